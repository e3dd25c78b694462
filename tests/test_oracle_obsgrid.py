"""Pins for the oracle with an EXPLICIT (non-uniform) observed wavelength array (reading R16;
SURVEY.md 8(f)-1 "arbitrary telescope grids"): F[k] = interpolant at lambda_obs[k] / ((1+z)(1+beta))."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C_KMS = 299792.458


def nonuniform(n_c, lo, hi, seed):
    rng = np.random.default_rng(seed)
    steps = rng.uniform(0.3, 1.7, n_c)
    lam = lo + (hi - lo) * np.cumsum(steps) / steps.sum()
    return lam.astype(np.float32)


def _ssp(log_grid, n_l=500, seed=2):
    rng = np.random.default_rng(seed)
    flux = rng.uniform(0.5, 2.0, (3, 3, n_l)).astype(np.float32)
    ax = (np.array([-1.0, 0.0, 1.0], np.float32), np.array([-3.0, -2.0, -1.5], np.float32))
    if log_grid:
        return synth.SSPGrid(*ax, np.float32(3500.0), np.float32(3.0e-4), flux, 1)
    return synth.SSPGrid(*ax, np.float32(3500.0), np.float32(3.0), flux, 0)


@pytest.mark.parametrize("log_grid", [False, True])
@pytest.mark.parametrize("v,z", [(0.0, 0.0), (420.0, 0.0), (-900.0, 0.1)])
def test_equals_numpy_interp_on_the_given_wavelengths(log_grid, v, z):
    ssp = _ssp(log_grid)
    lam = nonuniform(400, 3300.0 * (1 + z), 5300.0 * (1 + z), 7)
    t = synth.Telescope(1, 1, np.float32(1.0), 400, np.float32(0.0), np.float32(1.0), redshift=np.float32(z),
                        lambda_obs=lam)
    F = oracle.particle_spectrum(np.float32(1.5), np.float32(-1.0), np.float32(-3.0), np.float32(v), ssp, t)
    beta = float(np.float32(v)) / C_KMS
    rest = lam.astype(np.float64) / ((1 + float(np.float32(z))) * (1 + beta))
    T = ssp.flux[0, 0].astype(np.float64)
    if log_grid:
        ref = 1.5 * np.interp(np.log10(rest), np.log10(ssp.wavelengths()), T, left=0.0, right=0.0)
    else:
        ref = 1.5 * np.interp(rest, ssp.wavelengths(), T, left=0.0, right=0.0)
    edge = (np.abs(rest - ssp.wavelengths()[0]) < 1e-6) | (np.abs(rest - ssp.wavelengths()[-1]) < 1e-6)
    assert np.allclose(F[~edge], ref[~edge], rtol=1e-9, atol=1e-9)
    assert (F == 0).sum() > 10 and (F > 0).sum() > 200


def test_a_uniform_array_equals_the_uniform_grid_and_channels_permute_with_the_array():
    w = synth.make_workload("tiny", n=50)
    t = w.telescope
    lam = t.wavelengths().astype(np.float32)                       # k * dl + l0 rounded to fp32
    base = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    arr = oracle.build_cube(w.particles, w.rotation, w.ssp, dataclasses.replace(t, lambda_obs=lam))
    assert np.allclose(arr, base, rtol=0, atol=2e-3 * base.max())  # fp32 rounding of the wavelengths moves x_k by ~1e-4
    sub = lam[::3].copy()
    t3 = dataclasses.replace(t, n_channels=sub.size, lambda_obs=sub)
    assert np.array_equal(oracle.build_cube(w.particles, w.rotation, w.ssp, t3), arr[..., ::3])


@pytest.mark.parametrize("log_grid", [False, True])
def test_adjoint_matches_finite_differences_and_the_closed_form(log_grid):
    n = 300
    w = synth.make_workload("tiny", n=n)
    w.ssp = synth.make_ssp(6, 4, 600, 3500.0, 9500.0, seed=9, log_lambda=log_grid)
    lam = nonuniform(256, 4700.0, 9300.0, 3)
    t = dataclasses.replace(w.telescope.with_psf_lsf(), lambda_obs=lam)
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    resid = oracle.forward(w.particles, w.rotation, w.ssp, t) - oracle.forward(other, w.rotation, w.ssp, t)
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ok = key < t.n_spaxels
    if not log_grid:
        ok &= oracle.knot_clearance(vlos, ssp, t) > 1e-4
    else:
        beta = vlos.astype(np.float64)[:, None] / C_KMS
        xk = np.log10(lam.astype(np.float64)[None, :] / (1 + beta) / float(ssp.lambda0)) / float(ssp.dlambda)
        ok &= np.abs(xk - np.round(xk)).min(1) > 1e-4
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(5).choice(np.nonzero(ok)[0], 25, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), q
    if not log_grid:                                               # T = a + b lambda: dF_k/dv = -m b lambda_k / (c (1+beta)^2)
        n_l, a, b = 400, 2.0, 2.0 ** -12
        lin = synth.SSPGrid(np.array([-1, 0, 1], np.float32), np.array([-4, -3, -2], np.float32), np.float32(3000.0),
                            np.float32(2.5), np.ascontiguousarray(np.broadcast_to(a + b * (3000.0 + 2.5 * np.arange(n_l)),
                                                                                  (3, 3, n_l)), np.float32))
        lam2 = nonuniform(100, 3100.0, 3900.0, 11)
        tt = synth.Telescope(4, 4, np.float32(1.0), 100, np.float32(0.0), np.float32(1.0), lambda_obs=lam2)
        p.pos[:] = np.random.default_rng(0).uniform(-1.9, 1.9, p.pos.shape)
        R = np.eye(3, dtype=np.float32)
        G = np.random.default_rng(3).normal(size=(4, 4, 100))
        key, vlos = oracle.rotate_bin(p.pos, p.vel, R, 4, 4, 1.0)
        rows = G.reshape(16, -1)[key]
        be = vlos.astype(np.float64) / C_KMS
        g_v = oracle.adjoint(p, R, lin, tt, G)[3]
        assert np.allclose(g_v, -(p.mass * b / (C_KMS * (1 + be) ** 2)) * (rows * lam2.astype(np.float64)).sum(1), rtol=1e-9)
