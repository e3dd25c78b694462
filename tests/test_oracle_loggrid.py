"""Pins for the oracle on a LOG-SAMPLED SSP grid (reading R15; PAPER.md L44:
the experiment's library is `Mastar_CB19_SLOG_1_5`, a log-sampled grid): lambda_j = lambda0 * 10^(j d),
sampling coordinate x = log10(lambda_rest / lambda0) / d, interpolant linear in x between knots."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C_KMS = 299792.458


def _ssp(n_l=500, l0=3500.0, dlog=1.0e-4 * 3, seed=2):
    rng = np.random.default_rng(seed)
    flux = rng.uniform(0.5, 2.0, (3, 3, n_l)).astype(np.float32)
    return synth.SSPGrid(np.array([-1.0, 0.0, 1.0], np.float32), np.array([-3.0, -2.0, -1.5], np.float32),
                         np.float32(l0), np.float32(dlog), flux, 1)


def _tel(n_c, l0, dl, z=0.0):
    return synth.Telescope(1, 1, np.float32(1.0), n_c, np.float32(l0), np.float32(dl), redshift=np.float32(z))


@pytest.mark.parametrize("v,z", [(0.0, 0.0), (350.0, 0.0), (-1200.0, 0.04), (9000.0, 0.0)])
def test_equals_numpy_interp_in_log_lambda(v, z):
    ssp = _ssp()
    t = _tel(700, 3400.0 * (1 + z), 2.1 * (1 + z), z)               # starts below the coverage, ends above it
    F = oracle.particle_spectrum(np.float32(1.5), np.float32(-1.0), np.float32(-3.0), np.float32(v), ssp, t)
    beta = float(np.float32(v)) / C_KMS
    lam_rest = t.wavelengths() / ((1 + float(np.float32(z))) * (1 + beta))
    lam_ssp = ssp.wavelengths()
    ref = 1.5 * np.interp(np.log10(lam_rest), np.log10(lam_ssp), ssp.flux[0, 0].astype(np.float64), left=0.0, right=0.0)
    inside = (lam_rest > lam_ssp[0] * (1 + 1e-9)) & (lam_rest < lam_ssp[-1] * (1 - 1e-9))
    assert inside.sum() > 300 and (~inside).sum() > 20
    assert np.allclose(F[inside], ref[inside], rtol=1e-9, atol=1e-9)
    assert not F[lam_rest < lam_ssp[0] * (1 - 1e-9)].any() and not F[lam_rest > lam_ssp[-1] * (1 + 1e-9)].any()


def test_a_doppler_shift_is_a_constant_offset_in_x():
    """On a log grid, observing at velocity v equals observing at rest on the grid divided by (1 + beta)."""
    ssp = _ssp()
    v = 640.0
    beta = float(np.float32(v)) / C_KMS
    t = _tel(400, 3600.0, 2.0)
    moved = oracle.particle_spectrum(np.float32(1.0), np.float32(0.3), np.float32(-2.2), np.float32(v), ssp, t)
    # the same rest wavelengths reached at v = 0 from a grid shrunk by (1 + beta) (fp32 grid constants round)
    t0 = _tel(400, 3600.0 / (1 + beta), 2.0 / (1 + beta))
    rest = oracle.particle_spectrum(np.float32(1.0), np.float32(0.3), np.float32(-2.2), np.float32(0.0), ssp, t0)
    assert np.allclose(moved, rest, rtol=0, atol=2e-3 * moved.max())   # random template: slope ~1 per sample
    smooth = synth.make_ssp(4, 3, 800, 3500.0, 6500.0, seed=5, log_lambda=True)
    moved = oracle.particle_spectrum(np.float32(1.0), np.float32(0.3), np.float32(-2.2), np.float32(v), smooth, t)
    rest = oracle.particle_spectrum(np.float32(1.0), np.float32(0.3), np.float32(-2.2), np.float32(0.0), smooth, t0)
    assert np.allclose(moved, rest, rtol=2e-5)


def test_node_reproduction_and_template_linear_in_x():
    ssp = _ssp(n_l=300)
    lam = ssp.wavelengths()
    # observed exactly on the knots (to fp32 rounding of the observed grid this needs a linear stretch: use 2 knots)
    t = _tel(2, float(np.float32(lam[10])), float(np.float32(lam[11] - lam[10])))
    F = oracle.particle_spectrum(np.float32(2.0), np.float32(-1.0), np.float32(-3.0), np.float32(0.0), ssp, t)
    assert np.allclose(F, 2.0 * ssp.flux[0, 0, 10:12], rtol=2e-4)
    # T linear in x = log10(lambda/lambda0)/d is reproduced exactly anywhere
    n_l = 300
    x = np.arange(n_l)
    lin = synth.SSPGrid(ssp.log_age_axis, ssp.log_z_axis, ssp.lambda0, ssp.dlambda,
                        np.ascontiguousarray(np.broadcast_to(1.0 + 0.125 * x, (3, 3, n_l)), np.float32), 1)
    t = _tel(150, 3520.0, 4.0)
    F = oracle.particle_spectrum(np.float32(1.0), np.float32(0.2), np.float32(-2.5), np.float32(200.0), lin, t)
    beta = 200.0 / C_KMS
    xk = np.log10(t.wavelengths() / (1 + beta) / float(lin.lambda0)) / float(lin.dlambda)
    inside = (xk >= 0) & (xk <= n_l - 1)
    assert np.allclose(F[inside], 1.0 + 0.125 * xk[inside], rtol=1e-10)


def test_adjoint_on_a_log_grid_matches_finite_differences_and_the_closed_form():
    n = 400
    w = synth.make_workload("tiny", n=n)
    w.ssp = synth.make_ssp(8, 4, 700, 3500.0, 9500.0, seed=9, log_lambda=True)
    t = w.telescope.with_psf_lsf()
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    cube = oracle.forward(w.particles, w.rotation, w.ssp, t)
    resid = cube - oracle.forward(other, w.rotation, w.ssp, t)
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    beta = vlos.astype(np.float64)[:, None] / C_KMS
    xk = np.log10(t.wavelengths()[None, :] / (1 + beta) / float(ssp.lambda0)) / float(ssp.dlambda)
    ok = (key < t.n_spaxels) & (np.abs(xk - np.round(xk)).min(1) > 1e-4)
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(3).choice(np.nonzero(ok)[0], 30, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), q
    # closed form: T = a + b x  =>  F_k = m (a + b x_k), dF_k/dv = -m b / (c (1+beta) d ln 10)
    n_l, a, b = 400, 2.0, 0.25
    lin = synth.SSPGrid(np.array([-1, 0, 1], np.float32), np.array([-4, -3, -2], np.float32), np.float32(3000.0),
                        np.float32(4.0e-4), np.ascontiguousarray(np.broadcast_to(a + b * np.arange(n_l), (3, 3, n_l)),
                                                                 np.float32), 1)
    tt = synth.Telescope(4, 4, np.float32(1.0), 100, np.float32(3100.0), np.float32(7.5))
    p.pos[:] = np.random.default_rng(0).uniform(-1.9, 1.9, p.pos.shape)
    R = np.eye(3, dtype=np.float32)
    G = np.random.default_rng(3).normal(size=(4, 4, 100))
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, 4, 4, 1.0)
    rows = G.reshape(16, -1)[key]
    be = vlos.astype(np.float64) / C_KMS
    g_m, g_a, g_z, g_v = oracle.adjoint(p, R, lin, tt, G)
    assert np.allclose(g_v, -(p.mass * b / (C_KMS * (1 + be) * float(lin.dlambda) * np.log(10.0))) * rows.sum(1), rtol=1e-9)
