"""Pins for the oracle's cosmological redshift and flux scaling (reading R14; PAPER.md L40
"spectra are Doppler shifted based on the galaxy distance and line-of-sight velocity"):
lambda_rest = lambda_obs / ((1 + z)(1 + beta)), spectrum x flux_scale."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C_KMS = 299792.458


def _ssp(n_l=600, l0=3000.0, dl=1.5, seed=4):
    rng = np.random.default_rng(seed)
    flux = rng.uniform(0.5, 2.0, (3, 3, n_l)).astype(np.float32)
    return synth.SSPGrid(np.array([-1.0, 0.0, 1.0], np.float32), np.array([-3.0, -2.0, -1.5], np.float32),
                         np.float32(l0), np.float32(dl), flux)


def _tel(n_c, l0, dl, z=0.0, scale=1.0, resample=0):
    return synth.Telescope(1, 1, np.float32(1.0), n_c, np.float32(l0), np.float32(dl), resample=resample,
                           redshift=np.float32(z), flux_scale=np.float32(scale))


@pytest.mark.parametrize("z,v,scale", [(0.0, 0.0, 1.0), (0.05, 300.0, 1.0), (0.3, -700.0, 2.5e-3), (1.5, 90.0, 7.0)])
def test_equals_numpy_interp_at_the_doubly_shifted_wavelength(z, v, scale):
    ssp = _ssp()
    t = _tel(500, 3100.0 * (1 + z), 1.9 * (1 + z), z, scale)
    q = (np.float32(2.0), np.float32(-1.0), np.float32(-3.0))          # grid node (0, 0): blend = template
    F = oracle.particle_spectrum(q[0], q[1], q[2], np.float32(v), ssp, t)
    beta = float(np.float32(v)) / C_KMS
    zz, sc = float(np.float32(z)), float(np.float32(scale))
    lam_rest = t.wavelengths() / ((1 + zz) * (1 + beta))
    ref = sc * 2.0 * np.interp(lam_rest, ssp.wavelengths(), ssp.flux[0, 0].astype(np.float64), left=0.0, right=0.0)
    assert np.allclose(F, ref, rtol=1e-9, atol=1e-9)      # operation order of the two (1+z)(1+beta) divisions differs


def test_line_centroid_moves_to_lambda_1pz_1pvc():
    """BASELINE.json north_star pin 'a narrow synthetic line shifts to lambda(1+v/c)', with the cosmological
    factor: the absorption centroid lands on lambda_l (1+z)(1+v/c)."""
    n_l, lam_l, sig = 4000, 5000.0, 3.0
    lam = 4000.0 + 0.5 * np.arange(n_l)
    T = (1.0 - 0.6 * np.exp(-0.5 * ((lam - lam_l) / sig) ** 2)).astype(np.float32)
    ssp = synth.SSPGrid(np.array([-1.0, 1.0], np.float32), np.array([-3.0, -2.0], np.float32), np.float32(4000.0),
                        np.float32(0.5), np.ascontiguousarray(np.broadcast_to(T, (2, 2, n_l))))
    z, v = 0.2, 450.0
    for mode in (0, 1):
        t = _tel(3000, 5800.0, 0.2, z, 1.0, resample=mode)
        F = oracle.particle_spectrum(np.float32(1.0), np.float32(0.0), np.float32(-2.5), np.float32(v), ssp, t)
        depth = 1.0 - F
        centroid = (depth * t.wavelengths()).sum() / depth.sum()
        expect = lam_l * (1 + float(np.float32(z))) * (1 + v / C_KMS)
        assert abs(centroid - expect) < 0.01 * 0.2, (mode, centroid, expect)


def test_defaults_are_the_unshifted_unscaled_path_and_scale_is_linear():
    w = synth.make_workload("tiny", n=80)
    base = oracle.build_cube(w.particles, w.rotation, w.ssp, w.telescope)
    same = oracle.build_cube(w.particles, w.rotation, w.ssp,
                             dataclasses.replace(w.telescope, redshift=np.float32(0.0), flux_scale=np.float32(1.0)))
    assert np.array_equal(base, same)
    half = oracle.build_cube(w.particles, w.rotation, w.ssp, dataclasses.replace(w.telescope, flux_scale=np.float32(0.5)))
    assert np.allclose(half, 0.5 * base, rtol=1e-15)
    # z = 0.25 observed on a grid stretched by 1.25 is the z = 0 cube (rest-frame sampling is identical)
    t = w.telescope
    stretched = dataclasses.replace(t, lambda0=np.float32(float(t.lambda0) * 1.25), dlambda=np.float32(float(t.dlambda) * 1.25),
                                    redshift=np.float32(0.25))
    zc = oracle.build_cube(w.particles, w.rotation, w.ssp, stretched)
    assert np.allclose(zc, base, rtol=1e-6, atol=1e-9 * base.max())          # fp32 grid constants round


@pytest.mark.parametrize("mode", [0, 1])
def test_adjoint_with_redshift_and_scale_matches_finite_differences(mode):
    n = 400
    w = synth.make_workload("tiny", n=n)
    t0 = w.telescope.with_psf_lsf()
    t = dataclasses.replace(t0, lambda0=np.float32(float(t0.lambda0) * 1.1), dlambda=np.float32(float(t0.dlambda) * 1.1),
                            redshift=np.float32(0.1), flux_scale=np.float32(3.0e-2), resample=mode)
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    cube = oracle.forward(w.particles, w.rotation, w.ssp, t)
    resid = cube - oracle.forward(other, w.rotation, w.ssp, t)
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ok = key < t.n_spaxels
    if mode == 0:
        ok &= oracle.knot_clearance(vlos, ssp, t) > 1e-4
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(11).choice(np.nonzero(ok)[0], 30, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx, h_v=1e-3 if mode == 0 else 1e-2)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), (mode, q)


def test_linear_template_closed_form_with_redshift():
    """T = a + b lambda: F_k = s m (a + b lambda_k / ((1+z)(1+beta))), so
    dL/dv = -s m b sum_k G_k lambda_k / ((1+z) c (1+beta)^2) in both resampling modes (interior bins)."""
    n_l, a, b = 400, 2.0, 2.0 ** -12
    lam = 3000.0 + 2.5 * np.arange(n_l)
    ssp = synth.SSPGrid(np.array([-1, 0, 1], np.float32), np.array([-4, -3, -2], np.float32), np.float32(3000.0),
                        np.float32(2.5), np.ascontiguousarray(np.broadcast_to(a + b * lam, (3, 3, n_l)), np.float32))
    z, s = 0.25, 0.125
    w = synth.make_workload("tiny", n=30)
    p = w.particles
    p.pos[:] = np.random.default_rng(0).uniform(-1.9, 1.9, p.pos.shape)
    R = np.eye(3, dtype=np.float32)
    G = np.random.default_rng(3).normal(size=(4, 4, 100))
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, 4, 4, 1.0)
    rows = G.reshape(16, -1)[key]
    beta = vlos.astype(np.float64) / C_KMS
    for mode in (0, 1):
        t = synth.Telescope(4, 4, np.float32(1.0), 100, np.float32(3900.0), np.float32(7.5), resample=mode,
                            redshift=np.float32(z), flux_scale=np.float32(s))
        g_m, g_a, g_z, g_v = oracle.adjoint(p, R, ssp, t, G)
        lam_k = t.wavelengths()
        assert np.allclose(g_v, -(s * p.mass * b / ((1 + z) * C_KMS * (1 + beta) ** 2)) * (rows * lam_k).sum(1), rtol=1e-9)
        assert np.allclose(g_m, s * (rows * (a + b * lam_k[None, :] / ((1 + z) * (1 + beta[:, None])))).sum(1), rtol=1e-10)
