"""Pins for the oracle's wavelength-dependent PSF (reading R18):
sigma_k = psf_sigma (lambda_k / lambda_ref)^alpha, final = PSF_k(LSF(cube))."""
import dataclasses

import numpy as np
import pytest
from scipy import ndimage

import oracle
from paper_2412_08265_b200 import synth


def _tel(n_c=24, alpha=-0.2):
    t = synth.Telescope(11, 9, np.float32(1.0), n_c, np.float32(4800.0), np.float32(150.0)).with_psf_lsf()
    return dataclasses.replace(t, psf_alpha=np.float32(alpha), psf_lambda_ref=np.float32(6000.0))


def test_sigma_law_and_per_channel_scipy_convolution():
    t = _tel()
    sk = oracle.psf_sigma_k(t)
    lam = t.wavelengths()
    assert np.allclose(sk, float(t.psf_sigma) * (lam / 6000.0) ** float(np.float32(-0.2)), rtol=1e-12)
    assert sk[0] > float(t.psf_sigma) > sk[-1]                         # seeing improves towards the red
    cube = synth.synthetic_cube(t.n_x, t.n_y, t.n_channels, seed=4).astype(np.float64)
    got = oracle.convolve(cube, t.psf_size, t.psf_sigma, 0, 0.0, sk)
    for k in range(t.n_channels):                                      # library routine, channel by channel
        g = oracle.gauss_taps(t.psf_size, sk[k])
        ref = ndimage.convolve1d(ndimage.convolve1d(cube[..., k], g, axis=0, mode="constant"), g, axis=1, mode="constant")
        assert np.allclose(got[..., k], ref, rtol=1e-12, atol=1e-15)
    # delta response of channel k is its own normalised kernel
    d = np.zeros_like(cube)
    d[5, 4, :] = 1.0
    r = oracle.convolve(d, t.psf_size, t.psf_sigma, 0, 0.0, sk)
    assert np.allclose(r.sum((0, 1)), [oracle.gauss_taps(15, s)[2:13].sum() * oracle.gauss_taps(15, s)[3:12].sum() for s in sk])


def test_order_is_lsf_then_psf_and_alpha_zero_is_the_constant_psf():
    t = _tel()
    sk = oracle.psf_sigma_k(t)
    cube = synth.synthetic_cube(t.n_x, t.n_y, t.n_channels, seed=5).astype(np.float64)
    both = oracle.convolve(cube, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, sk)
    lsf_first = oracle.convolve(oracle.convolve(cube, 0, 0.0, t.lsf_size, t.lsf_sigma), t.psf_size, t.psf_sigma, 0, 0.0, sk)
    psf_first = oracle.convolve(oracle.convolve(cube, t.psf_size, t.psf_sigma, 0, 0.0, sk), 0, 0.0, t.lsf_size, t.lsf_sigma)
    assert np.allclose(both, lsf_first, rtol=1e-13)
    assert np.abs(both - psf_first).max() > 1e-5 * both.max()          # they no longer commute
    assert oracle.psf_sigma_k(dataclasses.replace(t, psf_alpha=np.float32(0.0))) is None
    same = oracle.convolve(cube, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, np.full(t.n_channels, float(t.psf_sigma)))
    assert np.allclose(same, oracle.convolve(cube, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma), rtol=1e-14)
    vox = np.random.default_rng(1).integers(0, cube.size, 40)
    brute = oracle.convolve_voxels_f32(cube.astype(np.float32), vox, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, sk)
    assert np.allclose(brute, oracle.convolve(cube.astype(np.float32).astype(np.float64), t.psf_size, t.psf_sigma, t.lsf_size,
                                              t.lsf_sigma, sk).reshape(-1)[vox], rtol=1e-12)


def test_transpose_is_the_adjoint_of_the_forward():
    t = _tel()
    sk = oracle.psf_sigma_k(t)
    rng = np.random.default_rng(2)
    x, y = rng.normal(size=(t.n_x, t.n_y, t.n_channels)), rng.normal(size=(t.n_x, t.n_y, t.n_channels))
    Ax = oracle.convolve(x, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, sk)
    Aty = oracle.convolve_transpose(y, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, sk)
    assert np.isclose((Ax * y).sum(), (x * Aty).sum(), rtol=1e-12)
    # and the transpose is NOT the forward any more (PSF_k and LSF do not commute)
    assert np.abs(Aty - oracle.convolve(y, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma, sk)).max() > 1e-6


def test_adjoint_through_the_wavelength_dependent_psf_matches_finite_differences():
    n = 300
    w = synth.make_workload("tiny", n=n)
    t = dataclasses.replace(w.telescope.with_psf_lsf(), psf_alpha=np.float32(-0.3), psf_lambda_ref=np.float32(7000.0))
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    resid = oracle.forward(w.particles, w.rotation, w.ssp, t) - oracle.forward(other, w.rotation, w.ssp, t)
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ok = (key < t.n_spaxels) & (oracle.knot_clearance(vlos, ssp, t) > 1e-4)
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(4).choice(np.nonzero(ok)[0], 25, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), q
    g0 = oracle.adjoint(w.particles, w.rotation, w.ssp, dataclasses.replace(t, psf_alpha=np.float32(0.0)), 2.0 * resid)
    assert np.abs(g0[0][idx] - g[0][idx]).max() > 1e-4 * np.abs(g[0][idx]).max()
