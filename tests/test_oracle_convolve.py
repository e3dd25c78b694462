"""Pins for the oracle's steps 7-8 (Gaussian PSF over (x, y), Gaussian LSF along the channel).
SURVEY.md 8(c) rows 7-8: delta response, partition of unity, scipy/numpy library routines,
flux conservation through PSF/LSF (BASELINE.json:north_star), commutation, transpose."""
import math

import numpy as np
import pytest
import scipy.ndimage as ndi

import oracle
from paper_2412_08265_b200 import synth

SIG_PSF = 3.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))     # FWHM 3 spaxels


def test_fwhm_to_sigma_constant():
    assert abs(SIG_PSF - 1.273983) < 5e-7                     # value quoted in SURVEY.md 8(c)-7
    assert abs(3.0 * synth.FWHM_TO_SIGMA - SIG_PSF) < 1e-15
    t = synth.make_telescope("medium")
    assert (t.psf_size, t.lsf_size) == (15, 9) and float(t.lsf_sigma) == 2.0
    assert abs(float(t.psf_sigma) - SIG_PSF) < 1e-7
    # half maximum at +-FWHM/2
    assert abs(math.exp(-(1.5 ** 2) / (2 * SIG_PSF ** 2)) - 0.5) < 1e-12


@pytest.mark.parametrize("size,sigma", [(15, SIG_PSF), (9, 2.0), (1, 0.7), (5, 10.0)])
def test_taps(size, sigma):
    g = oracle.gauss_taps(size, sigma)
    h = (size - 1) // 2
    assert g.shape == (size,) and abs(g.sum() - 1.0) < 1e-15
    assert np.array_equal(g, g[::-1]) and g.argmax() == h
    for i in range(1, h + 1):                                  # point-sampled Gaussian ratios
        assert math.isclose(g[h + i] / g[h], math.exp(-i * i / (2 * sigma * sigma)), rel_tol=1e-13)


def test_truncation_losses_quoted_in_the_survey():
    raw = np.exp(-np.arange(-200, 201) ** 2 / (2 * SIG_PSF ** 2))
    assert 1 - raw[200 - 7:200 + 8].sum() / raw.sum() < 1e-7   # +-7 taps keep all but ~2e-9..4e-8
    raw = np.exp(-np.arange(-200, 201) ** 2 / 8.0)
    assert abs((1 - raw[196:205].sum() / raw.sum()) - 0.0244) < 2e-3   # +-2 sigma drops ~2.3-2.4 %


def test_delta_response_is_the_kernel():
    cube = np.zeros((21, 23, 31))
    cube[10, 11, 15] = 2.0
    out = oracle.convolve(cube, 15, SIG_PSF, 9, 2.0)
    g, h = oracle.gauss_taps(15, SIG_PSF), oracle.gauss_taps(9, 2.0)
    ref = np.zeros_like(cube)
    ref[3:18, 4:19, 11:20] = 2.0 * g[:, None, None] * g[None, :, None] * h[None, None, :]
    assert np.allclose(out, ref, rtol=1e-13, atol=1e-300)
    assert abs(out.sum() - 2.0) < 1e-14                        # flux conserved away from the edges


def test_equals_scipy_and_numpy_library_routines():
    cube = np.random.default_rng(3).random((20, 17, 40))
    g, h = oracle.gauss_taps(15, SIG_PSF), oracle.gauss_taps(9, 2.0)
    out = oracle.convolve(cube, 15, SIG_PSF, 9, 2.0)
    ref = ndi.convolve1d(cube, h, axis=2, mode="constant", cval=0.0)
    ref = ndi.convolve1d(ref, g, axis=0, mode="constant", cval=0.0)
    ref = ndi.convolve1d(ref, g, axis=1, mode="constant", cval=0.0)
    assert np.allclose(out, ref, rtol=1e-12, atol=1e-15)
    lsf_only = oracle.convolve(cube, 0, 0.0, 9, 2.0)
    assert np.allclose(lsf_only[4, 5], np.convolve(cube[4, 5], h, "same"), rtol=1e-13)
    psf_only = oracle.convolve(cube, 15, SIG_PSF, 0, 0.0)
    direct = ndi.convolve(cube[:, :, 7], np.outer(g, g), mode="constant", cval=0.0)   # 225 taps
    assert np.allclose(psf_only[:, :, 7], direct, rtol=1e-12)
    assert np.array_equal(oracle.convolve(cube, 0, 0.0, 0, 0.0), cube)


def test_non_symmetric_axes_are_not_mixed_up():
    """A cube that varies along x only must be smoothed along x only (and so on)."""
    g = oracle.gauss_taps(15, SIG_PSF)
    ramp = np.arange(30.0)
    cube = np.broadcast_to(ramp[:, None, None], (30, 18, 12)).copy()
    out = oracle.convolve(cube, 15, SIG_PSF, 0, 0.0)
    assert np.allclose(out[7:23, 9, 5], ramp[7:23], rtol=1e-13)       # linear ramp is a fixed point
    edge_y = np.convolve(np.ones(18), g, "same")
    assert np.allclose(out[15, :, 5], 15.0 * edge_y, rtol=1e-13)      # zero padding dims the y edges


def test_flux_conservation_and_constant_interior():
    g, h = oracle.gauss_taps(15, SIG_PSF), oracle.gauss_taps(9, 2.0)
    cube = np.zeros((40, 40, 50))
    cube[7:33, 7:33, 4:46] = np.random.default_rng(4).random((26, 26, 42))   # >= 7 / 4 from edges
    out = oracle.convolve(cube, 15, SIG_PSF, 9, 2.0)
    assert math.isclose(out.sum(), cube.sum(), rel_tol=1e-13)
    # at the edge, the flux that left the cube is exactly the zero-padded halo's share
    ones = np.ones((20, 20, 12))
    out = oracle.convolve(ones, 15, SIG_PSF, 9, 2.0)
    ex, ec = np.convolve(np.ones(20), g, "same"), np.convolve(np.ones(12), h, "same")
    assert np.allclose(out, ex[:, None, None] * ex[None, :, None] * ec[None, None, :], rtol=1e-13)
    assert np.allclose(out[7:13, 7:13, 4:8], 1.0, rtol=1e-13)          # constant interior stays


def test_psf_and_lsf_commute():
    cube = np.random.default_rng(6).random((18, 16, 30))
    a = oracle.convolve(oracle.convolve(cube, 15, SIG_PSF, 0, 0.0), 0, 0.0, 9, 2.0)
    b = oracle.convolve(oracle.convolve(cube, 0, 0.0, 9, 2.0), 15, SIG_PSF, 0, 0.0)
    assert np.allclose(a, b, rtol=1e-12) and np.allclose(a, oracle.convolve(cube, 15, SIG_PSF, 9, 2.0), rtol=1e-12)


def test_sampled_voxels_equal_full_convolution():
    cube32 = synth.synthetic_cube(19, 22, 37, seed=8)
    full = oracle.convolve(cube32.astype(np.float64), 15, SIG_PSF, 9, 2.0)
    vox = np.random.default_rng(9).choice(cube32.size, 500, replace=False)
    vox[:4] = [0, cube32.size - 1, 36, 37 * 22 * 9 + 5]
    got = oracle.convolve_voxels_f32(cube32, vox, 15, SIG_PSF, 9, 2.0)
    assert np.allclose(got, full.reshape(-1)[vox], rtol=1e-12)
    got = oracle.convolve_voxels_f32(cube32, vox, 15, SIG_PSF, 0, 0.0)
    assert np.allclose(got, oracle.convolve(cube32.astype(np.float64), 15, SIG_PSF, 0, 0.0).reshape(-1)[vox], rtol=1e-12)


def test_transpose_dot_product_and_self_adjointness():
    rng = np.random.default_rng(10)
    x, y = rng.normal(size=(17, 19, 23)), rng.normal(size=(17, 19, 23))
    Ax = oracle.convolve(x, 15, SIG_PSF, 9, 2.0)
    ATy = oracle.convolve_transpose(y, 15, SIG_PSF, 9, 2.0)
    assert math.isclose((Ax * y).sum(), (x * ATy).sum(), rel_tol=1e-11)
    # zero-padded symmetric stencils are self-adjoint
    assert np.allclose(ATy, oracle.convolve(y, 15, SIG_PSF, 9, 2.0), rtol=1e-11, atol=1e-13)
