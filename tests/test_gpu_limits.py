"""The CUDA path at the limits of its implementation (include/rubix.h "Limits"; csrc/common.cuh): SSP axes of 512 x 128
nodes, 63-tap stencils, a key space that needs three radix passes, tens of channel tiles, windows close to the 4096-sample
table, the steepest sampling ratio the resampler takes -- each against the fp64 oracle, and the first value beyond each limit
refused with a status code."""
import dataclasses

import numpy as np
import pytest

import oracle
from sortcheck import check_perm
from paper_2412_08265_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no CPU fallback")
    from paper_2412_08265_b200 import binding
    binding.load()
    return binding


def check(B, w, what, sample=None):
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube(out=torch.full(dw.shape, float("nan"), device="cuda"))
    torch.cuda.synchronize()
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey) and np.array_equal(seg, oseg), what
    check_perm(perm, operm, oseg, w.particles, w.ssp, t.n_spaxels, None)
    assert torch.isfinite(cube).all(), what
    if sample is None:
        ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
        got = cube.cpu().numpy().astype(np.float64)
    else:                                                   # occupied spaxels drawn at random + the emptiness of the rest
        occ = np.unique(okey[okey < t.n_spaxels])
        sel = np.random.default_rng(1).choice(occ, min(sample, occ.size), replace=False).astype(np.int32)
        ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t, sel=sel)
        flat = cube.reshape(t.n_spaxels, t.n_channels)
        got = flat[torch.from_numpy(sel.astype(np.int64)).cuda()].cpu().numpy().astype(np.float64)
        empty = np.ones(t.n_spaxels, bool)
        empty[occ] = False
        assert not flat[torch.from_numpy(np.flatnonzero(empty)).cuda()].any(), what
    assert np.abs(got - ref).max() <= 1e-4 * np.abs(ref).max(), (what, np.abs(got - ref).max() / np.abs(ref).max())
    return dw, cube


def test_largest_ssp_axes(B):
    w = synth.make_workload("tiny", n=4000)
    w.ssp = synth.make_ssp(512, 128, 64, 3500.0, 9500.0, seed=7)                 # kMaxAge x kMaxZ nodes
    w.telescope = dataclasses.replace(w.telescope, n_channels=40, dlambda=np.float32(100.0))
    check(B, w, "512 x 128 SSP nodes")
    big = dataclasses.replace(w, ssp=synth.make_ssp(513, 4, 64, 3500.0, 9500.0, seed=7))
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(big).build_cube()
    assert B.rubix_last_error() != ""


def test_three_radix_passes_and_many_spaxels(B):
    w = synth.make_workload("small", n=300000)
    w.telescope = synth.Telescope(600, 620, np.float32(0.05), 8, np.float32(4750.0), np.float32(500.0))   # 372 000 keys: 19 bits
    w.ssp = synth.make_ssp(6, 4, 200, 3000.0, 10000.0, seed=3)
    dw, _ = check(B, w, "600 x 620 spaxels", sample=400)


def test_63_tap_stencils(B):
    w = synth.make_workload("tiny", n=500)
    w.telescope = dataclasses.replace(w.telescope.with_psf_lsf(fwhm_spaxels=9.0, psf_size=63, lsf_sigma=8.0, lsf_size=63), n_x=70, n_y=66,
                                      n_channels=130, dlambda=np.float32(30.0))
    t = w.telescope
    dw = B.DeviceWorkload(w)
    final = dw.forward().cpu().numpy().astype(np.float64)
    ref = oracle.forward(w.particles, w.rotation, w.ssp, t)
    assert np.abs(final - ref).max() <= 1e-4 * ref.max()
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(dataclasses.replace(w, telescope=dataclasses.replace(t, psf_size=65))).forward()


@pytest.mark.parametrize("resample", [0, 1])
def test_many_channel_tiles_and_the_steepest_sampling(B, resample):
    w = synth.make_workload("tiny", n=300)
    # 20 000 channels of 0.25 A on the 11.7 A grid (a window of a few hundred samples, six tiles of 29 x 128 channels)
    w.telescope = synth.Telescope(4, 4, np.float32(4.0), 20000, np.float32(4000.0), np.float32(0.25), resample=resample)
    check(B, w, "20 000 channels")
    # d x / d channel = 14.2 / (1 - 0.05): the steepest ratio the resampler takes; one channel per thread, table of 4096 samples
    ssp = synth.make_ssp(4, 3, 3000, 3500.0, 9500.0, seed=5)
    steep = synth.Telescope(4, 4, np.float32(4.0), 200, np.float32(3600.0), np.float32(2.0007 * 13.4), resample=resample)
    check(B, dataclasses.replace(w, ssp=ssp, telescope=steep), "steepest sampling ratio")
    too_steep = dataclasses.replace(steep, dlambda=np.float32(2.0007 * 14.3))
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(dataclasses.replace(w, ssp=ssp, telescope=too_steep)).build_cube()


def test_a_window_close_to_the_table_capacity(B):
    """One channel tile of 29 x 128 channels spanning ~3 900 of the 4 096 table samples (B = 1.05 with the Doppler margin)."""
    w = synth.make_workload("tiny", n=600)
    w.ssp = synth.make_ssp(4, 3, 4300, 3000.0, 10000.0, seed=11)
    w.telescope = synth.Telescope(5, 5, np.float32(3.0), 3712, np.float32(3100.0), np.float32(1.6283 * 1.0))
    w.particles.vel[:, :] = np.random.default_rng(2).uniform(-8000.0, 8000.0, w.particles.vel.shape).astype(np.float32)
    check(B, w, "window near the table capacity")
