"""rubix_forward (steps 1-8 in one device call, occupancy-masked PSF/LSF passes) against the two plain calls (bit for
bit) and against the fp64 oracle, through the C ABI.  SURVEY.md 8(a) rows 1-8, 8(d) rows K4-K6; VERDICT r01 item 4.

The workspace and the output are poisoned with NaN before every call: a stencil pass that read a row the accumulate
kernel did not write (an empty spaxel), or an unwritten row of the temporary, shows up as NaN in the result."""
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


def poisoned_forward(B, dw):
    dw.workspace.view(torch.float32).fill_(float("nan"))
    out = torch.full(dw.shape, float("nan"), dtype=torch.float32, device="cuda")
    dw.forward(out=out)
    torch.cuda.synchronize()
    return out


def check(B, w, what, oracle_too=True):
    t = w.telescope
    dw = B.DeviceWorkload(w)
    got = poisoned_forward(B, dw)
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey) and np.array_equal(seg, oseg), what
    check_perm(perm, operm, oseg, w.particles, w.ssp, t.n_spaxels, None)
    assert torch.isfinite(got).all(), what
    two = dw.forward_two_calls()
    torch.cuda.synchronize()
    assert torch.equal(got, two), (what, "rubix_forward differs from rubix_build_cube + rubix_convolve_psf_lsf")
    if oracle_too:
        ref = oracle.forward(w.particles, w.rotation, w.ssp, t)
        g = got.cpu().numpy().astype(np.float64)
        scale = max(np.abs(ref).max(), 1e-30)
        assert np.abs(g - ref).max() <= 1e-4 * scale, (what, np.abs(g - ref).max() / scale)
    return got


def sparse_workload(n_x, n_y, n_c, seed, n=400, clumps=3, **tel_kw):
    """A few clumps and a few isolated particles on an otherwise empty detector (most spaxels unoccupied)."""
    rng = np.random.default_rng(seed)
    w = synth.make_workload("tiny", n=n)
    s = 1.0
    centres = rng.uniform(-0.4, 0.4, (clumps, 2)) * np.array([n_x, n_y]) * s
    which = rng.integers(0, clumps, n)
    xy = centres[which] + rng.normal(0, 0.7, (n, 2))
    iso = rng.random(n) < 0.05
    xy[iso] = rng.uniform(-0.5, 0.5, (int(iso.sum()), 2)) * np.array([n_x, n_y]) * s
    w.particles.pos[:, 0] = xy[:, 0]
    w.particles.pos[:, 1] = xy[:, 1]
    w.rotation = np.eye(3, dtype=np.float32)
    w.telescope = synth.Telescope(n_x, n_y, np.float32(s), n_c, np.float32(4700.0), np.float32(4600.0 / max(n_c - 1, 1)),
                                  **tel_kw).with_psf_lsf()
    return w


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_configs_with_psf_lsf(B, name):
    w = synth.make_workload(name)
    w.telescope = w.telescope.with_psf_lsf()
    check(B, w, name)


@pytest.mark.parametrize("n_x,n_y,n_c", [(40, 36, 256), (33, 5, 130), (4, 47, 58), (1, 1, 64), (16, 16, 3700), (61, 17, 112)])
def test_sparse_detectors(B, n_x, n_y, n_c):
    w = sparse_workload(n_x, n_y, n_c, seed=n_x * 100 + n_y)
    t = w.telescope
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    check(B, w, f"{n_x}x{n_y}x{n_c}")
    if n_x * n_y > 500:
        assert np.unique(key[key < t.n_spaxels]).size < 0.5 * t.n_spaxels     # the mask really has holes


def test_stage_combinations_and_generic_stencils(B):
    base = sparse_workload(30, 28, 128, seed=5)
    t = base.telescope
    for what, tel in [
        ("LSF only", dataclasses.replace(t, psf_size=0)),
        ("PSF only", dataclasses.replace(t, lsf_size=0)),
        ("both off", dataclasses.replace(t, psf_size=0, lsf_size=0)),
        ("small stencils", dataclasses.replace(t, psf_size=5, lsf_size=3)),
        ("generic path: 17-tap PSF", dataclasses.replace(t, psf_size=17)),
        ("generic path: 11-tap LSF", dataclasses.replace(t, lsf_size=11)),
        ("generic path: odd channel count", dataclasses.replace(t, n_channels=127)),
        ("wavelength-dependent PSF", dataclasses.replace(t, psf_alpha=np.float32(-0.3), psf_lambda_ref=np.float32(6000.0))),
        ("flux-conserving rule", dataclasses.replace(t, resample=1)),
    ]:
        w = dataclasses.replace(base, telescope=tel)
        check(B, w, what)


def test_no_particles_and_all_dropped(B):
    w = sparse_workload(20, 20, 64, seed=9, n=50)
    w.particles.pos[:, 0] = 1e6                               # everything outside the field of view
    got = check(B, w, "all dropped", oracle_too=False)
    assert not got.any()
    w0 = dataclasses.replace(w, particles=w.particles.subset(np.arange(0)))
    got = check(B, w0, "n = 0", oracle_too=False)
    assert not got.any()


def test_one_particle_in_a_corner_and_dense_detector(B):
    w = sparse_workload(24, 24, 96, seed=11, n=1)
    w.particles.pos[0, :2] = (-11.5, 11.5)
    got = check(B, w, "corner").cpu().numpy()
    assert got[0:8, 16:24].any() and not got[8:, :16].any()
    wd = synth.make_workload("tiny", n=20000)                  # every spaxel occupied: the all-ones mask
    wd.telescope = wd.telescope.with_psf_lsf()
    t = wd.telescope
    key, _ = oracle.rotate_bin(wd.particles.pos, wd.particles.vel, wd.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert np.unique(key[key < t.n_spaxels]).size > 0.9 * t.n_spaxels
    check(B, wd, "dense")


def test_medium_sized_detector_against_two_calls(B):
    """BASELINE.json configs[2] geometry (300x300x3700, 24 % of the spaxels occupied) at the bench's launch configuration:
    bit-equal to the two plain calls (whose parity with the oracle test_gpu_parity.py checks on the whole cube)."""
    w = synth.make_workload("medium")
    dw = B.DeviceWorkload(w)
    got = poisoned_forward(B, dw)
    assert torch.isfinite(got).all()
    two = dw.forward_two_calls()
    torch.cuda.synchronize()
    assert torch.equal(got, two)
