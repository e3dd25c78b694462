"""rubix_forward_batched (many galaxies / many orientations per call) through the
C ABI: every element bit-equal to a single rubix_forward call, and compared with the fp64 oracle element by element."""
import dataclasses

import numpy as np
import pytest

import oracle
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


def rotations(batch, seed):
    return np.stack([synth.euler_rotation(*synth.random_euler(seed + b)) for b in range(batch)]).astype(np.float32)


def run_batched(B, parts, offsets, batch, ssp, tel, R):
    """parts: one synth.Particles (concatenated galaxies, or the shared galaxy when offsets is None)."""
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    arrays = [up(a) for a in (parts.pos, parts.vel, parts.mass, parts.log_age, parts.log_z)]
    flux = up(ssp.flux)
    cp, cs, ct = B.c_particles(*arrays), B.c_ssp(ssp, flux), B.c_telescope(tel)
    ws = torch.empty(B.rubix_forward_batched_workspace_bytes(parts.n, offsets, batch, cs, ct), dtype=torch.uint8, device="cuda")
    ws.view(torch.float32).fill_(float("nan"))
    cubes = torch.full((batch, tel.n_x, tel.n_y, tel.n_channels), float("nan"), dtype=torch.float32, device="cuda")
    B.rubix_forward_batched(cp, offsets, batch, cs, ct, R, cubes, ws)
    torch.cuda.synchronize()
    return cubes, B.rubix_last_launch_count()


def single(B, parts, ssp, tel, R):
    w = synth.Workload("one", parts, ssp, tel, R, (0.0, 0.0, 0.0))
    return B.DeviceWorkload(w).forward()


def concat(gals):
    return synth.Particles(*(np.concatenate([getattr(g, f) for g in gals]) for f in ("pos", "vel", "mass", "log_age", "log_z")))


@pytest.mark.parametrize("conv", [False, True])
def test_many_galaxies_per_call(B, conv):
    base = synth.make_workload("tiny")
    tel = base.telescope.with_psf_lsf() if conv else base.telescope
    sizes = [1000, 1, 0, 317, 2500, 40]                        # ragged, one empty, one single-particle galaxy
    gals = [synth.make_particles_for("tiny", n=max(n, 1), seed=500 + i).subset(np.arange(n)) for i, n in enumerate(sizes)]
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    R = rotations(len(sizes), 40)
    cubes, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R)
    assert torch.isfinite(cubes).all()
    for b, g in enumerate(gals):
        one = single(B, g, base.ssp, tel, R[b])
        assert torch.equal(cubes[b], one), b
        ref = oracle.forward(g, R[b], base.ssp, tel)
        got = cubes[b].cpu().numpy().astype(np.float64)
        assert np.abs(got - ref).max() <= 1e-4 * max(np.abs(ref).max(), 1e-30), b
    assert not cubes[2].any()


def test_many_orientations_of_one_galaxy(B):
    base = synth.make_workload("tiny", n=3000)
    tel = base.telescope.with_psf_lsf()
    batch = 9
    R = rotations(batch, 77)
    cubes, _ = run_batched(B, base.particles, None, batch, base.ssp, tel, R)
    for b in range(batch):
        assert torch.equal(cubes[b], single(B, base.particles, base.ssp, tel, R[b])), b
    ref = oracle.forward(base.particles, R[4], base.ssp, tel)
    assert np.abs(cubes[4].cpu().numpy() - ref).max() <= 1e-4 * np.abs(ref).max()
    assert not torch.equal(cubes[0], cubes[1])


def test_more_elements_than_one_group_and_small_spectral_cubes(B):
    """70 elements = two groups (64 + 6); the small config's 3700-channel spectra on a cut-down 6 x 5 detector."""
    base = synth.make_workload("small", n=2500)
    tel = dataclasses.replace(base.telescope, n_x=6, n_y=5, spaxel_size=np.float32(4.0)).with_psf_lsf(psf_size=5, lsf_size=5)
    batch = 70
    sizes = [(37 * b) % 50 + 1 for b in range(batch)]
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    parts = base.particles.subset(np.arange(int(offsets[-1])))
    R = rotations(batch, 900)
    cubes, launches = run_batched(B, parts, offsets, batch, base.ssp, tel, R)
    assert torch.isfinite(cubes).all() and launches <= 2 * 24
    for b in (0, 1, 63, 64, 69):
        g = parts.subset(np.arange(offsets[b], offsets[b + 1]))
        assert torch.equal(cubes[b], single(B, g, base.ssp, tel, R[b])), b
        ref = oracle.forward(g, R[b], base.ssp, tel)
        assert np.abs(cubes[b].cpu().numpy() - ref).max() <= 1e-4 * np.abs(ref).max(), b


def test_variants_and_bad_arguments(B):
    base = synth.make_workload("tiny", n=800)
    R = rotations(3, 5)
    for tel in (dataclasses.replace(base.telescope, resample=1),
                dataclasses.replace(base.telescope.with_psf_lsf(), psf_size=17),                       # generic stencils
                dataclasses.replace(base.telescope.with_psf_lsf(), psf_alpha=np.float32(-0.2), psf_lambda_ref=np.float32(6000.0))):
        cubes, _ = run_batched(B, base.particles, None, 3, base.ssp, tel, R)
        for b in range(3):
            assert torch.equal(cubes[b], single(B, base.particles, base.ssp, tel, R[b])), (tel, b)
    log_ssp = synth.make_ssp(8, 4, 512, 3500.0, 9500.0, 2100, log_lambda=True)
    cubes, _ = run_batched(B, base.particles, None, 3, log_ssp, base.telescope, R)
    assert torch.equal(cubes[1], single(B, base.particles, log_ssp, base.telescope, R[1]))
    with pytest.raises(B.RubixError):
        run_batched(B, base.particles, np.array([0, 500, 400, 800]), 3, base.ssp, base.telescope, R)
    with pytest.raises(B.RubixError):
        run_batched(B, base.particles, np.array([0, 500, 700, 801]), 3, base.ssp, base.telescope, R)
    with pytest.raises(B.RubixError):
        run_batched(B, base.particles, None, 0, base.ssp, base.telescope, R[:0])


def test_groups_either_side_of_a_sort_chunk_threshold(B):
    """65 elements = two launch sequences whose particle counts (262 208 and 262 000) sit either side of the count at which the
    radix sort doubles its warp chunks: the smaller group needs MORE histogram rows than the larger one, and both layouts are
    carved out of one workspace sized for the larger group (the layout must be monotone in n)."""
    base = synth.make_workload("tiny")
    tel = base.telescope
    sizes = [4097] * 64 + [262_000]
    big = synth.make_particles_for("tiny", n=262_000, seed=910)
    gals = [big.subset(np.arange(i * 4097, (i + 1) * 4097)) for i in range(63)] + \
           [synth.make_particles_for("tiny", n=4097, seed=911), big]
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    R = rotations(len(sizes), 123)
    cubes, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R)
    assert torch.isfinite(cubes).all()
    for b in (0, 17, 63, 64):
        assert torch.equal(cubes[b], single(B, gals[b], base.ssp, tel, R[b])), b
