"""The spaxel-sharded forward (paper_2412_08265_b200/sharded.py) with the CUDA backend: R ranks run
as threads of one process on one GPU (host-side waits only), every slab compared bit for bit with the single-GPU cube and
with the oracle.  Also the two C-ABI additions it needs: rubix_bin_particles and the row window of rubix_telescope."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import sharded, synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no CPU fallback")
    from paper_2412_08265_b200 import binding
    binding.load()
    return binding


def test_bin_particles_and_row_window(B):
    w = synth.make_workload("small", n=30000)
    t = w.telescope
    rec = sharded.pack_records(w.particles, "cuda")
    key = sharded.CudaBackend().bin(rec, t, w.rotation).cpu().numpy()
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert np.array_equal(key, okey)
    full = B.DeviceWorkload(w).build_cube()
    for x0, x1 in ((0, 25), (0, 9), (9, 17), (17, 25), (12, 13)):
        sub = dataclasses.replace(w, telescope=dataclasses.replace(t, n_x=x1 - x0, n_x_full=t.n_x, x_first=x0))
        dw = B.DeviceWorkload(sub)
        rows = dw.build_cube()
        assert torch.equal(rows, full[x0:x1]), (x0, x1)
        k2 = dw.sort_artifacts()[0].cpu().numpy()
        inside = (okey < t.n_spaxels) & (okey // t.n_y >= x0) & (okey // t.n_y < x1)
        assert np.array_equal(k2, np.where(inside, okey - x0 * t.n_y, (x1 - x0) * t.n_y))
    bad = dataclasses.replace(w, telescope=dataclasses.replace(t, n_x=10, n_x_full=t.n_x, x_first=20))
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(bad).build_cube()


def test_mirrored_build_writes_the_boundary_rows_twice(B):
    """rubix_build_cube_mirrored: the cube equals rubix_build_cube's, and the first / last rows also land in the mirrors
    (single- and multi-chunk spaxels: direct stores of k_accumulate and the sums of k_reduce_partials)."""
    w = synth.make_workload("small", n=60000)
    w.particles.pos[:4000, :2] *= np.float32(0.02)                       # a pile-up in the centre and ...
    w.particles.pos[4000:8000, 0] = np.float32(-14.5)                    # ... one in the first detector row (multi-chunk there)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    plain = dw.build_cube()
    for rows in (1, 7, t.n_x):
        cube = torch.full(dw.shape, float("nan"), device="cuda")
        lo = torch.full((rows, t.n_y, t.n_channels), float("nan"), device="cuda")
        hi = torch.full((rows, t.n_y, t.n_channels), float("nan"), device="cuda")
        B.rubix_build_cube_mirrored(dw.particles, dw.ssp, dw.tel, dw.R, cube, lo, hi, rows, dw.workspace)
        torch.cuda.synchronize()
        assert torch.equal(cube, plain) and torch.equal(lo, plain[:rows]) and torch.equal(hi, plain[t.n_x - rows:])
    cube = torch.full(dw.shape, float("nan"), device="cuda")
    hi = torch.full((3, t.n_y, t.n_channels), float("nan"), device="cuda")
    B.rubix_build_cube_mirrored(dw.particles, dw.ssp, dw.tel, dw.R, cube, None, hi, 3, dw.workspace)
    torch.cuda.synchronize()
    assert torch.equal(cube, plain) and torch.equal(hi, plain[t.n_x - 3:])
    with pytest.raises(B.RubixError):
        B.rubix_build_cube_mirrored(dw.particles, dw.ssp, dw.tel, dw.R, cube, None, hi, 0, dw.workspace)


@pytest.mark.parametrize("fuse_halo", [True, False])
@pytest.mark.parametrize("name,world,psf_size", [("tiny", 2, 15), ("tiny", 4, 7), ("small", 3, 15), ("small", 5, 9), ("tiny", 3, 0)])
def test_sharded_slabs_equal_the_single_gpu_cube(B, name, world, psf_size, fuse_halo):
    w = synth.make_workload(name, n=None if name == "tiny" else 40000)
    if psf_size:
        w.telescope = w.telescope.with_psf_lsf(psf_size=psf_size)
    t = w.telescope
    single = B.DeviceWorkload(w).forward()
    backend = sharded.CudaBackend()
    p = w.particles

    def rank_fn(comm):
        sl = sharded.slice_for_rank(p.n, comm.rank, comm.world)
        rec = sharded.pack_records(p.subset(np.arange(p.n)[sl]), "cuda")
        return sharded.forward_sharded(comm, backend, rec, w.rotation, w.ssp, t, fuse_halo=fuse_halo)

    slabs = sharded.run_threads(world, rank_fn)
    assert slabs[0].x0 == 0 and slabs[-1].x1 == t.n_x
    for s in slabs:
        assert torch.equal(s.cube, single[s.x0:s.x1]), (s.x0, s.x1)
    ref = oracle.forward(w.particles, w.rotation, w.ssp, t)
    got = torch.cat([s.cube for s in slabs]).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-4 * np.abs(ref).max()
    counts = [s.n_received for s in slabs]
    assert sum(counts) == int((oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)[0] < t.n_spaxels).sum())
    if psf_size == 0:                                         # no halo, so no minimum slab height: the work is split evenly
        assert max(counts) < 0.5 * sum(counts)
