"""Cell order and k_accumulate_cell (rubix_telescope.cell_order; SURVEY.md 8(d) row K3 "per-cell template reuse in heavy
spaxels", 7 "Contention config") through the C ABI: the cube against the fp64 oracle whichever kernel takes a spaxel, the
exported sort artefacts (unique parts bit for bit, the order inside a spaxel checked for validity), gradients independent
of the order."""
import dataclasses

import numpy as np
import pytest

import oracle
from sortcheck import check_perm
from paper_2412_08265_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

VOXEL_TOL = 1e-4


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no CPU fallback")
    from paper_2412_08265_b200 import binding
    binding.load()
    return binding


def with_order(w, order, **tel_changes):
    return dataclasses.replace(w, telescope=dataclasses.replace(w.telescope, cell_order=order, **tel_changes))


def artefacts(dw, w):
    t = w.telescope
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey) and np.array_equal(seg, oseg)
    return perm, operm, oseg


@pytest.mark.parametrize("name,resample", [("tiny", 0), ("tiny", 1), ("small", 0), ("small", 1)])
def test_forced_on_every_spaxel(B, name, resample):
    base = synth.make_workload(name, n=30000 if name == "small" else 4000)
    off = with_order(base, 1, resample=resample)
    on = with_order(base, 3, resample=resample)
    d_off, d_on = B.DeviceWorkload(off), B.DeviceWorkload(on)
    c_off, c_on = d_off.build_cube(), d_on.build_cube()
    torch.cuda.synchronize()
    perm, operm, oseg = artefacts(d_off, off)
    assert check_perm(perm, operm, oseg, base.particles, base.ssp, base.telescope.n_spaxels, False) == "stable"
    perm, operm, oseg = artefacts(d_on, on)
    if resample == 0:
        assert check_perm(perm, operm, oseg, base.particles, base.ssp, base.telescope.n_spaxels, True) == "cell"
        assert not np.array_equal(perm, operm)                 # the galaxies do spread over many cells
    else:                                                      # the cell order is for the point rule: silently off
        assert np.array_equal(perm, operm)
    ref = oracle.build_cube(base.particles, base.rotation, base.ssp, off.telescope)
    for cube in (c_off, c_on):
        got = cube.cpu().numpy().astype(np.float64)
        assert np.abs(got - ref).max() <= VOXEL_TOL * ref.max()
        assert not got[ref.sum(-1) == 0].any()
    # the two orders differ by fp32 rounding of the per-spaxel sums only
    assert (c_off - c_on).abs().max().item() <= 2e-6 * ref.max()
    again = d_on.build_cube()
    torch.cuda.synchronize()
    assert torch.equal(again, c_on)                            # bit-reproducible run to run


def test_forward_and_gradients_do_not_depend_on_the_order(B):
    base = synth.make_workload("adjoint", n=20000)
    off, on = with_order(base, 1), with_order(base, 3)
    d_off, d_on = B.DeviceWorkload(off), B.DeviceWorkload(on)
    f_off, f_on = d_off.forward(), d_on.forward()
    ref = oracle.forward(base.particles, base.rotation, base.ssp, base.telescope)
    for f in (f_off, f_on):
        assert np.abs(f.cpu().numpy() - ref).max() <= VOXEL_TOL * ref.max()
    rng = np.random.default_rng(3)
    grad = torch.from_numpy(rng.normal(size=d_on.shape).astype(np.float32)).cuda()
    g_off, g_on = d_off.adjoint(grad), d_on.adjoint(grad)
    torch.cuda.synchronize()
    for a, b2 in zip(g_off, g_on):                             # a particle's gradient is its own: no sum over particles
        assert torch.equal(a, b2)


def piled_up(n=200_000):
    """The contention galaxy (90 % in a Hernquist bulge of 0.2 kpc) on a 20 x 20 detector of 0.2 kpc spaxels: 500
    particles per spaxel on average, tens of thousands in the central ones, a handful at the rim."""
    base = synth.make_workload("contention", n=n)
    tel = dataclasses.replace(synth.make_telescope("contention"), n_x=20, n_y=20, psf_size=0, lsf_size=0)
    return dataclasses.replace(base, telescope=tel)


def test_auto_mode_splits_the_spaxels_between_the_kernels(B):
    w = piled_up(1_000_000)
    t = w.telescope
    assert t.cell_order == 0 and w.particles.n >= max(64 * t.n_spaxels, 1_000_000)
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    perm, operm, oseg = artefacts(dw, w)
    assert check_perm(perm, operm, oseg, w.particles, w.ssp, t.n_spaxels, True) == "cell"
    counts = np.diff(oseg)[:-1]
    threshold = 2 * w.ssp.log_age_axis.size * w.ssp.log_z_axis.size
    assert (counts >= threshold).sum() >= 4 and ((counts > 0) & (counts < threshold)).sum() >= 50   # both kernels get work
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    got = cube.cpu().numpy().astype(np.float64)
    assert np.abs(got - ref).max() <= VOXEL_TOL * ref.max()
    heavy = counts >= threshold
    g2, r2 = got.reshape(t.n_spaxels, -1), ref.reshape(t.n_spaxels, -1)
    for sel in (heavy, ~heavy):                                # each kernel's spaxels against their own maximum
        assert np.abs(g2[sel] - r2[sel]).max() <= VOXEL_TOL * r2[sel].max()
    pos = r2.sum(-1) > 0
    assert (np.abs(g2.sum(-1) - r2.sum(-1))[pos] / r2.sum(-1)[pos]).max() <= 1e-5
    # fewer than 10^6 particles: the auto mode stays off (stable order, k_accumulate alone); ON does what AUTO did above
    few = dataclasses.replace(w, particles=w.particles.subset(np.arange(200_000)))
    dw2 = B.DeviceWorkload(few)
    dw2.build_cube()
    torch.cuda.synchronize()
    perm, operm, oseg = artefacts(dw2, few)
    assert np.array_equal(perm, operm)
    on = with_order(w, 2)
    d_on = B.DeviceWorkload(on)
    assert torch.equal(d_on.build_cube(), cube)


def test_windows_too_far_apart_for_one_table(B):
    """Channel spacing close to the SSP spacing and line-of-sight speeds up to the 0.05 c cut: the windows of one unit no
    longer fit one table, so every particle loads its own range (the kernel's fallback) -- same cube."""
    ssp = synth.make_ssp(6, 3, 4300, 3000.0, 10000.0, 77)
    tel = synth.Telescope(4, 4, np.float32(1.0), 3800, np.float32(3300.0), np.float32(0.985 * float(ssp.dlambda)), cell_order=3)
    p = synth.make_particles(3000, 5, kind="gauss")
    rng = np.random.default_rng(8)
    p.pos[:] = rng.uniform(-1.9, 1.9, p.pos.shape).astype(np.float32)
    p.vel[:] = rng.uniform(-14500.0, 14500.0, p.vel.shape).astype(np.float32)    # |v_los| up to 0.048 c
    w = synth.Workload("spread", p, ssp, tel, np.eye(3, dtype=np.float32), (0.0, 0.0, 0.0))
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    ref = oracle.build_cube(p, w.rotation, ssp, tel)
    assert ref.max() > 0
    assert np.abs(cube.cpu().numpy() - ref).max() <= VOXEL_TOL * ref.max()
    tel_off = dataclasses.replace(tel, cell_order=1)
    c_off = B.DeviceWorkload(dataclasses.replace(w, telescope=tel_off)).build_cube()
    assert (cube - c_off).abs().max().item() <= 2e-6 * ref.max()


def test_batched_and_fused_calls_under_the_cell_order(B):
    """rubix_forward_batched keys are b N_s + spaxel: the composite sort key carries the cell below them."""
    base = synth.make_workload("tiny", n=3000)
    tel = dataclasses.replace(base.telescope.with_psf_lsf(), cell_order=3)
    batch = 5
    R = np.stack([synth.euler_rotation(*synth.random_euler(60 + b)) for b in range(batch)]).astype(np.float32)
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    p = base.particles
    arrays = [up(a) for a in (p.pos, p.vel, p.mass, p.log_age, p.log_z)]
    cp, cs, ct = B.c_particles(*arrays), B.c_ssp(base.ssp, up(base.ssp.flux)), B.c_telescope(tel)
    ws = torch.empty(B.rubix_forward_batched_workspace_bytes(p.n, None, batch, cs, ct), dtype=torch.uint8, device="cuda")
    cubes = torch.full((batch, tel.n_x, tel.n_y, tel.n_channels), float("nan"), dtype=torch.float32, device="cuda")
    B.rubix_forward_batched(cp, None, batch, cs, ct, R, cubes, ws)
    torch.cuda.synchronize()
    for b in range(batch):
        w1 = synth.Workload("one", p, base.ssp, tel, R[b], (0.0, 0.0, 0.0))
        assert torch.equal(cubes[b], B.DeviceWorkload(w1).forward()), b
    ref = oracle.forward(p, R[2], base.ssp, tel)
    assert np.abs(cubes[2].cpu().numpy() - ref).max() <= VOXEL_TOL * ref.max()


@pytest.mark.parametrize("order", [2, 3])
def test_mirrored_build_and_sharded_run_under_the_cell_order(B, order):
    """rubix_build_cube_mirrored through k_accumulate_cell (its own epilogue stores the mirrors) and the split between the two
    kernels (order 2: spaxels of >= 2 N_a N_z particles only); then the spaxel-sharded run, which fixes the order once for
    all ranks: slabs bit-equal to the single-GPU cube of the same order."""
    from paper_2412_08265_b200 import sharded
    base = synth.make_workload("tiny", n=6000)
    base.particles.pos[:2500, :2] *= np.float32(0.03)                    # a pile-up: multi-chunk spaxels above the threshold of order 2
    base.particles.pos[2500:3200, 0] = np.float32(-7.5)                  # ... and some in the first detector row
    w = with_order(base, order)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    plain = dw.build_cube()
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    assert np.abs(plain.cpu().numpy() - ref).max() <= VOXEL_TOL * ref.max()
    for rows in (1, 5, t.n_x):
        cube = torch.full(dw.shape, float("nan"), device="cuda")
        lo = torch.full((rows, t.n_y, t.n_channels), float("nan"), device="cuda")
        hi = torch.full((rows, t.n_y, t.n_channels), float("nan"), device="cuda")
        B.rubix_build_cube_mirrored(dw.particles, dw.ssp, dw.tel, dw.R, cube, lo, hi, rows, dw.workspace)
        torch.cuda.synchronize()
        assert torch.equal(cube, plain) and torch.equal(lo, plain[:rows]) and torch.equal(hi, plain[t.n_x - rows:])
    wc = dataclasses.replace(w, telescope=t.with_psf_lsf(psf_size=7))
    single = B.DeviceWorkload(wc).forward()
    backend = sharded.CudaBackend()
    p = wc.particles
    world = 3

    def rank_fn(comm):
        sl = sharded.slice_for_rank(p.n, comm.rank, comm.world)
        rec = sharded.pack_records(p.subset(np.arange(p.n)[sl]), "cuda")
        return sharded.forward_sharded(comm, backend, rec, wc.rotation, wc.ssp, wc.telescope)

    slabs = sharded.run_threads(world, rank_fn)
    torch.cuda.synchronize()
    for s in slabs:
        assert torch.equal(s.cube, single[s.x0:s.x1]), (s.x0, s.x1)
