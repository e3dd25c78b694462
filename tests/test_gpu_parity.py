"""Parity of the CUDA path (through the C ABI) against the fp64 oracle.  `-m gpu` only.

Tolerances are BASELINE.json:north_star's: spaxel assignment and sort order bit-exact; cube voxels
max|GPU - oracle| <= 1e-4 * max|oracle cube|; each spaxel's summed flux within 1e-5 relative;
empty spaxels exactly 0 before the PSF."""
import numpy as np
import pytest

import oracle
from sortcheck import check_perm
from gradcheck import assert_gradients
from paper_2412_08265_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

VOXEL_TOL = 1e-4
FLUX_TOL = 1e-5


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no CPU fallback")
    from paper_2412_08265_b200 import binding
    binding.load()
    return binding


def check_cube(gpu, ref, what=""):
    """gpu: fp32 array, ref: fp64 array of the same shape [..., n_c]."""
    gpu = np.asarray(gpu, np.float64)
    assert gpu.shape == ref.shape
    assert np.isfinite(gpu).all(), what
    scale = np.abs(ref).max()
    err = np.abs(gpu - ref).max()
    assert err <= VOXEL_TOL * scale, f"{what}: max err {err:.3e} vs {VOXEL_TOL * scale:.3e}"
    fs, fr = gpu.sum(-1), ref.sum(-1)
    pos = fr > 0
    rel = np.abs(fs[pos] - fr[pos]) / fr[pos]
    assert rel.size == 0 or rel.max() <= FLUX_TOL, f"{what}: spaxel flux rel err {rel.max():.3e}"
    assert not gpu[~pos].any(), f"{what}: empty spaxels must be exactly zero"
    return err / scale if scale > 0 else 0.0


def check_sort(dw, w):
    t = w.telescope
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey), "spaxel keys differ"
    assert np.array_equal(seg, oseg), "segment offsets differ"
    check_perm(perm, operm, oseg, w.particles, w.ssp, t.n_spaxels,
               {0: None, 1: False, 2: True, 3: True}[int(getattr(t, "cell_order", 0))])
    return okey, oseg


# ------------------------------------------------------------------ configs 0 and 1: whole cube
def test_tiny_whole_cube(B, tiny):
    dw = B.DeviceWorkload(tiny)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    check_sort(dw, tiny)
    ref = oracle.build_cube(tiny.particles, tiny.rotation, tiny.ssp, tiny.telescope)
    check_cube(cube.cpu().numpy(), ref, "tiny")


def test_small_whole_cube(B, small, small_oracle_cube):
    dw = B.DeviceWorkload(small)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    check_sort(dw, small)
    check_cube(cube.cpu().numpy(), small_oracle_cube, "small")
    again = dw.build_cube()
    torch.cuda.synchronize()
    assert torch.equal(cube, again), "build_cube must be bit-reproducible run to run"


def test_tiny_with_psf_lsf(B, tiny):
    w = synth.make_workload("tiny")
    w.telescope = w.telescope.with_psf_lsf()
    dw = B.DeviceWorkload(w)
    final = dw.forward()
    torch.cuda.synchronize()
    ref = oracle.forward(w.particles, w.rotation, w.ssp, w.telescope)
    g = final.cpu().numpy().astype(np.float64)
    assert np.abs(g - ref).max() <= VOXEL_TOL * ref.max()
    assert np.allclose(g.sum(-1), ref.sum(-1), rtol=FLUX_TOL, atol=FLUX_TOL * ref.sum(-1).max())


# ------------------------------------------------------------------ convolution alone
@pytest.mark.parametrize("shape,psf,lsf", [((19, 22, 37), 15, 9), ((8, 5, 64), 15, 9), ((30, 30, 100), 15, 0),
                                           ((30, 30, 101), 0, 9), ((12, 40, 256), 5, 3), ((6, 6, 16), 0, 0),
                                           ((1, 1, 33), 15, 9)])
def test_convolve_small_cubes(B, shape, psf, lsf):
    cube32 = synth.synthetic_cube(*shape, seed=11)
    tel = synth.Telescope(shape[0], shape[1], np.float32(1.0), shape[2], np.float32(5000.0), np.float32(1.0),
                          psf, np.float32(1.274 if psf else 0.0), lsf, np.float32(2.0 if lsf else 0.0))
    ctel = B.c_telescope(tel)
    d_in = torch.from_numpy(cube32).cuda()
    d_out = torch.full_like(d_in, float("nan"))
    ws = torch.empty(B.rubix_workspace_bytes(0, None, ctel), dtype=torch.uint8, device="cuda")
    B.rubix_convolve_psf_lsf(ctel, d_in, d_out, ws)
    torch.cuda.synchronize()
    ref = oracle.convolve(cube32.astype(np.float64), psf, tel.psf_sigma, lsf, tel.lsf_sigma)
    got = d_out.cpu().numpy().astype(np.float64)
    assert np.abs(got - ref).max() <= 2e-6 * np.abs(ref).max()
    assert torch.equal(d_in.cpu(), torch.from_numpy(cube32)), "input must not be modified"


def test_convolve_full_size_sampled_voxels(B):
    """300 x 300 x 3700 (the bench shape): brute-force oracle on sampled output voxels."""
    tel = synth.make_telescope("medium")
    cube32 = synth.synthetic_cube(tel.n_x, tel.n_y, tel.n_channels, seed=12)
    ctel = B.c_telescope(tel)
    d_in = torch.from_numpy(cube32).cuda()
    d_out = torch.empty_like(d_in)
    ws = torch.empty(B.rubix_workspace_bytes(0, None, ctel), dtype=torch.uint8, device="cuda")
    B.rubix_convolve_psf_lsf(ctel, d_in, d_out, ws)
    torch.cuda.synchronize()
    rng = np.random.default_rng(13)
    vox = rng.integers(0, cube32.size, 4000)
    nc, ny = tel.n_channels, tel.n_y
    corners = [((x * ny) + y) * nc + k for x in (0, 3, 150, 299) for y in (0, 149, 296, 299) for k in (0, 2, 1850, 3699)]
    vox = np.concatenate([vox, np.array(corners)])
    ref = oracle.convolve_voxels_f32(cube32, vox, tel.psf_size, tel.psf_sigma, tel.lsf_size, tel.lsf_sigma)
    got = d_out.view(-1)[torch.from_numpy(vox).cuda()].cpu().numpy().astype(np.float64)
    assert np.abs(got - ref).max() <= 2e-6 * np.abs(ref).max()
    # property that holds at any size: flux conservation away from the edges + linearity
    total_in = d_in[8:-8, 8:-8, 5:-5].double().sum().item()
    assert d_out.double().sum().item() >= total_in


# ------------------------------------------------------------------ config 2 (headline) at full size
@pytest.fixture(scope="module")
def medium():
    return synth.make_workload("medium")


def test_medium_full_size(B, medium):
    """The headline workload, WHOLE cube against the oracle: the build cube (steps 1-6) and the final cube (steps 7-8),
    every voxel; about 20 s of oracle time and 10 GB of host memory."""
    w = medium
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    okey, oseg = check_sort(dw, w)
    counts = np.diff(oseg)[:-1]
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    got = cube.cpu().numpy()
    # every empty spaxel is exactly zero (check_cube asserts it), every voxel within 1e-4 of the cube's maximum,
    # every spaxel's flux within 1e-5
    assert int((ref.reshape(t.n_spaxels, -1).sum(-1) > 0).sum()) == int((counts > 0).sum())
    check_cube(got, ref, "medium whole build cube")
    del got

    final = dw.convolve(cube)
    torch.cuda.synchronize()
    ref_final = oracle.convolve(ref, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma)
    del ref
    gotf = final.cpu().numpy()
    scale = ref_final.max()
    err = 0.0
    for x0 in range(0, t.n_x, 50):                         # in slabs: keeps the fp64 temporaries small
        d = gotf[x0:x0 + 50].astype(np.float64) - ref_final[x0:x0 + 50]
        err = max(err, float(np.abs(d).max()))
        fs, fr = gotf[x0:x0 + 50].astype(np.float64).sum(-1), ref_final[x0:x0 + 50].sum(-1)
        assert np.allclose(fs, fr, rtol=FLUX_TOL, atol=FLUX_TOL * float(ref_final.sum(-1).max()))
    assert err <= VOXEL_TOL * scale, f"medium whole final cube: max err {err:.3e} vs {VOXEL_TOL * scale:.3e}"


def test_forward_host_entries_against_the_oracle(B, small, small_oracle_cube):
    """rubix_forward_host and rubix_forward_host_pipelined (the calls bench.py's e2e leg times), HOST buffers in and
    out, compared with the oracle directly: config 1 as is (no PSF/LSF) and with config 2's PSF/LSF."""
    p = small.particles
    for tel, ref in ((small.telescope, small_oracle_cube),
                     (small.telescope.with_psf_lsf(), None)):
        if ref is None:
            ref = oracle.convolve(small_oracle_cube, tel.psf_size, tel.psf_sigma, tel.lsf_size, tel.lsf_sigma)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hp = [pin(x) for x in (p.pos, p.vel, p.mass, p.log_age, p.log_z)]
        hflux = pin(small.ssp.flux)
        cp, cs, ct = B.c_particles(*hp), B.c_ssp(small.ssp, hflux), B.c_telescope(tel)
        shape = (tel.n_x, tel.n_y, tel.n_channels)
        scratch = torch.empty(B.rubix_forward_host_pipelined_scratch_bytes(p.n, cs, ct), dtype=torch.uint8, device="cuda")
        h1 = torch.full(shape, float("nan"), dtype=torch.float32).pin_memory()
        B.rubix_forward_host(cp, cs, ct, small.rotation, h1, scratch)
        torch.cuda.synchronize()
        h2 = [torch.full(shape, float("nan"), dtype=torch.float32).pin_memory() for _ in range(3)]
        for h in h2:                                       # three back-to-back cubes through the pipeline
            B.rubix_forward_host_pipelined(cp, cs, ct, small.rotation, h, scratch)
        B.rubix_forward_host_drain()
        torch.cuda.synchronize()
        for h in [h1] + h2:
            got = h.numpy().astype(np.float64)
            assert np.isfinite(got).all()
            assert np.abs(got - ref).max() <= VOXEL_TOL * ref.max()
            assert np.allclose(got.sum(-1), ref.sum(-1), rtol=FLUX_TOL, atol=FLUX_TOL * ref.sum(-1).max())


# ------------------------------------------------------------------ config 3: contention
def test_contention(B):
    """10 M particles, 90 % in a compact bulge: sort bit-exact at full size; cube on sampled
    spaxels including the heaviest (the oracle spreads one spaxel over channel blocks)."""
    w = synth.make_workload("contention")
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    okey, oseg = check_sort(dw, w)
    counts = np.diff(oseg)[:-1]
    assert counts.max() > 0.03 * w.particles.n
    order = np.argsort(counts)
    rng = np.random.default_rng(15)
    # the heaviest spaxel (~1e6 particles x 3700 channels = a few 1e9 oracle samples, ~10 s), the
    # 5th..8th heaviest (still > 1e5 particles, thousands of chunks) plus lighter ones
    sel = np.unique(np.concatenate([order[-1:], order[-8:-4], order[-400:-8:60],
                                    rng.choice(np.nonzero(counts > 0)[0], 30)])).astype(np.int32)
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t, sel=sel)
    got = cube.view(t.n_spaxels, -1)[torch.from_numpy(sel.astype(np.int64)).cuda()].cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    # tolerance relative to the cube's global maximum, read from the GPU cube after checking the
    # sampled heavy spaxels against their own maximum (stricter)
    assert np.abs(got - ref).max() <= VOXEL_TOL * ref.max()
    pos = ref.sum(-1) > 0
    assert (np.abs(got.sum(-1) - ref.sum(-1))[pos] / ref.sum(-1)[pos]).max() <= FLUX_TOL
    empty = torch.from_numpy(counts == 0).cuda()
    assert not cube.view(t.n_spaxels, -1)[empty].any().item()
    # the brightest spaxel is one of the four central ones (their counts differ by a few per cent, so
    # which of them wins depends on the masses and ages it drew)
    assert int(cube.sum(-1).argmax().item()) in set(int(v) for v in order[-4:])


# ------------------------------------------------------------------ config 4: adjoint
def test_adjoint_config(B):
    w = synth.make_workload("adjoint")
    t = w.telescope
    other = synth.make_particles_for("adjoint", seed=synth.ADJOINT_TARGET_SEED)
    dw = B.DeviceWorkload(w)
    cube = dw.forward()
    # the target comes from the ORACLE, never from the CUDA path
    target = oracle.forward(other, w.rotation, w.ssp, t)
    ref_final = oracle.forward(w.particles, w.rotation, w.ssp, t)
    torch.cuda.synchronize()
    assert np.abs(cube.cpu().numpy() - ref_final).max() <= VOXEL_TOL * ref_final.max()
    resid = ref_final - target
    grad_cube = torch.from_numpy((2.0 * resid).astype(np.float32)).cuda()
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(grad_cube)]
    torch.cuda.synchronize()
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(grad_cube)]
    # 100 random particles against central finite differences of the oracle (BASELINE configs[4])
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ok = (key < t.n_spaxels) & (oracle.knot_clearance(vlos, ssp, t) > 1e-4)
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(synth.ADJOINT_FD_SEED).choice(np.nonzero(ok)[0], 100, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx)
    for q in range(4):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        rel = np.abs(g[q][idx] - fd[q]) / scale
        assert rel.max() <= 1e-3, (q, rel.max())
    # ALL particles against the oracle's analytic adjoint: maximum, not a percentile (readings R12 / R19)
    ana = oracle.adjoint(p, w.rotation, ssp, t, 2.0 * resid)
    stats = assert_gradients(g, ana, key, vlos, ssp, t, "configs[4]")
    print("configs[4] max relative gradient errors (excluded):", stats)
