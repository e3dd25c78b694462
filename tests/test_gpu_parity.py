"""Parity of the CUDA path (through the C ABI) against the fp64 oracle.  `-m gpu` only.

Tolerances are BASELINE.json:north_star's: spaxel assignment and sort order bit-exact; cube voxels
max|GPU - oracle| <= 1e-4 * max|oracle cube|; each spaxel's summed flux within 1e-5 relative;
empty spaxels exactly 0 before the PSF."""
import numpy as np
import pytest

import oracle
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
    assert np.array_equal(perm, operm), "sort order differs"
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
    w = medium
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    torch.cuda.synchronize()
    okey, oseg = check_sort(dw, w)
    counts = np.diff(oseg)[:-1]
    # every empty spaxel is exactly zero
    empty = torch.from_numpy(counts == 0).cuda()
    assert not cube.view(t.n_spaxels, -1)[empty].any().item()
    # sampled spaxels the oracle computes one by one: the heaviest, a ring of busy ones, random ones
    rng = np.random.default_rng(14)
    order = np.argsort(counts)
    sel = np.unique(np.concatenate([order[-12:], order[-3000:-12:250], rng.choice(np.nonzero(counts > 0)[0], 60),
                                    rng.choice(np.nonzero(counts == 0)[0], 4)])).astype(np.int32)
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t, sel=sel)
    got = cube.view(t.n_spaxels, -1)[torch.from_numpy(sel.astype(np.int64)).cuda()].cpu().numpy()
    # the global max of the cube is in the heaviest spaxels, which are part of the sample
    assert counts[sel].max() == counts.max()
    check_cube(got, ref, "medium sampled spaxels")
    # total flux per spaxel over the WHOLE cube against a property: positive where occupied
    sums = cube.double().sum(-1).view(-1).cpu().numpy()
    assert (sums[counts > 0] > 0).all()

    # final cube (PSF + LSF) on a patch around the brightest spaxel
    final = dw.convolve(cube)
    torch.cuda.synchronize()
    bx, by = divmod(int(order[-1]), t.n_y)
    bx, by = int(np.clip(bx, 12, t.n_x - 13)), int(np.clip(by, 12, t.n_y - 13))
    xs, ys = np.arange(bx - 10, bx + 11), np.arange(by - 10, by + 11)
    patch_sel = (xs[:, None] * t.n_y + ys[None, :]).reshape(-1).astype(np.int32)
    patch = oracle.build_cube(w.particles, w.rotation, w.ssp, t, sel=patch_sel).reshape(21, 21, -1)
    conv = oracle.convolve(patch, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma)[7:14, 7:14]
    gotp = final[bx - 3:bx + 4, by - 3:by + 4].cpu().numpy().astype(np.float64)
    assert np.abs(gotp - conv).max() <= VOXEL_TOL * conv.max()
    assert np.allclose(gotp.sum(-1), conv.sum(-1), rtol=FLUX_TOL)


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
    # all particles against the oracle's analytic adjoint
    ana = oracle.adjoint(p, w.rotation, ssp, t, 2.0 * resid)
    for q in range(4):
        scale = np.maximum(np.abs(ana[q]), 1e-3 * np.median(np.abs(ana[q][key < t.n_spaxels])))
        rel = np.abs(g[q] - ana[q]) / scale
        assert np.quantile(rel, 0.999) <= 1e-3, (q, rel.max())
        assert not g[q][key >= t.n_spaxels].any()
