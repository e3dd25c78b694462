"""Edge cases of the CUDA path against the oracle: empty input, everything out of the field of
view, one spaxel holding every particle (multi-chunk partial rows), multi-tile spectra, SSP grids
whose row length is not a multiple of 4 (scalar blend path), observed grids sticking out of the
SSP coverage (predicated resampling), non-square detectors, the host-buffer entry point."""
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


def run_and_check(B, w, what):
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube(out=torch.full((t.n_x, t.n_y, t.n_channels), float("nan"), device="cuda"))
    torch.cuda.synchronize()
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey) and np.array_equal(seg, oseg), what
    check_perm(perm, operm, oseg, w.particles, w.ssp, t.n_spaxels, None)
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    got = cube.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all(), what
    assert np.abs(got - ref).max() <= 1e-4 * max(np.abs(ref).max(), 1e-30), what
    fr = ref.sum(-1)
    pos = fr > 0
    if pos.any():
        assert (np.abs(got.sum(-1) - fr)[pos] / fr[pos]).max() <= 1e-5, what
    assert not got[~pos].any(), what
    return dw, got, ref


def test_no_particles(B):
    w = synth.make_workload("tiny", n=1000)
    w.particles = w.particles.subset(slice(0, 0))
    dw, got, _ = run_and_check(B, w, "n = 0")
    assert not got.any()


def test_all_particles_out_of_fov_or_too_fast(B):
    w = synth.make_workload("tiny", n=500)
    w.particles.pos[:250] += 1e3
    w.particles.vel[250:, 2] = 2.0e4
    w.particles.pos[7] = np.nan
    w.rotation = np.eye(3, dtype=np.float32)
    _, got, _ = run_and_check(B, w, "all dropped")
    assert not got.any()


def test_single_particle_and_node_reproduction(B):
    w = synth.make_workload("tiny", n=1)
    ssp = w.ssp
    w.telescope = synth.Telescope(3, 2, np.float32(1.0), 512, ssp.lambda0, ssp.dlambda)   # obs grid = SSP grid
    w.rotation = np.eye(3, dtype=np.float32)
    w.particles.pos[0] = [0.2, 0.3, 0.0]
    w.particles.vel[0] = [10.0, -20.0, 0.0]                      # v_los = 0
    w.particles.log_age[0], w.particles.log_z[0] = ssp.log_age_axis[5], ssp.log_z_axis[2]
    _, got, ref = run_and_check(B, w, "node")
    row = got[1, 1]
    assert np.allclose(row, float(w.particles.mass[0]) * ssp.flux[5, 2].astype(np.float64), rtol=3e-7)


def test_one_spaxel_holds_everything_multi_chunk(B):
    w = synth.make_workload("tiny", n=1000)
    w.particles.pos[:] = np.random.default_rng(0).uniform(0.05, 0.95, (1000, 3)).astype(np.float32)
    w.rotation = np.eye(3, dtype=np.float32)
    dw, got, ref = run_and_check(B, w, "one spaxel")
    assert (np.diff(dw.sort_artifacts()[2].cpu().numpy()) == 1000).sum() == 1


@pytest.mark.parametrize("n_c,dl", [(5000, 0.9), (257, 18.0), (1025, 4.0), (3841, 1.2)])
def test_multi_tile_and_ragged_channel_counts(B, n_c, dl):
    w = synth.make_workload("tiny", n=700)
    w.telescope = synth.Telescope(5, 7, np.float32(2.5), n_c, np.float32(4700.0), np.float32(dl))
    run_and_check(B, w, f"n_c={n_c}")


@pytest.mark.parametrize("n_x,n_y", [(33, 31), (32, 32), (41, 25), (64, 33)])
@pytest.mark.parametrize("n", [3000, 16384, 16385, 40000])
def test_unit_scan_around_the_tile_and_size_limits(B, n_x, n_y, n):
    """1023 / 1024 / 1025 / 2112 spaxels (one scan tile holds 1024) and particle counts either side of the limit up to which
    k_scan_units finds the segment offsets itself; a pile-up gives multi-chunk spaxels of more than 32 chunks (the warp path of
    the unit descriptors) next to ones of two or three."""
    w = synth.make_workload("tiny", n=n, seed=77)
    w.particles.pos[: n // 3, :2] *= np.float32(0.02)            # > 32 chunks of 128 in the central spaxels from n = 16384 on
    w.particles.pos[n // 3: n // 2, :2] *= np.float32(0.2)
    w.telescope = dataclasses.replace(w.telescope, n_x=n_x, n_y=n_y, spaxel_size=np.float32(0.5), n_channels=64)
    run_and_check(B, w, f"{n_x}x{n_y} n={n}")


def test_row_length_not_multiple_of_four_uses_scalar_blend(B):
    w = synth.make_workload("tiny", n=600)
    w.ssp = synth.make_ssp(6, 3, 511, 3500.0, 9500.0, seed=77)
    run_and_check(B, w, "n_lambda = 511")


def test_observed_grid_outside_ssp_coverage(B):
    w = synth.make_workload("tiny", n=600)
    w.telescope = synth.Telescope(6, 6, np.float32(3.0), 700, np.float32(3000.0), np.float32(10.0))  # 3000..9990
    _, got, ref = run_and_check(B, w, "coverage")
    assert not got[..., :40].any() and not got[..., -40:].any() and got[..., 300].any()
    w.telescope = synth.Telescope(6, 6, np.float32(3.0), 100, np.float32(9600.0), np.float32(10.0))  # all outside
    _, got, _ = run_and_check(B, w, "no coverage")
    assert not got.any()


def test_large_velocities_within_the_cap(B):
    w = synth.make_workload("tiny", n=400)
    w.particles.vel[:, :] = np.random.default_rng(3).uniform(-8000, 8000, (400, 3)).astype(np.float32)
    run_and_check(B, w, "fast particles")


def test_clamped_ages_and_metallicities(B):
    w = synth.make_workload("tiny", n=400)
    w.particles.log_age[:100] = 2.0
    w.particles.log_age[100:200] = -3.0
    w.particles.log_z[150:300] = -7.0
    w.particles.log_z[300:] = 0.5
    run_and_check(B, w, "clamped")


def test_forward_host_matches_device_path(B):
    w = synth.make_workload("small", n=20_000)
    w.telescope = w.telescope.with_psf_lsf()
    t = w.telescope
    dw = B.DeviceWorkload(w)
    ref = dw.forward()
    p = w.particles
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hp = [pin(x) for x in (p.pos, p.vel, p.mass, p.log_age, p.log_z)]
    hflux = pin(w.ssp.flux)
    hcube = torch.empty((t.n_x, t.n_y, t.n_channels), dtype=torch.float32).pin_memory()
    cp = B.c_particles(*hp)
    cs = B.c_ssp(w.ssp, hflux)
    ct = B.c_telescope(t)
    scratch = torch.empty(B.rubix_forward_host_scratch_bytes(p.n, cs, ct), dtype=torch.uint8, device="cuda")
    B.rubix_forward_host(cp, cs, ct, w.rotation, hcube, scratch)
    assert B.rubix_last_launch_count() > 5
    torch.cuda.synchronize()
    assert torch.equal(hcube, ref.cpu())


def test_gpu_error_paths(B):
    w = synth.make_workload("tiny")
    dw = B.DeviceWorkload(w)
    small_ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    cube = torch.empty(dw.shape, device="cuda")
    with pytest.raises(B.RubixError) as e:
        B.rubix_build_cube(dw.particles, dw.ssp, dw.tel, dw.R, cube, small_ws)
    assert e.value.status == B.RUBIX_ERR_WORKSPACE
    with pytest.raises(B.RubixError):
        B.rubix_convolve_psf_lsf(B.c_telescope(w.telescope.with_psf_lsf()), cube, cube, dw.workspace)


@pytest.mark.parametrize("var_psf", [False, True])
def test_calls_can_be_captured_in_a_cuda_graph(B, var_psf):
    """The library enqueues on the caller's stream, never synchronises and never allocates, so a
    build + PSF/LSF step is capturable and replays bit-identically (launch-bound small cubes gain).  Also with a
    wavelength-dependent PSF on a uniform channel grid (its per-channel taps come from a kernel)."""
    w = synth.make_workload("tiny")
    w.telescope = w.telescope.with_psf_lsf()
    if var_psf:
        w.telescope = dataclasses.replace(w.telescope, psf_alpha=np.float32(-0.2), psf_lambda_ref=np.float32(6000.0))
    dw = B.DeviceWorkload(w)
    cube = torch.empty(dw.shape, device="cuda")
    final = torch.empty_like(cube)

    def step():
        B.rubix_build_cube(dw.particles, dw.ssp, dw.tel, dw.R, cube, dw.workspace)
        B.rubix_convolve_psf_lsf(dw.tel, cube, final, dw.workspace)

    step()
    torch.cuda.synchronize()
    ref = final.clone()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        step()                                    # warm-up on the capture stream
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        step()
    for _ in range(3):
        final.zero_()
        cube.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(final, ref)


def test_pipelined_forward_host_matches_the_plain_call(B):
    """Back-to-back cubes with the device->host copies on the internal copy stream: every cube equals the plain
    end-to-end call's, also when host buffers alternate and when PSF/LSF is off (the raw buffer alternates)."""
    for conv in (True, False):
        w = synth.make_workload("tiny")
        if conv:
            w.telescope = w.telescope.with_psf_lsf()
        p = w.particles
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hflux = pin(w.ssp.flux)
        cs, ct = B.c_ssp(w.ssp, hflux), B.c_telescope(w.telescope)
        shape = (w.telescope.n_x, w.telescope.n_y, w.telescope.n_channels)
        scratch = torch.empty(B.rubix_forward_host_pipelined_scratch_bytes(p.n, cs, ct), dtype=torch.uint8, device="cuda")
        outs, refs = [], []
        for i in range(5):                                   # five galaxies differing by their masses
            hp = [pin(x) for x in (p.pos, p.vel, p.mass * np.float32(1.0 + i), p.log_age, p.log_z)]
            cp = B.c_particles(*hp)
            ref = torch.empty(shape).pin_memory()
            B.rubix_forward_host(cp, cs, ct, w.rotation, ref, scratch)
            torch.cuda.synchronize()
            refs.append(ref.clone())
            outs.append((torch.empty(shape).pin_memory(), cp, hp))
        for out, cp, _ in outs:
            B.rubix_forward_host_pipelined(cp, cs, ct, w.rotation, out, scratch)
        B.rubix_forward_host_drain()
        torch.cuda.current_stream().synchronize()            # the caller's stream alone: drain made it wait for the copies
        for (out, _, _), ref in zip(outs, refs):
            assert torch.equal(out, ref)
