"""Parity of the CUDA path on LOG-SAMPLED SSP grids (reading R15) against the
fp64 oracle, through the C ABI: forward (whole cubes, multi-tile, coverage edges, redshift) and adjoint."""
import dataclasses

import numpy as np
import pytest

import oracle
from gradcheck import assert_gradients, upstream_gradient
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


def log_ssp(name):
    if name == "tiny":
        return synth.make_ssp(8, 4, 512, 3500.0, 9500.0, 2100, log_lambda=True)
    return synth.make_ssp(50, 7, 4300, 3000.0, 10000.0, 2101, log_lambda=True)


def run_and_check(B, w, what):
    t = w.telescope
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube(out=torch.full((t.n_x, t.n_y, t.n_channels), float("nan"), device="cuda"))
    torch.cuda.synchronize()
    key, perm, seg = (a.cpu().numpy() for a in dw.sort_artifacts())
    okey, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(okey, t.n_spaxels)
    assert np.array_equal(key, okey) and np.array_equal(perm, operm) and np.array_equal(seg, oseg), what
    got = cube.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all(), what
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    scale = max(np.abs(ref).max(), 1e-30)
    assert np.abs(got - ref).max() <= 1e-4 * scale, (what, np.abs(got - ref).max() / scale)
    fr = ref.sum(-1)
    pos = fr > 0
    if pos.any():
        assert (np.abs(got.sum(-1) - fr)[pos] / fr[pos]).max() <= 1e-5, what
    assert not got[~pos].any(), what
    return got, ref


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_whole_cube(B, name):
    w = synth.make_workload(name)
    lin = oracle.build_cube(w.particles, w.rotation, w.ssp, w.telescope)
    w.ssp = log_ssp(name)
    got, ref = run_and_check(B, w, name)
    assert np.abs(ref - lin).max() > 1e-2 * ref.max()            # a different grid really is in use


@pytest.mark.parametrize("n_c,dl", [(5000, 0.9), (257, 18.0), (1025, 4.0), (3841, 1.2)])
def test_multi_tile_and_ragged_channel_counts(B, n_c, dl):
    w = synth.make_workload("tiny", n=700)
    w.ssp = log_ssp("tiny")
    w.telescope = synth.Telescope(5, 7, np.float32(2.5), n_c, np.float32(4700.0), np.float32(dl))
    run_and_check(B, w, f"n_c={n_c}")


def test_coverage_edges_redshift_and_fast_particles(B):
    w = synth.make_workload("tiny", n=600)
    w.ssp = log_ssp("tiny")
    w.telescope = synth.Telescope(6, 6, np.float32(3.0), 700, np.float32(3000.0), np.float32(10.0))   # 3000..9990
    got, _ = run_and_check(B, w, "coverage")
    assert not got[..., :40].any() and not got[..., -40:].any() and got[..., 300].any()
    w.telescope = dataclasses.replace(w.telescope, redshift=np.float32(0.2), flux_scale=np.float32(0.5))
    run_and_check(B, w, "redshift")
    w.particles.vel[:, :] = np.random.default_rng(3).uniform(-8000, 8000, (600, 3)).astype(np.float32)
    run_and_check(B, w, "fast particles")


def test_adjoint(B):
    w = synth.make_workload("adjoint", n=20000)
    w.ssp = log_ssp("small")
    t = w.telescope
    dw = B.DeviceWorkload(w)
    G = upstream_gradient(w)                               # 2 (cube - target) of two galaxies, as in configs[4]
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(torch.from_numpy(G).cuda())]
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, G.astype(np.float64))
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert_gradients(g, ana, key, vlos, w.ssp, t, "test_gpu_loggrid.py")


def test_flux_conserving_rule_is_refused_on_a_log_grid(B):
    w = synth.make_workload("tiny")
    w.ssp = log_ssp("tiny")
    w.telescope = dataclasses.replace(w.telescope, resample=1)
    dw = B.DeviceWorkload(w)
    with pytest.raises(B.RubixError):
        dw.build_cube()
    assert "RUBIX_RESAMPLE_POINT" in B.rubix_last_error()
