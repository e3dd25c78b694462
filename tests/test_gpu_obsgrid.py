"""Parity of the CUDA path with EXPLICIT (non-uniform) channel wavelengths (reading R16; SURVEY.md
8(f)-1 "arbitrary telescope grids") against the fp64 oracle, on linear and log-sampled SSP grids."""
import dataclasses

import numpy as np
import pytest

import oracle
from sortcheck import check_perm
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


def nonuniform(n_c, lo, hi, seed):
    rng = np.random.default_rng(seed)
    steps = rng.uniform(0.3, 1.7, n_c)
    return (lo + (hi - lo) * np.cumsum(steps) / steps.sum()).astype(np.float32)


def with_array(tel, lam):
    return dataclasses.replace(tel, n_channels=int(lam.size), lambda_obs=lam)


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


@pytest.mark.parametrize("log_grid", [False, True])
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_whole_cube(B, name, log_grid):
    w = synth.make_workload(name)
    if log_grid:
        w.ssp = synth.make_ssp(*w.ssp.flux.shape, 3000.0 if name == "small" else 3500.0,
                               10000.0 if name == "small" else 9500.0, 2200, log_lambda=True)
    t = w.telescope
    lam = nonuniform(t.n_channels, float(t.lambda0), float(t.lambda0) + float(t.dlambda) * (t.n_channels - 1), 5)
    w.telescope = with_array(t, lam)
    run_and_check(B, w, f"{name} log={log_grid}")


def test_uniform_array_matches_the_uniform_path(B):
    w = synth.make_workload("tiny")
    plain = B.DeviceWorkload(w).build_cube().cpu().numpy()
    w.telescope = with_array(w.telescope, w.telescope.wavelengths().astype(np.float32))
    arr = B.DeviceWorkload(w).build_cube().cpu().numpy()
    assert np.abs(arr - plain).max() <= 2e-3 * plain.max()       # fp32 rounding of the listed wavelengths


@pytest.mark.parametrize("n_c,lo,hi", [(5000, 4700.0, 9200.0), (257, 3000.0, 9990.0), (1025, 4700.0, 8800.0), (1, 6000.0, 6001.0)])
def test_multi_tile_coverage_edges_and_redshift(B, n_c, lo, hi):
    w = synth.make_workload("tiny", n=700)
    w.telescope = with_array(synth.Telescope(5, 7, np.float32(2.5), n_c, np.float32(0.0), np.float32(1.0)),
                             nonuniform(n_c, lo, hi, n_c))
    run_and_check(B, w, f"n_c={n_c}")
    w.telescope = dataclasses.replace(w.telescope, redshift=np.float32(0.15), flux_scale=np.float32(2.0))
    run_and_check(B, w, f"n_c={n_c} z")
    w.particles.vel[:, :] = np.random.default_rng(3).uniform(-8000, 8000, (700, 3)).astype(np.float32)
    run_and_check(B, w, f"n_c={n_c} fast")


@pytest.mark.parametrize("log_grid", [False, True])
def test_adjoint(B, log_grid):
    w = synth.make_workload("adjoint", n=20000)
    if log_grid:
        w.ssp = synth.make_ssp(50, 7, 4300, 3000.0, 10000.0, 2201, log_lambda=True)
    t = w.telescope
    w.telescope = with_array(t, nonuniform(t.n_channels, 4750.0, 9370.0, 8))
    t = w.telescope
    dw = B.DeviceWorkload(w)
    G = upstream_gradient(w)                               # 2 (cube - target) of two galaxies, as in configs[4]
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(torch.from_numpy(G).cuda())]
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, G.astype(np.float64))
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert_gradients(g, ana, key, vlos, w.ssp, t, "test_gpu_obsgrid.py")


def test_bad_arrays_are_refused(B):
    w = synth.make_workload("tiny")
    lam = w.telescope.wavelengths().astype(np.float32)
    bad = lam.copy()
    bad[10] = bad[9]
    w2 = dataclasses.replace(w, telescope=dataclasses.replace(w.telescope, lambda_obs=bad))
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(w2).build_cube()
    assert "increasing" in B.rubix_last_error()
    one = dataclasses.replace(w, telescope=dataclasses.replace(w.telescope, n_channels=1, lambda_obs=lam[:1], resample=1))
    with pytest.raises(B.RubixError):                           # a bin needs a neighbour to define its edges (R20)
        B.DeviceWorkload(one).build_cube()
    assert "n_channels >= 2" in B.rubix_last_error()
