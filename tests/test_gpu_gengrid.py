"""Parity of the CUDA path in the general-grid mode (readings R20, R21) against the fp64
oracle, through the C ABI: the bin average on log-sampled SSP grids and on listed channel wavelengths, listed (irregular)
SSP wavelengths under both rules -- forward (whole cubes, several channel tiles, coverage edges, redshift, fast
particles), PSF/LSF through rubix_forward, and the adjoint for every particle."""
import dataclasses

import numpy as np
import pytest

import oracle
from sortcheck import check_perm
from gradcheck import assert_gradients, upstream_gradient
from paper_2412_08265_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

COMBOS = [("log", False, 1), ("lin", True, 1), ("log", True, 1), ("irr", False, 0), ("irr", True, 0), ("irr", False, 1),
          ("irr", True, 1)]


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no CPU fallback")
    from paper_2412_08265_b200 import binding
    binding.load()
    return binding


def ssp_for(name, kind):
    if name == "tiny":
        return synth.make_ssp(8, 4, 512, 3500.0, 9500.0, 2100, log_lambda=kind == "log", irregular=kind == "irr")
    return synth.make_ssp(50, 7, 4300, 3000.0, 10000.0, 2101, log_lambda=kind == "log", irregular=kind == "irr")


def listed(tel, seed):
    """The telescope's channels moved by up to +-30 % of the spacing, with a slow stretch; fp32, strictly increasing."""
    rng = np.random.default_rng(seed)
    n_c = tel.n_channels
    k = np.arange(n_c) + rng.uniform(-0.3, 0.3, n_c)
    lam = float(tel.lambda0) + float(tel.dlambda) * k * (1.0 + 0.03 * np.arange(n_c) / max(n_c, 1))
    return np.sort(lam).astype(np.float32)


def configure(w, name, kind, listed_obs, rule, seed=1):
    w.ssp = ssp_for(name, kind)
    t = dataclasses.replace(w.telescope, resample=rule)
    if listed_obs:
        t = dataclasses.replace(t, lambda_obs=listed(t, seed))
    w.telescope = t
    return w


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


@pytest.mark.parametrize("kind,listed_obs,rule", COMBOS)
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_whole_cube(B, name, kind, listed_obs, rule):
    n = None if name == "tiny" else 20000
    w = configure(synth.make_workload(name, n=n), name, kind, listed_obs, rule)
    run_and_check(B, w, (name, kind, listed_obs, rule))


@pytest.mark.parametrize("kind,listed_obs,rule", COMBOS)
@pytest.mark.parametrize("n_c,dl", [(5000, 0.9), (257, 18.0), (3841, 1.2), (2, 90.0)])
def test_several_channel_tiles_and_ragged_counts(B, kind, listed_obs, rule, n_c, dl):
    w = synth.make_workload("tiny", n=500)
    w.telescope = synth.Telescope(5, 7, np.float32(2.5), n_c, np.float32(4700.0), np.float32(dl))
    run_and_check(B, configure(w, "tiny", kind, listed_obs, rule, seed=n_c), (kind, listed_obs, rule, n_c))


@pytest.mark.parametrize("kind,listed_obs,rule", COMBOS)
def test_coverage_edges_redshift_and_fast_particles(B, kind, listed_obs, rule):
    w = synth.make_workload("tiny", n=600)
    w.telescope = synth.Telescope(6, 6, np.float32(3.0), 700, np.float32(3000.0), np.float32(10.0))   # 3000..9990
    configure(w, "tiny", kind, listed_obs, rule)
    got, _ = run_and_check(B, w, "coverage")
    assert not got[..., :40].any() and not got[..., -30:].any() and got[..., 300].any()
    w.telescope = dataclasses.replace(w.telescope, redshift=np.float32(0.2), flux_scale=np.float32(0.5))
    run_and_check(B, w, "redshift")
    w.particles.vel[:, :] = np.random.default_rng(3).uniform(-8000, 8000, (600, 3)).astype(np.float32)
    run_and_check(B, w, "fast particles")


@pytest.mark.parametrize("kind,listed_obs,rule", COMBOS)
def test_forward_with_psf_lsf_and_adjoint(B, kind, listed_obs, rule):
    w = synth.make_workload("adjoint", n=12000)
    configure(w, "small", kind, listed_obs, rule)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    final = dw.forward().cpu().numpy().astype(np.float64)
    ref = oracle.forward(w.particles, w.rotation, w.ssp, t)
    assert np.abs(final - ref).max() <= 1e-4 * np.abs(ref).max()
    G = upstream_gradient(w)                               # 2 (cube - target) of two galaxies, as in configs[4]
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(torch.from_numpy(G).cuda())]
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, G.astype(np.float64))
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert_gradients(g, ana, key, vlos, w.ssp, t, ("test_gpu_gengrid.py", kind, listed_obs, rule))
    # the fused call: same gradients from one particle pass
    target = torch.from_numpy((ref - G.astype(np.float64) / 2.0).astype(np.float32)).cuda()
    loss, g2, _ = dw.loss_and_grad(target)
    for a, b in zip(g2, ana):
        scale = np.maximum(np.abs(b), 1e-3 * np.median(np.abs(b[key < t.n_spaxels])))
        rel = (np.abs(a.cpu().numpy() - b) / np.where(scale > 0, scale, 1.0))
        assert np.quantile(rel, 0.99) <= 3e-3               # upstream gradient from the GPU's own fp32 cube (R19)


def test_bad_listed_ssp_grids(B):
    w = synth.make_workload("tiny", n=50)
    good = ssp_for("tiny", "irr")
    bad = dataclasses.replace(good, lambda_grid=good.lambda_grid[::-1].copy())
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(dataclasses.replace(w, ssp=bad)).build_cube()
    assert "increasing" in B.rubix_last_error()
    both = dataclasses.replace(good, log_lambda=1)
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(dataclasses.replace(w, ssp=both)).build_cube()
    coarse = dataclasses.replace(w.telescope, dlambda=np.float32(400.0))      # one channel spans > 14 SSP samples
    with pytest.raises(B.RubixError):
        B.DeviceWorkload(dataclasses.replace(w, ssp=good, telescope=coarse)).build_cube()
