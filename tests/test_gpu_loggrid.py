"""Parity of the CUDA path on LOG-SAMPLED SSP grids (reading R15) against the
fp64 oracle, through the C ABI: forward (whole cubes, multi-tile, coverage edges, redshift) and adjoint."""
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


def _knot_sweep_workload(ssp, tel, k_star, j_star, half=220):
    """One particle per spaxel, identity rotation, v_los = v_z swept in steps of ~1e-7 SSP samples (or one fp32 ulp of
    v_los, if that is coarser) around the velocity that puts channel k_star's rest position exactly on SSP knot j_star
    (log-sampled grid: x_k = log10(lambda_k / lambda0) / d - log10(1 + beta) / d)."""
    lam_k = float(tel.wavelengths()[k_star])
    d, l0 = float(ssp.dlambda), float(ssp.lambda0)
    beta = lam_k / (l0 * 10.0 ** (j_star * d)) - 1.0
    v0 = np.float32(beta * synth.C_KMS)
    dv = max(1e-7 * d * np.log(10.0) * synth.C_KMS, float(np.spacing(np.abs(v0))))      # 1e-7 samples per step
    v = (np.float64(v0) + dv * np.arange(-half, half + 1)).astype(np.float32)
    n = v.size
    assert n <= tel.n_x * tel.n_y
    ix, iy = np.divmod(np.arange(n), tel.n_y)
    pos = np.zeros((n, 3), np.float32)
    pos[:, 0] = (ix + 0.5 - 0.5 * tel.n_x) * float(tel.spaxel_size)
    pos[:, 1] = (iy + 0.5 - 0.5 * tel.n_y) * float(tel.spaxel_size)
    vel = np.zeros((n, 3), np.float32)
    vel[:, 2] = v
    rng = np.random.default_rng(77)
    p = synth.Particles(pos, vel, rng.uniform(0.5e5, 2e5, n).astype(np.float32),
                        rng.uniform(ssp.log_age_axis[0], ssp.log_age_axis[-1], n).astype(np.float32),
                        rng.uniform(ssp.log_z_axis[0], ssp.log_z_axis[-1], n).astype(np.float32))
    return synth.Workload("knot-sweep", p, ssp, tel, np.eye(3, dtype=np.float32), (0.0, 0.0, 0.0))


@pytest.mark.parametrize("case", ["first covered channel on knot 0 (detector starts blueward of the grid)",
                                  "channel 0 on a knot that is a multiple of 32",
                                  "first channel of a later tile on a multiple of 32"])
def test_channel_within_a_fixed_point_unit_of_the_window_start(B, case):
    """ADVICE r01 (spectral.cu, table mode): the resampler adds separately truncated 2^-20 terms and may sit 1-2 units
    BELOW the exact x_k; with x_k within ~2e-6 samples above the first sample of the staged window that wrapped below
    zero and read a table entry outside the window.  Deterministic sweep: 441 particles whose x_k differ by ~1e-7
    samples, centred on the velocity that puts the critical channel exactly on the knot."""
    ssp = log_ssp("tiny")
    d = float(ssp.dlambda)
    if case.startswith("first covered"):
        tel = synth.Telescope(21, 21, np.float32(1.0), 700, np.float32(3000.0), np.float32(10.0))
        k_star = int(np.searchsorted(tel.wavelengths(), 3500.0 * 1.0005))     # first channel redward of knot 0
        w = _knot_sweep_workload(ssp, tel, k_star, 0)
    elif case.startswith("channel 0"):
        lam0 = np.float32(3500.0 * 10.0 ** (160.02 * d))
        tel = synth.Telescope(21, 21, np.float32(1.0), 256, lam0, np.float32(18.0))
        w = _knot_sweep_workload(ssp, tel, 0, 160)
    else:
        k_star = 1024                                                          # tiles of 8 x 128 channels
        lam0 = np.float32(3500.0 * 10.0 ** (224.02 * d) - 0.9 * k_star)        # puts x_1024 just above knot 224 = 7 x 32
        tel = synth.Telescope(21, 21, np.float32(1.0), 5000, lam0, np.float32(0.9))
        w = _knot_sweep_workload(ssp, tel, k_star, 224)
    assert np.abs(w.particles.vel[:, 2]).max() < 0.05 * synth.C_KMS
    got, ref = run_and_check(B, w, case)
    # every particle is alone in its spaxel: the bound holds per particle spectrum, not only against the cube maximum
    n = w.particles.n
    g2 = got.reshape(-1, got.shape[-1])[:n]
    r2 = ref.reshape(-1, ref.shape[-1])[:n]
    assert (np.abs(g2 - r2).max(1) <= 1e-4 * r2.max(1)).all(), case


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


def test_flux_conserving_rule_on_a_log_grid(B):
    """Refused in r01; reading R20 defines it (tests/test_gpu_gengrid.py holds the full set)."""
    w = synth.make_workload("tiny")
    w.ssp = log_ssp("tiny")
    w.telescope = dataclasses.replace(w.telescope, resample=1)
    run_and_check(B, w, "bin average on a log-sampled grid")
