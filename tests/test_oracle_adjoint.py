"""Pins for the oracle's step 9 (analytic adjoint).  SURVEY.md 8(c) row 9; BASELINE.json
north_star: "adjoint gradients match central finite differences"."""
import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C = synth.C_KMS


def _setup(n=600, psf=True):
    w = synth.make_workload("tiny", n=n)
    tel = w.telescope.with_psf_lsf() if psf else w.telescope
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    cube = oracle.forward(w.particles, w.rotation, w.ssp, tel)
    target = oracle.forward(other, w.rotation, w.ssp, tel)
    return w, tel, cube, target


def _fd_sample(w, tel, k, seed=synth.ADJOINT_FD_SEED):
    """In-FoV particles that are not clamped, not within 1e-3 dex of an SSP node, and whose
    channels all stay clear of a wavelength knot under the v_los step."""
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, tel.n_x, tel.n_y, tel.spaxel_size)
    ok = key < tel.n_spaxels
    ok &= oracle.knot_clearance(vlos, ssp, tel) > 1e-4          # 1e-3 km/s moves x_k by < 3e-5
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3)
        ok &= np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3
    cand = np.nonzero(ok)[0]
    return np.random.default_rng(seed).choice(cand, k, replace=False)


def test_analytic_adjoint_matches_central_finite_differences():
    w, tel, cube, target = _setup()
    resid = cube - target
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, tel, 2.0 * resid)
    idx = _fd_sample(w, tel, 40)
    fd = oracle.fd_gradients(w.particles, w.rotation, w.ssp, tel, resid, idx)
    # L is exactly quadratic in mass, and in log age / log Z inside one cell: FD is exact there
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), q


def test_fd_uses_the_loss_it_claims():
    """Cross-check fd_gradients' linearised loss against re-running the whole oracle pipeline.
    L is quadratic in each mass, so central differences are exact whatever the step."""
    w, tel, _, target = _setup(n=300)
    p = int(_fd_sample(w, tel, 1)[0])
    w.particles.mass[p] = 40000.0                                  # +-8192 stays exact in fp32
    cube = oracle.forward(w.particles, w.rotation, w.ssp, tel)
    resid = cube - target
    fd = oracle.fd_gradients(w.particles, w.rotation, w.ssp, tel, resid, [p])
    plus, minus = w.particles.copy(), w.particles.copy()
    plus.mass[p] = 48192.0
    minus.mass[p] = 31808.0
    Lp = ((oracle.forward(plus, w.rotation, w.ssp, tel) - target) ** 2).sum()
    Lm = ((oracle.forward(minus, w.rotation, w.ssp, tel) - target) ** 2).sum()
    assert Lp != (resid ** 2).sum()
    assert np.isclose((Lp - Lm) / (2.0 * 8192.0), fd[0][0], rtol=1e-7)


def test_linear_template_closed_form():
    """T = a + b*lambda everywhere: dF/dv = -m b lambda_k / (c (1+beta)^2), dF/dm = a + b lambda_k/(1+beta),
    and nothing depends on age or Z."""
    n_l, a, b = 400, 2.0, 2.0 ** -12
    lam = 3000.0 + 2.5 * np.arange(n_l)
    ssp = synth.SSPGrid(np.array([-1, 0, 1], np.float32), np.array([-4, -3, -2], np.float32),
                        np.float32(3000.0), np.float32(2.5),
                        np.ascontiguousarray(np.broadcast_to(a + b * lam, (3, 3, n_l)), np.float32))
    tel = synth.Telescope(4, 4, np.float32(1.0), 120, np.float32(3100.0), np.float32(6.0))
    w = synth.make_workload("tiny", n=50)
    p = w.particles
    p.pos[:] = np.random.default_rng(0).uniform(-1.9, 1.9, p.pos.shape)
    p.log_age[:] = np.random.default_rng(1).uniform(-0.9, 0.9, p.n)
    p.log_z[:] = np.random.default_rng(2).uniform(-3.9, -2.1, p.n)
    R = np.eye(3, dtype=np.float32)
    G = np.random.default_rng(3).normal(size=(4, 4, 120))
    g_m, g_a, g_z, g_v = oracle.adjoint(p, R, ssp, tel, G)
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, 4, 4, 1.0)
    assert (key < 16).all()
    beta = vlos.astype(np.float64) / C
    lam_k = tel.wavelengths()
    rows = G.reshape(16, -1)[key]
    assert np.allclose(g_v, -(p.mass * b / (C * (1 + beta) ** 2)) * (rows * lam_k).sum(1), rtol=1e-10)
    assert np.allclose(g_m, (rows * (a + b * lam_k[None, :] / (1 + beta[:, None]))).sum(1), rtol=1e-10)
    scale = np.abs(g_m * p.mass).max()
    assert np.abs(g_a).max() < 1e-9 * scale and np.abs(g_z).max() < 1e-9 * scale


def test_out_of_fov_and_clamped_particles():
    w, tel, cube, target = _setup(n=300, psf=False)
    p = w.particles
    p.log_age[:5] = 3.0          # beyond the oldest node: clamped, d/dlogAge = 0
    p.log_z[5:10] = -9.0
    p.pos[10:15] = 1e3           # out of the field of view
    g_m, g_a, g_z, g_v = oracle.adjoint(p, w.rotation, w.ssp, tel, 2.0 * (cube - target))
    assert not g_a[:5].any() and g_m[:5].all()
    assert not g_z[5:10].any() and g_m[5:10].all()
    for g in (g_m, g_a, g_z, g_v):
        assert not g[10:15].any()


def test_psf_lsf_enter_the_adjoint_through_the_transpose():
    """<G, P(dC)> = <P^T G, dC>: the gradient w.r.t. mass with PSF/LSF on equals the
    no-PSF gradient evaluated with the transposed-convolved upstream gradient."""
    w, tel, cube, target = _setup(n=200)
    G = 2.0 * (cube - target)
    bare = synth.make_telescope("tiny")
    Gp = oracle.convolve_transpose(G, tel.psf_size, tel.psf_sigma, tel.lsf_size, tel.lsf_sigma)
    a = oracle.adjoint(w.particles, w.rotation, w.ssp, tel, G)
    b = oracle.adjoint(w.particles, w.rotation, w.ssp, bare, Gp)
    for x, y in zip(a, b):
        assert np.allclose(x, y, rtol=1e-12, atol=0)
