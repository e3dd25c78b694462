"""Pins for the oracle's flux-conserving resampling (reading R13;
PAPER.md L40 "Additional resampling is performed to match the wavelength grid of the observed
telescope").  F[k] = bin average over [lambda_k - dl/2, lambda_k + dl/2] of the Doppler-shifted
piecewise-linear spectrum, zero outside the SSP coverage.  None of the expected values below comes
from the oracle's own knot walk: they are closed forms, an independent prefix-integral
formulation in numpy, and the exact telescoping of the total flux."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C_KMS = 299792.458


def grid(n_l=64, l0=4000.0, dl=2.0, n_a=3, n_z=3, fill=None, seed=0):
    rng = np.random.default_rng(seed)
    flux = rng.uniform(0.5, 2.0, (n_a, n_z, n_l)).astype(np.float32) if fill is None else fill
    return synth.SSPGrid(np.array([-1.0, 0.0, 1.0], np.float32)[:n_a], np.array([-3.0, -2.0, -1.5], np.float32)[:n_z],
                         np.float32(l0), np.float32(dl), flux)


def tel(n_c, l0, dl, resample=1):
    return synth.Telescope(1, 1, np.float32(1.0), n_c, np.float32(l0), np.float32(dl), resample=resample)


def prefix_integral_reference(S, x_lo, x_hi):
    """Independent formulation (the one SURVEY.md 8(f)-1 names): C(x) = cumulative integral of the
    piecewise-linear S (piecewise quadratic), F = C(x_hi) - C(x_lo), edges clipped to the coverage."""
    n = S.size
    cum = np.concatenate([[0.0], np.cumsum(0.5 * (S[1:] + S[:-1]))])

    def Cx(x):
        x = np.clip(x, 0.0, n - 1.0)
        j = np.minimum(np.floor(x).astype(int), n - 2)
        f = x - j
        return cum[j] + f * S[j] + 0.5 * f * f * (S[j + 1] - S[j])
    return Cx(x_hi) - Cx(x_lo)


@pytest.mark.parametrize("vlos,dl_obs", [(0.0, 1.3), (250.0, 1.25), (-800.0, 3.7), (12000.0, 0.4), (90.0, 9.1)])
def test_equals_prefix_integral_formulation(vlos, dl_obs):
    ssp = grid(n_l=300, l0=4000.0, dl=1.6, seed=3)
    t = tel(257, 3990.0, dl_obs)                         # starts below the coverage, may end above it
    q = (np.float32(1.7), np.float32(-0.35), np.float32(-2.4))
    got = oracle.particle_spectrum(q[0], q[1], q[2], np.float32(vlos), ssp, t)
    # blended samples from the POINT-sampled oracle on the SSP grid itself at v = 0 (pinned elsewhere)
    same = tel(ssp.flux.shape[2], float(ssp.lambda0), float(ssp.dlambda), resample=0)
    S = oracle.particle_spectrum(q[0], q[1], q[2], np.float32(0.0), ssp, same)
    beta = float(np.float32(vlos)) / C_KMS
    lam = t.wavelengths()
    d = float(t.dlambda)
    x_lo = ((lam - 0.5 * d) / (1 + beta) - float(ssp.lambda0)) / float(ssp.dlambda)
    x_hi = ((lam + 0.5 * d) / (1 + beta) - float(ssp.lambda0)) / float(ssp.dlambda)
    B = d / ((1 + beta) * float(ssp.dlambda))
    ref = prefix_integral_reference(S, x_lo, x_hi) / B
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()


def test_constant_template_gives_the_constant_inside_and_partial_bins_at_the_edges():
    ssp = grid(fill=np.full((3, 3, 64), 2.5, np.float32))
    t = tel(80, 3990.0, 2.0)                              # bins 3989..3991, 3991..3993, ...; coverage 4000..4126
    F = oracle.particle_spectrum(np.float32(2.0), np.float32(0.1), np.float32(-2.2), np.float32(0.0), ssp, t)
    lam = t.wavelengths()
    lo, hi = np.maximum(lam - 1.0, 4000.0), np.minimum(lam + 1.0, 4126.0)
    frac = np.clip(hi - lo, 0.0, None) / 2.0              # covered fraction of each bin
    assert np.allclose(F, 5.0 * frac, rtol=0, atol=1e-12)
    assert F[0] == 0.0 and F[-1] == 0.0 and np.isclose(F[5], 0.5 * 5.0)   # bin 3999..4001 is half covered


def test_linear_template_gives_the_value_at_the_shifted_bin_centre():
    lam_ssp = 4000.0 + 2.0 * np.arange(64)
    ssp = grid(fill=np.broadcast_to((0.25 + 1e-3 * lam_ssp).astype(np.float32), (3, 3, 64)).copy())
    t = tel(40, 4010.0, 2.7)
    for v in (0.0, 300.0, -1500.0):
        F = oracle.particle_spectrum(np.float32(3.0), np.float32(-0.4), np.float32(-1.8), np.float32(v), ssp, t)
        beta = float(np.float32(v)) / C_KMS
        T = ssp.flux[0, 0].astype(np.float64)
        slope = (T[-1] - T[0]) / (lam_ssp[-1] - lam_ssp[0])
        lam = t.wavelengths()
        expect = 3.0 * (T[0] + slope * (lam / (1 + beta) - lam_ssp[0]))
        inside = ((lam - 1.35) / (1 + beta) >= lam_ssp[0]) & ((lam + 1.35) / (1 + beta) <= lam_ssp[-1])
        assert inside.sum() >= 30
        # fp32 template values are linear only to fp32 rounding
        assert np.allclose(F[inside], expect[inside], rtol=5e-7, atol=0)


def test_same_grid_zero_velocity_is_the_1_6_1_over_8_stencil():
    ssp = grid(n_l=128, seed=5)
    t = tel(128, float(ssp.lambda0), float(ssp.dlambda))
    F = oracle.particle_spectrum(np.float32(1.0), np.float32(-1.0), np.float32(-3.0), np.float32(0.0), ssp, t)
    S = ssp.flux[0, 0].astype(np.float64)                 # node (0, 0): the blend is the template itself
    assert np.allclose(F[1:-1], (S[:-2] + 6.0 * S[1:-1] + S[2:]) / 8.0, rtol=1e-14, atol=0)
    assert np.isclose(F[0], (3.0 * S[0] + S[1]) / 8.0)    # half bin inside the coverage, averaged over the full bin


@pytest.mark.parametrize("vlos", [0.0, 420.0, -3000.0])
def test_total_flux_telescopes_exactly(vlos):
    """sum_k F[k] dl_obs = (1 + beta) * integral of the piecewise-linear spectrum over the coverage,
    when the observed grid covers the whole shifted coverage (BASELINE.json north_star: 'total flux
    is conserved')."""
    ssp = grid(n_l=200, l0=5000.0, dl=1.5, seed=11)
    t = tel(900, 4900.0, 0.77)
    m = np.float32(4.0)
    F = oracle.particle_spectrum(m, np.float32(0.3), np.float32(-1.9), np.float32(vlos), ssp, t)
    same = tel(200, 5000.0, 1.5, resample=0)
    S = oracle.particle_spectrum(m, np.float32(0.3), np.float32(-1.9), np.float32(0.0), ssp, same)
    beta = float(np.float32(vlos)) / C_KMS
    total = (1 + beta) * 1.5 * (S.sum() - 0.5 * (S[0] + S[-1]))
    assert np.isclose(F.sum() * float(t.dlambda), total, rtol=1e-12)
    assert F[0] == 0.0 and F[-1] == 0.0                   # the grid really covers everything


def test_cube_is_the_sum_of_particle_spectra_and_mode_0_is_untouched():
    w = synth.make_workload("tiny", n=60)
    t1 = dataclasses.replace(w.telescope, resample=1)
    cube = oracle.build_cube(w.particles, w.rotation, w.ssp, t1)
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t1.n_x, t1.n_y, t1.spaxel_size)
    ref = np.zeros((t1.n_spaxels, t1.n_channels))
    p = w.particles
    for i in range(p.n):
        if key[i] < t1.n_spaxels:
            ref[key[i]] += oracle.particle_spectrum(p.mass[i], p.log_age[i], p.log_z[i], vlos[i], w.ssp, t1)
    assert np.allclose(cube.reshape(ref.shape), ref, rtol=1e-13, atol=0)
    c0 = oracle.build_cube(w.particles, w.rotation, w.ssp, w.telescope)
    assert np.abs(c0 - cube).max() > 1e-4 * c0.max()      # the two rules do differ on this workload
    # a smooth spectrum sampled finely: bin average and point sample agree to second order
    assert np.abs(c0 - cube).max() < 0.2 * c0.max()


# ----------------------------------------------------------------------------- adjoint of the flux rule
def _fd_setup(n=500):
    w = synth.make_workload("tiny", n=n)
    tel_ = dataclasses.replace(w.telescope.with_psf_lsf(), resample=1)
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    cube = oracle.forward(w.particles, w.rotation, w.ssp, tel_)
    target = oracle.forward(other, w.rotation, w.ssp, tel_)
    return w, tel_, cube, target


def test_flux_adjoint_matches_central_finite_differences():
    """BASELINE.json north_star: 'adjoint gradients match central finite differences' -- for the
    flux-conserving rule.  F is C^1 in v_los here (an integral of a continuous function), so no knot
    clearance is needed; L is quadratic in mass, log age and log Z inside a cell (FD exact)."""
    w, tel_, cube, target = _fd_setup()
    resid = cube - target
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, tel_, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, _ = oracle.rotate_bin(p.pos, p.vel, w.rotation, tel_.n_x, tel_.n_y, tel_.spaxel_size)
    ok = key < tel_.n_spaxels
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(synth.ADJOINT_FD_SEED).choice(np.nonzero(ok)[0], 40, replace=False)
    fd = oracle.fd_gradients(w.particles, w.rotation, ssp, tel_, resid, idx, h_v=1e-2)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 1e-4)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), q
    # and it is not the point-sampled gradient
    g0 = oracle.adjoint(w.particles, w.rotation, w.ssp, dataclasses.replace(tel_, resample=0), 2.0 * resid)
    assert np.abs(g0[3][idx] - g[3][idx]).max() > 1e-3 * np.abs(g[3][idx]).max()


def test_flux_adjoint_closed_forms():
    """Constant template: F does not depend on v (interior bins) => d/dv = 0, d/dm = sum of G.
    Linear template a + b lambda: the bin average is the value at the bin centre, so the gradients
    equal the point-sampled closed forms  d/dv = -m b sum_k G_k lambda_k / (c (1+beta)^2)."""
    n_l = 400
    lam = 3000.0 + 2.5 * np.arange(n_l)
    t = synth.Telescope(4, 4, np.float32(1.0), 120, np.float32(3100.0), np.float32(6.0), resample=1)
    w = synth.make_workload("tiny", n=40)
    p = w.particles
    p.pos[:] = np.random.default_rng(0).uniform(-1.9, 1.9, p.pos.shape)
    p.log_age[:] = np.random.default_rng(1).uniform(-0.9, 0.9, p.n)
    p.log_z[:] = np.random.default_rng(2).uniform(-3.9, -2.1, p.n)
    R = np.eye(3, dtype=np.float32)
    G = np.random.default_rng(3).normal(size=(4, 4, 120))
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, 4, 4, 1.0)
    rows = G.reshape(16, -1)[key]
    beta = vlos.astype(np.float64) / C_KMS
    axes = (np.array([-1, 0, 1], np.float32), np.array([-4, -3, -2], np.float32))
    const = synth.SSPGrid(*axes, np.float32(3000.0), np.float32(2.5), np.full((3, 3, n_l), 1.5, np.float32))
    g_m, g_a, g_z, g_v = oracle.adjoint(p, R, const, t, G)
    assert np.allclose(g_m, 1.5 * rows.sum(1), rtol=1e-12)
    assert np.abs(g_v).max() <= 1e-12 * np.abs(g_m * p.mass).max()
    a, b = 2.0, 2.0 ** -12
    lin = synth.SSPGrid(*axes, np.float32(3000.0), np.float32(2.5),
                        np.ascontiguousarray(np.broadcast_to(a + b * lam, (3, 3, n_l)), np.float32))
    g_m, g_a, g_z, g_v = oracle.adjoint(p, R, lin, t, G)
    lam_k = t.wavelengths()
    assert np.allclose(g_v, -(p.mass * b / (C_KMS * (1 + beta) ** 2)) * (rows * lam_k).sum(1), rtol=1e-9)
    assert np.allclose(g_m, (rows * (a + b * lam_k[None, :] / (1 + beta[:, None]))).sum(1), rtol=1e-10)
