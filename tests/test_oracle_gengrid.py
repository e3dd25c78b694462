"""Pins for the oracle's step 5 on general grids (readings R20, R21; PAPER.md L40
"Additional resampling is performed to match the wavelength grid of the observed telescope", L44 the log-sampled
`Mastar_CB19_SLOG_1_5` library): the bin average on log-sampled SSP grids and on listed channel wavelengths, and
listed (irregular) SSP wavelengths for both rules.  Every pin is something other than the oracle itself: numpy.interp,
a prefix-integral restatement written here, closed forms, the exact telescoping sum, reduction to the already pinned
uniform-grid functions, central finite differences."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C_KMS = 299792.458
Q = np.array([1.7, -0.35, -2.4], np.float32)     # mass, log age, log Z of the probe particle


def ssp_grid(kind, n_l=300, seed=3, fill=None):
    """kind: 'lin' 4000 + 1.6 j, 'log' 4000 * 10^(1.5e-4 j), 'irr' listed knots (jittered, variable density)."""
    rng = np.random.default_rng(seed)
    flux = rng.uniform(0.5, 2.0, (3, 3, n_l)).astype(np.float32) if fill is None else fill
    age, zed = np.array([-1.0, 0.0, 1.0], np.float32), np.array([-3.0, -2.0, -1.5], np.float32)
    if kind == "lin":
        return synth.SSPGrid(age, zed, np.float32(4000.0), np.float32(1.6), flux)
    if kind == "log":
        return synth.SSPGrid(age, zed, np.float32(4000.0), np.float32(1.5e-4), flux, 1)
    lam = 4000.0 + 1.6 * np.arange(n_l) + np.concatenate([[0.0], rng.uniform(-0.5, 0.5, n_l - 2), [0.0]])
    lam[n_l // 2:] += 0.9 * np.arange(n_l - n_l // 2)                      # coarser sampling in the red half
    return synth.SSPGrid(age, zed, np.float32(lam[0]), np.float32(1.6), flux, 0, lam.astype(np.float32))


def blended_samples(ssp):
    """S_j of the probe particle from the (separately pinned) bilinear cell weights, written out here."""
    ia, iz, ta, tz = (v[0] for v in oracle.ssp_cells(Q[1:2], Q[2:3], ssp.log_age_axis, ssp.log_z_axis))
    T = ssp.flux.astype(np.float64)
    return float(Q[0]) * ((1 - ta) * (1 - tz) * T[ia, iz] + ta * (1 - tz) * T[ia + 1, iz]
                          + (1 - ta) * tz * T[ia, iz + 1] + ta * tz * T[ia + 1, iz + 1])


def coord(ssp, lam):
    """Sampling coordinate x of rest wavelength lam, written out here independently."""
    if ssp.lambda_grid is not None:
        knots = ssp.wavelengths()
        x = np.interp(lam, knots, np.arange(knots.size, dtype=np.float64))
        lo, hi = lam < knots[0], lam > knots[-1]                            # continued linearly outside the coverage
        x = np.where(lo, (lam - knots[0]) / (knots[1] - knots[0]), x)
        return np.where(hi, knots.size - 1 + (lam - knots[-1]) / (knots[-1] - knots[-2]), x)
    if ssp.log_lambda:
        return np.log10(lam / np.float64(ssp.lambda0)) / np.float64(ssp.dlambda)
    return (lam - np.float64(ssp.lambda0)) / np.float64(ssp.dlambda)


def edges(tel):
    lam = tel.wavelengths()
    if tel.lambda_obs is None:
        d = np.float64(tel.dlambda)
        return np.concatenate([lam - 0.5 * d, [lam[-1] + 0.5 * d]])
    mid = 0.5 * (lam[1:] + lam[:-1])
    return np.concatenate([[lam[0] - 0.5 * (lam[1] - lam[0])], mid, [lam[-1] + 0.5 * (lam[-1] - lam[-2])]])


def prefix_integral(S, x_lo, x_hi):
    n = S.size
    cum = np.concatenate([[0.0], np.cumsum(0.5 * (S[1:] + S[:-1]))])

    def Cx(x):
        x = np.clip(x, 0.0, n - 1.0)
        j = np.minimum(np.floor(x).astype(int), n - 2)
        f = x - j
        return cum[j] + f * S[j] + 0.5 * f * f * (S[j + 1] - S[j])
    return Cx(x_hi) - Cx(x_lo)


def listed(n_c, l0, dl, seed):
    """Strictly increasing channel wavelengths with a +-30 % jitter and a slow stretch (fp32, as the ABI takes them)."""
    rng = np.random.default_rng(seed)
    lam = l0 + dl * (np.arange(n_c) + rng.uniform(-0.3, 0.3, n_c)) * (1.0 + 0.1 * np.arange(n_c) / n_c)
    return np.sort(lam).astype(np.float32)


def telescope(n_c, l0, dl, resample, lam=None, z=0.0):
    return synth.Telescope(1, 1, np.float32(1.0), n_c, np.float32(l0), np.float32(dl), resample=resample,
                           lambda_obs=lam, redshift=np.float32(z))


COMBOS = [("log", False), ("lin", True), ("log", True), ("irr", False), ("irr", True)]


@pytest.mark.parametrize("kind,listed_obs", COMBOS)
@pytest.mark.parametrize("v,z", [(0.0, 0.0), (310.0, 0.0), (-2500.0, 0.02), (11000.0, 0.0)])
def test_bin_average_equals_the_prefix_integral_formulation(kind, listed_obs, v, z):
    ssp = ssp_grid(kind)
    lam_obs = listed(330, 3980.0 * (1 + z), 2.3 * (1 + z), 5) if listed_obs else None
    t = telescope(330, 3980.0 * (1 + z), 2.3 * (1 + z), 1, lam_obs, z)       # starts below the coverage, ends above it
    got = oracle.particle_spectrum(Q[0], Q[1], Q[2], np.float32(v), ssp, t)
    S = blended_samples(ssp)
    c = 1.0 / ((1.0 + float(np.float32(v)) / C_KMS) * (1.0 + float(np.float32(z))))
    x = coord(ssp, edges(t) * c)
    ref = prefix_integral(S, x[:-1], x[1:]) / (x[1:] - x[:-1])
    assert (ref > 0).sum() > 100 and (ref == 0).sum() > 3
    assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max()
    # the sum of F[k] W_k telescopes to the integral of the interpolant over the covered part of the detector
    total = (got * (x[1:] - x[:-1])).sum()
    assert abs(total - prefix_integral(S, x[:1], x[-1:])[0]) <= 1e-11 * abs(total)


@pytest.mark.parametrize("kind", ["lin", "log", "irr"])
def test_point_rule_equals_numpy_interp_on_the_knots(kind):
    ssp = ssp_grid(kind)
    lam_obs = listed(300, 3985.0, 2.0, 8)
    for t in (telescope(300, 3985.0, 2.0, 0), telescope(300, 3985.0, 2.0, 0, lam_obs)):
        for v in (0.0, 777.0, -13000.0):
            got = oracle.particle_spectrum(Q[0], Q[1], Q[2], np.float32(v), ssp, t)
            rest = t.wavelengths() / (1.0 + float(np.float32(v)) / C_KMS)
            knots = ssp.wavelengths()
            S = blended_samples(ssp)
            if kind == "log":
                ref = np.interp(np.log10(rest), np.log10(knots), S, left=0.0, right=0.0)
            else:
                ref = np.interp(rest, knots, S, left=0.0, right=0.0)
            inside = (rest > knots[0] * (1 + 1e-9)) & (rest < knots[-1] * (1 - 1e-9))
            assert inside.sum() > 100
            assert np.allclose(got[inside], ref[inside], rtol=1e-9, atol=1e-9)
            assert not got[(rest < knots[0] * (1 - 1e-9)) | (rest > knots[-1] * (1 + 1e-9))].any()


def test_listed_grids_that_happen_to_be_uniform_reduce_to_the_uniform_functions():
    """The general function against the separately pinned uniform-grid ones (R6, R13): listed channel wavelengths
    l0 + k dl (exact in fp32) give midpoint edges l_k +- dl/2, listed SSP knots l0 + j dl give x = (lambda - l0)/dl."""
    ssp = ssp_grid("lin")
    uniform_knots = dataclasses.replace(ssp, lambda_grid=(4000.0 + 1.6 * np.arange(300)).astype(np.float32))
    assert np.allclose(uniform_knots.wavelengths(), ssp.wavelengths(), rtol=0, atol=3e-4)     # fp32 knots
    n_c, l0, dl = 250, 3990.0, 2.25
    lam = (l0 + dl * np.arange(n_c)).astype(np.float32)
    assert np.array_equal(lam.astype(np.float64), l0 + dl * np.arange(n_c))
    for v in (0.0, 420.0, -9000.0):
        for rule in (0, 1):
            plain = oracle.particle_spectrum(Q[0], Q[1], Q[2], np.float32(v), ssp, telescope(n_c, l0, dl, rule))
            by_list = oracle.particle_spectrum(Q[0], Q[1], Q[2], np.float32(v), ssp, telescope(n_c, l0, dl, rule, lam))
            assert np.abs(plain - by_list).max() <= 1e-11 * plain.max(), (v, rule)
            # fp32 knots differ from l0 + j dl by up to 2.4e-4 A = 1.5e-4 samples; the random template has slope ~1 per sample
            by_knots = oracle.particle_spectrum(Q[0], Q[1], Q[2], np.float32(v), uniform_knots, telescope(n_c, l0, dl, rule))
            assert np.abs(plain - by_knots).max() <= 1e-3 * plain.max(), (v, rule)


@pytest.mark.parametrize("kind", ["log", "irr"])
def test_closed_forms_constant_and_linear_in_x(kind):
    n_l = 300
    const = ssp_grid(kind, fill=np.full((3, 3, n_l), 2.5, np.float32))
    t = telescope(200, 3990.0, 2.9, 1, listed(200, 3990.0, 2.9, 1))
    F = oracle.particle_spectrum(np.float32(2.0), Q[1], Q[2], np.float32(150.0), const, t)
    x = coord(const, edges(t) / (1.0 + float(np.float32(150.0)) / C_KMS))
    covered = (np.clip(x[1:], 0, n_l - 1) - np.clip(x[:-1], 0, n_l - 1)) / (x[1:] - x[:-1])
    assert np.allclose(F, 5.0 * covered, rtol=1e-12, atol=1e-12) and (covered == 1).sum() > 100 and (covered == 0).any()
    a, b = 3.0, 0.02
    ramp = ssp_grid(kind, fill=np.ascontiguousarray(np.broadcast_to(a + b * np.arange(n_l), (3, 3, n_l)), np.float32))
    F = oracle.particle_spectrum(np.float32(1.0), Q[1], Q[2], np.float32(150.0), ramp, t)
    inside = (x[:-1] > 0) & (x[1:] < n_l - 1)
    assert np.allclose(F[inside], (a + b * 0.5 * (x[:-1] + x[1:]))[inside], rtol=1e-6)     # fp32 samples of the ramp


@pytest.mark.parametrize("kind,listed_obs,rule", [("log", False, 1), ("lin", True, 1), ("log", True, 1),
                                                   ("irr", False, 0), ("irr", True, 0), ("irr", True, 1)])
def test_adjoint_matches_central_finite_differences(kind, listed_obs, rule):
    n = 300
    w = synth.make_workload("tiny", n=n)
    w.ssp = synth.make_ssp(8, 4, 700, 3500.0, 9500.0, seed=9, log_lambda=kind == "log", irregular=kind == "irr")
    t = w.telescope.with_psf_lsf()
    lam = listed(t.n_channels, float(t.lambda0), float(t.dlambda), 4) if listed_obs else None
    t = dataclasses.replace(t, resample=rule, lambda_obs=lam)
    other = synth.make_particles_for("tiny", n=n, seed=synth.ADJOINT_TARGET_SEED)
    resid = oracle.forward(w.particles, w.rotation, w.ssp, t) - oracle.forward(other, w.rotation, w.ssp, t)
    g = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    p, ssp = w.particles, w.ssp
    key, vlos = oracle.rotate_bin(p.pos, p.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ok = key < t.n_spaxels
    if rule == 0:                                               # the point rule has kinks where a channel crosses a knot
        ok &= oracle.knot_clearance(vlos, ssp, t) > 1e-4
    for q, ax in ((p.log_age, ssp.log_age_axis), (p.log_z, ssp.log_z_axis)):
        ok &= (q > ax[0] + 1e-3) & (q < ax[-1] - 1e-3) & (np.abs(q[:, None] - ax[None, :]).min(1) > 1e-3)
    idx = np.random.default_rng(3).choice(np.nonzero(ok)[0], 25, replace=False)
    fd = oracle.fd_gradients(p, w.rotation, ssp, t, resid, idx)
    for q, rtol in ((0, 1e-7), (1, 1e-6), (2, 1e-6), (3, 2e-3 if rule else 1e-3)):
        scale = np.maximum(np.abs(fd[q]), 1e-3 * np.median(np.abs(fd[q])))
        assert (np.abs(g[q][idx] - fd[q]) <= rtol * scale).all(), (q, (np.abs(g[q][idx] - fd[q]) / scale).max())


def test_cube_is_the_sum_of_particle_spectra_in_the_new_modes():
    w = synth.make_workload("tiny", n=150)
    w.ssp = synth.make_ssp(8, 4, 512, 3500.0, 9500.0, seed=2100, irregular=True)
    t = dataclasses.replace(w.telescope, resample=1, lambda_obs=listed(w.telescope.n_channels, 4700.0, 18.0, 2))
    cube = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    ref = np.zeros((t.n_spaxels, t.n_channels))
    p = w.particles
    for i in range(p.n):
        if key[i] < t.n_spaxels:
            ref[key[i]] += oracle.particle_spectrum(p.mass[i], p.log_age[i], p.log_z[i], vlos[i], w.ssp, t)
    assert np.abs(cube.reshape(ref.shape) - ref).max() <= 1e-12 * ref.max()
