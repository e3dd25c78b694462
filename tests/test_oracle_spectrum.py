"""Pins for the oracle's steps 4-6 (SSP lookup, Doppler + resample, accumulate).
SURVEY.md 8(c) rows 4-6; the five mandatory pins of BASELINE.json:north_star that live here:
node reproduction, line shift to lambda(1+v/c), flux conservation through binning."""
import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth

C = synth.C_KMS


def _ssp(flux, age_axis, z_axis, lam0, dlam):
    return synth.SSPGrid(np.asarray(age_axis, np.float32), np.asarray(z_axis, np.float32),
                         np.float32(lam0), np.float32(dlam), np.ascontiguousarray(flux, np.float32))


def _tel(n_c, lam0, dlam, n_x=1, n_y=1, s=1.0):
    return synth.Telescope(n_x, n_y, np.float32(s), n_c, np.float32(lam0), np.float32(dlam))


# ---------------------------------------------------------------- lookup (8c-4)
def test_particle_on_a_grid_node_at_rest_reproduces_its_template_exactly(tiny):
    ssp = tiny.ssp
    tel = _tel(ssp.flux.shape[2], ssp.lambda0, ssp.dlambda)       # observed grid = SSP grid
    for i, j in [(0, 0), (3, 1), (7, 3), (2, 3), (7, 0)]:          # n_age=8 != n_z=4: no transposition
        m = np.float32(123456.0)
        F = oracle.particle_spectrum(m, ssp.log_age_axis[i], ssp.log_z_axis[j], 0.0, ssp, tel)
        assert np.array_equal(F, np.float64(m) * ssp.flux[i, j].astype(np.float64))


def test_cells_weights_partition_of_unity_and_clamping(tiny):
    ssp = tiny.ssp
    rng = np.random.default_rng(5)
    la = rng.uniform(-2.0, 2.0, 2000).astype(np.float32)         # reaches outside the grid both sides
    lz = rng.uniform(-5.0, -1.0, 2000).astype(np.float32)
    ia, iz, ta, tz = oracle.ssp_cells(la, lz, ssp.log_age_axis, ssp.log_z_axis)
    assert ia.min() == 0 and ia.max() == ssp.log_age_axis.size - 2
    assert iz.min() == 0 and iz.max() == ssp.log_z_axis.size - 2
    assert ((ta >= 0) & (ta <= 1) & (tz >= 0) & (tz <= 1)).all()
    A = ssp.log_age_axis.astype(np.float64)
    inside = (la >= A[0]) & (la < A[-1])
    assert np.array_equal(ia[inside], np.searchsorted(A, la[inside].astype(np.float64), "right") - 1)
    assert np.allclose(A[ia[inside]] + ta[inside] * (A[ia[inside] + 1] - A[ia[inside]]),
                       la[inside], atol=1e-12)
    assert (ta[la < A[0]] == 0).all() and (ta[la >= A[-1]] == 1).all()
    # a node value belongs to the cell that starts there, with t = 0 (last node: t = 1)
    i2, _, t2, _ = oracle.ssp_cells(ssp.log_age_axis, np.full(8, -3, np.float32),
                                    ssp.log_age_axis, ssp.log_z_axis)
    assert i2.tolist() == [0, 1, 2, 3, 4, 5, 6, 6] and t2.tolist() == [0] * 7 + [1.0]


def test_bilinear_family_is_reproduced_exactly_on_nonuniform_axes():
    """T = f0 + a f1 + z f2 + a z f3 is bilinear in the axis values (a, z), so the lookup must
    return it exactly anywhere inside the grid.  Template values are dyadic (exact in fp32); only
    the interpolation parameter can round, hence 1e-14."""
    age_axis = np.array([-1.0, -0.5, 0.25, 0.375, 1.0])            # non-uniform
    z_axis = np.array([-4.0, -3.25, -2.0, -1.5])
    n_l = 16
    f = [np.arange(n_l) % 5 + 1.0, np.arange(n_l) % 3 + 0.5, (np.arange(n_l) % 4) * 0.25,
         np.arange(n_l) % 2 + 0.125]
    a, z = age_axis[:, None, None], z_axis[None, :, None]
    ssp = _ssp(f[0] + a * f[1] + z * f[2] + a * z * f[3] + 64.0, age_axis, z_axis, 4000.0, 2.0)
    tel = _tel(n_l, 4000.0, 2.0)
    for la, lz in [(-0.75, -3.5), (0.3125, -1.75), (0.0, -2.0), (0.9375, -3.9375), (0.25, -2.5)]:
        F = oracle.particle_spectrum(8.0, la, lz, 0.0, ssp, tel)
        assert np.allclose(F, 8.0 * (f[0] + la * f[1] + lz * f[2] + la * lz * f[3] + 64.0),
                           rtol=1e-14, atol=0)
    # midpoint of a cell = mean of its four corners
    F = oracle.particle_spectrum(1.0, -0.75, -3.625, 0.0, ssp, tel)
    assert np.allclose(F, ssp.flux[0:2, 0:2].astype(np.float64).mean((0, 1)), rtol=0, atol=1e-12)
    # outside the grid: clamped to the edge, no extrapolation
    F = oracle.particle_spectrum(1.0, 5.0, -9.0, 0.0, ssp, tel)
    assert np.array_equal(F, ssp.flux[-1, 0].astype(np.float64))


# ---------------------------------------------------------------- Doppler + resample (8c-5)
@pytest.mark.parametrize("v", [0.0, 137.5, -412.0, 3000.0])
def test_equals_numpy_interp(tiny, v):
    ssp, tel = tiny.ssp, tiny.telescope
    i, j = 4, 2
    F = oracle.particle_spectrum(1.0, ssp.log_age_axis[i], ssp.log_z_axis[j], v, ssp, tel)
    vf = float(np.float32(v))
    ref = np.interp(tel.wavelengths() / (1.0 + vf / C), ssp.wavelengths(),
                    ssp.flux[i, j].astype(np.float64), left=0.0, right=0.0)
    assert np.allclose(F, ref, rtol=1e-12, atol=0)


def test_linear_template_closed_form():
    """T = a + b*lambda is reproduced exactly by linear interpolation: F[k] = m (a + b lambda_k/(1+beta)).
    a, b and the wavelength grids are dyadic, so the fp32 template carries no rounding."""
    n_l, a, b = 300, 2.0, 2.0 ** -12
    lam = 3000.0 + 2.5 * np.arange(n_l)
    flux = np.broadcast_to(a + b * lam, (2, 2, n_l))
    assert np.array_equal(flux.astype(np.float32).astype(np.float64), flux)
    ssp = _ssp(flux, [0.0, 1.0], [-3.0, -2.0], 3000.0, 2.5)
    tel = _tel(100, 3100.0, 6.0)
    for v in (0.0, 250.0, -999.0):
        F = oracle.particle_spectrum(5.0, 0.3, -2.2, v, ssp, tel)
        beta = float(np.float32(v)) / C
        assert np.allclose(F, 5.0 * (a + b * tel.wavelengths() / (1 + beta)), rtol=1e-12, atol=0)


@pytest.mark.parametrize("v", [-600.0, -50.0, 0.0, 220.0, 1500.0])
def test_narrow_line_shifts_to_lambda_times_one_plus_v_over_c(v):
    lam_line, sig = 6562.8, 1.5
    n_l = 4001
    lam = 6000.0 + 0.25 * np.arange(n_l)                          # well sampled: sigma = 6 samples
    prof = 1.0 - 0.8 * np.exp(-0.5 * ((lam - lam_line) / sig) ** 2)
    ssp = _ssp(np.broadcast_to(prof, (2, 2, n_l)), [0.0, 1.0], [-3.0, -2.0], 6000.0, 0.25)
    tel = _tel(1200, 6400.0, 0.3)
    F = oracle.particle_spectrum(1.0, 0.5, -2.5, v, ssp, tel)
    absorb = 1.0 - F
    centroid = (absorb * tel.wavelengths()).sum() / absorb.sum()
    assert abs(centroid - lam_line * (1.0 + float(np.float32(v)) / C)) < 0.003   # 1% of a channel


def test_identity_at_rest_on_coincident_grids_and_zero_outside_coverage(tiny):
    ssp = tiny.ssp
    n_l = ssp.flux.shape[2]
    tel = _tel(n_l, ssp.lambda0, ssp.dlambda)
    F = oracle.particle_spectrum(1.0, ssp.log_age_axis[1], ssp.log_z_axis[1], 0.0, ssp, tel)
    assert np.array_equal(F, ssp.flux[1, 1].astype(np.float64))
    # observed grid sticking out on both sides of the SSP coverage
    tel = _tel(400, float(ssp.lambda0) - 500.0, 20.0)
    F = oracle.particle_spectrum(1.0, ssp.log_age_axis[1], ssp.log_z_axis[1], 100.0, ssp, tel)
    rest = tel.wavelengths() / (1 + float(np.float32(100.0)) / C)
    outside = (rest < ssp.wavelengths()[0]) | (rest > ssp.wavelengths()[-1])
    assert outside.sum() > 30 and (~outside).sum() > 100
    assert (F[outside] == 0).all() and (F[~outside] > 0).all()


# ---------------------------------------------------------------- accumulate (8c-6)
def _brute_force_cube(w):
    """Independent restatement with numpy library routines and a Python loop over particles."""
    p, t, ssp = w.particles, w.telescope, w.ssp
    R = w.rotation.astype(np.float32)
    cube = np.zeros((t.n_spaxels + 1, t.n_channels))
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, t.n_x, t.n_y, t.spaxel_size)   # pinned above
    A, Z = ssp.log_age_axis.astype(np.float64), ssp.log_z_axis.astype(np.float64)
    lam_s, lam_o = ssp.wavelengths(), t.wavelengths()
    T = ssp.flux.astype(np.float64)
    for q in range(p.n):
        i = int(np.clip(np.searchsorted(A, float(p.log_age[q]), "right") - 1, 0, A.size - 2))
        j = int(np.clip(np.searchsorted(Z, float(p.log_z[q]), "right") - 1, 0, Z.size - 2))
        ta = float(np.clip((p.log_age[q] - A[i]) / (A[i + 1] - A[i]), 0, 1))
        tz = float(np.clip((p.log_z[q] - Z[j]) / (Z[j + 1] - Z[j]), 0, 1))
        blend = ((1 - ta) * (1 - tz) * T[i, j] + ta * (1 - tz) * T[i + 1, j]
                 + (1 - ta) * tz * T[i, j + 1] + ta * tz * T[i + 1, j + 1])
        spec = np.interp(lam_o / (1 + float(vlos[q]) / C), lam_s, blend, 0, 0)
        cube[key[q]] += float(p.mass[q]) * spec
    return cube[:-1].reshape(t.n_x, t.n_y, t.n_channels), cube[-1]


def test_cube_equals_brute_force_on_tiny(tiny):
    ref, dropped = _brute_force_cube(tiny)
    cube = oracle.build_cube(tiny.particles, tiny.rotation, tiny.ssp, tiny.telescope)
    assert dropped.sum() > 0                                       # some particles are out of FoV
    assert np.allclose(cube, ref, rtol=1e-12, atol=0)


def test_superposition_permutation_linearity(tiny):
    p, R, ssp, t = tiny.particles, tiny.rotation, tiny.ssp, tiny.telescope
    full = oracle.build_cube(p, R, ssp, t)
    a = oracle.build_cube(p.subset(slice(0, 400)), R, ssp, t)
    b = oracle.build_cube(p.subset(slice(400, None)), R, ssp, t)
    assert np.allclose(a + b, full, rtol=1e-12)
    shuffled = oracle.build_cube(p.subset(np.random.default_rng(2).permutation(p.n)), R, ssp, t)
    assert np.allclose(shuffled, full, rtol=1e-12)
    heavy = p.copy()
    heavy.mass *= np.float32(4.0)                                  # exact in fp32
    assert np.allclose(oracle.build_cube(heavy, R, ssp, t), 4.0 * full, rtol=1e-13)
    empty = oracle.build_cube(p.subset(slice(0, 0)), R, ssp, t)
    assert empty.shape == full.shape and not empty.any()


def test_total_flux_is_conserved_through_binning(tiny):
    p, R, ssp, t = tiny.particles, tiny.rotation, tiny.ssp, tiny.telescope
    cube = oracle.build_cube(p, R, ssp, t)
    key, vlos = oracle.rotate_bin(p.pos, p.vel, R, t.n_x, t.n_y, t.spaxel_size)
    total = np.zeros(t.n_channels)
    for q in np.nonzero(key < t.n_spaxels)[0]:
        total += oracle.particle_spectrum(p.mass[q], p.log_age[q], p.log_z[q], vlos[q], ssp, t)
    assert np.allclose(cube.sum((0, 1)), total, rtol=1e-12)
    counts = np.bincount(key, minlength=t.n_spaxels + 1)[:-1].reshape(t.n_x, t.n_y)
    assert not cube[counts == 0].any() and (cube[counts > 0].sum(-1) > 0).all()


def test_selected_spaxels_equal_rows_of_the_full_cube(small, small_oracle_cube):
    t = small.telescope
    sel = np.array([0, 312, 313, 624, 100], np.int32)
    rows = oracle.build_cube(small.particles, small.rotation, small.ssp, t, sel=sel)
    assert np.array_equal(rows, small_oracle_cube.reshape(t.n_spaxels, -1)[sel])


def test_expected_trends_of_the_paper(small, small_oracle_cube):
    """centre spectra have higher flux than the outskirts."""
    img = small_oracle_cube.sum(-1)
    assert img[12, 12] > 20 * img[12, 2] > 0
