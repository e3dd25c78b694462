"""Pins for the oracle's steps 1-3 (rotate, project/bin, sort).  SURVEY.md 8(c) rows 1-3.

None of these retype the oracle's formula: they are invariants (orthonormality, counts),
hand-computed cases, and library routines (numpy.histogram2d, numpy.argsort)."""
import numpy as np
import pytest

import oracle
from paper_2412_08265_b200 import synth


def _eye():
    return np.eye(3, dtype=np.float32)


# ---------------------------------------------------------------- rotation (8c-1)
@pytest.mark.parametrize("euler", [(0, 0, 0), (0, 90, 0), (0, 60, 0), (33, 71, 250),
                                   synth.random_euler(3002), synth.random_euler(3003)])
def test_rotation_is_orthonormal_and_preserves_norms(euler):
    R = synth.euler_rotation(*euler).astype(np.float64)
    assert np.allclose(R.T @ R, np.eye(3), atol=1e-6)
    assert np.isclose(np.linalg.det(R), 1.0, atol=1e-6)
    r = np.random.default_rng(0).normal(size=(1000, 3))
    assert np.allclose(np.linalg.norm(r @ R.T, axis=1), np.linalg.norm(r, axis=1), rtol=1e-6)


def test_rotation_conventions():
    assert np.array_equal(synth.euler_rotation(0, 0, 0), _eye())
    # "edge-on (0,90,0)" = R_y(90 deg) maps z-hat onto x-hat: the disc normal lands in the sky plane
    R = synth.euler_rotation(0, 90, 0).astype(np.float64)
    assert np.allclose(R @ [0, 0, 1], [1, 0, 0], atol=1e-7)
    # inclination 60 deg: disc normal 60 deg away from the line of sight (+z')
    R = synth.euler_rotation(0, 60, 0).astype(np.float64)
    assert np.isclose((R @ [0, 0, 1])[2], 0.5, atol=1e-6)


def test_vlos_is_the_third_rotated_component():
    """Using R, and R with its rows cyclically permuted, as the orientation makes each rotated
    velocity component the line of sight once; their squares must add up to |v|^2."""
    rng = np.random.default_rng(1)
    vel = rng.normal(0, 200, (500, 3)).astype(np.float32)
    pos = np.zeros_like(vel)
    R = synth.euler_rotation(10, 40, 70)
    tot = np.zeros(500)
    for shift in range(3):
        _, vlos = oracle.rotate_bin(pos, vel, np.roll(R, shift, axis=0), 4, 4, 1.0)
        tot += vlos.astype(np.float64) ** 2
    assert np.allclose(tot, (vel.astype(np.float64) ** 2).sum(1), rtol=1e-5)
    # identity orientation: v_los = v_z exactly; receding = positive
    _, vlos = oracle.rotate_bin(pos, vel, _eye(), 4, 4, 1.0)
    assert np.array_equal(vlos, vel[:, 2])


def test_edge_on_projection_puts_z_on_the_x_axis():
    pos = np.array([[0.2, 0.3, 2.5]], np.float32)       # R_y(90): x' = z = 2.5, y' = y = 0.3
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), synth.euler_rotation(0, 90, 0), 16, 16, 1.0)
    assert key[0] == 10 * 16 + 8


# ---------------------------------------------------------------- binning (8c-2)
def test_spaxel_centres_land_in_their_spaxel_nonsquare():
    n_x, n_y, s = 7, 5, 0.5
    ix, iy = np.meshgrid(np.arange(n_x), np.arange(n_y), indexing="ij")
    pos = np.stack([(ix + 0.5) * s - 0.5 * n_x * s, (iy + 0.5) * s - 0.5 * n_y * s,
                    np.zeros_like(ix, dtype=float)], -1).reshape(-1, 3).astype(np.float32)
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), _eye(), n_x, n_y, s)
    assert np.array_equal(key, (ix * n_y + iy).reshape(-1))     # key = ix * N_y + iy


def test_edges_hand_checked():
    n_x, n_y, s = 4, 6, 2.0            # half widths 4 and 6 kpc; all values exact in fp32
    P = lambda x, y: [x, y, 0.0]
    pos = np.array([P(-4.0, 0.0),      # u = 0 exactly: lower edge inclusive -> ix 0, iy 3
                    P(4.0, 0.0),       # u = N_x exactly: upper edge exclusive -> out
                    P(0.0, -6.0),      # v = 0 -> iy 0, ix 2
                    P(0.0, 6.0),       # v = N_y -> out
                    P(-2.0, 2.0),      # u = 1, v = 4: integer u goes to the upper spaxel
                    P(3.999999, 5.999999),
                    P(-4.000001, 0.0),  # just outside
                    P(np.nan, 0.0), P(0.0, np.inf), P(-np.inf, 0.0)], np.float32)
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), _eye(), n_x, n_y, s)
    out = n_x * n_y
    assert key.tolist() == [0 * 6 + 3, out, 2 * 6 + 0, out, 1 * 6 + 4, 3 * 6 + 5, out, out, out, out]


def test_velocity_cap_and_nan_velocity_drop_the_particle():
    pos = np.zeros((4, 3), np.float32)
    vel = np.array([[0, 0, 14989.0], [0, 0, 14990.5], [0, 0, -14990.5], [0, 0, np.nan]], np.float32)
    key, _ = oracle.rotate_bin(pos, vel, _eye(), 2, 2, 1.0)
    assert key.tolist() == [3, 4, 4, 4]


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_histogram2d_brute_force(name):
    w = synth.make_workload(name)
    t = w.telescope
    # identity orientation: the fp32 coordinate u is a single add and a single divide
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, _eye(), t.n_x, t.n_y, t.spaxel_size)
    s = np.float32(t.spaxel_size)
    u = (w.particles.pos[:, 0] + np.float32(0.5 * t.n_x) * s) / s
    v = (w.particles.pos[:, 1] + np.float32(0.5 * t.n_y) * s) / s
    assert u.dtype == np.float32
    H, _, _ = np.histogram2d(u, v, bins=[np.arange(t.n_x + 1), np.arange(t.n_y + 1)])
    counts = np.bincount(key, minlength=t.n_spaxels + 1)
    assert np.array_equal(counts[:-1].reshape(t.n_x, t.n_y), H.astype(np.int64))
    assert counts.sum() == w.particles.n and counts[-1] == w.particles.n - int(H.sum())


def test_every_key_is_in_range_for_the_rotated_configs(tiny, small):
    for w in (tiny, small):
        t = w.telescope
        key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y,
                                   t.spaxel_size)
        assert key.min() >= 0 and key.max() <= t.n_spaxels
        # rotation by R then binning == binning the pre-rotated points with the identity
        # whenever the pre-rotated coordinates are far from an edge (fp32 vs fp64 rounding)
        rot = w.particles.pos.astype(np.float64) @ w.rotation.astype(np.float64).T
        u = rot[:, 0] / float(t.spaxel_size) + 0.5 * t.n_x
        v = rot[:, 1] / float(t.spaxel_size) + 0.5 * t.n_y
        safe = (np.abs(u - np.round(u)) > 1e-3) & (np.abs(v - np.round(v)) > 1e-3)
        inside = (u >= 0) & (u < t.n_x) & (v >= 0) & (v < t.n_y)
        ref = np.where(inside, np.floor(u) * t.n_y + np.floor(v), t.n_spaxels).astype(np.int64)
        assert safe.mean() > 0.99
        assert np.array_equal(key[safe], ref[safe])


# ---------------------------------------------------------------- sort (8c-3)
@pytest.mark.parametrize("n,n_s", [(0, 5), (1, 1), (1000, 7), (50_000, 625), (20_000, 90_000)])
def test_sort_equals_stable_argsort(n, n_s):
    key = np.random.default_rng(n + n_s).integers(0, n_s + 1, n).astype(np.int32)
    perm, seg = oracle.sort(key, n_s)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.int32))
    assert np.array_equal(np.sort(perm), np.arange(n))                      # bijection
    assert np.all(np.diff(key[perm]) >= 0)                                  # keys non-decreasing
    assert seg.shape == (n_s + 2,) and seg[0] == 0 and seg[-1] == n
    assert np.array_equal(np.diff(seg), np.bincount(key, minlength=n_s + 1))
    for s in np.unique(key)[:20]:
        assert np.all(np.diff(perm[seg[s]:seg[s + 1]]) > 0)                 # ties by original index


# ---------------------------------------------------------------- fp32 operation order (8c-2)
# SURVEY.md 8(c)-2 / DESIGN.md R2 DEFINE the binning in fp32: every * and + separately rounded, in the order
#   xr = (R00*x + R01*y) + R02*z ;  hx = (0.5f*N_x)*s ;  u = (xr + hx) / s
# (hx needs no case of its own: multiplying by 0.5 is exact, so every association of 0.5f, N_x and s agrees.)
# The cases below are built so that a different association, an FMA contraction or a re-arranged
# division moves u across a spaxel edge.  Expected keys: derived by hand (literal values, derivation in
# the comments) or evaluated with numpy.float32 ops, which round after every operation.
F = np.float32


def _key_in_order(pos, R, n_x, n_y, s, variant="spec"):
    """numpy.float32 evaluation (one rounding per op).  variant 'spec' is the order of 8(c)-2;
    the others are the plausible mistakes the cases must tell apart from it."""
    pos = np.asarray(pos, F)
    R = np.asarray(R, F).reshape(3, 3)
    s = F(s)
    x, y, z = pos[:, 0], pos[:, 1], pos[:, 2]

    def coord(r, n):
        a, b, c = r[0] * x, r[1] * y, r[2] * z                 # three separately rounded products
        if variant == "assoc_right":
            rot = a + (b + c)
        elif variant == "fma":                                  # fma(r0, x, r1*y): the first product unrounded
            rot = (r[0].astype(np.float64) * x.astype(np.float64) + b.astype(np.float64)).astype(F) + c
        else:
            rot = (a + b) + c
        h = (F(0.5) * F(n)) * s
        if variant == "div_split":
            return rot / s + h / s
        return (rot + h) / s

    u, v = coord(R[0], n_x), coord(R[1], n_y)
    assert u.dtype == np.float32
    inside = (u >= 0) & (u < n_x) & (v >= 0) & (v < n_y)
    with np.errstate(invalid="ignore"):
        return np.where(inside, np.floor(u).astype(np.int64) * n_y + np.floor(v).astype(np.int64), n_x * n_y)


def test_association_order_hand_built():
    """R00*x = 1, R01*y = R02*z = 2^-24.  (1 + 2^-24) is a tie and rounds to the even 1, and again
    1 + 2^-24 -> 1, so the specified order gives xr = 1; a + (b + c) gives 1 + 2^-23.
    With s = 1 + 2^-23 and N_x = 2: hx = s; spec: 1 + s = 2 + 2^-23 is a tie -> 2.0, u = 2/s < 2 -> ix = 1;
    other order: (1 + 2^-23) + s = 2 + 2^-22 exactly, u = 2 = N_x -> outside."""
    s = F(1.0) + F(2.0 ** -23)
    R = np.array([[0.5, 2.0 ** -10, 2.0 ** -12], [0.0, 0.0, 0.0], [0.0, 0.0, 1.0]], F)
    pos = np.array([[2.0, 2.0 ** -14, 2.0 ** -12]], F)          # products: 1, 2^-24, 2^-24 (all exact)
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), R, 2, 2, s)
    # y' = 0 -> v = (0 + s)/s = 1 -> iy = 1;  ix = 1  =>  key = 1*2 + 1
    assert key.tolist() == [3]
    assert _key_in_order(pos, R, 2, 2, s, "spec").tolist() == [3]
    assert _key_in_order(pos, R, 2, 2, s, "assoc_right").tolist() == [4]      # the mistake is visible


def test_fma_contraction_hand_built():
    """R00 = 1 + 2^-12, x = 4097: the exact product 4098 + 2^-12 is a tie in fp32 (spacing 2^-11) and
    rounds to the even 4098; R01*y = -4098.  Separately rounded: xr = 0; fma(R00, x, R01*y) = 2^-12.
    s = 2^-12, N_x = 2: hx = 2^-12; spec: u = 2^-12/2^-12 = 1 -> ix = 1; contracted: u = 2 = N_x -> outside."""
    s = F(2.0 ** -12)
    R = np.array([[1.0 + 2.0 ** -12, -1.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, 1.0]], F)
    pos = np.array([[4097.0, 4098.0, 0.0]], F)
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), R, 2, 2, s)
    assert key.tolist() == [1 * 2 + 1]
    assert _key_in_order(pos, R, 2, 2, s, "spec").tolist() == [3]
    assert _key_in_order(pos, R, 2, 2, s, "fma").tolist() == [4]


@pytest.mark.parametrize("euler,n_x,n_y,s", [((33.0, 71.0, 250.0), 25, 25, 1.2), (synth.random_euler(3002), 300, 300, 0.1),
                                             ((10.0, 40.0, 70.0), 7, 5, 0.37)])
def test_operation_order_on_edge_particles(euler, n_x, n_y, s):
    """Particles placed within a few ulp of spaxel edges under a real rotation: the oracle must equal the
    numpy.float32 evaluation in the specified order on ALL of them, and the set must contain particles
    that each plausible mistake bins differently (otherwise it would prove nothing)."""
    rng = np.random.default_rng(77)
    R = synth.euler_rotation(*euler)
    R64 = R.astype(np.float64)
    n = 200_000
    # pick a target edge coordinate in x', solve for the unrotated point, jitter by a few ulp
    ex = rng.integers(0, n_x + 1, n).astype(np.float64)
    ey = rng.uniform(0, n_y, n)
    zz = rng.normal(0, 3.0, n)
    target = np.stack([(ex - 0.5 * n_x) * s, (ey - 0.5 * n_y) * s, zz], 1)
    pos = (target @ R64).astype(F)                              # r = R^T r'
    pos = np.nextafter(pos, np.where(rng.random(pos.shape) < 0.5, -np.inf, np.inf).astype(F)).astype(F)
    key, _ = oracle.rotate_bin(pos, np.zeros_like(pos), R, n_x, n_y, F(s))
    spec = _key_in_order(pos, R, n_x, n_y, s, "spec")
    assert np.array_equal(key, spec)
    for variant in ("assoc_right", "fma", "div_split"):
        other = _key_in_order(pos, R, n_x, n_y, s, variant)
        assert (other != spec).sum() >= 20, variant           # the case set discriminates this mistake
