"""The seeded generator: shapes, ranges and determinism."""
import json
import os

import numpy as np

import oracle
from paper_2412_08265_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_generator_has_not_drifted(tiny, small):
    gold = json.load(open(os.path.join(GOLD, "synth_sha256.json")))
    for w in (tiny, small):
        for f in ("pos", "vel", "mass", "log_age", "log_z"):
            assert synth.sha256(getattr(w.particles, f)) == gold[f"{w.name}.particles.{f}"], f
        assert synth.sha256(w.ssp.flux) == gold[f"{w.name}.ssp.flux"]
        assert synth.sha256(w.rotation) == gold[f"{w.name}.rotation"]
    for name in ("medium", "contention"):
        assert np.allclose(synth.euler_for(name), gold[f"{name}.euler_deg"], atol=1e-8)


def test_oracle_tiny_fixture(tiny):
    gold = json.load(open(os.path.join(GOLD, "oracle_tiny.json")))
    t = tiny.telescope
    cube = oracle.forward(tiny.particles, tiny.rotation, tiny.ssp, t)
    assert np.isclose(cube.sum(), gold["total_flux"], rtol=1e-12)
    assert np.isclose(cube.max(), gold["max_voxel"], rtol=1e-12)
    assert list(np.unravel_index(cube.argmax(), cube.shape)) == gold["argmax"]
    for k, v in gold["voxels"].items():
        assert np.isclose(cube[tuple(int(i) for i in k.split(","))], v, rtol=1e-12)


def test_shapes_dtypes_and_ranges(tiny, small):
    for w, n, grid, det in ((tiny, 1000, (8, 4, 512), (16, 16, 256)),
                            (small, 100_000, (50, 7, 4300), (25, 25, 3700))):
        p = w.particles
        assert p.n == n and p.pos.shape == (n, 3) and p.vel.shape == (n, 3)
        for a in (p.pos, p.vel, p.mass, p.log_age, p.log_z, w.ssp.flux, w.rotation):
            assert a.dtype == np.float32 and a.flags.c_contiguous and np.isfinite(a).all()
        assert w.ssp.flux.shape == grid and (w.ssp.flux > 0).all()
        t = w.telescope
        assert (t.n_x, t.n_y, t.n_channels) == det
        assert np.all(np.diff(w.ssp.log_age_axis) > 0) and np.all(np.diff(w.ssp.log_z_axis) > 0)
        assert 10 ** p.log_age.min() >= 0.0999 and 10 ** p.log_age.max() <= 13.51
        assert 10 ** p.log_z.min() >= 0.99e-4 and 10 ** p.log_z.max() <= 0.0301
        assert 0.9e5 < np.median(p.mass) < 1.1e5
        # observed range sits inside the SSP coverage even after Doppler shifts
        assert w.ssp.wavelengths()[0] < t.wavelengths()[0] / 1.01
        assert w.ssp.wavelengths()[-1] > t.wavelengths()[-1] * 1.01
    assert np.isclose(tiny.telescope.wavelengths()[-1], 9300.0, atol=1e-3)
    assert np.isclose(small.telescope.wavelengths()[-1], 9373.75)
    assert np.isclose(small.ssp.wavelengths()[-1], 10000.0, atol=1e-2)


def test_disc_bulge_structure(small):
    r = np.linalg.norm(small.particles.pos[:, :2], axis=1)
    assert 4.5 < np.median(r) < 5.5            # Gamma(2, 3 kpc) disc median = 5.03 kpc, bulge pulls in
    assert np.mean(np.abs(small.particles.pos[:, 2]) < 0.3) > 0.55
    v_phi = (-small.particles.vel[:, 0] * small.particles.pos[:, 1]
             + small.particles.vel[:, 1] * small.particles.pos[:, 0]) / np.maximum(r, 1e-6)
    assert 190 < np.median(v_phi) < 210        # flat 200 km/s rotation curve


def test_contention_workload_is_centrally_concentrated():
    w = synth.make_workload("contention", n=200_000)
    t = w.telescope
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    counts = np.bincount(key, minlength=t.n_spaxels + 1)[:-1]
    assert np.sort(counts)[-4:].sum() > 0.25 * w.particles.n   # SURVEY: ~36 % in the central four
    assert w.ssp.flux.shape == (100, 12, 4300)
