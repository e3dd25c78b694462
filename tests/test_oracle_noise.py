"""Pins for the oracle's noise stage (reading R17; "add realistic noise"):
Philox4x32-10 known answers, the uniform -> normal map, moments of the deviates, the variance model."""
import os

import numpy as np

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]


def test_normals_follow_box_muller_of_the_philox_words():
    seed = 0x0123456789ABCDEF
    z = oracle.noise_normals(10, seed)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for q in range(3):
        r = oracle.philox4x32_10([q, 0, 0, 0], key)
        u = [((x >> 9) + 0.5) / 2.0 ** 23 for x in r]
        assert all(0.0 < v < 1.0 and np.float32(v) == v for v in u)          # exact in fp32, never 0 or 1
        exp = [np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]), np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
               np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3]), np.sqrt(-2 * np.log(u[2])) * np.sin(2 * np.pi * u[3])]
        for i in range(4):
            if 4 * q + i < 10:
                assert np.isclose(z[4 * q + i], exp[i], rtol=1e-13)


def test_deviates_are_standard_normal_and_seeds_are_independent_streams():
    n = 400_000
    z = oracle.noise_normals(n, 42)
    assert abs(z.mean()) < 5 / np.sqrt(n) and abs(z.var() - 1.0) < 5 * np.sqrt(2.0 / n)
    assert abs(np.mean(z ** 3)) < 0.03 and abs(np.mean(z ** 4) - 3.0) < 0.06
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 0.01 and abs(np.corrcoef(z[::2], z[1::2])[0, 1]) < 0.01
    # tail fractions of a normal law
    assert abs((np.abs(z) > 1.959964).mean() - 0.05) < 0.003
    z2 = oracle.noise_normals(n, 43)
    assert abs(np.corrcoef(z, z2)[0, 1]) < 0.01 and not np.array_equal(z[:8], z2[:8])
    assert np.array_equal(z[:1001], oracle.noise_normals(1001, 42))           # a prefix, whatever the length (ragged tail)


def test_variance_model_and_degenerate_cases():
    cube = np.full(200_000, 50.0)
    out = oracle.add_noise(cube, sigma_read=3.0, gain=0.5, seed=7)
    assert abs((out - cube).var() - (9.0 + 0.5 * 50.0)) < 0.5                  # sigma^2 = sigma_read^2 + gain F
    z = oracle.noise_normals(cube.size, 7)
    assert np.allclose(out, cube + np.sqrt(9.0 + 25.0) * z, rtol=1e-14)
    neg = np.array([-4.0, 0.0, 9.0, 100.0])
    o = oracle.add_noise(neg, sigma_read=0.0, gain=1.0, seed=1)
    zz = oracle.noise_normals(4, 1)
    assert np.allclose(o, neg + np.sqrt(np.maximum(neg, 0.0)) * zz)            # negative flux carries no shot noise
    assert np.array_equal(oracle.add_noise(neg, 0.0, 0.0, 5), neg)             # both terms off: identity
    assert oracle.add_noise(np.zeros(0), 1.0, 1.0, 3).size == 0
