"""rubix_add_noise (reading R17) against the fp64 oracle: both sides implement the same
counter-based generator (Philox4x32-10 + Box-Muller), so the noisy cubes agree voxel by voxel."""
import numpy as np
import pytest

import oracle
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


@pytest.mark.parametrize("n,sr,gain,seed", [(4096 * 37 + 3, 2.5, 0.3, 7), (1, 1.0, 0.0, 2 ** 63 + 5), (6, 0.0, 2.0, 11),
                                            (1000003, 0.7, 0.05, 0xDEADBEEFCAFE)])
def test_noisy_cube_matches_the_oracle(B, n, sr, gain, seed):
    cube = synth.synthetic_cube(1, 1, n, seed=3).reshape(-1) * np.float32(200.0) - np.float32(1.0)   # some negatives
    d_in = torch.from_numpy(cube).cuda()
    d_out = torch.full_like(d_in, float("nan"))
    B.rubix_add_noise(d_in, d_out, sr, gain, seed)
    torch.cuda.synchronize()
    ref = oracle.add_noise(cube.astype(np.float64), sr, gain, seed)
    got = d_out.cpu().numpy().astype(np.float64)
    sigma = np.sqrt(sr * sr + gain * np.maximum(cube.astype(np.float64), 0.0))
    # fp32 log / sincos / sqrt against fp64: a few 1e-6 of sigma (|n_v| <= 5.7), plus fp32 rounding of the sum
    assert np.abs(got - ref).max() <= 2e-5 * max(sigma.max(), 1e-30) + 1e-6 * np.abs(ref).max()
    assert np.abs(got - ref).max() <= 1e-4 * np.abs(ref).max()
    # in place, and an unaligned view (scalar path)
    B.rubix_add_noise(d_in, d_in, sr, gain, seed)
    assert torch.equal(d_in, d_out)
    if n > 8:
        src = torch.from_numpy(cube).cuda()
        dst = torch.empty(n + 1, device="cuda")
        B.rubix_add_noise(src[1:], dst[1:n], sr, gain, seed)
        ref1 = oracle.add_noise(cube[1:].astype(np.float64), sr, gain, seed)
        assert np.abs(dst[1:n].cpu().numpy() - ref1).max() <= 1e-4 * np.abs(ref1).max()


def test_extreme_uniform_words(B):
    """the largest uniform, u = 1 - 2^-24 (Philox word >> 9 = 0x7FFFFF), is where an approximate
    log loses all relative accuracy of -ln u and may even return a positive value (NaN after the square root).  With
    seed 4 the first 2^24 voxels contain that word three times (radius sqrt(-2 ln u) = 3.4527e-4; found with the oracle's
    generator); the deviates there and everywhere else must match the fp64 oracle."""
    n = 1 << 24
    z = oracle.noise_normals(n, 4)
    radius = np.hypot(z[0::2], z[1::2])
    extreme = np.flatnonzero(radius < 3.5e-4)
    assert extreme.size == 3 and abs(radius[extreme[0]] - np.sqrt(-2.0 * np.log(1.0 - 2.0 ** -24))) < 1e-12
    zero = torch.zeros(n, device="cuda")
    out = torch.empty_like(zero)
    B.rubix_add_noise(zero, out, 1.0, 0.0, 4)                 # cube = 0, sigma_read = 1: the output IS the deviate
    got = out.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    assert np.abs(got - z).max() <= 1e-5
    pair = np.stack([got[2 * extreme], got[2 * extreme + 1]], 1)
    ref = np.stack([z[2 * extreme], z[2 * extreme + 1]], 1)
    assert np.abs(pair - ref).max() <= 2e-8                   # 1e-4 relative of the 3.45e-4 radius


def test_zero_noise_is_the_identity_and_seeds_differ(B):
    cube = torch.from_numpy(synth.synthetic_cube(4, 4, 100, seed=1)).cuda()
    out = torch.empty_like(cube)
    B.rubix_add_noise(cube, out, 0.0, 0.0, 5)
    assert torch.equal(out, cube)
    a, b = torch.empty_like(cube), torch.empty_like(cube)
    B.rubix_add_noise(cube, a, 1.0, 0.0, 5)
    B.rubix_add_noise(cube, b, 1.0, 0.0, 6)
    assert not torch.equal(a, b)
    z = (a - cube).flatten().double()
    assert abs(float(z.mean())) < 0.2 and abs(float(z.var()) - 1.0) < 0.2


def test_bad_arguments(B):
    cube = torch.zeros(64, device="cuda")
    for sr, gain in ((-1.0, 0.0), (0.0, -2.0), (float("nan"), 0.0)):
        with pytest.raises(B.RubixError):
            B.rubix_add_noise(cube, cube, sr, gain, 1)
    with pytest.raises(B.RubixError):
        B.rubix_add_noise(cube[:32], cube[8:40], 1.0, 0.0, 1)             # partial overlap
