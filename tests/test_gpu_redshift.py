"""Parity of the CUDA path with a cosmological redshift and a flux scale (reading R14)
against the fp64 oracle, through the C ABI, in both resampling modes, forward and adjoint."""
import dataclasses

import numpy as np
import pytest

import oracle
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


def shifted(tel, z, scale, mode):
    """The same rest-frame coverage observed at redshift z: grid stretched by (1 + z)."""
    return dataclasses.replace(tel, lambda0=np.float32(float(tel.lambda0) * (1 + z)),
                               dlambda=np.float32(float(tel.dlambda) * (1 + z)), redshift=np.float32(z),
                               flux_scale=np.float32(scale), resample=mode)


@pytest.mark.parametrize("name,z,scale,mode", [("tiny", 0.1, 3.0e-2, 0), ("tiny", 0.1, 3.0e-2, 1),
                                               ("small", 0.35, 4.0, 0), ("small", 0.02, 1.0e-3, 1)])
def test_whole_cube(B, name, z, scale, mode):
    w = synth.make_workload(name)
    w.telescope = shifted(w.telescope, z, scale, mode)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    got = dw.build_cube().cpu().numpy().astype(np.float64)
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    assert np.abs(got - ref).max() <= 1e-4 * ref.max()
    fr = ref.sum(-1)
    pos = fr > 0
    assert (np.abs(got.sum(-1) - fr)[pos] / fr[pos]).max() <= 1e-5
    assert not got[~pos].any()
    # the factors are really applied: the unshifted, unscaled oracle cube is something else
    plain = oracle.build_cube(w.particles, w.rotation, w.ssp,
                              dataclasses.replace(t, redshift=np.float32(0.0), flux_scale=np.float32(1.0)))
    assert np.abs(got - plain).max() > 1e-2 * max(ref.max(), plain.max())


def test_unshifted_grid_at_high_redshift_runs_off_the_coverage(B):
    """z = 1 on the tiny detector grid: rest wavelengths 2350-4650 A, only the red part is covered."""
    w = synth.make_workload("tiny")
    w.telescope = dataclasses.replace(w.telescope, redshift=np.float32(1.0))
    got = B.DeviceWorkload(w).build_cube().cpu().numpy().astype(np.float64)
    ref = oracle.build_cube(w.particles, w.rotation, w.ssp, w.telescope)
    assert np.abs(got - ref).max() <= 1e-4 * ref.max()
    assert not got[..., :100].any() and got[..., -20:].any()


@pytest.mark.parametrize("mode", [0, 1])
def test_adjoint_with_redshift_and_scale(B, mode):
    w = synth.make_workload("adjoint", n=20000)
    w.telescope = shifted(w.telescope, 0.08, 2.5e-2, mode)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    G = upstream_gradient(w)                               # 2 (cube - target) of two galaxies, as in configs[4]
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(torch.from_numpy(G).cuda())]
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, G.astype(np.float64))
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert_gradients(g, ana, key, vlos, w.ssp, t, "test_gpu_redshift.py")


def test_bad_redshift_and_scale_are_rejected(B):
    w = synth.make_workload("tiny")
    for field, value in (("flux_scale", 0.0), ("flux_scale", float("inf")), ("redshift", -0.1), ("redshift", 25.0)):
        w2 = dataclasses.replace(w, telescope=dataclasses.replace(w.telescope, **{field: np.float32(value)}))
        with pytest.raises(B.RubixError):                 # rubix_workspace_bytes already validates the telescope
            B.DeviceWorkload(w2).build_cube()
        assert field.split("_")[0] in B.rubix_last_error()
