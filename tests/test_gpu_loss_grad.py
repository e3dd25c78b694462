"""rubix_loss_and_grad (fused forward + quadratic loss + adjoint) against the fp64
oracle: L = sum (final cube - target)^2 and its gradients (BASELINE.json configs[4])."""
import dataclasses

import numpy as np
import pytest

import oracle
from gradcheck import assert_gradients
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


def check(B, w, seed_other):
    """The fused call stage by stage (reading R19): the final cube against the oracle's (1e-4 of its maximum),
    the loss against the oracle's loss, and the gradients -- maximum over ALL particles, 1e-3 -- against the oracle's
    adjoint of the upstream gradient the call itself formed, 2 (cube_out - target).  (How the cube's own voxel error
    moves a gradient is linear, Adj(2 delta), and a property of the loss, not of the kernels: a particle whose gradient
    nearly cancels can see 1e-2 of its value from a 1e-6 voxel error; that composition is bounded below as well.)"""
    t = w.telescope
    other = synth.make_particles_for("tiny" if w.name == "tiny" else "adjoint", n=w.particles.n, seed=seed_other)
    target = oracle.forward(other, w.rotation, w.ssp, t)               # never from the CUDA path
    ref_final = oracle.forward(w.particles, w.rotation, w.ssp, t)
    target32 = target.astype(np.float32)
    dw = B.DeviceWorkload(w)
    loss, g, cube = dw.loss_and_grad(torch.from_numpy(target32).cuda(), want_cube=True)
    torch.cuda.synchronize()
    resid = ref_final - target32.astype(np.float64)
    L_ref = float((resid ** 2).sum())
    assert abs(float(loss.item()) - L_ref) <= 2e-4 * L_ref
    got_cube = cube.cpu().numpy().astype(np.float64)
    assert np.abs(got_cube - ref_final).max() <= 1e-4 * ref_final.max()
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    gg = [x.cpu().numpy() for x in g]
    # gradients of the upstream gradient the call formed: maximum over all particles
    up = (2.0 * (cube.cpu().numpy() - target32)).astype(np.float64)    # fp32 subtraction, as the kernel does it
    ana_own = oracle.adjoint(w.particles, w.rotation, w.ssp, t, up)
    stats = assert_gradients(gg, ana_own, key, vlos, w.ssp, t, "fused call")
    print("fused call, max relative gradient errors:", stats)
    # composition: against the oracle's own residual the difference is Adj(2 delta), delta = the cube's voxel error
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * resid)
    lin = oracle.adjoint(w.particles, w.rotation, w.ssp, t, 2.0 * (got_cube - ref_final))
    for q in range(4):
        scale = np.maximum(np.abs(ana[q]), 1e-3 * np.median(np.abs(ana[q][key < t.n_spaxels])))
        assert (np.abs(gg[q] - ana[q] - lin[q]) / np.where(scale > 0, scale, 1.0)).max() <= 1e-3
    # without cube_out the call runs the same kernels: loss and gradients bit for bit
    loss2, g2, none = dw.loss_and_grad(torch.from_numpy(target32).cuda(), want_cube=False)
    assert none is None and float(loss2.item()) == float(loss.item())  # fixed-order fp64 sum: bit-reproducible
    for a, b2 in zip(g, g2):
        assert torch.equal(a, b2)
    # and the fused call equals the three separate calls bit for bit (same kernels, same order)
    final = dw.forward()
    grad = 2.0 * (final - torch.from_numpy(target32).cuda())
    g_sep = dw.adjoint(grad)
    for a, b2 in zip(g, g_sep):
        assert torch.equal(a, b2)
    return float(loss.item())


@pytest.mark.parametrize("mode", [0, 1])
def test_config4_fused(B, mode):
    w = synth.make_workload("adjoint", n=30000)
    w.telescope = dataclasses.replace(w.telescope, resample=mode)
    check(B, w, synth.ADJOINT_TARGET_SEED)


def test_without_psf_lsf(B):
    w = synth.make_workload("tiny")
    check(B, w, synth.ADJOINT_TARGET_SEED)


def test_workspace_check(B):
    w = synth.make_workload("tiny")
    dw = B.DeviceWorkload(w)
    small = dw.workspace                                               # sized for the plain calls only
    t = torch.zeros(dw.shape, device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    g = [torch.empty(w.particles.n, device="cuda") for _ in range(4)]
    with pytest.raises(B.RubixError):
        B.rubix_loss_and_grad(dw.particles, dw.ssp, dw.tel, dw.R, t, loss, None, *g, small)
    assert "workspace" in B.rubix_last_error()
