"""rubix_residual_loss_static: the loss step without a workspace or any allocation (its partial sums sit in a file-scope
device array of the library, include/rubix.h) against the existing path, rubix_loss_and_grad / rubix_loss_and_grad_batched,
on two calls in a row.  Collected last on purpose (the file name): a failure here must not hide another test under -x."""
import numpy as np
import pytest

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


def existing_path(B, dw, target):
    """(loss, final cube) of the fused call that keeps its partial sums in the caller's workspace."""
    loss, _, cube = dw.loss_and_grad(target, want_cube=True)
    torch.cuda.synchronize()
    return loss.clone(), cube.clone()


def static_path(B, cube, target, batch=1):
    grads = torch.full_like(cube, float("nan"))
    loss = torch.full((batch,), float("nan"), dtype=torch.float64, device="cuda")
    B.rubix_residual_loss_static(cube, target, grads, loss, batch=batch)
    torch.cuda.synchronize()
    return loss, grads


def test_two_calls_in_a_row_match_the_workspace_path(B):
    w = synth.make_workload("adjoint", n=20000)                 # 25 x 25 x 3700 voxels, PSF + LSF
    dw = B.DeviceWorkload(w)
    rng = np.random.default_rng(11)
    shape = dw.shape
    scale = float(dw.forward().max().item())
    for call, spread in enumerate((0.3, 7.0)):                  # two calls, losses orders of magnitude apart: nothing of
        target = torch.from_numpy((rng.uniform(0.0, spread * scale, size=shape)).astype(np.float32)).cuda()   # call 1 leaks into 2
        loss_ref, cube = existing_path(B, dw, target)
        loss, grads = static_path(B, cube, target)
        assert torch.isfinite(loss).all()
        # same kernels, same fixed-order fp64 sum: equal to the last bit; the tolerance the loss tests use is 2e-4
        assert abs(float(loss[0].item()) - float(loss_ref[0].item())) <= 1e-13 * float(loss_ref[0].item()), call
        assert float(loss[0].item()) == float(loss_ref[0].item()), call
        assert torch.equal(grads, 2.0 * (cube - target)), call   # the upstream gradient of step 9, exact in fp32
        want = float(((cube - target).double() ** 2).sum().item())   # the residual is the fp32 difference, squared and summed in fp64
        assert abs(float(loss[0].item()) - want) <= 1e-12 * want
    # the gradients of the existing path follow from these grads through rubix_cube_adjoint (the three-call form)
    _, g_ref, _ = dw.loss_and_grad(target, want_cube=False)
    g = dw.adjoint(grads)
    torch.cuda.synchronize()
    for a, b2 in zip(g, g_ref):
        assert torch.equal(a, b2)


def test_batched_and_the_limit(B):
    base = synth.make_workload("tiny")
    t = base.telescope
    rng = np.random.default_rng(5)
    for batch in (1, 7, B.RESIDUAL_LOSS_STATIC_MAX_BATCH):      # 64 = every slot of the static array in use
        cubes = torch.from_numpy(rng.uniform(0.0, 3.0, size=(batch, t.n_x, t.n_y, t.n_channels)).astype(np.float32)).cuda()
        targets = torch.from_numpy(rng.uniform(0.0, 3.0, size=cubes.shape).astype(np.float32)).cuda()
        loss, grads = static_path(B, cubes, targets, batch)
        assert torch.equal(grads, 2.0 * (cubes - targets))
        want = ((cubes - targets).double() ** 2).sum(dim=(1, 2, 3))
        assert torch.allclose(loss, want, rtol=1e-12, atol=0.0)
        # every element alone gives the same bits as inside the batch (one row of partials per element)
        for b in (0, batch - 1):
            one, _ = static_path(B, cubes[b], targets[b])
            assert float(one[0].item()) == float(loss[b].item())
    too_many = B.RESIDUAL_LOSS_STATIC_MAX_BATCH + 1
    x = torch.zeros((too_many, 8), dtype=torch.float32, device="cuda")
    with pytest.raises(B.RubixError) as e:
        B.rubix_residual_loss_static(x, x.clone(), torch.empty_like(x), torch.zeros(too_many, dtype=torch.float64, device="cuda"),
                                     batch=too_many)
    assert e.value.status == B.RUBIX_ERR_UNSUPPORTED and "exceeds" in str(e.value) and "64" in str(e.value)


def test_odd_sizes_and_unaligned_views(B):
    rng = np.random.default_rng(9)
    for n, off in ((1, 0), (1027, 0), (4099, 1), (10_000_001, 3)):   # scalar path for views that are not 16-byte aligned
        c = torch.from_numpy(rng.normal(size=n + off).astype(np.float32)).cuda()[off:]
        t = torch.from_numpy(rng.normal(size=n + off).astype(np.float32)).cuda()[off:]
        grads = torch.full((n + off,), float("nan"), dtype=torch.float32, device="cuda")[off:]
        loss = torch.zeros(1, dtype=torch.float64, device="cuda")
        B.rubix_residual_loss_static(c, t, grads, loss)
        torch.cuda.synchronize()
        assert torch.equal(grads, 2.0 * (c - t))
        want = float(((c - t).double() ** 2).sum().item())
        assert abs(float(loss.item()) - want) <= 1e-12 * want
