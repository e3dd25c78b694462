"""rubix_loss_and_grad_batched (many galaxies per fused forward + loss + adjoint call, PAPER.md L32,
L86) through the C ABI: every element's cube and gradients bit-equal to a single rubix_loss_and_grad call on that
galaxy, its loss equal (bit-equal when the voxel count is a multiple of 4), and one element against the fp64 oracle."""
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


def rotations(batch, seed):
    return np.stack([synth.euler_rotation(*synth.random_euler(seed + b)) for b in range(batch)]).astype(np.float32)


def concat(gals):
    return synth.Particles(*(np.concatenate([getattr(g, f) for g in gals]) for f in ("pos", "vel", "mass", "log_age", "log_z")))


def run_batched(B, parts, offsets, batch, ssp, tel, R, targets, want_cubes=True):
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    arrays = [up(a) for a in (parts.pos, parts.vel, parts.mass, parts.log_age, parts.log_z)]
    flux = up(ssp.flux)
    cp, cs, ct = B.c_particles(*arrays), B.c_ssp(ssp, flux), B.c_telescope(tel)
    ws = torch.empty(B.rubix_loss_and_grad_batched_workspace_bytes(parts.n, offsets, batch, cs, ct), dtype=torch.uint8, device="cuda")
    ws.view(torch.float32)[: ws.numel() // 4].fill_(float("nan"))
    cubes = torch.full((batch, tel.n_x, tel.n_y, tel.n_channels), float("nan"), dtype=torch.float32, device="cuda") if want_cubes else None
    loss = torch.full((batch,), float("nan"), dtype=torch.float64, device="cuda")
    g = [torch.full((max(parts.n, 1),), float("nan"), dtype=torch.float32, device="cuda") for _ in range(4)]
    B.rubix_loss_and_grad_batched(cp, offsets, batch, cs, ct, R, targets, loss, cubes, *g, ws)
    torch.cuda.synchronize()
    return loss, cubes, [x[: parts.n] for x in g], B.rubix_last_launch_count()


def single(B, parts, ssp, tel, R, target):
    w = synth.Workload("one", parts, ssp, tel, R, (0.0, 0.0, 0.0))
    loss, g, cube = B.DeviceWorkload(w).loss_and_grad(target, want_cube=True)
    torch.cuda.synchronize()
    return loss, g, cube


def make_case(sizes, seed, tel):
    gals = [synth.make_particles_for("tiny", n=max(n, 1), seed=seed + i).subset(np.arange(n)) for i, n in enumerate(sizes)]
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    rng = np.random.default_rng(seed)
    targets = torch.from_numpy(rng.uniform(0.0, 1e-3, size=(len(sizes), tel.n_x, tel.n_y, tel.n_channels)).astype(np.float32)).cuda()
    return gals, offsets, targets


@pytest.mark.parametrize("conv,mode", [(False, 0), (True, 0), (True, 1)])
def test_elements_equal_single_calls(B, conv, mode):
    base = synth.make_workload("tiny")
    tel = base.telescope.with_psf_lsf() if conv else base.telescope
    tel = dataclasses.replace(tel, resample=mode)
    assert (tel.n_x * tel.n_y * tel.n_channels) % 4 == 0
    sizes = [1000, 1, 0, 317, 2500, 40]                        # ragged, one empty, one single-particle galaxy
    gals, offsets, targets = make_case(sizes, 900, tel)
    R = rotations(len(sizes), 11)
    loss, cubes, g, launches = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R, targets)
    assert launches > 0 and torch.isfinite(loss).all() and torch.isfinite(cubes).all()
    for x in g:
        assert torch.isfinite(x).all()
    for b, gal in enumerate(gals):
        if gal.n == 0:
            assert not cubes[b].any()
            want = float((targets[b].double() ** 2).sum().item())
            assert abs(float(loss[b].item()) - want) <= 1e-6 * want
            continue
        l1, g1, c1 = single(B, gal, base.ssp, tel, R[b], targets[b])
        assert torch.equal(cubes[b], c1), b
        assert float(loss[b].item()) == float(l1.item()), b    # same fixed-order fp64 sum
        lo, hi = int(offsets[b]), int(offsets[b + 1])
        for q in range(4):
            assert torch.equal(g[q][lo:hi], g1[q]), (b, q)
    # without cubes_out: same kernels, same numbers
    loss2, none, g2, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R, targets, want_cubes=False)
    assert none is None and torch.equal(loss, loss2)
    for a, b2 in zip(g, g2):
        assert torch.equal(a, b2)


def test_voxel_count_not_multiple_of_four(B):
    base = synth.make_workload("tiny")
    tel = dataclasses.replace(base.telescope.with_psf_lsf(), n_x=5, n_y=5, n_channels=base.telescope.n_channels | 1)
    assert (tel.n_x * tel.n_y * tel.n_channels) % 4 != 0
    sizes = [700, 1300, 90]
    gals, offsets, targets = make_case(sizes, 1300, tel)
    R = rotations(len(sizes), 5)
    loss, cubes, g, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R, targets)
    for b, gal in enumerate(gals):
        l1, g1, c1 = single(B, gal, base.ssp, tel, R[b], targets[b])
        assert torch.equal(cubes[b], c1), b
        assert abs(float(loss[b].item()) - float(l1.item())) <= 1e-13 * float(l1.item()), b   # fp64 sums in another order
        lo, hi = int(offsets[b]), int(offsets[b + 1])
        for q in range(4):
            assert torch.equal(g[q][lo:hi], g1[q]), (b, q)


def test_more_than_one_group(B):
    """70 elements: two launch sequences (64 + 6), the second one on offset particle arrays."""
    base = synth.make_workload("tiny")
    tel = base.telescope.with_psf_lsf()
    rng = np.random.default_rng(7)
    sizes = [int(s) for s in rng.integers(0, 400, size=70)]
    gals, offsets, targets = make_case(sizes, 2000, tel)
    R = rotations(len(sizes), 300)
    loss, cubes, g, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R, targets)
    for b in (0, 13, 63, 64, 69):
        if gals[b].n == 0:
            continue
        l1, g1, c1 = single(B, gals[b], base.ssp, tel, R[b], targets[b])
        assert torch.equal(cubes[b], c1) and float(loss[b].item()) == float(l1.item()), b
        lo, hi = int(offsets[b]), int(offsets[b + 1])
        for q in range(4):
            assert torch.equal(g[q][lo:hi], g1[q]), (b, q)


def test_against_oracle(B):
    base = synth.make_workload("tiny")
    tel = base.telescope.with_psf_lsf()
    sizes = [1500, 2200, 800]
    gals = [synth.make_particles_for("tiny", n=n, seed=3100 + i) for i, n in enumerate(sizes)]
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    R = rotations(len(sizes), 90)
    others = [synth.make_particles_for("tiny", n=n, seed=4100 + i) for i, n in enumerate(sizes)]
    target_np = np.stack([oracle.forward(o, R[b], base.ssp, tel) for b, o in enumerate(others)]).astype(np.float32)
    targets = torch.from_numpy(target_np).cuda()
    loss, cubes, g, _ = run_batched(B, concat(gals), offsets, len(sizes), base.ssp, tel, R, targets)
    for b, gal in enumerate(gals):
        ref = oracle.forward(gal, R[b], base.ssp, tel)
        got = cubes[b].cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-4 * ref.max()
        L_ref = float(((ref - target_np[b].astype(np.float64)) ** 2).sum())
        assert abs(float(loss[b].item()) - L_ref) <= 2e-4 * L_ref
        up = (2.0 * (got - target_np[b])).astype(np.float64)
        ana = oracle.adjoint(gal, R[b], base.ssp, tel, up)
        key, vlos = oracle.rotate_bin(gal.pos, gal.vel, R[b], tel.n_x, tel.n_y, tel.spaxel_size)
        lo, hi = int(offsets[b]), int(offsets[b + 1])
        assert_gradients([x[lo:hi].cpu().numpy() for x in g], ana, key, vlos, base.ssp, tel, f"element {b}")


def test_argument_checks(B):
    base = synth.make_workload("tiny", n=100)
    tel = base.telescope
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    p = base.particles
    arrays = [up(a) for a in (p.pos, p.vel, p.mass, p.log_age, p.log_z)]
    cp, cs, ct = B.c_particles(*arrays), B.c_ssp(base.ssp, up(base.ssp.flux)), B.c_telescope(tel)
    with pytest.raises(B.RubixError):
        B.rubix_loss_and_grad_batched_workspace_bytes(p.n, None, 2, cs, ct)      # needs offsets
    offsets = np.array([0, 40, 100], dtype=np.int64)
    need = B.rubix_loss_and_grad_batched_workspace_bytes(p.n, offsets, 2, cs, ct)
    ws = torch.empty(need - 256, dtype=torch.uint8, device="cuda")
    targets = torch.zeros((2, tel.n_x, tel.n_y, tel.n_channels), dtype=torch.float32, device="cuda")
    loss = torch.zeros(2, dtype=torch.float64, device="cuda")
    g = [torch.zeros(p.n, dtype=torch.float32, device="cuda") for _ in range(4)]
    with pytest.raises(B.RubixError) as e:
        B.rubix_loss_and_grad_batched(cp, offsets, 2, cs, ct, rotations(2, 1), targets, loss, None, *g, ws)
    assert e.value.status == B.RUBIX_ERR_WORKSPACE
