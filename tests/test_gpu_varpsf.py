"""Parity of the CUDA path with a WAVELENGTH-DEPENDENT PSF (reading R18) against
the fp64 oracle: standalone convolution, the whole forward path, and the adjoint (true transpose order)."""
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


def var(tel, alpha=-0.3, ref=6500.0):
    return dataclasses.replace(tel, psf_alpha=np.float32(alpha), psf_lambda_ref=np.float32(ref))


@pytest.mark.parametrize("shape,psf,lsf,alpha", [((19, 22, 38), 15, 9, -0.2), ((8, 5, 64), 15, 9, 1.5), ((30, 30, 100), 11, 0, -0.5),
                                                 ((12, 40, 130), 15, 5, -0.2), ((1, 1, 2), 3, 3, 0.7)])
def test_convolve_small_cubes(B, shape, psf, lsf, alpha):
    n_x, n_y, n_c = shape
    t = synth.Telescope(n_x, n_y, np.float32(1.0), n_c, np.float32(4800.0), np.float32(30.0), psf, np.float32(1.4),
                        lsf, np.float32(1.7 if lsf else 0.0))
    t = var(t, alpha)
    cube = synth.synthetic_cube(n_x, n_y, n_c, seed=11)
    tel = B.c_telescope(t)
    d_in = torch.from_numpy(cube).cuda()
    d_out = torch.full_like(d_in, float("nan"))
    ws = torch.empty(cube.nbytes + (1 << 20), dtype=torch.uint8, device="cuda")
    B.rubix_convolve_psf_lsf(tel, d_in, d_out, ws)
    ref = oracle.convolve(cube.astype(np.float64), psf, t.psf_sigma, lsf, t.lsf_sigma, oracle.psf_sigma_k(t))
    assert np.abs(d_out.cpu().numpy() - ref).max() <= 1e-4 * ref.max()
    const = oracle.convolve(cube.astype(np.float64), psf, t.psf_sigma, lsf, t.lsf_sigma)
    if n_c > 2:
        assert np.abs(ref - const).max() > 10 * np.abs(d_out.cpu().numpy() - ref).max()   # the law really is applied


def test_forward_and_adjoint_on_config4(B):
    w = synth.make_workload("adjoint", n=20000)
    w.telescope = var(w.telescope, -0.2, 7000.0)
    t = w.telescope
    dw = B.DeviceWorkload(w)
    final = dw.forward().cpu().numpy()
    ref_final = oracle.forward(w.particles, w.rotation, w.ssp, t)
    assert np.abs(final - ref_final).max() <= 1e-4 * ref_final.max()
    G = upstream_gradient(w)                               # 2 (cube - target) of two galaxies, as in configs[4]
    g = [x.cpu().numpy().astype(np.float64) for x in dw.adjoint(torch.from_numpy(G).cuda())]
    ana = oracle.adjoint(w.particles, w.rotation, w.ssp, t, G.astype(np.float64))
    key, vlos = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert_gradients(g, ana, key, vlos, w.ssp, t, "test_gpu_varpsf.py")
    # the wrong operator order (forward instead of transpose) would show: compare with the constant-PSF gradient
    ana0 = oracle.adjoint(w.particles, w.rotation, w.ssp, dataclasses.replace(t, psf_alpha=np.float32(0.0)), G.astype(np.float64))
    assert np.abs(ana0[0] - ana[0]).max() > 100 * np.quantile(np.abs(g[0] - ana[0]), 0.999)
    # fused call: loss and gradients through the same operators
    other = synth.make_particles_for("adjoint", n=20000, seed=synth.ADJOINT_TARGET_SEED)
    target = oracle.forward(other, w.rotation, w.ssp, t).astype(np.float32)
    loss, g2, cube2 = dw.loss_and_grad(torch.from_numpy(target).cuda(), want_cube=True)
    resid = ref_final - target.astype(np.float64)
    assert abs(float(loss.item()) - float((resid ** 2).sum())) <= 2e-4 * float((resid ** 2).sum())
    # gradients against the oracle's adjoint of the upstream gradient the call formed (reading R19)
    up = (2.0 * (cube2.cpu().numpy() - target)).astype(np.float64)
    ana2 = oracle.adjoint(w.particles, w.rotation, w.ssp, t, up)
    assert_gradients([x.cpu().numpy() for x in g2], ana2, key, vlos, w.ssp, t, "fused call, lambda-dependent PSF")


def test_unsupported_and_invalid_combinations(B):
    w = synth.make_workload("tiny")
    base = w.telescope.with_psf_lsf()
    for t, msg in ((var(dataclasses.replace(base, psf_size=21)), "psf_size <= 15"),
                   (var(dataclasses.replace(base, n_channels=255)), "even n_channels"),
                   (var(base, ref=0.0), "psf_lambda_ref")):
        w2 = dataclasses.replace(w, telescope=t)
        with pytest.raises(B.RubixError):
            B.DeviceWorkload(w2).forward()
        assert msg in B.rubix_last_error(), B.rubix_last_error()


def test_convolve_on_a_tiny_detector_keeps_the_sort_artefacts(B):
    """The per-channel taps (15 x (n_c + 2) floats) are larger than a cube of fewer than 15 spaxels: they must not land on
    the sort artefacts that rubix_build_cube left in the shared workspace (found by the r02 fuzz run, seed 118)."""
    w = synth.make_workload("tiny", n=200)
    w.telescope = dataclasses.replace(synth.Telescope(2, 3, np.float32(6.0), 88, np.float32(4700.0), np.float32(50.0)).with_psf_lsf(lsf_size=0),
                                      psf_alpha=np.float32(-0.2), psf_lambda_ref=np.float32(6000.0))
    dw = B.DeviceWorkload(w)
    cube = dw.build_cube()
    before = [a.clone() for a in dw.sort_artifacts()]
    final = dw.convolve(cube)
    torch.cuda.synchronize()
    for a, b in zip(before, dw.sort_artifacts()):
        assert torch.equal(a, b)
    t = w.telescope
    ref = oracle.convolve(oracle.build_cube(w.particles, w.rotation, w.ssp, t), t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma,
                          oracle.psf_sigma_k(t))
    assert np.abs(final.cpu().numpy() - ref).max() <= 1e-4 * ref.max()
