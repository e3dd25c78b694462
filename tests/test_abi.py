"""The C-ABI library: it builds, loads without a GPU, exports every symbol include/rubix.h
declares, and validates its arguments on the host before any launch.
No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2412_08265_b200 import binding as B
from paper_2412_08265_b200 import build as builder
from paper_2412_08265_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE = 0x10000          # non-NULL, 256-byte aligned "device" address that is never dereferenced


@pytest.fixture(scope="module")
def lib():
    builder.build()
    return B.load()


def test_every_declared_symbol_is_exported(lib):
    import glob
    header = "".join(open(h).read() for h in sorted(glob.glob(os.path.join(ROOT, "include", "*.h"))))
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(rubix_[a-z_]+)\s*\(", header))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_struct_layouts_match_the_header():
    assert C.sizeof(B.CParticles) == 48 and C.sizeof(B.CSSP) == 64 and C.sizeof(B.CTelescope) == 88


def test_abi_version_and_struct_size_are_checked(lib):
    """A caller built against another rubix.h (other struct size, or the pre-struct_size layout, whose first field was a
    small count) is refused before anything is read from the struct."""
    header = open(os.path.join(ROOT, "include", "rubix.h")).read()
    assert int(re.search(r"#define RUBIX_ABI_VERSION (\d+)", header).group(1)) == B.ABI_VERSION == lib.rubix_abi_version()
    P = _fake_particles()
    for which in ("ssp", "tel"):
        for bad in (0, 50, 300, C.sizeof(B.CSSP if which == "ssp" else B.CTelescope) + 8):
            ssp, tel = _structs()
            (ssp if which == "ssp" else tel).struct.struct_size = bad
            assert _call_build(lib, P, ssp, tel) == B.RUBIX_ERR_INVALID_ARG
            assert "struct_size" in B.rubix_last_error()
            assert lib.rubix_workspace_bytes(10, ssp.ref(), tel.ref()) == 0
            assert lib.rubix_forward_host_scratch_bytes(10, ssp.ref(), tel.ref()) == 0
            assert lib.rubix_forward(P.ref(), ssp.ref(), tel.ref(), np.eye(3, dtype=np.float32).ctypes.data, FAKE, FAKE,
                                     1 << 40, None) == B.RUBIX_ERR_INVALID_ARG
            if which == "tel":                             # (never reaches a launch: the addresses are fake)
                assert lib.rubix_convolve_psf_lsf(tel.ref(), FAKE, FAKE + (1 << 33), FAKE + (1 << 34), 1 << 40,
                                                  None) == B.RUBIX_ERR_INVALID_ARG


def _structs(tel=None, ssp=None):
    tel = tel or synth.make_telescope("medium")
    ssp = ssp or synth.make_ssp(8, 4, 512, 3500.0, 9500.0, 1)
    fake_flux = np.empty((ssp.flux.shape), np.float32)
    return B.c_ssp(ssp, fake_flux), B.c_telescope(tel)


def test_workspace_bytes(lib):
    ssp, tel = _structs()
    small = B.rubix_workspace_bytes(0, ssp, tel)
    big = B.rubix_workspace_bytes(1_000_000, ssp, tel)
    cube = 300 * 300 * 3700 * 4
    assert small >= 2 * cube and big > small and big < small + 1_000_000 * 120 + (1 << 28)
    with pytest.raises(B.RubixError):
        B.rubix_workspace_bytes(-1, ssp, tel)
    assert "n out of range" in B.rubix_last_error()


def _call_build(lib, particles, ssp, tel, R=None, cube=FAKE, ws=FAKE, ws_bytes=1 << 40):
    R = np.eye(3, dtype=np.float32).reshape(9) if R is None else R
    return lib.rubix_build_cube(particles.ref() if particles else None, ssp.ref() if ssp else None,
                                tel.ref() if tel else None, R.ctypes.data if R is not False else None,
                                cube, ws, ws_bytes, None)


def _fake_particles(n=10):
    class T:  # minimal stand-in with data_ptr/shape
        def __init__(self, shape): self.shape = shape
        def data_ptr(self): return FAKE
    return B.c_particles(T((n, 3)), T((n, 3)), T((n,)), T((n,)), T((n,)))


def test_argument_validation_happens_before_any_launch(lib):
    ssp, tel = _structs()
    P = _fake_particles()
    assert _call_build(lib, None, ssp, tel) == B.RUBIX_ERR_NULL
    assert _call_build(lib, P, None, tel) == B.RUBIX_ERR_NULL
    assert _call_build(lib, P, ssp, None) == B.RUBIX_ERR_NULL
    assert _call_build(lib, P, ssp, tel, R=False) == B.RUBIX_ERR_NULL
    assert _call_build(lib, P, ssp, tel, cube=None) == B.RUBIX_ERR_NULL
    assert _call_build(lib, P, ssp, tel, ws=None) == B.RUBIX_ERR_WORKSPACE
    assert _call_build(lib, P, ssp, tel, ws=FAKE + 8) == B.RUBIX_ERR_WORKSPACE          # misaligned
    assert _call_build(lib, P, ssp, tel, ws_bytes=1024) == B.RUBIX_ERR_WORKSPACE
    assert "needs" in B.rubix_last_error()
    neg = _fake_particles()
    neg.struct.n = -5
    assert _call_build(lib, neg, ssp, tel) == B.RUBIX_ERR_INVALID_ARG
    nullarr = _fake_particles()
    nullarr.struct.mass = None
    assert _call_build(lib, nullarr, ssp, tel) == B.RUBIX_ERR_NULL


@pytest.mark.parametrize("field,value,status", [
    ("psf_size", 14, B.RUBIX_ERR_INVALID_ARG), ("lsf_size", -1, B.RUBIX_ERR_INVALID_ARG),
    ("psf_size", 65, B.RUBIX_ERR_UNSUPPORTED), ("psf_sigma", 0.0, B.RUBIX_ERR_INVALID_ARG),
    ("dlambda", 0.0, B.RUBIX_ERR_INVALID_ARG), ("dlambda", float("nan"), B.RUBIX_ERR_INVALID_ARG),
    ("spaxel_size", -1.0, B.RUBIX_ERR_INVALID_ARG), ("n_x", 0, B.RUBIX_ERR_INVALID_ARG),
    ("n_channels", 0, B.RUBIX_ERR_INVALID_ARG), ("dlambda", 400.0, B.RUBIX_ERR_UNSUPPORTED)])
def test_bad_telescope(lib, field, value, status):
    ssp, tel = _structs()
    setattr(tel.struct, field, value)
    assert _call_build(lib, _fake_particles(), ssp, tel) == status
    assert B.rubix_last_error() != ""


def test_bad_ssp(lib):
    P = _fake_particles()
    base = synth.make_ssp(8, 4, 512, 3500.0, 9500.0, 1)
    for mutate, status in [
        (lambda s: s.log_age_axis.__setitem__(3, s.log_age_axis[2]), B.RUBIX_ERR_INVALID_ARG),
        (lambda s: s.log_z_axis.__setitem__(slice(None), s.log_z_axis[::-1].copy()), B.RUBIX_ERR_INVALID_ARG),
        (lambda s: setattr(s, "dlambda", np.float32(-1.0)), B.RUBIX_ERR_INVALID_ARG)]:
        s = synth.SSPGrid(base.log_age_axis.copy(), base.log_z_axis.copy(), base.lambda0, base.dlambda, base.flux)
        mutate(s)
        ssp, tel = _structs(ssp=s)
        assert _call_build(lib, P, ssp, tel) == status
    ssp, tel = _structs()
    ssp.struct.n_age = 1
    assert _call_build(lib, P, ssp, tel) == B.RUBIX_ERR_INVALID_ARG
    ssp, tel = _structs()
    ssp.struct.n_age = 600
    assert _call_build(lib, P, ssp, tel) == B.RUBIX_ERR_UNSUPPORTED
    ssp, tel = _structs()
    ssp.struct.flux = None
    assert _call_build(lib, P, ssp, tel) == B.RUBIX_ERR_NULL


def test_convolve_and_adjoint_validation(lib):
    ssp, tel = _structs()
    cube_bytes = 300 * 300 * 3700 * 4
    f = lib.rubix_convolve_psf_lsf
    assert f(tel.ref(), None, FAKE, FAKE, 1 << 40, None) == B.RUBIX_ERR_NULL
    assert f(tel.ref(), FAKE, FAKE + 4096, FAKE, 1 << 40, None) == B.RUBIX_ERR_INVALID_ARG   # overlap
    assert f(tel.ref(), FAKE, FAKE + 2 * cube_bytes, FAKE, 16, None) == B.RUBIX_ERR_WORKSPACE
    g = lib.rubix_cube_adjoint
    R = np.eye(3, dtype=np.float32).reshape(9)
    P = _fake_particles()
    assert g(P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, None, FAKE, FAKE, FAKE, FAKE, FAKE, 1 << 40, None) \
        == B.RUBIX_ERR_NULL
    assert g(P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, FAKE, FAKE, None, FAKE, FAKE, FAKE, 1 << 40, None) \
        == B.RUBIX_ERR_NULL
    assert g(P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, FAKE, FAKE, FAKE, FAKE, FAKE, FAKE, 64, None) \
        == B.RUBIX_ERR_WORKSPACE
    k = C.c_void_p()
    assert lib.rubix_get_sort_artifacts(0x20000, C.byref(k), C.byref(k), C.byref(k)) == B.RUBIX_ERR_INVALID_ARG


def test_loss_and_grad_validation(lib):
    ssp, tel = _structs()
    P = _fake_particles()
    R = np.eye(3, dtype=np.float32).reshape(9)
    f = lib.rubix_loss_and_grad
    args = lambda target=FAKE, loss=FAKE, ws_bytes=1 << 40: (P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, target, loss,
                                                             None, FAKE, FAKE, FAKE, FAKE, FAKE, ws_bytes, None)
    assert f(*args(target=None)) == B.RUBIX_ERR_NULL
    assert f(*args(loss=None)) == B.RUBIX_ERR_NULL
    plain = B.rubix_workspace_bytes(10, ssp, tel)
    fused = B.rubix_loss_and_grad_workspace_bytes(10, ssp, tel)
    assert fused >= plain + 300 * 300 * 3700 * 4
    assert f(*args(ws_bytes=plain)) == B.RUBIX_ERR_WORKSPACE            # one cube-sized buffer short


def test_add_noise_validation(lib):
    f = lib.rubix_add_noise
    assert f(None, FAKE, 16, 1.0, 0.0, 1, None) == B.RUBIX_ERR_NULL
    assert f(FAKE, FAKE, -1, 1.0, 0.0, 1, None) == B.RUBIX_ERR_INVALID_ARG
    assert f(FAKE, FAKE, 16, -1.0, 0.0, 1, None) == B.RUBIX_ERR_INVALID_ARG
    assert f(FAKE, FAKE + 16, 16, 1.0, 0.0, 1, None) == B.RUBIX_ERR_INVALID_ARG      # partial overlap
    assert f(None, None, 0, 1.0, 0.0, 1, None) == B.RUBIX_OK                          # nothing to do


def test_workspace_bytes_never_decrease_with_n(lib):
    """A batched call carves the layouts of its smaller groups out of the workspace sized for the largest group: every
    buffer must be monotone in n, also where the sort switches to larger warp chunks (fewer histogram rows)."""
    ssp, tel = _structs(tel=synth.make_telescope("tiny"))
    prev = 0
    for n in [0, 1, 127, 128, 129, 1000, 100_000, 262_143, 262_144, 262_145, 300_000, 524_288, 524_289, 1_048_576, 1_048_577,
              2_097_152, 2_097_153, 4_194_304, 4_194_305, 10_000_000]:
        b = lib.rubix_workspace_bytes(n, ssp.ref(), tel.ref())
        assert b >= prev > -1, n
        prev = b
    rng = np.random.default_rng(0)
    for _ in range(300):
        a, c = sorted(int(v) for v in rng.integers(1, 6_000_000, size=2))
        assert lib.rubix_workspace_bytes(a, ssp.ref(), tel.ref()) <= lib.rubix_workspace_bytes(c, ssp.ref(), tel.ref()), (a, c)


def test_residual_loss_static_validation(lib):
    """The no-allocation loss entry refuses bad arguments, and batches beyond its static scratch, before any launch."""
    f = lib.rubix_residual_loss_static
    a, b, c, d = FAKE, FAKE + (1 << 30), FAKE + (2 << 30), FAKE + (3 << 30)
    assert f(a, b, 16, B.RESIDUAL_LOSS_STATIC_MAX_BATCH + 1, c, d, None) == B.RUBIX_ERR_UNSUPPORTED
    assert "exceeds" in B.rubix_last_error() and str(B.RESIDUAL_LOSS_STATIC_MAX_BATCH) in B.rubix_last_error()
    assert f(a, b, 16, 0, c, d, None) == B.RUBIX_ERR_INVALID_ARG
    assert f(a, b, -1, 1, c, d, None) == B.RUBIX_ERR_INVALID_ARG
    assert f(a, b, 16, 1, c, None, None) == B.RUBIX_ERR_NULL
    assert f(None, b, 16, 1, c, d, None) == B.RUBIX_ERR_NULL
    assert f(a, b, 16, 1, None, d, None) == B.RUBIX_ERR_NULL
    header = open(os.path.join(ROOT, "include", "rubix.h")).read()
    assert f"#define RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH {B.RESIDUAL_LOSS_STATIC_MAX_BATCH}" in header


def test_no_cpu_fallback_without_the_library(monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/librubix_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.load()


def test_batched_sharded_and_mirrored_entries_validate_on_the_host(lib):
    """rubix_forward_batched / rubix_bin_particles / rubix_build_cube_mirrored / the row window: bad arguments are refused
    before any launch (fake device addresses, no GPU needed)."""
    ssp, tel = _structs(tel=synth.make_telescope("tiny"))
    P = _fake_particles(100)
    R = np.tile(np.eye(3, dtype=np.float32).reshape(1, 9), (3, 1))

    def batched(offsets, batch, ws_bytes=1 << 40):
        off = None if offsets is None else np.asarray(offsets, np.int64)
        return lib.rubix_forward_batched(P.ref(), None if off is None else off.ctypes.data, batch, ssp.ref(), tel.ref(),
                                         R.ctypes.data, FAKE + (1 << 41), FAKE, ws_bytes, None)

    assert batched(None, 0) == B.RUBIX_ERR_INVALID_ARG and "batch" in B.rubix_last_error()
    assert batched([0, 50, 40, 100], 3) == B.RUBIX_ERR_INVALID_ARG and "non-decreasing" in B.rubix_last_error()
    assert batched([0, 50, 60, 99], 3) == B.RUBIX_ERR_INVALID_ARG
    assert batched([1, 50, 60, 100], 3) == B.RUBIX_ERR_INVALID_ARG
    assert batched([0, 50, 60, 100], 3, ws_bytes=1024) == B.RUBIX_ERR_WORKSPACE
    assert lib.rubix_forward_batched_workspace_bytes(100, None, 3, ssp.ref(), tel.ref()) > \
        lib.rubix_forward_batched_workspace_bytes(100, None, 1, ssp.ref(), tel.ref()) > 0
    assert lib.rubix_forward_batched_workspace_bytes(100, None, 0, ssp.ref(), tel.ref()) == 0
    # the fused forward + loss + adjoint of many galaxies: offsets are required, the same checks apply
    def lg_batched(offsets, batch, ws_bytes=1 << 40, loss=FAKE):
        off = None if offsets is None else np.asarray(offsets, np.int64)
        return lib.rubix_loss_and_grad_batched(P.ref(), None if off is None else off.ctypes.data, batch, ssp.ref(), tel.ref(),
                                               R.ctypes.data, FAKE + (1 << 41), loss, None, FAKE, FAKE, FAKE, FAKE,
                                               FAKE + (1 << 42), ws_bytes, None)

    assert lg_batched(None, 3) == B.RUBIX_ERR_INVALID_ARG and "offsets" in B.rubix_last_error()
    assert lg_batched([0, 50, 40, 100], 3) == B.RUBIX_ERR_INVALID_ARG
    assert lg_batched([0, 50, 60, 100], 3, loss=None) == B.RUBIX_ERR_NULL
    assert lg_batched([0, 50, 60, 100], 3, ws_bytes=1024) == B.RUBIX_ERR_WORKSPACE
    off3 = np.asarray([0, 50, 60, 100], np.int64)
    assert lib.rubix_loss_and_grad_batched_workspace_bytes(100, off3.ctypes.data, 3, ssp.ref(), tel.ref()) > \
        lib.rubix_forward_batched_workspace_bytes(100, off3.ctypes.data, 3, ssp.ref(), tel.ref())
    assert lib.rubix_loss_and_grad_batched_workspace_bytes(100, None, 3, ssp.ref(), tel.ref()) == 0
    # cell order: 0 .. 3
    _, t3 = _structs(tel=synth.make_telescope("tiny"))
    t3.struct.cell_order = 4
    assert lib.rubix_workspace_bytes(10, ssp.ref(), t3.ref()) == 0 and "cell_order" in B.rubix_last_error()
    # row window of a sharded run
    for n_x, n_full, first, ok in ((4, 16, 12, True), (4, 16, 13, False), (4, 0, 2, False), (4, 16, -1, False)):
        _, t2 = _structs(tel=synth.make_telescope("tiny"))
        t2.struct.n_x, t2.struct.n_x_full, t2.struct.x_first = n_x, n_full, first
        st = lib.rubix_workspace_bytes(10, ssp.ref(), t2.ref())
        assert (st > 0) == ok, (n_x, n_full, first)
    assert lib.rubix_bin_particles(10, None, FAKE, tel.ref(), R.ctypes.data, FAKE, None, None) == B.RUBIX_ERR_NULL
    assert lib.rubix_bin_particles(-1, FAKE, FAKE, tel.ref(), R.ctypes.data, FAKE, None, None) == B.RUBIX_ERR_INVALID_ARG
    assert lib.rubix_build_cube_mirrored(P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, FAKE + (1 << 41), FAKE + (1 << 42), None, 0,
                                         FAKE, 1 << 40, None) == B.RUBIX_ERR_INVALID_ARG
    assert lib.rubix_build_cube_mirrored(P.ref(), ssp.ref(), tel.ref(), R.ctypes.data, FAKE + (1 << 41), None, FAKE + (1 << 42), 17,
                                         FAKE, 1 << 40, None) == B.RUBIX_ERR_INVALID_ARG
    # listed SSP wavelengths: validated on the host like the axes
    base = synth.make_ssp(8, 4, 64, 3500.0, 9500.0, 1, irregular=True)
    bad = synth.SSPGrid(base.log_age_axis, base.log_z_axis, base.lambda0, base.dlambda, base.flux, 0, base.lambda_grid[::-1].copy())
    s_bad, _ = _structs(ssp=bad)
    assert _call_build(lib, P, s_bad, tel) == B.RUBIX_ERR_INVALID_ARG and "lambda_grid" in B.rubix_last_error()
