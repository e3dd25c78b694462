"""Thin ctypes binding of ``librubix_b200.so`` (include/rubix.h): argument marshalling only.

Same names as the C ABI.  PyTorch is used for device memory and streams and nothing else: every
step of the path runs in the library's kernels.  There is no fallback of any kind -- a missing
library raises at load time and a failing call raises ``RubixError`` with the library's message.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librubix_b200.so")

RUBIX_OK, RUBIX_ERR_NULL, RUBIX_ERR_INVALID_ARG, RUBIX_ERR_UNSUPPORTED, RUBIX_ERR_WORKSPACE, \
    RUBIX_ERR_CUDA = range(6)

EXPORTS = ("rubix_workspace_bytes", "rubix_build_cube", "rubix_convolve_psf_lsf", "rubix_forward",
           "rubix_cube_adjoint", "rubix_get_sort_artifacts", "rubix_forward_host_scratch_bytes",
           "rubix_forward_batched_workspace_bytes", "rubix_forward_batched", "rubix_bin_particles", "rubix_build_cube_mirrored",
           "rubix_loss_and_grad_batched_workspace_bytes", "rubix_loss_and_grad_batched",
           "rubix_forward_host", "rubix_last_launch_count", "rubix_last_error", "rubix_abi_version",
           "rubix_forward_host_pipelined_scratch_bytes", "rubix_forward_host_pipelined", "rubix_forward_host_drain",
           "rubix_loss_and_grad_workspace_bytes", "rubix_loss_and_grad", "rubix_add_noise",
           "rubix_residual_loss_static",
           # include/rubix_peaks.h (measurement helpers)
           "rubix_measure_peaks", "rubix_stage_timing_enable", "rubix_stage_timing_read")
ABI_VERSION = 9          # RUBIX_ABI_VERSION of include/rubix.h
N_STAGES = 5
STAGES = ("particle_pass", "accumulate", "reduce_partials", "psf_lsf", "adjoint")


class RubixError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"rubix status {status}: {message}")
        self.status = status


class CParticles(C.Structure):
    _fields_ = [("n", C.c_int64), ("pos", C.c_void_p), ("vel", C.c_void_p), ("mass", C.c_void_p),
                ("log_age", C.c_void_p), ("log_z", C.c_void_p)]


class CSSP(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_age", C.c_int32), ("n_z", C.c_int32), ("n_lambda", C.c_int32),
                ("log_age_axis", C.c_void_p), ("log_z_axis", C.c_void_p),
                ("lambda0", C.c_float), ("dlambda", C.c_float), ("flux", C.c_void_p),
                ("log_lambda", C.c_int32), ("lambda_grid", C.c_void_p)]


class CTelescope(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_x", C.c_int32), ("n_y", C.c_int32), ("spaxel_size", C.c_float),
                ("n_channels", C.c_int32), ("lambda0", C.c_float), ("dlambda", C.c_float),
                ("psf_size", C.c_int32), ("psf_sigma", C.c_float),
                ("lsf_size", C.c_int32), ("lsf_sigma", C.c_float), ("resample", C.c_int32),
                ("redshift", C.c_float), ("flux_scale", C.c_float), ("lambda_obs", C.c_void_p),
                ("psf_alpha", C.c_float), ("psf_lambda_ref", C.c_float), ("n_x_full", C.c_int32), ("x_first", C.c_int32),
                ("cell_order", C.c_int32), ("reserved0", C.c_int32)]


_lib = None


def load():
    """Loads the in-tree library (build it with ``python -m paper_2412_08265_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2412_08265_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.rubix_workspace_bytes.restype = C.c_size_t
        lib.rubix_workspace_bytes.argtypes = [C.c_int64, C.POINTER(CSSP), C.POINTER(CTelescope)]
        lib.rubix_forward_host_scratch_bytes.restype = C.c_size_t
        lib.rubix_forward_host_scratch_bytes.argtypes = [C.c_int64, C.POINTER(CSSP), C.POINTER(CTelescope)]
        lib.rubix_build_cube.restype = C.c_int
        lib.rubix_build_cube.argtypes = [C.POINTER(CParticles), C.POINTER(CSSP), C.POINTER(CTelescope),
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.rubix_forward.restype = C.c_int
        lib.rubix_forward.argtypes = lib.rubix_build_cube.argtypes
        lib.rubix_forward_batched_workspace_bytes.restype = C.c_size_t
        lib.rubix_forward_batched_workspace_bytes.argtypes = [C.c_int64, C.c_void_p, C.c_int32, C.POINTER(CSSP),
                                                              C.POINTER(CTelescope)]
        lib.rubix_forward_batched.restype = C.c_int
        lib.rubix_forward_batched.argtypes = [C.POINTER(CParticles), C.c_void_p, C.c_int32, C.POINTER(CSSP),
                                              C.POINTER(CTelescope), C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t,
                                              C.c_void_p]
        lib.rubix_loss_and_grad_batched_workspace_bytes.restype = C.c_size_t
        lib.rubix_loss_and_grad_batched_workspace_bytes.argtypes = lib.rubix_forward_batched_workspace_bytes.argtypes
        lib.rubix_loss_and_grad_batched.restype = C.c_int
        lib.rubix_loss_and_grad_batched.argtypes = [C.POINTER(CParticles), C.c_void_p, C.c_int32, C.POINTER(CSSP),
                                                    C.POINTER(CTelescope)] + [C.c_void_p] * 9 + [C.c_size_t, C.c_void_p]
        lib.rubix_build_cube_mirrored.restype = C.c_int
        lib.rubix_build_cube_mirrored.argtypes = [C.POINTER(CParticles), C.POINTER(CSSP), C.POINTER(CTelescope), C.c_void_p,
                                                  C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.rubix_bin_particles.restype = C.c_int
        lib.rubix_bin_particles.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(CTelescope), C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p]
        lib.rubix_convolve_psf_lsf.restype = C.c_int
        lib.rubix_convolve_psf_lsf.argtypes = [C.POINTER(CTelescope), C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_size_t, C.c_void_p]
        lib.rubix_cube_adjoint.restype = C.c_int
        lib.rubix_cube_adjoint.argtypes = [C.POINTER(CParticles), C.POINTER(CSSP), C.POINTER(CTelescope),
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.rubix_loss_and_grad_workspace_bytes.restype = C.c_size_t
        lib.rubix_loss_and_grad_workspace_bytes.argtypes = [C.c_int64, C.POINTER(CSSP), C.POINTER(CTelescope)]
        lib.rubix_loss_and_grad.restype = C.c_int
        lib.rubix_loss_and_grad.argtypes = [C.POINTER(CParticles), C.POINTER(CSSP), C.POINTER(CTelescope),
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t,
                                            C.c_void_p]
        lib.rubix_residual_loss_static.restype = C.c_int
        lib.rubix_residual_loss_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.rubix_add_noise.restype = C.c_int
        lib.rubix_add_noise.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_float, C.c_uint64, C.c_void_p]
        lib.rubix_get_sort_artifacts.restype = C.c_int
        lib.rubix_get_sort_artifacts.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                                 C.POINTER(C.c_void_p)]
        lib.rubix_forward_host.restype = C.c_int
        lib.rubix_forward_host.argtypes = [C.POINTER(CParticles), C.POINTER(CSSP), C.POINTER(CTelescope),
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.rubix_forward_host_pipelined_scratch_bytes.restype = C.c_size_t
        lib.rubix_forward_host_pipelined_scratch_bytes.argtypes = [C.c_int64, C.POINTER(CSSP), C.POINTER(CTelescope)]
        lib.rubix_forward_host_pipelined.restype = C.c_int
        lib.rubix_forward_host_pipelined.argtypes = lib.rubix_forward_host.argtypes
        lib.rubix_forward_host_drain.restype = C.c_int
        lib.rubix_forward_host_drain.argtypes = [C.c_void_p]
        lib.rubix_measure_peaks.restype = C.c_int32
        lib.rubix_measure_peaks.argtypes = [C.POINTER(C.c_float), C.c_void_p, C.c_size_t, C.c_void_p]
        lib.rubix_stage_timing_enable.restype = None
        lib.rubix_stage_timing_enable.argtypes = [C.c_int32]
        lib.rubix_stage_timing_read.restype = C.c_int32
        lib.rubix_stage_timing_read.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_int32)]
        lib.rubix_last_launch_count.restype = C.c_int32
        lib.rubix_abi_version.restype = C.c_uint32
        if int(lib.rubix_abi_version()) != ABI_VERSION:
            raise RuntimeError(f"{LIB_PATH} has ABI version {int(lib.rubix_abi_version())}, this binding expects "
                               f"{ABI_VERSION}: rebuild with `python -m paper_2412_08265_b200.build --force`")
        lib.rubix_last_error.restype = C.c_char_p
        _lib = lib
    return _lib


def rubix_last_error() -> str:
    return load().rubix_last_error().decode()


def rubix_last_launch_count() -> int:
    return int(load().rubix_last_launch_count())


def _check(status):
    if status != RUBIX_OK:
        raise RubixError(status, rubix_last_error())


def _ptr(t):
    """Address of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _host_f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


class _Keep:
    """ctypes struct plus the host arrays it points to (kept alive for the call)."""

    def __init__(self, struct, *refs):
        self.struct, self.refs = struct, refs

    def ref(self):
        return C.byref(self.struct)


def c_telescope(tel) -> _Keep:
    lam = getattr(tel, "lambda_obs", None)
    lam = None if lam is None else np.ascontiguousarray(lam, dtype=np.float32)
    return _Keep(CTelescope(C.sizeof(CTelescope), int(tel.n_x), int(tel.n_y), float(tel.spaxel_size), int(tel.n_channels),
                            float(tel.lambda0), float(tel.dlambda), int(tel.psf_size),
                            float(tel.psf_sigma), int(tel.lsf_size), float(tel.lsf_sigma),
                            int(getattr(tel, "resample", 0)), float(getattr(tel, "redshift", 0.0)),
                            float(getattr(tel, "flux_scale", 1.0)),
                            None if lam is None else lam.ctypes.data, float(getattr(tel, "psf_alpha", 0.0)),
                            float(getattr(tel, "psf_lambda_ref", 1.0)), int(getattr(tel, "n_x_full", 0)),
                            int(getattr(tel, "x_first", 0)), int(getattr(tel, "cell_order", 0)), 0), lam)


def c_ssp(ssp, flux) -> _Keep:
    """``ssp``: object with log_age_axis, log_z_axis (host), lambda0, dlambda; ``flux``: the
    [n_age, n_z, n_lambda] array the struct should point to (device tensor, or host array for
    rubix_forward_host)."""
    age, zed = _host_f32(ssp.log_age_axis), _host_f32(ssp.log_z_axis)
    n_age, n_z, n_lambda = (int(v) for v in flux.shape)
    grid = getattr(ssp, "lambda_grid", None)
    grid = None if grid is None else _host_f32(grid)
    return _Keep(CSSP(C.sizeof(CSSP), n_age, n_z, n_lambda, age.ctypes.data, zed.ctypes.data, float(ssp.lambda0),
                      float(ssp.dlambda), _ptr(flux), int(getattr(ssp, "log_lambda", 0)),
                      None if grid is None else grid.ctypes.data), age, zed, flux, grid)


def c_particles(pos, vel, mass, log_age, log_z) -> _Keep:
    return _Keep(CParticles(int(mass.shape[0]), _ptr(pos), _ptr(vel), _ptr(mass), _ptr(log_age),
                            _ptr(log_z)), pos, vel, mass, log_age, log_z)


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


# ------------------------------------------------------------------------------ the C ABI
def rubix_workspace_bytes(n, ssp: _Keep, tel: _Keep) -> int:
    b = int(load().rubix_workspace_bytes(int(n), ssp.ref() if ssp is not None else None, tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_build_cube(particles: _Keep, ssp: _Keep, tel: _Keep, R, cube, workspace, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_build_cube(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(cube),
                                   _ptr(workspace), int(workspace.numel() * workspace.element_size()),
                                   _stream(stream)))


def rubix_forward(particles: _Keep, ssp: _Keep, tel: _Keep, R, cube, workspace, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_forward(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(cube),
                                _ptr(workspace), int(workspace.numel() * workspace.element_size()),
                                _stream(stream)))


def rubix_loss_and_grad_batched_workspace_bytes(n, offsets, batch, ssp: _Keep, tel: _Keep) -> int:
    off = _offsets(offsets)
    b = int(load().rubix_loss_and_grad_batched_workspace_bytes(int(n), _ptr(off), int(batch), ssp.ref(), tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_loss_and_grad_batched(particles: _Keep, offsets, batch, ssp: _Keep, tel: _Keep, R, targets, loss, cubes_out, g_mass,
                                g_log_age, g_log_z, g_vlos, workspace, stream=None):
    """``loss``: float64 device tensor [batch]; ``cubes_out``: device tensor [batch, n_x, n_y, n_channels] or None."""
    off = _offsets(offsets)
    R = _host_f32(R).reshape(-1)
    assert R.size == 9 * int(batch)
    _check(load().rubix_loss_and_grad_batched(particles.ref(), _ptr(off), int(batch), ssp.ref(), tel.ref(), R.ctypes.data,
                                              _ptr(targets), _ptr(loss), _ptr(cubes_out), _ptr(g_mass), _ptr(g_log_age),
                                              _ptr(g_log_z), _ptr(g_vlos), _ptr(workspace),
                                              int(workspace.numel() * workspace.element_size()), _stream(stream)))


def rubix_build_cube_mirrored(particles: _Keep, ssp: _Keep, tel: _Keep, R, cube, mirror_lo, mirror_hi, mirror_rows, workspace,
                              stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_build_cube_mirrored(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(cube), _ptr(mirror_lo),
                                            _ptr(mirror_hi), int(mirror_rows), _ptr(workspace),
                                            int(workspace.numel() * workspace.element_size()), _stream(stream)))


def rubix_bin_particles(pos, vel, tel: _Keep, R, key, vlos=None, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_bin_particles(int(pos.shape[0]), _ptr(pos), _ptr(vel), tel.ref(), R.ctypes.data, _ptr(key), _ptr(vlos),
                                      _stream(stream)))


def _offsets(offsets):
    return None if offsets is None else np.ascontiguousarray(offsets, dtype=np.int64)


def rubix_forward_batched_workspace_bytes(n, offsets, batch, ssp: _Keep, tel: _Keep) -> int:
    off = _offsets(offsets)
    b = int(load().rubix_forward_batched_workspace_bytes(int(n), _ptr(off), int(batch), ssp.ref(), tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_forward_batched(particles: _Keep, offsets, batch, ssp: _Keep, tel: _Keep, R, cubes, workspace, stream=None):
    """``offsets``: int64 host array [batch + 1] (concatenated galaxies) or None (one galaxy, ``batch`` rotations);
    ``R``: [batch, 3, 3]; ``cubes``: device tensor [batch, n_x, n_y, n_channels]."""
    off = _offsets(offsets)
    R = _host_f32(R).reshape(-1)
    assert R.size == 9 * int(batch)
    _check(load().rubix_forward_batched(particles.ref(), _ptr(off), int(batch), ssp.ref(), tel.ref(), R.ctypes.data,
                                        _ptr(cubes), _ptr(workspace),
                                        int(workspace.numel() * workspace.element_size()), _stream(stream)))


def rubix_convolve_psf_lsf(tel: _Keep, cube_in, cube_out, workspace, stream=None):
    nbytes = 0 if workspace is None else int(workspace.numel() * workspace.element_size())
    _check(load().rubix_convolve_psf_lsf(tel.ref(), _ptr(cube_in), _ptr(cube_out), _ptr(workspace),
                                         nbytes, _stream(stream)))


def rubix_cube_adjoint(particles: _Keep, ssp: _Keep, tel: _Keep, R, grad_cube, g_mass, g_log_age,
                       g_log_z, g_vlos, workspace, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_cube_adjoint(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data,
                                     _ptr(grad_cube), _ptr(g_mass), _ptr(g_log_age), _ptr(g_log_z),
                                     _ptr(g_vlos), _ptr(workspace),
                                     int(workspace.numel() * workspace.element_size()), _stream(stream)))


def rubix_loss_and_grad_workspace_bytes(n, ssp: _Keep, tel: _Keep) -> int:
    b = int(load().rubix_loss_and_grad_workspace_bytes(int(n), ssp.ref(), tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_loss_and_grad(particles: _Keep, ssp: _Keep, tel: _Keep, R, target, loss, cube_out, g_mass,
                        g_log_age, g_log_z, g_vlos, workspace, stream=None):
    """``loss``: one-element float64 device tensor; ``cube_out``: device tensor or None."""
    R = _host_f32(R).reshape(9)
    _check(load().rubix_loss_and_grad(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(target),
                                      _ptr(loss), _ptr(cube_out), _ptr(g_mass), _ptr(g_log_age),
                                      _ptr(g_log_z), _ptr(g_vlos), _ptr(workspace),
                                      int(workspace.numel() * workspace.element_size()), _stream(stream)))


RESIDUAL_LOSS_STATIC_MAX_BATCH = 64      # RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH of include/rubix.h


def rubix_residual_loss_static(cubes, targets, grads, loss, batch=1, stream=None):
    """grads = 2 (cubes - targets), loss[b] = sum (cubes[b] - targets[b])^2; no workspace, no allocation (batch <= 64)."""
    n_vox = int(cubes.numel()) // int(batch)
    assert int(cubes.numel()) == n_vox * int(batch) == int(targets.numel()) == int(grads.numel())
    _check(load().rubix_residual_loss_static(_ptr(cubes), _ptr(targets), n_vox, int(batch), _ptr(grads), _ptr(loss),
                                             _stream(stream)))


def rubix_add_noise(cube_in, cube_out, sigma_read, gain, seed, stream=None):
    _check(load().rubix_add_noise(_ptr(cube_in), _ptr(cube_out), int(cube_in.numel()), float(sigma_read), float(gain),
                                  int(seed) & 0xFFFFFFFFFFFFFFFF, _stream(stream)))


def rubix_get_sort_artifacts(workspace, n, n_s):
    """(key[n], perm[n], seg_off[n_s+2]) as int32 torch tensors copied out of the workspace."""
    import torch
    k, p, s = C.c_void_p(), C.c_void_p(), C.c_void_p()
    _check(load().rubix_get_sort_artifacts(_ptr(workspace), C.byref(k), C.byref(p), C.byref(s)))
    base = workspace.data_ptr()
    flat = workspace.view(torch.uint8)

    def view(addr, count):
        off = addr - base
        return flat[off:off + 4 * count].view(torch.int32).clone()

    return view(k.value, n), view(p.value, n), view(s.value, n_s + 2)


def rubix_forward_host_scratch_bytes(n, ssp: _Keep, tel: _Keep) -> int:
    b = int(load().rubix_forward_host_scratch_bytes(int(n), ssp.ref(), tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_forward_host(particles: _Keep, ssp: _Keep, tel: _Keep, R, h_cube, scratch, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_forward_host(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(h_cube),
                                     _ptr(scratch), int(scratch.numel() * scratch.element_size()),
                                     _stream(stream)))


def rubix_forward_host_pipelined_scratch_bytes(n, ssp: _Keep, tel: _Keep) -> int:
    b = int(load().rubix_forward_host_pipelined_scratch_bytes(int(n), ssp.ref(), tel.ref()))
    if b == 0:
        raise RubixError(RUBIX_ERR_INVALID_ARG, rubix_last_error())
    return b


def rubix_forward_host_pipelined(particles: _Keep, ssp: _Keep, tel: _Keep, R, h_cube, scratch, stream=None):
    R = _host_f32(R).reshape(9)
    _check(load().rubix_forward_host_pipelined(particles.ref(), ssp.ref(), tel.ref(), R.ctypes.data, _ptr(h_cube),
                                               _ptr(scratch), int(scratch.numel() * scratch.element_size()),
                                               _stream(stream)))


def rubix_forward_host_drain(stream=None):
    _check(load().rubix_forward_host_drain(_stream(stream)))


# ------------------------------------------------------------------------------ rubix_peaks.h
def rubix_measure_peaks(scratch, stream=None) -> dict:
    out = (C.c_float * 4)()
    _check(load().rubix_measure_peaks(out, _ptr(scratch), int(scratch.numel() * scratch.element_size()),
                                      _stream(stream)))
    return {"l2_gbs": out[0], "smem_gbs": out[1], "fma_tflops": out[2], "hbm_copy_gbs": out[3]}


def rubix_stage_timing_enable(on: bool):
    load().rubix_stage_timing_enable(1 if on else 0)


def rubix_stage_timing_read() -> dict:
    ms = (C.c_float * N_STAGES)()
    calls = (C.c_int32 * N_STAGES)()
    _check(load().rubix_stage_timing_read(ms, calls))
    return {name: {"ms": float(ms[i]), "calls": int(calls[i])} for i, name in enumerate(STAGES)}


# ------------------------------------------------------------------------------ conveniences
class DeviceWorkload:
    """A synth.Workload uploaded to the GPU, with the marshalled structs and a workspace."""

    def __init__(self, w, device="cuda:0", adjoint=False):
        import torch
        self.w = w
        self.device = torch.device(device)
        p = w.particles
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(self.device)
        self.pos, self.vel, self.mass = up(p.pos), up(p.vel), up(p.mass)
        self.log_age, self.log_z = up(p.log_age), up(p.log_z)
        self.flux = up(w.ssp.flux)
        self.particles = c_particles(self.pos, self.vel, self.mass, self.log_age, self.log_z)
        self.ssp = c_ssp(w.ssp, self.flux)
        self.tel = c_telescope(w.telescope)
        self.R = _host_f32(w.rotation)
        t = w.telescope
        self.shape = (t.n_x, t.n_y, t.n_channels)
        self.workspace = torch.empty(rubix_workspace_bytes(p.n, self.ssp, self.tel), dtype=torch.uint8,
                                     device=self.device)

    def build_cube(self, out=None):
        import torch
        cube = torch.empty(self.shape, dtype=torch.float32, device=self.device) if out is None else out
        rubix_build_cube(self.particles, self.ssp, self.tel, self.R, cube, self.workspace)
        return cube

    def convolve(self, cube, out=None):
        import torch
        res = torch.empty(self.shape, dtype=torch.float32, device=self.device) if out is None else out
        rubix_convolve_psf_lsf(self.tel, cube, res, self.workspace)
        return res

    def forward(self, out=None):
        """Steps 1-8 through the fused device call rubix_forward."""
        import torch
        cube = torch.empty(self.shape, dtype=torch.float32, device=self.device) if out is None else out
        rubix_forward(self.particles, self.ssp, self.tel, self.R, cube, self.workspace)
        return cube

    def forward_two_calls(self):
        cube = self.build_cube()
        t = self.w.telescope
        return self.convolve(cube) if (t.psf_size > 0 or t.lsf_size > 0) else cube

    def adjoint(self, grad_cube):
        import torch
        n = self.w.particles.n
        g = [torch.empty(n, dtype=torch.float32, device=self.device) for _ in range(4)]
        rubix_cube_adjoint(self.particles, self.ssp, self.tel, self.R, grad_cube, *g, self.workspace)
        return g

    def loss_and_grad(self, target, want_cube=False):
        """(loss [1] float64, (g_mass, g_log_age, g_log_z, g_vlos), final cube or None) in one fused call."""
        import torch
        n = self.w.particles.n
        need = rubix_loss_and_grad_workspace_bytes(n, self.ssp, self.tel)
        if self.workspace.numel() < need:
            self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
        loss = torch.zeros(1, dtype=torch.float64, device=self.device)
        cube = torch.empty(self.shape, dtype=torch.float32, device=self.device) if want_cube else None
        g = [torch.empty(n, dtype=torch.float32, device=self.device) for _ in range(4)]
        rubix_loss_and_grad(self.particles, self.ssp, self.tel, self.R, target, loss, cube, *g, self.workspace)
        return loss, g, cube

    def sort_artifacts(self):
        t = self.w.telescope
        return rubix_get_sort_artifacts(self.workspace, self.w.particles.n, t.n_x * t.n_y)
