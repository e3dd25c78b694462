"""ctypes front end of the fp64 CPU oracle (oracle/rubix_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2412_08265_b200`` (the CUDA
path) -- inputs arrive as plain numpy arrays or as objects with the attribute names used below
(``pos vel mass log_age log_z``; ``log_age_axis log_z_axis lambda0 dlambda flux``;
``n_x n_y spaxel_size n_channels lambda0 dlambda psf_size psf_sigma lsf_size lsf_sigma``).

Every wrapper only marshals arguments; the arithmetic is in the C file, which cites
PAPER.md / SURVEY.md section 8(c) per function.  ``fd_gradients`` (central finite differences of
the oracle's own loss, SURVEY.md 8(c)-9 "Primary") is the one piece written in Python: it
calls the C spectrum and LSF routines and exploits linearity exactly as that row describes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rubix_oracle.c")
# RUBIX_ORACLE_SANITIZE=1: a second build with -fsanitize=address,undefined (the process must then
# be started with LD_PRELOAD=libasan, as tests/test_oracle_sanitizers.py does)
_SANITIZE = os.environ.get("RUBIX_ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "librubix_oracle_san.so" if _SANITIZE else "librubix_oracle.so")
_lock = threading.Lock()
_lib = None

C_KMS = 299792.458


def build(force: bool = False) -> str:
    """gcc -O2, fp contraction off (the fp32 binning must round every op), OpenMP."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-g", "-O1"] if _SANITIZE else ["-O2"]
        subprocess.check_call(["gcc"] + san + ["-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-ffp-contract=off", "-fno-fast-math", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            build()
            _lib = C.CDLL(_LIB)
    return _lib


def n_threads() -> int:
    """Threads the OpenMP loops will use (OMP_NUM_THREADS or all cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    return int(env) if env else (os.cpu_count() or 1)


def _mode(tel, ssp):
    """bit 0: resampling rule (0 point-sampled, 1 bin average); bit 1: log-sampled SSP grid (R15);
    bit 2: listed SSP wavelengths (R21, ``ssp.lambda_grid``)."""
    resample, log_grid = int(getattr(tel, "resample", 0)), int(getattr(ssp, "log_lambda", 0))
    listed = getattr(ssp, "lambda_grid", None) is not None
    if listed and log_grid:
        raise ValueError("an SSP grid is either log-sampled or listed, not both")
    return resample | (log_grid << 1) | (4 if listed else 0)


class _grids:
    """Installs tel.lambda_obs (explicit observed wavelengths, reading R16) and ssp.lambda_grid (listed SSP
    wavelengths, reading R21) in the C oracle for one call."""

    def __init__(self, tel, ssp=None):
        arr = getattr(tel, "lambda_obs", None)
        self.arr = None if arr is None else np.ascontiguousarray(arr, dtype=np.float32)
        self.zp1 = 1.0 + float(getattr(tel, "redshift", 0.0))
        if self.arr is not None and int(getattr(tel, "resample", 0)) != 0 and self.arr.size < 2:
            raise ValueError("the bin average on listed channel wavelengths needs at least two channels")
        grid = None if ssp is None else getattr(ssp, "lambda_grid", None)
        self.grid = None if grid is None else np.ascontiguousarray(grid, dtype=np.float32)

    def __enter__(self):
        if self.arr is not None:
            assert self.arr.size == 0 or np.all(np.diff(self.arr) > 0)
            _load().orc_set_lambda_obs(_pf(self.arr), C.c_double(self.zp1))
        if self.grid is not None:
            assert np.all(np.diff(self.grid) > 0)
            _load().orc_set_lambda_ssp(_pf(self.grid))

    def __exit__(self, *exc):
        if self.arr is not None:
            _load().orc_set_lambda_obs(None, C.c_double(1.0))
        if self.grid is not None:
            _load().orc_set_lambda_ssp(None)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _pf(a):
    return _p(a, C.c_float)


def _pd(a):
    return _p(a, C.c_double)


def _pi(a):
    return _p(a, C.c_int32)


# ----------------------------------------------------------------------------- steps 1-3
def rotate_bin(pos, vel, R, n_x, n_y, spaxel_size):
    pos, vel, R = _f32(pos), _f32(vel), _f32(R).reshape(9)
    n = pos.shape[0]
    key = np.empty(n, np.int32)
    vlos = np.empty(n, np.float32)
    _load().orc_rotate_bin(C.c_int64(n), _pf(pos), _pf(vel), _pf(R), C.c_int32(n_x),
                           C.c_int32(n_y), C.c_float(float(spaxel_size)), _pi(key), _pf(vlos))
    return key, vlos


def sort(key, n_s):
    key = np.ascontiguousarray(key, dtype=np.int32)
    perm = np.empty(key.shape[0], np.int32)
    seg = np.empty(n_s + 2, np.int32)
    _load().orc_sort(C.c_int64(key.shape[0]), _pi(key), C.c_int32(n_s), _pi(perm), _pi(seg))
    return perm, seg


# ----------------------------------------------------------------------------- steps 4-5
def ssp_cells(log_age, log_z, age_axis, z_axis):
    log_age, log_z = _f32(log_age), _f32(log_z)
    age_axis, z_axis = _f32(age_axis), _f32(z_axis)
    n = log_age.shape[0]
    ia, iz = np.empty(n, np.int32), np.empty(n, np.int32)
    ta, tz = np.empty(n, np.float64), np.empty(n, np.float64)
    _load().orc_ssp_cells(C.c_int64(n), _pf(log_age), _pf(log_z), C.c_int32(age_axis.size),
                          C.c_int32(z_axis.size), _pf(age_axis), _pf(z_axis), _pi(ia), _pi(iz),
                          _pd(ta), _pd(tz))
    return ia, iz, ta, tz


def particle_spectrum(mass, log_age, log_z, vlos, ssp, tel):
    """One particle's spectrum on the observed grid; ``tel.resample`` picks the rule of step 5
    (0 point-sampled, 1 flux-conserving bin average)."""
    flux = _f32(ssp.flux)
    na, nz, nl = flux.shape
    age_axis, z_axis = _f32(ssp.log_age_axis), _f32(ssp.log_z_axis)
    out = np.empty(tel.n_channels, np.float64)
    with _grids(tel, ssp):
        _load().orc_particle_spectrum_mode(
            C.c_int32(_mode(tel, ssp)), C.c_double(float(getattr(tel, "redshift", 0.0))),
            C.c_double(float(getattr(tel, "flux_scale", 1.0))), C.c_float(float(mass)), C.c_float(float(log_age)), C.c_float(float(log_z)),
            C.c_float(float(vlos)), C.c_int32(na), C.c_int32(nz), C.c_int32(nl), _pf(age_axis),
            _pf(z_axis), C.c_float(float(ssp.lambda0)), C.c_float(float(ssp.dlambda)), _pf(flux),
            C.c_int32(tel.n_channels), C.c_float(float(tel.lambda0)), C.c_float(float(tel.dlambda)),
            _pd(out))
    return out


def particle_spectrum_f64(mass, log_age, log_z, vlos, ia, iz, ssp, tel):
    """fp64 parameters, cell (ia, iz) held fixed: the finite-difference evaluation."""
    flux = _f32(ssp.flux)
    na, nz, nl = flux.shape
    age_axis, z_axis = _f32(ssp.log_age_axis), _f32(ssp.log_z_axis)
    out = np.empty(tel.n_channels, np.float64)
    with _grids(tel, ssp):
        _load().orc_particle_spectrum_f64_mode(
            C.c_int32(_mode(tel, ssp)), C.c_double(float(getattr(tel, "redshift", 0.0))),
            C.c_double(float(getattr(tel, "flux_scale", 1.0))), C.c_double(float(mass)), C.c_double(float(log_age)), C.c_double(float(log_z)),
            C.c_double(float(vlos)), C.c_int32(na), C.c_int32(nz), C.c_int32(nl), _pf(age_axis),
            _pf(z_axis), C.c_float(float(ssp.lambda0)), C.c_float(float(ssp.dlambda)), _pf(flux),
            C.c_int32(tel.n_channels), C.c_float(float(tel.lambda0)), C.c_float(float(tel.dlambda)),
            C.c_int32(int(ia)), C.c_int32(int(iz)), _pd(out))
    return out


# ----------------------------------------------------------------------------- step 6
def build_cube(particles, R, ssp, tel, sel=None):
    """fp64 cube [n_x, n_y, n_c]; with ``sel`` (flat spaxel ids) -> [len(sel), n_c]."""
    pos, vel = _f32(particles.pos), _f32(particles.vel)
    mass, la, lz = _f32(particles.mass), _f32(particles.log_age), _f32(particles.log_z)
    R = _f32(R).reshape(9)
    flux = _f32(ssp.flux)
    na, nz, nl = flux.shape
    age_axis, z_axis = _f32(ssp.log_age_axis), _f32(ssp.log_z_axis)
    n_c = tel.n_channels
    if sel is None:
        sel_arr, n_sel = np.zeros(1, np.int32), 0
        cube = np.empty((tel.n_x, tel.n_y, n_c), np.float64)
    else:
        sel_arr = np.ascontiguousarray(sel, dtype=np.int32)
        n_sel = sel_arr.size
        cube = np.empty((n_sel, n_c), np.float64)
    with _grids(tel, ssp):
        _load().orc_build_cube_mode(
            C.c_int32(_mode(tel, ssp)), C.c_double(float(getattr(tel, "redshift", 0.0))),
            C.c_double(float(getattr(tel, "flux_scale", 1.0))), C.c_int64(mass.shape[0]), _pf(pos), _pf(vel), _pf(mass), _pf(la), _pf(lz), _pf(R),
            C.c_int32(na), C.c_int32(nz), C.c_int32(nl), _pf(age_axis), _pf(z_axis),
            C.c_float(float(ssp.lambda0)), C.c_float(float(ssp.dlambda)), _pf(flux),
            C.c_int32(tel.n_x), C.c_int32(tel.n_y), C.c_float(float(tel.spaxel_size)),
            C.c_int32(n_c), C.c_float(float(tel.lambda0)), C.c_float(float(tel.dlambda)),
            _pi(sel_arr), C.c_int32(n_sel), _pd(cube))
    return cube


# ----------------------------------------------------------------------------- steps 7-8
def psf_sigma_k(tel):
    """Per-channel PSF width of reading R18, or None when the PSF is the same for every channel:
    sigma_k = psf_sigma * (lambda_k / psf_lambda_ref) ** psf_alpha, lambda_k the observed wavelengths."""
    alpha = float(getattr(tel, "psf_alpha", 0.0))
    if alpha == 0.0 or tel.psf_size <= 0:
        return None
    return np.float64(tel.psf_sigma) * (tel.wavelengths() / np.float64(tel.psf_lambda_ref)) ** alpha


class _psf_sigma:
    """Installs a per-channel PSF width array in the C oracle for one call."""

    def __init__(self, sigma_k):
        self.arr = None if sigma_k is None else np.ascontiguousarray(sigma_k, dtype=np.float64)

    def __enter__(self):
        if self.arr is not None:
            _load().orc_set_psf_sigma(_pd(self.arr))

    def __exit__(self, *exc):
        if self.arr is not None:
            _load().orc_set_psf_sigma(None)


def gauss_taps(size, sigma):
    taps = np.empty(size, np.float64)
    _load().orc_gauss_taps(C.c_int32(size), C.c_double(float(sigma)), _pd(taps))
    return taps


def convolve(cube, psf_size, psf_sigma, lsf_size, lsf_sigma, sigma_k=None):
    """LSF along the channel, then the PSF over (x, y); ``sigma_k``: per-channel PSF widths (reading R18)."""
    cube = np.ascontiguousarray(cube, dtype=np.float64)
    n_x, n_y, n_c = cube.shape
    out = np.empty_like(cube)
    assert sigma_k is None or len(sigma_k) == n_c
    with _psf_sigma(sigma_k):
        _load().orc_convolve(_pd(cube), C.c_int32(n_x), C.c_int32(n_y), C.c_int32(n_c),
                             C.c_int32(psf_size), C.c_double(float(psf_sigma)), C.c_int32(lsf_size),
                             C.c_double(float(lsf_sigma)), _pd(out))
    return out


def convolve_transpose(gout, psf_size, psf_sigma, lsf_size, lsf_sigma, sigma_k=None):
    gout = np.ascontiguousarray(gout, dtype=np.float64)
    n_x, n_y, n_c = gout.shape
    gin = np.empty_like(gout)
    with _psf_sigma(sigma_k):
        _load().orc_convolve_transpose(_pd(gout), C.c_int32(n_x), C.c_int32(n_y), C.c_int32(n_c),
                                       C.c_int32(psf_size), C.c_double(float(psf_sigma)),
                                       C.c_int32(lsf_size), C.c_double(float(lsf_sigma)), _pd(gin))
    return gin


def convolve_voxels_f32(cube_f32, vox, psf_size, psf_sigma, lsf_size, lsf_sigma, sigma_k=None):
    """Brute-force value of sampled output voxels (flat indices) of an fp32 input cube."""
    assert cube_f32.dtype == np.float32 and cube_f32.flags.c_contiguous
    n_x, n_y, n_c = cube_f32.shape
    vox = np.ascontiguousarray(vox, dtype=np.int64)
    out = np.empty(vox.size, np.float64)
    with _psf_sigma(sigma_k):
        _load().orc_convolve_voxels_f32(
            _pf(cube_f32), C.c_int32(n_x), C.c_int32(n_y), C.c_int32(n_c), C.c_int32(psf_size),
            C.c_double(float(psf_sigma)), C.c_int32(lsf_size), C.c_double(float(lsf_sigma)),
            _p(vox, C.c_int64), C.c_int64(vox.size), _pd(out))
    return out


def forward(particles, R, ssp, tel):
    """Whole path: build + PSF/LSF (whatever ``tel`` switches on).  fp64 [n_x, n_y, n_c]."""
    cube = build_cube(particles, R, ssp, tel)
    if tel.psf_size > 0 or tel.lsf_size > 0:
        cube = convolve(cube, tel.psf_size, tel.psf_sigma, tel.lsf_size, tel.lsf_sigma, psf_sigma_k(tel))
    return cube


# ----------------------------------------------------------------------------- step 9
def adjoint(particles, R, ssp, tel, grad_cube):
    pos, vel = _f32(particles.pos), _f32(particles.vel)
    mass, la, lz = _f32(particles.mass), _f32(particles.log_age), _f32(particles.log_z)
    R = _f32(R).reshape(9)
    flux = _f32(ssp.flux)
    na, nz, nl = flux.shape
    age_axis, z_axis = _f32(ssp.log_age_axis), _f32(ssp.log_z_axis)
    grad_cube = np.ascontiguousarray(grad_cube, dtype=np.float64)
    n = mass.shape[0]
    out = [np.empty(n, np.float64) for _ in range(4)]
    with _grids(tel, ssp), _psf_sigma(psf_sigma_k(tel)):
        _load().orc_adjoint_mode(
            C.c_int32(_mode(tel, ssp)), C.c_double(float(getattr(tel, "redshift", 0.0))),
            C.c_double(float(getattr(tel, "flux_scale", 1.0))), C.c_int64(n), _pf(pos), _pf(vel), _pf(mass), _pf(la), _pf(lz), _pf(R), C.c_int32(na),
            C.c_int32(nz), C.c_int32(nl), _pf(age_axis), _pf(z_axis), C.c_float(float(ssp.lambda0)),
            C.c_float(float(ssp.dlambda)), _pf(flux), C.c_int32(tel.n_x), C.c_int32(tel.n_y),
            C.c_float(float(tel.spaxel_size)), C.c_int32(tel.n_channels),
            C.c_float(float(tel.lambda0)), C.c_float(float(tel.dlambda)), C.c_int32(tel.psf_size),
            C.c_double(float(tel.psf_sigma)), C.c_int32(tel.lsf_size),
            C.c_double(float(tel.lsf_sigma)), _pd(grad_cube), *(_pd(o) for o in out))
    return tuple(out)


def knot_clearance(vlos, ssp, tel, chunk=4096):
    """min over channels of |x_k - nearest integer|, x_k = rest position in SSP samples, per
    particle.  The spectrum has a kink in v_los wherever some x_k crosses an SSP knot; the
    finite-difference sample keeps away from those (non-differentiable points), and the
    all-particle gradient comparison leaves out the particles closer to a knot than the position resolution
    of the implementation under test (reading R19).  Linear and log-sampled SSP grids (R15), uniform
    and listed channel wavelengths (R16); evaluated in chunks of particles."""
    vlos = np.asarray(vlos, np.float64)
    lam = tel.wavelengths() / (1.0 + float(getattr(tel, "redshift", 0.0)))
    out = np.empty(vlos.shape[0], np.float64)
    for a in range(0, vlos.shape[0], chunk):
        beta = vlos[a:a + chunk, None] / C_KMS
        rest = lam[None, :] / (1.0 + beta)
        if getattr(ssp, "lambda_grid", None) is not None:              # listed SSP wavelengths (R21)
            knots = np.asarray(ssp.lambda_grid, np.float32).astype(np.float64)
            x = np.interp(rest, knots, np.arange(knots.size, dtype=np.float64))
            x = np.where((rest < knots[0]) | (rest > knots[-1]), 0.5, x)    # channels outside the coverage have no kink
        elif int(getattr(ssp, "log_lambda", 0)):
            x = np.log10(rest / np.float64(ssp.lambda0)) / np.float64(ssp.dlambda)
        else:
            x = (rest - np.float64(ssp.lambda0)) / np.float64(ssp.dlambda)
        out[a:a + chunk] = np.abs(x - np.round(x)).min(axis=1)
    return out


def fd_gradients(particles, R, ssp, tel, residual, idx, h_mass=1e-3, h_log=1e-4, h_v=1e-3):
    """Central finite differences of L = sum (cube_final - target)^2 for the particles ``idx``.

    ``residual`` = oracle final cube - target (fp64, [n_x, n_y, n_c]).  The pipeline is linear in
    each particle's spectrum, so perturbing particle p changes the final cube by
    P(delta) = (g (x) g)[x - sx, y - sy] * LSF(delta) around its spaxel (sx, sy), and
        L(theta +- h) - L0 = 2 <residual, P(delta+-)> + |P(delta+-)|^2 .
    Steps: mass h = 1e-3 m; log age / log Z h = 1e-4 dex; v_los h = 1e-3 km/s
    (reading R9: the survey's 0.05 km/s moves x_k by ~1e-3 SSP samples, which makes
    several of 3700 channels cross a knot for almost every particle).
    Returns four arrays (d/dmass, d/dlogAge, d/dlogZ, d/dv_los) aligned with ``idx``.
    """
    key, vlos = rotate_bin(particles.pos, particles.vel, R, tel.n_x, tel.n_y, tel.spaxel_size)
    ia, iz, _, _ = ssp_cells(particles.log_age, particles.log_z, ssp.log_age_axis, ssp.log_z_axis)
    n_c = tel.n_channels
    # PSF taps per channel, [n_c, psf_size] (all rows equal unless the PSF depends on wavelength, reading R18)
    if tel.psf_size > 0:
        sk = psf_sigma_k(tel)
        gk = np.stack([gauss_taps(tel.psf_size, tel.psf_sigma if sk is None else sk[k]) for k in range(n_c)]) \
            if sk is not None else np.broadcast_to(gauss_taps(tel.psf_size, tel.psf_sigma), (n_c, tel.psf_size))
    else:
        gk = np.ones((n_c, 1))
    hp = (gk.shape[1] - 1) // 2

    def lsf(row):
        if tel.lsf_size <= 0:
            return row
        return convolve(row.reshape(1, 1, n_c), 0, 0.0, tel.lsf_size, tel.lsf_sigma).reshape(n_c)

    def delta_loss(delta, sx, sy):
        row = lsf(delta)
        acc = 0.0
        for dx in range(-hp, hp + 1):
            for dy in range(-hp, hp + 1):
                x, y = sx + dx, sy + dy
                if 0 <= x < tel.n_x and 0 <= y < tel.n_y:
                    w = gk[:, dx + hp] * gk[:, dy + hp]            # per channel
                    wr = w * row
                    acc += 2.0 * float(residual[x, y] @ wr) + float(wr @ wr)
        return acc

    out = np.zeros((4, len(idx)), np.float64)
    for n_i, p in enumerate(idx):
        if key[p] >= tel.n_x * tel.n_y:
            continue
        sx, sy = divmod(int(key[p]), tel.n_y)
        theta0 = [float(particles.mass[p]), float(particles.log_age[p]),
                  float(particles.log_z[p]), float(vlos[p])]
        base = particle_spectrum_f64(*theta0, ia[p], iz[p], ssp, tel)
        for q, h in enumerate((h_mass * theta0[0], h_log, h_log, h_v)):
            dl = []
            for sign in (+1.0, -1.0):
                theta = list(theta0)
                theta[q] += sign * h
                spec = particle_spectrum_f64(*theta, ia[p], iz[p], ssp, tel)
                dl.append(delta_loss(spec - base, sx, sy))
            out[q, n_i] = (dl[0] - dl[1]) / (2.0 * h)
    return out[0], out[1], out[2], out[3]


# ----------------------------------------------------------------------------- noise stage (reading R17)
def philox4x32_10(counter, key):
    c = (C.c_uint32 * 4)(*[int(v) for v in counter])
    k = (C.c_uint32 * 2)(*[int(v) for v in key])
    out = (C.c_uint32 * 4)()
    _load().orc_philox4x32_10(c, k, out)
    return [int(v) for v in out]


def noise_normals(n, seed):
    z = np.empty(int(n), np.float64)
    _load().orc_noise_normals(C.c_int64(int(n)), C.c_uint64(int(seed)), _pd(z))
    return z


def add_noise(cube, sigma_read, gain, seed):
    cube = np.ascontiguousarray(cube, dtype=np.float64)
    out = np.empty_like(cube)
    _load().orc_add_noise(_pd(cube), C.c_int64(cube.size), C.c_double(float(sigma_read)), C.c_double(float(gain)),
                          C.c_uint64(int(seed)), _pd(out))
    return out
