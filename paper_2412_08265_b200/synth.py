"""Seeded synthetic inputs shaped like the paper's workloads (stand-ins, not the real data).

The paper runs on TNG50-1 subhalo particles, the MaStar CB19 SSP library and a MUSE
set-up (§4 "Qualitative Analysis"); none of these is available here, so
BASELINE.json:configs[0..4] and SURVEY.md §8(d) define synthetic galaxies, SSP grids and
detectors with the same shapes and value ranges.  This module produces those inputs and
NOTHING of the method's arithmetic: no binning, no interpolation, no Doppler shift, no
convolution.  Both the fp64 oracle (``oracle/``) and the CUDA path consume the arrays it
returns, so it must not import either of them.

Everything is drawn from ``numpy.random.Generator(PCG64(seed))`` in a fixed order, computed
in fp64 and cast to fp32 once at the end.  Seeds: galaxy 1000+i, SSP grid
2000+i, orientation 3000+i for config i; the adjoint target galaxy uses seed 4001 and the
finite-difference particle sample seed 4002.
"""
from __future__ import annotations

import dataclasses
import hashlib
import math

import numpy as np

C_KMS = 299792.458  # speed of light, km/s

# FWHM -> sigma of a Gaussian: sigma = FWHM / (2 sqrt(2 ln 2))
FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))


# --------------------------------------------------------------------------------------
# orientation ("orientate the galaxy in the field of view"; convention is
# this generator's: R = Rz(gamma) Ry(beta) Rx(alpha), degrees, right-handed, active)
# --------------------------------------------------------------------------------------
def euler_rotation(alpha_deg: float, beta_deg: float, gamma_deg: float) -> np.ndarray:
    a, b, g = (math.radians(v) for v in (alpha_deg, beta_deg, gamma_deg))
    rx = np.array([[1, 0, 0], [0, math.cos(a), -math.sin(a)], [0, math.sin(a), math.cos(a)]])
    ry = np.array([[math.cos(b), 0, math.sin(b)], [0, 1, 0], [-math.sin(b), 0, math.cos(b)]])
    rz = np.array([[math.cos(g), -math.sin(g), 0], [math.sin(g), math.cos(g), 0], [0, 0, 1]])
    return (rz @ ry @ rx).astype(np.float32)


def random_euler(seed: int) -> tuple[float, float, float]:
    rng = np.random.Generator(np.random.PCG64(seed))
    alpha = float(rng.uniform(0.0, 360.0))
    beta = float(np.degrees(np.arccos(1.0 - 2.0 * rng.uniform())))
    gamma = float(rng.uniform(0.0, 360.0))
    return alpha, beta, gamma


# --------------------------------------------------------------------------------------
# particles
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Particles:
    pos: np.ndarray      # [n,3] fp32 kpc, galaxy-centred
    vel: np.ndarray      # [n,3] fp32 km/s, systemic velocity removed
    mass: np.ndarray     # [n]   fp32 Msun
    log_age: np.ndarray  # [n]   fp32 log10(age / Gyr)
    log_z: np.ndarray    # [n]   fp32 log10(Z)

    @property
    def n(self) -> int:
        return int(self.mass.shape[0])

    def subset(self, idx) -> "Particles":
        return Particles(*(np.ascontiguousarray(getattr(self, f.name)[idx])
                           for f in dataclasses.fields(self)))

    def copy(self) -> "Particles":
        return Particles(*(getattr(self, f.name).copy() for f in dataclasses.fields(self)))


def _isotropic(rng, n):
    cos_t = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    sin_t = np.sqrt(1.0 - cos_t * cos_t)
    return np.stack([sin_t * np.cos(phi), sin_t * np.sin(phi), cos_t], axis=1)


def make_particles(n: int, seed: int, *, kind: str = "gauss", bulge_frac: float = 0.1,
                   bulge_a: float = 0.5, disc_h: float = 3.0, disc_z: float = 0.3,
                   sigma_v: float = 50.0, v_rot: float = 200.0) -> Particles:
    """kind='gauss': config 0 (isotropic Gaussian blob, sigma 3 kpc).
    kind='disc_bulge': configs 1-3 (exponential disc + Hernquist bulge; ``bulge_frac`` is the
    share of the particle COUNT in the bulge)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    if kind == "gauss":
        pos = rng.normal(0.0, 3.0, (n, 3))
    elif kind == "disc_bulge":
        n_b = int(round(bulge_frac * n))
        n_d = n - n_b
        rad = rng.gamma(2.0, disc_h, n_d)                      # surface density ~ exp(-R/h)
        phi = rng.uniform(0.0, 2.0 * np.pi, n_d)
        zed = disc_z * rng.exponential(1.0, n_d) * rng.choice([-1.0, 1.0], n_d)
        disc = np.stack([rad * np.cos(phi), rad * np.sin(phi), zed], axis=1)
        u = rng.uniform(0.0, 1.0, n_b)
        su = np.sqrt(u)
        r_b = bulge_a * su / (1.0 - su)                         # Hernquist M(<r) inverse
        bulge = r_b[:, None] * _isotropic(rng, n_b)
        pos = np.concatenate([disc, bulge], axis=0)
        pos = pos[rng.permutation(n)]                           # no spatial order in memory
    else:
        raise ValueError(kind)
    phi = np.arctan2(pos[:, 1], pos[:, 0])
    vel = v_rot * np.stack([-np.sin(phi), np.cos(phi), np.zeros(n)], axis=1)
    vel = vel + rng.normal(0.0, sigma_v, (n, 3))
    mass = 1e5 * np.exp(0.5 * rng.normal(0.0, 1.0, n))
    log_age = rng.uniform(math.log10(0.1), math.log10(13.5), n)
    log_z = rng.uniform(-4.0, math.log10(0.03), n)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return Particles(f32(pos), f32(vel), f32(mass), f32(log_age), f32(log_z))


# --------------------------------------------------------------------------------------
# SSP template grid
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class SSPGrid:
    log_age_axis: np.ndarray  # [n_age] fp32, strictly increasing, log10(age/Gyr)
    log_z_axis: np.ndarray    # [n_z]   fp32, strictly increasing, log10(Z)
    lambda0: np.float32       # first rest wavelength, Angstrom
    dlambda: np.float32       # uniform rest step: Angstrom, or dex (log10) when log_lambda = 1
    flux: np.ndarray          # [n_age, n_z, n_lambda] fp32, per unit mass, > 0
    log_lambda: int = 0       # 1: log-sampled grid, lambda_j = lambda0 * 10^(j dlambda)
    lambda_grid: np.ndarray | None = None   # listed rest wavelengths [n_lambda] fp32, strictly increasing (irregular grid)

    @property
    def shape(self):
        return self.flux.shape

    def wavelengths(self) -> np.ndarray:
        if self.lambda_grid is not None:
            return np.asarray(self.lambda_grid, np.float32).astype(np.float64)
        j = np.arange(self.flux.shape[2])
        if self.log_lambda:
            return np.float64(self.lambda0) * 10.0 ** (np.float64(self.dlambda) * j)
        return np.float64(self.lambda0) + np.float64(self.dlambda) * j


def _jittered_axis(rng, lo, hi, n):
    ax = np.linspace(lo, hi, n)
    if n > 2:
        step = (hi - lo) / (n - 1)
        ax[1:-1] += rng.uniform(-0.2, 0.2, n - 2) * step
    return ax


def make_ssp(n_age: int, n_z: int, n_lambda: int, lam_lo: float, lam_hi: float,
             seed: int, n_lines: int = 10, log_lambda: bool = False, irregular: bool = False) -> SSPGrid:
    """Smooth positive continuum times ``n_lines`` Gaussian absorption lines whose depths vary
    with age and Z (BASELINE.json configs[0]; recipe SURVEY.md §8(d)).  ``irregular``: the same recipe sampled at
    listed wavelengths -- the uniform knots with the interior ones moved by up to +-35 % of the spacing and a region
    of doubled sampling density in the middle third (as merged / multi-arm libraries have)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    age_ax = _jittered_axis(rng, math.log10(0.1), math.log10(13.5), n_age)
    z_ax = _jittered_axis(rng, -4.0, math.log10(0.03), n_z)
    dlam = (lam_hi - lam_lo) / (n_lambda - 1)
    lam = lam_lo + dlam * np.arange(n_lambda)
    dlog = math.log10(lam_hi / lam_lo) / (n_lambda - 1)
    if log_lambda:                                         # same recipe on a log-sampled grid (MaStar "SLOG")
        lam = lam_lo * 10.0 ** (dlog * np.arange(n_lambda))
    if irregular:                                          # own generator: the draws below stay those of the uniform grid
        rj = np.random.Generator(np.random.PCG64(seed + 1_000_003))
        t = np.linspace(0.0, 1.0, n_lambda)
        dens = 1.0 + ((t > 1.0 / 3.0) & (t < 2.0 / 3.0))     # doubled density in the middle third
        pos = np.concatenate([[0.0], np.cumsum(1.0 / (0.5 * (dens[1:] + dens[:-1])))])
        lam = lam_lo + (lam_hi - lam_lo) * pos / pos[-1]
        step = np.minimum(np.diff(lam)[1:], np.diff(lam)[:-1])
        lam[1:-1] += rj.uniform(-0.35, 0.35, n_lambda - 2) * step
        lam = lam.astype(np.float32).astype(np.float64)       # the knots the library sees
    u = ((age_ax - age_ax[0]) / (age_ax[-1] - age_ax[0]))[:, None, None]
    w = ((z_ax - z_ax[0]) / (z_ax[-1] - z_ax[0]))[None, :, None]
    ell = (lam / 5500.0)[None, None, :]
    span = lam_hi - lam_lo
    centre = rng.uniform(lam_lo + 0.05 * span, lam_hi - 0.05 * span, n_lines)
    width = rng.uniform(2.0, 6.0, n_lines) * dlam
    depth0 = rng.uniform(0.1, 0.6, n_lines)
    mix = rng.uniform(0.0, 1.0, n_lines)
    flux = 10.0 ** (-1.5 * u) * ell ** (-3.0 + 4.0 * u + 0.5 * w)
    for l in range(n_lines):
        d = depth0[l] * (0.3 + 0.7 * (mix[l] * u + (1.0 - mix[l]) * w))
        flux = flux * (1.0 - d * np.exp(-0.5 * ((lam[None, None, :] - centre[l]) / width[l]) ** 2))
    return SSPGrid(age_ax.astype(np.float32), z_ax.astype(np.float32),
                   np.float32(lam_lo), np.float32(dlog if log_lambda else dlam),
                   np.ascontiguousarray(flux, dtype=np.float32), 1 if log_lambda else 0,
                   lam.astype(np.float32) if irregular else None)


# --------------------------------------------------------------------------------------
# telescope / detector
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Telescope:
    n_x: int
    n_y: int
    spaxel_size: np.float32   # kpc; FoV centred on the origin
    n_channels: int
    lambda0: np.float32       # observed grid, Angstrom
    dlambda: np.float32
    psf_size: int = 0         # odd taps; 0 = off
    psf_sigma: np.float32 = np.float32(0.0)   # spaxels
    lsf_size: int = 0         # odd taps; 0 = off
    lsf_sigma: np.float32 = np.float32(0.0)   # channels
    resample: int = 0         # 0 = point-sampled linear interpolation, 1 = flux-conserving bin average
    redshift: np.float32 = np.float32(0.0)     # cosmological redshift of the galaxy
    flux_scale: np.float32 = np.float32(1.0)   # multiplies every spectrum (distance dimming / units)
    lambda_obs: np.ndarray | None = None       # explicit, increasing channel wavelengths [n_channels] fp32 (else uniform)
    psf_alpha: np.float32 = np.float32(0.0)    # PSF width ~ (lambda / psf_lambda_ref)^psf_alpha; 0 = the same for every channel
    psf_lambda_ref: np.float32 = np.float32(1.0)
    n_x_full: int = 0         # row window of a spaxel-sharded run: the whole detector has n_x_full rows and this
    x_first: int = 0          # telescope owns rows x_first .. x_first + n_x - 1 (0 / 0 = the whole detector)
    cell_order: int = 0       # per-cell template reuse in piled-up spaxels: 0 = auto, 1 = off, 2 = on, 3 = on for every spaxel

    @property
    def n_spaxels(self) -> int:
        return self.n_x * self.n_y

    def wavelengths(self) -> np.ndarray:
        if self.lambda_obs is not None:
            return np.asarray(self.lambda_obs, np.float32).astype(np.float64)
        return np.float64(self.lambda0) + np.float64(self.dlambda) * np.arange(self.n_channels)

    def with_psf_lsf(self, fwhm_spaxels=3.0, psf_size=15, lsf_sigma=2.0, lsf_size=9) -> "Telescope":
        return dataclasses.replace(self, psf_size=psf_size,
                                   psf_sigma=np.float32(fwhm_spaxels * FWHM_TO_SIGMA),
                                   lsf_size=lsf_size, lsf_sigma=np.float32(lsf_sigma))


# --------------------------------------------------------------------------------------
# the five workloads of BASELINE.json:configs
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Workload:
    name: str
    particles: Particles
    ssp: SSPGrid
    telescope: Telescope
    rotation: np.ndarray      # [3,3] fp32 row-major
    euler_deg: tuple


WORKLOADS = ("tiny", "small", "medium", "contention", "adjoint")
_INDEX = {n: i for i, n in enumerate(WORKLOADS)}


def make_telescope(name: str) -> Telescope:
    if name == "tiny":      # 16x16 of 1 kpc, 256 channels 4700..9300 inclusive
        return Telescope(16, 16, np.float32(1.0), 256, np.float32(4700.0),
                         np.float32(4600.0 / 255.0))
    if name == "small":     # 25x25 (30 kpc FoV), 3700 channels at 1.25 A from 4750 A
        return Telescope(25, 25, np.float32(1.2), 3700, np.float32(4750.0), np.float32(1.25))
    if name == "medium":
        return Telescope(300, 300, np.float32(0.1), 3700, np.float32(4750.0),
                         np.float32(1.25)).with_psf_lsf()
    if name == "contention":
        return Telescope(150, 150, np.float32(0.2), 3700, np.float32(4750.0),
                         np.float32(1.25)).with_psf_lsf()
    if name == "adjoint":   # config-1 detector + config-2 PSF/LSF (SURVEY.md §8(c)-9 reading)
        return make_telescope("small").with_psf_lsf()
    raise ValueError(name)


def make_ssp_for(name: str) -> SSPGrid:
    i = _INDEX["small" if name == "adjoint" else name]
    if name == "tiny":
        return make_ssp(8, 4, 512, 3500.0, 9500.0, 2000 + i)
    if name == "contention":
        return make_ssp(100, 12, 4300, 3000.0, 10000.0, 2000 + i)
    return make_ssp(50, 7, 4300, 3000.0, 10000.0, 2000 + i)


def make_particles_for(name: str, n: int | None = None, seed: int | None = None) -> Particles:
    i = _INDEX["small" if name == "adjoint" else name]
    seed = 1000 + i if seed is None else seed
    if name == "tiny":
        return make_particles(n or 1_000, seed, kind="gauss")
    if name in ("small", "adjoint"):
        return make_particles(n or 100_000, seed, kind="disc_bulge")
    if name == "medium":
        return make_particles(n or 1_000_000, seed, kind="disc_bulge")
    if name == "contention":
        return make_particles(n or 10_000_000, seed, kind="disc_bulge", bulge_frac=0.9,
                              bulge_a=0.2, sigma_v=150.0)
    raise ValueError(name)


def euler_for(name: str) -> tuple:
    if name == "tiny":
        return (0.0, 90.0, 0.0)
    if name in ("small", "adjoint"):
        return (0.0, 60.0, 0.0)
    return random_euler(3000 + _INDEX[name])


def make_workload(name: str, n: int | None = None, seed: int | None = None) -> Workload:
    """``n``/``seed`` override the particle count / galaxy seed (bench samples, replicas)."""
    euler = euler_for(name)
    return Workload(name, make_particles_for(name, n, seed), make_ssp_for(name),
                    make_telescope(name), euler_rotation(*euler), euler)


ADJOINT_TARGET_SEED = 4001
ADJOINT_FD_SEED = 4002


def synthetic_cube(n_x: int, n_y: int, n_c: int, seed: int) -> np.ndarray:
    """A positive fp32 cube with a bright centre and channel structure, for convolution tests
    that must not take their input from the CUDA path."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x = (np.arange(n_x) - 0.5 * (n_x - 1))[:, None, None] / max(n_x, 1)
    y = (np.arange(n_y) - 0.5 * (n_y - 1))[None, :, None] / max(n_y, 1)
    prof = np.exp(-8.0 * np.sqrt(x * x + y * y)).astype(np.float32)
    out = rng.random((n_x, n_y, n_c), dtype=np.float32)
    out *= prof
    out += np.float32(0.01)
    return out


def sha256(arr: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(arr).tobytes()).hexdigest()
