/*
 * rubix.h -- C ABI of the B200-native hot path of RUBIX's IFU forward model
 * (arXiv 2412.08265; section 3 "RUBIX Codebase", L40).
 *
 * The path, in the paper's order: "orientate the galaxy in the field of
 * view" -> "particles are assigned to the IFU spaxels" -> "Each star spectrum is calculated as
 * a lookup from a simple stellar population (SSP) library" -> "Doppler shifted based on ...
 * line-of-sight velocity" -> "resampling ... to match the wavelength grid of the observed
 * telescope" -> "the stellar spectra in each spaxel are summed up" -> "point-spread function
 * (PSF) and line-spread function (LSF) convolution"; plus "gradient computations through the
 * entire pipeline".  The paper gives no formulas: the numerical definition of
 * every step is BASELINE.json:north_star as spelled out in SURVEY.md section 8(a)/(c) and
 * restated in DESIGN.md ("The path" / "Readings").
 *
 * Conventions (all entry points)
 *   - Plain C: pointers and sizes only.  Each pointer is marked HOST or DEVICE.
 *   - The caller owns every buffer.  The library never allocates or frees device memory and
 *     never synchronises: all work is enqueued on `stream` (a cudaStream_t passed as void*)
 *     and is complete when the stream is.  Host arrays (R, the SSP axes, the structs) are
 *     read before the call returns and may be freed right after it.
 *     Consequently a sequence of calls can be captured in a CUDA graph (stage timing of
 *     rubix_peaks.h off) and replayed; the kernels read their sizes from the workspace, not
 *     from the host, after the call has returned.  NOT capturable: calls with rubix_telescope.lambda_obs
 *     or rubix_ssp.lambda_grid (the host arrays are copied to the workspace; with lambda_obs the per-channel taps of a
 *     wavelength-dependent PSF are also computed on the host and copied from pageable memory -- on a uniform channel grid
 *     they are computed by a kernel and the call stays capturable); the rubix_forward_host* entries (host buffers).
 *   - Every compute call is bracketed by an NVTX range carrying its name (visible in Nsight timelines).
 *   - Device arrays are dense, row-major, fp32 / int32 as stated, 16-byte aligned.
 *   - Errors: every call validates its arguments on the host BEFORE any launch and returns a
 *     rubix_status; nothing throws or aborts.  rubix_last_error() gives a thread-local message.
 *   - There is no CPU fallback: without a CUDA device the compute calls return RUBIX_ERR_CUDA.
 *
 * Notation: N particles; N_x x N_y spaxels, N_s = N_x*N_y; N_c channels; SSP grid
 * N_a x N_z x N_l; beta = v_los / c, c = 299792.458 km/s.
 */
#ifndef RUBIX_B200_H
#define RUBIX_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    RUBIX_OK = 0,
    RUBIX_ERR_NULL = 1,          /* a required pointer is NULL */
    RUBIX_ERR_INVALID_ARG = 2,   /* bad size, even stencil, non-increasing axis, dlambda <= 0 ... */
    RUBIX_ERR_UNSUPPORTED = 3,   /* valid but outside this build's limits (see each call) */
    RUBIX_ERR_WORKSPACE = 4,     /* workspace NULL / misaligned / smaller than rubix_workspace_bytes */
    RUBIX_ERR_CUDA = 5           /* a CUDA runtime call failed (message has the CUDA error string) */
} rubix_status;

/* Stellar particles ("star ... particle information"; BASELINE.json north_star:
 * "position, velocity, mass, age, metallicity").  All DEVICE, fp32. */
typedef struct {
    int64_t n;              /* number of particles, >= 0 (0 is valid: all-zero cube)        */
    const float *pos;       /* [n][3] kpc, galaxy-centred                                  */
    const float *vel;       /* [n][3] km/s, systemic velocity removed                      */
    const float *mass;      /* [n] Msun                                                    */
    const float *log_age;   /* [n] log10(age / Gyr)                                        */
    const float *log_z;     /* [n] log10(Z)                                                */
} rubix_particles;

/* SSP template library ("lookup from a simple stellar population (SSP) library").
 * Limits: n_age <= 512, n_z <= 128, n_age*n_z*n_lambda < 2^31. */
typedef struct {
    uint32_t struct_size;           /* = sizeof(rubix_ssp) of the header the CALLER was built against; a mismatch */
                                    /* is refused with RUBIX_ERR_INVALID_ARG (the struct grows with the library)    */
    int32_t n_age, n_z, n_lambda;   /* each >= 2                                            */
    const float *log_age_axis;      /* HOST [n_age], strictly increasing                    */
    const float *log_z_axis;        /* HOST [n_z],   strictly increasing                    */
    float lambda0, dlambda;         /* uniform rest-frame grid, Angstrom, dlambda > 0       */
    const float *flux;              /* DEVICE [n_age][n_z][n_lambda], per unit mass         */
    int32_t log_lambda;             /* 0: lambda_j = lambda0 + j dlambda (Angstrom);          */
                                    /* 1: log-sampled grid (e.g. MaStar "SLOG"): */
                                    /*    lambda_j = lambda0 * 10^(j dlambda), dlambda in dex; */
                                    /*    the interpolant is then linear in log lambda between */
                                    /*    knots                                                */
    const float *lambda_grid;       /* HOST [n_lambda] or NULL.  Non-NULL: LISTED rest wavelengths   */
                                    /* (Angstrom, > 0, strictly increasing; irregular sampling as in */
                                    /* merged libraries) replace lambda0 / dlambda / log_lambda (which */
                                    /* must be 0); the interpolant is linear between the listed knots. */
                                    /* Read and copied to the workspace before the call returns.       */
} rubix_ssp;

/* Detector ("telescope-specific configurations", L44 Gaussian PSF and LSF). */
typedef struct {
    uint32_t struct_size;           /* = sizeof(rubix_telescope), checked like rubix_ssp.struct_size */
    int32_t n_x, n_y;               /* spaxels; FoV centred on the origin                   */
    float spaxel_size;              /* kpc, > 0                                             */
    int32_t n_channels;             /* >= 1                                                 */
    float lambda0, dlambda;         /* observed grid, Angstrom, dlambda > 0                 */
    int32_t psf_size;               /* odd taps <= 63 along x and along y; 0 = PSF off      */
    float psf_sigma;                /* spaxels, > 0 when psf_size > 0                       */
    int32_t lsf_size;               /* odd taps <= 63 along the channel axis; 0 = LSF off   */
    float lsf_sigma;                /* channels, > 0 when lsf_size > 0                      */
    int32_t resample;               /* RUBIX_RESAMPLE_POINT (0) or RUBIX_RESAMPLE_FLUX (1)  */
    float redshift;                 /* cosmological redshift z of the galaxy, 0 <= z <= 20:  */
                                    /* lambda_rest = lambda_obs / ((1 + z)(1 + beta))        */
    float flux_scale;               /* > 0: every spectrum is multiplied by it (distance     */
                                    /* dimming / unit conversion chosen by the caller); 1 = off */
    const float *lambda_obs;        /* HOST [n_channels] or NULL.  Non-NULL: explicit channel   */
                                    /* wavelengths (Angstrom, > 0, strictly increasing) replace  */
                                    /* lambda0 + k dlambda.  With RUBIX_RESAMPLE_FLUX (needs       */
                                    /* n_channels >= 2) channel k is the bin between the midpoints  */
                                    /* to its neighbours (outer edges half a spacing outside).  Read */
                                    /* (and copied to the workspace) before the call returns.       */
    float psf_alpha;                /* wavelength-dependent PSF: channel k uses the width         */
    float psf_lambda_ref;           /* psf_sigma (lambda_k / psf_lambda_ref)^psf_alpha (e.g. -0.2 */
                                    /* for seeing); 0 = the same PSF for every channel.  Needs    */
                                    /* psf_size <= 15, lsf_size <= 9 and an even n_channels.      */
                                    /* The PSF then acts AFTER the LSF (they no longer commute).  */
    int32_t n_x_full, x_first;      /* Row window for spaxel-sharded runs:  */
                                    /* n_x_full > 0: the detector has n_x_full rows along x, binning  */
                                    /* uses THAT geometry (bit-equal keys), and this call owns the    */
                                    /* n_x rows x_first .. x_first + n_x - 1 (key = (ix - x_first)    */
                                    /* n_y + iy; particles in other rows are dropped).  0 = off.      */
    int32_t cell_order;             /* Per-cell template reuse in piled-up spaxels (SURVEY.md 8(d)    */
                                    /* K3): the particles of a spaxel are accumulated in the order    */
                                    /* (SSP cell, original index) and spaxels with >= 2 N_a N_z       */
                                    /* particles go to a kernel that keeps the corner templates of a  */
                                    /* cell in registers.  RUBIX_CELL_ORDER_AUTO (0): on when         */
                                    /* n >= 10^6 and n >= 64 x the spaxels of the whole detector      */
                                    /* (times the batch); _OFF (1); _ON (2); _ALL (3): on, and EVERY  */
                                    /* spaxel goes to that kernel.  Uniform grids and the point rule  */
                                    /* only (otherwise off).  Changes the fp32 summation order inside */
                                    /* a spaxel and the exported `perm` (rubix_get_sort_artifacts),   */
                                    /* nothing else; calls that must agree bit for bit (the ranks of  */
                                    /* a spaxel-sharded run) pass the same explicit value.            */
    int32_t reserved0;              /* 0 */
} rubix_telescope;

#define RUBIX_CELL_ORDER_AUTO 0
#define RUBIX_CELL_ORDER_OFF 1
#define RUBIX_CELL_ORDER_ON 2
#define RUBIX_CELL_ORDER_ALL 3

/* Version of this header's ABI (struct layouts and call signatures); bumped whenever either changes.
 * rubix_abi_version() returns the value the LIBRARY was built with. */
#define RUBIX_ABI_VERSION 9
uint32_t rubix_abi_version(void);

/* Resampling rule of step 5 ("Additional resampling is performed to match the
 * wavelength grid of the observed telescope"; the paper does not say which rule):
 *   RUBIX_RESAMPLE_POINT  F[k] = S~(lambda_k / (1+beta)): the piecewise-linear interpolant of the
 *                         blended SSP samples, point-sampled at the channel centre (SURVEY.md
 *                         8(c) row 5, numpy.interp with left = right = 0);
 *   RUBIX_RESAMPLE_FLUX   F[k] = (1/dlambda_obs) * integral of S~(lambda / (1+beta)) over the bin
 *                         [lambda_k - dlambda_obs/2, lambda_k + dlambda_obs/2], S~ = 0 outside the
 *                         SSP coverage (sum_k F[k] dlambda_obs telescopes to the
 *                         total flux exactly).  rubix_cube_adjoint differentiates whichever rule
 *                         the telescope selects.  On a log-sampled SSP grid, on listed channel
 *                         wavelengths and on listed SSP wavelengths the bin [e_k, e_{k+1}] of observed
 *                         wavelength is averaged IN THE SAMPLING COORDINATE x of the SSP grid,
 *                         F[k] = (1/(x_hi - x_lo)) * integral of S~(x) dx  (reading R20: identical
 *                         to the above on a linearly sampled grid; per unit log lambda on a log-sampled one). */
#define RUBIX_RESAMPLE_POINT 0
#define RUBIX_RESAMPLE_FLUX 1

/* Bytes of DEVICE scratch that any of the three compute calls below may need for this problem
 * size (the maximum over the three).  Returns 0 on invalid arguments (rubix_last_error says
 * why).  The workspace must be 256-byte aligned. */
size_t rubix_workspace_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel);

/* Steps 1-6: rotate into the field of view, project and bin to a
 * spaxel, sort by spaxel key, SSP bilinear lookup x mass, Doppler shift + linear resampling onto
 * the observed grid, per-spaxel sum.
 *   R     HOST  [9] row-major rotation; r' = R r, line of sight = +z' (receding positive).
 *   cube  DEVICE [n_x][n_y][n_channels] fp32, channel-contiguous; EVERY voxel is written
 *         exactly once (empty spaxels get 0); no atomics, bit-reproducible run to run.
 * Binning is the fp32 fixed-order arithmetic of SURVEY.md 8(c)-2 (bit-exact vs the oracle);
 * particles outside the FoV, with non-finite coordinates, or with |v_los| > 0.05 c are dropped.
 * Returns RUBIX_ERR_UNSUPPORTED if dlambda_obs/dlambda_ssp >= 15 (resampler fixed-point range).
 * Leaves the sort artefacts in `workspace` (see rubix_get_sort_artifacts). */
rubix_status rubix_build_cube(const rubix_particles *particles, const rubix_ssp *ssp,
                              const rubix_telescope *tel, const float *R, float *cube,
                              void *workspace, size_t workspace_bytes, void *stream);

/* Steps 7-8: Gaussian PSF over (x, y), the same for
 * every channel, and Gaussian LSF along the channel axis.  Taps exp(-i^2 / 2 sigma^2) sampled at
 * integer offsets and normalised to sum 1; 'same' output; zero padding.  A size of 0 switches
 * that stage off (both 0: plain copy).
 *   cube_in, cube_out  DEVICE [n_x][n_y][n_channels] fp32; must not overlap. */
rubix_status rubix_convolve_psf_lsf(const rubix_telescope *tel, const float *cube_in,
                                    float *cube_out, void *workspace, size_t workspace_bytes,
                                    void *stream);

/* Steps 1-2 alone: the spaxel key and the line-of-sight velocity of every particle, in the
 * caller's order, with the fp32 fixed-order arithmetic of rubix_build_cube (bit-equal keys).  Used by the spaxel-sharded
 * multi-GPU path (paper_2412_08265_b200/sharded.py) to route particles to the rank that owns their detector row.
 *   pos, vel  DEVICE [n][3];  key DEVICE [n] int32 (n_x*n_y = dropped);  vlos DEVICE [n] fp32 or NULL */
rubix_status rubix_bin_particles(int64_t n, const float *pos, const float *vel, const rubix_telescope *tel, const float *R,
                                 int32_t *key, float *vlos, void *stream);

/* rubix_build_cube with the halo exchange of a spaxel-sharded run FUSED into the producing kernels (
 * paper_2412_08265_b200/sharded.py): besides `cube`, the first `mirror_rows` detector rows (x < mirror_rows) are stored at
 * mirror_lo [mirror_rows][n_y][n_channels] and the last `mirror_rows` rows at mirror_hi, row by row as k_accumulate /
 * k_reduce_partials produce them.  The mirrors are the halo regions of the neighbouring ranks' buffers: any DEVICE address the
 * calling GPU can store to -- memory of the same GPU, or PEER memory of another GPU mapped into this process (NVLink stores);
 * NULL = no mirror on that side.  The neighbour may read its halo once this call's stream has completed (the caller
 * synchronises across ranks).  Everything else as rubix_build_cube. */
rubix_status rubix_build_cube_mirrored(const rubix_particles *particles, const rubix_ssp *ssp, const rubix_telescope *tel,
                                       const float *R, float *cube, float *mirror_lo, float *mirror_hi, int32_t mirror_rows,
                                       void *workspace, size_t workspace_bytes, void *stream);

/* Steps 1-8 in one call on DEVICE buffers (the whole forward model: rubix_build_cube followed by
 * rubix_convolve_psf_lsf, same arithmetic, same results bit for bit).  The raw cube of step 6 lives in the workspace; with
 * PSF/LSF on (psf_size <= 15, lsf_size <= 9, even n_channels) the sort's segment table tells the stencil passes which
 * spaxels hold particles: rows of empty spaxels are neither written by step 6 nor read by step 7, and all-zero rows of
 * the temporary between the two PSF passes are neither written nor read (the PSF/LSF floor is one read
 * and one write of the cube).  Other stencil shapes run the two plain stages.
 *   cube  DEVICE [n_x][n_y][n_channels] fp32: the FINAL cube (raw cube when PSF and LSF are off); every voxel written
 *         exactly once; must not overlap the workspace.
 * Arguments, limits, errors and sort artefacts as rubix_build_cube.  This is the device-resident call bench.py times. */
rubix_status rubix_forward(const rubix_particles *particles, const rubix_ssp *ssp, const rubix_telescope *tel,
                           const float *R, float *cube, void *workspace, size_t workspace_bytes, void *stream);

/* Batched steps 1-8 ("produce a sufficient number of samples required for statistical
 * analysis", L86 SBI): `batch` cubes per call with ONE launch sequence -- the detectors sit side by side in one key space
 * of batch * N_s spaxels, so the sort, the work units, the accumulate kernel and the PSF/LSF passes each run once for all
 * elements (small cubes are launch-latency bound one at a time).  Element b is computed exactly as rubix_forward would
 * (bit-equal cubes).
 *   particles  DEVICE arrays.  offsets != NULL: `batch` galaxies concatenated, element b = particles
 *              offsets[b] .. offsets[b+1]) (HOST [batch+1], offsets[0] = 0, offsets[batch] = particles->n, non-decreasing).
 *              offsets == NULL: the SAME particles->n particles for every element (one galaxy, `batch` orientations).
 *   R          HOST [batch][9], one rotation per element
 *   cubes      DEVICE [batch][n_x][n_y][n_channels] fp32, element-major; must not overlap the workspace
 * Elements are processed in groups of 64 (the rotations travel as kernel parameters); the sort artefacts left in the
 * workspace are those of the LAST group (keys are element * N_s + spaxel, dropped particles get group size * N_s).
 * Workspace: rubix_forward_batched_workspace_bytes (returns 0 on invalid arguments). */
size_t rubix_forward_batched_workspace_bytes(int64_t n, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                             const rubix_telescope *tel);
rubix_status rubix_forward_batched(const rubix_particles *particles, const int64_t *offsets, int32_t batch,
                                   const rubix_ssp *ssp, const rubix_telescope *tel, const float *R, float *cubes,
                                   void *workspace, size_t workspace_bytes, void *stream);

/* Step 9: gradients of a scalar loss L of the FINAL cube
 * (after PSF/LSF, if tel switches them on) with respect to each particle's mass, log age,
 * log Z and line-of-sight velocity.
 *   grad_cube  DEVICE [n_x][n_y][n_channels] fp32 = dL/d(final cube) (any loss: the caller
 *              forms it, e.g. 2 (cube - target) for BASELINE.json configs[4]).
 *   g_*        DEVICE [n] fp32, ORIGINAL particle order; dropped particles get 0; clamped
 *              ages / metallicities get 0 for that component.  g_vlos is per km/s.
 * Runs its own particle pass; no atomics (one warp owns one particle). */
rubix_status rubix_cube_adjoint(const rubix_particles *particles, const rubix_ssp *ssp,
                                const rubix_telescope *tel, const float *R,
                                const float *grad_cube, float *g_mass, float *g_log_age,
                                float *g_log_z, float *g_vlos, void *workspace,
                                size_t workspace_bytes, void *stream);

/* Fused forward + loss + adjoint for gradient-based fitting ("gradient computations
 * through the entire pipeline"; BASELINE.json configs[4]): steps 1-8, then
 *     L = sum over voxels of (final cube - target)^2       (fp64 sum in a fixed order: bit-reproducible)
 * and step 9 with the upstream gradient 2 (final cube - target), sharing ONE particle pass (rotate, bin,
 * sort, records) between the forward and the adjoint.  Equivalent to rubix_build_cube +
 * rubix_convolve_psf_lsf + (caller forms the residual) + rubix_cube_adjoint.
 *   target    DEVICE [n_x][n_y][n_channels] fp32
 *   loss      DEVICE, one double
 *   cube_out  DEVICE [n_x][n_y][n_channels] fp32 or NULL: receives the final cube when non-NULL
 *   g_*       as rubix_cube_adjoint
 * Needs rubix_loss_and_grad_workspace_bytes(...) bytes of workspace (one more cube-sized buffer than
 * rubix_workspace_bytes, plus the loss partials); returns 0 on invalid arguments. */
size_t rubix_loss_and_grad_workspace_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel);
rubix_status rubix_loss_and_grad(const rubix_particles *particles, const rubix_ssp *ssp,
                                 const rubix_telescope *tel, const float *R, const float *target,
                                 double *loss, float *cube_out, float *g_mass, float *g_log_age,
                                 float *g_log_z, float *g_vlos, void *workspace, size_t workspace_bytes,
                                 void *stream);

/* rubix_loss_and_grad for `batch` concatenated galaxies per call ("gradient based
 * optimization", L32): one launch sequence per group of 64 elements runs steps 1-8, the per-element losses
 *     loss[b] = sum over the voxels of element b of (final cube_b - target_b)^2
 * and step 9 for every particle, with one particle pass shared by forward and adjoint.  Element b gets the cube, the loss (when
 * n_x n_y n_channels is a multiple of 4: bit-equal; else equal to rounding of the fp64 sum) and the gradients of a single
 * rubix_loss_and_grad call on that galaxy.
 *   offsets    HOST [batch+1], required (the same-galaxy mode of rubix_forward_batched has no gradient counterpart)
 *   targets    DEVICE [batch][n_x][n_y][n_channels];  loss DEVICE [batch] doubles;  cubes_out DEVICE like targets, or NULL
 *   g_*        DEVICE [particles->n] in the order of the concatenated arrays
 * When cubes_out is NULL and PSF / LSF are on, the final cubes live in the workspace only. */
size_t rubix_loss_and_grad_batched_workspace_bytes(int64_t n, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                                   const rubix_telescope *tel);
rubix_status rubix_loss_and_grad_batched(const rubix_particles *particles, const int64_t *offsets, int32_t batch,
                                         const rubix_ssp *ssp, const rubix_telescope *tel, const float *R, const float *targets,
                                         double *loss, float *cubes_out, float *g_mass, float *g_log_age, float *g_log_z,
                                         float *g_vlos, void *workspace, size_t workspace_bytes, void *stream);

/* The loss step of rubix_loss_and_grad on its own, WITHOUT any workspace or allocation (for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 *     grads[b][v] = 2 (cubes[b][v] - targets[b][v]),   loss[b] = sum_v (cubes[b][v] - targets[b][v])^2   (fp64, fixed order)
 * for `batch` cubes of n_voxels voxels back to back -- the upstream gradient rubix_cube_adjoint takes (
 * SURVEY.md 8(f)-3).  Same kernels and summation order as inside rubix_loss_and_grad(_batched): the same values bit for bit.
 *   cubes, targets, grads  DEVICE [batch][n_voxels] fp32, three distinct arrays;  loss  DEVICE [batch] doubles
 * The per-block partial sums live in a file-scope device array of the library: 64 x 1184 doubles = 606 208 bytes, held by
 * every GPU that loads the library until the process exits.  LIMIT: batch <= RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH (64);
 * more is refused with RUBIX_ERR_UNSUPPORTED.  All calls on one device share that array: calls that may overlap on the GPU
 * (different streams without an ordering between them) race on it and return wrong losses -- order them on one stream or
 * with events.  Nothing in it has to be cleared between calls (every slot is written before it is read).  The call
 * launches two kernels on `stream`, never synchronises and calls no cudaMalloc / cudaFree. */
#define RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH 64
rubix_status rubix_residual_loss_static(const float *cubes, const float *targets, int64_t n_voxels, int32_t batch,
                                        float *grads, double *loss, void *stream);

/* Noise stage ("add realistic noise"; the paper names no model -- DESIGN.md reading R17):
 *     cube_out[v] = cube_in[v] + sqrt(sigma_read^2 + gain * max(cube_in[v], 0)) * n_v ,   n_v ~ N(0, 1)
 * (read noise plus shot noise, in the cube's flux units).  The deviates come from the counter-based
 * Philox4x32-10 generator keyed by `seed` with counter v / 4 and a Box-Muller map, so they depend only on
 * (seed, v): reproducible, independent of the launch configuration.
 *   cube_in, cube_out  DEVICE [n_voxels] fp32; cube_in == cube_out (in place) is allowed, partial overlap is not.
 * The noise is not differentiated: rubix_cube_adjoint / rubix_loss_and_grad act on the noise-free cube. */
rubix_status rubix_add_noise(const float *cube_in, float *cube_out, int64_t n_voxels, float sigma_read, float gain,
                             uint64_t seed, void *stream);

/* DEVICE pointers into the workspace last used by rubix_build_cube / rubix_forward / rubix_cube_adjoint /
 * rubix_loss_and_grad on this workspace address (the library remembers the 256 most recently used addresses) (compared bit for bit with the oracle):
 *   key     [n]      spaxel key of each particle in original order (n_s = dropped)
 *   perm    [n]      stable order by (key, original index); with the cell order active (rubix_telescope.cell_order)
 *                    by (key, SSP cell, original index): the same segments, each holding the same particles
 *   seg_off [n_s+2]  segment s is perm[seg_off[s] .. seg_off[s+1]); s = n_s: dropped particles
 * Valid once the stream of that call has completed. */
rubix_status rubix_get_sort_artifacts(const void *workspace, const int32_t **key,
                                      const int32_t **perm, const int32_t **seg_off);

/* Whole path with HOST buffers: copies the particle arrays and the SSP grid host->device,
 * runs rubix_forward (steps 1-8), and copies the final cube
 * device->host, all on `stream`; returns after enqueueing (pinned host memory makes the copies
 * asynchronous).  This is the end-to-end call bench.py times.
 *   h_particles  the five arrays are HOST pointers here;  h_ssp->flux is a HOST pointer here
 *   h_cube       HOST [n_x][n_y][n_channels] fp32
 *   device_scratch  DEVICE, at least rubix_forward_host_scratch_bytes(...) bytes, 256-B aligned */
size_t rubix_forward_host_scratch_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel);
rubix_status rubix_forward_host(const rubix_particles *h_particles, const rubix_ssp *h_ssp,
                                const rubix_telescope *tel, const float *R, float *h_cube,
                                void *device_scratch, size_t scratch_bytes, void *stream);

/* Pipelined variant of rubix_forward_host for back-to-back cubes (mock-catalogue generation): the device->host copy
 * of call i runs on an internal copy stream while call i + 1 computes on `stream`; two device buffers take the final
 * cube in turn (scratch: rubix_forward_host_pipelined_scratch_bytes, one cube more).  Everything else is as
 * rubix_forward_host, EXCEPT completion: h_cube of a call is complete once rubix_forward_host_drain(stream) has been
 * called after it and `stream` has completed (or the device has been synchronised).  Host buffers must be pinned
 * for the copies to overlap.  One pipeline per process (calls are serialised by a mutex). */
size_t rubix_forward_host_pipelined_scratch_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel);
rubix_status rubix_forward_host_pipelined(const rubix_particles *h_particles, const rubix_ssp *h_ssp,
                                          const rubix_telescope *tel, const float *R, float *h_cube,
                                          void *device_scratch, size_t scratch_bytes, void *stream);
/* Makes `stream` wait for every device->host copy the pipelined calls have enqueued so far. */
rubix_status rubix_forward_host_drain(void *stream);

/* Number of kernel launches the last compute call on this thread enqueued (bench.py's
 * gpu_launches claim is the sum over the timed region). */
int32_t rubix_last_launch_count(void);

/* Thread-local, NUL-terminated message of the last failing call on this thread ("" if none). */
const char *rubix_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RUBIX_B200_H */
