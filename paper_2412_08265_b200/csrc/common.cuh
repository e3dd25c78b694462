// Shared declarations of the CUDA path (never included by oracle/).
// Notation follows SURVEY.md section 8: N particles, N_s spaxels, N_c channels, SSP N_a x N_z x N_l.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/rubix.h"

namespace rubix {

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---- fixed constants of the method ------------------------------------
constexpr double kCkms = 299792.458;        // speed of light, km/s
constexpr float kVcapKms = 14989.623f;      // 0.05 c: |v_los| beyond this drops the particle
constexpr double kBetaCap = 0.05;

// ---- implementation constants ------------------------------------------------------------------
constexpr int kFxFrac = 28;                 // fractional bits of the rest-position fixed point
constexpr int kChunk = 128;                 // particles per work unit of the accumulate kernel
constexpr int kMaxAge = 512, kMaxZ = 128;   // SSP axes travel as kernel parameters
constexpr int kMaxTaps = 63;
constexpr int kAccThreads = 128;            // threads per CTA of the accumulate kernel (the 12.20 stride trick needs 128)
constexpr int kTabMax = 4096;               // table entries addressable by the 12.20 local format
constexpr int kSortWarps = 8;               // warps per CTA in the radix passes
constexpr int kSortItemsMax = 1024;         // keys per warp per radix pass: 128 .. 1024, chosen from n (Layout::sort_items)
constexpr int kSortMaxDigitBits = 9;
constexpr int kFluxPad = 2048;              // zero floats behind the workspace copy of the SSP grid
constexpr int kCellAutoMean = 64;           // cell order, auto: on when the detector holds >= this many particles per spaxel ...
constexpr int64_t kCellAutoMinN = 1000000;  // ... and at least this many particles (several waves of work units for BOTH kernels);
constexpr int kCellAutoRuns = 2;            // ... and a spaxel goes to k_accumulate_cell from this many particles per SSP cell
constexpr int kRowAlign = 32;               // rows of that copy are padded to 32 floats (128 B)

// Sorted-order particle record consumed by the accumulate kernel (48 B, 16-B aligned).
struct __align__(16) Rec {
    float w[4];        // mass x bilinear weights of corners (i,j) (i+1,j) (i,j+1) (i+1,j+1)
    int32_t cell;      // float offset of T[i][j][0] in the padded workspace copy of the grid
    uint32_t b_fx;     // B = dl_obs / (dl_ssp (1+beta)) in 4.28 fixed point
    int64_t a_fx;      // A = (l0_obs/(1+beta) - l0_ssp)/dl_ssp in 36.28 fixed point
    int32_t k_lo, k_hi;  // channels whose rest position lies inside the SSP coverage
    int32_t j0, nw;      // window of the whole spectrum: first SSP sample (multiple of 32), samples
};
static_assert(sizeof(Rec) == 48, "Rec layout");

// Per in-FoV particle, sorted order: what the adjoint kernel needs of the SSP cell (written by prepare_records_body).
struct __align__(16) AdjAux {
    float ta, tz;          // position inside the (log age, log Z) cell, in [0, 1]
    float inv_wa, inv_wz;  // 1 / cell width along each axis, 0 where the particle is clamped to the grid edge
};

// One work unit of the accumulate kernel: up to kChunk consecutive sorted particles of one spaxel.
struct __align__(16) Unit {
    int32_t start;     // first sorted index
    int32_t count;     // 0 = empty spaxel (zero fill)
    int32_t spaxel;
    int32_t part_row;  // >= 0: write a partial row (multi-chunk spaxel); -1: write the cube row
};

struct AxisParams {               // SSP axes, passed by value
    float age[kMaxAge];
    float z[kMaxZ];
    int32_t n_age, n_z;
};

struct Taps {
    float w[kMaxTaps];
    int32_t size;                 // 0 = stage off
};

// ---- workspace carve-up (host) ---------------------------------------------------------------
struct Layout {
    int64_t n;
    int32_t n_s, n_c;
    int32_t sort_passes, digit_bits, n_wchunks, sort_items;   // sort_items: keys per warp chunk (multiple of 32)
    int64_t max_units, max_part_rows, max_multi;
    size_t off_key, off_vlos, off_seg, off_keybuf[2], off_permbuf[2], off_hist, off_dtot,
        off_dbase, off_unitoff, off_partoff, off_multi, off_totals, off_tiletot, off_units, off_rec,
        off_partials, off_cube_a, off_cube_b, off_flux, off_xtab, off_lamobs, off_psftaps, off_aux, off_occ[2],
        off_gtab, off_gknots, off_ginvw, off_glut, off_glam;   // general-grid mode (gen_coord.cuh)
    int32_t n_rows, n_lambda, pitch;  // workspace copy of the SSP grid: n_rows = N_a*N_z rows of
                                      // `pitch` floats (zero padded), then kFluxPad zeros
    size_t bytes_total;           // two cube-sized buffers (convolve temp, adjoint G') + pass scratch
    int final_buf;                // which of the ping-pong buffers holds the final sort
};

Layout make_layout(int64_t n, int32_t n_s, int32_t n_c, int32_t n_rows, int32_t n_lambda);

// ---- host launchers (each returns the CUDA status of its launches) ----------------------------
constexpr int kMaxBatch = 64;              // batch elements per launch sequence (their rotations travel as kernel parameters)

struct PassInputs {
    const rubix_particles *p;
    const rubix_ssp *ssp;
    const rubix_telescope *tel;
    const float *R;                        // [batch][9]
    // Batched forward: `batch` detectors side by side in one key space of batch * N_s spaxels.
    // Logical particle i (0 <= i < Layout::n) belongs to element b with offsets[b] <= i < offsets[b+1] (concatenated
    // galaxies), or, with offsets == nullptr and batch > 1, to element i / p->n and is physical particle i % p->n
    // (the same galaxy seen under `batch` rotations).
    int32_t batch = 1;
    const int64_t *offsets = nullptr;      // HOST [batch + 1]
    // true: empty spaxels get NO work unit (the caller runs k_accumulate with skip_empty: nothing is written for them)
    bool compact_units = false;
};

// Cell order (rubix_telescope.cell_order, spectral_cell.cu): > 0 when the particle pass sorts by (spaxel, SSP cell) -- the
// number of cells, i.e. the multiplier of the composite sort key -- else 0.  *threshold (if given) receives the particle
// count from which a spaxel goes to k_accumulate_cell (0 = every spaxel).
int32_t cell_order_cells(const PassInputs &in, const Layout &L, int32_t *threshold = nullptr);
bool cell_kernel_fits(int32_t n_c, double b_max, bool flux);   // spectral_cell.cu
cudaError_t launch_particle_pass(const PassInputs &in, const Layout &L, char *ws, cudaStream_t st);
cudaError_t launch_bin_only(int64_t n, const float *pos, const float *vel, const rubix_telescope *tel, const float *R,
                            int32_t *key, float *vlos, cudaStream_t st);
// skip_empty: rows of spaxels without particles are NOT written (the masked PSF/LSF passes never read them)
// Mirrors of a spaxel-sharded run: the first / last `rows` detector rows are also stored at lo / hi (nullptr = none)
struct Mirrors { float *lo, *hi; int32_t rows; };
cudaError_t launch_accumulate(const PassInputs &in, const Layout &L, char *ws, float *cube, bool skip_empty,
                              cudaStream_t st, const Mirrors *mirrors = nullptr);
// taps_dev: device scratch of psf_taps_bytes(n_channels) for a wavelength-dependent PSF (reading R18), else unused.
// transpose: apply LSF^T PSF^T (PSF first, then LSF) instead of PSF LSF; only differs when the PSF depends on lambda.
// occ_in / occ_tmp (both or neither; forward order only): occ_in[s] != 0 marks the spaxel rows of `in` that hold data --
// the others are taken as zeros WITHOUT being read (they may be unwritten); occ_tmp [n_s] receives the same
// mask for the temporary after the first pass, so that all-zero rows cross HBM in neither direction.
cudaError_t launch_convolve(const rubix_telescope *tel, const float *in, float *out, float *tmp, float *taps_dev,
                            bool transpose, const uint8_t *occ_in, uint8_t *occ_tmp, cudaStream_t st, int32_t batch = 1);
// true when launch_convolve would take its marching (fast) path, the only one that honours the masks
bool convolve_fast_path(const rubix_telescope *tel, const float *in, const float *out, const float *tmp);
inline size_t psf_taps_bytes(int32_t n_c) { return align_up((size_t)15 * ((size_t)n_c + 2) * 4, 256); }
cudaError_t launch_adjoint(const PassInputs &in, const Layout &L, char *ws, const float *gconv,
                           float *g_mass, float *g_age, float *g_z, float *g_v, cudaStream_t st);

cudaError_t launch_add_noise(const float *in, float *out, int64_t n, float sigma_read, float gain, uint64_t seed,
                             cudaStream_t st);
constexpr int kLossStaticMaxBatch = 64;    // cubes per rubix_residual_loss_static call (size of its file-scope scratch)
// launch_residual_loss with the partials in a file-scope device array (loss.cu): no workspace, no allocation; batch <= 64
cudaError_t launch_residual_loss_static(const float *cube, const float *target, int64_t n_vox, float *grad, double *loss,
                                        cudaStream_t st, int32_t batch);
size_t loss_scratch_bytes(int32_t batch = 1);
cudaError_t launch_residual_loss(const float *cube, const float *target, int64_t n_vox, float *grad,
                                 double *partial, double *loss, cudaStream_t st, int32_t batch = 1);

// Table mode (readings R15 / R16): the rest position of channel k is x_k = Y[k] c + a with a per-launch
// table Y and per-particle (c, a); used for log-sampled SSP grids and for explicit channel wavelengths.
// General-grid mode (reading R21, gen_coord.cuh): listed SSP wavelengths; positions per sample in fp64.  Takes precedence
// over the table mode.
inline bool gen_mode(const rubix_ssp *s, const rubix_telescope *t)
{
    (void)t;
    return s->lambda_grid != nullptr;
}
// Table mode (readings R15 / R16, and R20 for the bin average): log-sampled SSP grid and / or listed channel wavelengths.
inline bool table_mode(const rubix_ssp *s, const rubix_telescope *t)
{
    return !gen_mode(s, t) && (s->log_lambda != 0 || t->lambda_obs != nullptr);
}
// table mode under the bin average: the per-launch table holds the n_c + 1 bin edges; the adjoint is k_adjoint_general
inline bool table_flux(const rubix_ssp *s, const rubix_telescope *t)
{
    return table_mode(s, t) && t->resample == RUBIX_RESAMPLE_FLUX;
}
struct GenGrid;
int gen_kind(const rubix_ssp *s);
// largest span of one channel (point rule: channel to channel; bin average: one bin) in SSP samples, Doppler cap included
double gen_step_max(const rubix_ssp *s, const rubix_telescope *t);
// samples spanned by tc consecutive channels (the table one channel tile needs)
double gen_window_max(const rubix_ssp *s, const rubix_telescope *t, int tc);
void gen_grid_params(const PassInputs &in, const Layout &L, char *ws, GenGrid *G);          // host only
cudaError_t launch_adjoint_general(const PassInputs &in, const Layout &L, char *ws, const float *gconv, float *g_mass,
                                   float *g_age, float *g_z, float *g_v, cudaStream_t st);
cudaError_t launch_gen_setup(const PassInputs &in, const Layout &L, char *ws, cudaStream_t st, GenGrid *G);   // + tables
// largest d x / d channel over the detector, including the largest Doppler stretch (host, fp64)
double table_step_max(const rubix_ssp *s, const rubix_telescope *t);

void make_taps(int size, float sigma, Taps *t);

extern thread_local int g_launches;

// Records a CUDA event pair around a stage when stage timing is on (include/rubix_peaks.h).
class StageTimer {
public:
    StageTimer(int stage, cudaStream_t st);
    ~StageTimer();
private:
    int stage_;
    cudaStream_t st_;
    cudaEvent_t a_;
};

#define RUBIX_LAUNCH_CHECK()                         \
    do {                                             \
        ++::rubix::g_launches;                       \
        cudaError_t e_ = cudaGetLastError();         \
        if (e_ != cudaSuccess) return e_;            \
    } while (0)

// ---- packed fp32x2 arithmetic (sm_100+): one issue slot, two FMAs ------------------------------
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long fmul2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float2 unpack2(unsigned long long v)
{
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}


}  // namespace rubix
