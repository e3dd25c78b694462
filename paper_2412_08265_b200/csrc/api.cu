// C ABI of include/rubix.h: argument validation, workspace carve-up, launches.  No CPU fallback.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <unordered_map>

#include <nvtx3/nvToolsExt.h>

#include "common.cuh"

namespace rubix {
thread_local int g_launches = 0;
}

using namespace rubix;

namespace {

thread_local char t_err[512] = "";

rubix_status fail(rubix_status st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return st;
}

rubix_status cuda_fail(cudaError_t e, const char *where)
{
    return fail(RUBIX_ERR_CUDA, "%s: %s", where, cudaGetErrorString(e));
}

// sort artefacts of the most recently used workspace addresses (bounded: the oldest entry is dropped)
struct Artifacts { const int32_t *key, *perm, *seg_off; uint64_t stamp; };
constexpr size_t kMaxArtifacts = 256;
std::mutex g_mu;
std::unordered_map<const void *, Artifacts> g_artifacts;
uint64_t g_stamp = 0;

// NVTX range around one ABI call (ranges around the compute calls)
struct Range {
    explicit Range(const char *name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
};

rubix_status check_ssp(const rubix_ssp *s, bool flux_required)
{
    if (!s) return fail(RUBIX_ERR_NULL, "ssp is NULL");
    if (s->struct_size != sizeof(rubix_ssp))
        return fail(RUBIX_ERR_INVALID_ARG, "rubix_ssp.struct_size is %u, this library expects %zu (ABI version %d): the "
                    "caller was built against another rubix.h", s->struct_size, sizeof(rubix_ssp), RUBIX_ABI_VERSION);
    if (!s->log_age_axis || !s->log_z_axis || (flux_required && !s->flux))
        return fail(RUBIX_ERR_NULL, "ssp axis / flux pointer is NULL");
    if (s->n_age < 2 || s->n_z < 2 || s->n_lambda < 2)
        return fail(RUBIX_ERR_INVALID_ARG, "ssp grid needs n_age, n_z, n_lambda >= 2");
    if (s->lambda_grid) {                                  // listed rest wavelengths replace lambda0 / dlambda
        if (s->log_lambda != 0)
            return fail(RUBIX_ERR_INVALID_ARG, "ssp lambda_grid (listed wavelengths) and log_lambda = 1 exclude each other");
        for (int j = 0; j < s->n_lambda; ++j)
            if (!(s->lambda_grid[j] > 0.0f) || !isfinite(s->lambda_grid[j]) || (j > 0 && !(s->lambda_grid[j] > s->lambda_grid[j - 1])))
                return fail(RUBIX_ERR_INVALID_ARG, "ssp lambda_grid must be positive, finite and strictly increasing");
    } else if (!(s->dlambda > 0.0f) || !isfinite(s->dlambda) || !isfinite(s->lambda0)) {
        return fail(RUBIX_ERR_INVALID_ARG, "ssp dlambda must be > 0 and finite");
    }
    if (s->log_lambda != 0 && s->log_lambda != 1)
        return fail(RUBIX_ERR_INVALID_ARG, "ssp log_lambda must be 0 or 1");
    if (s->log_lambda == 1 && !(s->lambda0 > 0.0f))
        return fail(RUBIX_ERR_INVALID_ARG, "a log-sampled ssp grid needs lambda0 > 0");
    if (s->n_age > kMaxAge || s->n_z > kMaxZ)
        return fail(RUBIX_ERR_UNSUPPORTED, "ssp axes limited to n_age <= %d, n_z <= %d", kMaxAge, kMaxZ);
    if ((double)s->n_age * s->n_z * s->n_lambda >= 2147483648.0)
        return fail(RUBIX_ERR_UNSUPPORTED, "ssp grid must have fewer than 2^31 samples");
    for (int i = 1; i < s->n_age; ++i)
        if (!(s->log_age_axis[i] > s->log_age_axis[i - 1]))
            return fail(RUBIX_ERR_INVALID_ARG, "log_age_axis must be strictly increasing");
    for (int i = 1; i < s->n_z; ++i)
        if (!(s->log_z_axis[i] > s->log_z_axis[i - 1]))
            return fail(RUBIX_ERR_INVALID_ARG, "log_z_axis must be strictly increasing");
    return RUBIX_OK;
}

rubix_status check_tel(const rubix_telescope *t)
{
    if (!t) return fail(RUBIX_ERR_NULL, "telescope is NULL");
    if (t->struct_size != sizeof(rubix_telescope))
        return fail(RUBIX_ERR_INVALID_ARG, "rubix_telescope.struct_size is %u, this library expects %zu (ABI version %d): "
                    "the caller was built against another rubix.h", t->struct_size, sizeof(rubix_telescope),
                    RUBIX_ABI_VERSION);
    if (t->n_x < 1 || t->n_y < 1 || t->n_channels < 1)
        return fail(RUBIX_ERR_INVALID_ARG, "detector needs n_x, n_y, n_channels >= 1");
    if ((double)t->n_x * t->n_y >= 2147483647.0 / 2 || (double)t->n_x * t->n_y * t->n_channels >= 9.0e15)
        return fail(RUBIX_ERR_UNSUPPORTED, "detector too large");
    if (!(t->spaxel_size > 0.0f) || !isfinite(t->spaxel_size))
        return fail(RUBIX_ERR_INVALID_ARG, "spaxel_size must be > 0");
    if (t->n_x_full < 0 || (t->n_x_full > 0 && (t->x_first < 0 || (int64_t)t->x_first + t->n_x > t->n_x_full)))
        return fail(RUBIX_ERR_INVALID_ARG, "row window: need 0 <= x_first and x_first + n_x <= n_x_full");
    if (t->n_x_full == 0 && t->x_first != 0)
        return fail(RUBIX_ERR_INVALID_ARG, "x_first needs n_x_full > 0");
    if (t->cell_order < 0 || t->cell_order > 3) return fail(RUBIX_ERR_INVALID_ARG, "cell_order must be 0 (auto), 1 (off), 2 (on) or 3 (all)");
    if (!(t->dlambda > 0.0f) || !isfinite(t->dlambda) || !isfinite(t->lambda0))
        return fail(RUBIX_ERR_INVALID_ARG, "telescope dlambda must be > 0 and finite");
    if (t->resample != RUBIX_RESAMPLE_POINT && t->resample != RUBIX_RESAMPLE_FLUX)
        return fail(RUBIX_ERR_INVALID_ARG, "resample must be RUBIX_RESAMPLE_POINT (0) or RUBIX_RESAMPLE_FLUX (1)");
    if (!(t->redshift >= 0.0f) || !(t->redshift <= 20.0f))
        return fail(RUBIX_ERR_INVALID_ARG, "redshift must be in [0, 20]");
    if (!(t->flux_scale > 0.0f) || !isfinite(t->flux_scale))
        return fail(RUBIX_ERR_INVALID_ARG, "flux_scale must be > 0 and finite (1 = no scaling)");
    if (t->psf_alpha != 0.0f && t->psf_size > 0) {
        if (!isfinite(t->psf_alpha) || fabsf(t->psf_alpha) > 4.0f || !(t->psf_lambda_ref > 0.0f) || !isfinite(t->psf_lambda_ref))
            return fail(RUBIX_ERR_INVALID_ARG, "psf_alpha must be finite with |psf_alpha| <= 4 and psf_lambda_ref > 0");
        if (t->psf_size > 15 || t->lsf_size > 9 || (t->n_channels % 2) != 0)
            return fail(RUBIX_ERR_UNSUPPORTED,
                        "a wavelength-dependent PSF needs psf_size <= 15, lsf_size <= 9 and an even n_channels");
        if (!t->lambda_obs && !((double)t->lambda0 > 0.0 && (double)t->lambda0 + (double)t->dlambda * (t->n_channels - 1) > 0.0))
            return fail(RUBIX_ERR_INVALID_ARG, "a wavelength-dependent PSF needs positive channel wavelengths");
    }
    if (t->lambda_obs) {
        if (t->resample == RUBIX_RESAMPLE_FLUX && t->n_channels < 2)
            return fail(RUBIX_ERR_INVALID_ARG, "the bin average on listed channel wavelengths needs n_channels >= 2");
        for (int k = 0; k < t->n_channels; ++k)
            if (!(t->lambda_obs[k] > 0.0f) || !isfinite(t->lambda_obs[k]) || (k > 0 && !(t->lambda_obs[k] > t->lambda_obs[k - 1])))
                return fail(RUBIX_ERR_INVALID_ARG, "lambda_obs must be positive, finite and strictly increasing");
    }
    const int sz[2] = {t->psf_size, t->lsf_size};
    const float sg[2] = {t->psf_sigma, t->lsf_sigma};
    for (int i = 0; i < 2; ++i) {
        if (sz[i] < 0 || (sz[i] > 0 && sz[i] % 2 == 0))
            return fail(RUBIX_ERR_INVALID_ARG, "stencil sizes must be 0 or odd");
        if (sz[i] > kMaxTaps) return fail(RUBIX_ERR_UNSUPPORTED, "stencil sizes limited to %d taps", kMaxTaps);
        if (sz[i] > 0 && (!(sg[i] > 0.0f) || !isfinite(sg[i])))
            return fail(RUBIX_ERR_INVALID_ARG, "stencil sigma must be > 0");
    }
    return RUBIX_OK;
}

rubix_status check_particles(const rubix_particles *p)
{
    if (!p) return fail(RUBIX_ERR_NULL, "particles is NULL");
    if (p->n < 0) return fail(RUBIX_ERR_INVALID_ARG, "n must be >= 0");
    if (p->n >= 2147483647LL) return fail(RUBIX_ERR_UNSUPPORTED, "n limited to < 2^31 particles");
    if (p->n > 0 && (!p->pos || !p->vel || !p->mass || !p->log_age || !p->log_z))
        return fail(RUBIX_ERR_NULL, "a particle array is NULL");
    return RUBIX_OK;
}

rubix_status check_resampler(const rubix_ssp *s, const rubix_telescope *t)
{
    if (gen_mode(s, t)) {                                  // readings R20 / R21: positions per sample in fp64
        const bool fl = t->resample == RUBIX_RESAMPLE_FLUX;
        const double first = t->lambda_obs ? (double)t->lambda_obs[0] - (fl ? 0.5 * ((double)t->lambda_obs[1] - (double)t->lambda_obs[0]) : 0.0)
                                           : (double)t->lambda0 - (fl ? 0.5 * (double)t->dlambda : 0.0);
        if (!(first > 0.0)) return fail(RUBIX_ERR_INVALID_ARG, "observed wavelengths (bin edges included) must be > 0");
        const double b0 = gen_step_max(s, t);
        if (!(b0 < 14.25))
            return fail(RUBIX_ERR_UNSUPPORTED, "one channel spans %.3f SSP samples: outside the resampler range (< 14.25)", b0);
        return RUBIX_OK;
    }
    if (table_mode(s, t)) {
        const bool fl = t->resample == RUBIX_RESAMPLE_FLUX;
        const double first = t->lambda_obs ? (double)t->lambda_obs[0] - (fl ? 0.5 * ((double)t->lambda_obs[1] - (double)t->lambda_obs[0]) : 0.0)
                                           : (double)t->lambda0 - (fl ? 0.5 * (double)t->dlambda : 0.0);
        if (!(first > 0.0)) return fail(RUBIX_ERR_INVALID_ARG, "observed wavelengths (bin edges included) must be > 0");
        const double b0 = table_step_max(s, t);
        if (!(b0 < 14.25))
            return fail(RUBIX_ERR_UNSUPPORTED, "d x / d channel = %.3f is outside the resampler range (< 14.25)", b0);
        return RUBIX_OK;
    }
    const double b_max = (double)t->dlambda / (double)s->dlambda / (1.0 - kBetaCap);
    if (b_max >= 15.0)
        return fail(RUBIX_ERR_UNSUPPORTED, "dlambda_obs / dlambda_ssp = %.3f is outside the resampler range (< 14.25)",
                    (double)t->dlambda / (double)s->dlambda);
    return RUBIX_OK;
}

rubix_status check_ws(const void *ws, size_t have, size_t need)
{
    if (!ws) return fail(RUBIX_ERR_WORKSPACE, "workspace is NULL");
    if (((uintptr_t)ws & 255u) != 0) return fail(RUBIX_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    if (have < need) return fail(RUBIX_ERR_WORKSPACE, "workspace has %zu bytes, needs %zu", have, need);
    return RUBIX_OK;
}

void remember(const void *ws, const Layout &L)
{
    const char *b = (const char *)ws;
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_artifacts.size() >= kMaxArtifacts && g_artifacts.find(ws) == g_artifacts.end()) {
        auto oldest = g_artifacts.begin();
        for (auto it = g_artifacts.begin(); it != g_artifacts.end(); ++it)
            if (it->second.stamp < oldest->second.stamp) oldest = it;
        g_artifacts.erase(oldest);
    }
    g_artifacts[ws] = Artifacts{(const int32_t *)(b + L.off_key),
                                (const int32_t *)(b + L.off_permbuf[L.final_buf]),
                                (const int32_t *)(b + L.off_seg), ++g_stamp};
}

}  // namespace

extern "C" {

const char *rubix_last_error(void) { return t_err; }
uint32_t rubix_abi_version(void) { return RUBIX_ABI_VERSION; }
int32_t rubix_last_launch_count(void) { return g_launches; }

size_t rubix_workspace_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel)
{
    t_err[0] = 0;
    if (n < 0 || n >= 2147483647LL) { fail(RUBIX_ERR_INVALID_ARG, "n out of range"); return 0; }
    if (check_tel(tel) != RUBIX_OK) return 0;
    if (ssp && ssp->struct_size != sizeof(rubix_ssp)) {
        fail(RUBIX_ERR_INVALID_ARG, "rubix_ssp.struct_size is %u, this library expects %zu", ssp->struct_size, sizeof(rubix_ssp));
        return 0;
    }
    if (ssp && (ssp->n_age < 2 || ssp->n_z < 2 || ssp->n_lambda < 2)) {
        fail(RUBIX_ERR_INVALID_ARG, "ssp grid needs n_age, n_z, n_lambda >= 2");
        return 0;
    }
    return make_layout(n, tel->n_x * tel->n_y, tel->n_channels, ssp ? ssp->n_age * ssp->n_z : 0,
                       ssp ? ssp->n_lambda : 0).bytes_total;
}

rubix_status rubix_build_cube(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                              const float *R, float *cube, void *workspace, size_t workspace_bytes,
                              void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_build_cube");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !cube) return fail(RUBIX_ERR_NULL, "R or cube is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    const Layout L = make_layout(p->n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z,
                                 ssp->n_lambda);
    if ((s = check_ws(workspace, workspace_bytes, L.bytes_total)) != RUBIX_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    PassInputs in{p, ssp, tel, R};
    cudaError_t e;
    {
        StageTimer t(0, st);
        e = launch_particle_pass(in, L, (char *)workspace, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "particle pass");
    e = launch_accumulate(in, L, (char *)workspace, cube, false, st);
    if (e != cudaSuccess) return cuda_fail(e, "accumulate");
    remember(workspace, L);
    return RUBIX_OK;
}

rubix_status rubix_bin_particles(int64_t n, const float *pos, const float *vel, const rubix_telescope *tel, const float *R,
                                 int32_t *key, float *vlos, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_bin_particles");
    g_launches = 0;
    rubix_status s;
    if (n < 0 || n >= 2147483647LL) return fail(RUBIX_ERR_INVALID_ARG, "n out of range");
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || (n > 0 && (!pos || !vel || !key))) return fail(RUBIX_ERR_NULL, "R, pos, vel or key is NULL");
    cudaError_t e = launch_bin_only(n, pos, vel, tel, R, key, vlos, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "bin");
    return RUBIX_OK;
}

rubix_status rubix_build_cube_mirrored(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                                       const float *R, float *cube, float *mirror_lo, float *mirror_hi, int32_t mirror_rows,
                                       void *workspace, size_t workspace_bytes, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_build_cube_mirrored");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !cube) return fail(RUBIX_ERR_NULL, "R or cube is NULL");
    if ((mirror_lo || mirror_hi) && (mirror_rows < 1 || mirror_rows > tel->n_x))
        return fail(RUBIX_ERR_INVALID_ARG, "mirror_rows must be in [1, n_x] when a mirror is given");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    const Layout L = make_layout(p->n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda);
    if ((s = check_ws(workspace, workspace_bytes, L.bytes_total)) != RUBIX_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    PassInputs in{p, ssp, tel, R};
    cudaError_t e;
    {
        StageTimer t(0, st);
        e = launch_particle_pass(in, L, (char *)workspace, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "particle pass");
    const Mirrors m{mirror_lo, mirror_hi, mirror_rows};
    e = launch_accumulate(in, L, (char *)workspace, cube, false, st, (mirror_lo || mirror_hi) ? &m : nullptr);
    if (e != cudaSuccess) return cuda_fail(e, "accumulate");
    remember(workspace, L);
    return RUBIX_OK;
}

// Steps 1-8 on device buffers.  With the marching PSF/LSF kernels the raw cube lives in the workspace and only the
// rows of occupied spaxels are written and read (launch_convolve's masks); otherwise the two plain stages run.
static rubix_status forward_device(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                                   const float *R, float *cube_out, const Layout &L, char *ws, cudaStream_t st,
                                   int32_t batch = 1, const int64_t *offsets = nullptr)
{
    PassInputs in{p, ssp, tel, R, batch, offsets};
    const bool conv = tel->psf_size > 0 || tel->lsf_size > 0;
    float *raw = (float *)(ws + L.off_cube_a), *tmp = (float *)(ws + L.off_cube_b);
    const bool sparse = conv && convolve_fast_path(tel, raw, cube_out, tmp);
    in.compact_units = sparse;                             // empty spaxels then need no work unit at all
    cudaError_t e;
    {
        StageTimer t(0, st);
        e = launch_particle_pass(in, L, ws, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "particle pass");
    if (!conv) {
        e = launch_accumulate(in, L, ws, cube_out, false, st);
        if (e != cudaSuccess) return cuda_fail(e, "accumulate");
        return RUBIX_OK;
    }
    e = launch_accumulate(in, L, ws, raw, sparse, st);
    if (e != cudaSuccess) return cuda_fail(e, "accumulate");
    {
        StageTimer t(3, st);
        e = launch_convolve(tel, raw, cube_out, tmp, (float *)(ws + L.off_psftaps), false,
                            sparse ? (const uint8_t *)(ws + L.off_occ[0]) : nullptr,
                            sparse ? (uint8_t *)(ws + L.off_occ[1]) : nullptr, st, batch);
    }
    if (e != cudaSuccess) return cuda_fail(e, "convolve");
    return RUBIX_OK;
}

// logical particles of the largest group of <= kMaxBatch elements, and that group's element count
static void batch_groups(int64_t n, int32_t batch, const int64_t *offsets, int64_t *n_max, int32_t *b_max)
{
    *b_max = batch < kMaxBatch ? batch : kMaxBatch;
    if (!offsets) { *n_max = n * *b_max; return; }
    int64_t m = 0;
    for (int32_t g0 = 0; g0 < batch; g0 += kMaxBatch) {
        const int32_t g1 = g0 + kMaxBatch < batch ? g0 + kMaxBatch : batch;
        if (offsets[g1] - offsets[g0] > m) m = offsets[g1] - offsets[g0];
    }
    *n_max = m;
}

static rubix_status check_batch(const rubix_particles *p, const int64_t *offsets, int32_t batch, const rubix_telescope *tel)
{
    if (batch < 1) return fail(RUBIX_ERR_INVALID_ARG, "batch must be >= 1");
    const int32_t bg = batch < kMaxBatch ? batch : kMaxBatch;
    if ((double)bg * tel->n_x * tel->n_y >= 2147483647.0 / 2)
        return fail(RUBIX_ERR_UNSUPPORTED, "batch x spaxels too large for one key space");
    if (offsets) {
        if (offsets[0] != 0 || offsets[batch] != p->n)
            return fail(RUBIX_ERR_INVALID_ARG, "offsets[0] must be 0 and offsets[batch] must equal particles->n");
        for (int32_t b = 0; b < batch; ++b)
            if (offsets[b + 1] < offsets[b]) return fail(RUBIX_ERR_INVALID_ARG, "offsets must be non-decreasing");
    } else if ((double)p->n * bg >= 2147483647.0) {
        return fail(RUBIX_ERR_UNSUPPORTED, "batch x particles must stay below 2^31 per group of %d elements", kMaxBatch);
    }
    return RUBIX_OK;
}

size_t rubix_forward_batched_workspace_bytes(int64_t n, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                             const rubix_telescope *tel)
{
    t_err[0] = 0;
    if (n < 0 || n >= 2147483647LL) { fail(RUBIX_ERR_INVALID_ARG, "n out of range"); return 0; }
    if (check_tel(tel) != RUBIX_OK || check_ssp(ssp, false) != RUBIX_OK) return 0;
    rubix_particles fake{n, nullptr, nullptr, nullptr, nullptr, nullptr};
    if (check_batch(&fake, offsets, batch, tel) != RUBIX_OK) return 0;
    int64_t n_max; int32_t b_max;
    batch_groups(n, batch, offsets, &n_max, &b_max);
    return make_layout(n_max, b_max * tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda).bytes_total;
}

rubix_status rubix_forward_batched(const rubix_particles *p, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                   const rubix_telescope *tel, const float *R, float *cubes, void *workspace,
                                   size_t workspace_bytes, void *stream)
{
    Range nvtx_range("rubix_forward_batched");
    t_err[0] = 0;
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !cubes) return fail(RUBIX_ERR_NULL, "R or cubes is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    if ((s = check_batch(p, offsets, batch, tel)) != RUBIX_OK) return s;
    int64_t n_max; int32_t b_max;
    batch_groups(p->n, batch, offsets, &n_max, &b_max);
    const int32_t n_s = tel->n_x * tel->n_y;
    const Layout Lmax = make_layout(n_max, b_max * n_s, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda);
    if ((s = check_ws(workspace, workspace_bytes, Lmax.bytes_total)) != RUBIX_OK) return s;
    const size_t cube_elems = (size_t)n_s * tel->n_channels;
    const char *c0 = (const char *)cubes, *w0 = (const char *)workspace;
    if (c0 < w0 + Lmax.bytes_total && w0 < c0 + cube_elems * 4 * (size_t)batch)
        return fail(RUBIX_ERR_INVALID_ARG, "cubes overlap the workspace");
    int launches = 0;
    for (int32_t g0 = 0; g0 < batch; g0 += kMaxBatch) {       // groups of <= kMaxBatch elements, one launch sequence each
        const int32_t bg = g0 + kMaxBatch < batch ? kMaxBatch : batch - g0;
        rubix_particles pg = *p;
        int64_t off_local[kMaxBatch + 1];
        if (offsets) {
            const int64_t first = offsets[g0];
            pg.n = offsets[g0 + bg] - first;
            pg.pos = p->pos ? p->pos + 3 * first : nullptr;
            pg.vel = p->vel ? p->vel + 3 * first : nullptr;
            pg.mass = p->mass ? p->mass + first : nullptr;
            pg.log_age = p->log_age ? p->log_age + first : nullptr;
            pg.log_z = p->log_z ? p->log_z + first : nullptr;
            for (int32_t b = 0; b <= bg; ++b) off_local[b] = offsets[g0 + b] - first;
        }
        const int64_t n_logical = offsets ? pg.n : p->n * bg;
        const Layout L = make_layout(n_logical, bg * n_s, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda);
        s = forward_device(&pg, ssp, tel, R + 9 * (size_t)g0, cubes + cube_elems * (size_t)g0, L, (char *)workspace,
                           (cudaStream_t)stream, bg, offsets ? off_local : nullptr);
        if (s != RUBIX_OK) return s;
        launches += g_launches;
        g_launches = 0;
        remember(workspace, L);
    }
    g_launches = launches;
    return RUBIX_OK;
}

rubix_status rubix_forward(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                           const float *R, float *cube, void *workspace, size_t workspace_bytes, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_forward");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !cube) return fail(RUBIX_ERR_NULL, "R or cube is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    const Layout L = make_layout(p->n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z,
                                 ssp->n_lambda);
    if ((s = check_ws(workspace, workspace_bytes, L.bytes_total)) != RUBIX_OK) return s;
    const char *c0 = (const char *)cube, *w0 = (const char *)workspace;
    if (c0 < w0 + L.bytes_total && w0 < c0 + (size_t)tel->n_x * tel->n_y * tel->n_channels * 4)
        return fail(RUBIX_ERR_INVALID_ARG, "cube overlaps the workspace");
    if ((s = forward_device(p, ssp, tel, R, cube, L, (char *)workspace, (cudaStream_t)stream)) != RUBIX_OK) return s;
    remember(workspace, L);
    return RUBIX_OK;
}

rubix_status rubix_convolve_psf_lsf(const rubix_telescope *tel, const float *cube_in, float *cube_out,
                                    void *workspace, size_t workspace_bytes, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_convolve_psf_lsf");
    g_launches = 0;
    rubix_status s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!cube_in || !cube_out) return fail(RUBIX_ERR_NULL, "cube_in or cube_out is NULL");
    const size_t cube_bytes = (size_t)tel->n_x * tel->n_y * tel->n_channels * 4;
    const char *a = (const char *)cube_in, *b = (const char *)cube_out;
    if (a < b + cube_bytes && b < a + cube_bytes)
        return fail(RUBIX_ERR_INVALID_ARG, "cube_in and cube_out overlap");
    float *tmp = nullptr, *taps = nullptr;
    if (tel->psf_size > 0) {
        const bool var = tel->psf_alpha != 0.0f;
        // first cube buffer = the temporary; the per-channel taps live behind BOTH cube buffers (make_layout), so a
        // workspace shared with rubix_build_cube keeps its sort artefacts
        const size_t need = var ? 2 * align_up(cube_bytes, 256) + psf_taps_bytes(tel->n_channels) : align_up(cube_bytes, 256);
        if ((s = check_ws(workspace, workspace_bytes, need)) != RUBIX_OK) return s;
        tmp = (float *)workspace;
        if (var) taps = (float *)((char *)workspace + 2 * align_up(cube_bytes, 256));
    }
    cudaError_t e;
    {
        StageTimer t(3, (cudaStream_t)stream);
        e = launch_convolve(tel, cube_in, cube_out, tmp, taps, false, nullptr, nullptr, (cudaStream_t)stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, "convolve");
    return RUBIX_OK;
}

rubix_status rubix_cube_adjoint(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                                const float *R, const float *grad_cube, float *g_mass, float *g_log_age,
                                float *g_log_z, float *g_vlos, void *workspace, size_t workspace_bytes,
                                void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_cube_adjoint");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !grad_cube) return fail(RUBIX_ERR_NULL, "R or grad_cube is NULL");
    if (p->n > 0 && (!g_mass || !g_log_age || !g_log_z || !g_vlos))
        return fail(RUBIX_ERR_NULL, "a gradient output is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    const Layout L = make_layout(p->n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z,
                                 ssp->n_lambda);
    if ((s = check_ws(workspace, workspace_bytes, L.bytes_total)) != RUBIX_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    PassInputs in{p, ssp, tel, R};
    cudaError_t e;
    {
        StageTimer t(0, st);
        e = launch_particle_pass(in, L, ws, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "particle pass");
    // G' = LSF^T PSF^T G: zero-padded symmetric stencils are self-adjoint
    const float *gconv = grad_cube;
    if (tel->psf_size > 0 || tel->lsf_size > 0) {
        {
            StageTimer t(3, st);
            e = launch_convolve(tel, grad_cube, (float *)(ws + L.off_cube_a), (float *)(ws + L.off_cube_b),
                                (float *)(ws + L.off_psftaps), true, nullptr, nullptr, st);
        }
        if (e != cudaSuccess) return cuda_fail(e, "adjoint convolve");
        gconv = (const float *)(ws + L.off_cube_a);
    }
    {
        StageTimer t(4, st);
        e = launch_adjoint(in, L, ws, gconv, g_mass, g_log_age, g_log_z, g_vlos, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "adjoint");
    remember(workspace, L);
    return RUBIX_OK;
}

size_t rubix_loss_and_grad_workspace_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel)
{
    const size_t base = rubix_workspace_bytes(n, ssp, tel);
    if (base == 0) return 0;
    const size_t cube_bytes = (size_t)tel->n_x * tel->n_y * tel->n_channels * 4;
    return base + align_up(cube_bytes, 256) + loss_scratch_bytes();
}

rubix_status rubix_loss_and_grad(const rubix_particles *p, const rubix_ssp *ssp, const rubix_telescope *tel,
                                 const float *R, const float *target, double *loss, float *cube_out,
                                 float *g_mass, float *g_log_age, float *g_log_z, float *g_vlos,
                                 void *workspace, size_t workspace_bytes, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_loss_and_grad");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !target || !loss) return fail(RUBIX_ERR_NULL, "R, target or loss is NULL");
    if (p->n > 0 && (!g_mass || !g_log_age || !g_log_z || !g_vlos))
        return fail(RUBIX_ERR_NULL, "a gradient output is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    const Layout L = make_layout(p->n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z,
                                 ssp->n_lambda);
    const int64_t n_vox = (int64_t)tel->n_x * tel->n_y * tel->n_channels;
    const size_t cube_al = align_up((size_t)n_vox * 4, 256);
    if ((s = check_ws(workspace, workspace_bytes, L.bytes_total + cube_al + loss_scratch_bytes())) != RUBIX_OK)
        return s;
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    float *buf_a = (float *)(ws + L.off_cube_a), *buf_b = (float *)(ws + L.off_cube_b);
    float *buf_c = (float *)(ws + L.bytes_total);
    double *partial = (double *)(ws + L.bytes_total + cube_al);
    const bool conv = tel->psf_size > 0 || tel->lsf_size > 0;
    PassInputs in{p, ssp, tel, R};
    cudaError_t e;
    {
        StageTimer t(0, st);
        e = launch_particle_pass(in, L, ws, st);           // ONE particle pass serves forward and adjoint
    }
    if (e != cudaSuccess) return cuda_fail(e, "particle pass");
    // forward: raw cube, then PSF/LSF
    float *raw = conv ? buf_a : (cube_out ? cube_out : buf_a);
    float *fin = cube_out ? cube_out : buf_c;
    const bool sparse = conv && convolve_fast_path(tel, raw, fin, buf_b);   // only occupied rows cross HBM
    e = launch_accumulate(in, L, ws, raw, sparse, st);
    if (e != cudaSuccess) return cuda_fail(e, "accumulate");
    const float *final_cube = raw;
    if (conv) {
        {
            StageTimer t(3, st);
            e = launch_convolve(tel, raw, fin, buf_b, (float *)(ws + L.off_psftaps), false,
                                sparse ? (const uint8_t *)(ws + L.off_occ[0]) : nullptr,
                                sparse ? (uint8_t *)(ws + L.off_occ[1]) : nullptr, st);
        }
        if (e != cudaSuccess) return cuda_fail(e, "convolve");
        final_cube = fin;
    }
    // loss and upstream gradient 2 (cube - target); the raw cube is no longer needed when conv is on
    float *grad = conv ? buf_a : buf_b;
    e = launch_residual_loss(final_cube, target, n_vox, grad, partial, loss, st);
    if (e != cudaSuccess) return cuda_fail(e, "loss");
    const float *gconv = grad;
    if (conv) {                                            // G' = LSF^T PSF^T G (self-adjoint stencils)
        {
            StageTimer t(3, st);
            e = launch_convolve(tel, grad, buf_c, buf_b, (float *)(ws + L.off_psftaps), true, nullptr, nullptr, st);   // buf_c is free
        }
        if (e != cudaSuccess) return cuda_fail(e, "adjoint convolve");
        gconv = buf_c;
    }
    {
        StageTimer t(4, st);
        e = launch_adjoint(in, L, ws, gconv, g_mass, g_log_age, g_log_z, g_vlos, st);
    }
    if (e != cudaSuccess) return cuda_fail(e, "adjoint");
    remember(workspace, L);
    return RUBIX_OK;
}

size_t rubix_loss_and_grad_batched_workspace_bytes(int64_t n, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                                   const rubix_telescope *tel)
{
    const size_t base = rubix_forward_batched_workspace_bytes(n, offsets, batch, ssp, tel);
    if (base == 0) return 0;
    if (!offsets) { fail(RUBIX_ERR_INVALID_ARG, "rubix_loss_and_grad_batched needs offsets (concatenated galaxies)"); return 0; }
    const int32_t bg = batch < kMaxBatch ? batch : kMaxBatch;
    const size_t cube_bytes = (size_t)bg * tel->n_x * tel->n_y * tel->n_channels * 4;
    return base + align_up(cube_bytes, 256) + loss_scratch_bytes(bg);
}

rubix_status rubix_loss_and_grad_batched(const rubix_particles *p, const int64_t *offsets, int32_t batch, const rubix_ssp *ssp,
                                         const rubix_telescope *tel, const float *R, const float *targets, double *loss,
                                         float *cubes_out, float *g_mass, float *g_log_age, float *g_log_z, float *g_vlos,
                                         void *workspace, size_t workspace_bytes, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_loss_and_grad_batched");
    g_launches = 0;
    rubix_status s;
    if ((s = check_particles(p)) != RUBIX_OK) return s;
    if ((s = check_ssp(ssp, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !targets || !loss) return fail(RUBIX_ERR_NULL, "R, targets or loss is NULL");
    if (!offsets) return fail(RUBIX_ERR_INVALID_ARG, "rubix_loss_and_grad_batched needs offsets (concatenated galaxies)");
    if (p->n > 0 && (!g_mass || !g_log_age || !g_log_z || !g_vlos))
        return fail(RUBIX_ERR_NULL, "a gradient output is NULL");
    if ((s = check_resampler(ssp, tel)) != RUBIX_OK) return s;
    if ((s = check_batch(p, offsets, batch, tel)) != RUBIX_OK) return s;
    int64_t n_max; int32_t b_max;
    batch_groups(p->n, batch, offsets, &n_max, &b_max);
    const int32_t n_s = tel->n_x * tel->n_y;
    const Layout Lmax = make_layout(n_max, b_max * n_s, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda);
    const int64_t n_vox = (int64_t)n_s * tel->n_channels;
    const size_t cube_al = align_up((size_t)b_max * n_vox * 4, 256);
    if ((s = check_ws(workspace, workspace_bytes, Lmax.bytes_total + cube_al + loss_scratch_bytes(b_max))) != RUBIX_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    const bool conv = tel->psf_size > 0 || tel->lsf_size > 0;
    int launches = 0;
    for (int32_t g0 = 0; g0 < batch; g0 += kMaxBatch) {       // groups of <= kMaxBatch elements, one launch sequence each
        const int32_t bg = g0 + kMaxBatch < batch ? kMaxBatch : batch - g0;
        const int64_t first = offsets[g0];
        rubix_particles pg = *p;
        pg.n = offsets[g0 + bg] - first;
        pg.pos = p->pos ? p->pos + 3 * first : nullptr;
        pg.vel = p->vel ? p->vel + 3 * first : nullptr;
        pg.mass = p->mass ? p->mass + first : nullptr;
        pg.log_age = p->log_age ? p->log_age + first : nullptr;
        pg.log_z = p->log_z ? p->log_z + first : nullptr;
        int64_t off_local[kMaxBatch + 1];
        for (int32_t b = 0; b <= bg; ++b) off_local[b] = offsets[g0 + b] - first;
        const Layout L = make_layout(pg.n, bg * n_s, tel->n_channels, ssp->n_age * ssp->n_z, ssp->n_lambda);
        float *buf_a = (float *)(ws + L.off_cube_a), *buf_b = (float *)(ws + L.off_cube_b);
        float *buf_c = (float *)(ws + Lmax.bytes_total);
        double *partial = (double *)(ws + Lmax.bytes_total + cube_al);
        PassInputs in{&pg, ssp, tel, R + 9 * (size_t)g0, bg, off_local};
        const float *target = targets + (size_t)g0 * n_vox;
        float *cube_g = cubes_out ? cubes_out + (size_t)g0 * n_vox : nullptr;
        float *raw = conv ? buf_a : (cube_g ? cube_g : buf_a);
        float *fin = cube_g ? cube_g : buf_c;
        const bool sparse = conv && convolve_fast_path(tel, raw, fin, buf_b);
        in.compact_units = false;                          // the adjoint kernels walk the same units
        cudaError_t e;
        {
            StageTimer t(0, st);
            e = launch_particle_pass(in, L, ws, st);       // ONE particle pass serves forward and adjoint of every element
        }
        if (e != cudaSuccess) return cuda_fail(e, "particle pass");
        e = launch_accumulate(in, L, ws, raw, sparse, st);
        if (e != cudaSuccess) return cuda_fail(e, "accumulate");
        const float *final_cube = raw;
        if (conv) {
            {
                StageTimer t(3, st);
                e = launch_convolve(tel, raw, fin, buf_b, (float *)(ws + L.off_psftaps), false,
                                    sparse ? (const uint8_t *)(ws + L.off_occ[0]) : nullptr,
                                    sparse ? (uint8_t *)(ws + L.off_occ[1]) : nullptr, st, bg);
            }
            if (e != cudaSuccess) return cuda_fail(e, "convolve");
            final_cube = fin;
        }
        float *grad = conv ? buf_a : buf_b;
        e = launch_residual_loss(final_cube, target, n_vox, grad, partial, loss + g0, st, bg);
        if (e != cudaSuccess) return cuda_fail(e, "loss");
        const float *gconv = grad;
        if (conv) {
            {
                StageTimer t(3, st);
                e = launch_convolve(tel, grad, buf_c, buf_b, (float *)(ws + L.off_psftaps), true, nullptr, nullptr, st, bg);
            }
            if (e != cudaSuccess) return cuda_fail(e, "adjoint convolve");
            gconv = buf_c;
        }
        {
            StageTimer t(4, st);
            e = launch_adjoint(in, L, ws, gconv, g_mass + first, g_log_age + first, g_log_z + first, g_vlos + first, st);
        }
        if (e != cudaSuccess) return cuda_fail(e, "adjoint");
        launches += g_launches;
        g_launches = 0;
        remember(workspace, L);
    }
    g_launches = launches;
    return RUBIX_OK;
}

rubix_status rubix_add_noise(const float *cube_in, float *cube_out, int64_t n_voxels, float sigma_read, float gain,
                             uint64_t seed, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_add_noise");
    g_launches = 0;
    if (n_voxels < 0) return fail(RUBIX_ERR_INVALID_ARG, "n_voxels must be >= 0");
    if (n_voxels > 0 && (!cube_in || !cube_out)) return fail(RUBIX_ERR_NULL, "cube_in or cube_out is NULL");
    if (!(sigma_read >= 0.0f) || !isfinite(sigma_read) || !(gain >= 0.0f) || !isfinite(gain))
        return fail(RUBIX_ERR_INVALID_ARG, "sigma_read and gain must be >= 0 and finite");
    if (cube_in != cube_out) {
        const char *a = (const char *)cube_in, *b = (const char *)cube_out;
        if (a < b + (size_t)n_voxels * 4 && b < a + (size_t)n_voxels * 4)
            return fail(RUBIX_ERR_INVALID_ARG, "cube_in and cube_out overlap (in place needs cube_in == cube_out)");
    }
    cudaError_t e = launch_add_noise(cube_in, cube_out, n_voxels, sigma_read, gain, seed, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "noise");
    return RUBIX_OK;
}

rubix_status rubix_residual_loss_static(const float *cubes, const float *targets, int64_t n_voxels, int32_t batch,
                                        float *grads, double *loss, void *stream)
{
    t_err[0] = 0;
    Range nvtx_range("rubix_residual_loss_static");
    g_launches = 0;
    if (n_voxels < 0) return fail(RUBIX_ERR_INVALID_ARG, "n_voxels must be >= 0");
    if (batch < 1) return fail(RUBIX_ERR_INVALID_ARG, "batch must be >= 1");
    if (batch > RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH)
        return fail(RUBIX_ERR_UNSUPPORTED, "batch = %d exceeds the %d cubes the static scratch of rubix_residual_loss_static holds "
                    "(split the call, or use rubix_loss_and_grad_batched with a workspace)", batch,
                    RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH);
    if (!loss) return fail(RUBIX_ERR_NULL, "loss is NULL");
    if (n_voxels > 0 && (!cubes || !targets || !grads)) return fail(RUBIX_ERR_NULL, "cubes, targets or grads is NULL");
    static_assert(RUBIX_RESIDUAL_LOSS_STATIC_MAX_BATCH == kLossStaticMaxBatch, "header and scratch size disagree");
    cudaError_t e = launch_residual_loss_static(cubes, targets, n_voxels, grads, loss, (cudaStream_t)stream, batch);
    if (e != cudaSuccess) return cuda_fail(e, "residual loss (static scratch)");
    return RUBIX_OK;
}

rubix_status rubix_get_sort_artifacts(const void *workspace, const int32_t **key, const int32_t **perm,
                                      const int32_t **seg_off)
{
    t_err[0] = 0;
    if (!workspace || !key || !perm || !seg_off) return fail(RUBIX_ERR_NULL, "NULL argument");
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_artifacts.find(workspace);
    if (it == g_artifacts.end())
        return fail(RUBIX_ERR_INVALID_ARG, "no rubix_build_cube / rubix_cube_adjoint call has used this workspace");
    *key = it->second.key;
    *perm = it->second.perm;
    *seg_off = it->second.seg_off;
    return RUBIX_OK;
}

// ---- end-to-end entry with host buffers ------------------------------------------------------
namespace {
struct HostLayout { size_t pos, vel, mass, age, z, flux, cube, cube2, ws, total; };
HostLayout host_layout(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel)
{
    HostLayout H{};
    size_t off = 0;
    auto take = [&](size_t b) { size_t o = off; off = align_up(off + b, 256); return o; };
    const size_t nn = (size_t)(n > 0 ? n : 1);
    H.pos = take(nn * 12);
    H.vel = take(nn * 12);
    H.mass = take(nn * 4);
    H.age = take(nn * 4);
    H.z = take(nn * 4);
    H.flux = take((size_t)ssp->n_age * ssp->n_z * ssp->n_lambda * 4);
    const size_t cube = (size_t)tel->n_x * tel->n_y * tel->n_channels * 4;
    H.cube = take(cube);
    H.cube2 = take(cube);
    H.ws = off;
    H.total = off + make_layout(n, tel->n_x * tel->n_y, tel->n_channels, ssp->n_age * ssp->n_z,
                                ssp->n_lambda).bytes_total;
    return H;
}
}  // namespace

size_t rubix_forward_host_scratch_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel)
{
    t_err[0] = 0;
    if (n < 0 || n >= 2147483647LL || !ssp || check_tel(tel) != RUBIX_OK || ssp->struct_size != sizeof(rubix_ssp) ||
        ssp->n_age < 2 || ssp->n_z < 2 || ssp->n_lambda < 2) {
        if (!t_err[0]) fail(RUBIX_ERR_INVALID_ARG, "bad arguments");
        return 0;
    }
    return host_layout(n, ssp, tel).total;
}

namespace {
// State of the pipelined end-to-end entry: the device->host copy of call i runs on an internal copy stream while
// call i + 1 computes on the caller's stream; two device buffers take the final cube in turn.
struct Pipe {
    cudaStream_t copy = nullptr;
    cudaEvent_t ready[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
    bool used[2] = {false, false};
    int next = 0;
};
Pipe g_pipe;
std::mutex g_pipe_mu;

cudaError_t pipe_init()
{
    if (g_pipe.copy) return cudaSuccess;
    cudaError_t e = cudaStreamCreateWithFlags(&g_pipe.copy, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&g_pipe.ready[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g_pipe.copied[i], cudaEventDisableTiming);
    }
    return e;
}

rubix_status forward_host_impl(const rubix_particles *hp, const rubix_ssp *hs, const rubix_telescope *tel,
                               const float *R, float *h_cube, void *scratch, size_t scratch_bytes, void *stream,
                               bool pipelined)
{
    Range nvtx_range(pipelined ? "rubix_forward_host_pipelined" : "rubix_forward_host");
    t_err[0] = 0;
    rubix_status s;
    if ((s = check_particles(hp)) != RUBIX_OK) return s;
    if ((s = check_ssp(hs, true)) != RUBIX_OK) return s;
    if ((s = check_tel(tel)) != RUBIX_OK) return s;
    if (!R || !h_cube) return fail(RUBIX_ERR_NULL, "R or h_cube is NULL");
    const HostLayout H = host_layout(hp->n, hs, tel);
    const size_t cube_bytes = (size_t)tel->n_x * tel->n_y * tel->n_channels * 4;
    const size_t extra = pipelined ? align_up(cube_bytes, 256) : 0;      // the second final-cube buffer, at the end
    if ((s = check_ws(scratch, scratch_bytes, H.total + extra)) != RUBIX_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    char *d = (char *)scratch;
    const size_t n = (size_t)hp->n;
    cudaError_t e = cudaSuccess;
    auto up = [&](size_t off, const void *src, size_t bytes) {
        if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(d + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    up(H.pos, hp->pos, n * 12);
    up(H.vel, hp->vel, n * 12);
    up(H.mass, hp->mass, n * 4);
    up(H.age, hp->log_age, n * 4);
    up(H.z, hp->log_z, n * 4);
    up(H.flux, hs->flux, (size_t)hs->n_age * hs->n_z * hs->n_lambda * 4);
    if (e != cudaSuccess) return cuda_fail(e, "host->device copy");
    rubix_particles dp{hp->n, (const float *)(d + H.pos), (const float *)(d + H.vel), (const float *)(d + H.mass),
                       (const float *)(d + H.age), (const float *)(d + H.z)};
    rubix_ssp ds = *hs;
    ds.flux = (const float *)(d + H.flux);
    const size_t ws_bytes = H.total - H.ws;
    const bool conv = tel->psf_size > 0 || tel->lsf_size > 0;
    // the buffer that takes the final cube of this call
    int slot = 0;
    float *final_cube = (float *)(d + (conv ? H.cube2 : H.cube));
    std::unique_lock<std::mutex> lk(g_pipe_mu, std::defer_lock);
    if (pipelined) {
        lk.lock();
        if ((e = pipe_init()) != cudaSuccess) return cuda_fail(e, "pipeline set-up");
        slot = g_pipe.next;
        g_pipe.next ^= 1;
        if (slot == 1) final_cube = (float *)(d + H.total);
        // the copy of the call before last read this buffer: it must have finished before we overwrite it
        if (g_pipe.used[slot] && (e = cudaStreamWaitEvent(st, g_pipe.copied[slot], 0)) != cudaSuccess)
            return cuda_fail(e, "pipeline wait");
    }
    // steps 1-8 in one call: with PSF/LSF on, the raw cube stays in the workspace and only occupied rows cross HBM
    s = rubix_forward(&dp, &ds, tel, R, final_cube, d + H.ws, ws_bytes, stream);
    if (s != RUBIX_OK) return s;
    if (!pipelined) {
        e = cudaMemcpyAsync(h_cube, final_cube, cube_bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return cuda_fail(e, "device->host copy");
        return RUBIX_OK;
    }
    if ((e = cudaEventRecord(g_pipe.ready[slot], st)) != cudaSuccess) return cuda_fail(e, "pipeline record");
    if ((e = cudaStreamWaitEvent(g_pipe.copy, g_pipe.ready[slot], 0)) != cudaSuccess) return cuda_fail(e, "pipeline wait");
    if ((e = cudaMemcpyAsync(h_cube, final_cube, cube_bytes, cudaMemcpyDeviceToHost, g_pipe.copy)) != cudaSuccess)
        return cuda_fail(e, "device->host copy");
    if ((e = cudaEventRecord(g_pipe.copied[slot], g_pipe.copy)) != cudaSuccess) return cuda_fail(e, "pipeline record");
    g_pipe.used[slot] = true;
    return RUBIX_OK;
}
}  // namespace

rubix_status rubix_forward_host(const rubix_particles *hp, const rubix_ssp *hs, const rubix_telescope *tel,
                                const float *R, float *h_cube, void *scratch, size_t scratch_bytes,
                                void *stream)
{
    return forward_host_impl(hp, hs, tel, R, h_cube, scratch, scratch_bytes, stream, false);
}

size_t rubix_forward_host_pipelined_scratch_bytes(int64_t n, const rubix_ssp *ssp, const rubix_telescope *tel)
{
    const size_t base = rubix_forward_host_scratch_bytes(n, ssp, tel);
    if (base == 0) return 0;
    return base + align_up((size_t)tel->n_x * tel->n_y * tel->n_channels * 4, 256);
}

rubix_status rubix_forward_host_pipelined(const rubix_particles *hp, const rubix_ssp *hs, const rubix_telescope *tel,
                                          const float *R, float *h_cube, void *scratch, size_t scratch_bytes,
                                          void *stream)
{
    return forward_host_impl(hp, hs, tel, R, h_cube, scratch, scratch_bytes, stream, true);
}

rubix_status rubix_forward_host_drain(void *stream)
{
    t_err[0] = 0;
    std::lock_guard<std::mutex> lk(g_pipe_mu);
    for (int i = 0; i < 2; ++i)
        if (g_pipe.used[i]) {
            cudaError_t e = cudaStreamWaitEvent((cudaStream_t)stream, g_pipe.copied[i], 0);
            if (e != cudaSuccess) return cuda_fail(e, "pipeline drain");
        }
    return RUBIX_OK;
}

}  // extern "C"
