// K4-K6: Gaussian LSF along the channel axis and separable Gaussian PSF over (x, y)
// ("Gaussian PSF and LSF").
// 'same' output, zero padding, taps point-sampled and normalised to 1 (host, fp64 -> fp32).
// The PSF kernel g (x) g factorises exactly, so two 1-D passes equal the size x size 2-D kernel.
//
// Fast path (psf_size <= 15, lsf_size <= 9, even n_channels): two "marching" kernels.  A thread
// owns one channel pair of one line and walks along the stencil axis with a ring of 15 partial
// sums in registers: every input is read exactly once (8-byte loads, 256 B contiguous per warp,
// five steps prefetched -- fifteen in the pass that fuses the LSF --), every output written exactly once, no shared
// memory.
//   pass 1  along y, with the LSF fused in: the 9 channel taps come from the neighbouring lanes
//           by warp shuffle (a warp covers 56 output channels plus 2 halo pairs on each side)
//   pass 2  along x
// Anything else (larger stencils, odd channel counts) takes the generic one-axis kernel.
#include <math.h>

#include <vector>

#include "common.cuh"

namespace rubix {

void make_taps(int size, float sigma, Taps *t)
{
    t->size = size;
    if (size <= 0) return;
    const int h = (size - 1) / 2;
    double w[kMaxTaps], sum = 0.0;
    for (int i = -h; i <= h; ++i) {
        w[i + h] = exp(-((double)i * (double)i) / (2.0 * (double)sigma * (double)sigma));
        sum += w[i + h];
    }
    for (int i = 0; i < size; ++i) t->w[i] = (float)(w[i] / sum);
}

// ------------------------------------------------------------------------------------------
// generic fallback: one 1-D stencil pass along an axis with element stride `stride`
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_stencil_axis(const float *__restrict__ in, float *__restrict__ out, int64_t n_vox, int64_t stride,
               int32_t len, const __grid_constant__ Taps T)
{
    const int h = (T.size - 1) / 2;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_vox;
         e += (int64_t)gridDim.x * blockDim.x) {
        const int32_t pos = (int32_t)((e / stride) % len);
        float acc = 0.0f;
        for (int d = -h; d <= h; ++d) {
            const int32_t pp = pos + d;
            if (pp < 0 || pp >= len) continue;
            acc = fmaf(T.w[d + h], __ldg(in + e + (int64_t)d * stride), acc);
        }
        out[e] = acc;
    }
}

static cudaError_t stencil_generic(const float *in, float *out, int64_t n_vox, int64_t stride, int32_t len,
                                   const Taps &T, cudaStream_t st)
{
    const int64_t blocks = (n_vox + 255) / 256;
    const unsigned grid = (unsigned)(blocks < 148 * 64 ? blocks : 148 * 64);
    k_stencil_axis<<<grid ? grid : 1, 256, 0, st>>>(in, out, n_vox, stride, len, T);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------
// marching kernels
// ------------------------------------------------------------------------------------------
struct MarchParams {
    const float *in;
    float *out;
    int64_t line_stride, step_stride;   // elements
    int32_t n_lines, n_steps, n_c, cblocks;
    float g[15];                        // stencil along the marching axis, zero padded, centred
    float h[9];                         // LSF taps along the channel, zero padded, centred, symmetric
    const float *taps;                  // VAR: per-channel PSF taps, tap-major [15][tstride] (reading R18)
    int32_t tstride;
    // MASK: spaxel of (line, step) = line * sp_line + step * sp_step; mask_in[spaxel] == 0: the input row is taken
    // as zeros without being read; mask_out (MASK == 1): 1 where the output row was written, 0 where it is all zero
    // and was NOT written
    const uint8_t *mask_in;
    uint8_t *mask_out;
    int32_t sp_line, sp_step;
    // batched cubes: gridDim.y = elements; element b starts batch_stride floats / sp_batch spaxels after
    // element b - 1; n_lines counts the lines of ONE cube, so a stencil never crosses into the next cube
    int32_t n_batch, sp_batch;
    int64_t batch_stride;
};

__device__ __forceinline__ float2 shfl_up2(float2 v, int d)
{
    return make_float2(__shfl_up_sync(0xffffffffu, v.x, d), __shfl_up_sync(0xffffffffu, v.y, d));
}
__device__ __forceinline__ float2 shfl_down2(float2 v, int d)
{
    return make_float2(__shfl_down_sync(0xffffffffu, v.x, d), __shfl_down_sync(0xffffffffu, v.y, d));
}

// 9-tap symmetric stencil (h[4 - j] = h[4 + j]) along the channel for the pair (c, c+1) held by
// this lane; lanes hold consecutive pairs, so offsets -4..+5 live in lanes -2..+2.  Even offsets
// use the lanes' aligned pairs, odd offsets the straddling ones; packed fp32x2 arithmetic.
// hp[j] = (h[4 + j], h[4 + j]).
__device__ __forceinline__ unsigned long long lsf_pair(float2 v, const unsigned long long *hp)
{
    const float2 m2 = shfl_up2(v, 2), m1 = shfl_up2(v, 1), p1 = shfl_down2(v, 1), p2 = shfl_down2(v, 2);
    unsigned long long o = fmul2(hp[0], pack2(v.x, v.y));
    o = ffma2(hp[2], pack2(m1.x + p1.x, m1.y + p1.y), o);
    o = ffma2(hp[4], pack2(m2.x + p2.x, m2.y + p2.y), o);
    o = ffma2(hp[1], pack2(m1.y + v.y, v.x + p1.x), o);        // offsets -1, +1
    o = ffma2(hp[3], pack2(m2.y + p1.y, m1.x + p2.x), o);      // offsets -3, +3
    return o;
}

// predicated 8-byte streaming load / store (no branch: the marching loops stay straight-line)
__device__ __forceinline__ float2 ldcs_pred(const float *p, uint32_t pred)
{
    float2 v;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\tmov.f32 %0, 0f00000000;\n\tmov.f32 %1, 0f00000000;\n\t"
                 "@p ld.global.cs.v2.f32 {%0, %1}, [%2];\n\t}"
                 : "=f"(v.x), "=f"(v.y) : "l"(p), "r"(pred));
    return v;
}
__device__ __forceinline__ void stcs_pred(float *p, float2 v, uint32_t pred)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t@p st.global.cs.v2.f32 [%0], {%1, %2};\n\t}"
                 :: "l"(p), "f"(v.x), "f"(v.y), "r"(pred) : "memory");
}
// steps prefetched per thread (divides 15) and resident CTAs per SM, for the pass with the fused LSF (1) and
// for the plain passes (0)
#ifndef RUBIX_MARCH_PF1
#define RUBIX_MARCH_PF1 15
#endif
#ifndef RUBIX_MARCH_MINB1
#define RUBIX_MARCH_MINB1 3
#endif
#ifndef RUBIX_MARCH_PF0
#define RUBIX_MARCH_PF0 5
#endif
#ifndef RUBIX_MARCH_MINB0
#define RUBIX_MARCH_MINB0 4
#endif

// VAR: the stencil along the marching axis differs per channel (wavelength-dependent PSF, reading R18): the
// thread loads the 15 taps of its two channels once; they then live in registers (two resident CTAs per SM).
// MASK (occupancy-aware passes of the fused forward, where the sort knows which spaxels hold particles):
//   1  first pass: rows with mask_in == 0 are not read; an output row whose 15 inputs are all unoccupied is NOT
//      written and gets mask_out = 0 (else 1);  2  second pass: rows with mask_in == 0 are not read, every output is
//      written.  A warp works on one line, so every mask decision is warp-uniform.  The mask bytes of the next 15
//      steps are fetched one iteration ahead (one byte per lane + ballot).
#ifndef RUBIX_MARCH_MINB2
#define RUBIX_MARCH_MINB2 4                  // the masked plain pass (second pass of rubix_forward)
#endif
template <bool LSF, bool VAR = false, int MASK = 0>
__global__ void __launch_bounds__(256, VAR ? 2 : (LSF ? RUBIX_MARCH_MINB1 : (MASK == 2 ? RUBIX_MARCH_MINB2 : RUBIX_MARCH_MINB0)))
k_march(const __grid_constant__ MarchParams P)
{
    constexpr int kMarchPf = LSF ? RUBIX_MARCH_PF1 : RUBIX_MARCH_PF0;
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * 256 + threadIdx.x) >> 5;
    const int line = (int)(gw / P.cblocks), cblock = (int)(gw % P.cblocks);
    if (line >= P.n_lines) return;
    const int c = LSF ? cblock * 56 + 2 * (lane - 2) : cblock * 64 + 2 * lane;
    const bool c_ok = c >= 0 && c + 1 < P.n_c;
    const bool st_ok = c_ok && (!LSF || (lane >= 2 && lane < 30));
    // batched cubes: blockIdx.y = element (no per-thread division: it cost the masked x pass 66 us in registers / spills)
    const int elem = blockIdx.y, lin = line;
    const size_t off = (size_t)elem * P.batch_stride + (size_t)lin * P.line_stride + (size_t)(c_ok ? c : 0);
    const float *src = P.in + off;
    float *dst = P.out + off;
    const int64_t sp0 = MASK ? (int64_t)elem * P.sp_batch + (int64_t)lin * P.sp_line : 0;
    auto mask_byte = [&](int base) -> uint32_t {           // lane i: occupancy of step base + i
        const int s = base + lane;
        return (lane < 15 && s < P.n_steps) ? (uint32_t)__ldg(P.mask_in + sp0 + (int64_t)s * P.sp_step) : 0u;
    };
    unsigned long long acc[15], g2[15], hp[5];
    float2 pf[kMarchPf];
#pragma unroll
    for (int i = 0; i < 15; ++i) {
        acc[i] = 0ull;
        if (VAR) {
            const float2 t = c_ok ? *reinterpret_cast<const float2 *>(P.taps + (size_t)i * P.tstride + c) : make_float2(0.f, 0.f);
            g2[i] = pack2(t.x, t.y);
        } else {
            g2[i] = pack2(P.g[i], P.g[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < 5; ++i) hp[i] = pack2(P.h[4 + i], P.h[4 + i]);
    // the next row to load / to store, advanced by one step per step (no per-step 64-bit multiplies)
    const float *lp = src;
    float *op = dst;
    // lane-dependent conditions as all-ones / zero words: a store predicate is then ONE and-with-uniform-bits test
    const uint32_t st_word = st_ok ? ~0u : 0u, ld_word = c_ok ? ~0u : 0u;
    // mq: occupancy shift register, bit 0 = the step loaded last, bit kMarchPf = the step consumed now,
    // bits kMarchPf .. kMarchPf + 14 = the 15 inputs of the output that completes now
    uint32_t mq = 0, mload = ~0u;
    {
        const uint32_t m0 = MASK ? __ballot_sync(0xffffffffu, mask_byte(0) != 0) : ~0u;
#pragma unroll
        for (int i = 0; i < kMarchPf; ++i) {
            const uint32_t o = i < P.n_steps ? (m0 >> i) & 1u : 0u;
            pf[i] = ldcs_pred(lp, ld_word & o);
            lp += P.step_stride;
            mq = (mq << 1) | o;
        }
        if (MASK) mload = __ballot_sync(0xffffffffu, mask_byte(kMarchPf) != 0);
    }
    for (int s0 = 0; s0 < P.n_steps + 7; s0 += 15) {
        const uint32_t mnext = MASK ? mask_byte(s0 + 15 + kMarchPf) : 0u;   // consumed at the end of this iteration
        uint32_t wbits = 0;                                   // MASK == 1: bit u = the output completed at position u was written
#pragma unroll
        for (int u = 0; u < 15; ++u) {
            const int s = s0 + u;
            const int slot = u % kMarchPf;
            const float2 raw = pf[slot];
            const uint32_t lo = s + kMarchPf < P.n_steps ? (mload >> u) & 1u : 0u;
            pf[slot] = ldcs_pred(lp, ld_word & lo);
            lp += P.step_stride;
            mq = (mq << 1) | lo;
            if (!MASK || ((mq >> kMarchPf) & 1u)) {          // warp-uniform: an unoccupied step adds nothing
                const unsigned long long v = LSF ? lsf_pair(raw, hp) : pack2(raw.x, raw.y);
#pragma unroll
                for (int d = -7; d <= 7; ++d) {
                    const int sl = (u - d + 15) % 15;         // output s - d
                    acc[sl] = ffma2(g2[d + 7], v, acc[sl]);
                }
            }
            const int so = (u + 8) % 15;                      // output s - 7 is complete
            if (s >= 7) {
                const uint32_t wr = (s - 7 < P.n_steps && (MASK != 1 || ((mq >> kMarchPf) & 0x7FFFu) != 0)) ? 1u : 0u;
                stcs_pred(op, unpack2(acc[so]), st_word & wr);
                op += P.step_stride;
                if (MASK == 1) wbits |= wr << u;
            }
            acc[so] = 0ull;
        }
        if (MASK == 1 && cblock == 0) {                       // lane u records the output that completed at position u
            const int o = s0 + lane - 7;
            if (lane < 15 && o >= 0 && o < P.n_steps) P.mask_out[sp0 + (int64_t)o * P.sp_step] = (uint8_t)((wbits >> lane) & 1u);
        }
        if (MASK) mload = __ballot_sync(0xffffffffu, mnext != 0);
    }
}

// LSF alone (PSF off): one pair per thread, same shuffle stencil
__global__ void __launch_bounds__(256)
k_lsf_rows(const __grid_constant__ MarchParams P)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * 256 + threadIdx.x) >> 5;
    const int64_t row = gw / P.cblocks;
    const int cblock = (int)(gw % P.cblocks);
    if (row >= P.n_lines) return;
    const int c = cblock * 56 + 2 * (lane - 2);
    const bool c_ok = c >= 0 && c + 1 < P.n_c;
    const size_t off = (size_t)row * P.n_c + (size_t)(c_ok ? c : 0);
    float2 v = make_float2(0.0f, 0.0f);
    const bool occ = P.mask_in == nullptr || __ldg(P.mask_in + row) != 0;   // unoccupied rows are zeros, not read
    if (c_ok && occ) v = __ldcs(reinterpret_cast<const float2 *>(P.in + off));
    unsigned long long hp[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) hp[i] = pack2(P.h[4 + i], P.h[4 + i]);
    const unsigned long long o = lsf_pair(v, hp);
    if (c_ok && lane >= 2 && lane < 30) __stcs(reinterpret_cast<float2 *>(P.out + off), unpack2(o));
}

static void centre_taps(const Taps &t, int width, float *dst)
{
    for (int i = 0; i < width; ++i) dst[i] = 0.0f;
    if (t.size <= 0) { dst[width / 2] = 1.0f; return; }
    const int shift = (width - t.size) / 2;
    for (int i = 0; i < t.size; ++i) dst[shift + i] = t.w[i];
}

// per-channel PSF taps (reading R18), tap-major [15][tstride], computed on the host in fp64 like make_taps
static void var_psf_taps(const rubix_telescope *tel, int tstride, float *dst)
{
    const int h = (tel->psf_size - 1) / 2, shift = (15 - tel->psf_size) / 2;
    for (int i = 0; i < 15 * tstride; ++i) dst[i] = 0.0f;
    const double zp1 = 1.0;                                // observed wavelengths: the telescope's own grid
    for (int k = 0; k < tel->n_channels; ++k) {
        const double lam = (tel->lambda_obs ? (double)tel->lambda_obs[k] : (double)tel->lambda0 + (double)tel->dlambda * k) / zp1;
        const double sigma = (double)tel->psf_sigma * pow(lam / (double)tel->psf_lambda_ref, (double)tel->psf_alpha);
        double w[15], sum = 0.0;
        for (int i = -h; i <= h; ++i) { w[i + h] = exp(-((double)i * i) / (2.0 * sigma * sigma)); sum += w[i + h]; }
        for (int i = 0; i < tel->psf_size; ++i) dst[(size_t)(shift + i) * tstride + k] = (float)(w[i] / sum);
    }
}

// The same on the device for a uniform channel grid (no host array to read): the call stays asynchronous and can be captured
// in a CUDA graph.  One thread per channel, fp64 like the host version (its values can differ from the host's in the last bit
// of an fp32 tap where the two exp / pow implementations round differently).
__global__ void __launch_bounds__(256)
k_var_psf_taps(int n_c, int psf_size, int tstride, double lambda0, double dlambda, double sigma0, double lambda_ref, double alpha,
               float *__restrict__ dst)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= tstride) return;
    const int h = (psf_size - 1) / 2, shift = (15 - psf_size) / 2;
#pragma unroll
    for (int i = 0; i < 15; ++i) dst[(size_t)i * tstride + k] = 0.0f;
    if (k >= n_c) return;
    const double lam = lambda0 + dlambda * k;
    const double sigma = sigma0 * pow(lam / lambda_ref, alpha);
    double w[15], sum = 0.0;
    for (int i = -h; i <= h; ++i) { w[i + h] = exp(-((double)i * i) / (2.0 * sigma * sigma)); sum += w[i + h]; }
    for (int i = 0; i < psf_size; ++i) dst[(size_t)(shift + i) * tstride + k] = (float)(w[i] / sum);
}

template <bool LSF, bool VAR, int MASK = 0>
static cudaError_t march(MarchParams &P, cudaStream_t st)
{
    P.cblocks = LSF ? (P.n_c + 55) / 56 : (P.n_c + 63) / 64;
    const int64_t warps = (int64_t)P.n_lines * P.cblocks;
    k_march<LSF, VAR, MASK><<<dim3((unsigned)((warps + 7) / 8), (unsigned)P.n_batch), 256, 0, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

static bool fast_path(const rubix_telescope *tel, const float *in, const float *out, const float *tmp)
{
    const bool aligned = (tel->n_channels % 2 == 0) && (((uintptr_t)in & 7u) == 0) && (((uintptr_t)out & 7u) == 0) &&
                         (tmp == nullptr || ((uintptr_t)tmp & 7u) == 0);
    return aligned && tel->psf_size <= 15 && tel->lsf_size <= 9;
}

bool convolve_fast_path(const rubix_telescope *tel, const float *in, const float *out, const float *tmp)
{
    return (tel->psf_size > 0 || tel->lsf_size > 0) && fast_path(tel, in, out, tmp);
}

cudaError_t launch_convolve(const rubix_telescope *tel, const float *in, float *out, float *tmp, float *taps_dev,
                            bool transpose, const uint8_t *occ_in, uint8_t *occ_tmp, cudaStream_t st, int32_t batch)
{
    const int32_t n_x = tel->n_x, n_y = tel->n_y, n_c = tel->n_channels;
    const int64_t n_vox = (int64_t)batch * n_x * n_y * n_c;   // `batch` cubes back to back
    if (n_vox == 0) return cudaSuccess;
    Taps lsf, psf;
    make_taps(tel->lsf_size, tel->lsf_sigma, &lsf);
    make_taps(tel->psf_size, tel->psf_sigma, &psf);
    if (lsf.size <= 0 && psf.size <= 0)
        return cudaMemcpyAsync(out, in, (size_t)n_vox * 4, cudaMemcpyDeviceToDevice, st);

    const bool var = psf.size > 0 && tel->psf_alpha != 0.0f;
    const bool fast = fast_path(tel, in, out, tmp);
    const bool masked = occ_in != nullptr && occ_tmp != nullptr && !transpose;
    cudaError_t e;
    if (!fast) {
        if (var || masked) return cudaErrorNotSupported;   // api.cu refuses / avoids these combinations beforehand
        const float *src = in;
        if (lsf.size > 0) {
            if ((e = stencil_generic(src, out, n_vox, 1, n_c, lsf, st)) != cudaSuccess) return e;
            src = out;
        }
        if (psf.size > 0) {
            if ((e = stencil_generic(src, tmp, n_vox, n_c, n_y, psf, st)) != cudaSuccess) return e;
            if ((e = stencil_generic(tmp, out, n_vox, (int64_t)n_c * n_y, n_x, psf, st)) != cudaSuccess) return e;
        }
        return cudaSuccess;
    }

    MarchParams P;
    P.n_c = n_c;
    P.taps = nullptr;
    P.tstride = 0;
    P.mask_in = nullptr;
    P.mask_out = nullptr;
    P.sp_line = P.sp_step = 0;
    P.n_batch = batch;
    P.sp_batch = n_x * n_y;
    P.batch_stride = (int64_t)n_x * n_y * n_c;
    centre_taps(psf, 15, P.g);
    centre_taps(lsf, 9, P.h);
    auto lsf_rows = [&](const float *src, float *dst) -> cudaError_t {
        P.in = src; P.out = dst;
        P.mask_in = masked ? occ_in : nullptr;
        P.n_lines = batch * n_x * n_y; P.n_steps = 1; P.line_stride = n_c; P.step_stride = 0;
        P.cblocks = (n_c + 55) / 56;
        const int64_t warps = (int64_t)P.n_lines * P.cblocks;
        k_lsf_rows<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(P);
        RUBIX_LAUNCH_CHECK();
        return cudaSuccess;
    };
    auto along_y = [&](const float *src, float *dst) {     // lines = x
        P.in = src; P.out = dst;
        P.n_lines = n_x; P.n_steps = n_y;
        P.line_stride = (int64_t)n_y * n_c; P.step_stride = n_c;
        P.sp_line = n_y; P.sp_step = 1;
    };
    auto along_x = [&](const float *src, float *dst) {     // lines = y
        P.in = src; P.out = dst;
        P.n_lines = n_y; P.n_steps = n_x;
        P.line_stride = n_c; P.step_stride = (int64_t)n_y * n_c;
        P.sp_line = 1; P.sp_step = n_y;
    };
    if (psf.size <= 0) return lsf_rows(in, out);           // LSF only

    if (var) {
        // wavelength-dependent PSF: per-channel taps go to the device once per call
        P.tstride = n_c + 2;
        P.taps = taps_dev;
        if (!tel->lambda_obs) {                            // uniform channel grid: taps on the device (asynchronous, capturable)
            k_var_psf_taps<<<(unsigned)((P.tstride + 255) / 256), 256, 0, st>>>(
                n_c, tel->psf_size, P.tstride, (double)tel->lambda0, (double)tel->dlambda, (double)tel->psf_sigma,
                (double)tel->psf_lambda_ref, (double)tel->psf_alpha, taps_dev);
            RUBIX_LAUNCH_CHECK();
        } else {                                           // listed channel wavelengths are a HOST array: taps on the host
            static thread_local std::vector<float> host_taps;
            host_taps.resize((size_t)15 * P.tstride);
            var_psf_taps(tel, P.tstride, host_taps.data());
            e = cudaMemcpyAsync(taps_dev, host_taps.data(), host_taps.size() * 4, cudaMemcpyHostToDevice, st);
            if (e != cudaSuccess) return e;
        }
        if (transpose && lsf.size > 0) {                   // LSF^T PSF^T: PSF first (y, x), then the LSF
            along_y(in, out);
            if ((e = march<false, true>(P, st)) != cudaSuccess) return e;
            along_x(out, tmp);
            if ((e = march<false, true>(P, st)) != cudaSuccess) return e;
            return lsf_rows(tmp, out);
        }
        along_y(in, tmp);                                  // PSF LSF: LSF fused into the pass along y
        if (masked) {
            P.mask_in = occ_in; P.mask_out = occ_tmp;
            e = lsf.size > 0 ? march<true, true, 1>(P, st) : march<false, true, 1>(P, st);
            if (e != cudaSuccess) return e;
            along_x(tmp, out);
            P.mask_in = occ_tmp; P.mask_out = nullptr;
            return march<false, true, 2>(P, st);
        }
        e = lsf.size > 0 ? march<true, true>(P, st) : march<false, true>(P, st);
        if (e != cudaSuccess) return e;
        along_x(tmp, out);
        return march<false, true>(P, st);
    }
    // pass 1: along y (lines = x), LSF fused when on; pass 2: along x (lines = y)
    along_y(in, tmp);
    if (masked) {
        P.mask_in = occ_in; P.mask_out = occ_tmp;
        e = lsf.size > 0 ? march<true, false, 1>(P, st) : march<false, false, 1>(P, st);
        if (e != cudaSuccess) return e;
        along_x(tmp, out);
        P.mask_in = occ_tmp; P.mask_out = nullptr;
        return march<false, false, 2>(P, st);
    }
    e = lsf.size > 0 ? march<true, false>(P, st) : march<false, false>(P, st);
    if (e != cudaSuccess) return e;
    along_x(tmp, out);
    return march<false, false>(P, st);
}

}  // namespace rubix
