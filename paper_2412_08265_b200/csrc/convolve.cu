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
template <bool LSF, bool VAR = false>
__global__ void __launch_bounds__(256, VAR ? 2 : (LSF ? RUBIX_MARCH_MINB1 : RUBIX_MARCH_MINB0))
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
    const size_t off = (size_t)line * P.line_stride + (size_t)(c_ok ? c : 0);
    const float *src = P.in + off;
    float *dst = P.out + off;
    auto load = [&](int s) -> float2 {
        if (c_ok && s < P.n_steps) return __ldcs(reinterpret_cast<const float2 *>(src + (size_t)s * P.step_stride));
        return make_float2(0.0f, 0.0f);
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
#pragma unroll
    for (int i = 0; i < kMarchPf; ++i) pf[i] = load(i);
    for (int s0 = 0; s0 < P.n_steps + 7; s0 += 15) {
#pragma unroll
        for (int u = 0; u < 15; ++u) {
            const int s = s0 + u;
            const float2 raw = pf[u % kMarchPf];
            pf[u % kMarchPf] = load(s + kMarchPf);
            const unsigned long long v = LSF ? lsf_pair(raw, hp) : pack2(raw.x, raw.y);
#pragma unroll
            for (int d = -7; d <= 7; ++d) {
                const int slot = (u - d + 15) % 15;           // output s - d
                acc[slot] = ffma2(g2[d + 7], v, acc[slot]);
            }
            const int o = s - 7, so = (u + 8) % 15;           // output o is complete
            if (st_ok && o >= 0 && o < P.n_steps)
                __stcs(reinterpret_cast<float2 *>(dst + (size_t)o * P.step_stride), unpack2(acc[so]));
            acc[so] = 0ull;
        }
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
    if (c_ok) v = __ldcs(reinterpret_cast<const float2 *>(P.in + off));
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

template <bool LSF, bool VAR>
static cudaError_t march(MarchParams &P, cudaStream_t st)
{
    P.cblocks = LSF ? (P.n_c + 55) / 56 : (P.n_c + 63) / 64;
    const int64_t warps = (int64_t)P.n_lines * P.cblocks;
    k_march<LSF, VAR><<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

cudaError_t launch_convolve(const rubix_telescope *tel, const float *in, float *out, float *tmp, float *taps_dev,
                            bool transpose, cudaStream_t st)
{
    const int32_t n_x = tel->n_x, n_y = tel->n_y, n_c = tel->n_channels;
    const int64_t n_vox = (int64_t)n_x * n_y * n_c;
    if (n_vox == 0) return cudaSuccess;
    Taps lsf, psf;
    make_taps(tel->lsf_size, tel->lsf_sigma, &lsf);
    make_taps(tel->psf_size, tel->psf_sigma, &psf);
    if (lsf.size <= 0 && psf.size <= 0)
        return cudaMemcpyAsync(out, in, (size_t)n_vox * 4, cudaMemcpyDeviceToDevice, st);

    const bool var = psf.size > 0 && tel->psf_alpha != 0.0f;
    const bool aligned = (n_c % 2 == 0) && (((uintptr_t)in & 7u) == 0) && (((uintptr_t)out & 7u) == 0) &&
                         (tmp == nullptr || ((uintptr_t)tmp & 7u) == 0);
    const bool fast = aligned && psf.size <= 15 && lsf.size <= 9;
    cudaError_t e;
    if (!fast) {
        if (var) return cudaErrorNotSupported;             // api.cu refuses this combination beforehand
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
    centre_taps(psf, 15, P.g);
    centre_taps(lsf, 9, P.h);
    auto lsf_rows = [&](const float *src, float *dst) -> cudaError_t {
        P.in = src; P.out = dst;
        P.n_lines = n_x * n_y; P.n_steps = 1; P.line_stride = n_c; P.step_stride = 0;
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
    };
    auto along_x = [&](const float *src, float *dst) {     // lines = y
        P.in = src; P.out = dst;
        P.n_lines = n_y; P.n_steps = n_x;
        P.line_stride = n_c; P.step_stride = (int64_t)n_y * n_c;
    };
    if (psf.size <= 0) return lsf_rows(in, out);           // LSF only

    if (var) {
        // wavelength-dependent PSF: per-channel taps go to the device once per call
        P.tstride = n_c + 2;
        P.taps = taps_dev;
        static thread_local std::vector<float> host_taps;
        host_taps.resize((size_t)15 * P.tstride);
        var_psf_taps(tel, P.tstride, host_taps.data());
        e = cudaMemcpyAsync(taps_dev, host_taps.data(), host_taps.size() * 4, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
        if (transpose && lsf.size > 0) {                   // LSF^T PSF^T: PSF first (y, x), then the LSF
            along_y(in, out);
            if ((e = march<false, true>(P, st)) != cudaSuccess) return e;
            along_x(out, tmp);
            if ((e = march<false, true>(P, st)) != cudaSuccess) return e;
            return lsf_rows(tmp, out);
        }
        along_y(in, tmp);                                  // PSF LSF: LSF fused into the pass along y
        e = lsf.size > 0 ? march<true, true>(P, st) : march<false, true>(P, st);
        if (e != cudaSuccess) return e;
        along_x(tmp, out);
        return march<false, true>(P, st);
    }
    // pass 1: along y (lines = x), LSF fused when on; pass 2: along x (lines = y)
    along_y(in, tmp);
    e = lsf.size > 0 ? march<true, false>(P, st) : march<false, false>(P, st);
    if (e != cudaSuccess) return e;
    along_x(tmp, out);
    return march<false, false>(P, st);
}

}  // namespace rubix
