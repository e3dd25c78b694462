// K4-K6: Gaussian LSF along the channel axis and separable Gaussian PSF over (x, y)
// ("Gaussian PSF and LSF").
// 'same' output, zero padding, taps point-sampled and normalised to 1 (host, fp64 -> fp32).
// The PSF kernel g (x) g factorises exactly, so two 1-D passes equal the size x size 2-D kernel.
#include <math.h>

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

// One 1-D stencil pass along an axis with element stride `stride` and extent `len`.
// Voxels are enumerated channel-fastest, so a warp always touches contiguous addresses.
template <int VEC>
__global__ void __launch_bounds__(256)
k_stencil_axis(const float *__restrict__ in, float *__restrict__ out, int64_t n_vec, int64_t stride,
               int32_t len, const __grid_constant__ Taps T)
{
    const int h = (T.size - 1) / 2;
    for (int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; v < n_vec;
         v += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = v * VEC;                        // first element of this thread's vector
        const int32_t pos = (int32_t)((e / stride) % len);  // coordinate along the stencil axis
        float acc[VEC];
#pragma unroll
        for (int q = 0; q < VEC; ++q) acc[q] = 0.0f;
        for (int d = -h; d <= h; ++d) {
            const int32_t pp = pos + d;
            if (pp < 0 || pp >= len) continue;
            const float w = T.w[d + h];
            const float *src = in + e + (int64_t)d * stride;
            if (VEC == 4) {
                const float4 x = __ldg(reinterpret_cast<const float4 *>(src));
                acc[0] = fmaf(w, x.x, acc[0]);
                acc[1] = fmaf(w, x.y, acc[1]);
                acc[2] = fmaf(w, x.z, acc[2]);
                acc[3] = fmaf(w, x.w, acc[3]);
            } else {
                acc[0] = fmaf(w, __ldg(src), acc[0]);
            }
        }
        if (VEC == 4) *reinterpret_cast<float4 *>(out + e) = make_float4(acc[0], acc[1], acc[2], acc[3]);
        else out[e] = acc[0];
    }
}

static cudaError_t stencil(const float *in, float *out, int64_t n_vox, int64_t stride, int32_t len,
                           const Taps &T, bool vec4, cudaStream_t st)
{
    // vectorised only across the channel axis and only when the stencil axis is not the channel
    if (vec4) {
        const int64_t n_vec = n_vox / 4;
        const unsigned grid = (unsigned)((n_vec + 255) / 256 < 148 * 64 ? (n_vec + 255) / 256 : 148 * 64);
        k_stencil_axis<4><<<grid ? grid : 1, 256, 0, st>>>(in, out, n_vec, stride, len, T);
    } else {
        const unsigned grid = (unsigned)((n_vox + 255) / 256 < 148 * 64 ? (n_vox + 255) / 256 : 148 * 64);
        k_stencil_axis<1><<<grid ? grid : 1, 256, 0, st>>>(in, out, n_vox, stride, len, T);
    }
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

cudaError_t launch_convolve(const rubix_telescope *tel, const float *in, float *out, float *tmp,
                            cudaStream_t st)
{
    const int32_t n_x = tel->n_x, n_y = tel->n_y, n_c = tel->n_channels;
    const int64_t n_vox = (int64_t)n_x * n_y * n_c;
    if (n_vox == 0) return cudaSuccess;
    Taps lsf, psf;
    make_taps(tel->lsf_size, tel->lsf_sigma, &lsf);
    make_taps(tel->psf_size, tel->psf_sigma, &psf);
    const bool v4 = (n_c % 4 == 0) && (((uintptr_t)in & 15u) == 0) && (((uintptr_t)out & 15u) == 0) &&
                    (((uintptr_t)tmp & 15u) == 0);
    cudaError_t e;
    if (lsf.size <= 0 && psf.size <= 0) {
        e = cudaMemcpyAsync(out, in, (size_t)n_vox * 4, cudaMemcpyDeviceToDevice, st);
        return e;
    }
    const float *src = in;
    if (lsf.size > 0) {
        e = stencil(src, out, n_vox, 1, n_c, lsf, false, st);          // along the channel
        if (e != cudaSuccess) return e;
        src = out;
    }
    if (psf.size > 0) {
        e = stencil(src, tmp, n_vox, n_c, n_y, psf, v4, st);           // along y
        if (e != cudaSuccess) return e;
        e = stencil(tmp, out, n_vox, (int64_t)n_c * n_y, n_x, psf, v4, st);   // along x
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace rubix
