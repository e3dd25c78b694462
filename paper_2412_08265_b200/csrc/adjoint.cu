// K7: adjoint of steps 4-6.  Input G' = LSF^T PSF^T dL/d(final cube)
// (the symmetric zero-padded stencils are self-adjoint, so G' comes from the forward convolve
// kernels).  One WARP owns one in-FoV particle (sorted order, so neighbouring warps read the same
// G' row from L1/L2); lanes stride over the channels and the five sums
//   D_c = sum_k G'[s][k] lerp(T_c; x_k)  (c = 4 cell corners),
//   E   = sum_k G'[s][k] lambda_k sum_c w_c (T_c[j+1] - T_c[j])
// are reduced with warp shuffles.  No atomics: each particle's four gradients are written once,
// in ORIGINAL particle order.
//   dL/dm = sum_c w_c D_c ;  dL/dlogA = m sum_c (dw_c/dta) D_c / (A[i+1]-A[i]) (0 if clamped) ;
//   dL/dlogZ likewise ;  dL/dv_los = -m E / (dl_ssp c (1+beta)^2).
// x_k uses the same fixed-point integers as the forward kernel (Rec.a_fx, Rec.b_fx).
#include "common.cuh"

namespace rubix {

struct AdjParams {
    AxisParams ax;
    int32_t n_lambda, pitch, n_z, n_c, n_s;
    float l0_obs, dl_obs, dl_ssp;
    int64_t n;
};

__device__ __forceinline__ void adj_axis_cell(const float *A, int n, float q, int *cell, double *t,
                                              double *width, bool *is_free)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (A[mid] <= q) lo = mid; else hi = mid - 1;
    }
    const int i = min(lo, n - 2);
    const double w = (double)A[i + 1] - (double)A[i];
    *t = fmin(fmax(((double)q - (double)A[i]) / w, 0.0), 1.0);
    *cell = i;
    *width = w;
    *is_free = (q > A[0]) && (q < A[n - 1]);
}

__global__ void __launch_bounds__(256)
k_adjoint(const int32_t *__restrict__ perm, const int32_t *__restrict__ seg_off,
          const int32_t *__restrict__ key, const float *__restrict__ vlos,
          const float *__restrict__ mass, const float *__restrict__ log_age,
          const float *__restrict__ log_z, const Rec *__restrict__ rec,
          const float *__restrict__ flux, const float *__restrict__ gconv,
          const __grid_constant__ AdjParams P, float *__restrict__ g_mass,
          float *__restrict__ g_age, float *__restrict__ g_z, float *__restrict__ g_v)
{
    const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // sorted position
    const int lane = threadIdx.x & 31;
    if (i >= P.n) return;
    const int p = perm[i];
    if (i >= seg_off[P.n_s]) {                              // dropped particle: zero gradient
        if (lane == 0) g_mass[p] = g_age[p] = g_z[p] = g_v[p] = 0.0f;
        return;
    }
    const Rec r = rec[i];
    const float *g = gconv + (size_t)key[p] * P.n_c;
    const float *T0 = flux + r.cell;
    const float *T1 = T0 + (size_t)P.n_z * P.pitch;      // flux = padded workspace copy of the grid
    const float *T2 = T0 + P.pitch;
    const float *T3 = T1 + P.pitch;
    int ia, iz;
    double ta, tz, wa, wz;
    bool a_free, z_free;
    adj_axis_cell(P.ax.age, P.ax.n_age, log_age[p], &ia, &ta, &wa, &a_free);
    adj_axis_cell(P.ax.z, P.ax.n_z, log_z[p], &iz, &tz, &wz, &z_free);
    const float u0 = (float)((1.0 - ta) * (1.0 - tz)), u1 = (float)(ta * (1.0 - tz));
    const float u2 = (float)((1.0 - ta) * tz), u3 = (float)(ta * tz);
    double D0 = 0, D1 = 0, D2 = 0, D3 = 0, E = 0;
    const float inv_scale = 1.0f / (float)(1 << kFxFrac);
    for (int k = r.k_lo + lane; k <= r.k_hi; k += 32) {
        const int64_t x = r.a_fx + (int64_t)r.b_fx * k;
        const int j = (int)(x >> kFxFrac);
        const int jn = min(j + 1, P.n_lambda - 1);
        const float f = (float)(uint32_t)(x & ((1 << kFxFrac) - 1)) * inv_scale;
        const float gk = __ldg(g + k);
        const float a0 = __ldg(T0 + j), b0 = __ldg(T0 + jn) - a0;
        const float a1 = __ldg(T1 + j), b1 = __ldg(T1 + jn) - a1;
        const float a2 = __ldg(T2 + j), b2 = __ldg(T2 + jn) - a2;
        const float a3 = __ldg(T3 + j), b3 = __ldg(T3 + jn) - a3;
        D0 += (double)(gk * fmaf(f, b0, a0));
        D1 += (double)(gk * fmaf(f, b1, a1));
        D2 += (double)(gk * fmaf(f, b2, a2));
        D3 += (double)(gk * fmaf(f, b3, a3));
        const float lam = fmaf(P.dl_obs, (float)k, P.l0_obs);
        E += (double)(gk * lam * fmaf(u3, b3, fmaf(u2, b2, fmaf(u1, b1, u0 * b0))));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        D0 += __shfl_xor_sync(0xffffffffu, D0, o);
        D1 += __shfl_xor_sync(0xffffffffu, D1, o);
        D2 += __shfl_xor_sync(0xffffffffu, D2, o);
        D3 += __shfl_xor_sync(0xffffffffu, D3, o);
        E += __shfl_xor_sync(0xffffffffu, E, o);
    }
    if (lane == 0) {
        const double m = (double)mass[p];
        const double opb = 1.0 + (double)vlos[p] / kCkms;
        g_mass[p] = (float)((1.0 - ta) * (1.0 - tz) * D0 + ta * (1.0 - tz) * D1 + (1.0 - ta) * tz * D2 + ta * tz * D3);
        g_age[p] = a_free ? (float)(m * (-(1.0 - tz) * D0 + (1.0 - tz) * D1 - tz * D2 + tz * D3) / wa) : 0.0f;
        g_z[p] = z_free ? (float)(m * (-(1.0 - ta) * D0 - ta * D1 + (1.0 - ta) * D2 + ta * D3) / wz) : 0.0f;
        g_v[p] = (float)(-m * E / ((double)P.dl_ssp * kCkms * opb * opb));
    }
}

cudaError_t launch_adjoint(const PassInputs &in, const Layout &L, char *ws, const float *gconv,
                           float *g_mass, float *g_age, float *g_z, float *g_v, cudaStream_t st)
{
    if (L.n == 0) return cudaSuccess;
    AdjParams P;
    P.ax.n_age = in.ssp->n_age;
    P.ax.n_z = in.ssp->n_z;
    for (int i = 0; i < in.ssp->n_age; ++i) P.ax.age[i] = in.ssp->log_age_axis[i];
    for (int i = 0; i < in.ssp->n_z; ++i) P.ax.z[i] = in.ssp->log_z_axis[i];
    P.n_lambda = in.ssp->n_lambda;
    P.pitch = L.pitch;
    P.n_z = in.ssp->n_z;
    P.n_c = L.n_c;
    P.n_s = L.n_s;
    P.l0_obs = in.tel->lambda0;
    P.dl_obs = in.tel->dlambda;
    P.dl_ssp = in.ssp->dlambda;
    P.n = L.n;
    const int64_t threads = L.n * 32;
    k_adjoint<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
        (const int32_t *)(ws + L.off_permbuf[L.final_buf]), (const int32_t *)(ws + L.off_seg),
        (const int32_t *)(ws + L.off_key), (const float *)(ws + L.off_vlos), in.p->mass,
        in.p->log_age, in.p->log_z, (const Rec *)(ws + L.off_rec), (const float *)(ws + L.off_flux), gconv, P,
        g_mass,
        g_age, g_z, g_v);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix
