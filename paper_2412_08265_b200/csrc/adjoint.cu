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
#include <type_traits>

#include "common.cuh"

namespace rubix {

struct AdjParams {
    AxisParams ax;
    int32_t n_lambda, pitch, n_z, n_c, n_s;
    float l0_obs, dl_obs, dl_ssp;     // observed grid already divided by (1 + z)
    float flux_scale;
    const int64_t *xtab;              // table mode (R15 / R16): x_k = xtab[k] c + a_fx, c = b_fx / 2^30
    int32_t log_grid;
    double l0_over_dl;                // lambda0_obs / dlambda_obs (the (1+z) factors cancel)
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

template <bool LOGX>
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
    int ia, iz;
    double ta, tz, wa, wz;
    bool a_free, z_free;
    adj_axis_cell(P.ax.age, P.ax.n_age, log_age[p], &ia, &ta, &wa, &a_free);
    adj_axis_cell(P.ax.z, P.ax.n_z, log_z[p], &iz, &tz, &wz, &z_free);
    const float u0 = (float)((1.0 - ta) * (1.0 - tz)), u1 = (float)(ta * (1.0 - tz));
    const float u2 = (float)((1.0 - ta) * tz), u3 = (float)(ta * tz);
    // Lane l owns channels k_lo + l + 32 m.  x_k advances by 32 B in exact 36.28 integer arithmetic;
    // the sample index is x >> 28 and the fraction comes from the top 23 fraction bits (2^-23
    // samples, far below the 1e-3 gradient tolerance).  The rows are padded with zeros, so T[j+1]
    // is always readable; x_k == N_l - 1 exactly (last knot) takes the interval N_l - 2 with f = 1,
    // as the forward kernel does.
    // Accumulated per channel, with v_c = lerp(T_c; x_k):
    //   P0 += g v_0, Pa += g (v_1 - v_0), Pz += g (v_2 - v_0), Pq += g (v_3 - v_2 - v_1 + v_0)
    // so that the bilinear combinations below never subtract two large sums (the D_c of the header
    // are P0, P0 + Pa, P0 + Pz, P0 + Pa + Pz + Pq).  fp32 partial sums over kAdjBlock channels are
    // flushed into fp64 running sums.
#ifndef RUBIX_ADJ_BLOCK
#define RUBIX_ADJ_BLOCK 4
#endif
    constexpr int kAdjBlock = RUBIX_ADJ_BLOCK;
    double P0 = 0, Pa = 0, Pz = 0, Pq = 0, E = 0;
    const int jmax = P.n_lambda - 2;
    const int64_t step = (int64_t)r.b_fx << 5;
    int64_t x = r.a_fx + (int64_t)r.b_fx * (r.k_lo + lane);
    const int64_t *xt = P.xtab + r.k_lo + lane;          // LOGX: x_k = xtab[k] + a_fx, and dx/dbeta is the same
    const float lam_log = (1.0f + vlos[p] / (float)kCkms) * 0.4342944819f;
    // table mode: the Doppler factor in full fp64 (the record's 2.30 value is 5e-6 samples off at x ~ 6000, enough to
    // put a channel on the other side of a knot, where d/dv_los jumps); the channel range stays the record's
    const double c_tab = P.log_grid ? 1.0 : 1.0 / (1.0 + (double)vlos[p] / kCkms);
    const float lam_step = 32.0f * P.dl_obs;
    float lam = fmaf(P.dl_obs, (float)(r.k_lo + lane), P.l0_obs);
    const float *T1 = T0 + (size_t)P.n_z * P.pitch, *T2 = T0 + P.pitch, *T3 = T1 + P.pitch;
    const float *gp = g + r.k_lo + lane;
    float s0, sa, sz, sq, se;
    auto channel = [&]() {
        if (LOGX) {                                         // table mode
            const int64_t y = __ldg(xt);
            x = max((int64_t)(r.a_fx + __double2ll_rn((double)y * c_tab)), (int64_t)0);
            // d x_k / d beta = -lambda_k / ((1+z)(1+beta)^2 dl_ssp) on a linear SSP grid (lambda_k/(1+z) = Y dl_ssp);
            // on a log-sampled one it is the same for every channel: lambda_k -> (1+beta) / ln 10
            lam = P.log_grid ? lam_log : (float)((double)y * (1.0 / (double)(1 << kFxFrac))) * P.dl_ssp;
            xt += 32;
        }
        int j = (int)(x >> kFxFrac);
        float f = __uint_as_float((((uint32_t)x >> 5) & 0x7FFFFFu) | 0x3F800000u) - 1.0f;
        if (j > jmax) { j = jmax; f = 1.0f; }
        const uint32_t ju = (uint32_t)j;                     // one 32 -> 64-bit widening add per corner
        const float gk = __ldg(gp);
        const float a0 = __ldg(T0 + ju), b0 = __ldg(T0 + ju + 1) - a0;
        const float a1 = __ldg(T1 + ju), b1 = __ldg(T1 + ju + 1) - a1;
        const float a2 = __ldg(T2 + ju), b2 = __ldg(T2 + ju + 1) - a2;
        const float a3 = __ldg(T3 + ju), b3 = __ldg(T3 + ju + 1) - a3;
        // difference basis on the samples (their differences are exact in fp32), then the interpolation
        const float v0 = fmaf(f, b0, a0);
        const float da = fmaf(f, b1 - b0, a1 - a0), dz = fmaf(f, b2 - b0, a2 - a0);
        const float dq = fmaf(f, (b3 - b2) - (b1 - b0), (a3 - a2) - (a1 - a0));
        s0 = fmaf(gk, v0, s0);
        sa = fmaf(gk, da, sa);
        sz = fmaf(gk, dz, sz);
        sq = fmaf(gk, dq, sq);
        se = fmaf(gk * lam, fmaf(u3, b3, fmaf(u2, b2, fmaf(u1, b1, u0 * b0))), se);
        x += step; lam += lam_step; gp += 32;
    };
    auto flush = [&]() {
        P0 += (double)s0; Pa += (double)sa; Pz += (double)sz; Pq += (double)sq; E += (double)se;
    };
    int k = r.k_lo + lane;
    for (; k + 32 * (kAdjBlock - 1) <= r.k_hi; k += 32 * kAdjBlock) {
        s0 = sa = sz = sq = se = 0.f;
#pragma unroll
        for (int m = 0; m < kAdjBlock; ++m) channel();
        flush();
    }
    s0 = sa = sz = sq = se = 0.f;
    for (; k <= r.k_hi; k += 32) channel();
    flush();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        P0 += __shfl_xor_sync(0xffffffffu, P0, o);
        Pa += __shfl_xor_sync(0xffffffffu, Pa, o);
        Pz += __shfl_xor_sync(0xffffffffu, Pz, o);
        Pq += __shfl_xor_sync(0xffffffffu, Pq, o);
        E += __shfl_xor_sync(0xffffffffu, E, o);
    }
    if (lane == 0) {
        const double m = (double)mass[p] * (double)P.flux_scale;
        const double opb = 1.0 + (double)vlos[p] / kCkms;
        g_mass[p] = (float)((double)P.flux_scale * (P0 + ta * Pa + tz * Pz + ta * tz * Pq));
        g_age[p] = a_free ? (float)(m * (Pa + tz * Pq) / wa) : 0.0f;
        g_z[p] = z_free ? (float)(m * (Pz + ta * Pq) / wz) : 0.0f;
        g_v[p] = (float)(-m * E / ((double)P.dl_ssp * kCkms * opb * opb));
    }
}

// ------------------------------------------------------------------------------------------
// Adjoint of the flux-conserving rule (RUBIX_RESAMPLE_FLUX, reading R13).
// Records carry the LOWER EDGE of bin 0 as a_fx: x_k = a_fx + b_fx k is the lower edge of bin k.
// One warp per particle; lane l owns bins / lower edges k_lo + l + 32 m.
//   bin k     F_c[k] = (1/B) sum_j W_j T_c[j],  W_j = H(x_hi - j) - H(x_lo - j)  (x clipped to the
//             coverage), H(t) = integral of the hat function from -1 to t.  Accumulated in the
//             difference basis of k_adjoint: P0, Pa, Pz, Pq (x 1/B at the end).
//   edge e    dF/dbeta needs the blended spectrum at the bin edges:
//             sum_k g_k dF_k/dbeta = [ sum_k g_k F_k - (1/dl_obs) sum_e lambda_e s(x_e) (g_{e-1} - g_e) ] / (1+beta),
//             s = 0 at edges outside the coverage (a clipped edge does not move), g = 0 outside
//             [k_lo, k_hi] (those bins do not overlap the coverage).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float hat_integral(float t)
{
    const float a = fminf(fmaxf(t, -1.0f), 1.0f);
    const float lo = 0.5f * (1.0f + a) * (1.0f + a);            // t in [-1, 0]
    const float hi = 1.0f - 0.5f * (1.0f - a) * (1.0f - a);      // t in [0, 1]
    return a <= 0.0f ? lo : hi;
}

__global__ void __launch_bounds__(256)
k_adjoint_flux(const int32_t *__restrict__ perm, const int32_t *__restrict__ seg_off,
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
    const float *T1 = T0 + (size_t)P.n_z * P.pitch, *T2 = T0 + P.pitch, *T3 = T1 + P.pitch;
    int ia, iz;
    double ta, tz, wa, wz;
    bool a_free, z_free;
    adj_axis_cell(P.ax.age, P.ax.n_age, log_age[p], &ia, &ta, &wa, &a_free);
    adj_axis_cell(P.ax.z, P.ax.n_z, log_z[p], &iz, &tz, &wz, &z_free);
    const int64_t x_max = (int64_t)(P.n_lambda - 1) << kFxFrac;
    const int64_t b = (int64_t)r.b_fx;
    const float inv_scale = 1.0f / (float)(1 << kFxFrac);
    double P0 = 0, Pa = 0, Pz = 0, Pq = 0, E = 0;
    const bool narrow = r.b_fx <= (1u << kFxFrac);
    const float width = (float)r.b_fx * inv_scale;
    // lambda_e s(x_e) (g_{e-1} - g_e) / dl_obs for one edge, in fp64: lambda_e / dl_obs ~ 3000 multiplies the blended
    // spectrum at the edge, and the sum over edges cancels to a derivative, so fp32 rounding of s(x_e) would show.
    // `xrel` = x_e minus its knot (or x_e itself: only the low 28 bits are used, except for f = 1 at the last knot).
    const double du0 = (1.0 - ta) * (1.0 - tz), du1 = ta * (1.0 - tz), du2 = (1.0 - ta) * tz, du3 = ta * tz;
    auto edge_term = [&](int64_t xrel, int k, float dg, float a0, float a1, float a2, float a3, float b0, float b1,
                         float b2, float b3) -> double {
        const double fd = xrel == ((int64_t)1 << kFxFrac) ? 1.0
                                                         : (double)(xrel & (((int64_t)1 << kFxFrac) - 1)) * (1.0 / (double)(1 << kFxFrac));
        const double sa_ = du0 * a0 + du1 * a1 + du2 * a2 + du3 * a3;
        const double sb_ = du0 * b0 + du1 * b1 + du2 * b2 + du3 * b3;
        return (double)dg * (P.l0_over_dl + ((double)k - 0.5)) * (sa_ + fd * (sb_ - sa_));
    };
    for (int k = r.k_lo + lane; k <= r.k_hi + 1; k += 32) {
        const int64_t xl = r.a_fx + b * k;                 // lower edge of bin k = edge k
        const float gk = k <= r.k_hi ? __ldg(g + k) : 0.0f;
        const float gm1 = k > r.k_lo ? __ldg(g + k - 1) : 0.0f;
        float s0 = 0.f, sa = 0.f, sz = 0.f, sq = 0.f, se = 0.f;
        if (narrow && k <= r.k_hi && xl >= 0 && xl + b <= x_max) {
            // interior bin no wider than one SSP sample: it touches knots j, j+1, j+2 only, and its
            // lower edge is sampled from the same loads.  w_0..2 = coefficients of the three samples in
            // I(f + B) - I(f), I(u) = integral of the interpolant from knot j to j + u (u < 2)
            const uint32_t j = (uint32_t)(xl >> kFxFrac);
            const float f = __uint_as_float((((uint32_t)xl >> 5) & 0x7FFFFFu) | 0x3F800000u) - 1.0f;
            const float u = f + width;
            const float uu1 = fminf(u, 1.0f), uu2 = fmaxf(u - 1.0f, 0.0f);
            const float q1 = 0.5f * (uu1 * uu1 - f * f);
            const float w0 = (uu1 - f) - q1, w2 = 0.5f * uu2 * uu2, w1 = q1 + uu2 - w2;
            const float a0 = __ldg(T0 + j), a1 = __ldg(T1 + j), a2 = __ldg(T2 + j), a3 = __ldg(T3 + j);
            const float b0 = __ldg(T0 + j + 1), b1 = __ldg(T1 + j + 1), b2 = __ldg(T2 + j + 1), b3 = __ldg(T3 + j + 1);
            const float c0 = __ldg(T0 + j + 2), c1 = __ldg(T1 + j + 2), c2 = __ldg(T2 + j + 2), c3 = __ldg(T3 + j + 2);
            // difference basis on the SAMPLES (exact in fp32), then the bin weights: no subtraction of rounded averages
            const float v0 = fmaf(w2, c0, fmaf(w1, b0, w0 * a0));
            const float da = fmaf(w2, c1 - c0, fmaf(w1, b1 - b0, w0 * (a1 - a0)));
            const float dz = fmaf(w2, c2 - c0, fmaf(w1, b2 - b0, w0 * (a2 - a0)));
            const float dq = fmaf(w2, (c3 - c2) - (c1 - c0), fmaf(w1, (b3 - b2) - (b1 - b0), w0 * ((a3 - a2) - (a1 - a0))));
            s0 = gk * v0;
            sa = gk * da;
            sz = gk * dz;
            sq = gk * dq;
            E += edge_term(xl & (((int64_t)1 << kFxFrac) - 1), k, gm1 - gk, a0, a1, a2, a3, b0, b1, b2, b3);
            P0 += (double)s0; Pa += (double)sa; Pz += (double)sz; Pq += (double)sq;
            continue;
        }
        if (k <= r.k_hi) {                                  // ---- bin k
            const int64_t cl = max(xl, (int64_t)0), ch = min(xl + b, x_max);
            const int jl = (int)(cl >> kFxFrac);
            const int ju = min((int)((ch + ((int64_t)1 << kFxFrac) - 1) >> kFxFrac), P.n_lambda - 1);
            float v0 = 0.f, da = 0.f, dz = 0.f, dq = 0.f;
            for (int j = jl; j <= ju; ++j) {
                const int64_t o = (int64_t)j << kFxFrac;
                const float w = hat_integral((float)(ch - o) * inv_scale) - hat_integral((float)(cl - o) * inv_scale);
                const uint32_t ju32 = (uint32_t)j;
                const float t0 = __ldg(T0 + ju32), t1 = __ldg(T1 + ju32), t2 = __ldg(T2 + ju32), t3 = __ldg(T3 + ju32);
                v0 = fmaf(w, t0, v0);
                da = fmaf(w, t1 - t0, da);
                dz = fmaf(w, t2 - t0, dz);
                dq = fmaf(w, (t3 - t2) - (t1 - t0), dq);
            }
            s0 = gk * v0;
            sa = gk * da;
            sz = gk * dz;
            sq = gk * dq;
        }
        if (xl >= 0 && xl <= x_max) {                       // ---- edge k inside the coverage
            const int j = min((int)(xl >> kFxFrac), P.n_lambda - 2);   // last knot: interval N_l - 2 with f = 1
            const uint32_t ju32 = (uint32_t)j;
            const int64_t xe = (int64_t)j << kFxFrac;      // edge_term re-derives the fraction from xl - (j << 28)
            E += edge_term(xl - xe, k, gm1 - gk, __ldg(T0 + ju32), __ldg(T1 + ju32), __ldg(T2 + ju32),
                           __ldg(T3 + ju32), __ldg(T0 + ju32 + 1), __ldg(T1 + ju32 + 1), __ldg(T2 + ju32 + 1),
                           __ldg(T3 + ju32 + 1));
        }
        P0 += (double)s0; Pa += (double)sa; Pz += (double)sz; Pq += (double)sq; E += (double)se;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        P0 += __shfl_xor_sync(0xffffffffu, P0, o);
        Pa += __shfl_xor_sync(0xffffffffu, Pa, o);
        Pz += __shfl_xor_sync(0xffffffffu, Pz, o);
        Pq += __shfl_xor_sync(0xffffffffu, Pq, o);
        E += __shfl_xor_sync(0xffffffffu, E, o);
    }
    if (lane == 0) {
        const double m = (double)mass[p] * (double)P.flux_scale;
        const double opb = 1.0 + (double)vlos[p] / kCkms;
        const double inv_b = (double)(1 << kFxFrac) / (double)r.b_fx;
        const double gm = inv_b * (P0 + ta * Pa + tz * Pz + ta * tz * Pq);
        g_mass[p] = (float)((double)P.flux_scale * gm);
        g_age[p] = a_free ? (float)(m * inv_b * (Pa + tz * Pq) / wa) : 0.0f;
        g_z[p] = z_free ? (float)(m * inv_b * (Pz + ta * Pq) / wz) : 0.0f;
        g_v[p] = (float)(m * (gm - E) / (kCkms * opb));       // E carries the 1 / dl_obs already
    }
}

// ------------------------------------------------------------------------------------------
// k_adjoint_units: the fast path of step 9 for the point-sampled rule on uniform grids.
// Same work decomposition as the forward kernel (one CTA per unit = up to kChunk consecutive sorted
// particles of ONE spaxel), with the resampling TRANSPOSED onto the SSP sample grid so that the
// four corner rows are read exactly like k_accumulate reads them: 16-byte, line-aligned, coalesced.
//   G' row      the unit's spaxel row of G' is staged in shared memory once per CTA;
//   per particle (one warp each), per pass of 128 samples, lane l owns the sample quad
//               j0 .. j0+3 (one 16-byte load per corner) and the channels whose rest position
//               x_k = A + B k falls into [j0, j0+4).  Per knot interval i of the quad it forms
//                   sigma_i = sum g_k,   beta_i = sum g_k frac(x_k)        (k with floor(x_k) = j0 + i)
//               from which  W_j = (sigma_j - beta_j) + beta_{j-1}   (the transposed hat weights) and
//               gamma_i = sum g_k (x_k + l0_ssp/dl_ssp) = (j0 + i + l0_ssp/dl_ssp) sigma_i + beta_i, and adds
//                   P0 += W_j T_0[j], Pa += W_j (T_1 - T_0)[j], Pz += W_j (T_2 - T_0)[j],
//                   Pq += W_j (T_3 - T_2 - T_1 + T_0)[j]             (difference basis: the template
//                                                                     differences are exact in fp32)
//                   Q_c += gamma_i (T_c[i+1] - T_c[i])               (slope term of d/dv_los)
//               fp32 inside a quad, fp64 across passes; fp64 warp-shuffle reduction at the end.
//   x_k         is evaluated here from v_los in 20.44 fixed point (A and B rounded to 2^-44 samples),
//               i.e. to 1e-10 samples of the oracle's fp64 value over 3700 channels: the derivative in
//               v_los jumps where some x_k crosses a knot, and a particle is compared with the oracle
//               only if its clearance from every knot exceeds that resolution (tests, R19).
// Each interval holds between NA and NA + NB channels (NA = floor(1/B_max), NA + NB = ceil(1/B_min) over
// the velocity cap); the first NA are consumed unconditionally (the staged row is zero padded on both
// sides, so virtual channels outside [0, N_c) contribute nothing), the next NB under a predicate.
// ------------------------------------------------------------------------------------------
#ifndef RUBIX_ADJU_MINB
#define RUBIX_ADJU_MINB 5
#endif
constexpr int kAdjUThreads = 128;
constexpr int kAdjUWarps = kAdjUThreads / 32;
constexpr int kAdjUSplit = 4;               // CTAs per unit: each takes kChunk / kAdjUSplit particles (finer tail)
// The staged G' row is zero padded: `front` floats before it (a pass starts up to 32 samples below the first
// lattice point: k >= -32/B - 2) and `back` behind it (a pass overshoots the last one by < 128/B + 8 points); both are
// multiples of 4, chosen by the host from the smallest B the velocity cap allows.
constexpr int kAdjUFrac = 44;               // fractional bits of x_k in this kernel
#ifndef RUBIX_ADJU_FLUSH
#define RUBIX_ADJU_FLUSH 8
#endif
#ifndef RUBIX_ADJU_DB
#define RUBIX_ADJU_DB 0                      // 1: the next pass's corner quads are loaded into a second register set before this pass is worked on
#endif
constexpr int kAdjUFlush = RUBIX_ADJU_FLUSH;  // passes accumulated in fp32 before the fp64 flush

struct AdjUParams {
    const int32_t *perm, *totals, *seg_off;
    const Unit *units;
    const Rec *rec;
    const AdjAux *aux;
    const float *vlos, *mass, *flux, *gconv;
    float *g_mass, *g_age, *g_z, *g_v;
    int32_t n_lambda, pitch, n_z, n_c, n_s;
    int32_t front, back;                        // zero padding of the staged G' row, floats
    int32_t na, nb;                             // lattice points per knot interval: at least na, at most na + nb
    double l0_obs, dl_obs, l0_ssp, dl_ssp;      // observed grid already divided by (1 + z)
    float flux_scale;
    int64_t n;
};

struct AdjQuad { unsigned long long lo, hi; };              // four consecutive samples as two packed pairs
__device__ __forceinline__ AdjQuad adj_ldg_quad(const float *p)
{
    AdjQuad q;
    asm volatile("ld.global.nc.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
    return q;
}
__device__ __forceinline__ uint32_t adj_and_or(uint32_t a, uint32_t b, uint32_t c)   // (a & b) | c in one LOP3
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

struct AdjCorners {                                         // one pass of one lane: 4 corners x 4 samples (+ the fifth)
    AdjQuad c[4];
    float e[4];                                             // lane 31 only: first sample of the next 128-sample block
};

// Per-particle state of one lane across the passes of k_adjoint_units.
struct AdjLane {
    int k;                                                  // first channel at or above the lane's first knot
    uint32_t d_lo, d_hi;                                    // x_k - j0 in 2^-44 samples, in [0, B)
    uint32_t b_lo, b_hi;                                    // B
    float bf;                                               // B as a float (fraction of the second channel of an interval)
    float xb;                                               // j0 + l0_ssp/dl_ssp - 1
    float beta_carry;                                       // beta of lane 31's last interval in the previous pass
    int na, nb;                                             // runtime step counts of the generic instance (NA < 0)
    unsigned long long p0, pa, pz, pq;                      // packed (even j, odd j) partial sums
    float q0, q1, q2, q3;
};

__device__ __forceinline__ void adj_add64(uint32_t &lo, uint32_t &hi, uint32_t blo, uint32_t bhi)
{
    asm("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, %3;" : "+r"(lo), "+r"(hi) : "r"(blo), "r"(bhi));
}

// One pass (one sample quad per lane) of one particle.  sg_bytes: byte address (shared window) of sg[0].
template <int NA, int NB, bool MASK>
__device__ __forceinline__ void adj_pass(const AdjCorners &C, AdjLane &L, uint32_t sg_addr, int lane, int lim,
                                         const AdjCorners *N = nullptr)
{
    // ---- channels of the quad, interval by interval: sigma_i = sum g, b1_i = sum g (1 + frac)
    uint32_t addr = sg_addr + ((uint32_t)L.k << 2);
    uint32_t lo = L.d_lo, hi = L.d_hi;
    float sig[4], b1[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        float s = 0.0f, b = 0.0f, f1 = 1.0f;
        const uint32_t bound = (uint32_t)(i + 1) << (kAdjUFrac - 32);
#pragma unroll
        for (int st = 0; st < (NA < 0 ? L.na + L.nb : NA + NB); ++st) {
            const bool take = st < (NA < 0 ? L.na : NA) || hi < bound;
            if (NA < 0 && !take) break;
            if (take) {
                float gk;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(gk) : "r"(addr));
                if (st == 0)                                // fraction from the top 23 bits below the binary point
                    f1 = __uint_as_float(adj_and_or(__funnelshift_r(lo, hi, kAdjUFrac - 23), 0x7FFFFFu, 0x3F800000u));
                else
                    f1 += L.bf;                             // same interval: the next channel sits B further on
                s += gk;
                b = fmaf(gk, f1, b);
                adj_add64(lo, hi, L.b_lo, L.b_hi);
                addr += 4;
            }
        }
        // intervals at or beyond the last knot carry no flux (x_k = N_l - 1 exactly: handled by the caller)
        const bool in_cov = !MASK || i < lim;
        sig[i] = in_cov ? s : 0.0f;
        b1[i] = in_cov ? b : 0.0f;
    }
    // ---- W_j = (sigma_j - beta_j) + beta_{j-1}, beta = b1 - sigma;  gamma_i = (x_i + l0/dl) sigma_i + beta_i
    const float bet0 = b1[0] - sig[0], bet1 = b1[1] - sig[1], bet2 = b1[2] - sig[2], bet3 = b1[3] - sig[3];
    float b_prev = __shfl_up_sync(0xffffffffu, bet3, 1);
    if (lane == 0) b_prev = L.beta_carry;
    L.beta_carry = __shfl_sync(0xffffffffu, bet3, 31);
    const float w0 = fmaf(2.0f, sig[0], -b1[0]) + b_prev, w1 = fmaf(2.0f, sig[1], -b1[1]) + bet0;
    const float w2 = fmaf(2.0f, sig[2], -b1[2]) + bet1, w3 = fmaf(2.0f, sig[3], -b1[3]) + bet2;
    const float gm0 = fmaf(L.xb, sig[0], b1[0]), gm1 = fmaf(L.xb + 1.0f, sig[1], b1[1]);
    const float gm2 = fmaf(L.xb + 2.0f, sig[2], b1[2]), gm3 = fmaf(L.xb + 3.0f, sig[3], b1[3]);
    // ---- P sums, two samples per instruction (difference basis; the template differences are exact)
    {
        const unsigned long long neg1 = pack2(-1.0f, -1.0f);
        const unsigned long long wl = pack2(w0, w1), wh = pack2(w2, w3);
        const unsigned long long dal = ffma2(C.c[0].lo, neg1, C.c[1].lo), dah = ffma2(C.c[0].hi, neg1, C.c[1].hi);
        const unsigned long long dzl = ffma2(C.c[0].lo, neg1, C.c[2].lo), dzh = ffma2(C.c[0].hi, neg1, C.c[2].hi);
        const unsigned long long dql = ffma2(dal, neg1, ffma2(C.c[2].lo, neg1, C.c[3].lo));
        const unsigned long long dqh = ffma2(dah, neg1, ffma2(C.c[2].hi, neg1, C.c[3].hi));
        L.p0 = ffma2(wh, C.c[0].hi, ffma2(wl, C.c[0].lo, L.p0));
        L.pa = ffma2(wh, dah, ffma2(wl, dal, L.pa));
        L.pz = ffma2(wh, dzh, ffma2(wl, dzl, L.pz));
        L.pq = ffma2(wh, dqh, ffma2(wl, dql, L.pq));
    }
    // ---- slope sums: gamma_i (T_c[i+1] - T_c[i]); the fifth sample comes from the next lane
    {
        float q[4] = {L.q0, L.q1, L.q2, L.q3};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float2 a = unpack2(C.c[c].lo), bq = unpack2(C.c[c].hi);
            float nx;
            if (N) {                                        // lane 0 publishes the NEXT pass's first sample for lane 31
                const float pub = lane == 0 ? unpack2(N->c[c].lo).x : a.x;
                nx = __shfl_sync(0xffffffffu, pub, (lane + 1) & 31);
            } else {
                nx = __shfl_down_sync(0xffffffffu, a.x, 1);
                if (lane == 31) nx = C.e[c];
            }
            q[c] = fmaf(gm3, nx - bq.y, fmaf(gm2, bq.y - bq.x, fmaf(gm1, bq.x - a.y, fmaf(gm0, a.y - a.x, q[c]))));
        }
        L.q0 = q[0]; L.q1 = q[1]; L.q2 = q[2]; L.q3 = q[3];
    }
}

// Flux-conserving rule (reading R13), same pass structure.  The lattice points are the n_c + 1 bin EDGES
// x_e = A + B e (A = lower edge of bin 0); with D_e = g_{e-1} - g_e (g = 0 outside the detector) summation by parts gives
//   B W_j = sum_e D_e H(x_e - j),  H = integral of the hat function  (edges beyond the coverage sit ON its end: H = 1/2 at
//           the last knot, 1 below it; edges below the coverage add -g/2 to W_0: the caller's fix-up)
//         = C_{j-1} + A_j + tail_j,   A_i = M0/2 + M1 - M2/2,  C_i = M2/2,  tail_j = g of the last edge below j + 1
// from the moments M_n = sum over the edges of interval i of D_e frac(x_e)^n.  The P sums use W as in the point rule.
// d/dv_los: inside the coverage dF_k/dbeta = -(1 / (B (1 + beta))) integral over bin k of (x + l0/dl) s'(x) dx, and s' is
// the constant S_{i+1} - S_i on knot interval i, so
//   sum_k g_k dF_k/dbeta = -(1 / (B (1 + beta))) sum_i Gamma_i (S_{i+1} - S_i),
//   Gamma_i = integral over [i, i+1) of g(x) (x + l0/dl) dx      (g(x) = g_k on bin k)
//           = g_start (xi + 1/2) - [xi (M0 - M1) + (M0 - M2) / 2],   xi = i + l0_ssp/dl_ssp,
// i.e. the point rule's slope sums with Gamma in place of gamma: exact template differences, no cancellation
// (the equivalent edge form sum_e D_e lambda_e s(x_e) cancels to this derivative and loses 3 digits in fp32).
// Bins cut by an end of the coverage add a boundary term each (the caller's fix-up).
template <int NA, int NB, bool MASK>
__device__ __forceinline__ void adj_pass_flux(const AdjCorners &C, AdjLane &L, float &c_carry, uint32_t sg_addr, int lane, int lim)
{
    uint32_t addr = sg_addr + ((uint32_t)L.k << 2);
    uint32_t lo = L.d_lo, hi = L.d_hi;
    float g_prev;
    asm volatile("ld.shared.f32 %0, [%1+-4];" : "=f"(g_prev) : "r"(addr));
    float wa[4], wc[4], gam[4];                             // A_i + tail_i, C_i, Gamma_i
    float xi = L.xb;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        float m0 = 0.0f, m1 = 0.0f, m2 = 0.0f, f = 0.0f;
        const float g_start = g_prev;
        const uint32_t bound = (uint32_t)(i + 1) << (kAdjUFrac - 32);
#pragma unroll
        for (int st = 0; st < (NA < 0 ? L.na + L.nb : NA + NB); ++st) {
            const bool take = st < (NA < 0 ? L.na : NA) || hi < bound;
            if (NA < 0 && !take) break;
            if (take) {
                float ge;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(ge) : "r"(addr));
                if (st == 0)
                    f = __uint_as_float(adj_and_or(__funnelshift_r(lo, hi, kAdjUFrac - 23), 0x7FFFFFu, 0x3F800000u)) - 1.0f;
                else
                    f += L.bf;
                const float dg = g_prev - ge;
                const float t = dg * f;
                m0 += dg;
                m1 += t;
                m2 = fmaf(t, f, m2);
                g_prev = ge;
                adj_add64(lo, hi, L.b_lo, L.b_hi);
                addr += 4;
            }
        }
        float a_i = fmaf(0.5f, m0 - m2, m1) + g_prev, c_i = 0.5f * m2;
        float gam_i = fmaf(g_start, xi + 0.5f, -fmaf(xi, m0 - m1, 0.5f * (m0 - m2)));
        if (MASK && i >= lim) {                             // at or beyond the last knot
            a_i = i == lim ? 0.5f * g_start : 0.0f;
            c_i = 0.0f; gam_i = 0.0f;
        }
        wa[i] = a_i; wc[i] = c_i; gam[i] = gam_i;
        xi += 1.0f;
    }
    float c_prev = __shfl_up_sync(0xffffffffu, wc[3], 1);
    if (lane == 0) c_prev = c_carry;
    c_carry = __shfl_sync(0xffffffffu, wc[3], 31);
    const float w0 = wa[0] + c_prev, w1 = wa[1] + wc[0], w2 = wa[2] + wc[1], w3 = wa[3] + wc[2];
    const unsigned long long neg1 = pack2(-1.0f, -1.0f);
    const unsigned long long wl = pack2(w0, w1), wh = pack2(w2, w3);
    const unsigned long long dal = ffma2(C.c[0].lo, neg1, C.c[1].lo), dah = ffma2(C.c[0].hi, neg1, C.c[1].hi);
    const unsigned long long dzl = ffma2(C.c[0].lo, neg1, C.c[2].lo), dzh = ffma2(C.c[0].hi, neg1, C.c[2].hi);
    const unsigned long long dql = ffma2(dal, neg1, ffma2(C.c[2].lo, neg1, C.c[3].lo));
    const unsigned long long dqh = ffma2(dah, neg1, ffma2(C.c[2].hi, neg1, C.c[3].hi));
    L.p0 = ffma2(wh, C.c[0].hi, ffma2(wl, C.c[0].lo, L.p0));
    L.pa = ffma2(wh, dah, ffma2(wl, dal, L.pa));
    L.pz = ffma2(wh, dzh, ffma2(wl, dzl, L.pz));
    L.pq = ffma2(wh, dqh, ffma2(wl, dql, L.pq));
    // slope sums: Gamma_i (T_c[i+1] - T_c[i]); the fifth sample comes from the next lane
    float q[4] = {L.q0, L.q1, L.q2, L.q3};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float2 a = unpack2(C.c[c].lo), bq = unpack2(C.c[c].hi);
        float nx = __shfl_down_sync(0xffffffffu, a.x, 1);
        if (lane == 31) nx = C.e[c];
        q[c] = fmaf(gam[3], nx - bq.y, fmaf(gam[2], bq.y - bq.x, fmaf(gam[1], bq.x - a.y, fmaf(gam[0], a.y - a.x, q[c]))));
    }
    L.q0 = q[0]; L.q1 = q[1]; L.q2 = q[2]; L.q3 = q[3];
}

template <int NA, int NB, bool FLUX>
__global__ void __launch_bounds__(kAdjUThreads, RUBIX_ADJU_MINB)
k_adjoint_units(const __grid_constant__ AdjUParams P)
{
    extern __shared__ __align__(16) float sg_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_units = P.totals[0];
    const int u = blockIdx.x / kAdjUSplit, part = blockIdx.x % kAdjUSplit;
    if (u >= n_units) {
        // spare CTAs of the (upper-bound) grid zero the gradients of the dropped particles
        const int64_t first = P.seg_off[P.n_s];
        const int64_t spare = (int64_t)gridDim.x - (int64_t)n_units * kAdjUSplit;
        for (int64_t i = first + ((int64_t)blockIdx.x - (int64_t)n_units * kAdjUSplit) * kAdjUThreads + tid; i < P.n;
             i += spare * kAdjUThreads) {
            const int p = P.perm[i];
            P.g_mass[p] = 0.0f; P.g_age[p] = 0.0f; P.g_z[p] = 0.0f; P.g_v[p] = 0.0f;
        }
        return;
    }
    const Unit U = P.units[u];
    constexpr int kPer = kChunk / kAdjUSplit;
    const int q_begin = part * kPer, q_end = min(U.count, q_begin + kPer);
    if (q_begin >= q_end) return;
    float *sg = sg_raw + P.front;                           // sg[k] = G'[spaxel][k], zeros outside [0, n_c)
    {
        const float *g = P.gconv + (size_t)U.spaxel * P.n_c;
        for (int k = tid - P.front; k < 0; k += kAdjUThreads) sg[k] = 0.0f;
        for (int k = P.n_c + tid; k < P.n_c + P.back; k += kAdjUThreads) sg[k] = 0.0f;
        if ((P.n_c & 3) == 0 && ((uintptr_t)P.gconv & 15u) == 0) {      // front is a multiple of 4: 16-byte stores
            const float4 *g4 = reinterpret_cast<const float4 *>(g);
            float4 *s4 = reinterpret_cast<float4 *>(sg);
            const int n4 = P.n_c >> 2;
            int k = tid;
            for (; k + 3 * kAdjUThreads < n4; k += 4 * kAdjUThreads) {  // four loads in flight per thread
                const float4 v0 = __ldg(g4 + k), v1 = __ldg(g4 + k + kAdjUThreads);
                const float4 v2 = __ldg(g4 + k + 2 * kAdjUThreads), v3 = __ldg(g4 + k + 3 * kAdjUThreads);
                s4[k] = v0; s4[k + kAdjUThreads] = v1; s4[k + 2 * kAdjUThreads] = v2; s4[k + 3 * kAdjUThreads] = v3;
            }
            for (; k < n4; k += kAdjUThreads) s4[k] = __ldg(g4 + k);
        } else {
            for (int k = tid; k < P.n_c; k += kAdjUThreads) sg[k] = __ldg(g + k);
        }
    }
    __syncthreads();
    const uint32_t sg_addr = (uint32_t)__cvta_generic_to_shared(sg);
    const int row_a = P.n_z * P.pitch, row_z = P.pitch;
    // lambda = (x + l0_ssp/dl_ssp) dl_ssp (1 + beta); point rule: -1 because b1 carries 1 + frac
    const float x_off = (float)(P.l0_ssp / P.dl_ssp) - (FLUX ? 0.0f : 1.0f);
    const int64_t x_top = (int64_t)(P.n_lambda - 1) << kAdjUFrac;
    const double inv_dl_ssp = 1.0 / P.dl_ssp;

    auto load = [&](AdjCorners &C, const float *t) {
        C.c[0] = adj_ldg_quad(t); C.c[1] = adj_ldg_quad(t + row_a);
        C.c[2] = adj_ldg_quad(t + row_z); C.c[3] = adj_ldg_quad(t + row_a + row_z);
        if (lane == 31) {                                   // fifth sample of each corner: the next block's first
            C.e[0] = __ldg(t + 4); C.e[1] = __ldg(t + row_a + 4);
            C.e[2] = __ldg(t + row_z + 4); C.e[3] = __ldg(t + row_a + row_z + 4);
        }
    };
    auto prefetch = [&](const float *t) {                   // the next pass's corner rows: L2 -> L1 while this pass is worked on
        asm volatile("prefetch.global.L1 [%0];" ::"l"(t));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(t + row_a));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(t + row_z));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(t + row_a + row_z));
    };
    // fp64 running sums of the thread live in shared memory (component-major: conflict-free), flushed every
    // kAdjUFlush passes; keeps the register count low enough for five resident CTAs
    double *acc = reinterpret_cast<double *>(sg_raw + ((P.n_c + P.front + P.back + 3) & ~3)) + tid;

    for (int q = q_begin + warp; q < q_end; q += kAdjUWarps) {
        const int64_t i_sorted = (int64_t)U.start + q;
        const int p = P.perm[i_sorted];
        const float *T0 = P.flux + P.rec[i_sorted].cell;
        const double opb = 1.0 + (double)P.vlos[p] / kCkms;
        const double inv = 1.0 / opb;
        const double scale = (double)((int64_t)1 << kAdjUFrac);
        // lattice: channel centres x_k (point rule, n_c points) or bin edges x_e (flux rule, n_c + 1 points)
        const int64_t a44 = __double2ll_rn(((P.l0_obs - (FLUX ? 0.5 * P.dl_obs : 0.0)) * inv - P.l0_ssp) * inv_dl_ssp * scale);
        const int64_t b44 = __double2ll_rn(P.dl_obs * inv * inv_dl_ssp * scale);
        const int64_t x_first = a44, x_last = a44 + (int64_t)(FLUX ? P.n_c : P.n_c - 1) * b44;
        const int64_t x_lo = max(x_first, (int64_t)0), x_hi = min(x_last, x_top);
#pragma unroll
        for (int c = 0; c < 8; ++c) acc[c * kAdjUThreads] = 0.0;
        if (x_lo <= x_hi) {
            const int j_begin = (int)(x_lo >> kAdjUFrac) & ~(kRowAlign - 1);
            // the sample above the last lattice point still receives weight (beta / C of its interval)
            const int j_last = min((int)(x_hi >> kAdjUFrac) + 1, P.n_lambda - 1);
            // channels per 128 samples: kstep = floor(128 / B); a pass moves the lane's first channel by kstep or
            // kstep + 1, decided in exact integers: delta = kstep B - 128 in (-B, 0]
            const double inv_b = 1.0 / (double)b44;
            const int64_t span = (int64_t)128 << kAdjUFrac;
            int kstep = (int)((double)span * inv_b);
            int64_t delta = (int64_t)kstep * b44 - span;
            if (delta > 0) { delta -= b44; --kstep; }
            if (delta <= -b44) { delta += b44; ++kstep; }
            // first channel at or above the lane's first knot: estimate in fp64, settle in exact integers
            int j0 = j_begin + 4 * lane;
            AdjLane L;
            int64_t d;
            {
                const int64_t J0 = (int64_t)j0 << kAdjUFrac;
                L.k = (int)ceil((double)(J0 - a44) * inv_b);
                int64_t X = a44 + (int64_t)L.k * b44;
                if (X - b44 >= J0) { X -= b44; --L.k; }
                if (X < J0) { X += b44; ++L.k; }
                d = X - J0;
            }
            L.b_lo = (uint32_t)b44; L.b_hi = (uint32_t)(b44 >> 32);
            L.bf = (float)((double)b44 * (1.0 / scale));
            L.xb = x_off + (float)j0;
            L.beta_carry = 0.0f;
            L.na = P.na; L.nb = P.nb;
            L.p0 = L.pa = L.pz = L.pq = 0ull;
            L.q0 = L.q1 = L.q2 = L.q3 = 0.f;
            float c_carry = 0.0f;                           // flux rule: C of lane 31's last interval in the previous pass
            const float *t = T0 + j0;
            int n_acc = 0;
            auto flush = [&]() {
                const float2 f0 = unpack2(L.p0), fa = unpack2(L.pa), fz = unpack2(L.pz), fq = unpack2(L.pq);
                acc[0 * kAdjUThreads] += (double)(f0.x + f0.y); acc[1 * kAdjUThreads] += (double)(fa.x + fa.y);
                acc[2 * kAdjUThreads] += (double)(fz.x + fz.y); acc[3 * kAdjUThreads] += (double)(fq.x + fq.y);
                acc[4 * kAdjUThreads] += (double)L.q0; acc[5 * kAdjUThreads] += (double)L.q1;
                acc[6 * kAdjUThreads] += (double)L.q2; acc[7 * kAdjUThreads] += (double)L.q3;
                L.q0 = L.q1 = L.q2 = L.q3 = 0.f;
                L.p0 = L.pa = L.pz = L.pq = 0ull;
                n_acc = 0;
            };
            auto advance = [&]() {                          // next pass: 128 samples on
                d += delta;
                L.k += kstep;
                if (d < 0) { d += b44; ++L.k; }
                j0 += 128; t += 128; L.xb += 128.0f;
                if (++n_acc == kAdjUFlush) flush();
            };
            const int j_main = min(j_last, P.n_lambda - 1 - 128);   // passes starting above this touch the last knot
            int jp = j_begin;
            AdjCorners A;
            A.e[0] = A.e[1] = A.e[2] = A.e[3] = 0.0f;
#if RUBIX_ADJU_DB
            if (!FLUX) {
                // two register sets: the quads of pass p + 1 are in flight while pass p is worked on (no L1 prefetch), and
                // lane 31's fifth sample is lane 0's first sample of the next set (no extra loads); the padded grid copy
                // makes the load behind the last pass harmless
                auto load4 = [&](AdjCorners &C, const float *tt) {
                    C.c[0] = adj_ldg_quad(tt); C.c[1] = adj_ldg_quad(tt + row_a);
                    C.c[2] = adj_ldg_quad(tt + row_z); C.c[3] = adj_ldg_quad(tt + row_a + row_z);
                };
                AdjCorners Bn;
                load4(A, t);
                for (; jp <= j_last; jp += 128) {
                    load4(Bn, t + 128);
                    L.d_lo = (uint32_t)d; L.d_hi = (uint32_t)((uint64_t)d >> 32);
                    if (jp <= j_main) adj_pass<NA, NB, false>(A, L, sg_addr, lane, 0, &Bn);
                    else adj_pass<NA, NB, true>(A, L, sg_addr, lane, P.n_lambda - 1 - j0, &Bn);
                    advance();
#pragma unroll
                    for (int c = 0; c < 4; ++c) A.c[c] = Bn.c[c];
                }
            } else
#endif
            {
            for (; jp <= j_main; jp += 128) {
                load(A, t);
                prefetch(t + 128);
                L.d_lo = (uint32_t)d; L.d_hi = (uint32_t)((uint64_t)d >> 32);
                if (FLUX) adj_pass_flux<NA, NB, false>(A, L, c_carry, sg_addr, lane, 0);
                else adj_pass<NA, NB, false>(A, L, sg_addr, lane, 0);
                advance();
            }
            for (; jp <= j_last; jp += 128) {               // passes that touch the last knot
                load(A, t);
                L.d_lo = (uint32_t)d; L.d_hi = (uint32_t)((uint64_t)d >> 32);
                if (FLUX) adj_pass_flux<NA, NB, true>(A, L, c_carry, sg_addr, lane, P.n_lambda - 1 - j0);
                else adj_pass<NA, NB, true>(A, L, sg_addr, lane, P.n_lambda - 1 - j0);
                advance();
            }
            }
            flush();
        }
        // sum the 32 lanes' running sums: lane l adds component (l & 7) of lanes 8 (l >> 3) .. + 7 from shared
        // memory, two shuffle rounds combine the four groups; fixed order, so the result is reproducible
        __syncwarp();
        double part = 0.0;
        {
            const double *col = acc - lane + (lane & 7) * kAdjUThreads + 8 * (lane >> 3);
#pragma unroll
            for (int r = 0; r < 8; ++r) part += col[r];
        }
        part += __shfl_xor_sync(0xffffffffu, part, 8);
        part += __shfl_xor_sync(0xffffffffu, part, 16);
        const double P0 = __shfl_sync(0xffffffffu, part, 0), Pa = __shfl_sync(0xffffffffu, part, 1);
        const double Pz = __shfl_sync(0xffffffffu, part, 2), Pq = __shfl_sync(0xffffffffu, part, 3);
        const double Q0 = __shfl_sync(0xffffffffu, part, 4), Q1 = __shfl_sync(0xffffffffu, part, 5);
        const double Q2 = __shfl_sync(0xffffffffu, part, 6), Q3 = __shfl_sync(0xffffffffu, part, 7);
        __syncwarp();
        if (lane == 0) {
            const AdjAux ax = P.aux[i_sorted];
            const double ta = (double)ax.ta, tz = (double)ax.tz;
            double p0 = P0, pa = Pa, pz = Pz, pq = Pq, q0 = Q0, q1 = Q1, q2 = Q2, q3 = Q3;
            const float *tl = T0 + (P.n_lambda - 1);
            const bool on_top = x_last >= x_top && x_first <= x_top && (x_top - a44) % b44 == 0;
            auto add_w = [&](double w, const float *tp) {  // weight w on one sample of the four corners
                const float t0 = tp[0], t1 = tp[row_a], t2 = tp[row_z], t3 = tp[row_a + row_z];
                p0 += w * t0;
                pa += w * ((double)t1 - t0);
                pz += w * ((double)t2 - t0);
                pq += w * (((double)t3 - t2) - ((double)t1 - t0));
            };
            if (!FLUX) {
                // a channel sitting exactly on the last knot (x_k = N_l - 1) takes the last sample with weight 1,
                // as the forward kernel does; its slope term is left out (the spectrum ends there)
                if (on_top) add_w((double)sg[(x_top - a44) / b44], tl);
            } else {
                const double off = P.l0_ssp * inv_dl_ssp;
                // bins cut by the first knot: the edges below it sit ON it, -g H(0) on W_0; and the cut bin's boundary term
                // -(0 + l0/dl) s(0) g of d/dv_los (a clipped edge does not move).  e0 = first edge at or above 0
                if (x_first < 0 && x_last >= 0) {
                    const int64_t e0 = (-a44 + b44 - 1) / b44;
                    const double gl = (double)sg[e0 - 1];
                    add_w(-0.5 * gl, T0);
                    const double v = gl * off;
                    q0 += v * T0[0]; q1 += v * T0[row_a]; q2 += v * T0[row_z]; q3 += v * T0[row_a + row_z];
                }
                // the bin cut by the last knot: boundary term +(N_l - 1 + l0/dl) s(N_l - 1) g
                if (x_first <= x_top && x_last > x_top) {
                    const int64_t kt = (x_top - a44) / b44;
                    const double v = -(double)sg[kt] * ((double)(P.n_lambda - 1) + off);
                    q0 += v * tl[0]; q1 += v * tl[row_a]; q2 += v * tl[row_z]; q3 += v * tl[row_a + row_z];
                }
            }
            const double m = (double)P.mass[p] * (double)P.flux_scale;
            const double E = (1.0 - ta) * (1.0 - tz) * q0 + ta * (1.0 - tz) * q1 + (1.0 - ta) * tz * q2 + ta * tz * q3;
            const double gm = p0 + ta * pa + tz * pz + ta * tz * pq;
            if (!FLUX) {
                P.g_mass[p] = (float)((double)P.flux_scale * gm);
                P.g_age[p] = (float)(m * (pa + tz * pq) * (double)ax.inv_wa);
                P.g_z[p] = (float)(m * (pz + ta * pq) * (double)ax.inv_wz);
                P.g_v[p] = (float)(-m * E * inv / kCkms);
            } else {
                // W carries a factor B (F_k = (1/B) integral);  d/dbeta sum g F = -(1 / (B (1 + beta))) sum_i Gamma_i dS_i + boundary
                const double inv_bw = scale / (double)b44;
                P.g_mass[p] = (float)((double)P.flux_scale * inv_bw * gm);
                P.g_age[p] = (float)(m * inv_bw * (pa + tz * pq) * (double)ax.inv_wa);
                P.g_z[p] = (float)(m * inv_bw * (pz + ta * pq) * (double)ax.inv_wz);
                P.g_v[p] = (float)(-m * inv_bw * E * inv / kCkms);
            }
        }
    }
}

template <int NA, int NB>
static cudaError_t launch_adjoint_units(const AdjUParams &P, bool flux, unsigned grid, size_t smem, cudaStream_t st)
{
    auto kern = flux ? k_adjoint_units<NA, NB, true> : k_adjoint_units<NA, NB, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kAdjUThreads, smem, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

// Lattice points per knot interval over the velocity cap: at least na, at most na + nb; zero padding of the staged row.
// Returns false when k_adjoint_units cannot take the problem (table mode, or the staged row would not fit in shared
// memory): the warp-per-particle kernels take over.
static bool adjoint_units_shape(const PassInputs &in, const Layout &L, AdjUParams *Q, size_t *smem)
{
    if (table_mode(in.ssp, in.tel)) return false;
    const double b0 = (double)in.tel->dlambda / ((1.0 + (double)in.tel->redshift) * (double)in.ssp->dlambda);
    const double b_lo = b0 / (1.0 + kBetaCap) * (1.0 - 1e-6), b_hi = b0 / (1.0 - kBetaCap) * (1.0 + 1e-6);
    if (!(b_lo > 0.0) || !(b_hi < 15.0)) return false;
    const double front = ceil(32.0 / b_lo) + 16.0, back = ceil(128.0 / b_lo) + 16.0;
    const double bytes = ((double)L.n_c + front + back + 8.0) * 4.0 + 8.0 * kAdjUThreads * sizeof(double);
    if (bytes > 200.0 * 1024.0) return false;
    Q->front = ((int32_t)front + 3) & ~3;
    Q->back = ((int32_t)back + 3) & ~3;
    Q->na = (int32_t)floor(1.0 / b_hi);
    Q->nb = (int32_t)ceil(1.0 / b_lo) - Q->na;
    *smem = (size_t)(((size_t)L.n_c + Q->front + Q->back + 3) & ~(size_t)3) * sizeof(float) +
            (size_t)8 * kAdjUThreads * sizeof(double);
    return true;
}

cudaError_t launch_adjoint(const PassInputs &in, const Layout &L, char *ws, const float *gconv,
                           float *g_mass, float *g_age, float *g_z, float *g_v, cudaStream_t st)
{
    if (L.n == 0) return cudaSuccess;
    if (gen_mode(in.ssp, in.tel) || table_flux(in.ssp, in.tel))
        return launch_adjoint_general(in, L, ws, gconv, g_mass, g_age, g_z, g_v, st);
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
    P.l0_obs = (float)((double)in.tel->lambda0 / (1.0 + (double)in.tel->redshift));
    P.dl_obs = (float)((double)in.tel->dlambda / (1.0 + (double)in.tel->redshift));
    P.flux_scale = in.tel->flux_scale;
    P.l0_over_dl = (double)in.tel->lambda0 / (double)in.tel->dlambda;
    P.xtab = (const int64_t *)(ws + L.off_xtab);
    P.log_grid = in.ssp->log_lambda;
    P.dl_ssp = in.ssp->dlambda;
    P.n = L.n;
    AdjUParams Q;
    size_t smem = 0;
    if (adjoint_units_shape(in, L, &Q, &smem)) {
        Q.perm = (const int32_t *)(ws + L.off_permbuf[L.final_buf]);
        Q.totals = (const int32_t *)(ws + L.off_totals);
        Q.seg_off = (const int32_t *)(ws + L.off_seg);
        Q.units = (const Unit *)(ws + L.off_units);
        Q.rec = (const Rec *)(ws + L.off_rec);
        Q.aux = (const AdjAux *)(ws + L.off_aux);
        Q.vlos = (const float *)(ws + L.off_vlos);
        Q.mass = in.p->mass;
        Q.flux = (const float *)(ws + L.off_flux);
        Q.gconv = gconv;
        Q.g_mass = g_mass; Q.g_age = g_age; Q.g_z = g_z; Q.g_v = g_v;
        Q.n_lambda = in.ssp->n_lambda; Q.pitch = L.pitch; Q.n_z = in.ssp->n_z; Q.n_c = L.n_c; Q.n_s = L.n_s;
        const double zp1 = 1.0 + (double)in.tel->redshift;
        Q.l0_obs = (double)in.tel->lambda0 / zp1;
        Q.dl_obs = (double)in.tel->dlambda / zp1;
        Q.l0_ssp = (double)in.ssp->lambda0;
        Q.dl_ssp = (double)in.ssp->dlambda;
        Q.flux_scale = in.tel->flux_scale;
        Q.n = L.n;
        const unsigned grid = (unsigned)(L.max_units * kAdjUSplit);
        const bool flux = in.tel->resample == RUBIX_RESAMPLE_FLUX;
        if (Q.na <= 3 && Q.nb <= 2) {
            switch (Q.na * 2 + (Q.nb - 1)) {
                case 0: return launch_adjoint_units<0, 1>(Q, flux, grid, smem, st);
                case 1: return launch_adjoint_units<0, 2>(Q, flux, grid, smem, st);
                case 2: return launch_adjoint_units<1, 1>(Q, flux, grid, smem, st);
                case 3: return launch_adjoint_units<1, 2>(Q, flux, grid, smem, st);
                case 4: return launch_adjoint_units<2, 1>(Q, flux, grid, smem, st);
                case 5: return launch_adjoint_units<2, 2>(Q, flux, grid, smem, st);
                case 6: return launch_adjoint_units<3, 1>(Q, flux, grid, smem, st);
                default: return launch_adjoint_units<3, 2>(Q, flux, grid, smem, st);
            }
        }
        return launch_adjoint_units<-1, 0>(Q, flux, grid, smem, st);       // step counts at run time
    }
    const int64_t threads = L.n * 32;
    auto kern = in.tel->resample == RUBIX_RESAMPLE_FLUX ? k_adjoint_flux
                                                        : (table_mode(in.ssp, in.tel) ? k_adjoint<true> : k_adjoint<false>);
    kern<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
        (const int32_t *)(ws + L.off_permbuf[L.final_buf]), (const int32_t *)(ws + L.off_seg),
        (const int32_t *)(ws + L.off_key), (const float *)(ws + L.off_vlos), in.p->mass,
        in.p->log_age, in.p->log_z, (const Rec *)(ws + L.off_rec), (const float *)(ws + L.off_flux), gconv, P,
        g_mass, g_age, g_z, g_v);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix
