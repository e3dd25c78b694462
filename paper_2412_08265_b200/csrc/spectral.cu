// K3: SSP lookup x mass, Doppler shift + resampling, per-spaxel accumulation
// ("The key part is the spectra calculation").
//
// Work unit = up to kChunk consecutive sorted particles of ONE spaxel x one channel tile.  One
// CTA (256 threads) per unit; thread t owns channels k0 + t + 256 i (i < CPT) and keeps their sums
// in registers, so a spaxel's spectrum is reduced without any atomic.  Per particle:
//   blend    the four corner templates are read once over the particle's rest-wavelength window
//            (16-byte loads, coalesced), blended with the mass-scaled bilinear weights and stored
//            in shared memory as interval entries  (S_j - D_j, D_j),  D_j = S_{j+1} - S_j ;
//   resample channel k reads ONE 8-byte entry: value = (S_j - D_j) + f1 * D_j with f1 = 1 + frac(x_k),
//            x_k from exact integer arithmetic (32-bit 12.20 local fixed point).
// The table is double buffered: the blend of particle p+1 overlaps the resampling of particle p
// with one __syncthreads per particle.
// Single-chunk spaxels write their cube row directly (each voxel exactly once, coalesced);
// spaxels with more particles write partial rows that k_reduce_partials sums in fixed order.
#include "common.cuh"

namespace rubix {

struct AccumParams {
    const float *flux;
    const Rec *rec;
    const Unit *units;
    const int32_t *totals;
    float *cube;
    float *partials;
    int32_t n_lambda, n_z, n_c, n_tiles, wcap;
};

__device__ __forceinline__ float4 ld4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }

template <int CPT, bool VEC4>
__global__ void __launch_bounds__(kAccThreads)
k_accumulate(const __grid_constant__ AccumParams P)
{
    extern __shared__ __align__(16) float2 tab[];           // [2][wcap] interval entries
    const int tid = threadIdx.x;
    const int tile = blockIdx.x % P.n_tiles;
    const int u = blockIdx.x / P.n_tiles;
    if (u >= P.totals[0]) return;
    const Unit U = P.units[u];
    constexpr int TC = CPT * kAccThreads;
    const int k0 = tile * TC;
    const int k_end = min(k0 + TC, P.n_c) - 1;              // last existing channel of this tile
    float *out = U.part_row >= 0 ? P.partials + (size_t)U.part_row * P.n_c
                                 : P.cube + (size_t)U.spaxel * P.n_c;
    float acc[CPT];
#pragma unroll
    for (int i = 0; i < CPT; ++i) acc[i] = 0.0f;

    // per-particle state of the particle being resampled (cur) and being blended (nxt)
    struct Win { int64_t base; uint32_t b; int32_t ka, kb; };
    Win cur{0, 0, 1, 0}, nxt{0, 0, 1, 0};
    const size_t row_a = (size_t)P.n_z * P.n_lambda;        // (i+1, j) - (i, j)
    const size_t row_z = (size_t)P.n_lambda;                // (i, j+1) - (i, j)

    auto blend = [&](int q, float2 *buf) -> Win {
        const int4 *rp = reinterpret_cast<const int4 *>(P.rec + U.start + q);
        const int4 ra = __ldg(rp), rb = __ldg(rp + 1), rc = __ldg(rp + 2);
        const float w0 = __int_as_float(ra.x), w1 = __int_as_float(ra.y);
        const float w2 = __int_as_float(ra.z), w3 = __int_as_float(ra.w);
        const uint32_t b = (uint32_t)rb.y;
        const int64_t a = (int64_t)(((uint64_t)(uint32_t)rb.w << 32) | (uint32_t)rb.z);
        Win W;
        W.b = b;
        W.ka = max(k0, rc.x);
        W.kb = min(k_end, rc.y);
        W.base = 0;
        if (W.ka > W.kb) return W;                          // nothing of this particle in the tile
        const int64_t xa = a + (int64_t)b * W.ka, xb = a + (int64_t)b * W.kb;
        const int j0 = (int)(xa >> kFxFrac) & ~3;
        const int jb = (int)(xb >> kFxFrac);                // <= n_lambda - 1
        W.base = a + (int64_t)b * k0 - ((int64_t)j0 << kFxFrac);
        const float *T = P.flux + rb.x;
        if (VEC4) {
            const int nq = min((jb - j0 + 4) >> 2, P.wcap >> 2);
            for (int qd = tid; qd < nq; qd += kAccThreads) {
                const int j = j0 + 4 * qd;
                const float *t = T + j;
                const float4 c0 = ld4(t), c1 = ld4(t + row_a), c2 = ld4(t + row_z), c3 = ld4(t + row_a + row_z);
                float s[5];
                s[0] = fmaf(w3, c3.x, fmaf(w2, c2.x, fmaf(w1, c1.x, w0 * c0.x)));
                s[1] = fmaf(w3, c3.y, fmaf(w2, c2.y, fmaf(w1, c1.y, w0 * c0.y)));
                s[2] = fmaf(w3, c3.z, fmaf(w2, c2.z, fmaf(w1, c1.z, w0 * c0.z)));
                s[3] = fmaf(w3, c3.w, fmaf(w2, c2.w, fmaf(w1, c1.w, w0 * c0.w)));
                if (j + 4 < P.n_lambda) {
                    s[4] = fmaf(w3, __ldg(t + row_a + row_z + 4),
                                fmaf(w2, __ldg(t + row_z + 4), fmaf(w1, __ldg(t + row_a + 4), w0 * __ldg(t + 4))));
                } else {
                    s[4] = s[3];                            // interval N_l-1: flat, only f = 0 reaches it
                }
                float4 e0, e1;
                e0.y = s[1] - s[0]; e0.x = s[0] - e0.y;
                e0.w = s[2] - s[1]; e0.z = s[1] - e0.w;
                e1.y = s[3] - s[2]; e1.x = s[2] - e1.y;
                e1.w = s[4] - s[3]; e1.z = s[3] - e1.w;
                float4 *dst = reinterpret_cast<float4 *>(buf + 4 * qd);
                dst[0] = e0;
                dst[1] = e1;
            }
        } else {
            const int nw = min(jb - j0 + 1, P.wcap);
            for (int e = tid; e < nw; e += kAccThreads) {
                const int j = j0 + e;
                const int jn = min(j + 1, P.n_lambda - 1);
                const float *t = T;
                const float s0 = fmaf(w3, __ldg(t + row_a + row_z + j),
                                      fmaf(w2, __ldg(t + row_z + j), fmaf(w1, __ldg(t + row_a + j), w0 * __ldg(t + j))));
                const float s1 = fmaf(w3, __ldg(t + row_a + row_z + jn),
                                      fmaf(w2, __ldg(t + row_z + jn), fmaf(w1, __ldg(t + row_a + jn), w0 * __ldg(t + jn))));
                const float d = s1 - s0;
                buf[e] = make_float2(s0 - d, d);
            }
        }
        return W;
    };

    auto resample = [&](const Win &W, const float2 *buf) {
        if (W.ka > W.kb) return;
        const char *bytes = reinterpret_cast<const char *>(buf);
        // 12.20 local fixed point: exact truncation of the 36.28 value (stride 256 b / 256 = b)
        const uint32_t x0 = (uint32_t)((W.base + (int64_t)W.b * tid) >> 8);
        if (W.ka == k0 && W.kb == k_end) {                  // whole tile inside the SSP coverage
#pragma unroll
            for (int i = 0; i < CPT; ++i) {
                const uint32_t x = x0 + (uint32_t)i * W.b;
                const float2 e = *reinterpret_cast<const float2 *>(bytes + ((x >> 17) & 0x7FF8u));
                const float f1 = __uint_as_float(((x << 3) & 0x7FFFF8u) | 0x3F800000u);
                acc[i] += fmaf(f1, e.y, e.x);
            }
        } else {
#pragma unroll
            for (int i = 0; i < CPT; ++i) {
                const int k = k0 + tid + i * kAccThreads;
                if (k >= W.ka && k <= W.kb) {
                    const uint32_t x = x0 + (uint32_t)i * W.b;
                    const float2 e = *reinterpret_cast<const float2 *>(bytes + ((x >> 17) & 0x7FF8u));
                    const float f1 = __uint_as_float(((x << 3) & 0x7FFFF8u) | 0x3F800000u);
                    acc[i] += fmaf(f1, e.y, e.x);
                }
            }
        }
    };

    if (U.count > 0) {
        cur = blend(0, tab);
        __syncthreads();
        for (int q = 0; q < U.count; ++q) {
            if (q + 1 < U.count) nxt = blend(q + 1, tab + (size_t)((q + 1) & 1) * P.wcap);
            resample(cur, tab + (size_t)(q & 1) * P.wcap);
            cur = nxt;
            __syncthreads();
        }
    }
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int k = k0 + tid + i * kAccThreads;
        if (k <= k_end) {
            if (U.part_row >= 0) out[k] = acc[i];
            else __stcs(out + k, acc[i]);                   // cube is written once, streamed
        }
    }
}

// Fixed-order second level for spaxels with more than kChunk particles: fp64 running sum over the
// chunk rows (the kernel is bandwidth bound; the fp64 adds are free and keep 1e6-term sums exact
// to fp32 rounding).
__global__ void __launch_bounds__(256)
k_reduce_partials(const float *__restrict__ partials, const int32_t *__restrict__ seg_off,
                  const int32_t *__restrict__ part_off, const int32_t *__restrict__ multi_list,
                  const int32_t *__restrict__ totals, int32_t n_c, float *__restrict__ cube)
{
    if ((int)blockIdx.x >= totals[2]) return;
    const int s = multi_list[blockIdx.x];
    const int cnt = seg_off[s + 1] - seg_off[s];
    const int chunks = (cnt + kChunk - 1) / kChunk;
    const float *rows = partials + (size_t)part_off[s] * n_c;
    for (int k = blockIdx.y * 256 + threadIdx.x; k < n_c; k += gridDim.y * 256) {
        double a = 0.0;
        for (int c = 0; c < chunks; ++c) a += (double)__ldcs(rows + (size_t)c * n_c + k);
        __stcs(cube + (size_t)s * n_c + k, (float)a);
    }
}

template <int CPT>
static cudaError_t launch_acc(const AccumParams &P, bool vec4, unsigned grid, size_t smem, cudaStream_t st)
{
    cudaError_t e;
    if (vec4) {
        e = cudaFuncSetAttribute(k_accumulate<CPT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k_accumulate<CPT, true><<<grid, kAccThreads, smem, st>>>(P);
    } else {
        e = cudaFuncSetAttribute(k_accumulate<CPT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k_accumulate<CPT, false><<<grid, kAccThreads, smem, st>>>(P);
    }
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

// Largest CPT in {15, 8, 4, 2, 1} whose table fits the 12.20 format; returns window capacity.
int choose_cpt(int n_c, double b_max, int *wcap_out)
{
    const int cand[5] = {15, 8, 4, 2, 1};
    for (int c = 0; c < 5; ++c) {
        const int cpt = cand[c];
        const int tc = cpt * kAccThreads;
        const int tiles = (n_c + tc - 1) / tc;
        // skip tilings that leave a whole 256-channel group of lanes idle (unless the smallest)
        if (cpt > 1 && (long long)tiles * tc - n_c >= kAccThreads) continue;
        const int wcap = (int)(b_max * tc) + 12;
        if (wcap > kTabMax) continue;
        *wcap_out = (wcap + 3) & ~3;
        return cpt;
    }
    *wcap_out = 0;
    return 0;
}

cudaError_t launch_accumulate(const PassInputs &in, const Layout &L, char *ws, float *cube, cudaStream_t st)
{
    const double b0 = (double)in.tel->dlambda / (double)in.ssp->dlambda;
    const double b_max = b0 / (1.0 - kBetaCap);
    int wcap = 0;
    const int cpt = choose_cpt(L.n_c, b_max, &wcap);
    if (cpt == 0) return cudaErrorInvalidConfiguration;
    AccumParams P;
    P.flux = in.ssp->flux;
    P.rec = (const Rec *)(ws + L.off_rec);
    P.units = (const Unit *)(ws + L.off_units);
    P.totals = (const int32_t *)(ws + L.off_totals);
    P.cube = cube;
    P.partials = (float *)(ws + L.off_partials);
    P.n_lambda = in.ssp->n_lambda;
    P.n_z = in.ssp->n_z;
    P.n_c = L.n_c;
    const int tc = cpt * kAccThreads;
    P.n_tiles = (L.n_c + tc - 1) / tc;
    P.wcap = wcap;
    const bool vec4 = (in.ssp->n_lambda % 4 == 0) && (((uintptr_t)in.ssp->flux & 15u) == 0);
    const size_t smem = (size_t)2 * wcap * sizeof(float2);
    const unsigned grid = (unsigned)(L.max_units * P.n_tiles);
    cudaError_t e = cudaSuccess;
    {
    StageTimer t(1, st);
    switch (cpt) {
        case 15: e = launch_acc<15>(P, vec4, grid, smem, st); break;
        case 8: e = launch_acc<8>(P, vec4, grid, smem, st); break;
        case 4: e = launch_acc<4>(P, vec4, grid, smem, st); break;
        case 2: e = launch_acc<2>(P, vec4, grid, smem, st); break;
        default: e = launch_acc<1>(P, vec4, grid, smem, st); break;
    }
    }
    if (e != cudaSuccess) return e;
    StageTimer t2(2, st);
    const unsigned gy = (unsigned)((L.n_c + 1023) / 1024);
    k_reduce_partials<<<dim3((unsigned)L.max_multi, gy), 256, 0, st>>>(
        P.partials, (const int32_t *)(ws + L.off_seg), (const int32_t *)(ws + L.off_partoff),
        (const int32_t *)(ws + L.off_multi), P.totals, L.n_c, cube);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix
