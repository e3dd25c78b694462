// K3: SSP lookup x mass, Doppler shift + resampling, per-spaxel accumulation
// ("The key part is the spectra calculation").
//
// Work unit = up to kChunk consecutive sorted particles of ONE spaxel x one channel tile.  One
// CTA (256 threads) per unit; thread t owns channels k0 + t + 256 i (i < CPT) and keeps their sums
// in registers, so a spaxel's spectrum is reduced without any atomic.  Per particle:
//   blend    the four corner templates are read once over the particle's rest-wavelength window
//            (8-byte loads, 256 B contiguous per warp instruction), blended with the mass-scaled
//            bilinear weights and stored in shared memory as interval entries
//            (S_j - D_j, D_j),  D_j = S_{j+1} - S_j   (S_{j+1} comes from the next lane by shuffle);
//   resample channel k reads ONE 8-byte entry: value = (S_j - D_j) + f1 * D_j with f1 = 1 + frac(x_k),
//            x_k from exact integer arithmetic (32-bit 12.20 local fixed point).
// The table is double buffered and the loop is software pipelined: the template loads of particle
// p+1 are issued, then particle p is resampled while they fly, then p+1 is blended (each further
// pass of loads is issued before the previous pass is consumed); one __syncthreads per particle.
// The unit's records are staged in shared memory once.
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

constexpr int kWarpSpan = 126;                       // table entries produced per warp per pass
constexpr int kPassSpan = kWarpSpan * (kAccThreads / 32);

__device__ __forceinline__ float2 ld2(const float *p) { return __ldg(reinterpret_cast<const float2 *>(p)); }

struct Win {                 // one particle's window in one channel tile
    const float *T;          // corner (i, j) template row
    int64_t base;            // x(k0) - j0 in 36.28 fixed point
    uint32_t b;              // step per channel, 4.28
    int32_t ka, kb;          // channels of this tile inside the SSP coverage (ka > kb: none)
    int32_t j0, nw;          // first SSP sample of the window (multiple of 4), entries needed
    float w0, w1, w2, w3;
};

struct LoadSet { float2 c[4][2]; };                  // 4 corners x 2 pair blocks

template <int CPT, bool VEC>
__global__ void __launch_bounds__(kAccThreads, 3)
k_accumulate(const __grid_constant__ AccumParams P)
{
    extern __shared__ __align__(16) float2 tab[];           // [2][wcap] interval entries, then records
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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

    if (U.count > 0) {
        int4 *srec = reinterpret_cast<int4 *>(tab + 2 * (size_t)P.wcap);
        {
            const int4 *g = reinterpret_cast<const int4 *>(P.rec + U.start);
            for (int i = tid; i < U.count * 3; i += kAccThreads) srec[i] = __ldg(g + i);
        }
        __syncthreads();
        const size_t row_a = (size_t)P.n_z * P.n_lambda;    // (i+1, j) - (i, j)
        const size_t row_z = (size_t)P.n_lambda;            // (i, j+1) - (i, j)
        const int nlm1 = P.n_lambda - 1, nlm2 = P.n_lambda - 2;

        auto window = [&](int q) -> Win {
            const int4 ra = srec[3 * q], rb = srec[3 * q + 1], rc = srec[3 * q + 2];
            Win W;
            W.w0 = __int_as_float(ra.x); W.w1 = __int_as_float(ra.y);
            W.w2 = __int_as_float(ra.z); W.w3 = __int_as_float(ra.w);
            W.b = (uint32_t)rb.y;
            const int64_t a = (int64_t)(((uint64_t)(uint32_t)rb.w << 32) | (uint32_t)rb.z);
            W.ka = max(k0, rc.x);
            W.kb = min(k_end, rc.y);
            W.T = P.flux + rb.x;
            W.base = 0; W.j0 = 0; W.nw = 0;
            if (W.ka <= W.kb) {
                const int64_t xa = a + (int64_t)W.b * W.ka, xb = a + (int64_t)W.b * W.kb;
                W.j0 = (int)(xa >> kFxFrac) & ~3;
                W.nw = min((int)(xb >> kFxFrac) - W.j0 + 1, P.wcap);    // last entry <= n_lambda-1
                W.base = a + (int64_t)W.b * k0 - ((int64_t)W.j0 << kFxFrac);
            }
            return W;
        };

        // ---- vector path: warp `warp`, pass starting at entry sb, lane handles entry pairs
        //      sb + 2 lane (+0, +64); lane 31 of the second block only feeds lane 30's neighbour
        auto issue = [&](LoadSet &L, const Win &W, int sb) {
            const int j1 = min(W.j0 + sb + 2 * lane, nlm2), j2 = min(W.j0 + sb + 64 + 2 * lane, nlm2);
            const float *t = W.T;
            L.c[0][0] = ld2(t + j1);                 L.c[0][1] = ld2(t + j2);
            L.c[1][0] = ld2(t + row_a + j1);         L.c[1][1] = ld2(t + row_a + j2);
            L.c[2][0] = ld2(t + row_z + j1);         L.c[2][1] = ld2(t + row_z + j2);
            L.c[3][0] = ld2(t + row_a + row_z + j1); L.c[3][1] = ld2(t + row_a + row_z + j2);
        };
        auto consume = [&](const LoadSet &L, const Win &W, int sb, float2 *buf) {
            const int p1 = sb + 2 * lane, p2 = p1 + 64;
            const float s10 = fmaf(W.w3, L.c[3][0].x, fmaf(W.w2, L.c[2][0].x, fmaf(W.w1, L.c[1][0].x, W.w0 * L.c[0][0].x)));
            const float s11 = fmaf(W.w3, L.c[3][0].y, fmaf(W.w2, L.c[2][0].y, fmaf(W.w1, L.c[1][0].y, W.w0 * L.c[0][0].y)));
            const float s20 = fmaf(W.w3, L.c[3][1].x, fmaf(W.w2, L.c[2][1].x, fmaf(W.w1, L.c[1][1].x, W.w0 * L.c[0][1].x)));
            const float s21 = fmaf(W.w3, L.c[3][1].y, fmaf(W.w2, L.c[2][1].y, fmaf(W.w1, L.c[1][1].y, W.w0 * L.c[0][1].y)));
            float nb1 = __shfl_sync(0xffffffffu, lane == 0 ? s20 : s10, (lane + 1) & 31);
            float nb2 = __shfl_down_sync(0xffffffffu, s20, 1);
            if (W.j0 + p1 + 2 > nlm1) nb1 = s11;            // interval N_l-1 is flat (only f = 0 reaches it)
            if (W.j0 + p2 + 2 > nlm1) nb2 = s21;
            float4 e1, e2;
            e1.y = s11 - s10; e1.x = s10 - e1.y; e1.w = nb1 - s11; e1.z = s11 - e1.w;
            e2.y = s21 - s20; e2.x = s20 - e2.y; e2.w = nb2 - s21; e2.z = s21 - e2.w;
            if (p1 < W.nw) *reinterpret_cast<float4 *>(buf + p1) = e1;
            if (lane < 31 && p2 < W.nw) *reinterpret_cast<float4 *>(buf + p2) = e2;
        };
        // ---- scalar path (row length odd or misaligned flux): plain per-entry blend
        auto blend_scalar = [&](const Win &W, float2 *buf) {
            for (int e = tid; e < W.nw; e += kAccThreads) {
                const int j = W.j0 + e, jn = min(j + 1, nlm1);
                const float *t = W.T;
                const float s0 = fmaf(W.w3, __ldg(t + row_a + row_z + j),
                                      fmaf(W.w2, __ldg(t + row_z + j), fmaf(W.w1, __ldg(t + row_a + j), W.w0 * __ldg(t + j))));
                const float s1 = fmaf(W.w3, __ldg(t + row_a + row_z + jn),
                                      fmaf(W.w2, __ldg(t + row_z + jn), fmaf(W.w1, __ldg(t + row_a + jn), W.w0 * __ldg(t + jn))));
                const float d = s1 - s0;
                buf[e] = make_float2(s0 - d, d);
            }
        };
        // all passes after the first one, software pipelined (A holds the pass being consumed)
        auto blend_rest = [&](LoadSet &A, const Win &W, float2 *buf) {
            LoadSet B;
            int sb = warp * kWarpSpan;
            while (true) {
                int nb = sb + kPassSpan;
                bool more = nb < W.nw;
                if (more) issue(B, W, nb);
                consume(A, W, sb, buf);
                if (!more) break;
                sb = nb; nb += kPassSpan; more = nb < W.nw;
                if (more) issue(A, W, nb);
                consume(B, W, sb, buf);
                if (!more) break;
                sb = nb;
            }
        };

        auto resample = [&](const Win &W, const float2 *buf) {
            const char *bytes = reinterpret_cast<const char *>(buf);
            // 12.20 local fixed point: exact truncation of the 36.28 value (stride 256 b / 256 = b)
            const uint32_t x0 = (uint32_t)((W.base + (int64_t)W.b * tid) >> 8);
            if (W.ka == k0 && W.kb == k_end) {              // whole tile inside the SSP coverage
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

        // prologue: table of particle 0
        Win cur = window(0);
        if (cur.ka <= cur.kb) {
            if (VEC) {
                LoadSet A;
                if (warp * kWarpSpan < cur.nw) { issue(A, cur, warp * kWarpSpan); blend_rest(A, cur, tab); }
            } else {
                blend_scalar(cur, tab);
            }
        }
        __syncthreads();
        for (int q = 0; q < U.count; ++q) {
            float2 *buf_next = tab + (size_t)((q + 1) & 1) * P.wcap;
            Win nxt;
            nxt.ka = 1; nxt.kb = 0;
            LoadSet A;
            bool blend_next = false;
            if (q + 1 < U.count) {
                nxt = window(q + 1);
                blend_next = (nxt.ka <= nxt.kb) && (!VEC || warp * kWarpSpan < nxt.nw);
                if (VEC && blend_next) issue(A, nxt, warp * kWarpSpan);     // loads fly during resample
            }
            if (cur.ka <= cur.kb) resample(cur, tab + (size_t)(q & 1) * P.wcap);
            if (blend_next) {
                if (VEC) blend_rest(A, nxt, buf_next);
                else blend_scalar(nxt, buf_next);
            }
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
static cudaError_t launch_acc(const AccumParams &P, bool vec, unsigned grid, size_t smem, cudaStream_t st)
{
    cudaError_t e;
    if (vec) {
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
    const bool vec = (in.ssp->n_lambda % 2 == 0) && (((uintptr_t)in.ssp->flux & 7u) == 0);
    const size_t smem = (size_t)2 * wcap * sizeof(float2) + (size_t)kChunk * sizeof(Rec);
    const unsigned grid = (unsigned)(L.max_units * P.n_tiles);
    cudaError_t e = cudaSuccess;
    {
        StageTimer t(1, st);
        switch (cpt) {
            case 15: e = launch_acc<15>(P, vec, grid, smem, st); break;
            case 8: e = launch_acc<8>(P, vec, grid, smem, st); break;
            case 4: e = launch_acc<4>(P, vec, grid, smem, st); break;
            case 2: e = launch_acc<2>(P, vec, grid, smem, st); break;
            default: e = launch_acc<1>(P, vec, grid, smem, st); break;
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
