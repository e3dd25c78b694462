// K3 for piled-up spaxels: per-cell template reuse (SURVEY.md 8(d) row K3 "cut by per-cell template reuse", 7 "Contention
// config").
//
// Where a spaxel holds far more particles than the SSP grid has (age, Z) cells, the particle pass orders the particles of a
// spaxel by cell (particle_pass.cu, cell order), so consecutive particles of a work unit mostly share their four corner
// templates.  k_accumulate reads those corner windows again for every particle (4 x 12 KB through L1, 53 % of its L1
// wavefronts); here a CTA keeps them in REGISTERS -- thread (warp w, lane l) holds samples J0 + 128 (w + 8 ps) + 4 l .. + 3 of
// the four corner rows for its NPASS passes -- and reloads them only when the next particle's cell differs or its window
// leaves the loaded range [J0, J0 + CAP).  Per particle the blend is then eight packed FMAs and one 16-byte table store per
// pass and lane, no global load at all; the resample phase is k_accumulate's.  The decision is taken per particle from the
// records, so the kernel is correct for any order; the order only decides how often it reloads.
//
// 256 threads (thread t owns channels t + 256 i, i < CPT), two CTAs per SM; uniform grids, point rule, one channel tile.
#include <type_traits>

#include "accumulate.cuh"

namespace rubix {

constexpr int kCellThreads = 256;
constexpr int kCellWarps = kCellThreads / 32;
constexpr int kCellStep = kCellWarps * kPass;           // samples per pass of the whole CTA
constexpr int kCellMargin = 64;                         // room for the spread of the window starts inside a unit (Doppler shifts)

struct WinC {
    float w0, w1, w2, w3;
    int64_t base;            // x(0) - J0 in 36.28 fixed point
    uint32_t b;
    int32_t first;           // flux index of (corner (i,j), sample J0)
    int32_t ka, kb;
    int32_t lo, hi;          // the particle's samples, relative to J0: [lo, hi)
    int32_t J0;
    bool reload, interior;
};

template <int CPT, int NPASS>
__global__ void __launch_bounds__(kCellThreads, 2)
k_accumulate_cell(const __grid_constant__ AccumParams P)
{
    extern __shared__ __align__(16) float tab[];            // [2][CAP] samples S_j, then the records
    __shared__ int s_jmin, s_jmax;
    constexpr int CAP = NPASS * kCellStep;
    constexpr int NP2 = (CPT + 1) / 2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int u = blockIdx.x;
    if (u >= P.totals[0]) return;
    const Unit U = P.units[u];
    if (U.count == 0 && P.skip_empty) return;
    if (P.cell_split && !cell_kernel_owns(P, U.spaxel)) return;
    const int k_end = P.n_c - 1;
    float *out = U.part_row >= 0 ? P.partials + (size_t)U.part_row * P.n_c : P.cube + (size_t)U.spaxel * P.n_c;
    unsigned long long acc2[NP2];                           // channels (2 m, 2 m + 1) of the thread, packed
#pragma unroll
    for (int i = 0; i < NP2; ++i) acc2[i] = 0ull;
    auto add_to = [&](int i, float v) {                     // (the rare, guarded paths)
        acc2[i >> 1] = fadd2(acc2[i >> 1], (i & 1) ? pack2(0.0f, v) : pack2(v, 0.0f));
    };

    if (U.count > 0) {
        int4 *srec = reinterpret_cast<int4 *>(tab + 2 * (size_t)CAP);
        {
            const int4 *g = reinterpret_cast<const int4 *>(P.rec + U.start);
            for (int i = tid; i < U.count * 3; i += kCellThreads) srec[i] = __ldg(g + i);
        }
        if (tid == 0) { s_jmin = 0x7fffffff; s_jmax = 0; }
        __syncthreads();
        // ---- per unit, once: thread q turns record q into the window parameters the loop needs.  All windows of the unit
        //      share one table origin J0 (the smallest j0) when they fit the table together -- then a reload is needed only
        //      where the SSP cell changes; otherwise every particle loads its own range.
        {
            int4 ra = make_int4(0, 0, 0, 0), rb = ra, rc = ra;
            int prev_cell = -1;
            bool covered = false;
            if (tid < U.count) {
                ra = srec[3 * tid]; rb = srec[3 * tid + 1]; rc = srec[3 * tid + 2];
                covered = rc.x <= rc.y;
                if (covered) {
                    atomicMin(&s_jmin, rc.z);
                    atomicMax(&s_jmax, rc.z + rc.w);
                    for (int t = tid - 1; t >= 0; --t) {    // the covered particle before this one
                        const int4 c = srec[3 * t + 2];
                        if (c.x <= c.y) { prev_cell = srec[3 * t + 1].x; break; }
                    }
                }
            }
            __syncthreads();
            const bool common = s_jmax - s_jmin <= CAP;
            if (tid < U.count) {
                const int64_t a = (int64_t)(((uint64_t)(uint32_t)rb.w << 32) | (uint32_t)rb.z);
                const int J0 = common ? s_jmin : rc.z;
                const int lo = covered ? rc.z - J0 : 0, hi = covered ? lo + rc.w : 0;
                const int64_t base = a - ((int64_t)J0 << kFxFrac);
                const bool interior = covered && rc.x == 0 && rc.y == k_end;
                const bool reload = covered && (!common || prev_cell != rb.x);
                srec[3 * tid + 1] = make_int4((int)(uint32_t)base, (int)(base >> 32), rb.y, rb.x + J0);
                srec[3 * tid + 2] = make_int4(covered ? rc.x : 1, covered ? rc.y : 0,
                                              lo | (hi << 13) | (reload ? 1 << 26 : 0) | (interior ? 1 << 27 : 0), J0);
            }
            __syncthreads();
        }
        const int row_a = P.n_z * P.pitch, row_z = P.pitch;
        LoadSet K[NPASS];                                   // the loaded corner windows

        auto window = [&](int q) -> WinC {
            const int4 ra = srec[3 * q], rb = srec[3 * q + 1], rc = srec[3 * q + 2];
            WinC W;
            W.w0 = __int_as_float(ra.x); W.w1 = __int_as_float(ra.y);
            W.w2 = __int_as_float(ra.z); W.w3 = __int_as_float(ra.w);
            W.base = (int64_t)(((uint64_t)(uint32_t)rb.y << 32) | (uint32_t)rb.x);
            W.b = (uint32_t)rb.z;
            W.first = rb.w;
            W.ka = rc.x; W.kb = rc.y;
            W.lo = rc.z & 0x1FFF;
            W.hi = (rc.z >> 13) & 0x1FFF;
            W.reload = (rc.z >> 26) & 1;
            W.interior = (rc.z >> 27) & 1;
            W.J0 = rc.w;
            return W;
        };
        // all NPASS passes of the row range [J0, J0 + CAP) that start inside the (padded) row; the pad behind the grid copy
        // absorbs the overshoot of the last one
        auto load = [&](const WinC &W) {
            const float *t0 = P.flux + (W.first + warp * kPass + 4 * lane);
#pragma unroll
            for (int ps = 0; ps < NPASS; ++ps) {
                if (W.J0 + (warp + ps * kCellWarps) * kPass <= P.pitch) {
                    const float *t = t0 + ps * kCellStep;
                    K[ps].c[0] = ldg_quad(t);
                    K[ps].c[1] = ldg_quad(t + row_a);
                    K[ps].c[2] = ldg_quad(t + row_z);
                    K[ps].c[3] = ldg_quad(t + row_a + row_z);
                }
            }
        };
        // (table stores go to 32-bit shared addresses at compile-time offsets from one per-thread base)
        uint32_t dst_s = (uint32_t)__cvta_generic_to_shared(tab + warp * kPass + 4 * lane);
        asm volatile("" : "+r"(dst_s));                     // (kept in a register: ptxas would rebuild it before every store)
        auto blend = [&](const WinC &W, uint32_t buf_off) {
            const unsigned long long w0 = pack2(W.w0, W.w0), w1 = pack2(W.w1, W.w1);
            const unsigned long long w2 = pack2(W.w2, W.w2), w3 = pack2(W.w3, W.w3);
#pragma unroll
            for (int ps = 0; ps < NPASS; ++ps) {
                const int s = (warp + ps * kCellWarps) * kPass;
                if (s + kPass > W.lo && s < W.hi) {         // this pass holds samples of the particle's window
                    const LoadSet &L = K[ps];
                    const unsigned long long lo = ffma2(w3, L.c[3].lo, ffma2(w2, L.c[2].lo, ffma2(w1, L.c[1].lo, fmul2(w0, L.c[0].lo))));
                    const unsigned long long hi = ffma2(w3, L.c[3].hi, ffma2(w2, L.c[2].hi, ffma2(w1, L.c[1].hi, fmul2(w0, L.c[0].hi))));
                    asm volatile("st.shared.v2.b64 [%0], {%1, %2};" ::"r"(dst_s + buf_off + (uint32_t)(ps * kCellStep * 4)), "l"(lo), "l"(hi)
                                 : "memory");
                }
            }
        };

        const uint32_t m_addr = 0x3FFCu, m_frac = 0x7FFFF8u, one_bits = 0x3F800000u;
        const unsigned long long minus1 = pack2(-1.0f, -1.0f);
        auto sample = [&](int i, uint32_t x, const char *bytes) {
            const float *e = reinterpret_cast<const float *>(bytes + ((x >> 18) & m_addr));
            const float s0 = e[0], s1 = e[1];
            const float f = __uint_as_float(and_or(x << 3, m_frac, one_bits)) - 1.0f;    // frac(x_k), exact
            add_to(i, fmaf(f, s1 - s0, s0));
        };
        // two channels per packed instruction: d = s1 - s0, v = s0 + f d, acc += v
        auto sample2 = [&](int m, uint32_t xa, uint32_t xb, const char *bytes) {
            const float *ea = reinterpret_cast<const float *>(bytes + ((xa >> 18) & m_addr));
            const float *eb = reinterpret_cast<const float *>(bytes + ((xb >> 18) & m_addr));
            const unsigned long long s0 = pack2(ea[0], eb[0]), s1 = pack2(ea[1], eb[1]);
            const unsigned long long f1 = pack2(__uint_as_float(and_or(xa << 3, m_frac, one_bits)),
                                                __uint_as_float(and_or(xb << 3, m_frac, one_bits)));   // 1 + frac
            const unsigned long long f = fadd2(f1, minus1);
            const unsigned long long d = ffma2(s0, minus1, s1);
            acc2[m] = fadd2(acc2[m], ffma2(f, d, s0));
        };
        // channel stride 256 b / 256 = b in the 2^-20 local format: exact for every b
        auto resample = [&](const WinC &W, const float *buf) {
            const char *bytes = reinterpret_cast<const char *>(buf);
            const uint32_t x0 = (uint32_t)((W.base + (int64_t)W.b * tid) >> 8);
            if (W.interior) {                               // the whole spectrum inside the SSP coverage
#pragma unroll
                for (int m = 0; m < CPT / 2; ++m) sample2(m, x0 + (uint32_t)(2 * m) * W.b, x0 + (uint32_t)(2 * m + 1) * W.b, bytes);
                if (CPT & 1) sample(CPT - 1, x0 + (uint32_t)(CPT - 1) * W.b, bytes);
            } else {
#pragma unroll
                for (int i = 0; i < CPT; ++i) {
                    const int k = tid + i * kCellThreads;
                    if (k >= W.ka && k <= W.kb) sample(i, x0 + (uint32_t)i * W.b, bytes);
                }
            }
        };

        // particle q is resampled from table PAR while particle q + 1 is blended into the other one (the loop is unrolled by
        // two so that both table addresses are compile-time offsets)
        WinC cur = window(0);
        if (cur.reload) load(cur);
        blend(cur, 0u);
        __syncthreads();
        auto step = [&](auto par_c, int q) {
            constexpr int PAR = decltype(par_c)::value;
            const bool have = q + 1 < U.count;
            WinC nxt = cur;
            if (have) {
                nxt = window(q + 1);
                if (nxt.reload) load(nxt);                  // K was consumed when `cur` was blended: the loads fly during the resample
            }
            resample(cur, tab + PAR * CAP);
            if (have) blend(nxt, (uint32_t)((PAR ^ 1) * CAP * 4));
            cur = nxt;
            __syncthreads();
        };
        for (int q = 0; q < U.count; q += 2) {
            step(std::integral_constant<int, 0>{}, q);
            if (q + 1 < U.count) step(std::integral_constant<int, 1>{}, q + 1);
        }
    }
    float *mirror = nullptr, *mirror2 = nullptr;
    if (U.part_row < 0) {
        const int sp = P.units[u].spaxel;
        if (P.mirror_lo && sp < P.mirror_lo_n) mirror = P.mirror_lo + (size_t)sp * P.n_c;
        if (P.mirror_hi && sp >= P.mirror_hi_first) mirror2 = P.mirror_hi + (size_t)(sp - P.mirror_hi_first) * P.n_c;
    }
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int k = tid + i * kCellThreads;
        const float2 pr = unpack2(acc2[i >> 1]);
        const float v = (i & 1) ? pr.y : pr.x;
        if (k <= k_end) {
            if (U.part_row >= 0) out[k] = v;
            else {
                __stcs(out + k, v);
                if (mirror) mirror[k] = v;
                if (mirror2) mirror2[k] = v;
            }
        }
    }
}

// ---- host --------------------------------------------------------------------------------------
static int cell_cpt(int32_t n_c) { return n_c <= 2 * kCellThreads ? 2 : (n_c <= 8 * kCellThreads ? 8 : 15); }

// samples the table must hold: every channel a thread may address (CPT x 256 of them) plus the spread of the window starts
static int cell_need(int32_t n_c, double b_max)
{
    const int tc = cell_cpt(n_c) * kCellThreads;
    return (int)(b_max * tc) + kRowAlign + 4 + kCellMargin;
}

// point rule only: under the bin average the kernel would be bound by its instruction count even harder (measured on the
// contention workload: 48.2 ms with the heavy spaxels here against 44 ms with k_accumulate<FLUX> alone)
bool cell_kernel_fits(int32_t n_c, double b_max, bool flux)
{
    return !flux && n_c <= 15 * kCellThreads && cell_need(n_c, b_max) <= kTabMax;
}

template <int CPT, int NPASS>
static cudaError_t launch_cell3(const AccumParams &P, unsigned grid, cudaStream_t st)
{
    // the masked 12.20 address of a lane beyond the last channel may point up to 16 KB past a table: pad
    const size_t smem = (size_t)2 * NPASS * kCellStep * sizeof(float) + (size_t)kChunk * sizeof(Rec) + (NPASS < 4 ? 16384 : 0);
    auto kern = k_accumulate_cell<CPT, NPASS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kCellThreads, smem, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

template <int CPT>
static cudaError_t launch_cell2(const AccumParams &P, int npass, unsigned grid, cudaStream_t st)
{
    return npass <= 2 ? launch_cell3<CPT, 2>(P, grid, st) : launch_cell3<CPT, 4>(P, grid, st);
}

cudaError_t launch_accumulate_cell(const AccumParams &P, double b_max, unsigned grid, cudaStream_t st)
{
    const int npass = (cell_need(P.n_c, b_max) + kCellStep - 1) / kCellStep;
    switch (cell_cpt(P.n_c)) {
        case 2: return launch_cell2<2>(P, npass, grid, st);
        case 8: return launch_cell2<8>(P, npass, grid, st);
        default: return launch_cell2<15>(P, npass, grid, st);
    }
}

}  // namespace rubix
