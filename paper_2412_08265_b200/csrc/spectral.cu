// K3: SSP lookup x mass, Doppler shift + resampling, per-spaxel accumulation
// ("The key part is the spectra calculation").
//
// Work unit = up to kChunk consecutive sorted particles of ONE spaxel x one channel tile.  One
// CTA (128 threads, five resident per SM) per unit; thread t owns channels k0 + t + 128 i (i < CPT, CPT = 29
// for 3700 channels) and keeps their sums in registers, so a spaxel's spectrum is reduced without any atomic.
// Small CTAs de-synchronise the load-heavy blend phases and the shared-memory-heavy resample phases of the
// CTAs sharing an SM, which keeps the L1 data pipe busier (r01: 3.51 -> 3.28 ms against 256-thread CTAs).
// Per particle:
//   blend    the four corner templates are read once over the particle's rest-wavelength window
//            and blended with the mass-scaled bilinear weights into a shared-memory table S_j.
//            The window starts on a multiple of 32 samples of the padded workspace copy of the grid
//            (rows padded to 128 B), so a warp pass is four 512-byte, line-aligned 16-byte-per-lane
//            loads (one per corner), eight packed fp32x2 FMAs and one 16-byte table store per lane:
//            every L1 wavefront moves a full 128 bytes;
//   resample channel k reads S_j and S_{j+1} (the 32 lanes of a warp read ~25 consecutive words: no
//            bank conflict) and adds S_j + f (S_{j+1} - S_j); j and f come from exact integer
//            arithmetic on x_k (32-bit 12.20 local fixed point).
// The table is double buffered and the loop is software pipelined: the template loads of particle
// p+1 are issued, then particle p is resampled while they fly, then p+1 is blended (each further
// pass of loads is issued before the previous pass is consumed); one __syncthreads per particle.
// The unit's records are staged in shared memory once.
// Single-chunk spaxels write their cube row directly (each voxel exactly once, coalesced);
// spaxels with more particles write partial rows that k_reduce_partials sums in fixed order.
#include "accumulate.cuh"

namespace rubix {

struct Win {                 // one particle's window in one channel tile
    int64_t base;            // x(k0) - j0 in 36.28 fixed point
    uint32_t b;              // step per channel, 4.28
    int32_t ka, kb;          // channels of this tile inside the SSP coverage (ka > kb: none)
    int32_t first, nw;       // flux index of (corner (i,j), sample j0); samples needed
    int32_t j0;              // first table sample (multiple of 32)
    float w0, w1, w2, w3;
    double g;                // GEN: the particle's Doppler value (gen_coord.cuh)
};

// SINGLE: the whole spectrum is one tile (n_tiles == 1): window (j0, nw) comes from the record.
// FLUX: flux-conserving resampling (RUBIX_RESAMPLE_FLUX): x_k is the lower edge of bin k and the
// channel value is the exact integral of the table's piecewise-linear interpolant over
// [x_k, x_{k+1}] (clipped to the SSP coverage), divided by the bin width B.
// LOGX: table mode (readings R15 / R16: log-sampled SSP grid, explicit channel wavelengths):
// x_k = Y[k] c + a with the per-launch table Y = xtab and the particle's (c, a); c (2.30 fixed point) travels in
// the record's b slot.  The thread keeps Y of its CPT channels relative to the tile start in registers (12.20).
// GEN: general-grid mode (readings R20 / R21, gen_coord.cuh): x = gen_coord(tab[e], g) per sample in fp64, e = channel
// (point rule) or bin edge (FLUX: channel k is the bin between edges k and k + 1, averaged over its FULL width in x).
// NARROW (GEN + FLUX): no bin is wider than one SSP sample, so a bin touches at most two knot intervals and is integrated
// through three samples without a branch (as the fixed-point kernel does for B <= 1).
// GEN = 0: off; 1 + kind of gen_coord.cuh otherwise (1 linear, 2 log-sampled, 3 listed SSP wavelengths).
template <int CPT, bool SINGLE, int DEPTH, int MINB, bool FLUX, bool LOGX, int GEN = 0, bool NARROW = false>
__global__ void __launch_bounds__(kAccThreads, MINB)
k_accumulate(const __grid_constant__ AccumParams P)
{
    extern __shared__ __align__(16) float tab[];            // [2][wcap] samples S_j, then the records
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = SINGLE ? 0 : blockIdx.x % P.n_tiles;
    const int u = SINGLE ? blockIdx.x : blockIdx.x / P.n_tiles;
    if (u >= P.totals[0]) return;
    const Unit U = P.units[u];
    if (U.count == 0 && P.skip_empty) return;
    if (P.cell_split && cell_kernel_owns(P, U.spaxel)) return;
    constexpr int TC = CPT * kAccThreads;
    const int k0 = tile * TC;
    const int k_end = min(k0 + TC, P.n_c) - 1;              // last existing channel of this tile
    float *out = U.part_row >= 0 ? P.partials + (size_t)U.part_row * P.n_c
                                 : P.cube + (size_t)U.spaxel * P.n_c;
    float acc[CPT];
    uint32_t xl[LOGX ? CPT : 1];
    uint32_t wd[(LOGX && FLUX) ? CPT : 1];                  // LOGX + FLUX: width of the thread's bins at beta = 0 (2^-20 samples)
    int64_t x_tile0 = 0;                                    // LOGX: xtab[k0]
#pragma unroll
    for (int i = 0; i < CPT; ++i) acc[i] = 0.0f;

    if (U.count > 0) {
        if (LOGX) {                                         // the table exists only when there are particles
            x_tile0 = P.xtab[k0];
#pragma unroll
            for (int i = 0; i < CPT; ++i) {
                const int k = k0 + tid + i * kAccThreads;
                xl[i] = (uint32_t)((P.xtab[min(k, P.n_c)] - x_tile0) >> 8);
                if (FLUX) wd[i] = (uint32_t)((P.xtab[min(k + 1, P.n_c)] - P.xtab[min(k, P.n_c)]) >> 8);
            }
        }
        int4 *srec = reinterpret_cast<int4 *>(tab + 2 * (size_t)P.wcap);
        {
            const int4 *g = reinterpret_cast<const int4 *>(P.rec + U.start);
            for (int i = tid; i < U.count * 3; i += kAccThreads) srec[i] = __ldg(g + i);
        }
        __syncthreads();
        const int row_a = P.n_z * P.pitch;                  // (i+1, j) - (i, j)
        const int row_z = P.pitch;                          // (i, j+1) - (i, j)

        auto window = [&](int q) -> Win {
            const int4 ra = srec[3 * q], rb = srec[3 * q + 1], rc = srec[3 * q + 2];
            Win W;
            W.w0 = __int_as_float(ra.x); W.w1 = __int_as_float(ra.y);
            W.w2 = __int_as_float(ra.z); W.w3 = __int_as_float(ra.w);
            W.b = (uint32_t)rb.y;
            const int64_t a = (int64_t)(((uint64_t)(uint32_t)rb.w << 32) | (uint32_t)rb.z);
            W.g = GEN ? __longlong_as_double(a) : 0.0;
            int j0;
            if (SINGLE) {                                   // k0 = 0, k_end = n_c - 1 >= k_hi
                W.ka = rc.x; W.kb = rc.y;
                j0 = rc.z; W.nw = rc.w;
            } else if (GEN) {
                W.ka = max(k0, rc.x);
                W.kb = min(k_end, rc.y);
                j0 = 0; W.nw = 0;
                if (W.ka <= W.kb) {                         // as prepare_records_body, for this tile's channels
                    const double x_top = (double)(P.n_lambda - 1);
                    const double xa = fmin(fmax(gen_coord_k<GEN - 1>(P.gen, P.gen.tab[W.ka], W.g) - 1e-6, 0.0), x_top);
                    const double xb = fmin(fmax(gen_coord_k<GEN - 1>(P.gen, P.gen.tab[W.kb + (FLUX ? 1 : 0)], W.g) + 1e-6, 0.0), x_top);
                    j0 = (int)xa & ~(kRowAlign - 1);
                    W.nw = (int)xb - j0 + 2;
                }
            } else {
                W.ka = max(k0, rc.x);
                W.kb = min(k_end, rc.y);
                j0 = 0; W.nw = 0;
                if (W.ka <= W.kb) {
                    int64_t xa = a + (int64_t)W.b * W.ka, xb = a + (int64_t)W.b * (W.kb + (FLUX ? 1 : 0));
                    if (LOGX) {
                        const double c = (double)W.b * (1.0 / (double)(1u << 30));
                        xa = a + __double2ll_rn((double)P.xtab[W.ka] * c);
                        xb = a + __double2ll_rn((double)P.xtab[W.kb + (FLUX ? 1 : 0)] * c);
                    }
                    if (FLUX) {                             // bins are clipped to the coverage
                        xa = max(xa, (int64_t)0);
                        xb = min(xb, (int64_t)(P.n_lambda - 1) << kFxFrac);
                    }
                    // LOGX: the resampler's x may sit up to 2 units of 2^-20 below the exact value, so the window
                    // starts one group earlier when x_ka is that close above a multiple of kRowAlign
                    j0 = (int)(max(xa - (LOGX ? 1024 : 0), (int64_t)0) >> kFxFrac) & ~(kRowAlign - 1);
                    W.nw = (int)(xb >> kFxFrac) - j0 + 2;   // samples j0 .. j_max + 1
                }
            }
            W.first = rb.x + j0;
            W.j0 = j0;
            W.base = GEN ? 0 : a + (LOGX ? __double2ll_rn((double)x_tile0 * ((double)W.b * (1.0 / (double)(1u << 30))))
                               : (int64_t)W.b * k0) - ((int64_t)j0 << kFxFrac);
            return W;
        };

        // ---- blend: warp `warp` produces samples [128 pass, 128 pass + 128) for pass = warp, warp+8..
        //      Loads and stores are unconditional: the padded grid copy and the table (a whole
        //      number of passes) absorb the overshoot.  A register ring of DEPTH load sets per warp:
        //      the first DEPTH passes of the next particle are issued before the current particle
        //      is resampled (their latency hides behind it), later passes refill the ring.
        constexpr int kStep = kAccWarps * kPass;            // samples between two passes of a warp
        auto tex_quad = [&](const float *t) -> Quad {
            const float4 v = tex1Dfetch<float4>(P.tex, (int)((t - P.flux) >> 2));
            Quad q;
            q.lo = pack2(v.x, v.y); q.hi = pack2(v.z, v.w);
            return q;
        };
        auto issue = [&](LoadSet &L, const float *t0) {
            constexpr bool NA = GEN == 3;
            L.c[0] = RUBIX_TEX_CORNERS >= 4 ? tex_quad(t0) : ldg_quad<NA>(t0);
            L.c[1] = RUBIX_TEX_CORNERS >= 3 ? tex_quad(t0 + row_a) : ldg_quad<NA>(t0 + row_a);
            L.c[2] = RUBIX_TEX_CORNERS >= 2 ? tex_quad(t0 + row_z) : ldg_quad<NA>(t0 + row_z);
            L.c[3] = RUBIX_TEX_CORNERS >= 1 ? tex_quad(t0 + row_a + row_z) : ldg_quad<NA>(t0 + row_a + row_z);
        };
        auto consume = [&](const LoadSet &L, const Win &W, float *dst) {
            const unsigned long long w0 = pack2(W.w0, W.w0), w1 = pack2(W.w1, W.w1);
            const unsigned long long w2 = pack2(W.w2, W.w2), w3 = pack2(W.w3, W.w3);
            const unsigned long long lo = ffma2(w3, L.c[3].lo, ffma2(w2, L.c[2].lo, ffma2(w1, L.c[1].lo, fmul2(w0, L.c[0].lo))));
            const unsigned long long hi = ffma2(w3, L.c[3].hi, ffma2(w2, L.c[2].hi, ffma2(w1, L.c[1].hi, fmul2(w0, L.c[0].hi))));
            sts_quad(dst, lo, hi);
        };
        auto prefetch = [&](LoadSet (&L)[DEPTH], const Win &W) {
            const float *t0 = P.flux + (W.first + warp * kPass + 4 * lane);
#pragma unroll
            for (int d = 0; d < DEPTH; ++d)
                if ((warp + d * kAccWarps) * kPass < W.nw) issue(L[d], t0 + d * kStep);
        };
        // every pass sits at a compile-time offset from one per-particle pointer (immediate load / store
        // offsets, no loop-carried address arithmetic); a warp has at most kTabMax / kStep passes
        constexpr int kMaxPass = kTabMax / kStep;
        auto blend_all = [&](LoadSet (&L)[DEPTH], const Win &W, float *buf) {
            const float *t0 = P.flux + (W.first + warp * kPass + 4 * lane);
            float *dst = buf + warp * kPass + 4 * lane;
            const int left = W.nw - warp * kPass;           // samples from this warp's first pass to the end
#pragma unroll
            for (int ps = 0; ps < kMaxPass; ++ps) {
                if (ps * kStep < left) {
                    consume(L[ps % DEPTH], W, dst + ps * kStep);
                    if (ps + DEPTH < kMaxPass && (ps + DEPTH) * kStep < left)
                        issue(L[ps % DEPTH], t0 + (ps + DEPTH) * kStep);
                }
            }
        };

        const uint32_t m_addr = 0x3FFCu, m_frac = 0x7FFFF8u, one_bits = 0x3F800000u;
        auto sample = [&](int i, uint32_t x, const char *bytes) {
            const float *e = reinterpret_cast<const float *>(bytes + ((x >> 18) & m_addr));
            const float s0 = e[0], s1 = e[1];
            const float f = __uint_as_float(and_or(x << 3, m_frac, one_bits)) - 1.0f;    // frac(x_k), exact
            acc[i] += fmaf(f, s1 - s0, s0);
        };
        // exact integral of the table's interpolant over local positions [xl, xh] (12.20), times inv_b
        auto flux_sample = [&](int i, uint32_t xl, uint32_t xh, float inv_b, const float *tabp) {
            const uint32_t jl = xl >> 20, jh = xh >> 20;
            const float fl = (float)(xl & 0xFFFFFu) * (1.0f / 1048576.0f);
            const float fh = (float)(xh & 0xFFFFFu) * (1.0f / 1048576.0f);
            const float a0 = tabp[jl], a1 = tabp[jl + 1];
            float tot;
            if (jl == jh) {
                tot = (fh - fl) * fmaf(0.5f * (fl + fh), a1 - a0, a0);
            } else {
                const float c0 = tabp[jh], c1 = tabp[jh + 1];
                tot = 0.5f * (1.0f - fl) * (fmaf(fl, a1 - a0, a0) + a1);
                tot = fmaf(0.5f * fh, c0 + fmaf(fh, c1 - c0, c0), tot);
                for (uint32_t j = jl + 1; j < jh; ++j) tot = fmaf(0.5f, tabp[j] + tabp[j + 1], tot);
            }
            acc[i] = fmaf(tot, inv_b, acc[i]);
        };
        auto resample = [&](const Win &W, const float *buf) {
            const char *bytes = reinterpret_cast<const char *>(buf);
            if (GEN) {
                // Branch-free per sample (a channel outside [ka, kb] or outside the coverage is computed on a clamped
                // position and masked), so that the unrolled iterations overlap their table loads and fp64 chains.
                const double x_top = (double)(P.n_lambda - 1), j0d = (double)W.j0;
                const int e_max = P.n_c - (FLUX ? 0 : 1);
                // local position -> (table index, fraction); one fp64 subtraction, then everything in fp32
                auto split = [&](double x, int &j, float &f) {
                    const double xl = x - j0d;
                    j = (int)xl;
                    f = (float)(xl - (double)j);
                };
#pragma unroll                                              // fully: acc[i] must stay in registers
                for (int i = 0; i < CPT; ++i) {
                    const int k = k0 + tid + i * kAccThreads;
                    const bool in_k = k >= W.ka && k <= W.kb;
                    const int kc = min(k, e_max);
                    if (!FLUX) {
                        const double x = gen_coord_k<GEN - 1>(P.gen, __ldg(P.gen.tab + kc), W.g);
                        const bool ok = in_k && x >= 0.0 && x <= x_top;
                        int j; float f;
                        split(ok ? x : j0d, j, f);
                        const float s0 = buf[j], s1 = buf[j + 1];
                        acc[i] += ok ? fmaf(f, s1 - s0, s0) : 0.0f;
                    } else {
                        const double xlo = gen_coord_k<GEN - 1>(P.gen, __ldg(P.gen.tab + kc), W.g);
                        const double xhi = gen_coord_k<GEN - 1>(P.gen, __ldg(P.gen.tab + min(kc + 1, e_max)), W.g);
                        const double cl = fmax(xlo, 0.0), ch = fmin(xhi, x_top);
                        const bool ok = in_k && ch > cl;
                        float tot;
                        if (NARROW) {
                            // I(u) = integral of the interpolant from knot ja to ja + u (u < 2) through a0, a1, a2
                            int ja; float fa;
                            split(ok ? cl : j0d, ja, fa);
                            const float u = fa + (ok ? (float)(ch - cl) : 0.0f);
                            const float u1 = fminf(u, 1.0f), u2 = fmaxf(u - 1.0f, 0.0f);
                            const float a0 = buf[ja], a1 = buf[ja + 1], a2r = buf[ja + 2];
                            const float a2 = u > 1.0f ? a2r : a1;         // buf[ja + 2] may lie beyond the blended window
                            const float d1 = a1 - a0, d2 = a2 - a1;
                            const float il = fa * fmaf(0.5f * fa, d1, a0);
                            float iu = u1 * fmaf(0.5f * u1, d1, a0);
                            iu = fmaf(u2, fmaf(0.5f * u2, d2, a1), iu);
                            tot = iu - il;
                        } else {
                            int ja, jb; float fa, fb;
                            split(ok ? cl : j0d, ja, fa);
                            split(ok ? ch : j0d, jb, fb);
                            const float a0 = buf[ja], a1 = buf[ja + 1], c0 = buf[jb], c1 = buf[jb + 1];
                            // same interval: (fb - fa) * value at the midpoint; else the two partial trapezoids + whole intervals
                            tot = (fb - fa) * fmaf(0.5f * (fa + fb), a1 - a0, a0);
                            if (ja != jb) {
                                tot = 0.5f * (1.0f - fa) * (fmaf(fa, a1 - a0, a0) + a1);
                                tot = fmaf(0.5f * fb, c0 + fmaf(fb, c1 - c0, c0), tot);
                                for (int j = ja + 1; j < jb; ++j) tot = fmaf(0.5f, buf[j] + buf[j + 1], tot);
                            }
                        }
                        const float inv_w = __fdividef(1.0f, (float)(xhi - xlo));   // the FULL width of the bin
                        acc[i] = ok ? fmaf(tot, inv_w, acc[i]) : acc[i];
                    }
                }
                return;
            }
            if (FLUX && LOGX) {
                // Bin average in table mode (reading R20): the table holds the bin edges, x_e = Y[e] c + a; the thread keeps
                // the lower edge and the width of its bins at beta = 0 (12.20), both scale with c.  Lower edge and width
                // are truncated separately, so neighbouring bins share their edge to 2^-20 samples (not bit for bit).
                const int64_t j0s = (int64_t)W.j0 << kFxFrac;
                const int64_t cov_lo = -j0s >> 8, cov_hi = (((int64_t)(P.n_lambda - 1) << kFxFrac) - j0s) >> 8;   // 2^-20
                const double cd = (double)W.b * (1.0 / (double)(1u << 30));
                const int64_t base20 = W.base >> 8;
                const int64_t last20 = base20 + (__double2ll_rn((double)(P.xtab[min(k_end + 1, P.n_c)] - x_tile0) * cd) >> 8);
                const bool interior = W.ka == k0 && W.kb == k_end && base20 >= cov_lo + 4 && last20 + 4 <= cov_hi;
                const uint32_t x0 = (uint32_t)base20;
                if (interior && P.narrow) {
#pragma unroll
                    for (int i = 0; i < CPT; ++i) {
                        const uint32_t x = x0 + (uint32_t)(((uint64_t)xl[i] * W.b) >> 30);
                        const float width = (float)(uint32_t)(((uint64_t)wd[i] * W.b) >> 30) * (1.0f / 1048576.0f);
                        const float *e = reinterpret_cast<const float *>(bytes + ((x >> 18) & m_addr));
                        const float a0 = e[0], a1 = e[1], a2r = e[2];
                        const float fl = __uint_as_float(and_or(x << 3, m_frac, one_bits)) - 1.0f;
                        const float u = fl + width;
                        const float u1 = fminf(u, 1.0f), u2 = fmaxf(u - 1.0f, 0.0f);
                        const float a2 = u > 1.0f ? a2r : a1;     // e[2] may lie beyond the table
                        const float d1 = a1 - a0, d2 = a2 - a1;
                        const float il = fl * fmaf(0.5f * fl, d1, a0);
                        float iu = u1 * fmaf(0.5f * u1, d1, a0);
                        iu = fmaf(u2, fmaf(0.5f * u2, d2, a1), iu);
                        acc[i] = fmaf(iu - il, __fdividef(1.0f, width), acc[i]);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < CPT; ++i) {
                        const int k = k0 + tid + i * kAccThreads;
                        if (k >= W.ka && k <= W.kb) {
                            const int64_t lo = base20 + (int64_t)(((uint64_t)xl[i] * W.b) >> 30);
                            const uint32_t wx = (uint32_t)(((uint64_t)wd[i] * W.b) >> 30);
                            const int64_t cl = max(lo, cov_lo), ch = min(lo + (int64_t)wx, cov_hi);
                            if (ch > cl) flux_sample(i, (uint32_t)cl, (uint32_t)ch, 1048576.0f / (float)wx, buf);
                        }
                    }
                }
                return;
            }
            if (FLUX) {
                const float inv_b = (float)(1 << kFxFrac) / (float)W.b;
                // coverage in local coordinates; W.base = x(k0) - (j0 << 28)
                const int64_t j0s = (int64_t)W.j0 << kFxFrac;
                const int64_t cov_lo = -j0s, cov_hi = ((int64_t)(P.n_lambda - 1) << kFxFrac) - j0s;
                const int64_t e0 = W.base + (int64_t)W.b * tid;          // lower edge of channel k0 + tid
                const bool interior = W.ka == k0 && W.kb == k_end && W.base >= cov_lo &&
                                      W.base + (int64_t)W.b * (k_end - k0 + 1) <= cov_hi;
                if (interior) {
                    // both edges are truncated by the same function of k, so neighbouring bins share
                    // their edge exactly (stride 128 b / 256 = b / 2 with even b keeps the truncation exact)
                    const uint32_t xl0 = (uint32_t)(e0 >> 8), xh0 = (uint32_t)((e0 + (int64_t)W.b) >> 8);
                    if (W.b <= (1u << kFxFrac)) {
                        // bins no wider than one SSP sample touch at most two knot intervals: branch-free
                        // I(u) = integral of the interpolant from knot jl to jl + u (u < 2) through
                        // the three samples a0, a1, a2;  F = (I(fl + width) - I(fl)) / B
                        const float width = (float)(xh0 - xl0) * (1.0f / 1048576.0f);
#pragma unroll
                        for (int i = 0; i < CPT; ++i) {
                            const uint32_t x = xl0 + (uint32_t)i * (W.b >> 1);
                            const float *e = reinterpret_cast<const float *>(bytes + ((x >> 18) & m_addr));
                            const float a0 = e[0], a1 = e[1], a2r = e[2];
                            const float fl = __uint_as_float(and_or(x << 3, m_frac, one_bits)) - 1.0f;
                            const float u = fl + width;
                            const float u1 = fminf(u, 1.0f), u2 = fmaxf(u - 1.0f, 0.0f);
                            const float a2 = u > 1.0f ? a2r : a1;     // e[2] may lie beyond the table
                            const float d1 = a1 - a0, d2 = a2 - a1;
                            const float il = fl * fmaf(0.5f * fl, d1, a0);
                            float iu = u1 * fmaf(0.5f * u1, d1, a0);
                            iu = fmaf(u2, fmaf(0.5f * u2, d2, a1), iu);
                            acc[i] = fmaf(iu - il, inv_b, acc[i]);
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < CPT; ++i)
                            flux_sample(i, xl0 + (uint32_t)i * (W.b >> 1), xh0 + (uint32_t)i * (W.b >> 1), inv_b, buf);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < CPT; ++i) {
                        const int k = k0 + tid + i * kAccThreads;
                        if (k >= W.ka && k <= W.kb) {
                            const int64_t lo = e0 + (int64_t)W.b * (i * kAccThreads);
                            const int64_t cl = max(lo, cov_lo), ch = min(lo + (int64_t)W.b, cov_hi);
                            if (ch > cl) flux_sample(i, (uint32_t)(cl >> 8), (uint32_t)(ch >> 8), inv_b, buf);
                        }
                    }
                }
                return;
            }
            // 12.20 local fixed point: exact truncation of the 36.28 value (channel stride 128 b / 256 = b / 2, b is even)
            // LOGX: x = (tile-relative table value of the channel) x c + (particle base), truncated to 2^-20
            const uint32_t x0 = LOGX ? (uint32_t)(W.base >> 8) : (uint32_t)((W.base + (int64_t)W.b * tid) >> 8);
            // LOGX: the sum of separately truncated terms can sit 1-2 units of 2^-20 BELOW the exact x_k that
            // prepare_records_body used for k_lo.  Where the window starts at knot 0 (j0 = 0) a channel just above
            // the knot would wrap below zero: such windows take the guarded branch, which clamps at the knot.
            if (W.ka == k0 && W.kb == k_end && !(LOGX && W.j0 == 0)) {   // whole tile inside the SSP coverage
#pragma unroll
                for (int i = 0; i < CPT; ++i) sample(i, LOGX ? x0 + (uint32_t)(((uint64_t)xl[i] * W.b) >> 30) : x0 + (uint32_t)i * (W.b >> 1), bytes);
            } else {
#pragma unroll
                for (int i = 0; i < CPT; ++i) {
                    const int k = k0 + tid + i * kAccThreads;
                    if (k >= W.ka && k <= W.kb) {
                        uint32_t x = LOGX ? x0 + (uint32_t)(((uint64_t)xl[i] * W.b) >> 30) : x0 + (uint32_t)i * (W.b >> 1);
                        if (LOGX) x = x >= 0xFFF00000u ? 0u : x;   // entry 4095 is never addressed: a wrap below 0
                        sample(i, x, bytes);
                    }
                }
            }
        };

        // prologue: table of particle 0
        Win cur = window(0);
        {
            LoadSet L[DEPTH];
            if (cur.ka <= cur.kb) {
                prefetch(L, cur);
                blend_all(L, cur, tab);
            }
        }
        __syncthreads();
        for (int q = 0; q < U.count; ++q) {
            float *buf_next = tab + (size_t)((q + 1) & 1) * P.wcap;
            Win nxt;
            nxt.ka = 1; nxt.kb = 0;
            LoadSet L[DEPTH];
            bool blend_next = false;
            if (q + 1 < U.count) {
                nxt = window(q + 1);
                blend_next = nxt.ka <= nxt.kb;
                if (blend_next) prefetch(L, nxt);           // loads fly during the resample
            }
            if (cur.ka <= cur.kb) resample(cur, tab + (size_t)(q & 1) * P.wcap);
            if (blend_next) blend_all(L, nxt, buf_next);
            cur = nxt;
            __syncthreads();
        }
    }
    // (derived here, not before the particle loop: the pointer must not occupy registers while the loop runs)
    // (a slab of fewer than two halos has rows that go to BOTH neighbours)
    float *mirror = nullptr, *mirror2 = nullptr;
    if (U.part_row < 0) {
        const int sp = P.units[u].spaxel;
        if (P.mirror_lo && sp < P.mirror_lo_n) mirror = P.mirror_lo + (size_t)sp * P.n_c;
        if (P.mirror_hi && sp >= P.mirror_hi_first) mirror2 = P.mirror_hi + (size_t)(sp - P.mirror_hi_first) * P.n_c;
    }
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int k = k0 + tid + i * kAccThreads;
        if (k <= k_end) {
            if (U.part_row >= 0) out[k] = acc[i];
            else {
                __stcs(out + k, acc[i]);                    // cube is written once, streamed
                if (mirror) mirror[k] = acc[i];             // ... and once more into the neighbour's halo, as it is produced
                if (mirror2) mirror2[k] = acc[i];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Experimental variant (kept for the measurement in profiles/r02_accumulate_async.md): the four corner
// windows of particle q + 1 are staged in shared memory by 1-D bulk async copies (cp.async.bulk, mbarrier completion)
// while particle q is resampled; the blend then reads shared memory instead of waiting on LDG results in registers.
// Point rule, uniform grids, one channel tile.  Built only with -DRUBIX_ACC_ASYNC=1.
// ------------------------------------------------------------------------------------------
#ifndef RUBIX_ACC_ASYNC
#define RUBIX_ACC_ASYNC 0
#endif
#ifndef RUBIX_ACC_ASYNC_TABLES
#define RUBIX_ACC_ASYNC_TABLES 2                     // 2: double-buffered table, one barrier per particle; 1: single table, two
#endif
#ifndef RUBIX_ACC_ASYNC_MINB
#define RUBIX_ACC_ASYNC_MINB 2
#endif
#if RUBIX_ACC_ASYNC
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\t"
                 "bra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ Quad lds_quad(const float *p)
{
    Quad q;
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "r"(smem_addr(p)));
    return q;
}

template <int CPT>
__global__ void __launch_bounds__(kAccThreads, RUBIX_ACC_ASYNC_MINB)
k_accumulate_async(const __grid_constant__ AccumParams P)
{
    extern __shared__ __align__(128) float sm[];            // stage[4][wcap] | tab[NT][wcap] | records | mbarrier
    constexpr int NT = RUBIX_ACC_ASYNC_TABLES;
    const int tid = threadIdx.x;
    const int u = blockIdx.x;
    if (u >= P.totals[0]) return;
    const Unit U = P.units[u];
    if (U.count == 0 && P.skip_empty) return;
    const int k_end = P.n_c - 1;
    float *out = U.part_row >= 0 ? P.partials + (size_t)U.part_row * P.n_c : P.cube + (size_t)U.spaxel * P.n_c;
    float acc[CPT];
#pragma unroll
    for (int i = 0; i < CPT; ++i) acc[i] = 0.0f;
    if (U.count > 0) {
        float *stage = sm, *tab = sm + 4 * (size_t)P.wcap;
        int4 *srec = reinterpret_cast<int4 *>(tab + NT * (size_t)P.wcap);
        const uint32_t bar = smem_addr(srec + 3 * kChunk);
        {
            const int4 *g = reinterpret_cast<const int4 *>(P.rec + U.start);
            for (int i = tid; i < U.count * 3; i += kAccThreads) srec[i] = __ldg(g + i);
        }
        if (tid == 0) {
            mbar_init(bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        const int row_a = P.n_z * P.pitch, row_z = P.pitch;
        // thread 0: start the copies of particle q's four corner windows (whole 128-sample groups; the padded grid copy
        // absorbs the overshoot); returns nothing -- every thread derives "has a window" from the record itself
        auto issue = [&](int q) {
            const int4 rb = srec[3 * q + 1], rc = srec[3 * q + 2];
            if (rc.x > rc.y) return;                          // no covered channel: no window
            const uint32_t bytes = (uint32_t)((rc.w + kPass - 1) / kPass * kPass) * 4u;
            const float *t0 = P.flux + (rb.x + rc.z);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic reads of the stage precede the async writes
            mbar_expect_tx(bar, 4u * bytes);
            bulk_g2s(smem_addr(stage), t0, bytes, bar);
            bulk_g2s(smem_addr(stage + P.wcap), t0 + row_a, bytes, bar);
            bulk_g2s(smem_addr(stage + 2 * (size_t)P.wcap), t0 + row_z, bytes, bar);
            bulk_g2s(smem_addr(stage + 3 * (size_t)P.wcap), t0 + row_a + row_z, bytes, bar);
        };
        auto blend = [&](int q, float *buf) {
            const int4 ra = srec[3 * q], rc = srec[3 * q + 2];
            const float f0 = __int_as_float(ra.x), f1 = __int_as_float(ra.y), f2 = __int_as_float(ra.z), f3 = __int_as_float(ra.w);
            const unsigned long long w0 = pack2(f0, f0), w1 = pack2(f1, f1), w2 = pack2(f2, f2), w3 = pack2(f3, f3);
            const int n = (rc.w + kPass - 1) / kPass * kPass;
            for (int s0 = 4 * tid; s0 < n; s0 += 4 * kAccThreads) {
                const Quad c0 = lds_quad(stage + s0), c1 = lds_quad(stage + P.wcap + s0);
                const Quad c2 = lds_quad(stage + 2 * (size_t)P.wcap + s0), c3 = lds_quad(stage + 3 * (size_t)P.wcap + s0);
                const unsigned long long lo = ffma2(w3, c3.lo, ffma2(w2, c2.lo, ffma2(w1, c1.lo, fmul2(w0, c0.lo))));
                const unsigned long long hi = ffma2(w3, c3.hi, ffma2(w2, c2.hi, ffma2(w1, c1.hi, fmul2(w0, c0.hi))));
                sts_quad(buf + s0, lo, hi);
            }
        };
        const uint32_t m_addr = 0x3FFCu, m_frac = 0x7FFFF8u, one_bits = 0x3F800000u;
        auto resample = [&](int q, const float *buf) {
            const int4 rb = srec[3 * q + 1], rc = srec[3 * q + 2];
            if (rc.x > rc.y) return;
            const char *bytes = reinterpret_cast<const char *>(buf);
            const uint32_t b = (uint32_t)rb.y;
            const int64_t a = (int64_t)(((uint64_t)(uint32_t)rb.w << 32) | (uint32_t)rb.z);
            const int64_t base = a - ((int64_t)rc.z << kFxFrac);
            const uint32_t x0 = (uint32_t)((base + (int64_t)b * tid) >> 8);
            auto sample = [&](int i, uint32_t x) {
                const float *e = reinterpret_cast<const float *>(bytes + ((x >> 18) & m_addr));
                const float s0 = e[0], s1 = e[1];
                const float f = __uint_as_float(and_or(x << 3, m_frac, one_bits)) - 1.0f;
                acc[i] += fmaf(f, s1 - s0, s0);
            };
            if (rc.x == 0 && rc.y == k_end) {
#pragma unroll
                for (int i = 0; i < CPT; ++i) sample(i, x0 + (uint32_t)i * (b >> 1));
            } else {
#pragma unroll
                for (int i = 0; i < CPT; ++i) {
                    const int k = tid + i * kAccThreads;
                    if (k >= rc.x && k <= rc.y) sample(i, x0 + (uint32_t)i * (b >> 1));
                }
            }
        };
        auto has_window = [&](int q) { const int4 rc = srec[3 * q + 2]; return rc.x <= rc.y; };
        uint32_t parity = 0;
        if (tid == 0) issue(0);
        if (has_window(0)) { mbar_wait(bar, parity); parity ^= 1u; blend(0, tab); }
        __syncthreads();
        for (int q = 0; q < U.count; ++q) {
            const bool more = q + 1 < U.count;
            if (more && tid == 0) issue(q + 1);               // the stage is free: its last reader passed the barrier
            resample(q, tab + (NT == 2 ? (size_t)(q & 1) * P.wcap : 0));
            if (NT == 1) __syncthreads();                     // single table: every thread is done reading it
            if (more && has_window(q + 1)) {
                mbar_wait(bar, parity);
                parity ^= 1u;
                blend(q + 1, tab + (NT == 2 ? (size_t)((q + 1) & 1) * P.wcap : 0));
            }
            __syncthreads();
        }
    }
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int k = tid + i * kAccThreads;
        if (k <= k_end) {
            if (U.part_row >= 0) out[k] = acc[i];
            else __stcs(out + k, acc[i]);
        }
    }
}
#endif  // RUBIX_ACC_ASYNC

// Fixed-order second level for spaxels with more than kChunk particles: fp64 running sum over the
// chunk rows (the kernel is bandwidth bound; the fp64 adds are free and keep 1e6-term sums exact
// to fp32 rounding).
// kReduceThreads channels per CTA: 256 normally; 32 where spaxels can hold thousands of rows (n >= 4 M particles), so that the
// rows of one piled-up spaxel are summed on n_c / 32 SMs at once (contention: 1.04 -> 0.43 ms; the sum order per channel is the same)
template <int kReduceThreads>
__global__ void __launch_bounds__(kReduceThreads)
k_reduce_partials(const float *__restrict__ partials, const int32_t *__restrict__ seg_off,
                  const int32_t *__restrict__ part_off, const int32_t *__restrict__ multi_list,
                  const int32_t *__restrict__ totals, int32_t n_c, float *__restrict__ cube, float *mirror_lo,
                  float *mirror_hi, int32_t mirror_lo_n, int32_t mirror_hi_first)
{
    for (int m = blockIdx.x; m < totals[2]; m += gridDim.x) {
    const int s = multi_list[m];
    const int cnt = seg_off[s + 1] - seg_off[s];
    const int chunks = (cnt + kChunk - 1) / kChunk;
    const float *rows = partials + (size_t)part_off[s] * n_c;
    // one thread per channel; eight chunk rows in flight per thread (the sum order stays c = 0, 1, ...)
    for (int k = blockIdx.y * kReduceThreads + threadIdx.x; k < n_c; k += gridDim.y * kReduceThreads) {
        const float *col = rows + k;
        double a = 0.0;
        int c = 0;
        for (; c + 32 <= chunks; c += 32) {                 // piled-up spaxels (thousands of rows): 32 loads in flight per thread
            float v[32];
#pragma unroll
            for (int u = 0; u < 32; ++u) v[u] = __ldcs(col + (size_t)(c + u) * n_c);
#pragma unroll
            for (int u = 0; u < 32; ++u) a += (double)v[u];
        }
        for (; c + 8 <= chunks; c += 8) {
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = __ldcs(col + (size_t)(c + u) * n_c);
#pragma unroll
            for (int u = 0; u < 8; ++u) a += (double)v[u];
        }
        for (; c < chunks; ++c) a += (double)__ldcs(col + (size_t)c * n_c);
        __stcs(cube + (size_t)s * n_c + k, (float)a);
        if (mirror_lo && s < mirror_lo_n) mirror_lo[(size_t)s * n_c + k] = (float)a;
        if (mirror_hi && s >= mirror_hi_first) mirror_hi[(size_t)(s - mirror_hi_first) * n_c + k] = (float)a;
    }
    }
}

template <int CPT, bool SINGLE, bool FLUX, bool LOGX = false, int GEN = 0, bool NARROW = false>
static cudaError_t launch_acc2(const AccumParams &P, unsigned grid, size_t smem, cudaStream_t st)
{
    auto kern = k_accumulate<CPT, SINGLE, kAccDepth, (LOGX || GEN) ? 3 : kAccMinBlocks, FLUX, LOGX, GEN, NARROW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kAccThreads, smem, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

template <int CPT>
static cudaError_t launch_acc(const AccumParams &P, bool flux, bool logx, unsigned grid, size_t smem, cudaStream_t st)
{
    if (logx && flux)
        return P.n_tiles == 1 ? launch_acc2<CPT, true, true, true>(P, grid, smem, st)
                              : launch_acc2<CPT, false, true, true>(P, grid, smem, st);
    if (logx)
        return P.n_tiles == 1 ? launch_acc2<CPT, true, false, true>(P, grid, smem, st)
                              : launch_acc2<CPT, false, false, true>(P, grid, smem, st);
    if (P.n_tiles == 1)
        return flux ? launch_acc2<CPT, true, true>(P, grid, smem, st) : launch_acc2<CPT, true, false>(P, grid, smem, st);
    return flux ? launch_acc2<CPT, false, true>(P, grid, smem, st) : launch_acc2<CPT, false, false>(P, grid, smem, st);
}

// general-grid mode: instantiated for CPT in {29, 8, 1} only (choose_cpt draws from that list then)
template <int CPT, int GEN>
static cudaError_t launch_acc_gen2(const AccumParams &P, bool flux, bool narrow, unsigned grid, size_t smem, cudaStream_t st)
{
    if (flux && narrow)
        return P.n_tiles == 1 ? launch_acc2<CPT, true, true, false, GEN, true>(P, grid, smem, st)
                              : launch_acc2<CPT, false, true, false, GEN, true>(P, grid, smem, st);
    if (P.n_tiles == 1)
        return flux ? launch_acc2<CPT, true, true, false, GEN>(P, grid, smem, st)
                    : launch_acc2<CPT, true, false, false, GEN>(P, grid, smem, st);
    return flux ? launch_acc2<CPT, false, true, false, GEN>(P, grid, smem, st)
                : launch_acc2<CPT, false, false, false, GEN>(P, grid, smem, st);
}
template <int CPT>
static cudaError_t launch_acc_gen(const AccumParams &P, bool flux, bool narrow, unsigned grid, size_t smem, cudaStream_t st)
{
    switch (P.gen.kind) {
        case 0: return launch_acc_gen2<CPT, 1>(P, flux, narrow, grid, smem, st);
        case 1: return launch_acc_gen2<CPT, 2>(P, flux, narrow, grid, smem, st);
        default: return launch_acc_gen2<CPT, 3>(P, flux, narrow, grid, smem, st);
    }
}

// Largest CPT in {29, 15, 8, 4, 2, 1} whose table fits the 12.20 format; returns the table capacity
// (samples, a whole number of passes).
int choose_cpt(int n_c, double b_max, bool flux, int *wcap_out, const rubix_ssp *gen_ssp = nullptr,
               const rubix_telescope *gen_tel = nullptr)
{
    const int cand[6] = {29, 15, 8, 4, 2, 1};
    for (int c = 0; c < 6; ++c) {
        const int cpt = cand[c];
        if (gen_ssp && cpt != 29 && cpt != 8 && cpt != 1) continue;   // the instantiated general-grid kernels
        const int tc = cpt * kAccThreads;
        const int tiles = (n_c + tc - 1) / tc;
        // skip tilings that leave a whole 256-channel group of lanes idle (unless the smallest)
        if (cpt > 1 && (long long)tiles * tc - n_c >= kAccThreads) continue;
        // samples j0 .. j_max + 1 with j0 rounded down to a multiple of kRowAlign
        // general-grid mode: the exact span of the widest tile (a listed grid is not equally dense everywhere)
        const int need = gen_ssp ? (int)gen_window_max(gen_ssp, gen_tel, tc < n_c ? tc : n_c) + kRowAlign + 6
                                 : (int)(b_max * (tc + (flux ? 1 : 0))) + kRowAlign + 4;
        const int wcap = (need + kPass - 1) / kPass * kPass;
        if (wcap > kTabMax) continue;
        *wcap_out = wcap;
        return cpt;
    }
    *wcap_out = 0;
    return 0;
}

cudaError_t launch_accumulate(const PassInputs &in, const Layout &L, char *ws, float *cube, bool skip_empty,
                              cudaStream_t st, const Mirrors *mirrors)
{
    const bool logx = table_mode(in.ssp, in.tel), gen = gen_mode(in.ssp, in.tel);
    const double b0 = (double)in.tel->dlambda / (double)in.ssp->dlambda;
    // table / general-grid mode: the steepest d x / d k of the detector, largest Doppler stretch included
    const double b_max = gen ? gen_step_max(in.ssp, in.tel) : (logx ? table_step_max(in.ssp, in.tel) : b0 / (1.0 - kBetaCap));
    int wcap = 0;
    const bool flux = in.tel->resample == RUBIX_RESAMPLE_FLUX;
    const int cpt = choose_cpt(L.n_c, b_max, flux, &wcap, gen ? in.ssp : nullptr, gen ? in.tel : nullptr);
    const bool narrow = (gen || logx) && flux && b_max <= 1.0;   // no bin wider than one SSP sample
    if (cpt == 0) return cudaErrorInvalidConfiguration;
    AccumParams P;
    P.flux = (const float *)(ws + L.off_flux);
    P.rec = (const Rec *)(ws + L.off_rec);
    P.units = (const Unit *)(ws + L.off_units);
    P.totals = (const int32_t *)(ws + L.off_totals);
    P.cube = cube;
    P.partials = (float *)(ws + L.off_partials);
    P.pitch = L.pitch;
    P.n_z = in.ssp->n_z;
    P.n_c = L.n_c;
    const int tc = cpt * kAccThreads;
    P.n_tiles = (L.n_c + tc - 1) / tc;
    P.wcap = wcap;
    P.n_lambda = in.ssp->n_lambda;
    P.skip_empty = skip_empty ? 1 : 0;
    P.narrow = narrow ? 1 : 0;
    P.mirror_lo = mirrors ? mirrors->lo : nullptr;
    P.mirror_hi = mirrors ? mirrors->hi : nullptr;
    P.mirror_lo_n = mirrors ? mirrors->rows * in.tel->n_y : 0;
    P.mirror_hi_first = mirrors ? (in.tel->n_x - mirrors->rows) * in.tel->n_y : 0;
    P.xtab = (const int64_t *)(ws + L.off_xtab);
    P.tex = 0;
    P.gen = GenGrid{};
    if (gen) gen_grid_params(in, L, ws, &P.gen);            // the tables the particle pass wrote
#if RUBIX_TEX_CORNERS > 0
    {
        static thread_local const void *cached_ptr = nullptr;
        static thread_local cudaTextureObject_t cached_tex = 0;
        if (cached_ptr != (const void *)P.flux) {
            if (cached_tex) cudaDestroyTextureObject(cached_tex);
            cudaResourceDesc rd{};
            rd.resType = cudaResourceTypeLinear;
            rd.res.linear.devPtr = (void *)P.flux;
            rd.res.linear.desc = cudaCreateChannelDesc<float4>();
            rd.res.linear.sizeInBytes = ((size_t)L.n_rows * L.pitch + kFluxPad) * 4;
            cudaTextureDesc td{};
            td.readMode = cudaReadModeElementType;
            cudaError_t te = cudaCreateTextureObject(&cached_tex, &rd, &td, nullptr);
            if (te != cudaSuccess) return te;
            cached_ptr = (const void *)P.flux;
        }
        P.tex = cached_tex;
    }
#endif
    int32_t cell_threshold = 0;
    const bool cell = cell_order_cells(in, L, &cell_threshold) > 0;    // as the particle pass decided
    P.seg = (const int32_t *)(ws + L.off_seg);
    P.cell_threshold = cell_threshold;
    P.cell_split = cell && cell_threshold > 0 ? 1 : 0;
    const size_t smem = (size_t)2 * wcap * sizeof(float) + (size_t)kChunk * sizeof(Rec);
    const unsigned grid = (unsigned)(L.max_units * P.n_tiles);
    cudaError_t e = cudaSuccess;
#if RUBIX_ACC_ASYNC
    if (!flux && !logx && !gen && P.n_tiles == 1 && cpt == 29) {     // the experimental staged variant (headline shape only)
        const size_t sm_async = (size_t)(4 + RUBIX_ACC_ASYNC_TABLES) * wcap * sizeof(float) + (size_t)kChunk * sizeof(Rec) + 16;
        {
            StageTimer t(1, st);
            auto kern = k_accumulate_async<29>;
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_async);
            if (e != cudaSuccess) return e;
            kern<<<grid, kAccThreads, sm_async, st>>>(P);
            RUBIX_LAUNCH_CHECK();
        }
    } else
#endif
    {
    StageTimer t(1, st);
    if (cell) {                                             // piled-up spaxels (all of them with RUBIX_CELL_ORDER_ALL)
        e = launch_accumulate_cell(P, b_max, (unsigned)L.max_units, st);
        if (e != cudaSuccess) return e;
    }
    if (!cell || P.cell_split) {
        if (gen) {
            switch (cpt) {
                case 29: e = launch_acc_gen<29>(P, flux, narrow, grid, smem, st); break;
                case 8: e = launch_acc_gen<8>(P, flux, narrow, grid, smem, st); break;
                default: e = launch_acc_gen<1>(P, flux, narrow, grid, smem, st); break;
            }
        } else {
            switch (cpt) {
                case 29: e = launch_acc<29>(P, flux, logx, grid, smem, st); break;
                case 15: e = launch_acc<15>(P, flux, logx, grid, smem, st); break;
                case 8: e = launch_acc<8>(P, flux, logx, grid, smem, st); break;
                case 4: e = launch_acc<4>(P, flux, logx, grid, smem, st); break;
                case 2: e = launch_acc<2>(P, flux, logx, grid, smem, st); break;
                default: e = launch_acc<1>(P, flux, logx, grid, smem, st); break;
            }
        }
    }
    }
    if (e != cudaSuccess) return e;
    StageTimer t2(2, st);
    const int rt = L.n >= 4000000 ? 32 : 256;
    const unsigned gy = (unsigned)((L.n_c + rt - 1) / rt);
    const unsigned gx = (unsigned)(L.max_multi < 1184 ? L.max_multi : 1184);   // grid-stride over the multi-chunk spaxels
    if (rt == 32)
        k_reduce_partials<32><<<dim3(gx, gy), 32, 0, st>>>(
            P.partials, (const int32_t *)(ws + L.off_seg), (const int32_t *)(ws + L.off_partoff),
            (const int32_t *)(ws + L.off_multi), P.totals, L.n_c, cube, P.mirror_lo, P.mirror_hi, P.mirror_lo_n, P.mirror_hi_first);
    else
        k_reduce_partials<256><<<dim3(gx, gy), 256, 0, st>>>(
            P.partials, (const int32_t *)(ws + L.off_seg), (const int32_t *)(ws + L.off_partoff),
            (const int32_t *)(ws + L.off_multi), P.totals, L.n_c, cube, P.mirror_lo, P.mirror_hi, P.mirror_lo_n, P.mirror_hi_first);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix
