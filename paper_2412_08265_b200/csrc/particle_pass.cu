// Particle pass: steps 1-3 of the hot path plus the per-particle records for steps 4-5.
//   K1  k_rotate_bin        rotate, project, bin  (fp32, fixed order)
//   K2  k_sort_*            stable LSD radix sort of (key, index)            (8(a) row 3)
//       k_unit_tile_totals, k_scan_units   seg_off[s] = lower_bound(sorted keys, s); work units (chunks of <= kChunk
//                           particles) per spaxel, partial rows: tiled three-way exclusive scan; unit descriptors
//                           -- no atomics on data anywhere (k_sort_rowscan counts its finished CTAs to pick the one that scans
//                           the digit totals, k_scan_units numbers the slots of a shared-memory list: neither changes a result)
//   K2c prepare_records_body (in k_scan_units_and_records)   SSP cell + bilinear weights x mass, fixed-point Doppler map (rows 4-5)
#include "common.cuh"
#include "gen_coord.cuh"

namespace rubix {

// --------------------------------------------------------------------------------------------
// K1.  Every * and + is a separately rounded fp32 op (no FMA contraction), in the order
//   xr = (R00*x + R01*y) + R02*z ;  u = (xr + (0.5f*N_x)*s) / s ;  key = floor(u)*N_y + floor(v)
// so the key equals the oracle's bit for bit.  NaN fails every comparison => dropped.
// --------------------------------------------------------------------------------------------
struct BinParams {
    float R[9];
    int32_t n_x, n_y;                      // rows owned by this call
    int32_t n_x_full, x_first;             // geometry of the whole detector along x and the first owned row (row window)
    float s;
    int64_t n;
    // the first pad_blocks CTAs of the launch write the padded workspace copy of the SSP grid instead (k_pad_flux's job: the
    // two tasks are independent and both come first, so they share a launch); 0 = binning only
    const float *pad_src;
    float *pad_dst;
    int64_t pad_total, pad_grid;
    int32_t pad_blocks, pad_n_lambda, pad_pitch;
};

// rows of n_lambda samples -> rows of `pitch` floats (zero padded), then zeros up to pad_total
__device__ __forceinline__ void pad_flux_part(const BinParams &P)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < P.pad_total; e += (int64_t)P.pad_blocks * blockDim.x) {
        float v = 0.0f;
        if (e < P.pad_grid) {
            const int64_t row = e / P.pad_pitch;
            const int32_t j = (int32_t)(e - row * P.pad_pitch);
            if (j < P.pad_n_lambda) v = __ldg(P.pad_src + row * P.pad_n_lambda + j);
        }
        P.pad_dst[e] = v;
    }
}

// key of (u, v) = detector coordinates in spaxels, or the sentinel n_x * n_y
__device__ __forceinline__ int32_t bin_key(const BinParams &P, float u, float v, float vl)
{
    const bool inside = (u >= 0.0f) && (u < (float)P.n_x_full) && (v >= 0.0f) && (v < (float)P.n_y) &&
                        (fabsf(vl) <= kVcapKms);
    const int32_t ix = (int32_t)floorf(u) - P.x_first;
    return (inside && ix >= 0 && ix < P.n_x) ? ix * P.n_y + (int32_t)floorf(v) : P.n_x * P.n_y;
}

__global__ void __launch_bounds__(256)
k_rotate_bin(const float *__restrict__ pos, const float *__restrict__ vel, BinParams P,
             int32_t *__restrict__ key, float *__restrict__ vlos)
{
    if ((int)blockIdx.x < P.pad_blocks) { pad_flux_part(P); return; }
    const int64_t i = (int64_t)(blockIdx.x - P.pad_blocks) * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    const float vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
    const float xr = __fadd_rn(__fadd_rn(__fmul_rn(P.R[0], x), __fmul_rn(P.R[1], y)), __fmul_rn(P.R[2], z));
    const float yr = __fadd_rn(__fadd_rn(__fmul_rn(P.R[3], x), __fmul_rn(P.R[4], y)), __fmul_rn(P.R[5], z));
    const float vl = __fadd_rn(__fadd_rn(__fmul_rn(P.R[6], vx), __fmul_rn(P.R[7], vy)), __fmul_rn(P.R[8], vz));
    const float hx = __fmul_rn(__fmul_rn(0.5f, (float)P.n_x_full), P.s);
    const float hy = __fmul_rn(__fmul_rn(0.5f, (float)P.n_y), P.s);
    const float u = __fdiv_rn(__fadd_rn(xr, hx), P.s);
    const float v = __fdiv_rn(__fadd_rn(yr, hy), P.s);
    key[i] = bin_key(P, u, v, vl);
    if (vlos) vlos[i] = vl;
}

// Batched variant: logical particle i belongs to batch element b (its own rotation) and gets the
// key b * N_s + (key inside its detector); dropped particles get batch * N_s.  Same fp32 arithmetic.
struct BinBatch {
    float R[kMaxBatch][9];
    int64_t off[kMaxBatch + 1];            // concatenated galaxies: element b = particles off[b] .. off[b+1]
    int32_t batch;
    int64_t n_phys;                        // > 0: shared galaxy, physical index = i % n_phys, element = i / n_phys
};

__global__ void __launch_bounds__(256)
k_rotate_bin_batched(const float *__restrict__ pos, const float *__restrict__ vel, BinParams P,
                     const __grid_constant__ BinBatch Bt, int32_t *__restrict__ key, float *__restrict__ vlos)
{
    if ((int)blockIdx.x < P.pad_blocks) { pad_flux_part(P); return; }
    const int64_t i = (int64_t)(blockIdx.x - P.pad_blocks) * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    int b;
    int64_t ip = i;
    if (Bt.n_phys > 0) {
        b = (int)(i / Bt.n_phys);
        ip = i - (int64_t)b * Bt.n_phys;
    } else {
        int lo = 0, hi = Bt.batch - 1;     // largest b with off[b] <= i
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (Bt.off[mid] <= i) lo = mid; else hi = mid - 1;
        }
        b = lo;
    }
    const float *R = Bt.R[b];
    const float x = pos[3 * ip], y = pos[3 * ip + 1], z = pos[3 * ip + 2];
    const float vx = vel[3 * ip], vy = vel[3 * ip + 1], vz = vel[3 * ip + 2];
    const float xr = __fadd_rn(__fadd_rn(__fmul_rn(R[0], x), __fmul_rn(R[1], y)), __fmul_rn(R[2], z));
    const float yr = __fadd_rn(__fadd_rn(__fmul_rn(R[3], x), __fmul_rn(R[4], y)), __fmul_rn(R[5], z));
    const float vl = __fadd_rn(__fadd_rn(__fmul_rn(R[6], vx), __fmul_rn(R[7], vy)), __fmul_rn(R[8], vz));
    const float hx = __fmul_rn(__fmul_rn(0.5f, (float)P.n_x_full), P.s);
    const float hy = __fmul_rn(__fmul_rn(0.5f, (float)P.n_y), P.s);
    const float u = __fdiv_rn(__fadd_rn(xr, hx), P.s);
    const float v = __fdiv_rn(__fadd_rn(yr, hy), P.s);
    const int32_t n_s = P.n_x * P.n_y;
    const int32_t kk = bin_key(P, u, v, vl);
    key[i] = kk < n_s ? b * n_s + kk : Bt.batch * n_s;
    vlos[i] = vl;
}

// --------------------------------------------------------------------------------------------
// K2.  Stable LSD radix sort.  Each WARP owns `items` consecutive keys ("warp chunk", Layout::sort_items) and is
// one column of the classic counting-sort histogram matrix histT[digit][warp chunk]; ranks
// inside a 32-key round come from __match_any_sync, so equal keys keep their index order.
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSortWarps * 32)
k_sort_hist(const int32_t *__restrict__ key_in, int64_t n, int shift, int mask, int n_wchunks, int items,
            int32_t *__restrict__ histT, int32_t *__restrict__ arrived)
{
    __shared__ int32_t cnt[kSortWarps][1 << kSortMaxDigitBits];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wc = blockIdx.x * kSortWarps + warp;
    if (blockIdx.x == 0 && threadIdx.x == 0) *arrived = 0;  // arrival counter of k_sort_rowscan (the next kernel on the stream)
    if (wc >= n_wchunks) return;
    for (int d = lane; d <= mask; d += 32) cnt[warp][d] = 0;
    __syncwarp();
    const int64_t base = (int64_t)wc * items;
    for (int r = 0; r < items; r += 32) {
        const int64_t i = base + r + lane;
        if (i < n) atomicAdd(&cnt[warp][(key_in[i] >> shift) & mask], 1);
    }
    __syncwarp();
    for (int d = lane; d <= mask; d += 32) histT[(int64_t)d * n_wchunks + wc] = cnt[warp][d];
}

// one CTA per digit: exclusive scan of its row of histT, row total to digit_total
// ... and the CTA that finishes last turns the row totals into the exclusive digit bases (one launch less per radix pass than a
// scan kernel of its own; `arrived` was zeroed by k_sort_hist)
__global__ void __launch_bounds__(256)
k_sort_rowscan(int32_t *__restrict__ histT, int n_wchunks, int32_t *digit_total, int n_digits, int32_t *__restrict__ digit_base,
               int32_t *arrived)
{
    __shared__ int32_t warp_sum[8];
    __shared__ int32_t carry_s;
    __shared__ int32_t s_last;
    __shared__ int32_t s_scan[1 << kSortMaxDigitBits];
    int32_t *row = histT + (int64_t)blockIdx.x * n_wchunks;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n_wchunks; base += 256) {
        const int i = base + threadIdx.x;
        const int32_t v = i < n_wchunks ? row[i] : 0;
        int32_t inc = v;
        for (int o = 1; o < 32; o <<= 1) {
            const int32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) warp_sum[warp] = inc;
        __syncthreads();
        int32_t wpre = 0;
        for (int w = 0; w < warp; ++w) wpre += warp_sum[w];
        const int32_t carry = carry_s;
        if (i < n_wchunks) row[i] = carry + wpre + inc - v;
        __syncthreads();
        if (threadIdx.x == 255) carry_s = carry + wpre + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        digit_total[blockIdx.x] = carry_s;
        __threadfence();                                    // the total is visible before the arrival is counted
        s_last = atomicAdd(arrived, 1) == (int32_t)gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    constexpr int kD = 1 << kSortMaxDigitBits;
    const volatile int32_t *dt = digit_total;               // written by the other CTAs: read past L1
    for (int t = threadIdx.x; t < kD; t += 256) s_scan[t] = t < n_digits ? dt[t] : 0;
    __syncthreads();
    for (int o = 1; o < kD; o <<= 1) {                      // inclusive scan, two entries per thread
        int32_t v[kD / 256];
#pragma unroll
        for (int i = 0; i < kD / 256; ++i) { const int t = threadIdx.x + 256 * i; v[i] = t >= o ? s_scan[t - o] : 0; }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < kD / 256; ++i) s_scan[threadIdx.x + 256 * i] += v[i];
        __syncthreads();
    }
    for (int t = threadIdx.x; t < n_digits; t += 256) digit_base[t] = s_scan[t] - dt[t];
}

template <bool FIRST>
__global__ void __launch_bounds__(kSortWarps * 32)
k_sort_scatter(const int32_t *__restrict__ key_in, const int32_t *__restrict__ perm_in, int64_t n,
               int shift, int mask, int n_wchunks, int items, const int32_t *__restrict__ histT,
               const int32_t *__restrict__ digit_base, int32_t *__restrict__ key_out,
               int32_t *__restrict__ perm_out)
{
    __shared__ int32_t cur[kSortWarps][1 << kSortMaxDigitBits];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wc = blockIdx.x * kSortWarps + warp;
    if (wc >= n_wchunks) return;
    for (int d = lane; d <= mask; d += 32)
        cur[warp][d] = digit_base[d] + histT[(int64_t)d * n_wchunks + wc];
    __syncwarp();
    const int64_t base = (int64_t)wc * items;
    const unsigned lt = (1u << lane) - 1u;
    for (int r = 0; r < items; r += 32) {
        const int64_t i = base + r + lane;
        const bool valid = i < n;
        const int32_t k = valid ? key_in[i] : 0;
        const int32_t v = valid ? (FIRST ? (int32_t)i : perm_in[i]) : 0;
        const int d = valid ? ((k >> shift) & mask) : (0x10000 + lane);   // invalid lanes never match
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        const int rank = __popc(peers & lt);
        int32_t dst = 0;
        if (valid) dst = cur[warp][d] + rank;
        __syncwarp();
        if (valid && rank == 0) cur[warp][d] += __popc(peers);
        __syncwarp();
        if (valid) {
            key_out[dst] = k;
            perm_out[dst] = v;
        }
    }
}

// seg_off[s] = first sorted position whose key is >= s   (s = 0 .. n_s+1)
// (cell order: the sorted keys are spaxel * mult + cell, dropped particles carry n_s * mult)
struct SegSource {
    const int32_t *key_sorted;         // non-null: seg_off is COMPUTED here (binary search) and written; null: read
    int64_t n;
    int32_t mult;
};

__global__ void __launch_bounds__(256)
k_segment_offsets(const int32_t *__restrict__ key_sorted, int64_t n, int32_t n_s, int32_t mult,
                  int32_t *__restrict__ seg_off)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s > n_s + 1) return;
    const int64_t want = (int64_t)s * mult;
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if ((int64_t)key_sorted[mid] < want) lo = mid + 1; else hi = mid;
    }
    seg_off[s] = (int32_t)lo;
}

constexpr int64_t kFusedSegMaxN = 16384;   // up to this many particles a one-tile detector finds its segment offsets inside k_scan_units

// Three exclusive scans over the spaxels, kScanTile spaxels per CTA:
//   unit_off: max(1, chunks(s))     part_off: chunks(s) if > 1 else 0     multi index: chunks(s) > 1
// Detectors of more than one tile: k_unit_tile_totals writes the three sums of every tile; k_scan_units adds the sums of the
// tiles before its own (a few hundred values at most), scans its tile and writes the unit descriptors.  A single tile needs no
// pre-pass, and with few particles k_scan_units also finds the segment offsets itself (SegSource).  totals = { n_units,
// n_part_rows, n_multi }.
constexpr int kScanItems = 4;
constexpr int kScanThreads = 256;
constexpr int kScanTile = kScanItems * kScanThreads;

// compact: an empty spaxel gets no unit (else one, which zero-fills its cube row).  first[i] = seg_off[s0 + i], i <= kScanItems
__device__ __forceinline__ void unit_counts(int32_t *__restrict__ seg_off, const SegSource &S, int32_t n_s, int s0, int compact,
                                            int32_t (&chunks)[kScanItems], int32_t (&first)[kScanItems + 1], int32_t (&tot)[3])
{
    tot[0] = tot[1] = tot[2] = 0;
    if (S.key_sorted) {
        // kScanItems + 1 binary searches in lockstep (one load of each per step: the chains overlap): first[i] = number of
        // sorted keys below (s0 + i) mult
        int64_t want[kScanItems + 1], pos[kScanItems + 1];
#pragma unroll
        for (int i = 0; i <= kScanItems; ++i) { want[i] = (int64_t)(s0 + i) * S.mult; pos[i] = 0; }
        int64_t step = 1;
        while (step * 2 <= S.n) step *= 2;
        for (; step > 0 && S.n > 0; step >>= 1) {
#pragma unroll
            for (int i = 0; i <= kScanItems; ++i) {
                const int64_t probe = pos[i] + step;
                if (probe <= S.n && (int64_t)__ldg(S.key_sorted + (probe - 1)) < want[i]) pos[i] = probe;
            }
        }
#pragma unroll
        for (int i = 0; i <= kScanItems; ++i) {
            first[i] = (int32_t)pos[i];
            if (s0 + i <= n_s + 1) seg_off[s0 + i] = first[i];   // (the entry shared with the next thread is written twice: same value)
        }
    } else {
#pragma unroll
        for (int i = 0; i <= kScanItems; ++i) first[i] = s0 + i <= n_s + 1 ? seg_off[s0 + i] : 0;
    }
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        const int s = s0 + i;
        chunks[i] = -1;
        if (s < n_s) {
            chunks[i] = (first[i + 1] - first[i] + kChunk - 1) / kChunk;
            tot[0] += chunks[i] > 1 ? chunks[i] : ((compact && chunks[i] == 0) ? 0 : 1);
            tot[1] += chunks[i] > 1 ? chunks[i] : 0;
            tot[2] += chunks[i] > 1 ? 1 : 0;
        }
    }
}

// block-wide sums of v[0..2]; every thread gets the results
__device__ __forceinline__ void block_sum3(int32_t (&v)[3], int32_t (*sm)[kScanThreads / 32])
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
        if (lane == 0) sm[q][warp] = v[q];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        v[q] = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) v[q] += sm[q][w];
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kScanThreads)
k_unit_tile_totals(int32_t *__restrict__ seg_off, const SegSource S, int32_t n_s, int compact, int32_t *__restrict__ tile_tot)
{
    __shared__ int32_t sm[3][kScanThreads / 32];
    int32_t chunks[kScanItems], first[kScanItems + 1], tot[3];
    unit_counts(seg_off, S, n_s, blockIdx.x * kScanTile + threadIdx.x * kScanItems, compact, chunks, first, tot);
    block_sum3(tot, sm);
    if (threadIdx.x < 3) tile_tot[3 * blockIdx.x + threadIdx.x] = tot[threadIdx.x];
}

// (one descriptor per unit; a spaxel of more than kChunk particles has several: the CTA writes those together)
struct ScanArgs {
    int32_t *seg_off;
    SegSource S;
    int32_t n_s, compact, n_tiles;
    const int32_t *tile_tot;
    int32_t *unit_off, *part_off, *multi_list, *totals;
    uint8_t *occ;
    Unit *units;
};

__device__ __forceinline__ void scan_units_body(const ScanArgs &A, const int tile)
{
    int32_t *__restrict__ seg_off = A.seg_off;
    const SegSource S = A.S;
    const int32_t n_s = A.n_s;
    const int compact = A.compact;
    const int32_t *__restrict__ tile_tot = A.tile_tot;
    int32_t *__restrict__ unit_off = A.unit_off, *__restrict__ part_off = A.part_off;
    int32_t *__restrict__ multi_list = A.multi_list, *__restrict__ totals = A.totals;
    uint8_t *__restrict__ occ = A.occ;
    Unit *__restrict__ units = A.units;
    __shared__ int32_t sm[3][kScanThreads / 32];
    __shared__ int32_t wsum[3][kScanThreads / 32];
    __shared__ int4 s_multi[kScanTile];                     // multi-chunk spaxels of this tile: (first, count, unit_off, part_off)
    __shared__ int32_t s_multi_s[kScanTile];
    __shared__ int32_t s_n_multi;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_n_multi = 0;
    // sums of the tiles before this one (and, in the last CTA, of all tiles)
    int32_t before[3] = {0, 0, 0};
    for (int t = threadIdx.x; t < tile; t += kScanThreads) {
#pragma unroll
        for (int q = 0; q < 3; ++q) before[q] += tile_tot[3 * t + q];
    }
    block_sum3(before, sm);
    const int s0 = tile * kScanTile + threadIdx.x * kScanItems;
    int32_t chunks[kScanItems], first[kScanItems + 1], tot[3], inc[3];
    unit_counts(seg_off, S, n_s, s0, compact, chunks, first, tot);
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        inc[q] = tot[q];
        for (int o = 1; o < 32; o <<= 1) {
            const int32_t t = __shfl_up_sync(0xffffffffu, inc[q], o);
            if (lane >= o) inc[q] += t;
        }
        if (lane == 31) wsum[q][warp] = inc[q];
    }
    __syncthreads();
    int32_t run[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        int32_t wpre = 0;
        for (int w = 0; w < warp; ++w) wpre += wsum[q][w];
        run[q] = before[q] + wpre + inc[q] - tot[q];
    }
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (chunks[i] >= 0) {
            const int s = s0 + i;
            const int32_t cnt = first[i + 1] - first[i];
            unit_off[s] = run[0];
            part_off[s] = run[1];
            occ[s] = chunks[i] > 0 ? 1 : 0;             // occupancy mask of the masked PSF/LSF passes
            if (chunks[i] > 1) {
                multi_list[run[2]] = s;
                const int slot = atomicAdd(&s_n_multi, 1);  // (shared memory, order irrelevant: every entry is written out below)
                s_multi[slot] = make_int4(first[i], cnt, run[0], run[1]);
                s_multi_s[slot] = s;
            } else if (!(compact && chunks[i] == 0)) {
                Unit U;
                U.start = first[i]; U.count = cnt; U.spaxel = s; U.part_row = -1;
                units[run[0]] = U;
            }
            run[0] += chunks[i] > 1 ? chunks[i] : ((compact && chunks[i] == 0) ? 0 : 1);
            run[1] += chunks[i] > 1 ? chunks[i] : 0;
            run[2] += chunks[i] > 1 ? 1 : 0;
        }
    }
    if (tile == A.n_tiles - 1 && threadIdx.x == kScanThreads - 1) {   // holds the grand totals
        unit_off[n_s] = run[0];
        part_off[n_s] = run[1];
        totals[0] = run[0];
        totals[1] = run[1];
        totals[2] = run[2];
    }
    __syncthreads();
    // the units of the multi-chunk spaxels: a thread per spaxel of up to 32 chunks, then a warp per heavier spaxel
    const int n_multi = s_n_multi;
    auto write_units = [&](const int4 e, int32_t sp, int c0, int c_step) {
        const int32_t n_chunks = (e.y + kChunk - 1) / kChunk;
        for (int c = c0; c < n_chunks; c += c_step) {
            Unit U;
            U.start = e.x + c * kChunk;
            U.count = min(kChunk, e.y - c * kChunk);
            U.spaxel = sp;
            U.part_row = e.w + c;
            units[e.z + c] = U;
        }
    };
    for (int m = threadIdx.x; m < n_multi; m += kScanThreads) {
        const int4 e = s_multi[m];
        if (e.y <= 32 * kChunk) write_units(e, s_multi_s[m], 0, 1);
    }
    for (int m = warp; m < n_multi; m += kScanThreads / 32) {
        const int4 e = s_multi[m];
        if (e.y > 32 * kChunk) write_units(e, s_multi_s[m], lane, 32);
    }
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_units(const ScanArgs A)
{
    scan_units_body(A, (int)blockIdx.x);
}

// --------------------------------------------------------------------------------------------
// K2c.  Per in-FoV particle, in sorted order:
//   cell i = clamp(max{j : A[j] <= q}, 0, n-2), t = clamp((q - A[i]) / (A[i+1] - A[i]), 0, 1)
//   w = mass * {(1-ta)(1-tz), ta(1-tz), (1-ta)tz, ta tz}                       (fp64 -> fp32)
//   rest position of channel k in SSP samples:  x_k = A + B k,
//   A = (l0_obs/(1+beta) - l0_ssp)/dl_ssp,  B = dl_obs/((1+beta) dl_ssp),  beta = v_los/c  (fp64)
//   stored as 28-bit-fraction fixed point so every kernel evaluates x_k with the same integers;
//   [k_lo, k_hi] = channels with 0 <= x_k <= N_l - 1 (zero contribution outside the coverage).
// --------------------------------------------------------------------------------------------
struct PrepParams {
    AxisParams ax;
    int32_t n_lambda, pitch, n_c, n_s, mode;
    float l0_ssp, dl_ssp, l0_obs, dl_obs;
    float redshift, flux_scale;         // DESIGN.md reading R14
    int32_t log_grid, table;            // table mode (R15 / R16): x_k = xtab[k] c + a
    const int64_t *xtab;
    int64_t n_phys;                     // > 0: batched call on a shared galaxy, physical particle = perm value % n_phys
    int32_t gen_on;                     // general-grid mode (gen_coord.cuh): positions per sample in fp64
    GenGrid gen;
};

__device__ __forceinline__ void axis_cell(const float *A, int n, float q, int *cell, double *t)
{
    int lo = 0, hi = n - 1;            // largest j with A[j] <= q, or 0
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (A[mid] <= q) lo = mid; else hi = mid - 1;
    }
    int i = min(lo, n - 2);
    double tt = ((double)q - (double)A[i]) / ((double)A[i + 1] - (double)A[i]);
    tt = fmin(fmax(tt, 0.0), 1.0);
    *cell = i;
    *t = tt;
}

struct PrepArgs {
    const int32_t *perm, *key_sorted;
    const float *vlos, *mass, *log_age, *log_z;
    Rec *rec;
    AdjAux *aux;
    int64_t n;
    int32_t drop_key;                           // sorted keys from here on belong to dropped particles
};

__device__ __forceinline__ void prepare_records_body(const PrepArgs &Q, const PrepParams &P, const int64_t i64)
{
    if (i64 >= Q.n) return;
    const int i = (int)i64;
    if (__ldg(Q.key_sorted + i) >= Q.drop_key) return;   // dropped particles sort last and get no record
    const int32_t *__restrict__ perm = Q.perm;
    const float *__restrict__ vlos = Q.vlos, *__restrict__ mass = Q.mass;
    const float *__restrict__ log_age = Q.log_age, *__restrict__ log_z = Q.log_z;
    Rec *__restrict__ rec = Q.rec;
    AdjAux *__restrict__ aux = Q.aux;
    const int pl = perm[i];                       // logical particle: indexes v_los
    const int p = P.n_phys > 0 ? (int)(pl % P.n_phys) : pl;   // physical particle: indexes the caller's arrays
    int ia, iz;
    double ta, tz;
    axis_cell(P.ax.age, P.ax.n_age, log_age[p], &ia, &ta);
    axis_cell(P.ax.z, P.ax.n_z, log_z[p], &iz, &tz);
    const double m = (double)mass[p] * (double)P.flux_scale;
    {
        const float qa = log_age[p], qz = log_z[p];
        AdjAux x;
        x.ta = (float)ta;
        x.tz = (float)tz;
        x.inv_wa = (qa > P.ax.age[0] && qa < P.ax.age[P.ax.n_age - 1])
                       ? (float)(1.0 / ((double)P.ax.age[ia + 1] - (double)P.ax.age[ia])) : 0.0f;
        x.inv_wz = (qz > P.ax.z[0] && qz < P.ax.z[P.ax.n_z - 1])
                       ? (float)(1.0 / ((double)P.ax.z[iz + 1] - (double)P.ax.z[iz])) : 0.0f;
        aux[i] = x;
    }
    Rec r;
    r.w[0] = (float)(m * (1.0 - ta) * (1.0 - tz));
    r.w[1] = (float)(m * ta * (1.0 - tz));
    r.w[2] = (float)(m * (1.0 - ta) * tz);
    r.w[3] = (float)(m * ta * tz);
#ifdef RUBIX_EXP_ONECELL
    ia = 3; iz = 2;                                     // timing experiment only: every particle in one SSP cell
#endif
    r.cell = (ia * P.ax.n_z + iz) * P.pitch;
    const double inv = 1.0 / ((1.0 + (double)vlos[pl] / kCkms) * (1.0 + (double)P.redshift));
    const double scale = (double)(1 << kFxFrac);
    const double A = ((double)P.l0_obs * inv - (double)P.l0_ssp) / (double)P.dl_ssp;
    const double B = (double)P.dl_obs * inv / (double)P.dl_ssp;
    int64_t a_fx = __double2ll_rn(A * scale);
    // B is rounded to an EVEN number of 2^-28 units: the accumulate kernel strides by kAccThreads = 128 channels,
    // i.e. by b / 2 in its 2^-20 local format, and that must stay exact
    const uint32_t b_fx = (uint32_t)(2 * __double2ll_rn(B * scale * 0.5));
    const int64_t b = (int64_t)b_fx;
    const int64_t x_max = (int64_t)(P.n_lambda - 1) << kFxFrac;
    int64_t k_lo, k_hi, x_first, x_last;
    uint32_t c_fx = 0;
    if (P.table) {
        // x_k = llrint(Y[k] c) + a_fx, c quantised to 2.30 fixed point so that every kernel uses the same value;
        // Y is increasing, so the covered channels are found by bisection
        const double opb = 1.0 + (double)vlos[pl] / kCkms;
        c_fx = P.log_grid ? (1u << 30) : (uint32_t)__double2ll_rn((double)(1u << 30) / opb);
        const double c = (double)c_fx * (1.0 / (double)(1u << 30));
        a_fx = P.log_grid ? -__double2ll_rn(log10(opb) / (double)P.dl_ssp * scale)
                          : -__double2ll_rn((double)P.l0_ssp / (double)P.dl_ssp * scale);
        auto xk = [&](int k) { return __double2ll_rn((double)P.xtab[k] * c) + a_fx; };
        const bool fl = P.mode == RUBIX_RESAMPLE_FLUX;     // the table then holds bin edges: bin k = [x_k, x_{k+1}]
        int lo = 0, hi = P.n_c;                            // point: first k with x_k >= 0; bins: first k with x_{k+1} > 0
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (fl ? xk(mid + 1) > 0 : xk(mid) >= 0) hi = mid; else lo = mid + 1;
        }
        k_lo = lo;
        lo = -1; hi = P.n_c - 1;                           // point: last k with x_k <= x_max; bins: last k with x_k < x_max
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (fl ? xk(mid) < x_max : xk(mid) <= x_max) lo = mid; else hi = mid - 1;
        }
        k_hi = lo;
        x_first = k_lo <= k_hi ? xk((int)k_lo) : 0;
        x_last = k_lo <= k_hi ? xk((int)k_hi + (fl ? 1 : 0)) : 0;
        if (x_first < 0) x_first = 0;
        if (x_last > x_max) x_last = x_max;
    } else if (P.mode == RUBIX_RESAMPLE_FLUX) {
        // x_k = a_fx + b k is the LOWER EDGE of bin k (upper edge = lower edge of bin k + 1);
        // [k_lo, k_hi] = bins that overlap the coverage [0, N_l - 1]
        a_fx -= (int64_t)(b_fx >> 1);
        const int64_t t = 1 - a_fx;                        // need a_fx + b (k + 1) >= 1
        k_lo = t <= 0 ? 0 : (t + b - 1) / b - 1;
        if (k_lo < 0) k_lo = 0;
        k_hi = x_max - 1 - a_fx < 0 ? -1 : (x_max - 1 - a_fx) / b;
        if (k_hi > P.n_c - 1) k_hi = P.n_c - 1;
        if (k_lo > P.n_c) k_lo = P.n_c;
        x_first = a_fx + b * k_lo;
        x_last = a_fx + b * (k_hi + 1);
        if (x_first < 0) x_first = 0;
        if (x_last > x_max) x_last = x_max;
    } else {
        k_lo = a_fx >= 0 ? 0 : (-a_fx + b - 1) / b;
        k_hi = a_fx > x_max ? -1 : (x_max - a_fx) / b;
        if (k_hi > P.n_c - 1) k_hi = P.n_c - 1;
        if (k_lo > P.n_c) k_lo = P.n_c;
        x_first = a_fx + b * k_lo;
        x_last = a_fx + b * k_hi;
    }
    if (P.gen_on) {
        // general-grid mode: x = gen_coord(tab[e], g) in fp64; the record carries g; the covered channels / bins are
        // found by bisection on the (increasing) table, the window gets a 1e-6-sample margin on either side
        const double g = gen_doppler(P.gen, 1.0 + (double)vlos[pl] / kCkms);
        const double x_top = (double)(P.n_lambda - 1);
        auto xe = [&](int e) { return gen_coord(P.gen, P.gen.tab[e], g); };
        const int fl = P.gen.flux;
        int lo = 0, hi = P.n_c;                            // point: first k with x_k >= 0; bins: first k with x_{k+1} > 0
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const bool ok = fl ? xe(mid + 1) > 0.0 : xe(mid) >= 0.0;
            if (ok) hi = mid; else lo = mid + 1;
        }
        k_lo = lo;
        lo = -1; hi = P.n_c - 1;                           // point: last k with x_k <= top; bins: last k with x_k < top
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            const bool ok = fl ? xe(mid) < x_top : xe(mid) <= x_top;
            if (ok) lo = mid; else hi = mid - 1;
        }
        k_hi = lo;
        r.a_fx = __double_as_longlong(g);
        r.b_fx = 0;
        r.k_lo = (int32_t)k_lo;
        r.k_hi = (int32_t)k_hi;
        r.j0 = 0;
        r.nw = 0;
        if (k_lo <= k_hi) {
            const double xa = fmin(fmax(xe((int)k_lo) - 1e-6, 0.0), x_top);
            const double xb = fmin(fmax(xe((int)k_hi + fl) + 1e-6, 0.0), x_top);
            r.j0 = (int32_t)xa & ~(kRowAlign - 1);
            r.nw = (int32_t)xb - r.j0 + 2;
        }
        rec[i] = r;
        return;
    }
    r.a_fx = a_fx;
    r.b_fx = P.table ? c_fx : b_fx;            // table mode: the Doppler factor c (2.30) takes B's slot
    r.k_lo = (int32_t)k_lo;
    r.k_hi = (int32_t)k_hi;
    r.j0 = 0;
    r.nw = 0;
    if (k_lo <= k_hi) {
        // table mode: k_accumulate<LOGX> adds separately truncated terms and may land up to 2 units of 2^-20 below
        // x_first; the window starts one group earlier when x_first is that close above a multiple of kRowAlign
        // (at j0 = 0 the kernel clamps at the knot instead)
        const int64_t x_j0 = P.table ? (x_first > 1024 ? x_first - 1024 : 0) : x_first;
        r.j0 = (int32_t)(x_j0 >> kFxFrac) & ~(kRowAlign - 1);
        r.nw = (int32_t)(x_last >> kFxFrac) - r.j0 + 2;   // samples j0 .. j_max + 1
    }
    rec[i] = r;
}

// The unit scan and the records are independent (both read the sorted keys): one launch, the first n_tiles CTAs scan
__global__ void __launch_bounds__(256)
k_scan_units_and_records(const ScanArgs S, const PrepArgs A, const __grid_constant__ PrepParams P)
{
    if ((int)blockIdx.x < S.n_tiles) { scan_units_body(S, (int)blockIdx.x); return; }
    prepare_records_body(A, P, (int64_t)(blockIdx.x - S.n_tiles) * blockDim.x + threadIdx.x);
}

// --------------------------------------------------------------------------------------------
// Table mode (readings R15 / R16): x_k = Y[k] c + a with (c, a) per particle and
//   log-sampled SSP grid:   Y[k] = log10(lambda_k / ((1+z) lambda0_ssp)) / dlog,   c = 1,  a = -log10(1+beta)/dlog
//   linear SSP grid:        Y[k] = lambda_k / ((1+z) dlambda_ssp),                 c = 1/(1+beta),  a = -lambda0_ssp/dlambda_ssp
// lambda_k = lam[k] (explicit channel wavelengths) or l0_obs + k dl_obs.  fp64 -> 36.28 fixed point.
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_positions(int32_t n_c, const float *__restrict__ lam, double l0_obs, double dl_obs, double zp1, int32_t log_grid,
            double l0_ssp, double dl_ssp, int32_t edges, int64_t *__restrict__ ytab)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > n_c) return;
    double l;
    if (!edges) {
        l = lam ? (double)lam[min(k, n_c - 1)] : l0_obs + dl_obs * (double)k;
    } else if (!lam) {                                     // bin average (reading R20): entry e = lower edge of bin e
        l = l0_obs + dl_obs * ((double)k - 0.5);
    } else if (k == 0) {
        l = (double)lam[0] - 0.5 * ((double)lam[1] - (double)lam[0]);
    } else if (k == n_c) {
        l = (double)lam[n_c - 1] + 0.5 * ((double)lam[n_c - 1] - (double)lam[n_c - 2]);
    } else {
        l = 0.5 * ((double)lam[k - 1] + (double)lam[k]);
    }
    l /= zp1;
    const double y = log_grid ? log10(l / l0_ssp) / dl_ssp : l / dl_ssp;
    ytab[k] = __double2ll_rn(y * (double)(1 << kFxFrac));
}

cudaError_t launch_bin_only(int64_t n, const float *pos, const float *vel, const rubix_telescope *tel, const float *R,
                            int32_t *key, float *vlos, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    BinParams B;
    for (int i = 0; i < 9; ++i) B.R[i] = R[i];
    B.n_x = tel->n_x;
    B.n_y = tel->n_y;
    B.n_x_full = tel->n_x_full > 0 ? tel->n_x_full : tel->n_x;
    B.x_first = tel->n_x_full > 0 ? tel->x_first : 0;
    B.s = tel->spaxel_size;
    B.n = n;
    B.pad_src = nullptr; B.pad_dst = nullptr; B.pad_total = B.pad_grid = 0; B.pad_blocks = 0; B.pad_n_lambda = B.pad_pitch = 0;
    k_rotate_bin<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pos, vel, B, key, vlos);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

double table_step_max(const rubix_ssp *s, const rubix_telescope *t)
{
    const double zp1 = 1.0 + (double)t->redshift;
    const bool edges = t->resample == RUBIX_RESAMPLE_FLUX;  // bin average: the table holds the n_c + 1 bin edges
    const int n_c = t->n_channels;
    auto y = [&](int k) {
        const float *lam = t->lambda_obs;
        double l;
        if (!edges) l = lam ? (double)lam[k] : (double)t->lambda0 + (double)t->dlambda * k;
        else if (!lam) l = (double)t->lambda0 + (double)t->dlambda * ((double)k - 0.5);
        else if (k == 0) l = (double)lam[0] - 0.5 * ((double)lam[1] - (double)lam[0]);
        else if (k == n_c) l = (double)lam[n_c - 1] + 0.5 * ((double)lam[n_c - 1] - (double)lam[n_c - 2]);
        else l = 0.5 * ((double)lam[k - 1] + (double)lam[k]);
        l /= zp1;
        return s->log_lambda ? log10(l / (double)s->lambda0) / (double)s->dlambda : l / (double)s->dlambda;
    };
    double m = 0.0;
    const int n_e = n_c + (edges ? 1 : 0);
    if (n_e < 2) return 0.0;
    if (!t->lambda_obs) {                                  // uniform grid: steepest at one of the two ends
        m = fmax(y(1) - y(0), y(n_e - 1) - y(n_e - 2));
    } else {
        for (int k = 1; k < n_e; ++k) m = fmax(m, y(k) - y(k - 1));
    }
    return s->log_lambda ? m : m / (1.0 - kBetaCap);
}

// --------------------------------------------------------------------------------------------
// Workspace copy of the SSP grid: every (age, Z) row padded with zeros to `pitch` floats (a
// multiple of 32, so every row and every 32-sample group starts on a 128-byte line) and kFluxPad
// zeros behind the last row.  The accumulate kernel then needs no bounds handling: a read past a
// row's end finds zeros.  6-20 MB, stays L2 resident.
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_pad_flux(const float *__restrict__ flux, int32_t n_lambda, int32_t pitch, int64_t n_total,
           int64_t n_grid, float *__restrict__ out)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_total;
         e += (int64_t)gridDim.x * blockDim.x) {
        float v = 0.0f;
        if (e < n_grid) {
            const int64_t row = e / pitch;
            const int32_t j = (int32_t)(e - row * pitch);
            if (j < n_lambda) v = __ldg(flux + row * n_lambda + j);
        }
        out[e] = v;
    }
}

// Cell order (spectral_cell.cu): composite sort key spaxel * cells + (i_age * n_z + i_z), so that the particles of a spaxel
// come grouped by SSP cell.  The cell found here only ORDERS the particles (prepare_records_body finds the cell it uses with the
// same search); dropped particles keep the last key.
struct CellKeyParams {
    AxisParams ax;
    int64_t n;
    int32_t n_s, cells;
    int64_t n_phys;
};

__global__ void __launch_bounds__(256)
k_cell_keys(const int32_t *__restrict__ key, const float *__restrict__ log_age, const float *__restrict__ log_z,
            const __grid_constant__ CellKeyParams P, int32_t *__restrict__ ckey)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const int32_t k = key[i];
    if (k >= P.n_s) { ckey[i] = P.n_s * P.cells; return; }
    const int64_t p = P.n_phys > 0 ? i % P.n_phys : i;
    int ia, iz;
    double ta, tz;
    axis_cell(P.ax.age, P.ax.n_age, log_age[p], &ia, &ta);
    axis_cell(P.ax.z, P.ax.n_z, log_z[p], &iz, &tz);
    ckey[i] = k * P.cells + ia * P.ax.n_z + iz;
}

// --------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------
static int bits_for(int32_t max_value)
{
    int b = 1;
    while ((1ll << b) <= (long long)max_value) ++b;
    return b;
}

int32_t cell_order_cells(const PassInputs &in, const Layout &L, int32_t *threshold)
{
    if (threshold) *threshold = 0;
    const rubix_telescope *t = in.tel;
    if (t->cell_order == RUBIX_CELL_ORDER_OFF || L.n <= 0 || !in.ssp) return 0;
    if (table_mode(in.ssp, t) || gen_mode(in.ssp, t)) return 0;                  // uniform grids only
    const int32_t cells = in.ssp->n_age * in.ssp->n_z;
    if ((double)(L.n_s + 2) * cells >= 2147483647.0) return 0;                   // composite key space
    const double b_max = (double)t->dlambda / (double)in.ssp->dlambda / (1.0 - kBetaCap);
    if (!cell_kernel_fits(L.n_c, b_max, t->resample == RUBIX_RESAMPLE_FLUX)) return 0;
    if (t->cell_order == RUBIX_CELL_ORDER_ALL) return cells;                     // every spaxel
    if (t->cell_order == RUBIX_CELL_ORDER_AUTO) {                                // piled-up detectors only
        const int64_t n_s_full = (int64_t)(t->n_x_full > 0 ? t->n_x_full : t->n_x) * t->n_y * (in.batch > 0 ? in.batch : 1);
        if (L.n < kCellAutoMinN || L.n < (int64_t)kCellAutoMean * n_s_full) return 0;
    }
    if (threshold) *threshold = kCellAutoRuns * cells;
    return cells;
}

Layout make_layout(int64_t n, int32_t n_s, int32_t n_c, int32_t n_rows, int32_t n_lambda)
{
    Layout L{};
    L.n = n;
    L.n_s = n_s;
    L.n_c = n_c;
    const int bits = bits_for(n_s);                      // keys are 0 .. n_s  (the cell order sorts wider keys: the pass
    L.sort_passes = (bits + kSortMaxDigitBits - 1) / kSortMaxDigitBits;   // count is then fixed in launch_particle_pass)
    L.digit_bits = (bits + L.sort_passes - 1) / L.sort_passes;
    // keys per warp chunk: about 2048 warps per radix pass, 128 .. 1024 keys each (measured: 10^5 particles are fastest at
    // 128, 10^6 at 512, 10^7 at 1024; the stable order does not depend on it)
    L.sort_items = 128;
    while (L.sort_items < kSortItemsMax && (int64_t)L.sort_items * 2048 < n) L.sort_items *= 2;
    L.n_wchunks = (int32_t)((n + L.sort_items - 1) / L.sort_items);
    L.max_units = (int64_t)n_s + n / kChunk + 1;
    L.max_part_rows = 2 * (n / kChunk) + 2;
    L.max_multi = n / kChunk + 1;
    L.final_buf = 0;                                     // the LAST radix pass always writes buffer 0
    const size_t nn = (size_t)(n > 0 ? n : 1);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    // two cube-sized buffers come first: rubix_convolve_psf_lsf (which does not know n) uses the
    // first one as its temporary, so it never touches the sort artefacts behind them
    const size_t cube = (size_t)n_s * (size_t)n_c * 4;
    L.off_cube_a = take(cube);
    L.off_cube_b = take(cube);
    // per-channel PSF taps (reading R18) sit right behind the two cubes, at an offset that depends on the detector
    // only: rubix_convolve_psf_lsf finds them without knowing n, and never touches the sort artefacts behind them
    L.off_psftaps = take(psf_taps_bytes(n_c));
    L.off_key = take(nn * 4);
    L.off_vlos = take(nn * 4);
    L.off_seg = take(((size_t)n_s + 2) * 4);
    for (int b = 0; b < 2; ++b) {
        L.off_keybuf[b] = take(nn * 4);
        L.off_permbuf[b] = take(nn * 4);
    }
    // rows reserved for the histogram matrix: n_wchunks itself DROPS where sort_items doubles, and a batched call carves the
    // layouts of its smaller groups out of the workspace sized for the largest -- so reserve a count that never decreases with n
    // (<= 2048 rows up to 262 144 particles, 4096 up to 4 M, then n / 1024)
    int64_t hist_rows = L.n_wchunks > 0 ? L.n_wchunks : 1;
    if (n > (int64_t)128 * 2048 && hist_rows < 4096) hist_rows = 4096;
    L.off_hist = take((size_t)(1 << kSortMaxDigitBits) * (size_t)hist_rows * 4);
    L.off_dtot = take(((size_t)(1 << kSortMaxDigitBits) + 1) * 4);   // + the arrival counter of k_sort_rowscan
    L.off_dbase = take((size_t)(1 << kSortMaxDigitBits) * 4);
    L.off_unitoff = take(((size_t)n_s + 1) * 4);
    L.off_partoff = take(((size_t)n_s + 1) * 4);
    L.off_multi = take((size_t)L.max_multi * 4);
    L.off_totals = take(16);
    L.off_tiletot = take(((size_t)n_s / kScanTile + 1) * 3 * 4);
    L.off_units = take((size_t)L.max_units * sizeof(Unit));
    L.off_rec = take(nn * sizeof(Rec));
    L.off_aux = take(nn * sizeof(AdjAux));
    L.off_partials = take((size_t)L.max_part_rows * (size_t)n_c * 4);
    L.n_rows = n_rows;
    L.n_lambda = n_lambda;
    L.pitch = (n_lambda + kRowAlign - 1) / kRowAlign * kRowAlign;
    off = align_up(off, 512);                            // (texture-alignment safe)
    L.off_flux = take(((size_t)n_rows * L.pitch + kFluxPad) * 4);
    L.off_xtab = take(((size_t)n_c + 1) * 8);           // Y[k] of the table mode (readings R15 / R16)
    L.off_lamobs = take(((size_t)n_c + 1) * 4);         // device copy of rubix_telescope.lambda_obs
    for (int b = 0; b < 2; ++b) L.off_occ[b] = take((size_t)n_s + 64);   // occupancy of the raw cube / of the PSF temporary
    // general-grid mode (gen_coord.cuh): table over channel centres / bin edges, knots, inverse widths, look-up table
    L.off_gtab = take(((size_t)n_c + 2) * 8);
    L.off_gknots = take(((size_t)n_lambda + 1) * 16);    // (knot, inverse interval width) pairs
    L.off_ginvw = L.off_gknots;
    L.off_glut = take(((size_t)kGenLutMaxPerKnot * n_lambda + 8) * 4);
    L.off_glam = take(((size_t)n_lambda + 1) * 4);
    L.bytes_total = off;
    return L;
}

cudaError_t launch_particle_pass(const PassInputs &in, const Layout &L, char *ws, cudaStream_t st)
{
    const int64_t n = L.n;
    const int32_t n_s = L.n_s;
    int32_t *key = (int32_t *)(ws + L.off_key);
    float *vlos = (float *)(ws + L.off_vlos);
    int32_t *seg = (int32_t *)(ws + L.off_seg);
    int32_t *kbuf[2] = {(int32_t *)(ws + L.off_keybuf[0]), (int32_t *)(ws + L.off_keybuf[1])};
    int32_t *pbuf[2] = {(int32_t *)(ws + L.off_permbuf[0]), (int32_t *)(ws + L.off_permbuf[1])};
    int32_t *histT = (int32_t *)(ws + L.off_hist);
    int32_t *dtot = (int32_t *)(ws + L.off_dtot);
    int32_t *dbase = (int32_t *)(ws + L.off_dbase);
    int32_t *arrived = dtot + (1 << kSortMaxDigitBits);   // behind the digit totals (Layout reserves one more word)
    int32_t *unit_off = (int32_t *)(ws + L.off_unitoff);
    int32_t *part_off = (int32_t *)(ws + L.off_partoff);
    int32_t *multi = (int32_t *)(ws + L.off_multi);
    int32_t *totals = (int32_t *)(ws + L.off_totals);
    Unit *units = (Unit *)(ws + L.off_units);
    Rec *rec = (Rec *)(ws + L.off_rec);

    const int64_t n_grid = (int64_t)L.n_rows * L.pitch, n_total = n_grid + kFluxPad;
    const unsigned pad_blocks = L.n_rows > 0 ? (unsigned)((n_total + 1023) / 1024) : 0u;
    if (pad_blocks > 0 && n == 0) {                         // no particles: the copy alone (the adjoint of an empty set reads nothing)
        k_pad_flux<<<pad_blocks, 256, 0, st>>>(in.ssp->flux, L.n_lambda, L.pitch, n_total, n_grid, (float *)(ws + L.off_flux));
        RUBIX_LAUNCH_CHECK();
    }
    if (n > 0) {
        BinParams B;
        B.pad_src = L.n_rows > 0 ? in.ssp->flux : nullptr;
        B.pad_dst = (float *)(ws + L.off_flux);
        B.pad_total = n_total; B.pad_grid = n_grid;
        B.pad_blocks = (int32_t)pad_blocks; B.pad_n_lambda = L.n_lambda; B.pad_pitch = L.pitch;
        for (int i = 0; i < 9; ++i) B.R[i] = in.R[i];
        B.n_x = in.tel->n_x;
        B.n_y = in.tel->n_y;
        B.n_x_full = in.tel->n_x_full > 0 ? in.tel->n_x_full : in.tel->n_x;
        B.x_first = in.tel->n_x_full > 0 ? in.tel->x_first : 0;
        B.s = in.tel->spaxel_size;
        B.n = n;
        if (in.batch > 1 || in.offsets) {
            BinBatch Bt;
            Bt.batch = in.batch;
            Bt.n_phys = in.offsets ? 0 : in.p->n;
            for (int b = 0; b < in.batch; ++b)
                for (int i = 0; i < 9; ++i) Bt.R[b][i] = in.R[9 * b + i];
            for (int b = 0; b <= in.batch; ++b) Bt.off[b] = in.offsets ? in.offsets[b] : 0;
            k_rotate_bin_batched<<<pad_blocks + (unsigned)((n + 255) / 256), 256, 0, st>>>(in.p->pos, in.p->vel, B, Bt, key, vlos);
        } else {
            k_rotate_bin<<<pad_blocks + (unsigned)((n + 255) / 256), 256, 0, st>>>(in.p->pos, in.p->vel, B, key, vlos);
        }
        RUBIX_LAUNCH_CHECK();

        // cell order: sort by spaxel * n_cells + cell instead (the composite keys go to the buffer the first pass does not write)
        const int32_t cells = cell_order_cells(in, L);
        int sort_passes = L.sort_passes, digit_bits = L.digit_bits;
        if (cells > 0) {
            const int bits = bits_for((int32_t)((int64_t)n_s * cells));
            sort_passes = (bits + kSortMaxDigitBits - 1) / kSortMaxDigitBits;
            digit_bits = (bits + sort_passes - 1) / sort_passes;
        }
        const int32_t *kin = key;
        if (cells > 0) {
            CellKeyParams C;
            C.ax.n_age = in.ssp->n_age;
            C.ax.n_z = in.ssp->n_z;
            for (int i = 0; i < in.ssp->n_age; ++i) C.ax.age[i] = in.ssp->log_age_axis[i];
            for (int i = 0; i < in.ssp->n_z; ++i) C.ax.z[i] = in.ssp->log_z_axis[i];
            C.n = n;
            C.n_s = n_s;
            C.cells = cells;
            C.n_phys = (in.batch > 1 && !in.offsets) ? in.p->n : 0;
            int32_t *ckey = kbuf[sort_passes & 1];
            k_cell_keys<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(key, in.p->log_age, in.p->log_z, C, ckey);
            RUBIX_LAUNCH_CHECK();
            kin = ckey;
        }
        const int mask = (1 << digit_bits) - 1;
        const int n_digits = 1 << digit_bits;
        const unsigned sort_grid = (unsigned)((L.n_wchunks + kSortWarps - 1) / kSortWarps);
        const int32_t *pin = nullptr;
        for (int pass = 0; pass < sort_passes; ++pass) {
            const int shift = pass * digit_bits;
            const int ob = (sort_passes - 1 - pass) & 1;   // the last pass writes buffer 0 = Layout::final_buf
            int32_t *kout = kbuf[ob], *pout = pbuf[ob];
            k_sort_hist<<<sort_grid, kSortWarps * 32, 0, st>>>(kin, n, shift, mask, L.n_wchunks, L.sort_items, histT, arrived);
            RUBIX_LAUNCH_CHECK();
            k_sort_rowscan<<<n_digits, 256, 0, st>>>(histT, L.n_wchunks, dtot, n_digits, dbase, arrived);
            RUBIX_LAUNCH_CHECK();
            if (pass == 0)
                k_sort_scatter<true><<<sort_grid, kSortWarps * 32, 0, st>>>(
                    kin, pin, n, shift, mask, L.n_wchunks, L.sort_items, histT, dbase, kout, pout);
            else
                k_sort_scatter<false><<<sort_grid, kSortWarps * 32, 0, st>>>(
                    kin, pin, n, shift, mask, L.n_wchunks, L.sort_items, histT, dbase, kout, pout);
            RUBIX_LAUNCH_CHECK();
            kin = kout;
            pin = pout;
        }
    }
    const int32_t *key_sorted = kbuf[L.final_buf];
    const int32_t *perm = pbuf[L.final_buf];
    const int32_t cells = n > 0 ? cell_order_cells(in, L) : 0;
    const int32_t mult = cells > 0 ? cells : 1;
    PrepParams P;
    if (n > 0) {                                           // what the records need, and the tables of the table / general-grid modes
        P.ax.n_age = in.ssp->n_age;
        P.ax.n_z = in.ssp->n_z;
        for (int i = 0; i < in.ssp->n_age; ++i) P.ax.age[i] = in.ssp->log_age_axis[i];
        for (int i = 0; i < in.ssp->n_z; ++i) P.ax.z[i] = in.ssp->log_z_axis[i];
        P.n_lambda = in.ssp->n_lambda;
        P.pitch = L.pitch;
        P.n_c = in.tel->n_channels;
        P.n_s = n_s;
        P.mode = in.tel->resample;
        P.log_grid = in.ssp->log_lambda;
        P.table = table_mode(in.ssp, in.tel) ? 1 : 0;
        P.gen_on = gen_mode(in.ssp, in.tel) ? 1 : 0;
        if (P.gen_on) {
            cudaError_t eg = launch_gen_setup(in, L, ws, st, &P.gen);
            if (eg != cudaSuccess) return eg;
        }
        P.n_phys = (in.batch > 1 && !in.offsets) ? in.p->n : 0;
        P.xtab = (const int64_t *)(ws + L.off_xtab);
        if (P.table) {
            const float *lam_dev = nullptr;
            if (in.tel->lambda_obs) {                      // host array -> workspace (read before this call returns)
                lam_dev = (const float *)(ws + L.off_lamobs);
                cudaError_t ec = cudaMemcpyAsync(ws + L.off_lamobs, in.tel->lambda_obs, (size_t)L.n_c * 4,
                                                 cudaMemcpyHostToDevice, st);
                if (ec != cudaSuccess) return ec;
            }
            k_positions<<<(unsigned)((L.n_c + 256) / 256), 256, 0, st>>>(
                L.n_c, lam_dev, (double)in.tel->lambda0, (double)in.tel->dlambda, 1.0 + (double)in.tel->redshift,
                P.log_grid, (double)in.ssp->lambda0, (double)in.ssp->dlambda, P.mode == RUBIX_RESAMPLE_FLUX ? 1 : 0,
                (int64_t *)(ws + L.off_xtab));
            RUBIX_LAUNCH_CHECK();
            if (P.mode == RUBIX_RESAMPLE_FLUX) {           // the adjoint of this combination is k_adjoint_general: its tables
                GenGrid Gt;
                cudaError_t eg = launch_gen_setup(in, L, ws, st, &Gt);
                if (eg != cudaSuccess) return eg;
            }
        }
        P.redshift = in.tel->redshift;
        P.flux_scale = in.tel->flux_scale;
        P.l0_ssp = in.ssp->lambda0;
        P.dl_ssp = in.ssp->dlambda;
        P.l0_obs = in.tel->lambda0;
        P.dl_obs = in.tel->dlambda;
    }
    {
        int32_t *tile_tot = (int32_t *)(ws + L.off_tiletot);
        const unsigned tiles = (unsigned)(n_s / kScanTile + 1);
        const int compact = in.compact_units ? 1 : 0;
        const SegSource compute{key_sorted, n, mult}, read{nullptr, 0, 1};
        // the segment offsets: inside the unit scan where that is one CTA and the searches are short, else a kernel of their own
        // (one search per thread; measured: five searches per thread in the 88 CTAs of the medium detector cost 40 us more)
        const bool fused_seg = tiles == 1 && n <= kFusedSegMaxN;
        if (!fused_seg) {
            k_segment_offsets<<<(unsigned)((n_s + 2 + 255) / 256), 256, 0, st>>>(key_sorted, n, n_s, mult, seg);
            RUBIX_LAUNCH_CHECK();
        }
        if (tiles > 1) {                                   // a single tile has nothing before it: k_scan_units reads no tile sums
            k_unit_tile_totals<<<tiles, kScanThreads, 0, st>>>(seg, read, n_s, compact, tile_tot);
            RUBIX_LAUNCH_CHECK();
        }
        const ScanArgs S{seg, fused_seg ? compute : read, n_s, compact, (int32_t)tiles, tile_tot, unit_off, part_off, multi, totals,
                         (uint8_t *)(ws + L.off_occ[0]), units};
        if (n > 0) {                                       // the unit scan and the records share a launch
            const PrepArgs A{perm, key_sorted, vlos, in.p->mass, in.p->log_age, in.p->log_z, rec, (AdjAux *)(ws + L.off_aux), n,
                             n_s * mult};
            k_scan_units_and_records<<<tiles + (unsigned)((n + 255) / 256), 256, 0, st>>>(S, A, P);
        } else {
            k_scan_units<<<tiles, kScanThreads, 0, st>>>(S);
        }
        RUBIX_LAUNCH_CHECK();
    }
    return cudaSuccess;
}

}  // namespace rubix
