// Shared by the accumulate kernels (spectral.cu: k_accumulate; spectral_cell.cu: k_accumulate_cell): launch parameters and the
// 16-byte load / store helpers of the blend.
#pragma once
#include "common.cuh"
#include "gen_coord.cuh"

namespace rubix {

struct AccumParams {
    const float *flux;       // padded workspace copy of the SSP grid (Layout::pitch)
    const Rec *rec;
    const Unit *units;
    const int32_t *totals;
    float *cube;
    float *partials;
    int32_t pitch, n_z, n_c, n_tiles, wcap, n_lambda;
    int32_t skip_empty;      // 1: empty spaxels are left unwritten (the masked PSF/LSF passes never read them)
    int32_t narrow;          // bin average in table / general-grid mode: no bin is wider than one SSP sample
    // Mirrors (spaxel-sharded runs, rubix_build_cube_mirrored): rows of spaxels < mirror_lo_n are ALSO stored at mirror_lo,
    // rows of spaxels >= mirror_hi_first at mirror_hi -- a neighbour's halo, possibly peer memory of another GPU.
    float *mirror_lo, *mirror_hi;
    int32_t mirror_lo_n, mirror_hi_first;
    const int64_t *xtab;     // LOGX: rest position of channel k at beta = 0 (36.28), see k_log_positions
    cudaTextureObject_t tex;
    GenGrid gen;             // GEN: general-grid mode (gen_coord.cuh)
    // Cell order (spectral_cell.cu): with cell_split, spaxels of >= cell_threshold particles (seg_off tells) are left to
    // k_accumulate_cell by k_accumulate and the others the other way round
    const int32_t *seg;
    int32_t cell_split, cell_threshold;
};

// which of the two accumulate kernels owns the unit's spaxel
__device__ __forceinline__ bool cell_kernel_owns(const AccumParams &P, int spaxel)
{
    return P.seg[spaxel + 1] - P.seg[spaxel] >= P.cell_threshold;
}

constexpr int kPass = 128;                           // table samples produced per warp per pass
constexpr int kAccWarps = kAccThreads / 32;
#ifndef RUBIX_LDG_MODE
#define RUBIX_LDG_MODE 0
#endif
#ifndef RUBIX_TEX_CORNERS
#define RUBIX_TEX_CORNERS 0
#endif
#ifndef RUBIX_ACC_DEPTH
#define RUBIX_ACC_DEPTH 1
#endif
#ifndef RUBIX_ACC_MINB
#define RUBIX_ACC_MINB 5
#endif
constexpr int kAccDepth = RUBIX_ACC_DEPTH;           // load sets (passes) in flight per warp
constexpr int kAccMinBlocks = RUBIX_ACC_MINB;

// (a & b) | c in one LOP3 (b, c stay in registers)
__device__ __forceinline__ uint32_t and_or(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

struct Quad { unsigned long long lo, hi; };          // four consecutive samples as two packed pairs

// NOALLOC: the corner windows stream past L1 (listed-knot mode: L1 then keeps the look-up table and the knots, which every
// sample reads; measured 37.7 -> 27.7 ms on the medium workload)
template <bool NOALLOC = false>
__device__ __forceinline__ Quad ldg_quad(const float *p)
{
    Quad q;
    if (NOALLOC) {
        asm volatile("ld.global.nc.L1::no_allocate.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
        return q;
    }
#if RUBIX_LDG_MODE == 1
    asm volatile("ld.global.nc.L1::no_allocate.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
#elif RUBIX_LDG_MODE == 2
    asm volatile("ld.global.cg.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
#elif RUBIX_LDG_MODE == 3
    asm volatile("ld.global.nc.L1::evict_first.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
#else
    asm volatile("ld.global.nc.v2.b64 {%0, %1}, [%2];" : "=l"(q.lo), "=l"(q.hi) : "l"(p));
#endif
    return q;
}
__device__ __forceinline__ void sts_quad(float *p, unsigned long long lo, unsigned long long hi)
{
    asm volatile("st.shared.v2.b64 [%0], {%1, %2};" ::"r"((uint32_t)__cvta_generic_to_shared(p)), "l"(lo), "l"(hi)
                 : "memory");
}

struct LoadSet { Quad c[4]; };                       // 4 corners x 4 samples

// spectral_cell.cu: the variant for piled-up spaxels (corner windows kept in registers across particles of one SSP cell)
cudaError_t launch_accumulate_cell(const AccumParams &P, double b_max, unsigned grid, cudaStream_t st);

}  // namespace rubix
