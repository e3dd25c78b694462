// Measurement helpers (include/rubix_peaks.h): on-chip peak micro-benchmarks and stage timing.
#include <vector>

#include "common.cuh"
#include "../../include/rubix_peaks.h"

namespace rubix {

// ---------------------------------------------------------------------------------------------
// stage timing: event pairs recorded on the caller's stream
// ---------------------------------------------------------------------------------------------
namespace {
bool g_timing = false;
struct Pair { cudaEvent_t a, b; int stage; };
std::vector<Pair> g_pairs;
std::vector<cudaEvent_t> g_free;
cudaEvent_t get_event()
{
    if (!g_free.empty()) { cudaEvent_t e = g_free.back(); g_free.pop_back(); return e; }
    cudaEvent_t e;
    cudaEventCreate(&e);
    return e;
}
}  // namespace

StageTimer::StageTimer(int stage, cudaStream_t st) : stage_(stage), st_(st), a_(nullptr)
{
    if (!g_timing) return;
    a_ = get_event();
    cudaEventRecord(a_, st_);
}
StageTimer::~StageTimer()
{
    if (!a_) return;
    cudaEvent_t b = get_event();
    cudaEventRecord(b, st_);
    g_pairs.push_back(Pair{a_, b, stage_});
}

// ---------------------------------------------------------------------------------------------
// micro-benchmarks
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_peak_l2(const float4 *__restrict__ buf, size_t n_vec, int iters, float *sink)
{
    float acc = 0.f;
    const size_t stride = (size_t)blockDim.x;
    // each CTA starts at a different place so that the SMs do not hit the same lines together
    size_t start = ((size_t)blockIdx.x * 7919u * 256u) % n_vec;
    for (int it = 0; it < iters; ++it) {
        size_t i = start + threadIdx.x;
#pragma unroll 8
        for (int r = 0; r < 2048; ++r) {
            if (i >= n_vec) i -= n_vec;
            float4 v;
            asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(buf + i));
            acc += v.x + v.y + v.z + v.w;
            i += stride;
        }
        start = (start + 2048 * stride) % n_vec;
    }
    if (acc == 123.456f) *sink = acc;
}

__global__ void __launch_bounds__(256) k_peak_smem(int iters, float *sink)
{
    __shared__ float4 s[1024];
    for (int i = threadIdx.x; i < 1024; i += 256) s[i] = make_float4(i, 1, 2, 3);
    __syncthreads();
    float acc = 0.f;
    int idx = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll 16
        for (int r = 0; r < 64; ++r) {
            float4 v;                                     // volatile: the compiler must not merge the loads
            asm volatile("ld.volatile.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                         : "r"((uint32_t)__cvta_generic_to_shared(&s[(idx + r * 256) & 1023])));
            acc += v.x + v.y + v.z + v.w;
        }
        idx = (idx + 1) & 1023;
    }
    if (acc == 123.456f) *sink = acc;
}

__global__ void __launch_bounds__(256) k_peak_fma(int iters, float seed, float *sink)
{
    float a[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) a[q] = seed + q + threadIdx.x;
    const float m = 1.0000001f + seed, c = seed * 0.5f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = fmaf(a[q], m, c);
        }
    }
    float acc = 0.f;
#pragma unroll
    for (int q = 0; q < 8; ++q) acc += a[q];
    if (acc == 123.456f) *sink = acc;
}

__global__ void __launch_bounds__(256) k_peak_copy(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n_vec)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = src[i];
}

}  // namespace rubix

using namespace rubix;

extern "C" {

void rubix_stage_timing_enable(int32_t on) { g_timing = on != 0; }

int32_t rubix_stage_timing_read(float ms[RUBIX_N_STAGES], int32_t calls[RUBIX_N_STAGES])
{
    for (auto &p : g_pairs) {
        cudaError_t e = cudaEventSynchronize(p.b);
        if (e != cudaSuccess) return RUBIX_ERR_CUDA;
        float t = 0.f;
        cudaEventElapsedTime(&t, p.a, p.b);
        if (p.stage >= 0 && p.stage < RUBIX_N_STAGES) {
            ms[p.stage] += t;
            calls[p.stage] += 1;
        }
        g_free.push_back(p.a);
        g_free.push_back(p.b);
    }
    g_pairs.clear();
    return RUBIX_OK;
}

int32_t rubix_measure_peaks(float out[4], void *scratch, size_t scratch_bytes, void *stream)
{
    if (!out || !scratch) return RUBIX_ERR_NULL;
    if (scratch_bytes < ((size_t)64 << 20)) return RUBIX_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return RUBIX_ERR_CUDA;
    float *sink = (float *)scratch;
    auto time_best = [&](auto launch, int reps) {
        float best = 1e30f;
        for (int r = 0; r < reps + 1; ++r) {
            cudaEventRecord(a, st);
            launch();
            cudaEventRecord(b, st);
            cudaEventSynchronize(b);
            float t = 0.f;
            cudaEventElapsedTime(&t, a, b);
            if (r > 0 && t < best) best = t;
        }
        return best;
    };
    const int grid = 148 * 8;
    {   // L2: 32 MiB buffer
        const size_t n_vec = ((size_t)32 << 20) / 16;
        cudaMemsetAsync(scratch, 0, (size_t)32 << 20, st);
        const int iters = 2;
        const float t = time_best([&] { k_peak_l2<<<grid, 256, 0, st>>>((const float4 *)scratch + 16, n_vec - 16, iters, sink); }, 5);
        out[0] = (float)((double)grid * 256 * iters * 2048 * 16 / (t * 1e-3) / 1e9);
    }
    {
        const int iters = 2000;
        const float t = time_best([&] { k_peak_smem<<<grid, 256, 0, st>>>(iters, sink); }, 5);
        out[1] = (float)((double)grid * 256 * iters * 64 * 16 / (t * 1e-3) / 1e9);
    }
    {
        const int iters = 4000;
        const float t = time_best([&] { k_peak_fma<<<grid, 256, 0, st>>>(iters, 1e-9f, sink); }, 5);
        out[2] = (float)((double)grid * 256 * iters * 16 * 8 * 2 / (t * 1e-3) / 1e12);
    }
    {
        size_t half = scratch_bytes / 2;
        if (half > ((size_t)1 << 30)) half = (size_t)1 << 30;
        half &= ~(size_t)255;
        const size_t n_vec = half / 16;
        const float t = time_best([&] { k_peak_copy<<<148 * 16, 256, 0, st>>>((const float4 *)scratch, (float4 *)((char *)scratch + half), n_vec); }, 5);
        out[3] = (float)(2.0 * (double)half / (t * 1e-3) / 1e9);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return cudaGetLastError() == cudaSuccess ? RUBIX_OK : RUBIX_ERR_CUDA;
}

}  // extern "C"
