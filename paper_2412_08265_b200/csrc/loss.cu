// Quadratic cube loss for the fused forward + adjoint entry point (BASELINE.json
// configs[4]: L = sum (cube - target)^2).  One pass over the final cube and the target:
//   grad[v] = 2 (cube[v] - target[v])                          (the upstream gradient of step 9)
//   L       = sum_v (cube[v] - target[v])^2                    in fp64, FIXED order: per-thread
//             grid-stride partial -> warp shuffle tree -> block tree -> one partial per CTA, then a
//             single CTA adds the partials in index order, so the value is bit-reproducible.
#include <mutex>

#include "common.cuh"

namespace rubix {

constexpr int kLossBlocks = 1184;          // 8 CTAs per SM
constexpr int kLossThreads = 256;

__device__ __forceinline__ double block_sum(double v, double *sm)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kLossThreads / 32; ++w) t += sm[w];
    return t;                               // valid in thread 0
}

// blockIdx.y = batch element (cubes back to back, n_vox voxels each; one row of partials per element)
__global__ void __launch_bounds__(kLossThreads)
k_residual_loss(const float *__restrict__ cube0, const float *__restrict__ target0, int64_t n_vox,
                float *__restrict__ grad0, double *__restrict__ partial0, int aligned)
{
    __shared__ double sm[kLossThreads / 32];
    const float *cube = cube0 + (size_t)blockIdx.y * n_vox, *target = target0 + (size_t)blockIdx.y * n_vox;
    float *grad = grad0 + (size_t)blockIdx.y * n_vox;
    double *partial = partial0 + (size_t)blockIdx.y * gridDim.x;
    double acc = 0.0;
    const int64_t n4 = aligned ? n_vox >> 2 : 0;            // 16-byte accesses only when all three arrays allow them
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const float4 c = __ldcs(reinterpret_cast<const float4 *>(cube) + i);
        const float4 t = __ldcs(reinterpret_cast<const float4 *>(target) + i);
        const float4 r = make_float4(c.x - t.x, c.y - t.y, c.z - t.z, c.w - t.w);
        __stcs(reinterpret_cast<float4 *>(grad) + i, make_float4(2.0f * r.x, 2.0f * r.y, 2.0f * r.z, 2.0f * r.w));
        acc += (double)r.x * r.x + (double)r.y * r.y + (double)r.z * r.z + (double)r.w * r.w;
    }
    for (int64_t i = (n4 << 2) + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vox; i += stride) {
        const float r = cube[i] - target[i];
        grad[i] = 2.0f * r;
        acc += (double)r * r;
    }
    const double tot = block_sum(acc, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kLossThreads)
k_loss_final(const double *__restrict__ partial0, int n, double *__restrict__ loss)
{
    __shared__ double sm[kLossThreads / 32];
    const double *partial = partial0 + (size_t)blockIdx.x * n;   // blockIdx.x = batch element
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += kLossThreads) acc += partial[i];
    const double tot = block_sum(acc, sm);
    if (threadIdx.x == 0) loss[blockIdx.x] = tot;
}

size_t loss_scratch_bytes(int32_t batch) { return align_up((size_t)batch * kLossBlocks * sizeof(double), 256); }

// `batch` cubes of n_vox voxels back to back: loss[b] and grad of every element, each summed exactly as a single call would
cudaError_t launch_residual_loss(const float *cube, const float *target, int64_t n_vox, float *grad,
                                 double *partial, double *loss, cudaStream_t st, int32_t batch)
{
    const int aligned = ((((uintptr_t)cube) | ((uintptr_t)target) | ((uintptr_t)grad)) & 15u) == 0 &&
                        (batch == 1 || (n_vox & 3) == 0);
    k_residual_loss<<<dim3(kLossBlocks, (unsigned)batch), kLossThreads, 0, st>>>(cube, target, n_vox, grad, partial, aligned);
    RUBIX_LAUNCH_CHECK();
    k_loss_final<<<(unsigned)batch, kLossThreads, 0, st>>>(partial, kLossBlocks, loss);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------
// No-allocation variant (rubix_residual_loss_static, include/rubix.h): the per-CTA partial sums of up to
// kLossStaticMaxBatch cubes live in a file-scope device array instead of a caller-provided workspace, for callers that
// cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads the library
// holds the array (kLossStaticMaxBatch x 1184 doubles = 606 208 bytes) until the process exits.
//
// In HOST code the name `s_loss_partials` is a stand-in for the symbol, not a device address: the address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current (each device has its own copy).
// Every block of k_residual_loss overwrites its slot before k_loss_final reads it, so nothing has to start at zero and the
// contents a previous call left behind are never read.  All calls on a device SHARE the array: calls that overlap on the
// GPU (different streams, no ordering between them) race on it.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) double s_loss_partials[(size_t)kLossStaticMaxBatch * kLossBlocks];

namespace {
constexpr int kMaxDevices = 64;
std::mutex s_mu;
double *s_partials_addr[kMaxDevices] = {};                  // device address of s_loss_partials, per device ordinal
}  // namespace

cudaError_t launch_residual_loss_static(const float *cube, const float *target, int64_t n_vox, float *grad, double *loss,
                                        cudaStream_t st, int32_t batch)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    double *partial = nullptr;
    {
        std::lock_guard<std::mutex> lk(s_mu);
        if (!s_partials_addr[dev]) {                        // set-up, once per device, with that device current
            double *ptr = nullptr;
            e = cudaGetSymbolAddress((void **)&ptr, s_loss_partials);
            if (e != cudaSuccess) return e;
            if (!ptr) return cudaErrorInvalidSymbol;
            s_partials_addr[dev] = ptr;
        }
        partial = s_partials_addr[dev];
    }
    const int aligned = ((((uintptr_t)cube) | ((uintptr_t)target) | ((uintptr_t)grad)) & 15u) == 0 &&
                        (batch == 1 || (n_vox & 3) == 0);
    k_residual_loss<<<dim3(kLossBlocks, (unsigned)batch), kLossThreads, 0, st>>>(cube, target, n_vox, grad, partial, aligned);
    RUBIX_LAUNCH_CHECK();
    k_loss_final<<<(unsigned)batch, kLossThreads, 0, st>>>(partial, kLossBlocks, loss);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix
