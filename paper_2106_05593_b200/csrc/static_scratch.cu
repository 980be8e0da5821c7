// static_scratch.cu -- mmc_mean_m_static (include/mmc.h): the magnetisation sums of the read-out kernel (kernels_layout.cu,
// observables_kernel: sum of m, of |m| and the number of non-empty cells) for callers that cannot
// allocate.  The per-block partial sums -- the scratch memory of that kernel, which the ctx path keeps in a cudaMalloc'ed
// buffer -- live here in a file-scope `static __device__` array; nothing in this file allocates, frees or synchronises.
//
// The array's name is a device symbol: in HOST code it is only a handle for cudaGetSymbolAddress, never an address a kernel
// may be given.  scratch_address() resolves it once per device, with that device current, and the launch passes the result.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/mmc.h"

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 16;
constexpr int kCellsPerBlock = kThreads * kCellsPerThread;                     // 4096
constexpr int kMaxBlocks = (int)(MMC_STATIC_MAX_CELLS / kCellsPerBlock);        // 4096
constexpr int kSums = 5;                                                        // mx, my, mz, |m|, count
constexpr int kHeadDoubles = 32;                                                // 256-byte control line: [0] = completion ticket
constexpr int kMaxDevices = 64;
static_assert((long long)kMaxBlocks * kCellsPerBlock == MMC_STATIC_MAX_CELLS, "whole blocks");
static_assert(sizeof(double) * (kHeadDoubles + kMaxBlocks * kSums) == MMC_STATIC_SCRATCH_BYTES, "size stated in mmc.h");

// One copy per GPU that loads the library, held until the process exits.  Shared by every call on that GPU.
static __device__ __align__(256) double g_static_scratch[kHeadDoubles + kMaxBlocks * kSums];

std::mutex g_mu;
double* g_scratch_addr[kMaxDevices] = {};       // device address of g_static_scratch per device ordinal, nullptr = not resolved

// Needs `device` current.  No allocation: the look-up returns the address of memory the module already owns.
int scratch_address(int device, double** out)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_addr[device]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { (void)cudaGetLastError(); return MMC_E_CUDA; }
        g_scratch_addr[device] = static_cast<double*>(p);
    }
    *out = g_scratch_addr[device];
    return MMC_OK;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sums of the block in a fixed order: lanes by the shuffle tree, then the 8 warps in index order.  Result in thread 0.
__device__ __forceinline__ void block_sum(double (&v)[kSums], double (*s_w)[kSums])
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < kSums; ++q) { const double w = warp_sum(v[q]); if (lane == 0) s_w[warp][q] = w; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < kSums; ++q) { double t = 0.0; for (int w = 0; w < kThreads / 32; ++w) t += s_w[w][q]; v[q] = t; }
    }
    __syncthreads();
}

// Block b sums cells [4096 b, 4096 (b + 1)) into scratch[32 + 5 b ..]; the block that draws the last ticket adds the
// partials of all blocks in index order and writes the means.  scratch[0] (the ticket, an unsigned) must be 0 at launch.
__global__ void __launch_bounds__(kThreads) mean_m_static_kernel(const float* __restrict__ mx, const float* __restrict__ my,
                                                                 const float* __restrict__ mz, long long n,
                                                                 double* __restrict__ scratch, double* __restrict__ out5)
{
    __shared__ double s_w[kThreads / 32][kSums];
    __shared__ bool s_last;
    double acc[kSums] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    const long long base = (long long)blockIdx.x * kCellsPerBlock + threadIdx.x;
    float x[kCellsPerThread], y[kCellsPerThread], z[kCellsPerThread];
#pragma unroll
    for (int r = 0; r < kCellsPerThread; ++r) {                  // all loads first: 48 independent coalesced requests per thread
        const long long c = base + (long long)r * kThreads;
        const bool in = c < n;
        x[r] = in ? __ldg(mx + c) : 0.f; y[r] = in ? __ldg(my + c) : 0.f; z[r] = in ? __ldg(mz + c) : 0.f;
    }
#pragma unroll
    for (int r = 0; r < kCellsPerThread; ++r) {
        // the arithmetic of observables_kernel: fp64 sums of the fp32 components, |m| = fp32 square root of the fp64 square sum
        const double a = x[r], b = y[r], c = z[r];
        const double l2 = a * a + b * b + c * c;
        if (l2 > 0.0) { acc[0] += a; acc[1] += b; acc[2] += c; acc[3] += (double)sqrtf((float)l2); acc[4] += 1.0; }
    }
    block_sum(acc, s_w);
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    double* part = scratch + kHeadDoubles;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < kSums; ++q) part[(size_t)blockIdx.x * kSums + q] = acc[q];
        __threadfence();                                         // partials visible before the ticket is drawn
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double tot[kSums] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (unsigned b = threadIdx.x; b < gridDim.x; b += kThreads) {
#pragma unroll
        for (int q = 0; q < kSums; ++q) tot[q] += __ldcg(part + (size_t)b * kSums + q);      // L2: written by other SMs
    }
    block_sum(tot, s_w);
    if (threadIdx.x == 0) {
        const double na = tot[4] > 0.0 ? tot[4] : 1.0;           // divisions, as the host side of the ctx read-out does
        out5[0] = tot[0] / na; out5[1] = tot[1] / na; out5[2] = tot[2] / na; out5[3] = tot[3] / na; out5[4] = tot[4];
    }
}

struct DeviceScope {
    int prev = -1; bool ok;
    explicit DeviceScope(int dev) { ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

extern "C" int mmc_mean_m_static(const float* mx, const float* my, const float* mz, long long n_cells, double* out5,
                                 int device, void* cuda_stream)
{
    if (n_cells < 0 || device < 0 || device >= kMaxDevices) return MMC_E_INVALID;
    if (n_cells > MMC_STATIC_MAX_CELLS) return MMC_E_TOO_LARGE;                 // before anything is enqueued
    if (n_cells > 0 && (!mx || !my || !mz || !out5)) return MMC_E_INVALID;
    DeviceScope ds(device);
    if (!ds.ok) { (void)cudaGetLastError(); return MMC_E_CUDA; }
    double* scratch = nullptr;
    const int rc = scratch_address(device, &scratch);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n_cells == 0) {
        if (out5 && cudaMemsetAsync(out5, 0, kSums * sizeof(double), st) != cudaSuccess) { (void)cudaGetLastError(); return MMC_E_CUDA; }
        return MMC_OK;
    }
    // the array still holds the previous call's ticket and partials: the ticket must start at zero, every partial that is
    // read is written first by this launch
    if (cudaMemsetAsync(scratch, 0, kHeadDoubles * sizeof(double), st) != cudaSuccess) { (void)cudaGetLastError(); return MMC_E_CUDA; }
    const unsigned blocks = (unsigned)((n_cells + kCellsPerBlock - 1) / kCellsPerBlock);
    mean_m_static_kernel<<<blocks, kThreads, 0, st>>>(mx, my, mz, n_cells, scratch, out5);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
