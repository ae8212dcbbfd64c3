// bonsai_diagnostics_static: the conserved-quantity diagnostics (R24 of DESIGN.md) for a caller that has nothing but
// its particle arrays and a 96-byte result buffer on the device.
//
// Who this is for.  bonsai_diagnostics() needs a context, and a context needs a caller-allocated workspace of
// bonsai_workspace_bytes() (hundreds of bytes per particle), although the reduction itself only needs ~111 KB of
// scratch: one row of 12 partial sums per thread block and a "last block done" ticket.  Some callers cannot provide
// even that: an in-situ energy monitor hooked into somebody else's simulation whose device memory pool is fully
// committed; a plug-in running under a fixed memory budget where the host application forbids cudaMalloc; a
// latency-critical loop that must not call cudaMalloc / cudaFree because both may synchronise the whole device; code
// that runs between two phases of an application that has already carved up every byte of HBM.  For those callers the
// scratch lives HERE, in a file-scope __device__ array that is part of the library image: every GPU that loads
// libbonsai holds these kDiagStaticBytes (113 920 bytes) from the moment the module is loaded until the process
// exits, whether or not the entry point is ever called.  Nothing in this file calls cudaMalloc, cudaFree, or any
// library routine that allocates.
//
// The kernel is a variant of k_diagnostics (integrate.cu): same grid rule, same accumulation and fold order, so the
// result is meant to equal bonsai_diagnostics() (tests/test_zz_no_alloc.py checks it within that path's own
// tolerance); only where the scratch and the ticket live differs.  integrate.cu is untouched.
//
// Rules that follow from one shared array:
//   * every call on a device uses the same scratch, and it keeps whatever the last call left in it.  The only word
//     that has to start at zero is the ticket; it is cleared on the stream before every launch (the partial rows are
//     overwritten before they are read).
//   * two calls that overlap on the GPU (different streams, or different host threads on different streams) race on
//     the scratch and give wrong sums.  Calls on ONE stream are ordered and safe.  The caller serialises.
//   * the first call on a device looks up the array's device address (cudaGetSymbolAddress, below).  That look-up can
//     load the module, which is not a stream operation: make the first call on each device before any stream capture
//     starts.  (No claim is made here about capturing later calls.)
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "bonsai.h"

namespace bonsai {
namespace {

constexpr int kN = 12;              // K, W, P[3], L[3], M, C[3]
constexpr int kThreads = 256;
constexpr int kRows = 1184;         // grid cap of the reduction: 8 blocks per SM on 148 SMs (as k_diagnostics)
constexpr int kMaxDevices = 64;

// Layout of the static scratch: a 256-byte header that holds the ticket, then kRows rows of kN doubles.
struct DiagScratch {
    unsigned int ticket;
    unsigned int pad[63];
    double partial[kRows * kN];
};
constexpr size_t kDiagStaticBytes = sizeof(DiagScratch);
static_assert(kDiagStaticBytes == BONSAI_DIAG_STATIC_SCRATCH_BYTES, "header and scratch layout disagree");

// The scratch itself.  In HOST code the name `g_diag_scratch` is only a handle for the runtime's symbol table -- it
// is not a device address and must never be handed to a kernel; scratch_for_current_device() asks the runtime for
// the real address.
static __device__ __align__(256) unsigned char g_diag_scratch[kDiagStaticBytes];

std::mutex g_mu;
DiagScratch* g_addr[kMaxDevices] = {};  // device address of g_diag_scratch, per device ordinal, filled on first use

// Set-up, once per device, with that device current: resolve the symbol to its address on the current device.
cudaError_t scratch_for_current_device(DiagScratch** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_diag_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_addr[dev] = static_cast<DiagScratch*>(p);
    }
    *out = g_addr[dev];
    return cudaSuccess;
}

__device__ __forceinline__ void warp_fold(double (&s)[kN]) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int k = 0; k < kN; ++k) s[k] += __shfl_down_sync(0xFFFFFFFFu, s[k], o);
}

// R24: fp64 sums of the fp32 state.  Per thread a strided accumulation, per warp a shuffle tree, per block a fold in
// warp order, and the block that draws the last ticket folds the rows in block order: the bits of the result do not
// depend on how the blocks were scheduled.
__global__ void __launch_bounds__(kThreads) k_diagnostics_static(const float4* __restrict__ pos,
                                                                 const float4* __restrict__ vel,
                                                                 const float4* __restrict__ acc, uint32_t n,
                                                                 DiagScratch* __restrict__ scratch,
                                                                 double* __restrict__ out) {
    __shared__ double s_w[kThreads / 32][kN];
    __shared__ bool s_last;
    double s[kN];
#pragma unroll
    for (int k = 0; k < kN; ++k) s[k] = 0.0;
    for (uint32_t i = blockIdx.x * kThreads + threadIdx.x; i < n; i += gridDim.x * kThreads) {
        const float4 p = __ldg(&pos[i]), v = __ldg(&vel[i]), a = __ldg(&acc[i]);
        const double x = p.x, y = p.y, z = p.z, m = p.w, vx = v.x, vy = v.y, vz = v.z;
        s[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        s[1] += 0.5 * m * (double)a.w;
        s[2] += m * vx; s[3] += m * vy; s[4] += m * vz;
        s[5] += m * (y * vz - z * vy);
        s[6] += m * (z * vx - x * vz);
        s[7] += m * (x * vy - y * vx);
        s[8] += m;
        s[9] += m * x; s[10] += m * y; s[11] += m * z;
    }
    warp_fold(s);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0)
#pragma unroll
        for (int k = 0; k < kN; ++k) s_w[w][k] = s[k];
    __syncthreads();
    if (threadIdx.x < kN) {
        double t = 0.0;
        for (int k = 0; k < kThreads / 32; ++k) t += s_w[k][threadIdx.x];
        __stcg(&scratch->partial[(size_t)blockIdx.x * kN + threadIdx.x], t);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&scratch->ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x < kN) {
        double t = 0.0;
        for (uint32_t b = 0; b < gridDim.x; ++b) t += __ldcg(&scratch->partial[(size_t)b * kN + threadIdx.x]);
        out[threadIdx.x] = t;
    }
}

}  // namespace
}  // namespace bonsai

using namespace bonsai;

extern "C" int bonsai_diagnostics_static(const float* pos_mass_dev, const float* vel_dev, const float* acc_pot_dev,
                                         uint32_t n, double* out12_dev, void* cuda_stream) {
    if (!pos_mass_dev || !vel_dev || !acc_pot_dev || !out12_dev) return BONSAI_EINVAL;
    if ((reinterpret_cast<uintptr_t>(pos_mass_dev) | reinterpret_cast<uintptr_t>(vel_dev) |
         reinterpret_cast<uintptr_t>(acc_pot_dev)) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(out12_dev) % 8 != 0)
        return BONSAI_EINVAL;
    if (n == 0 || n > BONSAI_DIAG_STATIC_MAX_N) return BONSAI_EINVAL;  // checked before any CUDA call
    DiagScratch* scratch = nullptr;
    if (scratch_for_current_device(&scratch) != cudaSuccess) return BONSAI_ECUDA;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    // the scratch still holds the previous call's ticket and rows (and anything an aborted launch left behind)
    if (cudaMemsetAsync(&scratch->ticket, 0, sizeof(unsigned int), stream) != cudaSuccess) return BONSAI_ECUDA;
    const uint32_t per_block = kThreads * 4;
    uint32_t blocks = n / per_block + (n % per_block != 0);
    if (blocks > (uint32_t)kRows) blocks = kRows;  // never more rows than the static array has
    k_diagnostics_static<<<blocks, kThreads, 0, stream>>>(reinterpret_cast<const float4*>(pos_mass_dev),
                                                          reinterpret_cast<const float4*>(vel_dev),
                                                          reinterpret_cast<const float4*>(acc_pot_dev), n, scratch,
                                                          out12_dev);
    return cudaGetLastError() == cudaSuccess ? BONSAI_OK : BONSAI_ECUDA;
}
