// Device-wide exclusive prefix sum of u32 (one of the "primitive algorithms" of P:L44 / P:L48 that the
// sort, tree-build and group stages are assembled from).  Three launches: per-block sums, one block
// scanning the block sums, per-block rescan with the carried-in offset.
#include "internal.cuh"

namespace bonsai {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
    __shared__ uint32_t wsum[kScanThreads / 32];
    __shared__ uint32_t tot;
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
        if (l >= o) x += y;
    }
    __syncthreads();  // protects wsum/tot against the previous call
    if (l == 31) wsum[w] = x;
    __syncthreads();
    uint32_t pre = 0;
#pragma unroll
    for (int k = 0; k < kScanThreads / 32; ++k) {
        uint32_t t = wsum[k];
        if (k < w) pre += t;
    }
    if (threadIdx.x == kScanThreads - 1) tot = pre + x;
    __syncthreads();
    *total = tot;
    return pre + x - v;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_sums(const uint32_t* __restrict__ in, uint32_t n,
                                                            uint32_t* __restrict__ sums) {
    const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < n) s += in[base + k];
    uint32_t total;
    block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// single block: sums[0..m) -> exclusive, sums[m] = grand total
__global__ void __launch_bounds__(kScanThreads) k_scan_top(uint32_t* __restrict__ sums, uint32_t m) {
    uint32_t carry = 0;
    for (uint32_t t0 = 0; t0 < m; t0 += kScanThreads) {
        uint32_t t = t0 + threadIdx.x;
        uint32_t v = (t < m) ? sums[t] : 0u;
        uint32_t total;
        uint32_t e = block_exclusive_scan(v, &total);
        if (t < m) sums[t] = carry + e;
        carry += total;
    }
    if (threadIdx.x == 0) sums[m] = carry;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const uint32_t* in, uint32_t* out, uint32_t n,
                                                             const uint32_t* __restrict__ sums, uint32_t m) {
    const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0u;
        s += v[k];
    }
    uint32_t total;
    uint32_t run = block_exclusive_scan(s, &total) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) out[base + k] = run;
        run += v[k];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = sums[m];
}

cudaError_t exclusive_scan_u32(Ctx* c, const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* tmp) {
    const uint32_t m = div_up(n, kScanTile);
    k_scan_sums<<<m, kScanThreads, 0, c->stream>>>(in, n, tmp);
    k_scan_top<<<1, kScanThreads, 0, c->stream>>>(tmp, m);
    k_scan_apply<<<m, kScanThreads, 0, c->stream>>>(in, out, n, tmp, m);
    c->launches += 3;
    return cudaGetLastError();
}

}  // namespace bonsai
