// Device-wide exclusive prefix sum of u32 (one of the "primitive algorithms" of P:L44 / P:L48 that the
// sort, tree-build and group stages are assembled from).  Two launches: per-block sums, then a per-block rescan in
// which every block first adds up the sums of the blocks before it (at most n / 2048 values, 8 KB at N = 2^22, out of
// L2) -- cheaper than a third launch with a single block scanning the sums (round 1: 10 us + a launch gap).
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
    // offset of this block = sum of the block sums before it (every block computes its own: no third kernel)
    uint32_t before = 0;
    for (uint32_t j = threadIdx.x; j < blockIdx.x; j += kScanThreads) before += sums[j];
    uint32_t offset;
    block_exclusive_scan(before, &offset);
    uint32_t total;
    uint32_t run = block_exclusive_scan(s, &total) + offset;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) out[base + k] = run;
        run += v[k];
    }
    if (blockIdx.x == m - 1 && threadIdx.x == 0) out[n] = offset + total;  // the last block knows the grand total
}

cudaError_t exclusive_scan_u32(Ctx* c, const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* tmp) {
    const uint32_t m = div_up(n, kScanTile);
    k_scan_sums<<<m, kScanThreads, 0, c->stream>>>(in, n, tmp);
    k_scan_apply<<<m, kScanThreads, 0, c->stream>>>(in, out, n, tmp, m);
    c->launches += 2;
    return cudaGetLastError();
}

}  // namespace bonsai
