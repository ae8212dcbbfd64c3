// Stages a0 (bounding box), a1 (Morton keys), a2 (radix sort), a3 (reorder).
// P:L30 (Results): "Sorting of the particles along a Space Filling Curve (Morton (1966))" and
// "reordering of the particle properties ('moving')".  Readings R1-R6 of DESIGN.md.
#include "internal.cuh"

namespace bonsai {

// ------------------------------------------------------------------------------------------------
// a0  Bounding box -> root cube (R3): lo = per-axis minimum, side = smallest power of two strictly
// greater than the largest per-axis extent (extent evaluated in fp64 on the fp32 values; 0 -> 1).
// One grid-stride pass of float4 loads; warp shuffles, then one partial per block; the last block to
// finish (ticket) folds the partials and writes the cube.  min/max are exact in any order.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void warp_minmax(float (&mn)[3], float (&mx)[3]) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            mn[a] = fminf(mn[a], __shfl_xor_sync(0xFFFFFFFFu, mn[a], o));
            mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xFFFFFFFFu, mx[a], o));
        }
}

__global__ void __launch_bounds__(256) k_bbox(const float4* __restrict__ pos, uint32_t n, float* __restrict__ partial,
                                              Control* __restrict__ ctl) {
    __shared__ float s_mn[8][3], s_mx[8][3];
    __shared__ bool s_last;
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(&pos[i]);
        mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
        mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
        mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
    }
    warp_minmax(mn, mx);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0)
        for (int a = 0; a < 3; ++a) { s_mn[w][a] = mn[a]; s_mx[w][a] = mx[a]; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k)
            for (int a = 0; a < 3; ++a) { mn[a] = fminf(mn[a], s_mn[k][a]); mx[a] = fmaxf(mx[a], s_mx[k][a]); }
        for (int a = 0; a < 3; ++a) { partial[6 * blockIdx.x + a] = mn[a]; partial[6 * blockIdx.x + 3 + a] = mx[a]; }
        __threadfence();
        uint32_t t = atomicAdd(&ctl->bbox_ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int a = 0; a < 3; ++a) { mn[a] = INFINITY; mx[a] = -INFINITY; }
    for (uint32_t k = threadIdx.x; k < gridDim.x; k += blockDim.x)
        for (int a = 0; a < 3; ++a) {
            mn[a] = fminf(mn[a], __ldcg(&partial[6 * k + a]));
            mx[a] = fmaxf(mx[a], __ldcg(&partial[6 * k + 3 + a]));
        }
    warp_minmax(mn, mx);
    __syncthreads();
    if (l == 0)
        for (int a = 0; a < 3; ++a) { s_mn[w][a] = mn[a]; s_mx[w][a] = mx[a]; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k)
            for (int a = 0; a < 3; ++a) { mn[a] = fminf(mn[a], s_mn[k][a]); mx[a] = fmaxf(mx[a], s_mx[k][a]); }
        double ext = 0.0;
        for (int a = 0; a < 3; ++a) {
            ctl->lo[a] = mn[a];
            double e = (double)mx[a] - (double)mn[a];
            if (e > ext) ext = e;
        }
        double side = 1.0;
        if (ext > 0.0) {
            int e;
            frexp(ext, &e);  // ext = f 2^e, f in [0.5, 1)  =>  2^e > ext
            side = ldexp(1.0, e);
        }
        ctl->side = side;
        ctl->side_f = (float)side;
        ctl->scale = (float)(1073741824.0 / side);
        ctl->bbox_ticket = 0;  // ready for the next step
    }
}

// ------------------------------------------------------------------------------------------------
// a1  Morton keys (R1, R2, R4).  Per axis in fp32, round-to-nearest, no contraction:
//   t = x - lo;  u = t * (2^30 / side);  i = trunc(u) clamped to [0, 2^30 - 1].
// Octal digit of level L (1..30) = 4 x_bit + 2 y_bit + z_bit at bit 30 - L; words hi/mid/lo hold levels
// 1-10 / 11-20 / 21-30.  One thread per particle; 16 B in, 4 x 4 B out, all coalesced.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t spread10(uint32_t v) {  // 10 bits -> every third bit of 30
    v &= 0x3FFu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__device__ __forceinline__ uint32_t quantise(float x, float lo, float scale) {
    float u = __fmul_rn(__fsub_rn(x, lo), scale);
    if (!(u >= 0.0f)) return 0u;
    if (u >= 1073741824.0f) return 1073741823u;
    return (uint32_t)u;  // truncation
}

__global__ void __launch_bounds__(256) k_keys(const float4* __restrict__ pos, uint32_t n, const Control* __restrict__ ctl,
                                              uint32_t* __restrict__ khi, uint32_t* __restrict__ kmid,
                                              uint32_t* __restrict__ klo, uint32_t* __restrict__ idx) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float scale = ctl->scale;
    float4 p = __ldg(&pos[i]);
    uint32_t qx = quantise(p.x, ctl->lo[0], scale);
    uint32_t qy = quantise(p.y, ctl->lo[1], scale);
    uint32_t qz = quantise(p.z, ctl->lo[2], scale);
    khi[i] = (spread10(qx >> 20) << 2) | (spread10(qy >> 20) << 1) | spread10(qz >> 20);
    kmid[i] = (spread10(qx >> 10) << 2) | (spread10(qy >> 10) << 1) | spread10(qz >> 10);
    klo[i] = (spread10(qx) << 2) | (spread10(qy) << 1) | spread10(qz);
    idx[i] = i;
}

// ------------------------------------------------------------------------------------------------
// a2  Stable LSD radix sort of (90-bit key, index) records (R5): 9 passes of 10-bit digits (3 per key
// word, lo word first).  Per pass:
//   k_sort_count    per-tile digit histogram (shared-memory atomics), digit-major [digit][tile]
//   k_sort_scan     one block per digit: exclusive prefix over tiles, plus the digit's global base taken
//                   from the all-pass histogram that k_sort_ghist builds once per sort
//   k_sort_scatter  stable in-tile ranking with __match_any_sync + per-warp digit counters, then the
//                   record (3 key words + index) is written to its final slot
// Records are kept as four u32 arrays so every read and the key-word of interest are coalesced.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_sort_ghist(const uint32_t* __restrict__ khi, const uint32_t* __restrict__ kmid,
                                                    const uint32_t* __restrict__ klo, uint32_t n,
                                                    uint32_t* __restrict__ ghist) {
    __shared__ uint32_t h[kSortPasses * kRadix];
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += blockDim.x) h[k] = 0;
    __syncthreads();
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        uint32_t w[3] = {__ldg(&klo[i]), __ldg(&kmid[i]), __ldg(&khi[i])};
#pragma unroll
        for (int p = 0; p < kSortPasses; ++p) {
            uint32_t d = (w[p / 3] >> (kRadixBits * (p % 3))) & (kRadix - 1);
            atomicAdd(&h[p * kRadix + d], 1u);
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += blockDim.x)
        if (h[k]) atomicAdd(&ghist[k], h[k]);
}

// exclusive scan of each pass's histogram: ghist[p][d] <- sum_{d' < d} ghist[p][d'].  One block per pass.
__global__ void __launch_bounds__(kRadix) k_sort_gscan(uint32_t* __restrict__ ghist) {
    __shared__ uint32_t s[kRadix];
    __shared__ uint32_t wsum[kRadix / 32];
    uint32_t* h = ghist + blockIdx.x * kRadix;
    uint32_t v = h[threadIdx.x];
    uint32_t x = v;
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
        if (l >= o) x += y;
    }
    if (l == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        uint32_t t = wsum[l];
        uint32_t y = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t z = __shfl_up_sync(0xFFFFFFFFu, y, o);
            if (l >= o) y += z;
        }
        wsum[l] = y - t;
    }
    __syncthreads();
    (void)s;
    h[threadIdx.x] = x - v + wsum[w];
}

__global__ void __launch_bounds__(kSortThreads) k_sort_count(const uint32_t* __restrict__ word, uint32_t n, int shift,
                                                             uint32_t n_tiles, uint32_t* __restrict__ tile_count) {
    __shared__ uint32_t h[kRadix];
    for (int k = threadIdx.x; k < kRadix; k += kSortThreads) h[k] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kSortTile;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        uint32_t i = base + r * kSortThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[(__ldg(&word[i]) >> shift) & (kRadix - 1)], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < kRadix; k += kSortThreads) tile_count[(size_t)k * n_tiles + blockIdx.x] = h[k];
}

// One block per digit: tile_count[d][t] <- ghist_base[d] + sum_{t' < t} tile_count[d][t'].
__global__ void __launch_bounds__(256) k_sort_scan(uint32_t* __restrict__ tile_count, uint32_t n_tiles,
                                                   const uint32_t* __restrict__ gbase) {
    __shared__ uint32_t wsum[8];
    __shared__ uint32_t carry;
    uint32_t* row = tile_count + (size_t)blockIdx.x * n_tiles;
    if (threadIdx.x == 0) carry = gbase[blockIdx.x];
    __syncthreads();
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (uint32_t t0 = 0; t0 < n_tiles; t0 += 256) {
        uint32_t t = t0 + threadIdx.x;
        uint32_t v = (t < n_tiles) ? row[t] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
            if (l >= o) x += y;
        }
        if (l == 31) wsum[w] = x;
        __syncthreads();
        uint32_t pre = carry;
        for (int k = 0; k < w; ++k) pre += wsum[k];
        if (t < n_tiles) row[t] = pre + x - v;
        __syncthreads();
        if (threadIdx.x == 255) carry = pre + x;
        __syncthreads();
    }
}

struct SortIO {
    const uint32_t* in_key[3];
    const uint32_t* in_idx;
    uint32_t* out_key[3];
    uint32_t* out_idx;
};

__global__ void __launch_bounds__(kSortThreads) k_sort_scatter(SortIO io, int word, int shift, uint32_t n,
                                                               uint32_t n_tiles,
                                                               const uint32_t* __restrict__ tile_offset) {
    extern __shared__ uint32_t s_cnt[];  // [warps][kRadix]
    constexpr int kWarps = kSortThreads / 32;
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < kWarps * kRadix; k += kSortThreads) s_cnt[k] = 0;
    __syncthreads();
    uint32_t* cnt = s_cnt + w * kRadix;
    // warp w owns the contiguous run [base_w, base_w + 32 * kSortItems) of the tile: round r, lane l
    const uint32_t base_w = blockIdx.x * kSortTile + w * (32 * kSortItems);
    const uint32_t* __restrict__ wsrc = io.in_key[word];
    uint32_t dig[kSortItems];
    uint32_t rnk[kSortItems];
    const uint32_t lt = (1u << l) - 1u;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        uint32_t i = base_w + r * 32 + l;
        bool valid = i < n;
        uint32_t d = valid ? ((__ldg(&wsrc[i]) >> shift) & (kRadix - 1)) : (uint32_t)kRadix;  // kRadix = "no key"
        uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
        uint32_t pre = 0;
        if (valid) pre = cnt[d];
        __syncwarp();
        if (valid && (peers & lt) == 0) cnt[d] = pre + __popc(peers);
        __syncwarp();
        dig[r] = d;
        rnk[r] = pre + __popc(peers & lt);
    }
    __syncthreads();
    // per digit: exclusive prefix over warps + the tile's global offset
    for (int d = threadIdx.x; d < kRadix; d += kSortThreads) {
        uint32_t run = tile_offset[(size_t)d * n_tiles + blockIdx.x];
#pragma unroll
        for (int k = 0; k < kWarps; ++k) {
            uint32_t t = s_cnt[k * kRadix + d];
            s_cnt[k * kRadix + d] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        uint32_t i = base_w + r * 32 + l;
        if (i < n) {
            uint32_t dst = cnt[dig[r]] + rnk[r];
            io.out_key[0][dst] = __ldg(&io.in_key[0][i]);
            io.out_key[1][dst] = __ldg(&io.in_key[1][i]);
            io.out_key[2][dst] = __ldg(&io.in_key[2][i]);
            io.out_idx[dst] = __ldg(&io.in_idx[i]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a3  Reorder ("moving"): sorted_pos[i] = pos_mass[perm[i]].  Gather of 16-byte records.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_reorder(const float4* __restrict__ pos, const uint32_t* __restrict__ perm,
                                                 uint32_t n, float4* __restrict__ sorted_pos) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) sorted_pos[i] = __ldg(&pos[__ldg(&perm[i])]);
}

// ------------------------------------------------------------------------------------------------
cudaError_t stage_bbox(Ctx* c) {
    uint32_t blocks = min(div_up(c->n, 256 * 8), (uint32_t)(c->num_sms * 8));
    k_bbox<<<blocks, 256, 0, c->stream>>>(c->pos_mass, c->n, c->b.bbox_partial, c->b.ctl);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_keys(Ctx* c) {
    k_keys<<<div_up(c->n, 256), 256, 0, c->stream>>>(c->pos_mass, c->n, c->b.ctl, c->b.key[0][0], c->b.key[0][1],
                                                     c->b.key[0][2], c->b.idx[0]);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_sort(Ctx* c) {
    const uint32_t n = c->n;
    const uint32_t n_tiles = div_up(n, kSortTile);
    Buffers& b = c->b;
    cudaError_t e = cudaMemsetAsync(b.ghist, 0, sizeof(uint32_t) * kSortPasses * kRadix, c->stream);
    if (e != cudaSuccess) return e;
    uint32_t hb = min(div_up(n, 256 * 16), (uint32_t)(c->num_sms * 4));
    k_sort_ghist<<<hb, 256, 0, c->stream>>>(b.key[0][0], b.key[0][1], b.key[0][2], n, b.ghist);
    k_sort_gscan<<<kSortPasses, kRadix, 0, c->stream>>>(b.ghist);
    c->launches += 2;
    static bool attr_set = false;
    const size_t smem = sizeof(uint32_t) * (kSortThreads / 32) * kRadix;
    if (!attr_set) {
        e = cudaFuncSetAttribute(k_sort_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    int cur = 0;
    for (int p = 0; p < kSortPasses; ++p) {
        const int word = 2 - p / 3;  // lo word (index 2) first
        const int shift = kRadixBits * (p % 3);
        SortIO io;
        for (int k = 0; k < 3; ++k) { io.in_key[k] = b.key[cur][k]; io.out_key[k] = b.key[cur ^ 1][k]; }
        io.in_idx = b.idx[cur];
        io.out_idx = b.idx[cur ^ 1];
        k_sort_count<<<n_tiles, kSortThreads, 0, c->stream>>>(b.key[cur][word], n, shift, n_tiles, b.tile_count);
        k_sort_scan<<<kRadix, 256, 0, c->stream>>>(b.tile_count, n_tiles, b.ghist + p * kRadix);
        k_sort_scatter<<<n_tiles, kSortThreads, smem, c->stream>>>(io, word, shift, n, n_tiles, b.tile_count);
        c->launches += 3;
        cur ^= 1;
    }
    c->sorted_buf = cur;
    return cudaGetLastError();
}

cudaError_t stage_reorder(Ctx* c) {
    k_reorder<<<div_up(c->n, 256), 256, 0, c->stream>>>(c->pos_mass, c->b.idx[c->sorted_buf], c->n, c->b.sorted_pos);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace bonsai
