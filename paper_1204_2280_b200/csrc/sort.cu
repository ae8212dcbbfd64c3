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
                                              Control* __restrict__ ctl, const Gate gate) {
    __shared__ float s_mn[8][3], s_mx[8][3];
    __shared__ bool s_last;
    if (gate_closed(gate)) return;
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    // four independent 16-byte loads in flight per thread: with one, the pass is latency-bound (13 % issue-active, 48
    // long-scoreboard stalls per issue, 2.6 TB/s; profiles/r2_nonwalk_ncu.md)
    const uint32_t stride = gridDim.x * blockDim.x;
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3u * stride < n; i += 4u * stride) {
        float4 p[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) p[k] = __ldg(&pos[i + k * stride]);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            mn[0] = fminf(mn[0], p[k].x); mx[0] = fmaxf(mx[0], p[k].x);
            mn[1] = fminf(mn[1], p[k].y); mx[1] = fmaxf(mx[1], p[k].y);
            mn[2] = fminf(mn[2], p[k].z); mx[2] = fmaxf(mx[2], p[k].z);
        }
    }
    for (; i < n; i += stride) {
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
        // one epoch per sort pass of this build (kSortPasses of them); on wrap-around of the 30-bit tag the look-back
        // table is cleared by k_sort_gscan before the first pass
        uint32_t ep = ctl->sort_epoch + 8u;
        ctl->look_wrap = 0u;
        if (ep >= (1u << 30) - 16u) {
            ep = 8u;
            ctl->look_wrap = 1u;
        }
        ctl->sort_epoch = ep;
    }
}

// ------------------------------------------------------------------------------------------------
// a1  Morton keys (R1, R2, R4).  Per axis in fp32, round-to-nearest, no contraction:
//   t = x - lo;  u = t * (2^30 / side);  i = trunc(u) clamped to [0, 2^30 - 1].
// Octal digit of level L (1..30) = 4 x_bit + 2 y_bit + z_bit at bit 30 - L; words hi/mid/lo hold levels
// 1-10 / 11-20 / 21-30.  Grid-stride, 16 B in, 3 x 4 B out, all coalesced.  The same pass builds the
// digit histograms of the sort passes that will run in shared memory (a histogram does not depend on the order
// of the keys, so the sort never has to count again).
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

// w[0] = lo word (levels 21-30), w[1] = mid, w[2] = hi: the order the LSD passes consume them in.
__device__ __forceinline__ void morton_words(const float4 p, const float lox, const float loy, const float loz,
                                             const float scale, uint32_t (&w)[3]) {
    const uint32_t qx = quantise(p.x, lox, scale);
    const uint32_t qy = quantise(p.y, loy, scale);
    const uint32_t qz = quantise(p.z, loz, scale);
    w[2] = (spread10(qx >> 20) << 2) | (spread10(qy >> 20) << 1) | spread10(qz >> 20);
    w[1] = (spread10(qx >> 10) << 2) | (spread10(qy >> 10) << 1) | spread10(qz >> 10);
    w[0] = (spread10(qx) << 2) | (spread10(qy) << 1) | spread10(qz);
}

__global__ void __launch_bounds__(kKeysThreads) k_keys(const float4* __restrict__ pos, uint32_t n,
                                                       const Control* __restrict__ ctl, uint32_t* __restrict__ khi,
                                                       uint32_t* __restrict__ kmid, uint32_t* __restrict__ klo,
                                                       uint32_t* __restrict__ ghist, const int first_pass, const Gate gate) {
    __shared__ uint32_t h[kSortPasses * kRadix];
    if (gate_closed(gate)) return;
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += kKeysThreads) h[k] = 0;
    __syncthreads();
    const float scale = ctl->scale, lox = ctl->lo[0], loy = ctl->lo[1], loz = ctl->lo[2];
    const uint32_t lane = threadIdx.x & 31;
    // warp-uniform trip count: the vote below needs the whole warp
    for (uint32_t base = blockIdx.x * kKeysThreads + (threadIdx.x & ~31u); base < n; base += gridDim.x * kKeysThreads) {
        const uint32_t i = base + lane;
        const bool valid = i < n;
        uint32_t w[3] = {0u, 0u, 0u};
        if (valid) {
            morton_words(__ldg(&pos[i]), lox, loy, loz, scale, w);
            klo[i] = w[0];
            kmid[i] = w[1];
            khi[i] = w[2];
        }
#pragma unroll
        for (int p = 0; p < kSortPasses; ++p) {  // pass p sorts digit p % 3 of word 1 + p / 3 (mid, then hi)
            if (p < first_pass) continue;        // (the lowest mid digits may be left to the tie repair, see stage_sort)
            const uint32_t d = (w[1 + p / 3] >> (kRadixBits * (p % 3))) & (kRadix - 1);
            // a warp whose 32 keys share the digit (the leading digits of clustered or pre-sorted input)
            // adds once instead of serialising 32 same-address atomics; only the hi word's digits (levels 1-10) are
            // ever that uniform, the mid word's are as good as random and skip the vote
            if (p >= 3) {
                const uint32_t d0 = __shfl_sync(0xFFFFFFFFu, d, 0);
                if (__all_sync(0xFFFFFFFFu, valid && d == d0)) {
                    if (lane == 0) atomicAdd(&h[p * kRadix + d], 32u);
                } else if (valid) {
                    atomicAdd(&h[p * kRadix + d], 1u);
                }
            } else if (valid) {
                atomicAdd(&h[p * kRadix + d], 1u);
            }
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < kSortPasses * kRadix; k += kKeysThreads)
        if (h[k]) atomicAdd(&ghist[k], h[k]);
}

// exclusive scan of each pass's histogram: ghist[p][d] <- sum_{d' < d} ghist[p][d'].  One block per pass.
__global__ void __launch_bounds__(kRadix) k_sort_gscan(uint32_t* __restrict__ ghist, Control* __restrict__ ctl,
                                                       unsigned long long* __restrict__ look, size_t look_entries,
                                                       const Gate gate) {
    __shared__ uint32_t wsum[kRadix / 32];
    if (gate_closed(gate)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        ctl->n_long_runs = 0;
        ctl->tree_fresh = 1;  // R30: a new tree is being built; the next recorded walk is its reference
    }
    if (ctl->look_wrap != 0u)  // the epoch tag wrapped (k_bbox): forget every stale entry of the look-back table
        for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < look_entries; k += (size_t)gridDim.x * blockDim.x)
            look[k] = 0ull;
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
    h[threadIdx.x] = x - v + wsum[w];
}

// ------------------------------------------------------------------------------------------------
// a2  Stable radix sort of (90-bit key, index) records (R5).  LSD passes of 10-bit digits over (current
// 30-bit word, index) PAIRS: a pass reads 8 B and writes 8 B per particle.  When the passes of one word are
// done the next word is fetched through the index (gather from the load-order key arrays); the sorted
// 90-bit keys are re-derived from the reordered positions in k_reorder (a key is a pure function of the
// position and the root cube).  The sort runs FOUR to SIX passes, over the leading 40 to 60 bits of the
// mid and hi words (by size, see sort_first_pass): the remaining bits almost never decide the order; the
// runs of equal leading bits are put in order after the reorder, short ones in place by k_sort_ties, long
// ones (coincident particles, clumps far smaller than the cells the passes resolve) by k_sort_long_runs
// (see stage_sort_ties).
//
// One kernel per pass, single sweep with decoupled look-back:
//   * tiles of kSortTile pairs are handed out by an atomic ticket, so a tile's predecessors have
//     always started;
//   * stable in-tile ranking with warp ballots and per-warp digit counters (warp w owns a
//     contiguous run of the tile, round r, lane l  ->  order = (warp, round, lane));
//   * each tile publishes, per digit, first its own count (AGGREGATE) and, after summing its
//     predecessors' entries back to the nearest INCLUSIVE one, its inclusive prefix; an entry is one
//     64-bit word {epoch : 30, flag : 2, value : 32}, the epoch (one per pass launch) makes stale
//     entries of earlier passes read as "not yet written", so the table is never cleared; the epoch
//     lives on the device (Control::sort_epoch, advanced by k_bbox once per build) so that a captured
//     CUDA graph of the step can be replayed;
//   * the digit's global base comes from the all-pass histogram k_keys built;
//   * pairs are first permuted into tile-sorted order in shared memory (aliasing the counters), so
//     the global stores are runs of consecutive addresses per digit.
// ------------------------------------------------------------------------------------------------
struct SortPass {
    const uint32_t* key_in;    // MODE 1: pair keys of the previous pass
    const uint32_t* idx_in;    // MODE 1, 2: indices of the previous pass
    const uint32_t* src_word;  // MODE 0, 2: load-order key word of this phase
    uint32_t* key_out;         // nullptr on the last pass
    uint32_t* idx_out;
    const uint32_t* gbase;     // [kRadix] exclusive digit bases of this pass
    unsigned long long* look;  // [n_tiles][kRadix]
    uint32_t* ticket;
    const Control* ctl;
    Gate gate;                 // the pass only runs when this gate is open (R30)
    uint32_t n, n_tiles, pass; // pass = 0 .. kSortPasses - 1: epoch of the launch = ctl->sort_epoch + pass
    int shift;
};

constexpr uint32_t kFlagAgg = 1u, kFlagIncl = 2u;

__device__ __forceinline__ unsigned long long look_pack(uint32_t epoch, uint32_t flag, uint32_t value) {
    return ((unsigned long long)((epoch << 2) | flag) << 32) | value;
}
__device__ __forceinline__ unsigned long long look_load(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void look_store(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// MODE 0: key = src_word[i], idx = i.   MODE 1: key = key_in[i], idx = idx_in[i].
// MODE 2: idx = idx_in[i], key = src_word[idx].
template <int MODE>
__global__ void __launch_bounds__(kSortThreads, kSortBlocksPerSM) k_sort_pass(const SortPass a) {
    extern __shared__ __align__(16) uint32_t smem[];
    constexpr int kWarps = kSortThreads / 32;
    constexpr int kDig = kRadix / kSortThreads;      // digits per thread in the per-digit steps
    struct __align__(4 * kDig) DigVec { uint32_t x[kDig]; };
    uint32_t* s_cnt = smem;                          // [kWarps][kRadix]; later the staging area
    uint32_t* s_tstart = smem + kWarps * kRadix;     // [kRadix] first tile-sorted slot of the digit
    uint32_t* s_gdst = s_tstart + kRadix;            // [kRadix] global slot of tile-sorted slot 0 of the digit
    __shared__ uint32_t s_tile;
    __shared__ uint32_t s_wsum[kWarps];
    const int tid = threadIdx.x, l = tid & 31, w = tid >> 5;
    if (gate_closed(a.gate)) return;
    const uint32_t epoch = __ldcg(&a.ctl->sort_epoch) + a.pass;

    if (tid == 0) {
        const uint32_t t = atomicAdd(a.ticket, 1u);
        if (t == a.n_tiles - 1) *a.ticket = 0;  // every tile has drawn: ready for the next pass
        s_tile = t;
    }
    {
        uint4* z = reinterpret_cast<uint4*>(s_cnt);
        for (int k = tid; k < kWarps * kRadix / 4; k += kSortThreads) z[k] = make_uint4(0, 0, 0, 0);
    }
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base_w = tile * kSortTile + w * (32 * kSortItems);
    uint32_t* cnt = s_cnt + w * kRadix;

    uint32_t key[kSortItems];
    uint32_t rnk[kSortItems];
    if (MODE == 2) {
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) {
            const uint32_t i = base_w + r * 32 + l;
            rnk[r] = (i < a.n) ? __ldg(&a.idx_in[i]) : 0u;
        }
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) key[r] = __ldg(&a.src_word[rnk[r]]);
    } else {
        const uint32_t* __restrict__ src = (MODE == 0) ? a.src_word : a.key_in;
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) {
            const uint32_t i = base_w + r * 32 + l;
            key[r] = (i < a.n) ? __ldg(&src[i]) : 0u;
        }
    }
    // Ranking: lanes with the same digit elect their lowest lane, which reserves popc(peers) consecutive
    // ranks in the warp's counter with one shared-memory atomic and broadcasts the old value.  Rounds are
    // independent instructions (no warp barrier in between), so the 16 match / atomic / shuffle chains
    // overlap; the atomics of one warp reach the counter in program order, which keeps the ranks stable.
    const uint32_t lt = (1u << l) - 1u;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const bool valid = base_w + r * 32 + l < a.n;
        const uint32_t d = valid ? ((key[r] >> a.shift) & (kRadix - 1)) : (uint32_t)kRadix;  // kRadix = "no key"
        // lanes holding the same digit, one ballot per digit bit (MATCH.ANY serialises over the distinct values
        // of the warp and is several times slower here: 1024 bins make almost every lane distinct)
        uint32_t peers = __ballot_sync(0xFFFFFFFFu, valid);
        if (!valid) peers = ~peers;
#pragma unroll
        for (int bit = 0; bit < kRadixBits; ++bit) {
            const bool on = (d >> bit) & 1u;
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, on);
            peers &= on ? m : ~m;
        }
        const int leader = __ffs(peers) - 1;
        uint32_t pre = 0;
        if (valid && l == leader) pre = atomicAdd(&cnt[d], (uint32_t)__popc(peers));
        pre = __shfl_sync(0xFFFFFFFFu, pre, leader);
        rnk[r] = pre + __popc(peers & lt);
    }
    __syncthreads();

    // per digit (kDig consecutive digits per thread): exclusive prefix over warps, tile total
    const int d0 = kDig * tid;
    uint32_t tot[kDig];
#pragma unroll
    for (int q = 0; q < kDig; ++q) tot[q] = 0u;
#pragma unroll
    for (int k = 0; k < kWarps; ++k) {
        DigVec* pv = reinterpret_cast<DigVec*>(&s_cnt[k * kRadix + d0]);
        DigVec v = *pv, o;
#pragma unroll
        for (int q = 0; q < kDig; ++q) {
            o.x[q] = tot[q];
            tot[q] += v.x[q];
        }
        *pv = o;
    }
    unsigned long long* my_look = a.look + (size_t)tile * kRadix + d0;
    const uint32_t first_flag = (tile == 0) ? kFlagIncl : kFlagAgg;
#pragma unroll
    for (int q = 0; q < kDig; ++q) look_store(my_look + q, look_pack(epoch, first_flag, tot[q]));
    // block-wide exclusive scan of the digit totals -> first tile-sorted slot of each digit
    uint32_t x = 0;
#pragma unroll
    for (int q = 0; q < kDig; ++q) x += tot[q];
    const uint32_t mine = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
        if (l >= o) x += y;
    }
    if (l == 31) s_wsum[w] = x;
    __syncthreads();
    uint32_t tstart = x - mine;
#pragma unroll
    for (int k = 0; k < kWarps; ++k)
        if (k < w) tstart += s_wsum[k];
    // The tile's aggregates are out; everything that only needs tile-local information comes BEFORE the look-back
    // (first slot of each digit, slot of every pair, staging into shared memory), so the predecessors get that much
    // more time to publish and the wait below is that much shorter.
    {
        uint32_t ts = tstart;
#pragma unroll
        for (int q = 0; q < kDig; ++q) {
            s_tstart[d0 + q] = ts;
            ts += tot[q];
        }
    }
    __syncthreads();

    // tile-sorted slot of every pair (the counters now hold the exclusive prefix over warps)
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const bool valid = base_w + r * 32 + l < a.n;
        if (valid) {
            const uint32_t d = (key[r] >> a.shift) & (kRadix - 1);
            rnk[r] += s_tstart[d] + cnt[d];
        }
    }
    __syncthreads();  // counters are dead: reuse them as the staging area
    uint32_t* s_key = smem;
    uint32_t* s_idx = smem + kSortTile;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t i = base_w + r * 32 + l;
        if (i < a.n) {
            s_key[rnk[r]] = key[r];
            s_idx[rnk[r]] = (MODE == 0) ? i : __ldg(&a.idx_in[i]);
        }
    }

    // decoupled look-back, all of the thread's digits in flight together
    uint32_t excl[kDig];
#pragma unroll
    for (int q = 0; q < kDig; ++q) excl[q] = 0u;
    if (tile > 0) {
        uint32_t j[kDig];
        uint32_t pending = (1u << kDig) - 1u;
#pragma unroll
        for (int q = 0; q < kDig; ++q) j[q] = tile - 1;
        const uint32_t want = epoch;
        // kLookBatch predecessors per digit are fetched together and consumed nearest-first: when a whole wave of
        // tiles publishes its aggregates at the same moment, the inclusive prefixes ripple forward one L2 round
        // trip per kLookBatch tiles instead of one per tile.
        while (pending) {
            bool missed = false;
            unsigned long long v[kDig][kLookBatch];
#pragma unroll
            for (int q = 0; q < kDig; ++q)
#pragma unroll
                for (int t = 0; t < kLookBatch; ++t)
                    if ((pending & (1u << q)) && j[q] >= (uint32_t)t)
                        v[q][t] = look_load(a.look + (size_t)(j[q] - t) * kRadix + d0 + q);
#pragma unroll
            for (int q = 0; q < kDig; ++q) {
                const uint32_t jq = j[q];
#pragma unroll
                for (int t = 0; t < kLookBatch; ++t) {
                    if (!(pending & (1u << q)) || jq < (uint32_t)t || j[q] != jq - t) continue;
                    const uint32_t tag = (uint32_t)(v[q][t] >> 32);
                    if ((tag >> 2) != want) {          // not written yet in this pass: retry from here, a little later
                        if (t == 0) missed = true;
                        continue;
                    }
                    excl[q] += (uint32_t)v[q][t];
                    if ((tag & 3u) == kFlagIncl) pending &= ~(1u << q);
                    else --j[q];                       // tile 0 always publishes INCLUSIVE, so j never passes 0
                }
            }
            if (missed) __nanosleep(kLookSleepNs);     // keeps a waiting wave from flooding L2 with re-reads
        }
#pragma unroll
        for (int q = 0; q < kDig; ++q) look_store(my_look + q, look_pack(epoch, kFlagIncl, excl[q] + tot[q]));
    }
#pragma unroll
    for (int q = 0; q < kDig; ++q) {
        s_gdst[d0 + q] = __ldg(&a.gbase[d0 + q]) + excl[q] - tstart;
        tstart += tot[q];
    }
    __syncthreads();
    const uint32_t tile_base = tile * kSortTile;
    const uint32_t n_valid = min((uint32_t)kSortTile, a.n - tile_base);
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t s = r * kSortThreads + tid;
        if (s < n_valid) {
            const uint32_t k = s_key[s];
            const uint32_t dst = s_gdst[(k >> a.shift) & (kRadix - 1)] + s;
            if (a.key_out) a.key_out[dst] = k;
            a.idx_out[dst] = s_idx[s];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a3  Reorder ("moving"): sorted_pos[i] = pos_mass[perm[i]], a gather of 16-byte records; the
// sorted key words are re-derived from the record in flight (12 B more written, nothing more read).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_reorder(const float4* __restrict__ pos, const uint32_t* __restrict__ perm,
                                                 uint32_t n, const Control* __restrict__ ctl,
                                                 float4* __restrict__ sorted_pos, uint32_t* __restrict__ khi,
                                                 uint32_t* __restrict__ kmid, uint32_t* __restrict__ klo,
                                                 const Gate gate) {
    if (gate_closed(gate)) return;
    const float lox = ctl->lo[0], loy = ctl->lo[1], loz = ctl->lo[2], scale = ctl->scale;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 p = __ldg(&pos[__ldg(&perm[i])]);
        sorted_pos[i] = p;
        if (khi == nullptr) continue;  // refresh of a frozen tree (R25): the keys stay those of the last build
        uint32_t w[3];
        morton_words(p, lox, loy, loz, scale, w);
        klo[i] = w[0];
        kmid[i] = w[1];
        khi[i] = w[2];
    }
}

// ------------------------------------------------------------------------------------------------
cudaError_t stage_bbox(Ctx* c) {
    uint32_t blocks = min(min(div_up(c->n, 256 * 8), (uint32_t)(c->num_sms * 8)), (uint32_t)kBboxMaxBlocks);
    k_bbox<<<blocks, 256, 0, c->stream>>>(c->pos_mass, c->n, c->b.bbox_partial, c->b.ctl, c->gate);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_keys(Ctx* c) {
    Buffers& b = c->b;
    cudaError_t e = cudaMemsetAsync(b.ghist, 0, sizeof(uint32_t) * kSortPasses * kRadix, c->stream);
    if (e != cudaSuccess) return e;
    const uint32_t blocks = min(div_up(c->n, kKeysThreads), (uint32_t)(c->num_sms * 2));
    k_keys<<<blocks, kKeysThreads, 0, c->stream>>>(c->pos_mass, c->n, b.ctl, b.key[0][0], b.key[0][1], b.key[0][2],
                                                   b.ghist, sort_first_pass(c), c->gate);
    c->launches += 1;
    return cudaGetLastError();
}

// Ties of the sort.  After the passes the particles are ordered by the leading 60 - cut bits of (hi, mid) -- cut = 0,
// 10 or 20 low bits of the mid word are skipped with the first passes, see stage_sort -- and, inside a run of equal
// leading bits, by load index (LSD passes are stable).  Such runs are cells of side 2^-20 (cut = 0) to 2^-13.3
// (cut = 20) of the root cube: they hold one particle almost always, a handful in the densest part of the largest
// systems.  The thread at the head of a run of up to kTieRun particles orders it by (low mid bits, lo word, load
// index) with an insertion sort over perm, sorted_pos and the key words; the start of a longer run is appended to a
// device list that k_sort_long_runs works off.
constexpr uint32_t kTieRun = 32;

__device__ __forceinline__ unsigned long long tie_key(uint32_t mid, uint32_t lo, uint32_t cut) {
    return ((unsigned long long)(mid & ((1u << cut) - 1u)) << 30) | lo;
}

__device__ __noinline__ void sort_tie_run(uint32_t i, uint32_t h, uint32_t m, uint32_t cut, const uint32_t* __restrict__ khi,
                                          uint32_t* __restrict__ kmid, uint32_t* __restrict__ klo,
                                          uint32_t* __restrict__ perm, float4* __restrict__ sorted_pos, uint32_t n,
                                          Control* __restrict__ ctl, uint32_t* __restrict__ long_start) {
    uint32_t len = 2;
    while (i + len < n && len <= kTieRun && khi[i + len] == h && (kmid[i + len] >> cut) == m) ++len;
    if (len > kTieRun) {
        long_start[atomicAdd(&ctl->n_long_runs, 1u)] = i;  // at most n / (kTieRun + 1) such runs
        return;
    }
    // (skipping the loads of perm / sorted_pos for particles that are already in place was measured: 45.6 against
    // 39.5 us at N = 2^22 -- the extra compare chain costs more than the loads it saves)
    for (uint32_t k = 1; k < len; ++k) {  // stable insertion sort: equal keys keep their ascending load index
        const uint32_t lo = klo[i + k], mk = kmid[i + k], pk = perm[i + k];
        const unsigned long long key = tie_key(mk, lo, cut);
        const float4 xk = sorted_pos[i + k];
        uint32_t j = k;
        while (j > 0 && tie_key(kmid[i + j - 1], klo[i + j - 1], cut) > key) {
            klo[i + j] = klo[i + j - 1];
            kmid[i + j] = kmid[i + j - 1];
            perm[i + j] = perm[i + j - 1];
            sorted_pos[i + j] = sorted_pos[i + j - 1];
            --j;
        }
        klo[i + j] = lo;
        kmid[i + j] = mk;
        perm[i + j] = pk;
        sorted_pos[i + j] = xk;
    }
}

// Four consecutive sorted particles per thread (16-byte loads of the hi and mid words plus one neighbour on each
// side); a particle that ties with its successor but not with its predecessor heads a run.
__global__ void __launch_bounds__(256) k_sort_ties(const uint32_t* __restrict__ khi, uint32_t* __restrict__ kmid,
                                                   uint32_t* __restrict__ klo, uint32_t* __restrict__ perm,
                                                   float4* __restrict__ sorted_pos, uint32_t n, Control* __restrict__ ctl,
                                                   uint32_t* __restrict__ long_start, const uint32_t cut, const Gate gate) {
    if (gate_closed(gate)) return;
    const uint32_t i0 = 4u * (blockIdx.x * blockDim.x + threadIdx.x);
    if (i0 >= n) return;
    uint32_t h[6], m[6];  // positions i0 - 1 .. i0 + 4; out-of-range slots get a value no key has
    if (i0 + 4 <= n) {
        // (plain loads: a neighbouring thread's repair may be rewriting mid words of ITS run, never of this thread's
        // leading bits -- a repair only permutes words whose leading bits are equal)
        const uint4 hv = __ldg(reinterpret_cast<const uint4*>(khi + i0)), mv = *reinterpret_cast<const uint4*>(kmid + i0);
        h[1] = hv.x; h[2] = hv.y; h[3] = hv.z; h[4] = hv.w;
        m[1] = mv.x; m[2] = mv.y; m[3] = mv.z; m[4] = mv.w;
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            h[1 + k] = (i0 + k < n) ? __ldg(&khi[i0 + k]) : 0xFFFFFFFFu;
            m[1 + k] = (i0 + k < n) ? kmid[i0 + k] : 0xFFFFFFFFu;
        }
    }
    h[0] = (i0 > 0) ? __ldg(&khi[i0 - 1]) : 0xFFFFFFFFu;
    m[0] = (i0 > 0) ? kmid[i0 - 1] : 0xFFFFFFFFu;
    h[5] = (i0 + 4 < n) ? __ldg(&khi[i0 + 4]) : 0xFFFFFFFFu;
    m[5] = (i0 + 4 < n) ? kmid[i0 + 4] : 0xFFFFFFFFu;
#pragma unroll
    for (int k = 0; k < 6; ++k) m[k] >>= cut;  // the leading bits the passes have sorted (0xFFFFFFFF >> cut: still no key)
#pragma unroll
    for (int k = 1; k <= 4; ++k) {
        if (h[k] == 0xFFFFFFFFu) break;  // past the end (key words have 30 bits)
        const bool ties_next = (h[k + 1] == h[k]) && (m[k + 1] == m[k]);
        const bool ties_prev = (h[k - 1] == h[k]) && (m[k - 1] == m[k]);
        if (ties_next && !ties_prev)
            sort_tie_run(i0 + k - 1, h[k], m[k], cut, khi, kmid, klo, perm, sorted_pos, n, ctl, long_start);
    }
}

// Long runs of equal leading bits: one WARP per run (runs are taken from the list by an atomic ticket) sorts the run
// by (low mid bits, lo word, position in the run) -- a stable LSD radix sort over the 30 + cut bits of that key in 8-bit
// digits.  Only the local indices move between passes (the digit of an element is read through its index from the
// run's own key words); one gather of perm, sorted_pos and the key words through the resulting order ends it.
// Positions in a run ascend with the load index (the passes are stable), so this is exactly the order (key, load index)
// of R5.  The launch returns at once when the list is empty (every Plummer / merger workload); a degenerate input --
// all particles coincident, or a clump far smaller than the cells the passes resolve -- costs this kernel a few
// milliseconds instead of costing every step more passes.
struct LongRunScratch {
    uint32_t *idx_a, *idx_b;  // [n] each, indexed by global position: runs are disjoint
    uint32_t *perm_tmp, *lo_tmp, *mid_tmp;
    float4* pos_tmp;
};

constexpr int kLongWarps = 4;

__global__ void __launch_bounds__(kLongWarps * 32) k_sort_long_runs(const uint32_t* __restrict__ khi,
                                                                    uint32_t* __restrict__ kmid,
                                                                    uint32_t* __restrict__ klo, uint32_t* __restrict__ perm,
                                                                    float4* __restrict__ sorted_pos, uint32_t n,
                                                                    Control* __restrict__ ctl,
                                                                    const uint32_t* __restrict__ long_start,
                                                                    LongRunScratch sc, const uint32_t cut, const Gate gate) {
    __shared__ uint32_t s_hist[kLongWarps][256];
    if (gate_closed(gate)) return;
    const uint32_t n_runs = __ldcg(&ctl->n_long_runs);
    if (n_runs == 0u) return;
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t lt = (1u << l) - 1u;
    uint32_t* hist = s_hist[w];
    for (;;) {
        uint32_t r = 0;
        if (l == 0) r = atomicAdd(&ctl->long_ticket, 1u);
        r = __shfl_sync(0xFFFFFFFFu, r, 0);
        if (r >= n_runs) break;
        const uint32_t s0 = __ldcg(&long_start[r]);
        const uint32_t h = khi[s0], m = kmid[s0] >> cut;
        // length of the run: first position that leaves it
        uint32_t len = 0;
        for (uint32_t base = s0;; base += 32u) {
            const uint32_t i = base + l;
            const bool in = i < n && khi[i] == h && (kmid[i] >> cut) == m;
            const uint32_t out = ~__ballot_sync(0xFFFFFFFFu, in);
            if (out) { len = base - s0 + (uint32_t)(__ffs(out) - 1); break; }
        }
        uint32_t *ia = sc.idx_a + s0, *ib = sc.idx_b + s0;
        for (uint32_t k = l; k < len; k += 32u) ia[k] = k;
        __syncwarp();
        for (uint32_t shift = 0; shift < 30u + cut; shift += 8u) {
            for (int d = l; d < 256; d += 32) hist[d] = 0u;
            __syncwarp();
            for (uint32_t k = l; k < len; k += 32u)
                atomicAdd(&hist[(uint32_t)(tie_key(kmid[s0 + k], klo[s0 + k], cut) >> shift) & 255u], 1u);
            __syncwarp();
            // exclusive scan of the 256 counts: 8 per lane, then across lanes
            uint32_t v[8], sum = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) { v[q] = hist[8 * l + q]; sum += v[q]; }
            uint32_t incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                if (l >= o) incl += y;
            }
            uint32_t run = incl - sum;
#pragma unroll
            for (int q = 0; q < 8; ++q) { hist[8 * l + q] = run; run += v[q]; }
            __syncwarp();
            // stable scatter, 32 elements at a time in order: equal digits keep their order (lane order inside a
            // chunk, chunk order through the running offsets)
            for (uint32_t base = 0; base < len; base += 32u) {
                const uint32_t k = base + l;
                const bool valid = k < len;
                const uint32_t e = valid ? ia[k] : 0u;
                const uint32_t d = valid ? ((uint32_t)(tie_key(kmid[s0 + e], klo[s0 + e], cut) >> shift) & 255u)
                                         : 256u + (uint32_t)l;  // invalid lanes match nobody
                const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
                uint32_t off = 0;
                if (valid) off = hist[d];
                __syncwarp();
                if (valid) {
                    ib[off + (uint32_t)__popc(peers & lt)] = e;
                    if ((peers >> l) <= 1u) hist[d] = off + (uint32_t)__popc(peers);  // the highest peer advances the offset
                }
                __syncwarp();
            }
            uint32_t* t = ia; ia = ib; ib = t;
            __threadfence_block();
            __syncwarp();
        }
        // ia[k] = position (in the run) of the particle that belongs at k
        for (uint32_t k = l; k < len; k += 32u) {
            sc.perm_tmp[s0 + k] = perm[s0 + k];
            sc.lo_tmp[s0 + k] = klo[s0 + k];
            sc.mid_tmp[s0 + k] = kmid[s0 + k];
            sc.pos_tmp[s0 + k] = sorted_pos[s0 + k];
        }
        __threadfence_block();
        __syncwarp();
        for (uint32_t k = l; k < len; k += 32u) {
            const uint32_t src = s0 + ia[k];
            perm[s0 + k] = sc.perm_tmp[src];
            klo[s0 + k] = sc.lo_tmp[src];
            kmid[s0 + k] = sc.mid_tmp[src];
            sorted_pos[s0 + k] = sc.pos_tmp[src];
        }
        __syncwarp();
    }
    // the last warp to leave resets the ticket for the next build (n_long_runs is reset by k_sort_gscan)
    if (l == 0) {
        __threadfence();
        if (atomicAdd(&ctl->long_done, 1u) == gridDim.x * kLongWarps - 1u) {
            ctl->long_done = 0u;
            ctl->long_ticket = 0u;
        }
    }
}

constexpr size_t kSortSmem = sizeof(uint32_t) * ((kSortThreads / 32) * kRadix + 2 * kRadix);

// per device, at context creation (see walk_prepare)
cudaError_t sort_prepare(Ctx* c) {
    (void)c;
    cudaError_t e = cudaFuncSetAttribute(k_sort_pass<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSortSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sort_pass<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSortSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sort_pass<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSortSmem);
    return e;
}

// How many of the six passes run.  The passes go over the mid word's three digits, then the hi word's; leaving out the
// first one or two leaves particles that agree in the leading 50 or 40 key bits (cells of side 2^-16.7 / 2^-13.3 of the
// root cube) in load order, and the tie repair after the reorder (k_sort_ties, k_sort_long_runs) puts exactly those
// runs in order of their remaining bits -- the result is the same permutation bit for bit, whatever the choice.  What it
// costs is the repair: measured on the Plummer sphere, 40 leading bits leave 0.3 % of the particles in runs (of 2) at
// N = 2^15 and 17 % (runs of <= 8) at N = 2^22; 50 bits leave 0.02 % at 2^22.  The rule below keeps the expected run of
// a Plummer core short; params.sort_passes overrides it (a strongly clustered system wants more passes).
int sort_first_pass(const Ctx* c) {
    if (c->prm.sort_passes) return kSortPasses - (int)c->prm.sort_passes;
    if (c->n <= (1u << 23)) return 2;  // measured, sort + repair: 0.681 (4) against 0.698 ms (5) at 2^23, 1.451 against 1.375 at 2^24
    if (c->n <= (1u << 25)) return 1;
    return 0;
}

// The sort: LSD passes over the mid and hi words (pass p: word mid, hi = p / 3; digit p % 3), starting from the identity
// permutation at pass sort_first_pass(); the starting pair buffer is chosen so that the permutation ends in idx[0].
cudaError_t stage_sort(Ctx* c) {
    Buffers& b = c->b;
    const size_t look_entries = (size_t)div_up(c->n_max, kSortTile) * kRadix;
    k_sort_gscan<<<kSortPasses, kRadix, 0, c->stream>>>(b.ghist, b.ctl, b.look, look_entries, c->gate);
    c->launches += 1;
    c->perm = b.idx[0];
    SortPass a;
    a.n = c->n;
    a.n_tiles = div_up(c->n, kSortTile);
    a.look = b.look;
    a.ticket = &b.ctl->sort_ticket;
    a.ctl = b.ctl;
    a.gate = c->gate;
    const int first = sort_first_pass(c);
    int cur = first & 1;
    for (int p = first; p < kSortPasses; ++p) {
        a.pass = (uint32_t)p;
        a.shift = kRadixBits * (p % 3);
        a.gbase = b.ghist + p * kRadix;
        a.src_word = b.key[0][1 - p / 3];  // load-order word of this phase: mid, then hi
        const int out = cur ^ 1;
        a.key_in = b.pair_key[cur];
        a.idx_in = b.idx[cur];
        a.key_out = (p == kSortPasses - 1) ? nullptr : b.pair_key[out];
        a.idx_out = b.idx[out];
        if (p == first) k_sort_pass<0><<<a.n_tiles, kSortThreads, kSortSmem, c->stream>>>(a);
        else if (p % 3 == 0) k_sort_pass<2><<<a.n_tiles, kSortThreads, kSortSmem, c->stream>>>(a);
        else k_sort_pass<1><<<a.n_tiles, kSortThreads, kSortSmem, c->stream>>>(a);
        c->launches += 1;
        cur = out;
    }
    return (cur == 0) ? cudaGetLastError() : cudaErrorUnknown;
}

cudaError_t stage_reorder(Ctx* c, bool write_keys) {
    Buffers& b = c->b;
    k_reorder<<<div_up(c->n, 256), 256, 0, c->stream>>>(c->pos_mass, c->perm, c->n, b.ctl, b.sorted_pos,
                                                        write_keys ? b.key[1][0] : nullptr, b.key[1][1], b.key[1][2], c->gate);
    c->launches += 1;
    c->sorted_buf = 1;
    return cudaGetLastError();
}

// After the reorder of a fresh sort: put the runs of equal leading key bits in order of their remaining bits -- short
// runs in place, long ones (coincident particles, clumps far smaller than the cells the passes resolve) by
// k_sort_long_runs, which returns at once when there are none.  Scratch of the long-run sort: the pair buffers and the
// load-order key words (dead after the passes) and tie_pos, an n-sized array of its own (the cell arrays are sized by
// cap_cells, which the caller may set far below n).
cudaError_t stage_sort_ties(Ctx* c) {
    Buffers& b = c->b;
    const uint32_t cut = (uint32_t)(kRadixBits * sort_first_pass(c));  // low bits of the mid word the passes skipped
    k_sort_ties<<<div_up(div_up(c->n, 4), 256), 256, 0, c->stream>>>(b.key[1][0], b.key[1][1], b.key[1][2], c->perm, b.sorted_pos, c->n,
                                                          b.ctl, b.long_start, cut, c->gate);
    LongRunScratch sc{b.pair_key[0], b.idx[1], b.key[0][0], b.key[0][1], b.key[0][2], b.tie_pos};
    k_sort_long_runs<<<c->num_sms, kLongWarps * 32, 0, c->stream>>>(b.key[1][0], b.key[1][1], b.key[1][2], c->perm, b.sorted_pos, c->n,
                                                                 b.ctl, b.long_start, sc, cut, c->gate);
    c->launches += 2;
    return cudaGetLastError();
}

}  // namespace bonsai
