// Stage a4: octree construction from the sorted Morton keys ("construction of the
// tree-datastructure"; P:L22 fn.1 "we use an octree data-structure"; reading R7 of DESIGN.md).
//
// The paper-era design builds the tree level by level (one pass over the keys per level).  Here the
// whole tree comes out of ONE pass over a 1-byte-per-particle array, in four launches, because every
// property of the canonical tree is a local function of the sorted keys:
//
//   lcp[i]        = number of leading octal digits shared by key[i-1] and key[i]  (-1 at i = 0 and i = n).
//                   The level-L cell containing particle i is the maximal run around i with lcp < L ... >= L
//                   inside, i.e. it starts at the last boundary b <= i with lcp[b] < L.
//   leaf_level[i] = the level of the leaf holding particle i = the smallest L whose level-L run around i has
//                   <= nleaf particles (capped at 30).  Because nleaf <= 64 this only needs lcp within
//                   +-nleaf of i:  leaf_level = 1 + min over boundaries b <= i < e, e - b <= nleaf, of
//                   max(lcp[b], lcp[e]).
//   A level-L cell starts at boundary b  <=>  lcp[b] < L <= leaf_level[b];  it ends at boundary e  <=>
//   lcp[e] < L <= leaf_level[e-1].  Breadth-first numbering = level offset + rank of the start among the
//   level-L starts, so ids come from one per-level count/scan over blocks and warp ballots inside a block.
//
// Launches: k_tree_levels (lcp + leaf levels + per-block per-level start counts),
// k_tree_scan_levels (prefix over blocks per level, level offsets, n_cells), k_tree_emit (cell records),
// k_tree_finalize (count = end - first, n_child = last_child - first_child + 1).
#include "internal.cuh"

namespace bonsai {

__device__ __forceinline__ int common_digits(uint32_t ahi, uint32_t amid, uint32_t alo, uint32_t bhi, uint32_t bmid,
                                             uint32_t blo) {
    uint32_t x = ahi ^ bhi;  // 30-bit words: the most significant digit sits in bits 29..27
    if (x) return (__clz(x) - 2) / 3;
    x = amid ^ bmid;
    if (x) return 10 + (__clz(x) - 2) / 3;
    x = alo ^ blo;
    if (x) return 20 + (__clz(x) - 2) / 3;
    return 30;
}

// bits (lo_excl, hi_incl] of a 31-bit level mask; lo_excl may be -1
__device__ __forceinline__ uint32_t level_range_mask(int lo_excl, int hi_incl) {
    if (hi_incl <= lo_excl) return 0u;
    uint32_t hi = (2u << hi_incl) - 1u;
    uint32_t lo = (lo_excl < 0) ? 0u : ((2u << lo_excl) - 1u);
    return hi & ~lo;
}

// Boundary handled by (warp w, round r, lane l) of a block: consecutive lanes = consecutive boundaries.
__device__ __forceinline__ uint32_t tree_item(uint32_t block, int w, int r, int l) {
    return block * kTreeTile + w * (32 * kTreeItems) + r * 32 + l;
}

// lcp[] is computed here, from the sorted keys, for the block's span plus a halo of kMaxNleaf boundaries on each
// side (the keys are read once more per halo -- 12 % more than a separate lcp pass, which this saves), and stored for
// k_tree_emit.
__global__ void __launch_bounds__(kTreeThreads) k_tree_levels(const uint32_t* __restrict__ khi,
                                                              const uint32_t* __restrict__ kmid,
                                                              const uint32_t* __restrict__ klo, uint32_t n, int nleaf,
                                                              uint32_t n_blocks, int8_t* __restrict__ lcp,
                                                              int8_t* __restrict__ leaf_level,
                                                              uint32_t* __restrict__ blk_level_count, const Gate gate) {
    constexpr int H = kMaxNleaf;
    if (gate_closed(gate)) return;
    __shared__ int8_t s_lcp[kTreeTile + 2 * H + 1];
    __shared__ uint32_t s_cnt[kLevelSlots];
    const long long base = (long long)blockIdx.x * kTreeTile;
    for (int j = threadIdx.x; j < kTreeTile + 2 * H + 1; j += kTreeThreads) {
        const long long b = base - H + j;
        int v = -1;  // boundaries 0 and n, and everything outside [0, n]
        if (b > 0 && b < (long long)n)
            v = common_digits(__ldg(&khi[b - 1]), __ldg(&kmid[b - 1]), __ldg(&klo[b - 1]), __ldg(&khi[b]), __ldg(&kmid[b]),
                              __ldg(&klo[b]));
        s_lcp[j] = (int8_t)v;
        if (j >= H && j < H + kTreeTile && b <= (long long)n) lcp[b] = (int8_t)v;  // this block's own boundaries
    }
    if (threadIdx.x < kLevelSlots) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < kTreeItems; ++r) {
        const uint32_t i = tree_item(blockIdx.x, w, r, l);
        uint32_t mask = 0;
        if (i < n) {
            const int j = (int)(i - base) + H;  // s_lcp index of boundary i
            // candidate start b = i - nleaf + 1 + t, candidate ends (i, b + nleaf].  No range checks: boundaries outside
            // [0, n] read -1 like boundaries 0 and n themselves, so an end past n repeats what the end n already
            // contributed, and a start before 0 sees fewer ends than the start 0 that is then a candidate too.
            int best = 127, rmin = 127;
            const int8_t* lo_side = &s_lcp[j - nleaf + 1];
            const int8_t* hi_side = &s_lcp[j + 1];
#pragma unroll 8
            for (int t = 0; t < nleaf; ++t) {
                rmin = min(rmin, (int)hi_side[t]);
                best = min(best, max((int)lo_side[t], rmin));
            }
            const int ll = min(best + 1, kMaxLevel);
            leaf_level[i] = (int8_t)ll;
            mask = level_range_mask((int)s_lcp[j], ll);
        }
        uint32_t orm = __reduce_or_sync(0xFFFFFFFFu, mask);
        while (orm) {
            const int L = __ffs(orm) - 1;
            orm &= orm - 1;
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, (mask >> L) & 1u);
            if (l == 0) atomicAdd(&s_cnt[L], (uint32_t)__popc(b));
        }
    }
    __syncthreads();
    if (threadIdx.x < kLevelSlots) blk_level_count[(size_t)threadIdx.x * n_blocks + blockIdx.x] = s_cnt[threadIdx.x];
}

// One block per level: exclusive prefix over blocks in place; the last block to finish turns the level totals
// into level offsets and n_cells.
constexpr int kScanLvThreads = 1024;

__global__ void __launch_bounds__(kScanLvThreads) k_tree_scan_levels(uint32_t* __restrict__ blk_level_count, uint32_t n_blocks,
                                                                     uint32_t* __restrict__ level_total,
                                                                     Control* __restrict__ ctl, uint32_t cap_cells,
                                                                     const Gate gate) {
    __shared__ uint32_t wsum[kScanLvThreads / 32];
    __shared__ uint32_t carry;
    __shared__ bool s_last;
    if (gate_closed(gate)) return;
    uint32_t* row = blk_level_count + (size_t)blockIdx.x * n_blocks;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (uint32_t t0 = 0; t0 < n_blocks; t0 += kScanLvThreads) {
        const uint32_t t = t0 + threadIdx.x;
        const uint32_t v = (t < n_blocks) ? row[t] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
            if (l >= o) x += y;
        }
        if (l == 31) wsum[w] = x;
        __syncthreads();
        if (w == 0) {  // exclusive scan of the 32 warp totals
            const uint32_t tw = wsum[l];
            uint32_t y = tw;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t z = __shfl_up_sync(0xFFFFFFFFu, y, o);
                if (l >= o) y += z;
            }
            wsum[l] = y - tw;
        }
        __syncthreads();
        const uint32_t pre = carry + wsum[w];
        if (t < n_blocks) row[t] = pre + x - v;
        __syncthreads();
        if (threadIdx.x == kScanLvThreads - 1) carry = pre + x;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        level_total[blockIdx.x] = carry;
        __threadfence();
        s_last = (atomicAdd(&ctl->level_ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last || threadIdx.x != 0) return;
    __threadfence();
    uint32_t off = 0;
    for (int L = 0; L <= kMaxLevel; ++L) {
        ctl->level_offsets[L] = off;
        off += __ldcg(&level_total[L]);
    }
    ctl->level_offsets[kMaxLevel + 1] = off;
    ctl->n_cells = off;
    if (off > cap_cells) ctl->status = BONSAI_ECAPACITY;
    ctl->level_ticket = 0;
}

struct CellArrays {
    uint32_t *level, *first, *count, *first_child, *n_child, *parent;
};

// Cell records.  Every boundary i in [0, n] is handled by one thread: it STARTS the cells of levels
// (lcp[i], leaf_level[i]] and ENDS the cells of levels (lcp[i], leaf_level[i-1]].  The absolute id of a level-L
// start is  level_offsets[L] + (level-L starts in earlier blocks) + (rank inside the block).
// count[] receives the END boundary and n_child[] the LAST child id; k_tree_finalize turns them into counts.
__global__ void __launch_bounds__(kTreeThreads) k_tree_emit(const int8_t* __restrict__ lcp,
                                                            const int8_t* __restrict__ leaf_level, uint32_t n,
                                                            uint32_t n_blocks,
                                                            const uint32_t* __restrict__ blk_level_prefix,
                                                            const Control* __restrict__ ctl, uint32_t cap_cells,
                                                            CellArrays ca, const Gate gate) {
    constexpr int kWarps = kTreeThreads / 32;
    if (gate_closed(gate)) return;
    __shared__ uint32_t s_pre[kWarps][kTreeItems][kLevelSlots];
    for (int k = threadIdx.x; k < kWarps * kTreeItems * kLevelSlots; k += kTreeThreads) (&s_pre[0][0][0])[k] = 0;
    __syncthreads();
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t lt = (1u << l) - 1u;
    uint32_t smask[kTreeItems], emask[kTreeItems];
    int8_t ll_here[kTreeItems], ll_before[kTreeItems];
#pragma unroll
    for (int r = 0; r < kTreeItems; ++r) {
        const uint32_t i = tree_item(blockIdx.x, w, r, l);
        smask[r] = emask[r] = 0;
        ll_here[r] = ll_before[r] = -1;
        if (i <= n) {
            const int c = lcp[i];
            if (i < n) ll_here[r] = leaf_level[i];
            if (i > 0) ll_before[r] = leaf_level[i - 1];
            smask[r] = level_range_mask(c, ll_here[r]);
            emask[r] = level_range_mask(c, ll_before[r]);
        }
        uint32_t orm = __reduce_or_sync(0xFFFFFFFFu, smask[r]);
        while (orm) {
            const int L = __ffs(orm) - 1;
            orm &= orm - 1;
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, (smask[r] >> L) & 1u);
            if (l == 0) s_pre[w][r][L] = __popc(b);
        }
    }
    __syncthreads();
    if (threadIdx.x <= kMaxLevel) {  // one thread per level: exclusive prefix in (warp, round) order + absolute base
        const int L = threadIdx.x;
        uint32_t run = ctl->level_offsets[L] + blk_level_prefix[(size_t)L * n_blocks + blockIdx.x];
        for (int k = 0; k < kWarps * kTreeItems; ++k) {
            uint32_t t = s_pre[k / kTreeItems][k % kTreeItems][L];
            s_pre[k / kTreeItems][k % kTreeItems][L] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kTreeItems; ++r) {
        const uint32_t i = tree_item(blockIdx.x, w, r, l);
        const uint32_t sm = smask[r], em = emask[r];
        const uint32_t allm = __reduce_or_sync(0xFFFFFFFFu, sm | em);
        if (allm == 0) continue;
        const int Lmin = __ffs(allm) - 1, Lmax = 31 - __clz(allm);
        const int L0 = max(Lmin - 1, 0);
        uint32_t rk_prev = 0;
        uint32_t rk_cur = s_pre[w][r][L0] + __popc(__ballot_sync(0xFFFFFFFFu, (sm >> L0) & 1u) & lt);
        for (int L = L0; L <= Lmax; ++L) {
            uint32_t rk_next = 0;
            if (L < kMaxLevel)
                rk_next = s_pre[w][r][L + 1] + __popc(__ballot_sync(0xFFFFFFFFu, (sm >> (L + 1)) & 1u) & lt);
            if ((sm >> L) & 1u) {  // a level-L cell starts here
                const uint32_t id = rk_cur;
                if (id < cap_cells) {
                    ca.level[id] = (uint32_t)L;
                    ca.first[id] = i;
                    ca.parent[id] = (L == 0) ? kNone : (rk_prev - (((sm >> (L - 1)) & 1u) ? 0u : 1u));
                    if (L == ll_here[r]) {
                        ca.first_child[id] = 0;
                        ca.n_child[id] = 0;
                    } else {
                        ca.first_child[id] = rk_next;  // the level-(L+1) cell starting at this same boundary
                    }
                }
            }
            if ((em >> L) & 1u) {  // the level-L cell holding particle i-1 ends here
                const uint32_t id = rk_cur - 1u;
                if (id < cap_cells) {
                    ca.count[id] = i;
                    if (L < ll_before[r]) ca.n_child[id] = rk_next - 1u;
                }
            }
            rk_prev = rk_cur;
            rk_cur = rk_next;
        }
    }
}

__global__ void __launch_bounds__(256) k_tree_finalize(const Control* __restrict__ ctl, uint32_t cap_cells,
                                                       CellArrays ca, const Gate gate) {
    if (gate_closed(gate)) return;
    // grid-stride: the number of cells is only known on the device, a grid sized for cap_cells would be mostly empty
    const uint32_t n_cells = min(ctl->n_cells, cap_cells);
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cells; c += gridDim.x * blockDim.x) {
        ca.count[c] = ca.count[c] - ca.first[c];
        const uint32_t fc = ca.first_child[c];
        if (fc != 0) ca.n_child[c] = ca.n_child[c] - fc + 1u;
    }
}

cudaError_t stage_build(Ctx* c) {
    const uint32_t n = c->n;
    Buffers& b = c->b;
    const int s = c->sorted_buf;
    const uint32_t n_blocks = div_up(n + 1, kTreeTile);
    CellArrays ca{b.c_level, b.c_first, b.c_count, b.c_first_child, b.c_n_child, b.c_parent};
    k_tree_levels<<<n_blocks, kTreeThreads, 0, c->stream>>>(b.key[s][0], b.key[s][1], b.key[s][2], n, (int)c->prm.nleaf, n_blocks,
                                                            b.lcp, b.leaf_level, b.blk_level_count, c->gate);
    k_tree_scan_levels<<<kMaxLevel + 1, kScanLvThreads, 0, c->stream>>>(b.blk_level_count, n_blocks, b.level_total, b.ctl,
                                                             c->cap_cells, c->gate);
    k_tree_emit<<<n_blocks, kTreeThreads, 0, c->stream>>>(b.lcp, b.leaf_level, n, n_blocks, b.blk_level_count, b.ctl,
                                                          c->cap_cells, ca, c->gate);
    k_tree_finalize<<<min(div_up(c->cap_cells, 256), (uint32_t)c->num_sms * 16u), 256, 0, c->stream>>>(b.ctl, c->cap_cells, ca, c->gate);
    c->launches += 4;
    return cudaGetLastError();
}

}  // namespace bonsai
