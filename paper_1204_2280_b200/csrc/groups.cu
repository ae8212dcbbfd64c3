// Stage a4': walk groups (the traversal follows "the method used for tree-traversion on vector
// machines (Barnes 1990)" -- one shared traversal per group of neighbouring particles; readings R13, R19).
//
//   rank[i]        exclusive count of ACTIVE particles among sorted particles 0..i-1  (rank[n] = n_active)
//   active_list[k] sorted index of the k-th active particle
//                  (all particles active: both are the identity and are NOT materialised -- the kernels below and the
//                  walk take a null pointer to mean rank[i] = i, active_list[k] = k; bonsai_get_groups fills
//                  active_list on demand)
//   mode 1 (sorted chunks): group g = active particles [g ncrit, min((g+1) ncrit, n_active))
//   mode 0 (tree cells):    the cells with count <= ncrit (or childless) whose parent has count > ncrit, in key
//                           order, each keeping only its active members, dropped when none remain
//   mode 2 (cell chunks):   the active members of every container cell (count <= group_cell or childless, parent
//                           count > group_cell) are cut into consecutive runs of ncrit: no group straddles the
//                           boundary of a big cell, which bounds the most expensive group
//   bmin / bmax            exact fp32 per-axis min / max over the group's members
#include "internal.cuh"

namespace bonsai {

// introspection only (bonsai_get_groups after an all-active build)
__global__ void __launch_bounds__(256) k_groups_identity(uint32_t n, uint32_t* __restrict__ active_list) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) active_list[i] = i;
}

__device__ __forceinline__ uint32_t rank_at(const uint32_t* __restrict__ rank, uint32_t i) { return rank ? rank[i] : i; }

// flags in sorted order from a mask in load order
__global__ void __launch_bounds__(256) k_groups_flags(const uint8_t* __restrict__ mask, const uint32_t* __restrict__ perm,
                                                      uint32_t n, uint32_t* __restrict__ flag) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = mask[__ldg(&perm[i])] ? 1u : 0u;
}

__global__ void __launch_bounds__(256) k_groups_compact(const uint32_t* __restrict__ rank, uint32_t n,
                                                        uint32_t* __restrict__ active_list) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const uint32_t r = rank[i];
        if (rank[i + 1] != r) active_list[r] = i;
    }
}

// mode 1: first / count of every chunk
__global__ void __launch_bounds__(256) k_groups_chunks(const uint32_t* __restrict__ rank, uint32_t n, uint32_t ncrit,
                                                       uint32_t* __restrict__ g_first, uint32_t* __restrict__ g_count,
                                                       Control* __restrict__ ctl) {
    const uint32_t na = rank_at(rank, n);
    const uint32_t ng = (na + ncrit - 1) / ncrit;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g == 0) {
        ctl->n_groups = ng;
        ctl->n_active = na;
    }
    if (g >= ng) return;
    g_first[g] = g * ncrit;
    g_count[g] = min(ncrit, na - g * ncrit);
}

// mode 0, step 1: mark the first particle of every non-empty group cell
__global__ void __launch_bounds__(256) k_groups_mark(const Control* __restrict__ ctl, uint32_t cap_cells, uint32_t limit,
                                                     uint32_t chunk,
                                                     const uint32_t* __restrict__ c_first,
                                                     const uint32_t* __restrict__ c_count,
                                                     const uint32_t* __restrict__ c_n_child,
                                                     const uint32_t* __restrict__ c_parent,
                                                     const uint32_t* __restrict__ rank, uint32_t* __restrict__ g_flag,
                                                     uint32_t* __restrict__ g_cell) {
    // grid-stride: the number of cells is only known on the device
    const uint32_t n_cells = min(ctl->n_cells, cap_cells);
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cells; c += gridDim.x * blockDim.x) {
        const uint32_t cnt = c_count[c];
        if (!(cnt <= limit || c_n_child[c] == 0)) continue;
        const uint32_t p = c_parent[c];
        if (p != kNone && c_count[p] <= limit) continue;  // an ancestor already is the group / container
        const uint32_t f = c_first[c];
        const uint32_t a = rank_at(rank, f + cnt) - rank_at(rank, f);
        if (a == 0) continue;                              // no active member
        g_flag[f] = chunk ? (a + chunk - 1u) / chunk : 1u;  // number of groups this cell contributes
        g_cell[f] = c + 1u;
    }
}

// mode 0, step 2 (after the scan of g_flag): first / count of every group
__global__ void __launch_bounds__(256) k_groups_cells(const uint32_t* __restrict__ g_index,
                                                      const uint32_t* __restrict__ g_cell, uint32_t n,
                                                      const uint32_t* __restrict__ c_count,
                                                      const uint32_t* __restrict__ rank, uint32_t chunk,
                                                      uint32_t* __restrict__ g_first, uint32_t* __restrict__ g_count,
                                                      Control* __restrict__ ctl) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        ctl->n_groups = g_index[n];
        ctl->n_active = rank_at(rank, n);
    }
    if (i >= n) return;
    const uint32_t c1 = g_cell[i];
    if (c1 == 0) return;
    const uint32_t g = g_index[i];
    const uint32_t r0 = rank_at(rank, i);
    const uint32_t a = rank_at(rank, i + c_count[c1 - 1]) - r0;
    if (chunk == 0u) {
        g_first[g] = r0;
        g_count[g] = a;
    } else {
        uint32_t k = 0;
        for (uint32_t o = 0; o < a; o += chunk, ++k) {
            g_first[g + k] = r0 + o;
            g_count[g + k] = min(chunk, a - o);
        }
    }
}

// one warp per group (grid-stride): exact fp32 box
__global__ void __launch_bounds__(256) k_groups_box(const Control* __restrict__ ctl, const uint32_t* __restrict__ g_first,
                                                    const uint32_t* __restrict__ g_count,
                                                    const uint32_t* __restrict__ active_list,
                                                    const float4* __restrict__ sorted_pos, float* __restrict__ g_bmin,
                                                    float* __restrict__ g_bmax) {
    const uint32_t ng = ctl->n_groups;
    const int l = threadIdx.x & 31;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; g < ng; g += warps) {
        const uint32_t f = g_first[g], cnt = g_count[g];
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        for (uint32_t k = l; k < cnt; k += 32) {
            const float4 p = __ldg(&sorted_pos[active_list ? __ldg(&active_list[f + k]) : f + k]);
            mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
            mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
            mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xFFFFFFFFu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xFFFFFFFFu, mx[a], o));
            }
        if (l < 3) {
            g_bmin[3 * g + l] = (l == 0) ? mn[0] : (l == 1) ? mn[1] : mn[2];
            g_bmax[3 * g + l] = (l == 0) ? mx[0] : (l == 1) ? mx[1] : mx[2];
        }
    }
}

cudaError_t stage_groups(Ctx* c, const uint8_t* mask_load_order) {
    const uint32_t n = c->n;
    Buffers& b = c->b;
    cudaError_t e;
    const uint32_t* rank = (mask_load_order == nullptr) ? nullptr : b.rank;  // nullptr = identity (see the header)
    const uint32_t* active_list = (mask_load_order == nullptr) ? nullptr : b.active_list;
    if (mask_load_order != nullptr) {
        k_groups_flags<<<div_up(n, 256), 256, 0, c->stream>>>(mask_load_order, c->perm, n, b.rank);
        c->launches += 1;
        if ((e = exclusive_scan_u32(c, b.rank, b.rank, n, b.scan_tmp)) != cudaSuccess) return e;
        k_groups_compact<<<div_up(n, 256), 256, 0, c->stream>>>(b.rank, n, b.active_list);
        c->launches += 1;
    }
    if (c->prm.group_mode == 1) {
        k_groups_chunks<<<div_up(div_up(n, c->prm.ncrit), 256), 256, 0, c->stream>>>(rank, n, c->prm.ncrit, b.g_first,
                                                                                   b.g_count, b.ctl);
        c->launches += 1;
    } else {
        if ((e = cudaMemsetAsync(b.g_flag, 0, sizeof(uint32_t) * (size_t)(n + 1), c->stream)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(b.g_cell, 0, sizeof(uint32_t) * (size_t)n, c->stream)) != cudaSuccess) return e;
        const bool cells = (c->prm.group_mode == 0);
        const uint32_t limit = cells ? c->prm.ncrit : c->prm.group_cell;
        const uint32_t chunk = cells ? 0u : c->prm.ncrit;
        k_groups_mark<<<min(div_up(c->cap_cells, 256), (uint32_t)c->num_sms * 16u), 256, 0, c->stream>>>(b.ctl, c->cap_cells, limit, chunk, b.c_first,
                                                                        b.c_count, b.c_n_child, b.c_parent, rank,
                                                                        b.g_flag, b.g_cell);
        c->launches += 1;
        if ((e = exclusive_scan_u32(c, b.g_flag, b.g_flag, n, b.scan_tmp)) != cudaSuccess) return e;
        k_groups_cells<<<div_up(n, 256), 256, 0, c->stream>>>(b.g_flag, b.g_cell, n, b.c_count, rank, chunk,
                                                              b.g_first, b.g_count, b.ctl);
        c->launches += 1;
    }
    k_groups_box<<<c->num_sms * 8, 256, 0, c->stream>>>(b.ctl, b.g_first, b.g_count, active_list, b.sorted_pos,
                                                        b.g_bmin, b.g_bmax);
    c->launches += 1;
    c->groups_all_active = (mask_load_order == nullptr);
    return cudaGetLastError();
}

// bonsai_get_groups after an all-active build: materialise the identity list the getter hands out
cudaError_t groups_fill_identity(Ctx* c) {
    k_groups_identity<<<div_up(c->n, 256), 256, 0, c->stream>>>(c->n, c->b.active_list);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace bonsai
