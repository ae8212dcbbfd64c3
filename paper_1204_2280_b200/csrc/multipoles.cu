// Stage a5: multipole moments ("computation of the tree-properties (multipole moments)", P:L30;
// BASELINE.json north_star: monopole + quadrupole; reading R8 of DESIGN.md).
//
// Per cell: M, centre of mass, the 6 raw second moments about the centre of mass, delta = |COM - geometric
// centre| and the geometric side l.  Everything is accumulated in fp64 and rounded ONCE to fp32, because the
// fp32 opening test of the walk must see the same COM / delta as the reference to the last bit (R9).
//
// One launch, bottom-up without level barriers: a lane per cell, tiles of 32 cells handed out deepest-first; leaves sum
// their particles (in particle order, without FMA contraction), internal cells wait until their children have
// published and combine the children's fp64 moments (parallel-axis shift about the parent's COM; moments about
// the origin would cancel catastrophically in the halo).  See k_multipoles for the scheduling argument.
// The exact fp32 bounding box of every cell's members rides along; a refreshed tree (R25) uses it to let l
// grow when particles have drifted out of their cell.
#include "internal.cuh"

namespace bonsai {

__device__ __forceinline__ uint32_t compact10(uint32_t v) {  // every third bit of 30 -> 10 bits
    v &= 0x09249249u;
    v = (v | (v >> 2)) & 0x030C30C3u;
    v = (v | (v >> 4)) & 0x0300F00Fu;
    v = (v | (v >> 8)) & 0x030000FFu;
    v = (v | (v >> 16)) & 0x3FFu;
    return v;
}

struct Mom {
    double m, cx, cy, cz, xx, yy, zz, xy, xz, yz;
};

// kBox: the exact fp32 bounding box of the cell's members is available (mn, mx) and is stored for the parent;
// kTight: R28 -- the side and centre that enter the opening test are those of that box (mac_mode = 1); otherwise, with
// kBox alone, R25 -- a refreshed tree lets the geometric side grow to contain the members.
template <bool kBox, bool kTight>
__device__ __forceinline__ void store_cell(const Mom& q, const float (&mn)[3], const float (&mx)[3],
                                           uint32_t c, int L, uint32_t khi, uint32_t kmid, uint32_t klo,
                                           const Control* __restrict__ ctl, uint32_t link_first, uint32_t link_info,
                                           double* __restrict__ c_mom, float* __restrict__ c_box,
                                           CellMac* __restrict__ c_mac, CellQuad* __restrict__ c_quad,
                                           float* __restrict__ c_qraw, const bool grow) {
    // geometric centre: integer cell coordinate = top L bits of the quantised coordinate of any member (R8)
    double l = ldexp(ctl->side, -L);
    double g[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int sh = 2 - a;
        const uint32_t qa = (compact10(khi >> sh) << 20) | (compact10(kmid >> sh) << 10) | compact10(klo >> sh);
        const uint32_t ca = (L == 0) ? 0u : (qa >> (kMaxLevel - L));
        g[a] = __dadd_rn((double)ctl->lo[a], __dmul_rn(__dadd_rn((double)ca, 0.5), l));
    }
    if (kBox) {
        float2* bx = reinterpret_cast<float2*>(c_box + (size_t)c * 6);  // only refreshed trees and the tight MAC need the boxes
        __stcg(&bx[0], make_float2(mn[0], mn[1]));
        __stcg(&bx[1], make_float2(mn[2], mx[0]));
        __stcg(&bx[2], make_float2(mx[1], mx[2]));
        // R25 (refreshed tree): the side becomes the side of the smallest cube about the geometric centre that
        // holds every member, never less than the geometric side: l = max(l, 2 max_axis max(g - min, max - g)), fp64
        if (kTight) {
            // R28: l_t = longest side of the particle box, centre = its midpoint (fp64 on the exact fp32 bounds)
            l = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                l = fmax(l, __dadd_rn((double)mx[d], -(double)mn[d]));
                g[d] = __dmul_rn(0.5, __dadd_rn((double)mn[d], (double)mx[d]));
            }
        } else if (grow) {
            double e = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) e = fmax(e, fmax(__dadd_rn(g[d], -(double)mn[d]), __dadd_rn((double)mx[d], -g[d])));
            l = fmax(l, __dmul_rn(2.0, e));
        }
    }
    Mom o = q;
    if (!(q.m > 0.0)) {  // only zero-mass members: COM is undefined, take the geometric centre (R8)
        o.cx = g[0]; o.cy = g[1]; o.cz = g[2];
        o.xx = o.yy = o.zz = o.xy = o.xz = o.yz = 0.0;
    }
    const double ex = __dadd_rn(o.cx, -g[0]), ey = __dadd_rn(o.cy, -g[1]), ez = __dadd_rn(o.cz, -g[2]);
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
    // 16-byte stores: the record is written (and read back by the parent) in 5 L2 transactions instead of 10
    double2* mo = reinterpret_cast<double2*>(c_mom + (size_t)c * 10);
    __stcg(&mo[0], make_double2(o.m, o.cx));
    __stcg(&mo[1], make_double2(o.cy, o.cz));
    __stcg(&mo[2], make_double2(o.xx, o.yy));
    __stcg(&mo[3], make_double2(o.zz, o.xy));
    __stcg(&mo[4], make_double2(o.xz, o.yz));
    CellMac cm;
    cm.cx = (float)o.cx; cm.cy = (float)o.cy; cm.cz = (float)o.cz; cm.m = (float)o.m;
    cm.delta = (float)sqrt(d2);
    cm.lside = (float)l;
    cm.first = link_first;
    cm.info = link_info;
    c_mac[c] = cm;
    (void)c_qraw;  // the fp32 raw moments are introspection only: k_cells_qraw derives them from c_mom on demand
    const double tr = o.xx + o.yy + o.zz;
    CellQuad cq;
    cq.pxx = (float)(tr - 3.0 * o.xx); cq.pyy = (float)(tr - 3.0 * o.yy); cq.pzz = (float)(tr - 3.0 * o.zz);
    cq.pxy = (float)(-3.0 * o.xy); cq.pxz = (float)(-3.0 * o.xz); cq.pyz = (float)(-3.0 * o.yz);
    cq.tr = (float)tr;
    cq.pad = 0.0f;
    c_quad[c] = cq;
}

struct TreeView {
    const uint32_t *level, *first, *count, *first_child, *n_child, *parent;
};

// Leaf: sums over its particles, in particle order, without FMA contraction.
template <bool kBox>
__device__ __forceinline__ void leaf_moments(const float4* __restrict__ sorted_pos, uint32_t f, uint32_t cnt, Mom& q,
                                             float (&mn)[3], float (&mx)[3]) {
    double sx = 0.0, sy = 0.0, sz = 0.0;
    q.m = 0.0;
    q.cx = q.cy = q.cz = 0.0;
    q.xx = q.yy = q.zz = q.xy = q.xz = q.yz = 0.0;
    for (uint32_t k = 0; k < cnt; ++k) {
        const float4 p = __ldg(&sorted_pos[f + k]);
        const double m = (double)p.w;
        if (kBox) {
            mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
            mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
            mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
        }
        q.m = __dadd_rn(q.m, m);
        sx = __dadd_rn(sx, __dmul_rn(m, (double)p.x));
        sy = __dadd_rn(sy, __dmul_rn(m, (double)p.y));
        sz = __dadd_rn(sz, __dmul_rn(m, (double)p.z));
    }
    if (q.m > 0.0) {
        q.cx = sx / q.m; q.cy = sy / q.m; q.cz = sz / q.m;
        for (uint32_t k = 0; k < cnt; ++k) {
            const float4 p = __ldg(&sorted_pos[f + k]);
            const double m = (double)p.w;
            const double dx = __dadd_rn((double)p.x, -q.cx), dy = __dadd_rn((double)p.y, -q.cy),
                         dz = __dadd_rn((double)p.z, -q.cz);
            q.xx = __dadd_rn(q.xx, __dmul_rn(__dmul_rn(m, dx), dx));
            q.yy = __dadd_rn(q.yy, __dmul_rn(__dmul_rn(m, dy), dy));
            q.zz = __dadd_rn(q.zz, __dmul_rn(__dmul_rn(m, dz), dz));
            q.xy = __dadd_rn(q.xy, __dmul_rn(__dmul_rn(m, dx), dy));
            q.xz = __dadd_rn(q.xz, __dmul_rn(__dmul_rn(m, dx), dz));
            q.yz = __dadd_rn(q.yz, __dmul_rn(__dmul_rn(m, dy), dz));
        }
    }
}

// Internal cell: ONE pass over the children's fp64 records (each fetched once, two children's loads in flight per
// trip).  Moments are gathered about the first child's centre c0 -- at most a cell diagonal away from every other child,
// so the shift to the centre of mass below cancels at most one digit of the fp64 sums -- and moved to the COM at the
// end (parallel-axis theorem):
//   M = sum m_k,  S = sum m_k d_k,  T = sum (Q_k + m_k d_k d_k^T),  d_k = c_k - c0;
//   COM = c0 + S / M,  Q = T - M (S / M)(S / M)^T.
// A massless child has Q = 0 and m = 0 and drops out by itself.
template <bool kBox>
__device__ __forceinline__ void combine_children(const double* __restrict__ c_mom, const float* __restrict__ c_box, uint32_t fc,
                                                 uint32_t nc, Mom& q, float (&mn)[3], float (&mx)[3]) {
    const double2* mo0 = reinterpret_cast<const double2*>(c_mom + (size_t)fc * 10);
    double c0x = 0.0, c0y = 0.0, c0z = 0.0;
    double M = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
    double txx = 0.0, tyy = 0.0, tzz = 0.0, txy = 0.0, txz = 0.0, tyz = 0.0;
#pragma unroll 2
    for (uint32_t k = 0; k < nc; ++k) {
        const double2 r0 = __ldcg(&mo0[5 * k + 0]), r1 = __ldcg(&mo0[5 * k + 1]), r2 = __ldcg(&mo0[5 * k + 2]),
                      r3 = __ldcg(&mo0[5 * k + 3]), r4 = __ldcg(&mo0[5 * k + 4]);
        if (kBox) {
            const float2* bx = reinterpret_cast<const float2*>(c_box + (size_t)(fc + k) * 6);
            const float2 b0 = __ldcg(&bx[0]), b1 = __ldcg(&bx[1]), b2 = __ldcg(&bx[2]);
            mn[0] = fminf(mn[0], b0.x); mn[1] = fminf(mn[1], b0.y); mn[2] = fminf(mn[2], b1.x);
            mx[0] = fmaxf(mx[0], b1.y); mx[1] = fmaxf(mx[1], b2.x); mx[2] = fmaxf(mx[2], b2.y);
        }
        if (k == 0) { c0x = r0.y; c0y = r1.x; c0z = r1.y; }
        const double m = r0.x;
        const double dx = r0.y - c0x, dy = r1.x - c0y, dz = r1.y - c0z;
        M += m;
        sx += m * dx; sy += m * dy; sz += m * dz;
        txx += r2.x + m * dx * dx;
        tyy += r2.y + m * dy * dy;
        tzz += r3.x + m * dz * dz;
        txy += r3.y + m * dx * dy;
        txz += r4.x + m * dx * dz;
        tyz += r4.y + m * dy * dz;
    }
    q.m = M;
    q.cx = q.cy = q.cz = 0.0;
    q.xx = q.yy = q.zz = q.xy = q.xz = q.yz = 0.0;
    if (M > 0.0) {
        const double ux = sx / M, uy = sy / M, uz = sz / M;
        q.cx = c0x + ux; q.cy = c0y + uy; q.cz = c0z + uz;
        q.xx = txx - M * ux * ux;
        q.yy = tyy - M * uy * uy;
        q.zz = tzz - M * uz * uz;
        q.xy = txy - M * ux * uy;
        q.xz = txz - M * ux * uz;
        q.yz = tyz - M * uy * uz;
    }
}

// Small systems (n < kMultTilesMinN): one thread per cell, the LAST child to arrive at a parent combines its siblings
// and climbs on -- nobody waits.  Most of the time one lane per warp is active, but the chain from the deepest leaf
// to the root (which is all a small tree has) is one acq_rel atomic + one round of loads per level, shorter than the
// publish / poll hand-off of the tiled kernel below: 0.056 against 0.078 ms at N = 2^15, 0.097 against 0.107 ms at 2^20.
template <bool kBox, bool kTight>
__global__ void __launch_bounds__(128, 8) k_multipoles_climb(Control* __restrict__ ctl, uint32_t cap_cells, TreeView t,
                                                    const float4* __restrict__ sorted_pos,
                                                    const uint32_t* __restrict__ khi, const uint32_t* __restrict__ kmid,
                                                    const uint32_t* __restrict__ klo, double* __restrict__ c_mom,
                                                    CellMac* __restrict__ c_mac, CellQuad* __restrict__ c_quad,
                                                    float* __restrict__ c_qraw, float* __restrict__ c_box,
                                                    uint32_t* __restrict__ c_arrived, const Gate grow_gate) {
    const bool grow = !gate_closed(grow_gate);  // (see k_multipoles)
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (ctl->status != 0) return;               // (see k_multipoles)
    if (c >= min(ctl->n_cells, cap_cells)) return;
    if (t.n_child[c] != 0) return;  // internal cells are produced by their last child
    {
        const uint32_t f = t.first[c], cnt = t.count[c];
        Mom q;
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        leaf_moments<kBox>(sorted_pos, f, cnt, q, mn, mx);
        store_cell<kBox, kTight>(q, mn, mx, c, (int)t.level[c], __ldg(&khi[f]), __ldg(&kmid[f]), __ldg(&klo[f]), ctl, f,
                   kLeafBit | cnt, c_mom, c_box, c_mac, c_quad, c_qraw, grow);
    }
    for (;;) {
        const uint32_t p = t.parent[c];
        if (p == kNone) return;
        const uint32_t nc = t.n_child[p];
        // release: this cell's moments are visible (gpu scope) before the arrival is; acquire: the last child to
        // arrive sees its siblings' moments.  One acq_rel atomic instead of two full fences around a relaxed one.
        uint32_t arrived;
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(arrived) : "l"(&c_arrived[p]) : "memory");
        if (arrived + 1u != nc) return;
        c_arrived[p] = 0;  // ready for the next step
        const uint32_t fc = t.first_child[p];
        Mom q;
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        combine_children<kBox>(c_mom, c_box, fc, nc, q, mn, mx);
        const uint32_t f = t.first[p];
        store_cell<kBox, kTight>(q, mn, mx, p, (int)t.level[p], __ldg(&khi[f]), __ldg(&kmid[f]), __ldg(&klo[f]), ctl, fc, nc,
                   c_mom, c_box, c_mac, c_quad, c_qraw, grow);
        c = p;
    }
}

// Scheduler: tiles of 32 consecutive cells, one per warp, are handed out by an atomic ticket from the END of the cell
// array (breadth-first numbering: children have larger ids than their parent, so the deepest cells come first).  A warp
// that holds ticket t therefore knows that every tile with children of its cells has been STARTED by a running warp, and
// may wait for them: an internal cell spins (acquire) on its arrival counter until all children have published their
// moments (release: one gpu-scope fence per warp after a warp barrier, then relaxed increments).  Waiting is rare -- the
// children's tiles were drawn thousands of tickets earlier -- except near the root.  Inside a tile the levels are
// processed deepest first with a warp barrier in between (a tile can hold a parent and its children only near the root,
// where levels are shorter than a tile).  No block-wide barrier anywhere: the warps of a block are independent.
// (Until round 2 the last child to arrive combined its siblings and climbed on: one active lane per warp for most of
// the kernel, 28 % of the warp slots in use, 0.204 ms at N = 2^22; tiles of 128 cells per block with block barriers:
// 0.178 ms, 15 % of the stall samples at the barrier and 6 % in per-thread release fences; this form: 0.173 ms.
// Fetching the leaf particles two or four at a time spills at 64 registers: 0.198 / 0.219 ms.)
constexpr int kMultThreads = 128;
constexpr uint32_t kMultTilesMinN = 1u << 21;  // below: k_multipoles_climb (measured crossover between 2^20 and 2^22)

template <bool kBox, bool kTight>
__global__ void __launch_bounds__(kMultThreads, 8) k_multipoles(Control* __restrict__ ctl, uint32_t cap_cells, TreeView t,
                                                    const float4* __restrict__ sorted_pos,
                                                    const uint32_t* __restrict__ khi, const uint32_t* __restrict__ kmid,
                                                    const uint32_t* __restrict__ klo, double* __restrict__ c_mom,
                                                    CellMac* __restrict__ c_mac, CellQuad* __restrict__ c_quad,
                                                    float* __restrict__ c_qraw, float* __restrict__ c_box,
                                                    uint32_t* __restrict__ c_arrived, const Gate grow_gate) {
    // R25 growth of the cell side applies to a REFRESHED tree only; whether this tree was refreshed may have been
    // decided on the device (R30): the gate is open (or absent) when it was
    const bool grow = !gate_closed(grow_gate);
    // a cell-capacity overflow leaves child links that point past the arrays: nothing downstream of the build may
    // follow them (bonsai_sync reports the status; the next build recovers)
    if (ctl->status != 0) return;
    const uint32_t n_cells = min(ctl->n_cells, cap_cells);
    const uint32_t n_tiles = (n_cells + 31u) / 32u;
    const int lane = threadIdx.x & 31;
    for (;;) {
        uint32_t ticket = 0;
        if (lane == 0) ticket = atomicAdd(&ctl->mult_ticket, 1u);
        ticket = __shfl_sync(0xFFFFFFFFu, ticket, 0);
        if (ticket >= n_tiles) break;
        const uint32_t c = (n_tiles - 1u - ticket) * 32u + (uint32_t)lane;
        const bool valid = c < n_cells;
        const int level = valid ? (int)t.level[c] : -1;
        const int lmax = __reduce_max_sync(0xFFFFFFFFu, level);
        const int lmin = __reduce_min_sync(0xFFFFFFFFu, valid ? level : 64);
        for (int L = lmax; L >= lmin; --L) {
            const bool mine = valid && level == L;
            uint32_t parent = kNone;
            if (mine) {
                const uint32_t nc = t.n_child[c];
                Mom q;
                float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
                const uint32_t f = t.first[c];
                uint32_t link_first, link_info;
                if (nc == 0) {
                    const uint32_t cnt = t.count[c];
                    leaf_moments<kBox>(sorted_pos, f, cnt, q, mn, mx);
                    link_first = f;
                    link_info = kLeafBit | cnt;
                } else {
                    // internal cell: wait for the children (acquire), then combine their fp64 moments
                    uint32_t arrived;
                    for (;;) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(arrived) : "l"(&c_arrived[c]) : "memory");
                        if (arrived == nc) break;
                        __nanosleep(40);
                    }
                    c_arrived[c] = 0;  // ready for the next step
                    const uint32_t fc = t.first_child[c];
                    combine_children<kBox>(c_mom, c_box, fc, nc, q, mn, mx);
                    link_first = fc;
                    link_info = nc;
                }
                store_cell<kBox, kTight>(q, mn, mx, c, L, __ldg(&khi[f]), __ldg(&kmid[f]), __ldg(&klo[f]), ctl, link_first,
                                         link_info, c_mom, c_box, c_mac, c_quad, c_qraw, grow);
                parent = t.parent[c];
            }
            // release, once per warp: the warp barrier orders the lanes' stores before lane 0's gpu-scope fence
            // (cumulative), the arrivals after it may then be relaxed
            __syncwarp();
            if (lane == 0) __threadfence();
            __syncwarp();
            if (parent != kNone) asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(&c_arrived[parent]) : "memory");
        }
    }
    // the last block to leave resets the scheduler for the next pass
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(&ctl->mult_done, 1u) == gridDim.x - 1) {
        ctl->mult_done = 0;
        ctl->mult_ticket = 0;
    }
}

// Introspection (bonsai_get_cells): the six raw second moments as fp32, rounded once from the fp64 record (R8).
__global__ void __launch_bounds__(256) k_cells_qraw(const Control* __restrict__ ctl, uint32_t cap_cells,
                                                    const double* __restrict__ c_mom, float* __restrict__ c_qraw) {
    const uint32_t n_cells = min(ctl->n_cells, cap_cells);
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cells; c += gridDim.x * blockDim.x)
#pragma unroll
        for (int k = 0; k < 6; ++k) c_qraw[(size_t)c * 6 + k] = (float)c_mom[(size_t)c * 10 + 4 + k];
}

cudaError_t cells_qraw(Ctx* c) {
    k_cells_qraw<<<c->num_sms * 8, 256, 0, c->stream>>>(c->b.ctl, c->cap_cells, c->b.c_mom, c->b.c_qraw);
    c->launches += 1;
    return cudaGetLastError();
}

// Recovery after a capacity overflow (guarded: returns at once when the device status is clear).  An overflow of the
// cell arrays leaves arrival counters of cells whose children were cut off non-zero, which would corrupt every
// later multipole pass of this context; the counters are re-zeroed and the sticky status is cleared by the last
// block to finish, so that the status read by bonsai_sync() covers the work since the last bonsai_build_tree().
__global__ void __launch_bounds__(256) k_recover(Control* __restrict__ ctl, uint32_t cap_cells,
                                                 uint32_t* __restrict__ c_arrived) {
    if (ctl->status == 0) return;  // the same answer in every block: only the last block to finish clears it
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < cap_cells; c += gridDim.x * blockDim.x) c_arrived[c] = 0;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(&ctl->recover_ticket, 1u) == gridDim.x - 1) {
        ctl->recover_ticket = 0;
        ctl->status = 0;
    }
}

cudaError_t stage_recover(Ctx* c) {
    k_recover<<<c->num_sms * 2, 256, 0, c->stream>>>(c->b.ctl, c->cap_cells, c->b.c_arrived);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_multipoles(Ctx* c) {
    Buffers& b = c->b;
    const int s = c->sorted_buf;
    TreeView t{b.c_level, b.c_first, b.c_count, b.c_first_child, b.c_n_child, b.c_parent};
    using Kernel = void (*)(Control*, uint32_t, TreeView, const float4*, const uint32_t*, const uint32_t*, const uint32_t*,
                            double*, CellMac*, CellQuad*, float*, float*, uint32_t*, Gate);
    const int which = (c->prm.mac_mode == 1) ? 2 : (c->tree_refreshed || c->tree_auto) ? 1 : 0;
    static const Kernel kTiles[3] = {k_multipoles<false, false>, k_multipoles<true, false>, k_multipoles<true, true>};
    static const Kernel kClimb[3] = {k_multipoles_climb<false, false>, k_multipoles_climb<true, false>,
                                     k_multipoles_climb<true, true>};
    // a tree handled by the device-side rebuild decision (R30) was refreshed iff rebuild_flag == 0
    const Gate grow = c->tree_auto ? Gate{&b.ctl->rebuild_flag, 0u} : Gate{nullptr, 0u};
    const bool tiles = c->prm.mult_kernel == 2 || (c->prm.mult_kernel == 0 && c->n >= kMultTilesMinN);
    if (tiles) {
        // persistent blocks (8 per SM) draw tiles of 32 cells until the device-side cell count is exhausted
        const dim3 grid(min(div_up(c->cap_cells, (uint32_t)kMultThreads), (uint32_t)c->num_sms * 8u));
        kTiles[which]<<<grid, kMultThreads, 0, c->stream>>>(b.ctl, c->cap_cells, t, b.sorted_pos, b.key[s][0], b.key[s][1],
                                                            b.key[s][2], b.c_mom, b.c_mac, b.c_quad, b.c_qraw, b.c_box,
                                                            b.c_arrived, grow);
    } else {
        kClimb[which]<<<div_up(c->cap_cells, 128u), 128, 0, c->stream>>>(b.ctl, c->cap_cells, t, b.sorted_pos, b.key[s][0],
                                                                         b.key[s][1], b.key[s][2], b.c_mom, b.c_mac, b.c_quad,
                                                                         b.c_qraw, b.c_box, b.c_arrived, grow);
    }
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace bonsai
