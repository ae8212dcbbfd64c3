// Stage a6 / a7: the tree-walk ("tree-traverse"; more than 90 % of the step at theta = 0.75).
// Readings R9 (opening criterion, defined in fp32), R10 (softening), R11 (self term), R12 (potential),
// R14 (accepted leaf = p-c), R19 (active mask), R21 (interaction counts) of DESIGN.md.
//
// One warp per group (Barnes 1990: one shared traversal per group of neighbouring particles), groups handed out
// by an atomic ticket so consecutive (= spatially adjacent) groups run at the same time and share the cell
// data they pull through L2 / L1.  Each lane holds one sink, or two when the group has more than 32.
//
// Traversal: a per-warp stack in shared memory whose entries are RUNS of sibling cells (first_child, n_child) --
// children are consecutive in the breadth-first numbering, so one entry expands into up to 8 lanes.  Per round
// the warp pops as many entries as fit into 32 cells, every lane applies the opening test to one cell, then
//   accepted cell      -> ring buffer of cell ids      (flushed 32 at a time through the p-c kernel)
//   rejected leaf      -> its particles -> ring buffer  (flushed 32 at a time through the p-p kernel)
//   rejected internal  -> its child run is pushed.
// Few groups (a small active subset): one group's walk is a serial chain of ~0.4 ms, so when there are fewer
// groups than resident warps the kernel would last as long as its slowest group.  The warps of a block then form
// TEAMS of S = 2, 4 or 8 (chosen on the device from the number of groups) that walk ONE group together: the stack of
// sibling runs is shared by the team (the members' private stacks, concatenated); per round every member takes its
// own four runs off the top (eight lanes per run, no scan), tests those cells, keeps the cells it accepts and the
// leaves it opens in its OWN rings and evaluates them itself, and pushes the children of the cells it opens back
// onto the shared stack (two team barriers per round: counts, then stack).  Traversal and evaluation are both
// divided by S; the union of the members' lists is exactly the group's list, so counts are unchanged, and the
// members' partial sums and counts are folded in member order at the end.  (Round 1 let every member repeat the
// whole traversal and only divided the evaluation: the traversal, ~15 % of a group-walk, bounded a team of 8 at ~4x.)
// Interaction kernels run in fp32 (FFMA + MUFU.RSQ); each batch of <= 32 sources is summed in fp32 starting
// from zero and the batch total is added to an fp64 running total, which keeps the round-off of the long sum
// out of the result at the cost of 4 DADD per 32 interactions.
#include "internal.cuh"

namespace bonsai {

struct WalkArgs {
    Control* ctl;
    const CellMac* mac;
    const CellQuad* quad;
    const float4* pos;       // sorted particles
    const uint32_t* perm;    // sorted -> load index
    const uint32_t* active_list;
    const uint32_t *g_first, *g_count;
    const float *g_bmin, *g_bmax;
    float inv_theta, eps2;
    uint32_t warps_small, warps_big;  // resident warps of the 8-warp and of the 16-warp team kernel (regime choice)
    float4* out;             // load order
    uint32_t *n_pp, *n_pc;   // load order
};

struct __align__(16) WarpSmem {
    float4 pp[64];                 // ring of p-p sources
    float4 pc[32][3];              // staged p-c sources: (cx,cy,cz,m) (Pxx,Pyy,Pzz,Pxy) (Pxz,Pyz,tr eps^2,-)
    uint32_t stack[kWalkStack];    // runs of sibling cells: (first << 3) | (n - 1)
    uint32_t pc_ids[64];           // ring of accepted cell ids
    uint32_t leaf_first[32];
    uint32_t leaf_pref[36];
    float2 sink_xyz[3][32];        // per lane: negated (x0, x1), (y0, y1), (z0, z1) of its two sinks, see walk_chunk
};

size_t walk_smem_bytes(uint32_t) { return sizeof(WarpSmem) * kWalkWarps; }
constexpr int kWalkWarpsBig = 16;  // the team kernel for very few groups: one block of 16 warps per SM, teams of up to 16

__device__ __forceinline__ float rsqrt_fast(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Packed fp32x2 arithmetic (sm_100: FFMA2 / FMUL2 / FADD2).  One instruction does the same IEEE operation on the
// two halves of a 64-bit register pair, so a lane that holds two sinks spends ONE issue slot per operation for
// both of them.  Measured on B200 (profiles/r2_microbench.md): FFMA2 runs at half the instruction rate
// of FFMA -- the same 74 TFLOP/s -- which turns the interaction loops from issue-bound into FP32-pipe-bound.
typedef unsigned long long f32x2;  // two fp32 values in one 64-bit register pair: .x = low half, .y = high half
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float lo2(f32x2 v) {
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return a;
}
__device__ __forceinline__ float hi2(f32x2 v) {
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return b;
}
__device__ __forceinline__ f32x2 bc(float v) { return pack2(v, v); }
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 rsqrt2(f32x2 v) { return pack2(rsqrt_fast(lo2(v)), rsqrt_fast(hi2(v))); }

template <int NS>
struct Sinks {
    f32x2 nx2, ny2, nz2;     // NS = 2: (-x0, -x1), (-y0, -y1), (-z0, -z1), kept packed for the whole walk
    float x[NS], y[NS], z[NS];
    double ax[NS], ay[NS], az[NS], ph[NS];  // ph accumulates +sum m/r (negated on output)
    int pair0, pair_step;    // NS = 1: this lane evaluates the source pairs pair0, pair0 + pair_step, ... (lane split)
};

// NS = 2: the two sinks of a lane ride in the two halves of packed registers; operation for operation (and
// rounding for rounding) the same arithmetic as the scalar loop below.
template <bool kZeroEps>
__device__ __forceinline__ void eval_pp_packed(WarpSmem& S, uint32_t r0, int nb, float eps2, Sinks<2>& s) {
    const f32x2 nsx = s.nx2, nsy = s.ny2, nsz = s.nz2;
    const f32x2 e2 = bc(eps2);
    f32x2 ax = bc(0.0f), ay = bc(0.0f), az = bc(0.0f), ph = bc(0.0f);
    const float4* src = &S.pp[r0 & 63u];  // batches start at ring slot 0 or 32 and hold <= 32 sources: no wrap
#pragma unroll 4
    for (int j = 0; j < nb; ++j) {
        const float4 q = src[j];
        const f32x2 dx = fadd2(bc(q.x), nsx), dy = fadd2(bc(q.y), nsy), dz = fadd2(bc(q.z), nsz);
        f32x2 rinv;
        if (kZeroEps) {
            const f32x2 r2 = ffma2(dx, dx, ffma2(dy, dy, fmul2(dz, dz)));
            rinv = pack2((lo2(r2) > 0.0f) ? rsqrt_fast(lo2(r2)) : 0.0f, (hi2(r2) > 0.0f) ? rsqrt_fast(hi2(r2)) : 0.0f);
        } else {
            rinv = rsqrt2(ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2))));
        }
        const f32x2 mr = fmul2(bc(q.w), rinv);
        const f32x2 rinv2 = fmul2(rinv, rinv);
        const f32x2 mr3 = fmul2(mr, rinv2);
        ph = fadd2(ph, mr);
        ax = ffma2(mr3, dx, ax);
        ay = ffma2(mr3, dy, ay);
        az = ffma2(mr3, dz, az);
    }
    s.ax[0] += (double)lo2(ax); s.ay[0] += (double)lo2(ay); s.az[0] += (double)lo2(az); s.ph[0] += (double)lo2(ph);
    s.ax[1] += (double)hi2(ax); s.ay[1] += (double)hi2(ay); s.az[1] += (double)hi2(az); s.ph[1] += (double)hi2(ph);
    __syncwarp();
}

// NS = 1 (a group of <= 32 sinks: the short last run of a container): one sink per lane would leave half of every
// packed operation empty, and scalar FFMA gives the shared-memory loads, MUFU and loop control no FFMA2 shadow to hide
// in (measured with ncrit = 32: 1.4x the time per interaction).  Instead the lane's ONE sink rides in both halves
// and the two halves take two DIFFERENT sources: the rings are kept in pair layout (pair p = sources 2p, 2p + 1 stored
// as (x0, x1, y0, y1) (z0, z1, m0, m1)), so every operand is an aligned register pair straight out of an LDS.128.
// An odd batch is padded with a massless source far away (contributes exactly 0).
constexpr float kPadFar = 1.0e15f;

__device__ __forceinline__ void pp_put_pairs(WarpSmem& S, uint32_t slot, const float4 v) {
    float* f = reinterpret_cast<float*>(S.pp);
    const uint32_t t = slot & 63u, base = (t >> 1) * 8u + (t & 1u);
    f[base] = v.x; f[base + 2] = v.y; f[base + 4] = v.z; f[base + 6] = v.w;
}

template <bool kZeroEps>
__device__ __forceinline__ void eval_pp_pairs(WarpSmem& S, uint32_t r0, int nb, float eps2, int lane, Sinks<1>& s) {
    if (nb & 1) {  // (tails only: full batches hold 32 sources)
        if (lane == 0) pp_put_pairs(S, r0 + (uint32_t)nb, make_float4(kPadFar, kPadFar, kPadFar, 0.0f));
        __syncwarp();
    }
    const f32x2 nsx = s.nx2, nsy = s.ny2, nsz = s.nz2;
    const f32x2 e2 = bc(eps2);
    f32x2 ax = bc(0.0f), ay = bc(0.0f), az = bc(0.0f), ph = bc(0.0f);
    const float4* src = &S.pp[r0 & 63u];  // batches start at ring slot 0 or 32: pair-aligned, no wrap
    const int np = (nb + 1) >> 1;
    const int pstep = s.pair_step;
#pragma unroll 4
    for (int p = s.pair0; p < np; p += pstep) {
        const float4 u = src[2 * p], v = src[2 * p + 1];
        const f32x2 dx = fadd2(pack2(u.x, u.y), nsx), dy = fadd2(pack2(u.z, u.w), nsy), dz = fadd2(pack2(v.x, v.y), nsz);
        f32x2 rinv;
        if (kZeroEps) {  // eps = 0: the self term (and only it, R11) has r = 0 and must drop out
            const f32x2 r2 = ffma2(dx, dx, ffma2(dy, dy, fmul2(dz, dz)));
            rinv = pack2((lo2(r2) > 0.0f) ? rsqrt_fast(lo2(r2)) : 0.0f, (hi2(r2) > 0.0f) ? rsqrt_fast(hi2(r2)) : 0.0f);
        } else {         // eps > 0: the self term adds exactly m/eps to ph and 0 to a; removed at the end
            rinv = rsqrt2(ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2))));
        }
        const f32x2 mr = fmul2(pack2(v.z, v.w), rinv);
        const f32x2 rinv2 = fmul2(rinv, rinv);
        const f32x2 mr3 = fmul2(mr, rinv2);
        ph = fadd2(ph, mr);
        ax = ffma2(mr3, dx, ax);
        ay = ffma2(mr3, dy, ay);
        az = ffma2(mr3, dz, az);
    }
    s.ax[0] += (double)(lo2(ax) + hi2(ax)); s.ay[0] += (double)(lo2(ay) + hi2(ay));
    s.az[0] += (double)(lo2(az) + hi2(az)); s.ph[0] += (double)(lo2(ph) + hi2(ph));
    __syncwarp();
}

template <int NS, bool kZeroEps>
__device__ __forceinline__ void eval_pp(WarpSmem& S, uint32_t r0, int nb, float eps2, int lane, Sinks<NS>& s) {
    if constexpr (NS == 2) eval_pp_packed<kZeroEps>(S, r0, nb, eps2, s);
    else eval_pp_pairs<kZeroEps>(S, r0, nb, eps2, lane, s);
}

template <int NS>
__device__ __forceinline__ void eval_pc(WarpSmem& S, const WalkArgs& a, uint32_t r0, int nb, int lane, Sinks<NS>& s) {
    if constexpr (NS == 2) {
        if (lane < nb) {
            const uint32_t c = S.pc_ids[(r0 + lane) & 63];
            const float4* m = reinterpret_cast<const float4*>(a.mac + c);
            const float4* q = reinterpret_cast<const float4*>(a.quad + c);
            S.pc[lane][0] = __ldg(m);
            S.pc[lane][1] = __ldg(q);
            float4 q1 = __ldg(q + 1);
            q1.z = q1.z * a.eps2;  // tr eps^2: the softening term of the quadrupole (see CellQuad), once per cell
            S.pc[lane][2] = q1;
        }
        __syncwarp();
        const f32x2 nsx = s.nx2, nsy = s.ny2, nsz = s.nz2;
        const f32x2 e2 = bc(a.eps2);
        f32x2 ax = bc(0.0f), ay = bc(0.0f), az = bc(0.0f), ph = bc(0.0f);
#pragma unroll 2
        for (int j = 0; j < nb; ++j) {
            const float4 c0 = S.pc[j][0], c1 = S.pc[j][1], c2 = S.pc[j][2];
            const f32x2 dx = fadd2(bc(c0.x), nsx), dy = fadd2(bc(c0.y), nsy), dz = fadd2(bc(c0.z), nsz);
            const f32x2 rinv = rsqrt2(ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2))));
            const f32x2 rinv2 = fmul2(rinv, rinv);
            // c1 = (Pxx, Pyy, Pzz, Pxy), c2 = (Pxz, Pyz, tr eps^2, -)
            const f32x2 prx = ffma2(bc(c1.x), dx, ffma2(bc(c1.w), dy, fmul2(bc(c2.x), dz)));
            const f32x2 pry = ffma2(bc(c1.w), dx, ffma2(bc(c1.y), dy, fmul2(bc(c2.y), dz)));
            const f32x2 prz = ffma2(bc(c2.x), dx, ffma2(bc(c2.y), dy, fmul2(bc(c1.z), dz)));
            const f32x2 sq = ffma2(dx, prx, ffma2(dy, pry, ffma2(dz, prz, bc(c2.z))));  // dr.P.dr + tr eps^2
            const f32x2 rinv3 = fmul2(rinv, rinv2);
            const f32x2 rinv5 = fmul2(rinv3, rinv2);
            const f32x2 q5 = fmul2(sq, rinv5);
            // ph accumulates -phi = M/r - (dr.P.dr + tr eps^2) / (2 r^5)
            ph = ffma2(bc(c0.w), rinv, ph);
            ph = ffma2(bc(-0.5f), q5, ph);
            // a = dr (M/r^3 - 5/2 q5/r^2) + P.dr / r^5
            const f32x2 f = ffma2(bc(-2.5f), fmul2(q5, rinv2), fmul2(bc(c0.w), rinv3));
            ax = ffma2(dx, f, ax); ax = ffma2(rinv5, prx, ax);
            ay = ffma2(dy, f, ay); ay = ffma2(rinv5, pry, ay);
            az = ffma2(dz, f, az); az = ffma2(rinv5, prz, az);
        }
        s.ax[0] += (double)lo2(ax); s.ay[0] += (double)lo2(ay); s.az[0] += (double)lo2(az); s.ph[0] += (double)lo2(ph);
        s.ax[1] += (double)hi2(ax); s.ay[1] += (double)hi2(ay); s.az[1] += (double)hi2(az); s.ph[1] += (double)hi2(ph);
        __syncwarp();
    } else {
        // pair layout (see eval_pp_pairs): pair p = cells 2p, 2p + 1 as six float4
        //   (cx0, cx1, cy0, cy1) (cz0, cz1, M0, M1) (Pxx0, Pxx1, Pyy0, Pyy1) (Pzz0, Pzz1, Pxy0, Pxy1)
        //   (Pxz0, Pxz1, Pyz0, Pyz1) (tr0 eps^2, tr1 eps^2, -, -);  S.pc holds 16 pairs
        float* f = reinterpret_cast<float*>(S.pc);
        if (lane < nb) {
            const uint32_t c = S.pc_ids[(r0 + lane) & 63];
            const float4* m = reinterpret_cast<const float4*>(a.mac + c);
            const float4* q = reinterpret_cast<const float4*>(a.quad + c);
            const float4 m0 = __ldg(m), q0 = __ldg(q), q1 = __ldg(q + 1);
            const uint32_t base = ((uint32_t)lane >> 1) * 24u + ((uint32_t)lane & 1u);
            f[base] = m0.x; f[base + 2] = m0.y; f[base + 4] = m0.z; f[base + 6] = m0.w;
            f[base + 8] = q0.x; f[base + 10] = q0.y; f[base + 12] = q0.z; f[base + 14] = q0.w;
            f[base + 16] = q1.x; f[base + 18] = q1.y; f[base + 20] = q1.z * a.eps2;
        } else if (lane == nb && (nb & 1)) {  // odd tail: a massless cell far away contributes exactly 0
            const uint32_t base = ((uint32_t)lane >> 1) * 24u + 1u;
            f[base] = kPadFar; f[base + 2] = kPadFar; f[base + 4] = kPadFar; f[base + 6] = 0.0f;
            f[base + 8] = 0.0f; f[base + 10] = 0.0f; f[base + 12] = 0.0f; f[base + 14] = 0.0f;
            f[base + 16] = 0.0f; f[base + 18] = 0.0f; f[base + 20] = 0.0f;
        }
        __syncwarp();
        const f32x2 nsx = s.nx2, nsy = s.ny2, nsz = s.nz2;
        const f32x2 e2 = bc(a.eps2);
        f32x2 ax = bc(0.0f), ay = bc(0.0f), az = bc(0.0f), ph = bc(0.0f);
        const float4* src = &S.pc[0][0];
        const int np = (nb + 1) >> 1;
        const int pstep = s.pair_step;
#pragma unroll 2
        for (int p = s.pair0; p < np; p += pstep) {
            const float4 A = src[6 * p], B = src[6 * p + 1], C = src[6 * p + 2], D = src[6 * p + 3], E = src[6 * p + 4],
                         F = src[6 * p + 5];
            const f32x2 dx = fadd2(pack2(A.x, A.y), nsx), dy = fadd2(pack2(A.z, A.w), nsy), dz = fadd2(pack2(B.x, B.y), nsz);
            const f32x2 M = pack2(B.z, B.w);
            const f32x2 pxx = pack2(C.x, C.y), pyy = pack2(C.z, C.w), pzz = pack2(D.x, D.y), pxy = pack2(D.z, D.w),
                        pxz = pack2(E.x, E.y), pyz = pack2(E.z, E.w);
            const f32x2 rinv = rsqrt2(ffma2(dx, dx, ffma2(dy, dy, ffma2(dz, dz, e2))));
            const f32x2 rinv2 = fmul2(rinv, rinv);
            const f32x2 prx = ffma2(pxx, dx, ffma2(pxy, dy, fmul2(pxz, dz)));
            const f32x2 pry = ffma2(pxy, dx, ffma2(pyy, dy, fmul2(pyz, dz)));
            const f32x2 prz = ffma2(pxz, dx, ffma2(pyz, dy, fmul2(pzz, dz)));
            const f32x2 sq = ffma2(dx, prx, ffma2(dy, pry, ffma2(dz, prz, pack2(F.x, F.y))));  // dr.P.dr + tr eps^2
            const f32x2 rinv3 = fmul2(rinv, rinv2);
            const f32x2 rinv5 = fmul2(rinv3, rinv2);
            const f32x2 q5 = fmul2(sq, rinv5);
            ph = ffma2(M, rinv, ph);
            ph = ffma2(bc(-0.5f), q5, ph);
            const f32x2 g = ffma2(bc(-2.5f), fmul2(q5, rinv2), fmul2(M, rinv3));
            ax = ffma2(dx, g, ax); ax = ffma2(rinv5, prx, ax);
            ay = ffma2(dy, g, ay); ay = ffma2(rinv5, pry, ay);
            az = ffma2(dz, g, az); az = ffma2(rinv5, prz, az);
        }
        s.ax[0] += (double)(lo2(ax) + hi2(ax)); s.ay[0] += (double)(lo2(ay) + hi2(ay));
        s.az[0] += (double)(lo2(az) + hi2(az)); s.ph[0] += (double)(lo2(ph) + hi2(ph));
        __syncwarp();
    }
}

// Size of the traversal stack (kWalkStack runs of siblings per warp).  A round pops runs from the top until 32 cells
// are gathered and pushes at most one run per tested cell, all one level below their parents.  New level-L runs
// appear only when level-(L-1) cells are tested, and those lie BELOW every level-L run still on the stack, so a
// round that reaches them has first consumed the level-L runs above: at any time at most 32 runs of one level are
// stacked, and the stack never holds more than 32 x (levels that branch) entries.  A Plummer sphere of 2^22 particles
// is 13 levels deep (32 x 13 = 416); single-child chains (coincident or very close particles) add one run per
// level.  512 entries therefore cover every tree whose opened frontier branches over <= 16 levels; the theoretical
// maximum of 30 levels (960) would cost twice the shared memory for trees that do not occur in practice, and is
// not silently wrong either: an overflow stops the group and sets the sticky BONSAI_ECAPACITY status.
__device__ __forceinline__ void team_barrier(int team, int warps) {
    asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "r"(warps * 32) : "memory");
}

// kTeam: this warp is member `slot` of a team of `tsize` warps (WarpSmem of member j = (&S)[j - slot]) that walks
// the chunk together; see the header.  kTeam = false compiles to the single-warp walk.
constexpr int kTeamRuns = 4;  // runs a team member takes per round: 4 x 8 lanes
// kMono: R29 -- accepted cells act as monopoles only: (COM, M) is a point source like any particle, so it joins the
// p-p ring and the p-c kernel is never called; lists and counts are those of the quadrupole walk.
template <int NS, bool kZeroEps, bool kTeam, bool kMono>
__device__ __forceinline__ bool walk_chunk(WarpSmem& S, const WalkArgs& a, int lane, uint32_t sink_first, uint32_t ns,
                                           const float (&bmin)[3], const float (&bmax)[3], int team, int slot,
                                           int tsize) {
    constexpr uint32_t tmask = 0u, uslot = 0u;  // (every warp evaluates all the batches of its own rings)
    const uint32_t lt = (1u << lane) - 1u;
    // team scratch in member 0's shared memory (its sink_xyz area, free once the sinks are in registers):
    // T[0] = entries on the shared stack, T[1 + j] = runs member j pushes this round
    volatile uint32_t* T = reinterpret_cast<volatile uint32_t*>(&(&S)[-slot].sink_xyz[0][0]);
    auto team_stack = [&](uint32_t e) -> uint32_t& { return (&S)[(int)(e / kWalkStack) - slot].stack[e % kWalkStack]; };
    const uint32_t team_cap = (uint32_t)tsize * kWalkStack;
    Sinks<NS> s;
    uint32_t sidx[NS];
    float smass[NS];
    // Lane split (NS = 1): a group of ns <= 16 sinks would leave half of the lanes (or more) idle.  With m = the
    // smallest power of two >= ns, lane l holds sink l mod m and is replica l / m of 32 / m; replica r evaluates the
    // source pairs r, r + 32/m, ... of every batch, and the replicas' partial sums are added by a butterfly at the end.
    uint32_t split_m = 32u;
    if constexpr (NS == 1) {
        while (split_m > 1u && (split_m >> 1) >= ns) split_m >>= 1;
        s.pair_step = (int)(32u / split_m);
        s.pair0 = lane / (int)split_m;
    }
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        // NS = 1 with ns <= 16: the sinks are replicated over the lanes (sink = lane mod m, m = the power of two >= ns)
        // and the 32 / m replicas share the sources of every batch between them -- see the lane split below
        const uint32_t off = (NS == 1 ? ((uint32_t)lane & (split_m - 1u)) : (uint32_t)lane) + 32u * k;
        const uint32_t at = sink_first + (off < ns ? off : 0u);
        sidx[k] = a.active_list ? __ldg(&a.active_list[at]) : at;  // nullptr: all particles active, identity
        const float4 p = __ldg(&a.pos[sidx[k]]);
        s.x[k] = p.x; s.y[k] = p.y; s.z[k] = p.z;
        smass[k] = p.w;
        s.ax[k] = s.ay[k] = s.az[k] = s.ph[k] = 0.0;
    }
    if constexpr (NS == 2) {
        // The packed loops want (-x0, -x1) etc. in ALIGNED register pairs.  Left as halves of the two float4 loads
        // above, ptxas re-pairs them with two MOVs per coordinate in every loop iteration (ALU-pipe slots that
        // FFMA2 cannot overlap, profiles/r2_microbench.md); a round trip through shared memory as 64-bit words makes each pair
        // the destination of one LDS.64.
        S.sink_xyz[0][lane] = make_float2(-s.x[0], -s.x[1]);
        S.sink_xyz[1][lane] = make_float2(-s.y[0], -s.y[1]);
        S.sink_xyz[2][lane] = make_float2(-s.z[0], -s.z[1]);
        __syncwarp();
        const uint32_t sa = (uint32_t)__cvta_generic_to_shared(&S.sink_xyz[0][lane]);
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(s.nx2) : "r"(sa));
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(s.ny2) : "r"(sa + 256u));
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(s.nz2) : "r"(sa + 512u));
    }
    if constexpr (NS == 1) {  // the one sink in both halves (eval_pp_pairs)
        s.nx2 = pack2(-s.x[0], -s.x[0]);
        s.ny2 = pack2(-s.y[0], -s.y[0]);
        s.nz2 = pack2(-s.z[0], -s.z[0]);
    }
    uint32_t pc_r = 0, pc_w = 0, pp_r = 0, pp_w = 0;
    uint32_t npc = 0, npp = 0;
    int sp = 1;
    if (!kTeam || slot == 0) {
        if (lane == 0) {
            S.stack[0] = 0u;  // the root alone: first = 0, n = 1
            if (kTeam) T[0] = 1u;
        }
    }
    bool ok = true;
    while (sp > 0) {
        bool valid;
        uint32_t cell;
        int take = 0;
        if constexpr (kTeam) {
            team_barrier(team, tsize);  // (A) the stack and its size as the last round left them
            sp = (int)T[0];
            if (sp == 0) break;
            // ---- pop: member `slot` takes runs slot * 4 .. slot * 4 + 3 from the top, eight lanes per run ----
            take = min(sp, kTeamRuns * tsize);
            const int r = slot * kTeamRuns + (lane >> 3);
            uint32_t e = 0;
            int cnt = 0;
            if (r < take) {
                e = team_stack((uint32_t)(sp - 1 - r));
                cnt = (int)(e & 7u) + 1;
            }
            valid = (lane & 7) < cnt;
            cell = (e >> 3) + (uint32_t)(lane & 7);
        } else {
        __syncwarp();
        // ---- pop as many runs as fit into 32 lanes ----
        const int navail = min(sp, 32);
        uint32_t e = 0;
        int cnt = 0;
        if (lane < navail) {
            e = S.stack[sp - 1 - lane];
            cnt = (int)(e & 7u) + 1;
        }
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += y;
        }
        const bool take_run = (lane < navail) && (incl <= 32);
        const int k_taken = __popc(__ballot_sync(0xFFFFFFFFu, take_run));
        const int total = __shfl_sync(0xFFFFFFFFu, incl, k_taken - 1);
        sp -= k_taken;
        const uint32_t startbits = __reduce_or_sync(0xFFFFFFFFu, take_run ? (1u << (incl - cnt)) : 0u);
        const int j = __popc(startbits & (0xFFFFFFFFu >> (31 - lane))) - 1;
        const uint32_t ej = __shfl_sync(0xFFFFFFFFu, e, j);
        const int exj = __shfl_sync(0xFFFFFFFFu, incl - cnt, j);
        valid = lane < total;
        cell = (ej >> 3) + (uint32_t)(lane - exj);
        }
        // ---- opening test (R9), every operation rounded once, in this order ----
        bool accept = false, leaf = false;
        uint32_t link_first = 0, info = 0;
        float4 m0 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (valid) {
            const float4* m = reinterpret_cast<const float4*>(a.mac + cell);
            m0 = __ldg(m);
            const float4 m1 = __ldg(m + 1);
            const float dx = fmaxf(0.0f, fmaxf(__fsub_rn(bmin[0], m0.x), __fsub_rn(m0.x, bmax[0])));
            const float dy = fmaxf(0.0f, fmaxf(__fsub_rn(bmin[1], m0.y), __fsub_rn(m0.y, bmax[1])));
            const float dz = fmaxf(0.0f, fmaxf(__fsub_rn(bmin[2], m0.z), __fsub_rn(m0.z, bmax[2])));
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const float rc = __fmaf_rn(m1.y, a.inv_theta, m1.x);
            const float rc2 = __fmul_rn(rc, rc);
            accept = d2 > rc2;
            link_first = __float_as_uint(m1.z);
            info = __float_as_uint(m1.w);
            leaf = (info & kLeafBit) != 0u;
        }
        // ---- rejected internal cells: push their child runs ----
        const bool open = valid && !accept && !leaf;
        const uint32_t om = __ballot_sync(0xFFFFFFFFu, open);
        if constexpr (kTeam) {
            if (lane == 0) T[1 + slot] = (uint32_t)__popc(om);
            team_barrier(team, tsize);  // (B) every member has read its runs and published its count
            uint32_t off = 0, total = 0;
            for (int j = 0; j < tsize; ++j) {
                const uint32_t v = T[1 + j];
                if (j < slot) off += v;
                total += v;
            }
            const uint32_t base = (uint32_t)(sp - take);
            if (base + total > team_cap) { ok = false; break; }  // the same decision in every member
            if (open) team_stack(base + off + (uint32_t)__popc(om & lt)) = (link_first << 3) | (info - 1u);
            if (slot == 0 && lane == 0) T[0] = base + total;
            sp = (int)(base + total);
        } else {
        if (open) {
            const int pos = sp + __popc(om & lt);
            if (pos < kWalkStack) S.stack[pos] = (link_first << 3) | (info - 1u);
        }
        sp += __popc(om);
        if (sp > kWalkStack) { ok = false; break; }
        }
        // ---- accepted cells ----
        const bool acc = valid && accept;
        const uint32_t am = __ballot_sync(0xFFFFFFFFu, acc);
        if constexpr (kMono) {
            if (am) {
                if (acc) {
                    const uint32_t slot_w = pp_w + __popc(am & lt);
                    if (!kTeam || ((slot_w >> 5) & tmask) == uslot) {  // (COM, M)
                        if constexpr (NS == 1) pp_put_pairs(S, slot_w, m0);
                        else S.pp[slot_w & 63u] = m0;
                    }
                }
                pp_w += __popc(am);
                npc += __popc(am);
                __syncwarp();
                if (pp_w - pp_r >= 32u) {
                    if (!kTeam || ((pp_r >> 5) & tmask) == uslot) eval_pp<NS, kZeroEps>(S, pp_r, 32, a.eps2, lane, s);
                    pp_r += 32u;
                }
            }
        } else {
        if (acc) S.pc_ids[(pc_w + __popc(am & lt)) & 63u] = cell;
        pc_w += __popc(am);
        npc += __popc(am);
        __syncwarp();
        if (pc_w - pc_r >= 32u) {
            if (!kTeam || ((pc_r >> 5) & tmask) == uslot) eval_pc<NS>(S, a, pc_r, 32, lane, s);
            pc_r += 32u;
        }
        }
        // ---- rejected leaves: expand into particles ----
        const bool oleaf = valid && !accept && leaf;
        const uint32_t lm = __ballot_sync(0xFFFFFFFFu, oleaf);
        if (lm) {
            const uint32_t lc = oleaf ? (info & ~kLeafBit) : 0u;
            uint32_t lincl = lc;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, lincl, o);
                if (lane >= o) lincl += y;
            }
            const uint32_t T = __shfl_sync(0xFFFFFFFFu, lincl, 31);
            if (oleaf) {
                const int r = __popc(lm & lt);
                S.leaf_first[r] = link_first;
                S.leaf_pref[r] = lincl - lc;
            }
            __syncwarp();
            npp += T;
            const uint32_t lpre = lincl - lc;  // first particle slot of this lane's leaf (oleaf lanes)
            for (uint32_t base = 0; base < T; base += 32u) {
                const uint32_t t = base + lane;
                // which leaf does slot t belong to?  Leaves are non-empty, so their first slots are distinct: one bit
                // per leaf starting inside this batch, and the rank of slot t's leaf = (leaves starting before the
                // batch) + (start bits at or below the lane) - 1.
                const uint32_t off = lpre - base;  // wraps for leaves that start before the batch
                const uint32_t starts = __reduce_or_sync(0xFFFFFFFFu, (oleaf && off < 32u) ? (1u << off) : 0u);
                const int before = __popc(__ballot_sync(0xFFFFFFFFu, oleaf && lpre < base));
                if (t < T) {
                    const int r = before + __popc(starts & (0xFFFFFFFFu >> (31 - lane))) - 1;
                    if (!kTeam || (((pp_w + lane) >> 5) & tmask) == uslot) {  // only the batches this member evaluates
                        const float4 src = __ldg(&a.pos[S.leaf_first[r] + (t - S.leaf_pref[r])]);
                        if constexpr (NS == 1) pp_put_pairs(S, pp_w + lane, src);
                        else S.pp[(pp_w + lane) & 63u] = src;
                    }
                }
                pp_w += min(32u, T - base);
                __syncwarp();
                if (pp_w - pp_r >= 32u) {
                    if (!kTeam || ((pp_r >> 5) & tmask) == uslot) eval_pp<NS, kZeroEps>(S, pp_r, 32, a.eps2, lane, s);
                    pp_r += 32u;
                }
            }
        }
    }
    if (!ok) return false;  // the same decision in every member of a team
    __syncwarp();
    if (pc_w != pc_r && (!kTeam || ((pc_r >> 5) & tmask) == uslot)) eval_pc<NS>(S, a, pc_r, (int)(pc_w - pc_r), lane, s);
    if (pp_w != pp_r && (!kTeam || ((pp_r >> 5) & tmask) == uslot))
        eval_pp<NS, kZeroEps>(S, pp_r, (int)(pp_w - pp_r), a.eps2, lane, s);
    if constexpr (NS == 1) {  // lane split: add the replicas' partial sums (every replica ends with the same bits)
        for (uint32_t o = split_m; o < 32u; o <<= 1) {
            s.ax[0] += __shfl_xor_sync(0xFFFFFFFFu, s.ax[0], o);
            s.ay[0] += __shfl_xor_sync(0xFFFFFFFFu, s.ay[0], o);
            s.az[0] += __shfl_xor_sync(0xFFFFFFFFu, s.az[0], o);
            s.ph[0] += __shfl_xor_sync(0xFFFFFFFFu, s.ph[0], o);
        }
    }
    if (kTeam) {
        // fold the members' partial sums: each member parks its 4 NS doubles per lane in its own source rings
        // (dead now), member 0 adds them in member order
        static_assert(sizeof(S.pp) + sizeof(S.pc) >= 2 * 4 * 32 * sizeof(double), "partials do not fit the rings");
        __syncwarp();
        if (slot != 0) {
            double* park = reinterpret_cast<double*>(S.pp);
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                park[(4 * k + 0) * 32 + lane] = s.ax[k];
                park[(4 * k + 1) * 32 + lane] = s.ay[k];
                park[(4 * k + 2) * 32 + lane] = s.az[k];
                park[(4 * k + 3) * 32 + lane] = s.ph[k];
            }
            if (lane == 0) {  // this member's share of the lists
                S.leaf_first[0] = npc;
                S.leaf_first[1] = npp;
            }
        }
        team_barrier(team, tsize);  // every member's partials are parked
        if (slot == 0)
        for (int j = 1; j < tsize; ++j) {
            const double* park = reinterpret_cast<const double*>((&S)[j].pp);
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                s.ax[k] += park[(4 * k + 0) * 32 + lane];
                s.ay[k] += park[(4 * k + 1) * 32 + lane];
                s.az[k] += park[(4 * k + 2) * 32 + lane];
                s.ph[k] += park[(4 * k + 3) * 32 + lane];
            }
            npc += (&S)[j].leaf_first[0];
            npp += (&S)[j].leaf_first[1];
        }
        team_barrier(team, tsize);  // ... and consumed: the rings are free for the next chunk
        if (slot != 0) return true;
    }
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        if (lane + 32u * k < ns) {
            double ph = s.ph[k];
            if (!kZeroEps) ph -= (double)(smass[k] * rsqrt_fast(a.eps2));  // the self term, bit for bit as it was added
            const uint32_t dst = __ldg(&a.perm[sidx[k]]);
            a.out[dst] = make_float4((float)s.ax[k], (float)s.ay[k], (float)s.az[k], (float)(-ph));
            a.n_pp[dst] = npp - 1u;
            a.n_pc[dst] = npc;
        }
    }
    if (lane == 0) {
        atomicAdd(&a.ctl->sum_pp, (unsigned long long)ns * (npp - 1u));
        atomicAdd(&a.ctl->sum_pc, (unsigned long long)ns * npc);
    }
    return true;
}

template <bool kZeroEps, bool kTeam, bool kMono>
__device__ __forceinline__ void walk_groups(WarpSmem& S, const WalkArgs& a, uint32_t n_groups, int lane, int w, int tsize,
                                            uint32_t* s_team_g) {
    const int team = kTeam ? w / tsize : w, slot = kTeam ? w % tsize : 0;
    for (;;) {
        uint32_t g = 0;
        if (kTeam) {
            if (slot == 0 && lane == 0) s_team_g[team] = atomicAdd(&a.ctl->walk_ticket, 1u);
            team_barrier(team, tsize);
            g = s_team_g[team];
            team_barrier(team, tsize);  // everybody has read it before member 0 can draw the next ticket
        } else {
            if (lane == 0) g = atomicAdd(&a.ctl->walk_ticket, 1u);
            g = __shfl_sync(0xFFFFFFFFu, g, 0);
        }
        if (g >= n_groups) break;
        const uint32_t gf = __ldg(&a.g_first[g]), gc = __ldg(&a.g_count[g]);
        float bmin[3], bmax[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bmin[k] = __ldg(&a.g_bmin[3 * g + k]);
            bmax[k] = __ldg(&a.g_bmax[3 * g + k]);
        }
        // a group larger than 64 (only a level-30 leaf of coincident keys, or nleaf > ncrit) is walked in chunks
        // of 64 sinks that all use the group's box, hence the same lists
        for (uint32_t c0 = 0; c0 < gc; c0 += 64u) {
            const uint32_t ns = min(64u, gc - c0);
            bool ok;
            if (ns > 32u) ok = walk_chunk<2, kZeroEps, kTeam, kMono>(S, a, lane, gf + c0, ns, bmin, bmax, team, slot, tsize);
            else ok = walk_chunk<1, kZeroEps, kTeam, kMono>(S, a, lane, gf + c0, ns, bmin, bmax, team, slot, tsize);
            if (!ok && lane == 0) a.ctl->status = BONSAI_ECAPACITY;
            __syncwarp();
        }
    }
}

// Cost model of a team configuration: with dynamic tickets a walk lasts about ceil(n_groups S / warps) rounds of one
// group-walk each, and a team of S shortens a group-walk to ~(0.05 + 0.95 / S) of a single warp's.  Returns the
// cheapest S <= max_team (the smaller one on near-ties) and its cost.
__device__ __forceinline__ int best_team(uint32_t n_groups, uint32_t warps, int max_team, float* cost_out) {
    int tsize = 1;
    float best = 3.0e38f;
    for (int ts = 1; ts <= max_team; ts *= 2) {
        const float rounds = (float)(((unsigned long long)n_groups * ts + warps - 1) / warps);
        const float cost = rounds * (0.05f + 0.95f / (float)ts);
        if (cost < 0.95f * best) { best = cost; tsize = ts; }
    }
    *cost_out = best;
    return tsize;
}

// kTeams = false: the plain one-warp-per-group kernel (all particles active: always enough groups).
// kTeams = true: launched for masked walks and small systems; picks the team size from the number of groups on the
// device.  Two instances are launched back to back, blocks of 8 warps (3 per SM) and blocks of 16 warps (1 per SM,
// teams of up to 16); both evaluate the same cost model on the same group count, the cheaper one does the walk, the
// other returns at once.
template <bool kZeroEps, bool kTeams, bool kMono, int kWarps>
__global__ void __launch_bounds__(kWarps * 32, kWarps == kWalkWarps ? 3 : 1) k_walk(WalkArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_team_g[kWarps];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    WarpSmem& S = reinterpret_cast<WarpSmem*>(smem_raw)[w];
    const uint32_t n_groups = a.ctl->n_groups;
    // after a cell-capacity overflow in the build the child links of the tree point past the arrays: do not follow them
    // (one read per block: the walk itself may raise the status later, and a team must not split over it)
    __shared__ int s_status;
    if (threadIdx.x == 0) s_status = a.ctl->status;
    __syncthreads();
    if (s_status != 0) return;
    if constexpr (kTeams) {
        float cost_small, cost_big;
        const int t_small = best_team(n_groups, a.warps_small, kWalkWarps, &cost_small);
        const int t_big = best_team(n_groups, a.warps_big, kWalkWarpsBig, &cost_big);
        const bool big_wins = cost_big < 0.9f * cost_small;
        if (big_wins != (kWarps == kWalkWarpsBig)) return;
        const int tsize = big_wins ? t_big : t_small;
        if (tsize > 1) {
            walk_groups<kZeroEps, true, kMono>(S, a, n_groups, lane, w, tsize, s_team_g);
            return;
        }
    }
    walk_groups<kZeroEps, false, kMono>(S, a, n_groups, lane, w, 1, s_team_g);
}

using WalkKernel = void (*)(WalkArgs);
// index = (eps == 0) + 2 (team-capable) + 4 (monopole only)
static const WalkKernel kWalkKernels[8] = {k_walk<false, false, false, kWalkWarps>, k_walk<true, false, false, kWalkWarps>,
                                           k_walk<false, true, false, kWalkWarps>,  k_walk<true, true, false, kWalkWarps>,
                                           k_walk<false, false, true, kWalkWarps>,  k_walk<true, false, true, kWalkWarps>,
                                           k_walk<false, true, true, kWalkWarps>,   k_walk<true, true, true, kWalkWarps>};
// the 16-warp team kernels: index = (eps == 0) + 2 (monopole only)
static const WalkKernel kWalkKernelsBig[4] = {k_walk<false, true, false, kWalkWarpsBig>, k_walk<true, true, false, kWalkWarpsBig>,
                                              k_walk<false, true, true, kWalkWarpsBig>,  k_walk<true, true, true, kWalkWarpsBig>};

// Kernel attributes are per device (and cheap to set again): done for every context at creation, so a second
// device or a second host thread in the same process never launches without the dynamic shared memory opt-in.
cudaError_t walk_prepare(Ctx* c) {
    const size_t smem = walk_smem_bytes(c->prm.nleaf);
    cudaError_t e;
    for (int k = 0; k < 8; ++k) {
        if ((e = cudaFuncSetAttribute(kWalkKernels[k], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->walk_blocks_per_sm[k], kWalkKernels[k], kWalkWarps * 32, smem)) != cudaSuccess) return e;
        if (c->walk_blocks_per_sm[k] < 1) c->walk_blocks_per_sm[k] = 1;
    }
    for (int k = 0; k < 4; ++k)
        if ((e = cudaFuncSetAttribute(kWalkKernelsBig[k], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)(sizeof(WarpSmem) * kWalkWarpsBig))) != cudaSuccess) return e;
    return cudaSuccess;
}

cudaError_t stage_walk(Ctx* c, float theta, float eps, float4* acc_pot_out) {
    Buffers& b = c->b;
    WalkArgs a;
    a.ctl = b.ctl;
    a.mac = b.c_mac;
    a.quad = b.c_quad;
    a.pos = b.sorted_pos;
    a.perm = c->perm;
    a.active_list = c->groups_all_active ? nullptr : b.active_list;
    a.g_first = b.g_first;
    a.g_count = b.g_count;
    a.g_bmin = b.g_bmin;
    a.g_bmax = b.g_bmax;
    a.inv_theta = 1.0f / theta;  // IEEE fp32 division on the host; theta = 0 -> +inf -> nothing is accepted
    a.eps2 = eps * eps;
    a.out = acc_pot_out;
    a.n_pp = b.n_pp;
    a.n_pc = b.n_pc;
    const size_t smem = walk_smem_bytes(c->prm.nleaf);
    cudaError_t e;
    // reset the ticket and the interaction totals (adjacent fields of the control block)
    if ((e = cudaMemsetAsync(&b.ctl->walk_ticket, 0, sizeof(uint32_t), c->stream)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&b.ctl->sum_pp, 0, 2 * sizeof(unsigned long long), c->stream)) != cudaSuccess) return e;
    // a masked walk, or a small system, may have fewer groups than resident warps: the team-capable kernel adapts on
    // the device; n / ncrit is a lower bound of the all-active group count known on the host (measured at
    // N = 2^17 / 2^18 / 2^19: teams 0.41 / 0.75 / 1.26 ms against 0.55 / 0.72 / 1.27 ms for the plain kernel, so the
    // team kernel is taken up to one group per resident warp)
    const unsigned long long resident_warps = (unsigned long long)c->num_sms * c->walk_blocks_per_sm[2] * kWalkWarps;
    const bool few_groups = !c->groups_all_active || c->n / c->prm.ncrit <= resident_warps;
    const int which = ((a.eps2 == 0.0f) ? 1 : 0) + (few_groups ? 2 : 0) + (c->prm.order == 1 ? 4 : 0);
    const int grid = c->num_sms * c->walk_blocks_per_sm[which];
    a.warps_small = (uint32_t)grid * kWalkWarps;
    a.warps_big = (uint32_t)c->num_sms * kWalkWarpsBig;
    kWalkKernels[which]<<<grid, kWalkWarps * 32, smem, c->stream>>>(a);
    c->launches += 1;
    if (few_groups) {  // the 16-warp instance: does the walk instead when teams of 16 pay (see k_walk)
        const int big = ((a.eps2 == 0.0f) ? 1 : 0) + (c->prm.order == 1 ? 2 : 0);
        kWalkKernelsBig[big]<<<c->num_sms, kWalkWarpsBig * 32, sizeof(WarpSmem) * kWalkWarpsBig, c->stream>>>(a);
        c->launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace bonsai
