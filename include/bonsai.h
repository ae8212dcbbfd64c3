/* =====================================================================================
 * libbonsai -- C-ABI boundary of the B200-native Barnes-Hut force step.
 *
 * Method: "Bonsai: A GPU Tree-Code" (arXiv 1204.2280), cited as P:Lnn = line nn of the
 * paper text.  The five timed sections of the paper (Results: "Sorting of
 * the particles along a Space Filling Curve", "reordering of the particle properties
 * ('moving')", "construction of the tree-datastructure", "computation of the multipole
 * moments", "tree-traverse") map onto the calls below.  "All parts of the algorithm are
 * executed on the GPU" (Abstract): every pointer documented "device" below is a
 * CUDA device pointer and the host only sequences stages.  No call copies particle data
 * between host and device, with ONE exception that exists for end-to-end measurement and
 * for callers without device buffers: bonsai_step_host() (host pointers in and out, copies
 * inside).  The paper states no formula or constant; the exact arithmetic of every stage
 * is the set of readings R1..R31 in DESIGN.md.
 *
 * Conventions
 *   - All calls return an int: 0 (BONSAI_OK) or a negative BONSAI_E* code.  No exceptions, no
 *     aborts, no output on stdout/stderr.
 *   - All work is enqueued on the CUDA stream passed to bonsai_create() and the calls return
 *     without waiting for it, except bonsai_sync() and bonsai_get_stage_ms().
 *   - Memory: the CALLER owns every buffer (particles, masks, outputs and the workspace); the
 *     library never allocates device memory.  The workspace must stay alive and untouched
 *     between bonsai_create() and bonsai_destroy().  Device pointers handed out by the
 *     bonsai_get_* calls point into the workspace and are valid until the next
 *     bonsai_build_tree()/bonsai_walk() that rewrites them, or bonsai_destroy().
 *   - "sorted order" = Morton order produced by bonsai_build_tree(); "load order" = the order of
 *     the array given to bonsai_load().
 * ===================================================================================== */
#ifndef BONSAI_H_
#define BONSAI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BONSAI_OK          0
#define BONSAI_EINVAL     (-1)  /* null / misaligned pointer, n = 0, n > n_max, bad parameter, NaN        */
#define BONSAI_ESTATE     (-2)  /* call out of order (e.g. walk before multipoles)                        */
#define BONSAI_ECAPACITY  (-3)  /* more cells than cap_cells, or traversal stack overflow (sticky, device) */
#define BONSAI_ECUDA      (-4)  /* a CUDA runtime call failed                                             */
#define BONSAI_ENOMEM     (-5)  /* workspace smaller than bonsai_workspace_bytes()                        */

#define BONSAI_THETA_MAX   1.15f /* R9/R11: largest opening angle accepted; below 2/sqrt(3) a sink's own leaf is
                                    always opened, which the arithmetic removal of the self term relies on      */
#define BONSAI_MAX_LEVEL   30   /* R1: 30 bits per axis, 90-bit Morton key (BASELINE.json north_star)     */
#define BONSAI_N_STAGES    9

typedef struct bonsai_ctx bonsai_ctx; /* opaque, host memory, owned by the library */

/* Tunables.  A zeroed field takes the default in brackets. */
typedef struct {
    uint32_t nleaf;      /* [16] a cell with <= nleaf particles is a leaf (R7); 1..64                        */
    uint32_t ncrit;      /* [64] maximum particles per walk group (R13); 1..64                               */
    uint32_t group_mode; /* 0 = tree-cell groups, 1 = consecutive sorted chunks, 2 = chunks of ncrit inside the
                            cells with <= group_cell particles [2] (R13).  NOTE: because 0 is a legal value,
                            group_mode is only defaulted when params == NULL.                                 */
    uint32_t cap_cells;  /* [2 n_max + 256] capacity of the cell arrays                                      */
    uint32_t group_cell; /* [512]  mode 2: a group never crosses the boundary of a cell holding more than
                            group_cell particles (the containers are the cells with count <= group_cell whose
                            parent has more); >= ncrit                                                        */
    uint32_t mac_mode;   /* [0] size and centre of a cell in the opening test ("MAC"): 0 = geometric cell
                            (side l = root side / 2^level, geometric centre; R9), 1 = tight: the exact bounding box
                            of the cell's particles, l_t = its longest side, centre = its midpoint (R28)         */
    uint32_t order;      /* [2] multipole order of a particle-cell interaction: 2 = monopole + quadrupole (R8),
                            1 = monopole only (R29); 0 = default                                                */
    uint32_t no_graph;   /* [0] 1 = bonsai_step / bonsai_leapfrog_step enqueue their kernels one by one; 0 = they
                            are captured as a CUDA graph and replayed while buffers and parameters repeat         */
    float rebuild_factor;/* [1.25] bonsai_block_tick(rebuild = -1) rebuilds the tree when the interactions per
                            walked sink of the last walk exceed rebuild_factor x those of the first walk after the
                            last build (R30); >= 1                                                       */
    uint32_t mult_kernel;/* [0] which of the two multipole kernels runs (same results to the last bit of the fp64 sums'
                            rounding order within a cell): 0 = by size (tiles from n = 2^21), 1 = the last child to
                            arrive climbs (small systems), 2 = tiles of cells deepest first, parents wait            */
    uint32_t sort_passes;/* [0] radix passes of the key sort (a2): 4, 5 or 6 passes of 10 bits over the leading 40, 50 or 60
                            key bits; particles that agree in those are put in order of their remaining bits after the
                            reorder (the permutation is the same bit for bit).  0 = by size: 4 up to n = 2^23, 5 up to
                            2^25, else 6 (a strongly clustered system wants more passes)                             */
} bonsai_params;

/* Bytes of device workspace bonsai_create() needs for up to n_max particles (0 on bad arguments). */
size_t bonsai_workspace_bytes(uint32_t n_max, const bonsai_params* params);

/* Create a context for up to n_max particles.
 *   params         host pointer or NULL (all defaults, group_mode = 2)
 *   workspace_dev  device pointer, 256-byte aligned, >= bonsai_workspace_bytes() bytes, caller-owned
 *   cuda_stream    a cudaStream_t (NULL = the legacy default stream)
 *   out            host pointer receiving the context
 * Zero-fills the control block of the workspace on the stream.  EINVAL / ENOMEM / ECUDA. */
int bonsai_create(uint32_t n_max, const bonsai_params* params, void* workspace_dev, size_t workspace_bytes,
                  void* cuda_stream, bonsai_ctx** out);

/* Hand the particles of this step to the library (particle arrays live on the device).
 *   pos_mass_dev   device, float4[n] = (x, y, z, m), 16-byte aligned, load order.  NOT copied: it is read by
 *                  bonsai_build_tree() (bounding box, keys, reorder) and must stay valid and unchanged until
 *                  that call has completed on the stream.  Finite positions and m >= 0 are preconditions.
 *   n              1 .. n_max
 * Invalidates tree, multipoles and walk results.  EINVAL. */
int bonsai_load(bonsai_ctx* ctx, const float* pos_mass_dev, uint32_t n);

/* Stages a0..a4' ("sorting", "moving", "construction of the tree-datastructure"):
 *   bounding box -> root cube (R3); 90-bit Morton keys (R1, R2, R4); stable radix sort of (key, index) (R5);
 *   reorder of pos_mass into sorted order; octree over the sorted keys (R7: leaf <=> count <= nleaf or level 30,
 *   sparse, chains kept, breadth-first numbering); walk groups over all particles with exact fp32 boxes (R13).
 * ESTATE if nothing is loaded.  A cell overflow sets the sticky ECAPACITY flag reported by bonsai_sync(). */
int bonsai_build_tree(bonsai_ctx* ctx);

/* Stage a5 ("computation of the tree-properties (multipole moments)"): per cell the mass, centre
 * of mass, the 6 raw second moments about the centre of mass (xx, yy, zz, xy, xz, yz), delta = |COM - geometric
 * centre| and the cell side l (R8).  Accumulated in fp64, stored rounded once to fp32.  ESTATE before build. */
int bonsai_compute_multipoles(bonsai_ctx* ctx);

/* Stage a6 / a7 ("tree-traverse"): for every group, traverse from the root with the opening
 * criterion  d2 > (l / theta + delta)^2  evaluated in fp32 exactly as R9 orders it (d = distance from the group's
 * box to the cell's COM); accepted cells act on every particle of the group as monopole + quadrupole
 * (particle-cell), rejected leaves particle by particle, with Plummer softening eps in every power of r (R10).
 *   0 <= theta <= BONSAI_THETA_MAX (0 = open everything = direct summation through the tree; above 2/sqrt(3) a
 *   cell containing a sink could be accepted, see R9), eps >= 0 and finite
 *   active_mask_dev  device u8[n] in LOAD order, or NULL = all particles are sinks.  A non-NULL mask rebuilds
 *                    the group list over the active particles for this call (R13, R19); all particles stay
 *                    sources.  Must stay valid until the call completed on the stream.
 *   acc_pot_dev_out  device float4[n] = (ax, ay, az, phi), load order, 16-byte aligned.  G = 1; phi is the
 *                    potential per unit mass with the self term excluded (R11, R12).  Only entries of active
 *                    particles are written.
 * Per-particle interaction counts are kept for bonsai_get_counts().  EINVAL, ESTATE before multipoles. */
int bonsai_walk(bonsai_ctx* ctx, float theta, float eps, const uint8_t* active_mask_dev, float* acc_pot_dev_out);

/* One full force step = bonsai_load, bonsai_build_tree, bonsai_compute_multipoles, bonsai_walk (arguments as
 * there), as ONE call.  Unless params.no_graph is set or stage timing is on, the sequence is captured as a CUDA graph
 * the first time a combination (pos_mass_dev, n, theta, eps, active_mask_dev, acc_pot_dev_out) is seen -- on a stream
 * the library owns, so the caller's stream may be the legacy default stream -- and replayed with one graph launch
 * from then on (the four most recent combinations are kept): below ~10^5 particles a step is bound by launch gaps
 * (P:L32).  The replay enqueues exactly the kernels of the staged calls; results are bit-identical.  The graph reads
 * the buffers, not a snapshot of them: new particle data in the same buffers needs no new capture.  A caller that
 * passes different buffers on every call gains nothing (after 16 misses in a row the next 256 calls are enqueued kernel
 * by kernel, then capturing is tried again).
 * EINVAL / ESTATE / ECUDA as the staged calls. */
int bonsai_step(bonsai_ctx* ctx, const float* pos_mass_dev, uint32_t n, float theta, float eps,
                const uint8_t* active_mask_dev, float* acc_pot_dev_out);

/* One full force step for a caller whose particles live in HOST memory (the end-to-end path of bench.py):
 * copies pos_mass_host (float4[n]; pinned memory recommended) to a staging buffer in the workspace, runs
 * bonsai_load .. bonsai_walk exactly as above, copies acc_pot (float4[n], load order) back and WAITS for the
 * stream.  active_mask_host: host u8[n] or NULL; with a mask, entries of inactive particles are returned unchanged.
 * Both directions are staged through the workspace (one copy each way, 16 n bytes each).
 * Returns what bonsai_sync() returns, or EINVAL / ECUDA. */
int bonsai_step_host(bonsai_ctx* ctx, const float* pos_mass_host, uint32_t n, float theta, float eps,
                     const uint8_t* active_mask_host, float* acc_pot_host_out);

/* Release the context (host memory only; the workspace belongs to the caller).  NULL is allowed. */
void bonsai_destroy(bonsai_ctx* ctx);

/* Wait for the stream and return the sticky device status (OK / ECAPACITY) or ECUDA.  The status covers the work
 * enqueued since the last bonsai_build_tree(): that call clears it (and repairs the internal counters an overflow
 * leaves behind), so one failed step does not poison the context. */
int bonsai_sync(bonsai_ctx* ctx);

/* ---- introspection (parity tests and reporting).  All pointers returned are DEVICE pointers. ---- */

/* Root cube on the device: float[4] = (lo_x, lo_y, lo_z, side) (R3; side is a power of two). */
int bonsai_get_box(bonsai_ctx* ctx, const float** box4_dev);

/* Sorted keys, one u32 array per 30-bit word: hi = levels 1-10, mid = 11-20, lo = 21-30 (R1). */
int bonsai_get_keys(bonsai_ctx* ctx, const uint32_t** hi_dev, const uint32_t** mid_dev, const uint32_t** lo_dev);

/* perm[i] = load index of the i-th sorted particle; sorted pos_mass float4[n]. */
int bonsai_get_perm(bonsai_ctx* ctx, const uint32_t** perm_dev);
int bonsai_get_sorted_pos(bonsai_ctx* ctx, const float** pos_mass_dev);

typedef struct {
    uint32_t cap_cells;
    const uint32_t* n_cells;       /* device u32[1]                                                     */
    const uint32_t* level_offsets; /* device u32[32]: first cell of level L, [31] = n_cells             */
    const uint32_t* level;         /* device u32[cap] each, structure of arrays (R7)                    */
    const uint32_t* first;         /*   first sorted particle                                           */
    const uint32_t* count;         /*   number of particles                                             */
    const uint32_t* first_child;   /*   0 for a leaf                                                    */
    const uint32_t* n_child;       /*   0 for a leaf                                                    */
    const uint32_t* parent;        /*   0xFFFFFFFF for the root                                         */
    const float* mac;              /* device, 8 x 4 bytes per cell (after multipoles; the walk's layout):
                                      f32 COM x, y, z, mass, delta = |COM - geometric centre|, l = cell side,
                                      then u32 link (leaf: first particle; else first child) and u32 info
                                      (leaf: 0x80000000 | count; else n_child)                                */
    const float* quad;             /* device, 6 floats per cell: xx, yy, zz, xy, xz, yz (raw second moments
                                      about the COM, R8); filled by bonsai_get_cells() itself (one small
                                      kernel on the stream), valid after bonsai_compute_multipoles()        */
    const float* walk_quad;        /* device, 8 floats per cell, the walk's second record: P = tr I - 3 Q as
                                      Pxx, Pyy, Pzz, Pxy, Pxz, Pyz, then tr = Qxx + Qyy + Qzz and a pad      */
} bonsai_cells_view;
int bonsai_get_cells(bonsai_ctx* ctx, bonsai_cells_view* out);

typedef struct {
    const uint32_t* n_groups;    /* device u32[1]                                                       */
    const uint32_t* n_active;    /* device u32[1]                                                       */
    const uint32_t* active_list; /* device u32[n_active]: sorted index of the k-th active particle      */
    const uint32_t* first;       /* device u32[n_groups]: offset into active_list                       */
    const uint32_t* count;       /* device u32[n_groups]                                                */
    const float* bmin;           /* device float[3*n_groups]                                            */
    const float* bmax;           /* device float[3*n_groups]                                            */
} bonsai_groups_view;
/* The group list of the last bonsai_build_tree() (all active) or of the last masked bonsai_walk(). */
int bonsai_get_groups(bonsai_ctx* ctx, bonsai_groups_view* out);

/* Interaction counts of the last walk, per particle in LOAD order (R21): n_pp = particles in the opened
 * leaves of the particle's group minus itself, n_pc = accepted cells of its group. */
int bonsai_get_counts(bonsai_ctx* ctx, const uint32_t** n_pp_dev, const uint32_t** n_pc_dev);

/* Totals of the last walk over all sinks: sum of n_pp and of n_pc (R21).  Waits for the stream. */
int bonsai_get_interaction_totals(bonsai_ctx* ctx, uint64_t* sum_pp, uint64_t* sum_pc);

/* Re-use the sorted order and the tree of the last bonsai_build_tree() after the particles have moved (P:L52:
 * sorting, moving and tree-construction "do not have to be executed during each time-step when using the block
 * time-step method. It is sufficient to only recompute the multipole moments ..."; reading R25 of DESIGN.md).
 * The array given to bonsai_load() must hold the SAME particles in the SAME load order as at the last build, with
 * new positions (e.g. after bonsai_drift()).  Keeps permutation, keys, cells, links, geometric centres and group
 * membership; re-gathers the particles into sorted order and recomputes the group boxes.  The next
 * bonsai_compute_multipoles() then recomputes every moment from the new positions and lets the cell side that
 * enters the opening test grow to the extent of the cell's members:
 *     l' = max(l, 2 max_i max_a |x_ia - g_a|)   (fp64, rounded once).
 * Forces stay valid Barnes-Hut forces for the new positions; the interaction count grows with the drift, and the
 * caller decides when to rebuild (bonsai_get_interaction_totals()).  ESTATE when no tree for this n exists. */
int bonsai_refresh_tree(bonsai_ctx* ctx);

/* ---- Time integration around the force step (DESIGN.md row f2) ----------------------------------------
 * The paper integrates with "the block time-step method" (P:L24 Introduction; P:L32 Results: only "particles
 * that have to be updated" are walked) and states no scheme; BASELINE.json configs[2] fixes leapfrog steps with
 * a shared time-step and the tree rebuilt every step.  Readings R22 (kick-drift-kick), R23 (fp32 state, each
 * component updated by ONE fused multiply-add rounded once), R24 (diagnostics) of DESIGN.md.
 *
 * All arrays are device, 16-byte aligned float4[n] in LOAD order, caller-owned:
 *   pos_mass (x, y, z, m)   vel (vx, vy, vz, unused -- carried through)   acc_pot (ax, ay, az, phi) as bonsai_walk
 *   writes it.  n <= n_max.  Asynchronous on the context's stream.  EINVAL on null / misaligned / n / non-finite step. */

/* Kick: vel[i].xyz = fma(acc_pot[i].xyz, step, vel[i].xyz) for every i whose mask byte is non-zero (all i when
 * active_mask_dev is NULL; u8[n], load order -- the same mask bonsai_walk takes, R19). */
int bonsai_kick(bonsai_ctx* ctx, float* vel_dev, const float* acc_pot_dev, uint32_t n, float step,
                const uint8_t* active_mask_dev);

/* Drift: pos_mass[i].xyz = fma(vel[i].xyz, step, pos_mass[i].xyz); masses untouched; every particle drifts.
 * If pos_mass_dev is the array given to bonsai_load(), the context falls back to the "loaded" state: the tree no
 * longer matches the positions and bonsai_build_tree() must run before the next walk (ESTATE otherwise). */
int bonsai_drift(bonsai_ctx* ctx, float* pos_mass_dev, const float* vel_dev, uint32_t n, float step);

/* One kick-drift-kick step of size dt with a shared time-step (R22):
 *   vel += acc (dt/2);  pos += vel dt;  [load, build_tree, compute_multipoles, walk(theta, eps, all active)];
 *   vel += acc_new (dt/2).
 * On entry acc_pot_dev holds the force at the current positions (from a previous bonsai_walk or
 * bonsai_leapfrog_step); on return it holds the force at the new positions.  The opening kick and the drift run
 * as one fused pass with the same arithmetic as bonsai_kick followed by bonsai_drift. */
int bonsai_leapfrog_step(bonsai_ctx* ctx, float* pos_mass_dev, float* vel_dev, float* acc_pot_dev, uint32_t n,
                         float theta, float eps, float dt);

/* Diagnostics (R24), fp64 sums of the fp32 state, G = 1; writes 12 doubles to out12_dev (device, 8-byte aligned):
 *   [0] K = 1/2 sum m |v|^2   [1] W = 1/2 sum m phi   [2..4] P = sum m v   [5..7] L = sum m (x cross v)
 *   [8] M = sum m             [9..11] C = sum m x.
 * Deterministic for a given n (fixed reduction tree). */
int bonsai_diagnostics(bonsai_ctx* ctx, const float* pos_mass_dev, const float* vel_dev, const float* acc_pot_dev,
                       uint32_t n, double* out12_dev);

/* The same diagnostics (R24; the 12 sums documented at bonsai_diagnostics) for callers that CANNOT ALLOCATE device
 * memory: no context, no workspace.  bonsai_diagnostics() is only reachable through a context, and a context wants a
 * workspace of several hundred bytes per particle from the caller; a monitor that is hooked into a running
 * simulation whose memory pool is spent, a plug-in whose host forbids cudaMalloc, or a loop that must avoid the
 * device-wide synchronisation cudaMalloc / cudaFree can cause, has no such buffer to give.  This call needs only the
 * three particle arrays and the result buffer.  Its scratch (block partials + a ticket) is a fixed array inside the
 * library image:
 *     BONSAI_DIAG_STATIC_SCRATCH_BYTES = 113 920 bytes of device memory, held on EVERY GPU that loads libbonsai,
 *     from load until the process exits, used or not.
 * The call allocates nothing, on the host or on the device (no cudaMalloc / cudaFree / allocating library routine).
 *   pos_mass_dev, vel_dev, acc_pot_dev   device float4[n], 16-byte aligned, caller-owned, read only
 *   n            1 .. BONSAI_DIAG_STATIC_MAX_N (2^30, the ceiling bonsai_create puts on n_max; the kernel's 32-bit
 *                strided index is safe up to there).  Larger n, like n = 0, is refused with BONSAI_EINVAL before any
 *                CUDA call is made; the scratch itself (1184 rows, the grid cap) serves every n up to the limit.
 *   out12_dev    device double[12], 8-byte aligned, caller-owned, written by the kernel
 *   cuda_stream  a cudaStream_t of the CURRENT device (NULL = legacy default stream); asynchronous on it
 * Sharing.  All calls on a device share the one array and it keeps the last call's contents; the ticket is cleared on
 * the stream before each launch, the rows are rewritten before they are read.  Calls that may run on the GPU at the
 * same time (two streams, two threads) RACE on it and return wrong sums: keep them on one stream or order them
 * yourself.  Calls on different devices do not interfere.
 * First call.  The first call on each device resolves the array's device address (with that device current) and may
 * load the module while doing so; issue it once per device before any stream capture begins.
 * Result.  Same grid rule and summation order as bonsai_diagnostics(); deterministic for a given n.
 * EINVAL (null / misaligned / n out of range), ECUDA. */
#define BONSAI_DIAG_STATIC_MAX_N          (1u << 30)
#define BONSAI_DIAG_STATIC_SCRATCH_BYTES  113920u
int bonsai_diagnostics_static(const float* pos_mass_dev, const float* vel_dev, const float* acc_pot_dev, uint32_t n,
                              double* out12_dev, void* cuda_stream);

/* ---- Block time-steps (R26, R27; "block time-step algorithm", "N_active") -----------------
 * The paper states no criterion or scheme.  R26: particle i steps with dt_i = dt_max 2^-k_i, its rung k_i in
 * [0, kmax] the smallest k with dt_max 2^-k <= eta sqrt(eps / |a_i|) (fp64 on the fp32 acceleration).  Time is
 * counted in ticks of dt_min = dt_max 2^-kmax; i is active at tick t iff t mod 2^(kmax - k_i) == 0.  kmax <= 30.
 * rung / mask arrays are device u8[n] in load order, caller-owned.  Asynchronous on the context's stream. */

/* init != 0: rung[i] = R26 for every particle.  init == 0: the update at the end of a tick for the particles with
 * mask != 0 (NULL = all): a finer rung at once, a coarser one by one rung and only if `tick` is a multiple of the
 * coarser step (steps stay nested). */
int bonsai_timestep_rungs(bonsai_ctx* ctx, const float* acc_pot_dev, uint32_t n, float eta, float eps, float dt_max,
                          uint32_t kmax, const uint8_t* active_mask_dev, uint64_t tick, uint8_t* rung_dev, int init);

/* mask[i] = 1 if particle i is active at `tick`, else 0: the mask bonsai_walk / bonsai_kick_rungs take. */
int bonsai_active_mask(bonsai_ctx* ctx, const uint8_t* rung_dev, uint32_t n, uint32_t kmax, uint64_t tick,
                       uint8_t* mask_dev_out);

/* Half a step of each masked-in particle's own size: vel.xyz = fma(acc.xyz, dt_max 2^-(rung+1), vel.xyz) (R23). */
int bonsai_kick_rungs(bonsai_ctx* ctx, float* vel_dev, const float* acc_pot_dev, const uint8_t* rung_dev,
                      const uint8_t* active_mask_dev, uint32_t n, float dt_max);

/* One tick of the block scheme (R27), everything on the device, no host read-back:
 *   opening kick of the particles active at `tick`; drift of ALL particles by dt_min; force on the particles active
 *   at tick + 1 (masked walk) from a rebuilt (rebuild > 0) or refreshed (rebuild == 0, bonsai_refresh_tree) tree;
 *   closing kick of those; their new rungs.
 *   rebuild < 0: the library decides ON THE DEVICE (rebuild "only when the tree-traverse shows a considerable
 *   decline in performance"; R30): rebuild iff the interactions per walked sink of the previous tick's walk exceed
 *   params.rebuild_factor times those of the first tick after the last build; both kernel sequences are enqueued
 *   behind a device flag, the one not taken returns at once.  Without a tree for this array / n it rebuilds.
 * acc_pot_dev holds every particle's force at its last force time and is updated for the walked particles only.
 * With kmax = 0 this is bonsai_leapfrog_step.  ESTATE if rebuild == 0 and no tree for this array / n exists. */
int bonsai_block_tick(bonsai_ctx* ctx, float* pos_mass_dev, float* vel_dev, float* acc_pot_dev, uint8_t* rung_dev,
                      uint32_t n, uint64_t tick, float theta, float eps, float eta, float dt_max, uint32_t kmax,
                      int rebuild);

/* R30 bookkeeping of bonsai_block_tick: decisions taken and rebuilds decided on the device since bonsai_create,
 * the reference and the latest interactions per walked sink.  Any pointer may be NULL.  Waits for the stream. */
int bonsai_get_rebuild_stats(bonsai_ctx* ctx, uint32_t* n_decisions, uint32_t* n_rebuilds, double* ipp_ref,
                             double* ipp_last);

/* Per-stage device times.  bonsai_set_timing(ctx, 1) records CUDA events around every stage from then on;
 * bonsai_get_stage_ms() waits for the stream and writes, per stage, the milliseconds SUMMED over its executions
 * since the previous bonsai_get_stage_ms() (or bonsai_set_timing) call (any number of executions; every 9th execution of a
 * stage waits for the previous eight to fold their times into a host-side sum):
 * 0 bbox, 1 keys, 2 sort, 3 reorder, 4 build, 5 groups, 6 multipoles, 7 walk, 8 integrate (kicks, drifts). */
int bonsai_set_timing(bonsai_ctx* ctx, int enable);
int bonsai_get_stage_ms(bonsai_ctx* ctx, float out_ms[BONSAI_N_STAGES]);

/* Number of kernel launches the library has enqueued since bonsai_create() (kernels inside replayed graphs
 * included), and how many calls were served by replaying a captured graph. */
uint64_t bonsai_get_launch_count(bonsai_ctx* ctx);
uint64_t bonsai_get_graph_replays(bonsai_ctx* ctx);

/* Measurement support (not a step of the method): the FP32 throughput of the current CUDA device, measured with a
 * register-only loop of independent chains of the instruction the walk's interaction loops are made of --
 * packed != 0: fma.rn.f32x2 (SASS FFMA2), packed == 0: scalar FFMA -- `iters` rounds per thread, 64 warps per SM,
 * best of three timed launches on `cuda_stream` (CUDA events).  Writes TFLOP/s (FMA = 2 flop) to *tflops_out.
 * Blocks until done.  bench.py reports the walk's flop/s against this next to the derived peak.  EINVAL / ECUDA. */
int bonsai_measure_fp32_peak(void* cuda_stream, int packed, int iters, double* tflops_out);

const char* bonsai_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* BONSAI_H_ */
