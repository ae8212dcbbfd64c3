// Internal declarations shared by the stage translation units of libbonsai (CUDA, sm_100a only).
// Nothing here is part of the C-ABI; see include/bonsai.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "bonsai.h"

namespace bonsai {

constexpr int kMaxLevel = BONSAI_MAX_LEVEL;
constexpr uint32_t kNone = 0xFFFFFFFFu;
constexpr uint32_t kLeafBit = 0x80000000u;

// ---- radix sort geometry (sort.cu) -------------------------------------------------------------
constexpr int kRadixBits = 10;             // one 30-bit key word = 3 digits
constexpr int kRadix = 1 << kRadixBits;
constexpr int kSortPasses = 6;              // mid and hi words; the lo word is settled by the tie kernels
constexpr int kSortThreads = 512;
constexpr int kSortBlocksPerSM = 2;
constexpr int kLookBatch = 1;              // look-back entries in flight per digit
constexpr unsigned kLookSleepNs = 200;     // back-off of a look-back chain whose next entry is not published yet
constexpr int kSortItems = 16;             // pairs per thread per tile
constexpr int kSortTile = kSortThreads * kSortItems;
constexpr int kKeysThreads = 512;

// ---- tree build geometry (tree.cu) -------------------------------------------------------------
constexpr int kTreeThreads = 256;
constexpr int kTreeItems = 4;
constexpr int kTreeTile = kTreeThreads * kTreeItems;  // particles per block
constexpr int kLevelSlots = 32;                       // levels 0..30, padded
constexpr int kMaxNleaf = 64;

constexpr int kBboxMaxBlocks = 2048;       // rows of bbox_partial; stage_bbox clamps its grid to this
constexpr uint32_t kGraphPause = 256;      // calls enqueued directly after 16 graph misses in a row
constexpr int kStageIntervals = 8;         // event pairs per stage: a stage that runs several times between two
                                           // bonsai_get_stage_ms() calls (groups in build and in a masked walk, the
                                           // kicks of a tick) is summed over its intervals

// ---- diagnostics (integrate.cu) ----------------------------------------------------------------
constexpr int kDiagMaxBlocks = 1184;       // 8 blocks per SM on 148 SMs

// ---- walk geometry (walk.cu) -------------------------------------------------------------------
constexpr int kWalkWarps = 8;              // warps per block, one group per warp at a time
constexpr int kWalkStack = 512;            // traversal stack entries (runs of siblings) per warp; bound derived in walk.cu
constexpr int kMaxNcrit = 64;

// Device-resident control block at the start of the workspace (zeroed by bonsai_create).
struct Control {
    float lo[3];               // root cube corner (R3)
    float side_f;              // root cube side as fp32 (power of two, exact)
    float scale;               // 2^30 / side (exact)
    int status;                // sticky device status (0 or BONSAI_ECAPACITY)
    double side;               // root cube side
    uint32_t n_cells;
    uint32_t n_groups;
    uint32_t n_active;
    uint32_t bbox_ticket;
    uint32_t walk_ticket;      // dynamic group scheduler of the walk
    uint32_t level_ticket;     // last-block-done counter of k_tree_scan_levels
    uint32_t sort_ticket;      // tile scheduler of k_sort_pass (reset by the tile that draws the last ticket)
    uint32_t diag_ticket;      // last-block-done counter of k_diagnostics
    uint32_t n_long_runs;      // runs of equal (hi, mid) longer than kTieRun found by k_sort_ties (k_sort_long_runs)
    uint32_t recover_ticket;   // last-block-done counter of k_recover
    uint32_t rebuild_flag;     // R30: decision of k_rebuild_decide for the current tick (1 = rebuild, 0 = refresh)
    uint32_t tree_fresh;       // R30: set by a build; the next recorded walk becomes the reference and clears it
    uint32_t level_offsets[32];  // first cell of level L; [31] = n_cells
    unsigned long long sum_pp;   // interaction totals of the last walk (sink-source pairs)
    unsigned long long sum_pc;
    double ipp_ref;              // R30: interactions per walked sink of the first recorded walk after the last build
    double ipp_last;             // R30: ... of the last recorded walk
    uint32_t n_rebuilds;         // R30: rebuilds decided on the device since bonsai_create
    uint32_t n_decisions;
    uint32_t sort_epoch;         // tag base of the look-back entries of this build's sort passes (k_bbox advances it)
    uint32_t look_wrap;          // the epoch wrapped: k_sort_gscan clears the look-back table
    uint32_t long_ticket;        // run scheduler / last-warp-done counter of k_sort_long_runs
    uint32_t long_done;
    uint32_t mult_ticket;        // tile scheduler of k_multipoles (tiles of cells, deepest first)
    uint32_t mult_done;          // ... and its last-block-out counter, which resets both
};

// A launch that only does its work when a device flag has a given value.  The flag is written by an earlier kernel
// on the same stream (k_sort_ties: the sort's fallback chain; k_rebuild_decide: R30), so a data-dependent choice
// between two kernel sequences needs no host read-back: both are enqueued, one of them returns at once.
struct Gate {
    const uint32_t* flag;      // nullptr: always open
    uint32_t want;
};
__device__ __forceinline__ bool gate_closed(const Gate g) { return g.flag != nullptr && __ldcg(g.flag) != g.want; }

// Walk layout of a cell, two 32-byte records (one DRAM/L2 sector each):
//   CellMac : what the opening test and the monopole need + the links
//   CellQuad: what only an accepted cell needs
struct __align__(16) CellMac {
    float cx, cy, cz, m;       // centre of mass, mass (fp32, rounded once from fp64)
    float delta, lside;        // |COM - geometric centre|, geometric side
    uint32_t first;            // internal: first child;  leaf: first sorted particle
    uint32_t info;             // internal: n_child (1..8);  leaf: kLeafBit | count
};
struct __align__(16) CellQuad {
    // P = tr I - 3 Q  (minus the trace-free quadrupole; Q = raw second moments about the COM, tr = Qxx + Qyy + Qzz),
    // formed in fp64 and rounded once.  With r^2 = |dr|^2 + eps^2 in every power (R10) the raw-moment formulas are
    //   phi = -M/r + (dr.P.dr + tr eps^2) / (2 r^5),   a = dr (M/r^3 - 5 (dr.P.dr + tr eps^2) / (2 r^7)) + P.dr / r^5
    // exactly, which is 33 FP32 operations per particle-cell interaction instead of 36 (walk.cu).
    float pxx, pyy, pzz, pxy, pxz, pyz;
    float tr;
    float pad;
};

struct Buffers {
    Control* ctl;
    // keys, structure of arrays: key[0] = load order (k_keys), key[1] = sorted order (k_reorder)
    uint32_t* key[2][3];       // [order][word]: hi, mid, lo
    // sort: ping-pong (30-bit word, index) pairs
    uint32_t* pair_key[2];
    uint32_t* idx[2];
    uint32_t* ghist;           // [kSortPasses][kRadix] global digit histograms -> exclusive bases
    unsigned long long* look;  // [n_tiles][kRadix] decoupled look-back table of k_sort_pass
    uint32_t* long_start;      // [n / 32 + 1] first position of every long run of equal (hi, mid)
    float* bbox_partial;       // [blocks][6]
    float4* sorted_pos;
    // tree
    int8_t* lcp;               // [n+1] common leading digits of key[i-1], key[i]; -1 at both ends
    int8_t* leaf_level;        // [n] level of the leaf containing particle i
    uint32_t* blk_level_count; // [kLevelSlots][n_blocks] cells per level per block -> exclusive prefix over blocks
    uint32_t* level_total;     // [kLevelSlots]
    uint32_t *c_level, *c_first, *c_count, *c_first_child, *c_n_child, *c_parent;
    // multipoles
    CellMac* c_mac;            // [cap]
    CellQuad* c_quad;          // [cap]
    float* c_qraw;             // [cap][6] raw second moments xx, yy, zz, xy, xz, yz as fp32 (introspection, R8)
    double* c_mom;             // [cap][10] fp64: M, COMx, COMy, COMz, Qxx, Qyy, Qzz, Qxy, Qxz, Qyz
    uint32_t* c_arrived;       // [cap] children that have finished
    float* c_box;              // [cap][6] exact fp32 bounding box of each cell's members (min xyz, max xyz)
    // groups
    uint32_t* rank;            // [n+1] exclusive count of active particles (sorted order)
    uint32_t* active_list;     // [n]
    uint32_t* g_flag;          // [n+1] scan scratch (mode 0: 1 where a non-empty group starts)
    uint32_t* g_cell;          // [n] mode 0: 1 + id of the group cell starting at particle i (0 = none)
    uint32_t *g_first, *g_count;
    float *g_bmin, *g_bmax;
    uint32_t* scan_tmp;        // block sums of the device-wide scan
    // walk
    uint32_t *n_pp, *n_pc;     // [n] load order
    double* diag_partial;      // [kDiagMaxBlocks][12] block partials of k_diagnostics
    // staging of bonsai_step_host
    float4 *host_in, *host_out;
    float4* tie_pos;           // [n] scratch of k_sort_long_runs: a run's particles while they are permuted
    uint8_t* host_mask;
    uint8_t* tick_mask;        // [n] active mask of bonsai_block_tick
};

// A whole call sequence (bonsai_step, bonsai_leapfrog_step) captured once as a CUDA graph and replayed while the
// caller keeps passing the same buffers and parameters: one graph launch instead of ~27 kernel launches -- below
// N ~ 10^5 the step is bound by launch gaps, not by the kernels ("the algorithms require more than 10^5
// particles to saturate the GPU").  Nothing in a step depends on host-side values that change between replays
// (grid sizes depend on n only; the sort's look-back epoch lives on the device).
struct GraphKey {
    int kind;                  // 1 = bonsai_step, 2 = bonsai_leapfrog_step
    const void* ptr[4];
    uint32_t n;
    float f[3];
    bool operator==(const GraphKey& o) const {
        return kind == o.kind && ptr[0] == o.ptr[0] && ptr[1] == o.ptr[1] && ptr[2] == o.ptr[2] && ptr[3] == o.ptr[3] &&
               n == o.n && f[0] == o.f[0] && f[1] == o.f[1] && f[2] == o.f[2];
    }
};
struct HostState {            // what a captured sequence leaves behind in the Ctx (restored on replay)
    const float4* pos_mass;
    uint32_t n, tree_n;
    int state, sorted_buf;
    bool groups_all_active, tree_refreshed, tree_auto;
    uint32_t* perm;
};
struct GraphSlot {
    bool valid;
    GraphKey key;
    cudaGraphExec_t exec;
    HostState after;
    uint64_t launches, last_use;
};
constexpr int kGraphSlots = 4;

struct Ctx {
    uint32_t n_max, n;
    bonsai_params prm;
    uint32_t cap_cells;
    cudaStream_t stream;
    Buffers b;
    const float4* pos_mass;    // caller's particles (load order)
    int sorted_buf;            // which key[] holds the sorted keys (1 once k_reorder has run)
    uint32_t* perm;            // perm[i] = load index of the i-th sorted particle (one of b.idx[])
    int state;                 // 0 created, 1 loaded, 2 tree built, 3 multipoles done, 4 walked
    bool groups_all_active;    // the group list on the device is the all-active one
    uint32_t tree_n;           // particle count of the tree on the device (0 = none): bonsai_refresh_tree may reuse it
    bool tree_refreshed;       // positions were re-gathered into a frozen tree: multipoles take l from the extents (R25)
    bool timing;
    cudaEvent_t ev[BONSAI_N_STAGES][kStageIntervals][2];
    int ev_count[BONSAI_N_STAGES];  // intervals recorded since the last bonsai_get_stage_ms() or fold
    double ms_acc[BONSAI_N_STAGES]; // ms of the intervals already folded (a stage ran more than kStageIntervals times)
    uint64_t launches;
    int num_sms;
    int device;                // the CUDA device the context was created on
    cudaStream_t capture_stream;  // library-owned stream the sequences are captured on (any caller stream can replay)
    cudaStream_t side_stream;     // library-owned: the group kernels of bonsai_step run here, beside the multipole pass
    cudaEvent_t ev_fork, ev_join; // fork / join of that branch (no timing)
    GraphSlot graphs[kGraphSlots];
    uint64_t graph_clock, graph_replays;
    uint32_t graph_misses;     // consecutive calls that found no captured graph (16 in a row pause capturing)
    uint32_t graph_pause;      // calls left to enqueue directly before capturing is tried again
    Gate gate;                 // applied to every launch of the build chain (bbox .. tree) while it is set (R30)
    bool tree_auto;            // the tree on the device was rebuilt OR refreshed by a device-side decision (R30)
    int walk_blocks_per_sm[8]; // occupancy of the k_walk instances on this device (set in bonsai_create)
};

inline uint32_t div_up(uint32_t a, uint32_t b) { return (a + b - 1) / b; }

// Stage entry points (each enqueues kernels on ctx->stream and bumps ctx->launches).
cudaError_t stage_bbox(Ctx* c);
cudaError_t stage_keys(Ctx* c);
cudaError_t stage_sort(Ctx* c);
int sort_first_pass(const Ctx* c);  // the passes sort_first_pass() .. 5 run (params.sort_passes, else a rule on n)
cudaError_t stage_reorder(Ctx* c, bool write_keys);
cudaError_t stage_sort_ties(Ctx* c);
cudaError_t stage_build(Ctx* c);
cudaError_t stage_groups(Ctx* c, const uint8_t* mask_load_order);
cudaError_t groups_fill_identity(Ctx* c);  // active_list of an all-active group list, on demand (introspection)
cudaError_t stage_multipoles(Ctx* c);
cudaError_t cells_qraw(Ctx* c);  // fills c_qraw from c_mom (introspection)
cudaError_t stage_walk(Ctx* c, float theta, float eps, float4* acc_pot_out);
cudaError_t walk_prepare(Ctx* c);  // per-device kernel attributes and occupancy (bonsai_create)
cudaError_t sort_prepare(Ctx* c);
cudaError_t stage_rebuild_decide(Ctx* c, float factor);  // R30 (policy.cu)
cudaError_t stage_walk_stats(Ctx* c);
cudaError_t stage_recover(Ctx* c); // guarded: re-zeroes the arrival counters after a capacity overflow, clears the status
size_t walk_smem_bytes(uint32_t nleaf);
cudaError_t stage_kick(Ctx* c, float4* vel, const float4* acc, uint32_t n, float h, const uint8_t* mask);
cudaError_t stage_drift(Ctx* c, float4* pos, const float4* vel, uint32_t n, float h);
cudaError_t stage_kick_drift(Ctx* c, float4* pos, float4* vel, const float4* acc, uint32_t n, float hk, float hd);
cudaError_t stage_rungs(Ctx* c, const float4* acc, uint32_t n, float eta, float eps, float dt_max, uint32_t kmax,
                        const uint8_t* mask, unsigned long long tick, uint8_t* rung, int init);
cudaError_t stage_active_mask(Ctx* c, const uint8_t* rung, uint32_t n, uint32_t kmax, unsigned long long tick,
                              uint8_t* mask);
cudaError_t stage_kick_rungs(Ctx* c, float4* vel, const float4* acc, const uint8_t* rung, const uint8_t* mask,
                             uint32_t n, float dt_max);
cudaError_t stage_diagnostics(Ctx* c, const float4* pos, const float4* vel, const float4* acc, uint32_t n, double* out);

// Device-wide exclusive scan of u32 (scan.cu): out[i] = sum_{j<i} in[j], i in [0, n]; out has n+1 entries
// (out[n] = total).  in may alias out.  tmp needs div_up(n, 2048) + 1 entries.
cudaError_t exclusive_scan_u32(Ctx* c, const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* tmp);

}  // namespace bonsai
