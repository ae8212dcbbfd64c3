// The C-ABI of libbonsai (include/bonsai.h): context, workspace carve-up, call sequencing, introspection.
// No arithmetic of the method lives here; each call enqueues the stage kernels of sort.cu / tree.cu /
// groups.cu / multipoles.cu / walk.cu on the caller's stream.
#include <cmath>
#include <new>

#include "internal.cuh"

using namespace bonsai;

struct bonsai_ctx {
    Ctx c;
};

namespace {

constexpr size_t kAlign = 256;

struct Carver {
    unsigned char* base;
    size_t off = 0;
    template <typename T>
    T* take(size_t count) {
        off = (off + kAlign - 1) / kAlign * kAlign;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += sizeof(T) * count;
        return p;
    }
};

bool resolve_params(uint32_t n_max, const bonsai_params* in, bonsai_params* out) {
    bonsai_params p;
    p.nleaf = 16; p.ncrit = 64; p.group_mode = 2; p.cap_cells = 0; p.group_cell = 0; p.mac_mode = 0; p.order = 2; p.rebuild_factor = 0.0f; p.no_graph = 0; p.mult_kernel = 0; p.sort_passes = 0;
    if (in) {
        p.no_graph = in->no_graph;
        p.mult_kernel = in->mult_kernel;
        p.sort_passes = in->sort_passes;
        p.rebuild_factor = in->rebuild_factor;
        p.mac_mode = in->mac_mode;
        if (in->order) p.order = in->order;
        if (in->nleaf) p.nleaf = in->nleaf;
        if (in->ncrit) p.ncrit = in->ncrit;
        p.group_mode = in->group_mode;
        p.cap_cells = in->cap_cells;
        p.group_cell = in->group_cell;
    }
    if (p.group_cell == 0) p.group_cell = 512;  // measured at 2^22: 9.75 ms per step against 9.88 (1024) and 10.07 (256)
    if (p.group_cell < p.ncrit) p.group_cell = p.ncrit;
    if (p.cap_cells == 0) {
        unsigned long long cap = 2ull * n_max + 256ull;
        if (cap >= (1ull << 29)) cap = (1ull << 29) - 1;
        p.cap_cells = (uint32_t)cap;
    }
    if (n_max == 0 || n_max > (1u << 30)) return false;
    if (p.nleaf < 1 || p.nleaf > (uint32_t)kMaxNleaf) return false;
    if (p.ncrit < 1 || p.ncrit > (uint32_t)kMaxNcrit) return false;
    if (p.group_mode > 2) return false;
    if (p.mac_mode > 1 || p.order < 1 || p.order > 2 || p.mult_kernel > 2) return false;
    if (p.sort_passes != 0 && (p.sort_passes < 4 || p.sort_passes > 6)) return false;
    if (p.rebuild_factor == 0.0f) p.rebuild_factor = 1.25f;
    if (!(p.rebuild_factor >= 1.0f) || std::isinf(p.rebuild_factor)) return false;
    if (p.cap_cells < 1 || p.cap_cells >= (1u << 29)) return false;  // walk stack entries pack the id into 29 bits
    *out = p;
    return true;
}

// Lays the buffers out in the workspace; with base = nullptr it only measures.
size_t carve(unsigned char* base, uint32_t n, const bonsai_params& p, Buffers* b) {
    Carver cv{base};
    const size_t cap = p.cap_cells;
    const uint32_t n_tiles = div_up(n, kSortTile);
    const uint32_t n_tblocks = div_up(n + 1, kTreeTile);
    Buffers t{};
    t.ctl = cv.take<Control>(1);
    for (int k = 0; k < 2; ++k) {
        for (int w = 0; w < 3; ++w) t.key[k][w] = cv.take<uint32_t>(n);
        t.pair_key[k] = cv.take<uint32_t>(n);
        t.idx[k] = cv.take<uint32_t>(n);
    }
    t.ghist = cv.take<uint32_t>((size_t)kSortPasses * kRadix);
    t.look = cv.take<unsigned long long>((size_t)kRadix * n_tiles);
    t.long_start = cv.take<uint32_t>((size_t)n / 32 + 1);
    t.bbox_partial = cv.take<float>(6 * kBboxMaxBlocks);
    t.sorted_pos = cv.take<float4>(n);
    t.lcp = cv.take<int8_t>((size_t)n + 1);
    t.leaf_level = cv.take<int8_t>((size_t)n + 1);
    t.blk_level_count = cv.take<uint32_t>((size_t)kLevelSlots * n_tblocks);
    t.level_total = cv.take<uint32_t>(kLevelSlots);
    t.c_level = cv.take<uint32_t>(cap);
    t.c_first = cv.take<uint32_t>(cap);
    t.c_count = cv.take<uint32_t>(cap);
    t.c_first_child = cv.take<uint32_t>(cap);
    t.c_n_child = cv.take<uint32_t>(cap);
    t.c_parent = cv.take<uint32_t>(cap);
    t.c_mac = cv.take<CellMac>(cap);
    t.c_quad = cv.take<CellQuad>(cap);
    t.c_qraw = cv.take<float>(cap * 6);
    t.c_mom = cv.take<double>(cap * 10);
    t.c_arrived = cv.take<uint32_t>(cap);
    t.c_box = cv.take<float>(cap * 6);
    t.rank = cv.take<uint32_t>((size_t)n + 1);
    t.active_list = cv.take<uint32_t>(n);
    t.g_flag = cv.take<uint32_t>((size_t)n + 1);
    t.g_cell = cv.take<uint32_t>(n);
    const size_t max_groups = (p.group_mode == 1) ? div_up(n, p.ncrit) : n;
    t.g_first = cv.take<uint32_t>(max_groups);
    t.g_count = cv.take<uint32_t>(max_groups);
    t.g_bmin = cv.take<float>(3 * max_groups);
    t.g_bmax = cv.take<float>(3 * max_groups);
    t.scan_tmp = cv.take<uint32_t>((size_t)div_up(n + 1, 2048) + 2);
    t.n_pp = cv.take<uint32_t>(n);
    t.n_pc = cv.take<uint32_t>(n);
    t.diag_partial = cv.take<double>((size_t)kDiagMaxBlocks * 12);
    t.host_in = cv.take<float4>(n);
    t.host_out = cv.take<float4>(n);
    t.host_mask = cv.take<uint8_t>(n);
    t.tick_mask = cv.take<uint8_t>(n);
    t.tie_pos = cv.take<float4>(n);
    if (b) *b = t;
    return (cv.off + kAlign - 1) / kAlign * kAlign;
}

// One timed interval of a stage.  A stage may run several times between two bonsai_get_stage_ms() calls (the
// groups in bonsai_build_tree and again in a masked bonsai_walk, the kicks of a tick): every run takes the next
// event pair of the stage and bonsai_get_stage_ms() sums them; when all kStageIntervals pairs are in use the next run
// first folds them into Ctx::ms_acc (a host wait on the last pair) and starts over.
struct StageTimer {
    Ctx* c;
    int stage, slot;
    StageTimer(Ctx* c_, int s) : c(c_), stage(s), slot(0) {
        if (c->timing) {
            if (c->ev_count[stage] == kStageIntervals) fold();
            slot = c->ev_count[stage];
            cudaEventRecord(c->ev[stage][slot][0], c->stream);
        }
    }
    ~StageTimer() {
        if (c->timing) {
            cudaEventRecord(c->ev[stage][slot][1], c->stream);
            c->ev_count[stage] += 1;
        }
    }
    // every event pair of this stage is in use: wait for the last one, add the intervals to the host-side sum and start
    // over with the first pair, so that no interval is lost (timing mode only; this is the one place a stage call waits)
    void fold() {
        cudaEventSynchronize(c->ev[stage][kStageIntervals - 1][1]);
        for (int i = 0; i < kStageIntervals; ++i) {
            float ms = 0.0f;
            if (cudaEventElapsedTime(&ms, c->ev[stage][i][0], c->ev[stage][i][1]) == cudaSuccess) c->ms_acc[stage] += ms;
        }
        c->ev_count[stage] = 0;
    }
};

// R9 / R11: the walk removes the self term arithmetically, which requires every sink's own leaf to be opened.  A cell
// that contains the sink has d <= |x - COM| <= (sqrt(3)/2) l + delta, so it is never accepted while
// l / theta > (sqrt(3)/2) l, i.e. theta < 2 / sqrt(3) = 1.1547; the library accepts theta in [0, 1.15].
constexpr float kThetaMax = BONSAI_THETA_MAX;
inline bool theta_ok(float theta) { return theta >= 0.0f && theta <= kThetaMax; }

#define BONSAI_TRY(expr)                                  \
    do {                                                  \
        cudaError_t e_ = (expr);                          \
        if (e_ != cudaSuccess) return BONSAI_ECUDA;       \
    } while (0)

}  // namespace

extern "C" {

size_t bonsai_workspace_bytes(uint32_t n_max, const bonsai_params* params) {
    bonsai_params p;
    if (!resolve_params(n_max, params, &p)) return 0;
    return carve(nullptr, n_max, p, nullptr);
}

int bonsai_create(uint32_t n_max, const bonsai_params* params, void* workspace_dev, size_t workspace_bytes,
                  void* cuda_stream, bonsai_ctx** out) {
    if (!out) return BONSAI_EINVAL;
    *out = nullptr;
    bonsai_params p;
    if (!resolve_params(n_max, params, &p)) return BONSAI_EINVAL;
    if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) % kAlign) != 0) return BONSAI_EINVAL;
    if (workspace_bytes < carve(nullptr, n_max, p, nullptr)) return BONSAI_ENOMEM;
    bonsai_ctx* h = new (std::nothrow) bonsai_ctx();
    if (!h) return BONSAI_ENOMEM;
    Ctx& c = h->c;
    c.n_max = n_max;
    c.n = 0;
    c.prm = p;
    c.cap_cells = p.cap_cells;
    c.stream = static_cast<cudaStream_t>(cuda_stream);
    carve(static_cast<unsigned char*>(workspace_dev), n_max, p, &c.b);
    c.pos_mass = nullptr;
    c.sorted_buf = 1;
    c.perm = c.b.idx[0];
    c.state = 0;
    c.groups_all_active = false;
    c.tree_n = 0;
    c.tree_refreshed = false;
    c.timing = false;
    c.launches = 0;
    for (int s = 0; s < BONSAI_N_STAGES; ++s) {
        c.ev_count[s] = 0;
        for (int k = 0; k < kStageIntervals; ++k) c.ev[s][k][0] = c.ev[s][k][1] = nullptr;
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&c.num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete h;
        return BONSAI_ECUDA;
    }
    c.device = dev;
    c.gate = Gate{nullptr, 0u};
    c.tree_auto = false;
    c.capture_stream = nullptr;
    c.side_stream = nullptr;
    c.ev_fork = c.ev_join = nullptr;
    c.graph_clock = c.graph_replays = 0;
    c.graph_misses = 0;
    c.graph_pause = 0;
    for (int s = 0; s < BONSAI_N_STAGES; ++s) c.ms_acc[s] = 0.0;
    for (int k = 0; k < kGraphSlots; ++k) c.graphs[k].valid = false;
    // kernel attributes and occupancy are per device: set for every context (idempotent), never behind a
    // process-wide flag
    if (walk_prepare(&c) != cudaSuccess || sort_prepare(&c) != cudaSuccess) {
        delete h;
        return BONSAI_ECUDA;
    }
    // control block, the self-cleaning arrival counters and the sort's look-back table (epoch 0 = never written)
    // start at zero
    if (cudaMemsetAsync(c.b.ctl, 0, sizeof(Control), c.stream) != cudaSuccess ||
        cudaMemsetAsync(c.b.c_arrived, 0, sizeof(uint32_t) * (size_t)c.cap_cells, c.stream) != cudaSuccess ||
        cudaMemsetAsync(c.b.look, 0, sizeof(unsigned long long) * (size_t)kRadix * div_up(n_max, kSortTile), c.stream) !=
            cudaSuccess) {
        delete h;
        return BONSAI_ECUDA;
    }
    *out = h;
    return BONSAI_OK;
}

int bonsai_load(bonsai_ctx* h, const float* pos_mass_dev, uint32_t n) {
    if (!h || !pos_mass_dev) return BONSAI_EINVAL;
    if ((reinterpret_cast<uintptr_t>(pos_mass_dev) % 16) != 0) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max) return BONSAI_EINVAL;
    h->c.pos_mass = reinterpret_cast<const float4*>(pos_mass_dev);
    h->c.n = n;
    h->c.state = 1;
    return BONSAI_OK;
}

// Stages a0..a4 (everything of bonsai_build_tree but the groups); every launch honours c->gate.
static int build_chain(Ctx* c) {
    { StageTimer t(c, 0); BONSAI_TRY(stage_bbox(c)); }
    { StageTimer t(c, 1); BONSAI_TRY(stage_keys(c)); }
    { StageTimer t(c, 2); BONSAI_TRY(stage_sort(c)); }
    {
        StageTimer t(c, 3);
        BONSAI_TRY(stage_reorder(c, true));
        BONSAI_TRY(stage_sort_ties(c));
    }
    { StageTimer t(c, 4); BONSAI_TRY(stage_build(c)); }
    return BONSAI_OK;
}

int bonsai_build_tree(bonsai_ctx* h) {
    if (!h) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    if (c->state < 1) return BONSAI_ESTATE;
    // the sticky status reports the work since the last build: a capacity overflow of an earlier step (reported by
    // the bonsai_sync of that step) must not poison this one
    BONSAI_TRY(stage_recover(c));
    int rc;
    if ((rc = build_chain(c)) != BONSAI_OK) return rc;
    { StageTimer t(c, 5); BONSAI_TRY(stage_groups(c, nullptr)); }
    c->tree_n = c->n;
    c->tree_refreshed = false;
    c->tree_auto = false;
    c->state = 2;
    return BONSAI_OK;
}

// bonsai_build_tree + bonsai_compute_multipoles as bonsai_step enqueues them: the group kernels (a4') and the
// multipole pass (a5) both need only the finished tree and neither reads what the other writes, and both are
// latency-bound, so the groups run on a side stream beside the multipole pass (fork / join by events; inside a
// capture this becomes two branches of the graph).  The same kernels with the same arguments as the two calls, so
// the results are bit-identical.  With stage timing on the two run one after the other, as the separate calls do.
static int build_tree_and_multipoles(Ctx* c) {
    if (c->state < 1) return BONSAI_ESTATE;
    BONSAI_TRY(stage_recover(c));
    int rc;
    if ((rc = build_chain(c)) != BONSAI_OK) return rc;
    bool fork = !c->timing;
    if (fork && !c->side_stream) {
        if (cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError();
            fork = false;
        }
    }
    if (fork) {
        cudaStream_t main_stream = c->stream;
        BONSAI_TRY(cudaEventRecord(c->ev_fork, main_stream));
        BONSAI_TRY(cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0));
        c->stream = c->side_stream;
        const cudaError_t e = stage_groups(c, nullptr);
        c->stream = main_stream;
        BONSAI_TRY(e);
        BONSAI_TRY(cudaEventRecord(c->ev_join, c->side_stream));
        BONSAI_TRY(stage_multipoles(c));
        BONSAI_TRY(cudaStreamWaitEvent(main_stream, c->ev_join, 0));
    } else {
        { StageTimer t(c, 5); BONSAI_TRY(stage_groups(c, nullptr)); }
        { StageTimer t(c, 6); BONSAI_TRY(stage_multipoles(c)); }
    }
    c->tree_n = c->n;
    c->tree_refreshed = false;
    c->tree_auto = false;
    c->state = 3;
    return BONSAI_OK;
}

// R30: rebuild or refresh, decided on the device from the interaction totals of the last recorded walk.  Both
// sequences are enqueued behind opposite gates on Control::rebuild_flag; there is no host read-back.
static int build_or_refresh_on_device(Ctx* c) {
    BONSAI_TRY(stage_rebuild_decide(c, c->prm.rebuild_factor));
    BONSAI_TRY(stage_recover(c));  // a set status made the decision "rebuild" (policy.cu): as every build, clear it first
    Buffers& b = c->b;
    c->gate = Gate{&b.ctl->rebuild_flag, 1u};
    int rc = build_chain(c);
    c->gate = Gate{&b.ctl->rebuild_flag, 0u};
    if (rc == BONSAI_OK) {
        StageTimer t(c, 3);
        if (stage_reorder(c, false) != cudaSuccess) rc = BONSAI_ECUDA;
    }
    c->gate = Gate{nullptr, 0u};
    if (rc != BONSAI_OK) return rc;
    { StageTimer t(c, 5); BONSAI_TRY(stage_groups(c, nullptr)); }
    c->tree_refreshed = false;
    c->tree_auto = true;  // the multipole pass asks the device flag whether the cell sides grow (R25)
    c->state = 2;
    return BONSAI_OK;
}

int bonsai_refresh_tree(bonsai_ctx* h) {
    if (!h) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    if (c->state < 1 || c->tree_n == 0 || c->tree_n != c->n) return BONSAI_ESTATE;
    { StageTimer t(c, 3); BONSAI_TRY(stage_reorder(c, false)); }
    { StageTimer t(c, 5); BONSAI_TRY(stage_groups(c, nullptr)); }
    c->tree_refreshed = true;
    c->tree_auto = false;
    c->state = 2;
    return BONSAI_OK;
}

int bonsai_compute_multipoles(bonsai_ctx* h) {
    if (!h) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    if (c->state < 2) return BONSAI_ESTATE;
    { StageTimer t(c, 6); BONSAI_TRY(stage_multipoles(c)); }
    c->state = 3;
    return BONSAI_OK;
}

int bonsai_walk(bonsai_ctx* h, float theta, float eps, const uint8_t* active_mask_dev, float* acc_pot_dev_out) {
    if (!h || !acc_pot_dev_out) return BONSAI_EINVAL;
    if ((reinterpret_cast<uintptr_t>(acc_pot_dev_out) % 16) != 0) return BONSAI_EINVAL;
    if (!theta_ok(theta) || !(eps >= 0.0f) || std::isinf(eps)) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    if (c->state < 3) return BONSAI_ESTATE;
    if (active_mask_dev != nullptr || !c->groups_all_active) {
        StageTimer t(c, 5);
        BONSAI_TRY(stage_groups(c, active_mask_dev));
    }
    { StageTimer t(c, 7); BONSAI_TRY(stage_walk(c, theta, eps, reinterpret_cast<float4*>(acc_pot_dev_out))); }
    c->state = 4;
    return BONSAI_OK;
}


}  // extern "C"

// ---- captured sequences (GraphKey / GraphSlot, internal.cuh) ------------------------------------------------------------

namespace {

HostState host_state(const Ctx* c) {
    return HostState{c->pos_mass, c->n, c->tree_n, c->state, c->sorted_buf, c->groups_all_active, c->tree_refreshed,
                     c->tree_auto, c->perm};
}

void restore_host_state(Ctx* c, const HostState& s) {
    c->pos_mass = s.pos_mass; c->n = s.n; c->tree_n = s.tree_n; c->state = s.state; c->sorted_buf = s.sorted_buf;
    c->groups_all_active = s.groups_all_active; c->tree_refreshed = s.tree_refreshed; c->tree_auto = s.tree_auto;
    c->perm = s.perm;
}

// Runs `enqueue` (a sequence of C-ABI calls on h) either directly on the caller's stream, or -- when graphs are
// enabled and stage timing is off -- as a CUDA graph: captured on the library's own stream the first time this key
// is seen, replayed on the caller's stream from then on.  A failed capture falls back to the direct path.
template <class F>
int run_sequence(bonsai_ctx* h, const GraphKey& key, F&& enqueue) {
    Ctx* c = &h->c;
    if (c->prm.no_graph || c->timing) return enqueue();
    c->graph_clock += 1;
    for (int k = 0; k < kGraphSlots; ++k) {
        GraphSlot& g = c->graphs[k];
        if (g.valid && g.key == key) {
            if (cudaGraphLaunch(g.exec, c->stream) != cudaSuccess) return BONSAI_ECUDA;
            restore_host_state(c, g.after);
            c->launches += g.launches;
            c->graph_replays += 1;
            c->graph_misses = 0;
            g.last_use = c->graph_clock;
            return BONSAI_OK;
        }
    }
    // a caller that passes fresh buffers every call would pay a capture + instantiation each time: after 16 misses in
    // a row the next kGraphPause calls are enqueued directly (no look-up of new keys, no capture), then capturing is
    // tried again -- a caller whose arguments settle later gets its graphs back
    if (c->graph_pause > 0) {
        c->graph_pause -= 1;
        return enqueue();
    }
    if (++c->graph_misses > 16) {
        c->graph_misses = 0;
        c->graph_pause = kGraphPause;
        return enqueue();
    }
    if (!c->capture_stream && cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
        (void)cudaGetLastError();
        return enqueue();
    }
    const HostState before = host_state(c);
    const uint64_t launches0 = c->launches;
    cudaStream_t user = c->stream;
    if (cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        (void)cudaGetLastError();
        return enqueue();
    }
    c->stream = c->capture_stream;
    const int rc = enqueue();
    c->stream = user;
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(c->capture_stream, &graph);
    cudaGraphExec_t exec = nullptr;
    if (rc != BONSAI_OK || ce != cudaSuccess || graph == nullptr ||
        cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        (void)cudaGetLastError();
        restore_host_state(c, before);
        c->launches = launches0;
        if (rc != BONSAI_OK) return rc;  // an argument / state error: the same answer without a graph
        return enqueue();
    }
    cudaGraphDestroy(graph);
    int slot = 0;  // a free slot, else the least recently used
    for (int k = 0; k < kGraphSlots; ++k) {
        if (!c->graphs[k].valid) { slot = k; break; }
        if (c->graphs[k].last_use < c->graphs[slot].last_use) slot = k;
    }
    GraphSlot& g = c->graphs[slot];
    if (g.valid) cudaGraphExecDestroy(g.exec);
    g.valid = true;
    g.key = key;
    g.exec = exec;
    g.after = host_state(c);
    g.launches = c->launches - launches0;
    g.last_use = c->graph_clock;
    if (cudaGraphLaunch(exec, c->stream) != cudaSuccess) return BONSAI_ECUDA;
    return BONSAI_OK;
}

}  // namespace

extern "C" {

int bonsai_step(bonsai_ctx* h, const float* pos_mass_dev, uint32_t n, float theta, float eps,
                const uint8_t* active_mask_dev, float* acc_pot_dev_out) {
    if (!h || !pos_mass_dev || !acc_pot_dev_out) return BONSAI_EINVAL;
    const GraphKey key{1, {pos_mass_dev, active_mask_dev, acc_pot_dev_out, nullptr}, n, {theta, eps, 0.0f}};
    return run_sequence(h, key, [&]() -> int {
        int rc;
        if ((rc = bonsai_load(h, pos_mass_dev, n)) != BONSAI_OK) return rc;
        if ((rc = build_tree_and_multipoles(&h->c)) != BONSAI_OK) return rc;
        return bonsai_walk(h, theta, eps, active_mask_dev, acc_pot_dev_out);
    });
}

int bonsai_step_host(bonsai_ctx* h, const float* pos_mass_host, uint32_t n, float theta, float eps,
                     const uint8_t* active_mask_host, float* acc_pot_host_out) {
    if (!h || !pos_mass_host || !acc_pot_host_out) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    if (n == 0 || n > c->n_max) return BONSAI_EINVAL;
    if (!theta_ok(theta) || !(eps >= 0.0f) || std::isinf(eps)) return BONSAI_EINVAL;
    Buffers& b = c->b;
    // (Measured and dropped, profiles/r2_tried_and_dropped.md: letting the walk write its 16-byte rows straight into
    // page-locked host memory hides the device-to-host copy but the scattered PCIe writes slow the walk by more than
    // the copy costs -- 13.9 ms against 12.9 ms end to end at 2^22.)
    float4* out_dev = b.host_out;
    BONSAI_TRY(cudaMemcpyAsync(b.host_in, pos_mass_host, sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
    if (active_mask_host) {
        BONSAI_TRY(cudaMemcpyAsync(b.host_mask, active_mask_host, (size_t)n, cudaMemcpyHostToDevice, c->stream));
        // entries of inactive particles are defined to stay untouched: the staged result starts from the caller's values
        BONSAI_TRY(cudaMemcpyAsync(b.host_out, acc_pot_host_out, sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
    }
    int rc;
    if ((rc = bonsai_step(h, reinterpret_cast<const float*>(b.host_in), n, theta, eps,
                          active_mask_host ? b.host_mask : nullptr, reinterpret_cast<float*>(out_dev))) != BONSAI_OK)
        return rc;
    BONSAI_TRY(cudaMemcpyAsync(acc_pot_host_out, b.host_out, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToHost, c->stream));
    return bonsai_sync(h);
}


// ---- row f2: integrator and diagnostics (integrate.cu) --------------------------------------------

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) % 16) == 0; }

int bonsai_kick(bonsai_ctx* h, float* vel_dev, const float* acc_pot_dev, uint32_t n, float step,
                const uint8_t* active_mask_dev) {
    if (!h || !vel_dev || !acc_pot_dev || !aligned16(vel_dev) || !aligned16(acc_pot_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || !std::isfinite(step)) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    StageTimer t(c, 8);
    BONSAI_TRY(stage_kick(c, reinterpret_cast<float4*>(vel_dev), reinterpret_cast<const float4*>(acc_pot_dev), n, step,
                          active_mask_dev));
    return BONSAI_OK;
}

int bonsai_drift(bonsai_ctx* h, float* pos_mass_dev, const float* vel_dev, uint32_t n, float step) {
    if (!h || !pos_mass_dev || !vel_dev || !aligned16(pos_mass_dev) || !aligned16(vel_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || !std::isfinite(step)) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    StageTimer t(c, 8);
    BONSAI_TRY(stage_drift(c, reinterpret_cast<float4*>(pos_mass_dev), reinterpret_cast<const float4*>(vel_dev), n, step));
    if (c->pos_mass == reinterpret_cast<const float4*>(pos_mass_dev) && c->state > 1) c->state = 1;  // the tree is stale
    return BONSAI_OK;
}

int bonsai_diagnostics(bonsai_ctx* h, const float* pos_mass_dev, const float* vel_dev, const float* acc_pot_dev,
                       uint32_t n, double* out12_dev) {
    if (!h || !pos_mass_dev || !vel_dev || !acc_pot_dev || !out12_dev) return BONSAI_EINVAL;
    if (!aligned16(pos_mass_dev) || !aligned16(vel_dev) || !aligned16(acc_pot_dev) ||
        (reinterpret_cast<uintptr_t>(out12_dev) % 8) != 0)
        return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    BONSAI_TRY(stage_diagnostics(c, reinterpret_cast<const float4*>(pos_mass_dev), reinterpret_cast<const float4*>(vel_dev),
                                 reinterpret_cast<const float4*>(acc_pot_dev), n, out12_dev));
    return BONSAI_OK;
}

int bonsai_leapfrog_step(bonsai_ctx* h, float* pos_mass_dev, float* vel_dev, float* acc_pot_dev, uint32_t n, float theta,
                         float eps, float dt) {
    if (!h || !pos_mass_dev || !vel_dev || !acc_pot_dev) return BONSAI_EINVAL;
    if (!aligned16(pos_mass_dev) || !aligned16(vel_dev) || !aligned16(acc_pot_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || !std::isfinite(dt)) return BONSAI_EINVAL;
    if (!theta_ok(theta) || !(eps >= 0.0f) || std::isinf(eps)) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    const float half = 0.5f * dt;  // exact
    const GraphKey key{2, {pos_mass_dev, vel_dev, acc_pot_dev, nullptr}, n, {theta, eps, dt}};
    return run_sequence(h, key, [&]() -> int {
        {
            StageTimer t(c, 8);
            BONSAI_TRY(stage_kick_drift(c, reinterpret_cast<float4*>(pos_mass_dev), reinterpret_cast<float4*>(vel_dev),
                                        reinterpret_cast<const float4*>(acc_pot_dev), n, half, dt));
        }
        int rc;
        if ((rc = bonsai_load(h, pos_mass_dev, n)) != BONSAI_OK) return rc;
        if ((rc = build_tree_and_multipoles(c)) != BONSAI_OK) return rc;
        if ((rc = bonsai_walk(h, theta, eps, nullptr, acc_pot_dev)) != BONSAI_OK) return rc;
        {
            StageTimer t(c, 8);
            BONSAI_TRY(stage_kick(c, reinterpret_cast<float4*>(vel_dev), reinterpret_cast<const float4*>(acc_pot_dev), n, half,
                                  nullptr));
        }
        return BONSAI_OK;
    });
}

// ---- block time-steps (R26, R27) --------------------------------------------------------------------------

int bonsai_timestep_rungs(bonsai_ctx* h, const float* acc_pot_dev, uint32_t n, float eta, float eps, float dt_max,
                          uint32_t kmax, const uint8_t* active_mask_dev, uint64_t tick, uint8_t* rung_dev, int init) {
    if (!h || !acc_pot_dev || !rung_dev || !aligned16(acc_pot_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || kmax > 30u) return BONSAI_EINVAL;
    if (!(eta > 0.0f) || !(eps > 0.0f) || !(dt_max > 0.0f) || std::isinf(eta) || std::isinf(eps) || std::isinf(dt_max))
        return BONSAI_EINVAL;
    BONSAI_TRY(stage_rungs(&h->c, reinterpret_cast<const float4*>(acc_pot_dev), n, eta, eps, dt_max, kmax, active_mask_dev,
                           tick, rung_dev, init));
    return BONSAI_OK;
}

int bonsai_active_mask(bonsai_ctx* h, const uint8_t* rung_dev, uint32_t n, uint32_t kmax, uint64_t tick,
                       uint8_t* mask_dev_out) {
    if (!h || !rung_dev || !mask_dev_out) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || kmax > 30u) return BONSAI_EINVAL;
    BONSAI_TRY(stage_active_mask(&h->c, rung_dev, n, kmax, tick, mask_dev_out));
    return BONSAI_OK;
}

int bonsai_kick_rungs(bonsai_ctx* h, float* vel_dev, const float* acc_pot_dev, const uint8_t* rung_dev,
                      const uint8_t* active_mask_dev, uint32_t n, float dt_max) {
    if (!h || !vel_dev || !acc_pot_dev || !rung_dev || !aligned16(vel_dev) || !aligned16(acc_pot_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || !std::isfinite(dt_max)) return BONSAI_EINVAL;
    Ctx* c = &h->c;
    StageTimer t(c, 8);
    BONSAI_TRY(stage_kick_rungs(c, reinterpret_cast<float4*>(vel_dev), reinterpret_cast<const float4*>(acc_pot_dev), rung_dev,
                                active_mask_dev, n, dt_max));
    return BONSAI_OK;
}

int bonsai_block_tick(bonsai_ctx* h, float* pos_mass_dev, float* vel_dev, float* acc_pot_dev, uint8_t* rung_dev, uint32_t n,
                      uint64_t tick, float theta, float eps, float eta, float dt_max, uint32_t kmax, int rebuild) {
    if (!h || !pos_mass_dev || !vel_dev || !acc_pot_dev || !rung_dev) return BONSAI_EINVAL;
    if (!aligned16(pos_mass_dev) || !aligned16(vel_dev) || !aligned16(acc_pot_dev)) return BONSAI_EINVAL;
    if (n == 0 || n > h->c.n_max || kmax > 30u) return BONSAI_EINVAL;
    if (!theta_ok(theta) || !(eta > 0.0f) || !(eps > 0.0f) || !(dt_max > 0.0f) || std::isinf(eta) ||
        std::isinf(eps) || std::isinf(dt_max))
        return BONSAI_EINVAL;
    Ctx* c = &h->c;
    const bool have_tree = c->tree_n == n && c->pos_mass == reinterpret_cast<const float4*>(pos_mass_dev);
    if (rebuild == 0 && !have_tree) return BONSAI_ESTATE;
    if (rebuild < 0 && !have_tree) rebuild = 1;  // R30 needs a tree to decide about
    float4* vel = reinterpret_cast<float4*>(vel_dev);
    const float4* acc = reinterpret_cast<const float4*>(acc_pot_dev);
    uint8_t* mask = c->b.tick_mask;
    const float dt_min = std::ldexp(dt_max, -(int)kmax);
    int rc;
    BONSAI_TRY(stage_active_mask(c, rung_dev, n, kmax, tick, mask));
    {
        StageTimer t(c, 8);
        BONSAI_TRY(stage_kick_rungs(c, vel, acc, rung_dev, mask, n, dt_max));
        BONSAI_TRY(stage_drift(c, reinterpret_cast<float4*>(pos_mass_dev), vel, n, dt_min));
    }
    BONSAI_TRY(stage_active_mask(c, rung_dev, n, kmax, tick + 1, mask));
    if ((rc = bonsai_load(h, pos_mass_dev, n)) != BONSAI_OK) return rc;
    if (rebuild < 0) rc = build_or_refresh_on_device(c);
    else rc = rebuild ? bonsai_build_tree(h) : bonsai_refresh_tree(h);
    if (rc != BONSAI_OK) return rc;
    if ((rc = bonsai_compute_multipoles(h)) != BONSAI_OK) return rc;
    if ((rc = bonsai_walk(h, theta, eps, mask, acc_pot_dev)) != BONSAI_OK) return rc;
    BONSAI_TRY(stage_walk_stats(c));  // R30: interactions per walked sink; the first walk after a build is the reference
    {
        StageTimer t(c, 8);
        BONSAI_TRY(stage_kick_rungs(c, vel, acc, rung_dev, mask, n, dt_max));
    }
    BONSAI_TRY(stage_rungs(c, acc, n, eta, eps, dt_max, kmax, mask, tick + 1, rung_dev, 0));
    return BONSAI_OK;
}

void bonsai_destroy(bonsai_ctx* h) {
    if (!h) return;
    for (int k = 0; k < kGraphSlots; ++k)
        if (h->c.graphs[k].valid) cudaGraphExecDestroy(h->c.graphs[k].exec);
    if (h->c.capture_stream) cudaStreamDestroy(h->c.capture_stream);
    if (h->c.side_stream) cudaStreamDestroy(h->c.side_stream);
    if (h->c.ev_fork) cudaEventDestroy(h->c.ev_fork);
    if (h->c.ev_join) cudaEventDestroy(h->c.ev_join);
    for (int s = 0; s < BONSAI_N_STAGES; ++s)
        for (int i = 0; i < kStageIntervals; ++i)
            for (int k = 0; k < 2; ++k)
                if (h->c.ev[s][i][k]) cudaEventDestroy(h->c.ev[s][i][k]);
    delete h;
}

int bonsai_sync(bonsai_ctx* h) {
    if (!h) return BONSAI_EINVAL;
    int status = 0;
    if (cudaMemcpyAsync(&status, &h->c.b.ctl->status, sizeof(int), cudaMemcpyDeviceToHost, h->c.stream) != cudaSuccess)
        return BONSAI_ECUDA;
    if (cudaStreamSynchronize(h->c.stream) != cudaSuccess) return BONSAI_ECUDA;
    return status;
}

// ---- introspection ---------------------------------------------------------------------------------

int bonsai_get_box(bonsai_ctx* h, const float** box4_dev) {
    if (!h || !box4_dev) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    *box4_dev = h->c.b.ctl->lo;  // lo[3] followed by side_f
    return BONSAI_OK;
}

int bonsai_get_keys(bonsai_ctx* h, const uint32_t** hi_dev, const uint32_t** mid_dev, const uint32_t** lo_dev) {
    if (!h || !hi_dev || !mid_dev || !lo_dev) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    const int s = h->c.sorted_buf;
    *hi_dev = h->c.b.key[s][0];
    *mid_dev = h->c.b.key[s][1];
    *lo_dev = h->c.b.key[s][2];
    return BONSAI_OK;
}

int bonsai_get_perm(bonsai_ctx* h, const uint32_t** perm_dev) {
    if (!h || !perm_dev) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    *perm_dev = h->c.perm;
    return BONSAI_OK;
}

int bonsai_get_sorted_pos(bonsai_ctx* h, const float** pos_mass_dev) {
    if (!h || !pos_mass_dev) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    *pos_mass_dev = reinterpret_cast<const float*>(h->c.b.sorted_pos);
    return BONSAI_OK;
}

int bonsai_get_cells(bonsai_ctx* h, bonsai_cells_view* out) {
    if (!h || !out) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    const Buffers& b = h->c.b;
    if (h->c.state >= 3) BONSAI_TRY(cells_qraw(&h->c));  // quad[] is derived from the fp64 record on demand
    out->cap_cells = h->c.cap_cells;
    out->n_cells = &b.ctl->n_cells;
    out->level_offsets = b.ctl->level_offsets;
    out->level = b.c_level;
    out->first = b.c_first;
    out->count = b.c_count;
    out->first_child = b.c_first_child;
    out->n_child = b.c_n_child;
    out->parent = b.c_parent;
    out->mac = reinterpret_cast<const float*>(b.c_mac);
    out->quad = b.c_qraw;
    out->walk_quad = reinterpret_cast<const float*>(b.c_quad);
    return BONSAI_OK;
}

int bonsai_get_groups(bonsai_ctx* h, bonsai_groups_view* out) {
    if (!h || !out) return BONSAI_EINVAL;
    if (h->c.state < 2) return BONSAI_ESTATE;
    const Buffers& b = h->c.b;
    if (h->c.groups_all_active) BONSAI_TRY(groups_fill_identity(&h->c));  // not materialised by the step itself
    out->n_groups = &b.ctl->n_groups;
    out->n_active = &b.ctl->n_active;
    out->active_list = b.active_list;
    out->first = b.g_first;
    out->count = b.g_count;
    out->bmin = b.g_bmin;
    out->bmax = b.g_bmax;
    return BONSAI_OK;
}

int bonsai_get_counts(bonsai_ctx* h, const uint32_t** n_pp_dev, const uint32_t** n_pc_dev) {
    if (!h || !n_pp_dev || !n_pc_dev) return BONSAI_EINVAL;
    if (h->c.state < 4) return BONSAI_ESTATE;
    *n_pp_dev = h->c.b.n_pp;
    *n_pc_dev = h->c.b.n_pc;
    return BONSAI_OK;
}

int bonsai_get_interaction_totals(bonsai_ctx* h, uint64_t* sum_pp, uint64_t* sum_pc) {
    if (!h || !sum_pp || !sum_pc) return BONSAI_EINVAL;
    if (h->c.state < 4) return BONSAI_ESTATE;
    unsigned long long v[2] = {0, 0};
    if (cudaMemcpyAsync(v, &h->c.b.ctl->sum_pp, sizeof(v), cudaMemcpyDeviceToHost, h->c.stream) != cudaSuccess)
        return BONSAI_ECUDA;
    if (cudaStreamSynchronize(h->c.stream) != cudaSuccess) return BONSAI_ECUDA;
    *sum_pp = v[0];
    *sum_pc = v[1];
    return BONSAI_OK;
}

int bonsai_get_rebuild_stats(bonsai_ctx* h, uint32_t* n_decisions, uint32_t* n_rebuilds, double* ipp_ref, double* ipp_last) {
    if (!h) return BONSAI_EINVAL;
    Control host;
    if (cudaMemcpyAsync(&host, h->c.b.ctl, sizeof(Control), cudaMemcpyDeviceToHost, h->c.stream) != cudaSuccess)
        return BONSAI_ECUDA;
    if (cudaStreamSynchronize(h->c.stream) != cudaSuccess) return BONSAI_ECUDA;
    if (n_decisions) *n_decisions = host.n_decisions;
    if (n_rebuilds) *n_rebuilds = host.n_rebuilds;
    if (ipp_ref) *ipp_ref = host.ipp_ref;
    if (ipp_last) *ipp_last = host.ipp_last;
    return BONSAI_OK;
}

int bonsai_set_timing(bonsai_ctx* h, int enable) {
    if (!h) return BONSAI_EINVAL;
    Ctx& c = h->c;
    if (enable && !c.ev[0][0][0]) {
        for (int s = 0; s < BONSAI_N_STAGES; ++s)
            for (int i = 0; i < kStageIntervals; ++i)
                for (int k = 0; k < 2; ++k)
                    if (cudaEventCreate(&c.ev[s][i][k]) != cudaSuccess) return BONSAI_ECUDA;
    }
    c.timing = enable != 0;
    for (int s = 0; s < BONSAI_N_STAGES; ++s) { c.ev_count[s] = 0; c.ms_acc[s] = 0.0; }
    return BONSAI_OK;
}

int bonsai_get_stage_ms(bonsai_ctx* h, float out_ms[BONSAI_N_STAGES]) {
    if (!h || !out_ms) return BONSAI_EINVAL;
    Ctx& c = h->c;
    if (cudaStreamSynchronize(c.stream) != cudaSuccess) return BONSAI_ECUDA;
    for (int s = 0; s < BONSAI_N_STAGES; ++s) {
        out_ms[s] = (float)c.ms_acc[s];
        c.ms_acc[s] = 0.0;
        for (int i = 0; i < c.ev_count[s]; ++i) {
            float ms = 0.0f;
            if (cudaEventElapsedTime(&ms, c.ev[s][i][0], c.ev[s][i][1]) != cudaSuccess) return BONSAI_ECUDA;
            out_ms[s] += ms;
        }
        c.ev_count[s] = 0;
    }
    return BONSAI_OK;
}

uint64_t bonsai_get_launch_count(bonsai_ctx* h) { return h ? h->c.launches : 0; }

uint64_t bonsai_get_graph_replays(bonsai_ctx* h) { return h ? h->c.graph_replays : 0; }

const char* bonsai_strerror(int code) {
    switch (code) {
        case BONSAI_OK: return "ok";
        case BONSAI_EINVAL: return "invalid argument";
        case BONSAI_ESTATE: return "call out of order";
        case BONSAI_ECAPACITY: return "cell capacity or traversal stack exceeded";
        case BONSAI_ECUDA: return "CUDA runtime error";
        case BONSAI_ENOMEM: return "workspace too small";
        default: return "unknown error";
    }
}

}  // extern "C"
