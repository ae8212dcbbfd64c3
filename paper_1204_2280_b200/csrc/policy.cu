// Row f1, the rebuild policy (Discussion): "only when the tree-traverse shows a considerable decline in
// performance does the complete tree-structure has to be rebuild.  This decline is the result of ... an increase of
// the average number of particle-cell and particle-particle interactions."  No number is given.  Reading R30:
//
//   I_t   = (sum n_pp + sum n_pc over the sinks walked in tick t) / (number of sinks walked)      (fp64 division)
//   I_ref = I of the first recorded walk after the last full build
//   at the start of a tick:  rebuild  <=>  a reference exists  and  I_last > factor I_ref      (fp64, factor fp32)
//
// Outside the method: a tick that finds the sticky device status set (cell capacity or walk stack overflow in an
// earlier tick) rebuilds whatever the totals say -- only a build clears the status (k_recover), and with the status set
// the multipole pass and the walk return at once, so a refreshed tick would silently compute nothing.
//
// The decision is taken ON THE DEVICE (the totals of the last walk never travel to the host): k_rebuild_decide writes
// Control::rebuild_flag, and bonsai_block_tick enqueues the build chain behind Gate{rebuild_flag, 1} and the refresh
// behind Gate{rebuild_flag, 0} (internal.cuh); the side not taken costs its empty launches.
#include "internal.cuh"

namespace bonsai {

__global__ void k_rebuild_decide(Control* __restrict__ ctl, float factor) {
    const bool have_ref = ctl->tree_fresh == 0u;
    const bool rebuild = ctl->status != 0 || (have_ref && ctl->ipp_last > __dmul_rn((double)factor, ctl->ipp_ref));
    ctl->rebuild_flag = rebuild ? 1u : 0u;
    ctl->n_decisions += 1u;
    if (rebuild) ctl->n_rebuilds += 1u;
}

// after a walk: record I of that walk; the first one after a build becomes the reference
__global__ void k_walk_stats(Control* __restrict__ ctl) {
    const uint32_t n = ctl->n_active;
    if (n == 0u) return;
    const double ipp = __ddiv_rn((double)(ctl->sum_pp + ctl->sum_pc), (double)n);
    ctl->ipp_last = ipp;
    if (ctl->tree_fresh != 0u) {
        ctl->ipp_ref = ipp;
        ctl->tree_fresh = 0u;
    }
}

cudaError_t stage_rebuild_decide(Ctx* c, float factor) {
    k_rebuild_decide<<<1, 1, 0, c->stream>>>(c->b.ctl, factor);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_walk_stats(Ctx* c) {
    k_walk_stats<<<1, 1, 0, c->stream>>>(c->b.ctl);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace bonsai
