// Row f2: the time integration around the force step ("block time-step method"; BASELINE.json
// configs[2]: leapfrog, shared time-step, tree rebuilt every step) and the conserved-quantity diagnostics.
// Readings R22 (kick-drift-kick), R23 (fp32 state, one fused multiply-add per component), R24 (fp64 sums).
//
// All three kernels stream float4 records once: kick 16 + 16 B in, 16 B out; drift likewise; the fused
// kick+drift that opens a step 48 B in, 32 B out; the diagnostics 48 B in.  HBM-bound, no reuse.
#include "internal.cuh"

namespace bonsai {

// v <- fma(a, h, v) per component; the fourth lane of vel is carried through untouched.
__global__ void __launch_bounds__(256) k_kick(float4* __restrict__ vel, const float4* __restrict__ acc, uint32_t n,
                                              float h, const uint8_t* __restrict__ mask) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (mask && !mask[i]) return;
    float4 v = vel[i];
    const float4 a = __ldg(&acc[i]);
    v.x = __fmaf_rn(a.x, h, v.x);
    v.y = __fmaf_rn(a.y, h, v.y);
    v.z = __fmaf_rn(a.z, h, v.z);
    vel[i] = v;
}

// x <- fma(v, h, x) per component; the mass is carried through untouched.
__global__ void __launch_bounds__(256) k_drift(float4* __restrict__ pos, const float4* __restrict__ vel, uint32_t n,
                                               float h) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = pos[i];
    const float4 v = __ldg(&vel[i]);
    p.x = __fmaf_rn(v.x, h, p.x);
    p.y = __fmaf_rn(v.y, h, p.y);
    p.z = __fmaf_rn(v.z, h, p.z);
    pos[i] = p;
}

// The opening half of a KDK step in one pass: kick by hk, then drift by hd with the kicked velocity --
// operation for operation what k_kick followed by k_drift computes.
__global__ void __launch_bounds__(256) k_kick_drift(float4* __restrict__ pos, float4* __restrict__ vel,
                                                    const float4* __restrict__ acc, uint32_t n, float hk, float hd) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = vel[i];
    const float4 a = __ldg(&acc[i]);
    v.x = __fmaf_rn(a.x, hk, v.x);
    v.y = __fmaf_rn(a.y, hk, v.y);
    v.z = __fmaf_rn(a.z, hk, v.z);
    vel[i] = v;
    float4 p = pos[i];
    p.x = __fmaf_rn(v.x, hd, p.x);
    p.y = __fmaf_rn(v.y, hd, p.y);
    p.z = __fmaf_rn(v.z, hd, p.z);
    pos[i] = p;
}

// R24: K, W, P[3], L[3], M, C[3] as fp64 sums of fp32 data.  Grid-stride accumulation per thread, shuffle tree per
// warp, fixed-order fold per block, and the last block to finish (ticket) folds the block partials in block order,
// so the result does not depend on scheduling.
constexpr int kDiagN = 12;
constexpr int kDiagThreads = 256;

__device__ __forceinline__ void diag_warp_reduce(double (&s)[kDiagN]) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int k = 0; k < kDiagN; ++k) s[k] += __shfl_down_sync(0xFFFFFFFFu, s[k], o);
}

__global__ void __launch_bounds__(kDiagThreads) k_diagnostics(const float4* __restrict__ pos,
                                                              const float4* __restrict__ vel,
                                                              const float4* __restrict__ acc, uint32_t n,
                                                              double* __restrict__ partial, Control* __restrict__ ctl,
                                                              double* __restrict__ out) {
    __shared__ double s_w[kDiagThreads / 32][kDiagN];
    __shared__ bool s_last;
    double s[kDiagN];
#pragma unroll
    for (int k = 0; k < kDiagN; ++k) s[k] = 0.0;
    for (uint32_t i = blockIdx.x * kDiagThreads + threadIdx.x; i < n; i += gridDim.x * kDiagThreads) {
        const float4 p = __ldg(&pos[i]), v = __ldg(&vel[i]), a = __ldg(&acc[i]);
        const double x = p.x, y = p.y, z = p.z, m = p.w, vx = v.x, vy = v.y, vz = v.z;
        s[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        s[1] += 0.5 * m * (double)a.w;
        s[2] += m * vx; s[3] += m * vy; s[4] += m * vz;
        s[5] += m * (y * vz - z * vy);
        s[6] += m * (z * vx - x * vz);
        s[7] += m * (x * vy - y * vx);
        s[8] += m;
        s[9] += m * x; s[10] += m * y; s[11] += m * z;
    }
    diag_warp_reduce(s);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0)
#pragma unroll
        for (int k = 0; k < kDiagN; ++k) s_w[w][k] = s[k];
    __syncthreads();
    if (threadIdx.x < kDiagN) {
        double t = 0.0;
        for (int k = 0; k < kDiagThreads / 32; ++k) t += s_w[k][threadIdx.x];
        __stcg(&partial[(size_t)blockIdx.x * kDiagN + threadIdx.x], t);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&ctl->diag_ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x < kDiagN) {
        double t = 0.0;
        for (uint32_t b = 0; b < gridDim.x; ++b) t += __ldcg(&partial[(size_t)b * kDiagN + threadIdx.x]);
        out[threadIdx.x] = t;
    }
    if (threadIdx.x == 0) ctl->diag_ticket = 0;  // ready for the next call
}

// ---- block time-steps (R26, R27) -----------------------------------------------------------------------
// Rung of a particle: the smallest k with dt_max 2^-k <= eta sqrt(eps / |a|), fp64 on the fp32 acceleration, every
// operation rounded once in the order written (no contraction), clamped to kmax.
__device__ __forceinline__ uint32_t rung_of(const float4 a, double eta, double eps, double dt_max, uint32_t kmax) {
    const double ax = a.x, ay = a.y, az = a.z;
    const double a2 = __dadd_rn(__dadd_rn(__dmul_rn(ax, ax), __dmul_rn(ay, ay)), __dmul_rn(az, az));
    if (!(a2 > 0.0)) return 0u;
    const double crit = __dmul_rn(eta, sqrt(eps / sqrt(a2)));
    uint32_t k = 0;
    while (k < kmax && ldexp(dt_max, -(int)k) > crit) ++k;
    return k;
}

__global__ void __launch_bounds__(256) k_rungs(const float4* __restrict__ acc, uint32_t n, float eta, float eps,
                                               float dt_max, uint32_t kmax, const uint8_t* __restrict__ mask,
                                               unsigned long long tick, uint8_t* __restrict__ rung, int init) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (!init && mask && !mask[i]) return;
    const uint32_t want = rung_of(__ldg(&acc[i]), (double)eta, (double)eps, (double)dt_max, kmax);
    if (init) {
        rung[i] = (uint8_t)want;
        return;
    }
    const uint32_t cur = rung[i];
    if (want > cur) rung[i] = (uint8_t)want;                                          // finer at once
    else if (want < cur && (tick % (1ull << (kmax - (cur - 1u)))) == 0ull) rung[i] = (uint8_t)(cur - 1u);  // nested
}

__global__ void __launch_bounds__(256) k_active_mask(const uint8_t* __restrict__ rung, uint32_t n, uint32_t kmax,
                                                     unsigned long long tick, uint8_t* __restrict__ mask) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    mask[i] = ((tick % (1ull << (kmax - rung[i]))) == 0ull) ? 1 : 0;
}

// v <- fma(a, dt_max 2^-(rung+1), v) for the masked-in particles: half a step of the particle's own size.
__global__ void __launch_bounds__(256) k_kick_rungs(float4* __restrict__ vel, const float4* __restrict__ acc,
                                                    const uint8_t* __restrict__ rung, const uint8_t* __restrict__ mask,
                                                    uint32_t n, float dt_max) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (mask && !mask[i]) return;
    const float h = ldexpf(dt_max, -(int)rung[i] - 1);
    float4 v = vel[i];
    const float4 a = __ldg(&acc[i]);
    v.x = __fmaf_rn(a.x, h, v.x);
    v.y = __fmaf_rn(a.y, h, v.y);
    v.z = __fmaf_rn(a.z, h, v.z);
    vel[i] = v;
}

cudaError_t stage_rungs(Ctx* c, const float4* acc, uint32_t n, float eta, float eps, float dt_max, uint32_t kmax,
                        const uint8_t* mask, unsigned long long tick, uint8_t* rung, int init) {
    k_rungs<<<div_up(n, 256), 256, 0, c->stream>>>(acc, n, eta, eps, dt_max, kmax, mask, tick, rung, init);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_active_mask(Ctx* c, const uint8_t* rung, uint32_t n, uint32_t kmax, unsigned long long tick,
                              uint8_t* mask) {
    k_active_mask<<<div_up(n, 256), 256, 0, c->stream>>>(rung, n, kmax, tick, mask);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_kick_rungs(Ctx* c, float4* vel, const float4* acc, const uint8_t* rung, const uint8_t* mask,
                             uint32_t n, float dt_max) {
    k_kick_rungs<<<div_up(n, 256), 256, 0, c->stream>>>(vel, acc, rung, mask, n, dt_max);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_kick(Ctx* c, float4* vel, const float4* acc, uint32_t n, float h, const uint8_t* mask) {
    k_kick<<<div_up(n, 256), 256, 0, c->stream>>>(vel, acc, n, h, mask);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_drift(Ctx* c, float4* pos, const float4* vel, uint32_t n, float h) {
    k_drift<<<div_up(n, 256), 256, 0, c->stream>>>(pos, vel, n, h);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_kick_drift(Ctx* c, float4* pos, float4* vel, const float4* acc, uint32_t n, float hk, float hd) {
    k_kick_drift<<<div_up(n, 256), 256, 0, c->stream>>>(pos, vel, acc, n, hk, hd);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t stage_diagnostics(Ctx* c, const float4* pos, const float4* vel, const float4* acc, uint32_t n, double* out) {
    const uint32_t blocks = min(div_up(n, kDiagThreads * 4), (uint32_t)kDiagMaxBlocks);
    k_diagnostics<<<blocks, kDiagThreads, 0, c->stream>>>(pos, vel, acc, n, c->b.diag_partial, c->b.ctl, out);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace bonsai
