// =====================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY (see bonsai_oracle.cpp for the rules that apply).
//
// Row f2 of DESIGN.md section 0: the time integration around the force step, and the
// conserved-quantity diagnostics.  The paper integrates with "the block time-step method"
// (P:L24 Introduction; P:L32 Results: "particles that have to be updated") and gives no
// scheme, order or precision; BASELINE.json configs[2] fixes "leapfrog steps with dt = 1/1024 and
// a shared time-step, with the tree rebuilt every step" on fp32 particle data.  Readings taken
// (R22-R24):
//
//   R22  kick-drift-kick leapfrog.  One step of size dt from (x_n, v_n, a_n = a(x_n)):
//          v_{n+1/2} = v_n + a_n (dt/2);  x_{n+1} = x_n + v_{n+1/2} dt;
//          a_{n+1} = a(x_{n+1});          v_{n+1} = v_{n+1/2} + a_{n+1} (dt/2).
//   R23  Particle state is fp32 (configs: "fp32"), so the update is DEFINED in fp32: each
//        component is ONE fused multiply-add rounded once,  v <- fma(a, h, v),  x <- fma(v, h, x),
//        with h the fp32 step passed in (the caller forms dt/2 as 0.5f * dt, exact).  A masked
//        kick touches only particles whose mask byte is non-zero (block time-steps, R19).
//   R24  Diagnostics in fp64 from the fp32 state, G = 1:
//          K = 1/2 sum m |v|^2,   W = 1/2 sum m phi   (phi = the potential the force step returned),
//          P = sum m v,   L = sum m (x cross v),   M = sum m,   C = sum m x.
//
// Pins (tests/test_oracle_integrator.py, -m "not gpu"):
//   oracle_kick / oracle_drift   exact agreement with the once-rounded fp64 evaluation of a h + v
//                                (numpy, independent route); mask semantics
//   leapfrog (python loop over these + the force oracle)
//                                two-body circular orbit against the closed form x(t) = r cos(wt):
//                                error after one period falls 4x when dt is halved (2nd order);
//                                time reversal returns to the start; energy and momentum are
//                                conserved on a Plummer sphere
//   oracle_diagnostics           closed forms for the two-body orbit (K, W, L); Plummer sphere in
//                                Henon units: K ~ 1/4, W ~ -1/2 (virial equilibrium); numpy sums
// =====================================================================================
#include <cmath>
#include <cstdint>

extern "C" {

// R23: v_a <- fma(acc_a, h, v_a) for a = x, y, z; vel4 is float[n][4] (vx, vy, vz, unused),
// acc_pot is float[n][4] (ax, ay, az, phi); mask (may be null) selects the particles that are kicked.
void oracle_kick(float* vel4, const float* acc_pot, uint32_t n, float h, const uint8_t* mask) {
    for (uint32_t i = 0; i < n; ++i) {
        if (mask && !mask[i]) continue;
        for (int a = 0; a < 3; ++a) vel4[4 * i + a] = std::fmaf(acc_pot[4 * i + a], h, vel4[4 * i + a]);
    }
}

// R23: x_a <- fma(v_a, h, x_a); the mass (pos_mass[.][3]) is untouched.  Every particle drifts.
void oracle_drift(float* pos_mass, const float* vel4, uint32_t n, float h) {
    for (uint32_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) pos_mass[4 * i + a] = std::fmaf(vel4[4 * i + a], h, pos_mass[4 * i + a]);
}

// R24: out[12] = K, W, Px, Py, Pz, Lx, Ly, Lz, M, Cx, Cy, Cz, plain fp64 sums in particle order.
void oracle_diagnostics(const float* pos_mass, const float* vel4, const float* acc_pot, uint32_t n, double* out) {
    double K = 0, W = 0, P[3] = {0, 0, 0}, L[3] = {0, 0, 0}, M = 0, Cm[3] = {0, 0, 0};
    for (uint32_t i = 0; i < n; ++i) {
        const double x = pos_mass[4 * i + 0], y = pos_mass[4 * i + 1], z = pos_mass[4 * i + 2], m = pos_mass[4 * i + 3];
        const double vx = vel4[4 * i + 0], vy = vel4[4 * i + 1], vz = vel4[4 * i + 2];
        const double phi = acc_pot[4 * i + 3];
        K += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        W += 0.5 * m * phi;
        P[0] += m * vx; P[1] += m * vy; P[2] += m * vz;
        L[0] += m * (y * vz - z * vy);
        L[1] += m * (z * vx - x * vz);
        L[2] += m * (x * vy - y * vx);
        M += m;
        Cm[0] += m * x; Cm[1] += m * y; Cm[2] += m * z;
    }
    out[0] = K; out[1] = W;
    for (int a = 0; a < 3; ++a) { out[2 + a] = P[a]; out[5 + a] = L[a]; out[9 + a] = Cm[a]; }
    out[8] = M;
}

}  // extern "C"

// =====================================================================================
// Block time-steps (row f1/f2 of DESIGN.md; "block time-step algorithm", "N_active ... the number of
// particles that have to be updated").  The paper gives no criterion or scheme.  Readings taken (R26, R27):
//
//   R26  Rungs.  Particle i steps with dt_i = dt_max 2^-k_i, k_i in [0, kmax] the SMALLEST k with
//            dt_max 2^-k <= eta sqrt(eps / |a_i|)          (fp64 on the fp32 acceleration; |a| = 0 -> k = 0),
//        clamped to kmax.  Time is counted in ticks of dt_min = dt_max 2^-kmax; i is ACTIVE at tick t iff
//        t mod 2^(kmax - k_i) == 0 (its step ends / begins there).
//   R27  One tick of the block scheme (kick-drift-kick per particle, every step aligned to its own rung):
//          opening kick of the particles active at t:      v += a (dt_i / 2)
//          drift of ALL particles:                          x += v dt_min
//          force on the particles active at t + 1 (masked walk; tree rebuilt or refreshed, R25)
//          closing kick of those:                           v += a_new (dt_i / 2)     (same rung as the opening kick)
//          new rung for those from a_new: finer at once; coarser by ONE rung, and only if t + 1 is a multiple of
//          the coarser step (so steps stay nested).
//        Kicks are the fp32 fma of R23 with h = dt_max 2^-(k+1) (an exact power-of-two scaling).
//        With kmax = 0 this is the shared-step leapfrog of R22, operation for operation.
//
// Pins (tests/test_oracle_integrator.py): rung formula against numpy; activity pattern and counts; kmax = 0
// reproduces oracle.leapfrog bit for bit; rungs only coarsen at synchronised ticks; a Plummer core with block steps
// conserves energy better than the shared dt_max step at a fraction of the force evaluations of the shared dt_min step.
// =====================================================================================
extern "C" {

static uint32_t rung_of(const float* a, double eta, double eps, double dt_max, uint32_t kmax) {
    const double ax = a[0], ay = a[1], az = a[2];
    const double a2 = (ax * ax + ay * ay) + az * az;
    if (!(a2 > 0.0)) return 0;
    const double crit = eta * std::sqrt(eps / std::sqrt(a2));
    uint32_t k = 0;
    while (k < kmax && std::ldexp(dt_max, -(int)k) > crit) ++k;
    return k;
}

// init != 0: rung[i] = R26 for every particle (mask ignored).  init == 0: the R27 update at `tick` for the particles
// with mask[i] != 0 (mask null = all).
void oracle_rungs(const float* acc_pot, uint32_t n, float eta, float eps, float dt_max, uint32_t kmax,
                  const uint8_t* mask, uint64_t tick, uint8_t* rung, int init) {
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t want = rung_of(&acc_pot[4 * i], eta, eps, dt_max, kmax);
        if (init) { rung[i] = (uint8_t)want; continue; }
        if (mask && !mask[i]) continue;
        const uint32_t cur = rung[i];
        if (want > cur) rung[i] = (uint8_t)want;
        else if (want < cur && (tick % (1ull << (kmax - (cur - 1)))) == 0) rung[i] = (uint8_t)(cur - 1);
    }
}

void oracle_active_mask(const uint8_t* rung, uint32_t n, uint32_t kmax, uint64_t tick, uint8_t* mask) {
    for (uint32_t i = 0; i < n; ++i) mask[i] = (tick % (1ull << (kmax - rung[i]))) == 0 ? 1 : 0;
}

// v_a <- fma(acc_a, dt_max 2^-(rung+1), v_a) for the particles with mask != 0 (null = all).
void oracle_kick_rungs(float* vel4, const float* acc_pot, const uint8_t* rung, const uint8_t* mask, uint32_t n, float dt_max) {
    for (uint32_t i = 0; i < n; ++i) {
        if (mask && !mask[i]) continue;
        const float h = std::ldexp(dt_max, -(int)rung[i] - 1);
        for (int a = 0; a < 3; ++a) vel4[4 * i + a] = std::fmaf(acc_pot[4 * i + a], h, vel4[4 * i + a]);
    }
}

}  // extern "C"
