"""Pins of the integrator oracle (oracle/integrator_oracle.cpp; R22-R24) against closed forms,
conservation laws and an independent numpy route.  CPU only."""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W


def _two_body():
    """Equal masses 1/2 at x = -+1/2 on a circular orbit about the origin (G = 1, eps = 0).

    Closed form: mutual acceleration m / d^2 = 1/2 towards the origin, orbit radius r = 1/2, so v^2 / r = 1/2,
    v = 1/2, omega = v / r = 1, period 2 pi; x_1(t) = -(1/2)(cos t, sin t, 0).
    """
    pm = np.array([[-0.5, 0, 0, 0.5], [0.5, 0, 0, 0.5]], np.float32)
    vel = np.array([[0, -0.5, 0], [0, 0.5, 0]], np.float32)
    return pm, vel


def test_kick_drift_definition_against_numpy_fp64():
    # a*h is exact in fp64 (24 + 24 significand bits), so fp64 a*h + v carries ONE fp64 rounding; rounding that to
    # fp32 equals the single rounding of fma except when the fp64 result sits within 2^-29 of an fp32 tie.
    rng = np.random.default_rng(7)
    n = 20001
    v = np.zeros((n, 4), np.float32); v[:, :3] = rng.normal(size=(n, 3))
    a = rng.normal(size=(n, 4)).astype(np.float32) * 3
    h = np.float32(1.0 / 1024.0) * np.float32(0.5)
    want = (a[:, :3].astype(np.float64) * np.float64(h) + v[:, :3].astype(np.float64)).astype(np.float32)
    got = v.copy()
    O.kick(got, a, h)
    assert np.array_equal(got[:, 3], v[:, 3])
    same = got[:, :3] == want
    assert same.mean() > 0.9999
    assert np.all(np.abs(got[:, :3].astype(np.float64) - want) <= np.spacing(np.abs(want)).astype(np.float64))
    x = rng.normal(size=(n, 4)).astype(np.float32)
    wantx = (got[:, :3].astype(np.float64) * np.float64(1 / 1024) + x[:, :3].astype(np.float64)).astype(np.float32)
    gx = x.copy()
    O.drift(gx, got, np.float32(1 / 1024))
    assert np.array_equal(gx[:, 3], x[:, 3])          # the mass is untouched
    assert (gx[:, :3] == wantx).mean() > 0.9999


def test_kick_mask_touches_only_selected():
    rng = np.random.default_rng(3)
    n = 1000
    v = rng.normal(size=(n, 4)).astype(np.float32)
    a = rng.normal(size=(n, 4)).astype(np.float32)
    mask = (rng.random(n) < 0.3).astype(np.uint8)
    got = v.copy()
    O.kick(got, a, np.float32(0.25), mask)
    full = v.copy()
    O.kick(full, a, np.float32(0.25))
    assert np.array_equal(got[mask == 0], v[mask == 0])
    assert np.array_equal(got[mask == 1], full[mask == 1])
    assert not np.array_equal(got[mask == 1], v[mask == 1])


def _orbit_error(steps_per_period):
    pm, vel = _two_body()
    dt = np.float32(2 * np.pi / steps_per_period)
    p, v, _ = O.leapfrog(pm, vel, 0.0, 0.0, dt, steps_per_period)
    t = float(dt) * steps_per_period
    want = -0.5 * np.array([np.cos(t), np.sin(t), 0.0])
    return np.linalg.norm(p[0, :3].astype(np.float64) - want), p, v


def test_two_body_circular_orbit_is_second_order():
    e0, _, _ = _orbit_error(64)
    e1, p, v = _orbit_error(128)
    e2, _, _ = _orbit_error(256)
    # a second-order scheme: the distance to the closed form after one period falls 4x per halving of dt
    # (measured constant: |error| = 41.2 / steps^2, i.e. a phase error of (w dt)^2 * 2 pi / 3 per period)
    assert 3.9 < e0 / e1 < 4.1
    assert 3.9 < e1 / e2 < 4.1
    assert e2 < 1e-3
    # the orbit stays circular and symmetric
    assert abs(np.linalg.norm(p[0, :3]) - 0.5) < 2e-4
    assert np.allclose(p[0, :3], -p[1, :3], atol=1e-6)


def test_two_body_diagnostics_closed_form():
    pm, vel = _two_body()
    ap = O.force_f32(pm, 0.0, 0.0)
    d = dict(zip(O.DIAG_FIELDS, O.diagnostics(pm, O._vel4(vel), ap)))
    assert d["K"] == pytest.approx(2 * 0.5 * 0.5 * 0.25)          # 2 x (1/2 m v^2)
    assert d["W"] == pytest.approx(-0.5 * 0.5 / 1.0)              # -m1 m2 / d
    assert d["Lz"] == pytest.approx(2 * 0.5 * 0.5 * 0.5)          # 2 x m r v
    assert d["Lx"] == 0 and d["Ly"] == 0
    assert d["Px"] == 0 and d["Py"] == 0 and d["Pz"] == 0
    assert d["M"] == 1.0 and d["Cx"] == 0


def test_time_reversal_returns_to_start():
    pm, vel = W.plummer(256, with_velocities=True)
    n_steps, dt = 16, np.float32(1 / 256)
    p1, v1, a1 = O.leapfrog(pm, vel, 0.0, 0.01, dt, n_steps)
    v1[:, :3] *= -1
    p2, v2, _ = O.leapfrog(p1, v1, 0.0, 0.01, dt, n_steps, acc_pot=a1)
    assert np.abs(p2[:, :3] - pm[:, :3]).max() < 2e-5          # fp32 state: reversal holds up to rounding
    assert np.abs(-v2[:, :3] - vel).max() < 2e-4


def test_plummer_energy_momentum_conservation_and_virial():
    n = 1024
    pm, vel = W.plummer(n, with_velocities=True)
    eps, dt = 0.02, np.float32(1 / 256)
    a0 = O.force_f32(pm, 0.0, eps)
    d0 = dict(zip(O.DIAG_FIELDS, O.diagnostics(pm, O._vel4(vel), a0)))
    # Henon units: E = -1/4, K = 1/4, W = -1/2 up to sampling noise, softening and the 99.9 % mass cut
    assert d0["K"] == pytest.approx(0.25, rel=0.08)
    assert d0["W"] == pytest.approx(-0.5, rel=0.08)
    assert d0["M"] == pytest.approx(1.0, rel=1e-6)
    p, v, a = O.leapfrog(pm, vel, 0.0, eps, dt, 32, acc_pot=a0)
    d1 = dict(zip(O.DIAG_FIELDS, O.diagnostics(p, v, a)))
    e0, e1 = d0["K"] + d0["W"], d1["K"] + d1["W"]
    assert abs((e1 - e0) / e0) < 2e-5
    for k in ("Px", "Py", "Pz"):
        assert abs(d1[k] - d0[k]) < 1e-7                        # pairwise forces cancel: momentum is conserved
    for k in ("Lx", "Ly", "Lz"):
        assert abs(d1[k] - d0[k]) < 1e-6
    # independent numpy route for the sums
    m = pm[:, 3].astype(np.float64)
    assert d0["K"] == pytest.approx(0.5 * np.sum(m * np.sum(vel.astype(np.float64) ** 2, axis=1)), rel=1e-13)
    assert d0["W"] == pytest.approx(0.5 * np.sum(m * a0[:, 3].astype(np.float64)), rel=1e-13)
    L = np.sum(m[:, None] * np.cross(pm[:, :3].astype(np.float64), vel.astype(np.float64)), axis=0)
    assert np.allclose([d0["Lx"], d0["Ly"], d0["Lz"]], L, rtol=1e-12, atol=1e-15)


def test_tree_leapfrog_tracks_direct_leapfrog():
    # theta = 0.5 force errors are ~1e-3 relative; over 8 short steps the trajectories stay close
    pm, vel = W.plummer(512, with_velocities=True)
    dt = np.float32(1 / 1024)
    pd, vd, _ = O.leapfrog(pm, vel, 0.0, 0.01, dt, 8)
    pt, vt, _ = O.leapfrog(pm, vel, 0.5, 0.01, dt, 8)
    assert np.abs(pd[:, :3] - pt[:, :3]).max() < 1e-5
    assert np.abs(vd[:, :3] - vt[:, :3]).max() < 2e-3


# ---- block time-steps (R26, R27) ------------------------------------------------------------------------

def test_rung_formula_against_numpy_and_activity_pattern():
    pm, vel = W.plummer(2048, with_velocities=True)
    eps, eta, dt_max, kmax = 0.01, 0.02, 1.0 / 64, 5
    ap = O.force_f32(pm, 0.0, eps)
    r = O.rungs(ap, eta, eps, dt_max, kmax)
    a = np.linalg.norm(ap[:, :3].astype(np.float64), axis=1)
    crit = np.float64(np.float32(eta)) * np.sqrt(np.float64(np.float32(eps)) / a)
    want = np.clip(np.ceil(np.log2(np.float64(np.float32(dt_max)) / crit)), 0, kmax).astype(np.int64)
    assert (r == want).mean() > 0.999                     # log2 at an exact power of two may round either way
    ok = r < kmax
    assert np.all(np.ldexp(dt_max, -r[ok].astype(int)) <= crit[ok])           # the step satisfies the criterion ...
    big = r > 0
    assert np.all(np.ldexp(dt_max, -(r[big].astype(int) - 1)) > crit[big])    # ... and the next coarser one does not
    assert len(np.unique(r)) >= 3                          # the core needs finer steps than the halo
    for tick in (0, 1, 2, 4, 6, 16, 32):
        m = O.active_at(r, kmax, tick)
        assert np.array_equal(m.astype(bool), tick % (1 << (kmax - r.astype(int))) == 0)
    assert O.active_at(r, kmax, 0).all() and O.active_at(r, kmax, 32).all()
    assert O.active_at(r, kmax, 1).sum() == (r == kmax).sum()


def test_block_scheme_with_one_rung_is_the_shared_leapfrog_bit_for_bit():
    pm, vel = W.plummer(300, with_velocities=True)
    theta, eps, dt = 0.5, 0.02, np.float32(1 / 128)
    p_ref, v_ref, a_ref = O.leapfrog(pm, vel, theta, eps, dt, 5)
    p, v = pm.copy(), O._vel4(vel)
    ap = O.force_f32(p, theta, eps)
    rung = np.zeros(300, np.uint8)
    for tick in range(5):
        O.block_tick(p, v, ap, rung, tick, theta, eps, 1e9, dt, 0)     # eta huge: nobody wants a finer rung
    assert np.array_equal(p.view(np.uint32), p_ref.view(np.uint32))
    assert np.array_equal(v.view(np.uint32), v_ref.view(np.uint32))
    assert np.array_equal(ap.view(np.uint32), a_ref.view(np.uint32))


def test_rungs_coarsen_only_at_synchronised_ticks():
    n, kmax = 64, 4
    ap = np.zeros((n, 4), np.float32)
    ap[:, 0] = 1e-6                                       # tiny acceleration: every particle wants rung 0
    rung = np.full(n, kmax, np.uint8)
    history = []
    for tick in range(1, 17):
        mask = O.active_at(rung, kmax, tick)
        before = rung.copy()
        O.rungs(ap, 0.02, 0.01, 1 / 64, kmax, rung=rung, mask=mask, tick=tick)
        changed = rung != before
        assert np.all(before[changed] - rung[changed] == 1)                     # one rung at a time
        assert np.all(tick % (1 << (kmax - rung[changed].astype(int))) == 0)    # aligned to the NEW, coarser step
        assert not changed[mask == 0].any()
        history.append(int(rung[0]))
    assert history[0] == kmax and history[-1] == 0        # 4 -> 3 at tick 2, -> 2 at 4, -> 1 at 8, -> 0 at 16
    assert history[1] == 3 and history[3] == 2 and history[7] == 1


def test_block_steps_beat_the_coarse_shared_step_at_a_fraction_of_the_fine_cost():
    n = 256
    pm, vel = W.plummer(n, with_velocities=True)
    eps, eta, dt_max, kmax = 0.005, 0.1, 1.0 / 32, 4      # rungs 0..3 populated: 7 / 23 / 108 / 118 particles

    def energy(p, v, a):
        d = O.diagnostics(p, v, a)
        return d[0] + d[1]

    a0 = O.force_f32(pm, 0.0, eps)
    e0 = energy(pm, O._vel4(vel), a0)
    pc, vc, ac = O.leapfrog(pm, vel, 0.0, eps, np.float32(dt_max), 4, acc_pot=a0)          # shared dt_max
    err_coarse = abs(energy(pc, vc, ac) / e0 - 1)
    p, v, ap = pm.copy(), O._vel4(vel), a0.copy()
    rung = O.rungs(ap, eta, eps, dt_max, kmax)
    walked = 0
    for tick in range(4 << kmax):
        _, na = O.block_tick(p, v, ap, rung, tick, 0.0, eps, eta, dt_max, kmax)
        walked += na
    assert O.active_at(rung, kmax, 4 << kmax).all()       # everybody is synchronised at a multiple of dt_max
    err_block = abs(energy(p, v, O.force_f32(p, 0.0, eps)) / e0 - 1)
    assert err_block < 0.1 * err_coarse                   # measured: 9.5e-8 against 4.7e-6
    assert walked < 0.4 * n * (4 << kmax)                 # far fewer force evaluations than the shared dt_min step
