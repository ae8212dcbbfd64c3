"""Pins of the refreshed-tree oracle (oracle/refresh_oracle.cpp, oracle.refresh; R25).  CPU only."""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W

N, THETA, EPS = 4096, 0.75, 0.01


@pytest.fixture(scope="module")
def base():
    pm, vel = W.plummer(N, with_velocities=True)
    return pm, vel, O.full_step(pm, THETA, EPS)


def _drifted(pm, vel, t):
    out = pm.copy()
    out[:, :3] = (pm[:, :3].astype(np.float64) + vel.astype(np.float64) * t).astype(np.float32)
    return out


def _centres(step):
    """Geometric centres of all cells from the frozen keys, independent numpy route (R8)."""
    t = step.tree
    q = np.array([O.decode_key(step.sorted_keys[f]) for f in t.first], dtype=np.int64)   # [n_cells, 3]
    L = t.level.astype(np.int64)
    ca = np.where(L[:, None] == 0, 0, q >> (30 - L[:, None]))
    l = step.side / 2.0 ** L
    return step.lo.astype(np.float64)[None, :] + (ca + 0.5) * l[:, None], l


def test_zero_motion_reproduces_the_fresh_build(base):
    pm, vel, s = base
    r = O.refreshed_step(s, pm, THETA, EPS)
    assert np.array_equal(r.sorted_pos_mass, s.sorted_pos_mass)
    for name in ("com_m", "quad", "delta"):
        assert np.array_equal(getattr(r.tree, name), getattr(s.tree, name)), name
    assert np.all(r.tree.lside >= s.tree.lside)
    assert (r.tree.lside == s.tree.lside).mean() > 0.999      # only R4 rounding can push a member out of its cell
    assert np.array_equal(r.groups.first, s.groups.first) and np.array_equal(r.groups.bmin, s.groups.bmin)
    same = r.tree.lside == s.tree.lside
    if same.all():
        assert np.array_equal(r.walk.n_pc, s.walk.n_pc)
        assert np.array_equal(r.walk.acc, s.walk.acc)


@pytest.mark.parametrize("t", [0.0, 0.02, 0.2])
def test_extent_side_contains_members_and_is_minimal(base, t):
    pm, vel, s = base
    r = O.refresh(s, _drifted(pm, vel, t))
    g, l = _centres(s)
    tr = r.tree
    x = r.sorted_pos_mass[:, :3].astype(np.float64)
    grew = 0
    for c in range(tr.n_cells):
        xs = x[tr.first[c]:tr.first[c] + tr.count[c]]
        ext = np.abs(xs - g[c]).max()
        want = max(l[c], 2.0 * ext)
        assert tr.lside[c] == np.float32(want), c
        grew += want > l[c]
    if t == 0.2:
        assert grew > 0.5 * tr.n_cells       # most cells have lost a member across their boundary by then
    # topology, keys and membership are frozen
    for name in ("level", "first", "count", "first_child", "n_child", "parent"):
        assert np.array_equal(getattr(tr, name), getattr(s.tree, name))
    assert np.array_equal(r.perm, s.perm) and np.array_equal(r.sorted_keys, s.sorted_keys)
    assert np.array_equal(r.groups.first, s.groups.first) and np.array_equal(r.groups.count, s.groups.count)
    # group boxes follow the particles
    k = 3
    f, cnt = r.groups.first[k], r.groups.count[k]
    members = r.sorted_pos_mass[r.groups.active_list[f:f + cnt], :3]
    assert np.array_equal(r.groups.bmin[k], members.min(axis=0)) and np.array_equal(r.groups.bmax[k], members.max(axis=0))


def test_theta_zero_on_refreshed_tree_is_direct_sum(base):
    pm, vel, s = base
    pm2 = _drifted(pm[:512].copy(), vel[:512], 0.1)
    s0 = O.build(pm[:512])
    r = O.refreshed_step(s0, pm2, 0.0, EPS)
    acc_d, pot_d = O.direct(r.sorted_pos_mass, EPS)
    assert np.allclose(r.walk.acc, acc_d, rtol=1e-12, atol=1e-13)
    assert np.allclose(r.walk.pot, pot_d, rtol=1e-12)


def test_refreshed_force_stays_accurate_and_costs_more(base):
    pm, vel, s = base
    errs, cost = {}, {}
    for t in (0.02, 0.1):
        pm2 = _drifted(pm, vel, t)
        r = O.refreshed_step(s, pm2, THETA, EPS)
        f = O.full_step(pm2, THETA, EPS)
        for tag, st in (("refresh", r), ("fresh", f)):
            acc_d, _ = O.direct(st.sorted_pos_mass, EPS)
            e = np.linalg.norm(st.walk.acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
            errs[tag, t] = np.median(e)
            cost[tag, t] = st.walk.n_pc.mean() + st.walk.n_pp.mean()
        # a refreshed tree is still a valid Barnes-Hut force for the new positions: same order of error as a rebuild
        assert errs["refresh", t] < 2.0 * errs["fresh", t]
        # and it costs more, increasingly so
        assert cost["refresh", t] > cost["fresh", t]
    assert cost["refresh", 0.1] / cost["fresh", 0.1] > cost["refresh", 0.02] / cost["fresh", 0.02]


def test_rebuild_policy_fires_after_the_drift_and_not_before(base):
    """R30: the rule compares the interactions per walked sink of the last walk with those of the first walk
    after the last build.  Pinned on the very drift that test_refreshed_force_stays_accurate_and_costs_more shows to
    raise the cost: fed with a fresh walk (reference) and then refreshed walks after growing drifts, the policy stays
    quiet while the ratio is below the factor and fires once it is above -- the ratios recomputed here from the
    walk counts by numpy."""
    pm, vel, s = base
    pol = O.RebuildPolicy(factor=1.25)
    assert pol.decide() is False                       # no reference yet: never rebuild
    everyone = np.ones(N, bool)
    pol.record(s.walk, everyone)
    ref = (s.walk.n_pp.astype(np.float64).sum() + s.walk.n_pc.astype(np.float64).sum()) / N
    assert pol.ref == ref and pol.last == ref and pol.fresh is False
    assert pol.decide() is False                       # ratio 1
    fired = []
    for t in (0.01, 0.05, 0.2, 0.5):
        r = O.refreshed_step(s, _drifted(pm, vel, t), THETA, EPS)
        pol.record(r.walk, everyone)
        ratio = (r.walk.n_pp.astype(np.float64).sum() + r.walk.n_pc.astype(np.float64).sum()) / N / ref
        assert pol.ref == ref                          # the reference is the walk after the build, not a later one
        fired.append((ratio, pol.decide()))
        assert fired[-1][1] == (ratio > float(np.float32(1.25)))
    assert fired[0][1] is False and fired[-1][1] is True, fired
    assert all(fired[k][0] < fired[k + 1][0] for k in range(3)), fired     # the cost grows with the drift
    # a rebuild resets the reference
    pol.built()
    f = O.full_step(_drifted(pm, vel, 0.5), THETA, EPS)
    pol.record(f.walk, everyone)
    assert pol.decide() is False and pol.ref < fired[-1][0] * ref


def test_block_ticks_with_the_policy_rebuild_when_it_says_so():
    """oracle.block_tick(policy=...) rebuilds exactly at the ticks the policy fires, refreshes otherwise, and a
    masked tick records only the walked sinks."""
    n, theta, eps, eta, dt_max, kmax = 2048, 0.75, 0.01, 0.3, 1 / 4, 2
    pm, vel = W.plummer(n, with_velocities=True)
    p, v = pm.copy(), O._vel4(vel)
    ap = O.force_f32(p, theta, eps)
    r = O.rungs(ap, eta, eps, dt_max, kmax)
    pol = O.RebuildPolicy(factor=1.02)
    prev = None
    kinds = []
    for tick in range(12):
        s, na = O.block_tick(p, v, ap, r, tick, theta, eps, eta, dt_max, kmax, prev=prev, policy=pol)
        fresh_tree = np.array_equal(s.lo, O.box(p)[0]) and np.array_equal(s.perm, O.sort(O.keys(p, *O.box(p))))
        kinds.append(fresh_tree)
        prev = s
    assert kinds[0] is True                               # no tree yet: built
    assert len(pol.decisions) == 11                       # one decision per tick that had a tree
    for k, d in enumerate(pol.decisions):                 # a fired decision means a fresh sort of the CURRENT positions
        if d:
            assert kinds[k + 1]
    assert any(pol.decisions) and not all(pol.decisions)
