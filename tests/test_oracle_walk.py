"""Pins for oracle_walk / oracle_direct (CPU only).

None of these compares the oracle with itself through the same formula: oracle_direct is pinned by an
independent vectorised numpy O(N^2) sum and by the two-body closed form; oracle_walk is pinned by
theta = 0 == direct sum (BASELINE.json north_star), by the error against the direct sum falling as theta -> 0,
by exact mass accounting of every group's lists, by the exact potential of point clusters (the
quadrupole-accurate p-c term must converge with the order a multipole expansion truncated after the
quadrupole has: relative error ~ (s/d)^3; any wrong coefficient, sign or index leaves an (s/d)^2
residual), by acc = -grad(pot) through finite differences, and by the closed forms of SURVEY.md 8(c)
(cube corners: quadrupole terms vanish; dumbbell on-axis series).
"""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W


def _numpy_direct(pm, eps, sinks):
    x = pm[:, :3].astype(np.float64)
    m = pm[:, 3].astype(np.float64)
    acc = np.zeros((len(sinks), 3))
    pot = np.zeros(len(sinks))
    for k, i in enumerate(sinks):
        d = x - x[i]
        r2 = (d * d).sum(axis=1) + float(eps) ** 2
        r2[i] = 1.0  # self term: weight set to zero below
        w = m / r2 ** 1.5
        w[i] = 0.0
        p = m / np.sqrt(r2)
        p[i] = 0.0
        acc[k] = (w[:, None] * d).sum(axis=0)
        pot[k] = -p.sum()
    return acc, pot


def test_direct_two_body_closed_form():
    # softened Newton: a = m2 d / (d^2 + eps^2)^(3/2) towards the other body, pot = -m2 / sqrt(d^2+eps^2)
    pm = np.array([[0, 0, 0, 2.0], [3.0, 4.0, 0, 5.0]], np.float32)
    eps = np.float32(0.5)
    acc, pot = O.direct(pm, eps)
    r2 = 25.0 + 0.25
    assert np.allclose(acc[0], 5.0 * np.array([3.0, 4.0, 0]) / r2 ** 1.5, rtol=1e-14)
    assert np.allclose(acc[1], -2.0 * np.array([3.0, 4.0, 0]) / r2 ** 1.5, rtol=1e-14)
    assert np.isclose(pot[0], -5.0 / np.sqrt(r2), rtol=1e-14)
    assert np.isclose(pot[1], -2.0 / np.sqrt(r2), rtol=1e-14)


def test_direct_vs_numpy():
    pm = W.plummer(1500)
    sinks = np.arange(0, 1500, 7, dtype=np.uint32)
    acc, pot = O.direct(pm, 0.01, sinks)
    a2, p2 = _numpy_direct(pm, np.float32(0.01), sinks)
    assert np.allclose(acc, a2, rtol=1e-11, atol=1e-13)
    assert np.allclose(pot, p2, rtol=1e-12)
    # momentum conservation of the full pairwise sum: sum m_i a_i = 0
    acc_all, pot_all = O.direct(pm, 0.01)
    f = (pm[:, 3:4].astype(np.float64) * acc_all).sum(axis=0)
    assert np.abs(f).max() < 1e-12


@pytest.mark.parametrize("mode,ncrit", [(1, 32), (0, 64)])
def test_theta_zero_equals_direct(mode, ncrit):
    n, eps = 3000, 0.01
    pm = W.plummer(n)
    s = O.full_step(pm, 0.0, eps, ncrit=ncrit, group_mode=mode)
    acc, pot = O.direct(s.sorted_pos_mass, eps)
    w = s.walk
    assert (w.n_pc == 0).all() and (w.n_pp == n - 1).all()
    assert np.allclose(w.acc, acc, rtol=1e-11, atol=1e-12)
    assert np.allclose(w.pot, pot, rtol=1e-12)


def test_error_falls_with_theta_and_matches_direct_at_4096():
    """BASELINE.json north_star: BH vs direct O(N^2) at N <= 4096, error decreasing as theta -> 0."""
    n, eps = 4096, 0.01
    pm = W.plummer(n)
    b = O.build(pm, ncrit=64, group_mode=0)
    acc_d, pot_d = O.direct(b.sorted_pos_mass, eps)
    med = []
    for theta in (1.0, 0.75, 0.5, 0.3, 0.2):
        w = O.walk(theta, eps, b.sorted_pos_mass, b.tree, b.groups)
        err = np.linalg.norm(w.acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
        perr = np.abs((w.pot - pot_d) / pot_d)
        med.append((np.median(err), np.median(perr), err.max()))
    for k in range(1, len(med)):
        assert med[k][0] < med[k - 1][0] and med[k][1] < med[k - 1][1]
    # magnitudes in the range the survey's probe saw (5e-4 at 0.75, 5e-6 at 0.2 for 2^15)
    assert med[1][0] < 2e-3 and med[-1][0] < 2e-5 and med[-1][2] < 1e-3


@pytest.mark.parametrize("mode,ncrit,theta", [(1, 32, 0.75), (0, 64, 0.75), (0, 64, 0.3), (1, 64, 1.0)])
def test_lists_account_for_all_mass_exactly_once(mode, ncrit, theta):
    """Every group's p-c cells and p-p leaves are disjoint and tile [0, n): no source lost or doubled."""
    n = 6000
    s = O.build(W.plummer(n), ncrit=ncrit, group_mode=mode)
    t, g = s.tree, s.groups
    for G in range(0, g.n_groups, max(1, g.n_groups // 40)):
        pc, pp = O.walk_lists(theta, t, g.bmin[G], g.bmax[G])
        cover = np.zeros(n, np.int32)
        for c in np.concatenate([pc, pp]):
            cover[t.first[c]:t.first[c] + t.count[c]] += 1
        assert (cover == 1).all()
        assert (t.n_child[pp] == 0).all()
        # the group's own particles are never inside an accepted cell (d2 = 0 for those cells)
        mine = g.active_list[g.first[G]:g.first[G] + g.count[G]]
        for c in pc:
            assert not ((mine >= t.first[c]) & (mine < t.first[c] + t.count[c])).any()
    w = O.walk(theta, 0.01, s.sorted_pos_mass, t, g)
    assert (w.n_pp.astype(np.int64) + 1 >= g.count.min()).all()
    # counts are per group: equal for all members
    for G in range(0, g.n_groups, max(1, g.n_groups // 40)):
        mem = g.active_list[g.first[G]:g.first[G] + g.count[G]]
        assert len(set(w.n_pc[mem])) == 1 and len(set(w.n_pp[mem])) == 1
        # oracle_walk carries its own copy of the traversal: it must visit exactly the lists oracle_walk_lists returns
        # (the copy the mass-accounting and stated-inequality pins run on), group by group (R21: n_pc = accepted cells,
        # n_pp = particles of the opened leaves minus the sink itself)
        pc, pp = O.walk_lists(theta, t, g.bmin[G], g.bmax[G])
        assert int(w.n_pc[mem[0]]) == len(pc)
        assert int(w.n_pp[mem[0]]) + 1 == int(t.count[pp].astype(np.int64).sum())


def test_mac_is_the_stated_inequality():
    """accept iff d > l/theta + delta with d = distance from the group box to the cell COM (R9)."""
    n, theta = 5000, 0.6
    s = O.build(W.plummer(n), ncrit=32, group_mode=1)
    t, g = s.tree, s.groups
    G = g.n_groups // 3
    pc, pp = O.walk_lists(theta, t, g.bmin[G], g.bmax[G])
    com = t.com_m[:, :3].astype(np.float64)
    d = np.maximum(0, np.maximum(g.bmin[G].astype(np.float64) - com, com - g.bmax[G].astype(np.float64)))
    dist = np.sqrt((d * d).sum(axis=1))
    rc = t.lside.astype(np.float64) / theta + t.delta.astype(np.float64)
    margin = 1e-5 * rc
    assert (dist[pc] > rc[pc] - margin[pc]).all()
    assert (dist[pp] <= rc[pp] + margin[pp]).all()
    # every accepted cell's parent was NOT acceptable; every visited cell's ancestors were opened
    for c in np.concatenate([pc, pp]):
        p = t.parent[c]
        while p != 0xFFFFFFFF:
            assert dist[p] <= rc[p] + margin[p]
            p = t.parent[p]


def _hand_tree(cluster, sink):
    """Root (opened) -> [cluster leaf (accepted), sink leaf (own leaf, never accepted)]."""
    nc = len(cluster)
    spm = np.asarray(list(cluster) + [list(sink) + [1.0]], np.float32)
    t = O.Tree(3, np.array([0, 1, 1], np.uint32), np.array([0, 0, nc], np.uint32),
               np.array([nc + 1, nc, 1], np.uint32), np.array([1, 0, 0], np.uint32),
               np.array([2, 0, 0], np.uint32), np.array([0xFFFFFFFF, 0, 0], np.uint32), np.zeros(32, np.uint32))
    x = spm[:nc, :3].astype(np.float64)
    m = spm[:nc, 3].astype(np.float64)
    M = m.sum()
    com = (m[:, None] * x).sum(axis=0) / M
    dx = x - com
    Q = np.einsum("i,ia,ib->ab", m, dx, dx)
    t.com_m = np.zeros((3, 4), np.float32)
    t.quad = np.zeros((3, 6), np.float32)
    t.com_m[1] = [*com, M]
    t.quad[1] = [Q[0, 0], Q[1, 1], Q[2, 2], Q[0, 1], Q[0, 2], Q[1, 2]]
    t.com_m[2] = spm[nc]
    t.com_m[0] = spm[nc]            # root COM placed on the sink: d2 = 0, always opened
    t.delta = np.zeros(3, np.float32)
    t.lside = np.array([1e30, 1e-30, 1e-30], np.float32)
    g = O.Groups(1, 1, np.array([nc], np.uint32), np.array([0], np.uint32), np.array([1], np.uint32),
                 spm[nc:nc + 1, :3].copy(), spm[nc:nc + 1, :3].copy())
    return spm, t, g


def _pc_at(cluster, sink, eps=0.0):
    spm, t, g = _hand_tree(cluster, sink)
    w = O.walk(0.75, eps, spm, t, g)
    nc = len(cluster)
    assert w.n_pc[nc] == 1 and w.n_pp[nc] == 0
    return w.acc[nc], w.pot[nc], spm


def test_pc_term_converges_at_quadrupole_order():
    rng = np.random.default_rng(5)
    x = rng.uniform(-0.5, 0.5, (12, 3))
    m = rng.uniform(0.5, 1.5, 12)
    cluster = np.concatenate([x, m[:, None]], axis=1).astype(np.float32)
    u = np.array([0.36, -0.48, 0.8])
    rel_a, rel_p = [], []
    for d in (8.0, 16.0, 32.0):
        sink = (u * d).astype(np.float32)
        acc, pot, spm = _pc_at(cluster, sink)
        a_ex, p_ex = _numpy_direct(spm, 0.0, [12])
        rel_a.append(np.linalg.norm(acc - a_ex[0]) / np.linalg.norm(a_ex[0]))
        rel_p.append(abs((pot - p_ex[0]) / p_ex[0]))
    # truncation after the quadrupole: relative error ~ d^-3  (monopole only or any wrong
    # quadrupole coefficient: d^-2, ratio 4 instead of 8)
    for r in (rel_a, rel_p):
        assert 6.0 < r[0] / r[1] < 10.5 and 6.0 < r[1] / r[2] < 10.5
    assert rel_a[0] < 2e-3 and rel_p[0] < 5e-4


def test_pc_acc_is_minus_gradient_of_pot_with_softening():
    rng = np.random.default_rng(6)
    x = rng.uniform(-0.5, 0.5, (9, 3))
    cluster = np.concatenate([x, rng.uniform(0.5, 1.5, (9, 1))], axis=1).astype(np.float32)
    # sink coordinates and steps exactly representable in fp32
    s0 = np.array([2.0, -1.5, 1.25])
    h = 2.0 ** -10
    eps = 0.75
    acc, _, _ = _pc_at(cluster, s0, eps)
    grad = np.zeros(3)
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        _, pp_, _ = _pc_at(cluster, s0 + e, eps)
        _, pm_, _ = _pc_at(cluster, s0 - e, eps)
        grad[a] = (pp_ - pm_) / (2 * h)
    assert np.allclose(acc, -grad, rtol=2e-6, atol=1e-9)


def test_pc_closed_forms():
    # cube corners (half-edge s), eps = 0: Q = M s^2 I  =>  quadrupole terms vanish identically
    s_ = 0.25
    cube = [[sx * s_, sy * s_, sz * s_, 0.125] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    sink = np.array([3.0, -2.0, 6.0])
    acc, pot, _ = _pc_at(cube, sink)
    assert np.isclose(pot, -1.0 / 7.0, rtol=1e-14)
    assert np.allclose(acc, -sink / 343.0, rtol=1e-13)
    # dumbbell m at +-s on x, seen on-axis at distance d: pot = -(2m/d)(1 + s^2/d^2),
    # a = -(2m/d^2)(1 + 3 s^2/d^2)  (SURVEY.md 8(c) "p-c formula")
    m, s_, d = 0.5, 0.5, 4.0
    acc, pot, _ = _pc_at([[s_, 0, 0, m], [-s_, 0, 0, m]], np.array([d, 0, 0]))
    assert np.isclose(pot, -(2 * m / d) * (1 + s_ ** 2 / d ** 2), rtol=1e-14)
    assert np.allclose(acc, [-(2 * m / d ** 2) * (1 + 3 * s_ ** 2 / d ** 2), 0, 0], rtol=1e-14, atol=1e-18)
    # the same dumbbell seen from the perpendicular axis: pot = -(2m/d)(1 - s^2/(2 d^2)),
    # a_y = -(2m/d^2)(1 - 3 s^2/(2 d^2))   (expansion of -2m/sqrt(d^2+s^2))
    acc, pot, _ = _pc_at([[s_, 0, 0, m], [-s_, 0, 0, m]], np.array([0, d, 0]))
    assert np.isclose(pot, -(2 * m / d) * (1 - s_ ** 2 / (2 * d ** 2)), rtol=1e-14)
    assert np.allclose(acc, [0, -(2 * m / d ** 2) * (1 - 3 * s_ ** 2 / (2 * d ** 2)), 0], rtol=1e-14, atol=1e-18)


def test_two_body_through_the_tree():
    pm = np.array([[0, 0, 0, 2.0], [3.0, 4.0, 0, 5.0]], np.float32)
    s = O.full_step(pm, 0.75, 0.5, ncrit=1, group_mode=1)
    acc = s.to_load_order(s.walk.acc)
    pot = s.to_load_order(s.walk.pot)
    r2 = 25.25
    assert np.allclose(acc[0], 5.0 * np.array([3.0, 4.0, 0]) / r2 ** 1.5, rtol=1e-14)
    assert np.isclose(pot[1], -2.0 / np.sqrt(r2), rtol=1e-14)


def test_active_mask_semantics():
    """R19: the mask selects sinks only; all particles remain sources; inactive rows untouched."""
    n, eps = 3000, 0.01
    pm = W.plummer(n)
    mask = W.active_mask(pm, n // 16, "scattered")
    for mode in (0, 1):
        s = O.full_step(pm, 0.0, eps, ncrit=32, group_mode=mode, active_mask=mask)
        act_sorted = mask[s.perm].astype(bool)
        assert s.groups.n_active == n // 16
        assert (np.sort(s.groups.active_list) == np.nonzero(act_sorted)[0]).all()
        acc_d, pot_d = O.direct(s.sorted_pos_mass, eps, np.nonzero(act_sorted)[0].astype(np.uint32))
        assert np.allclose(s.walk.acc[act_sorted], acc_d, rtol=1e-11, atol=1e-12)
        assert np.isnan(s.walk.acc[~act_sorted]).all()


def test_pc_count_rises_with_n():
    """Weak pin from the paper (Results): the average number of particle-cell interactions
    grows with N (it 'doubles between N ~ 32k and 1M'); checked here on 2^12 -> 2^15."""
    out = []
    for n in (1 << 12, 1 << 15):
        s = O.build(W.plummer(n), ncrit=64, group_mode=0)
        sel = np.arange(0, s.groups.n_groups, 8, dtype=np.uint32)
        w = O.walk(0.75, 0.01, s.sorted_pos_mass, s.tree, s.groups, sel)
        walked = ~np.isnan(w.pot)
        out.append(w.n_pc[walked].mean())
    assert out[1] > 1.3 * out[0]
