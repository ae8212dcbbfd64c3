"""Pins for the MAC / accuracy variants of row f3 (CPU only): oracle/mac_oracle.cpp (R28, tight particle boxes for the
cell size and centre) and the monopole-only branch of oracle_walk (R29).  P:L30: the MAC "sets the trade-off between
speed and accuracy".

Nothing here re-types the oracle's formula: the boxes are pinned by numpy brute force (containment + minimality),
delta_t by the numpy COM, the monopole branch by its convergence ORDER on a point cluster ((s/d)^2 where the
quadrupole-accurate term has (s/d)^3) and by theta = 0 == direct summation, the variants together by the ordering
the mathematics fixes: l_t <= l, so at equal theta the tight MAC accepts a superset of the geometric MAC's cells and
costs less; a quadrupole walk is more accurate than a monopole walk on the same lists; every variant's error against
direct summation falls monotonically with theta.
"""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W


def test_tight_box_contains_members_and_is_minimal():
    n = 5000
    s = O.build(W.plummer(n))
    t = s.tree
    geo_l, geo_delta = t.lside.copy(), t.delta.copy()
    box = O.tight_mac(s.sorted_pos_mass, t)
    x = s.sorted_pos_mass[:, :3]
    m = s.sorted_pos_mass[:, 3].astype(np.float64)
    for c in range(0, t.n_cells, 3):
        xs = x[t.first[c]:t.first[c] + t.count[c]]
        mn, mx = xs.min(axis=0), xs.max(axis=0)
        assert np.array_equal(box[c, :3], mn) and np.array_equal(box[c, 3:], mx)      # exact fp32 min / max
        lt = (mx.astype(np.float64) - mn.astype(np.float64)).max()
        assert t.lside[c] == np.float32(lt)
        mm = m[t.first[c]:t.first[c] + t.count[c]]
        com = (mm[:, None] * xs.astype(np.float64)).sum(axis=0) / mm.sum()
        centre = 0.5 * (mn.astype(np.float64) + mx.astype(np.float64))
        assert np.isclose(t.delta[c], np.linalg.norm(com - centre), rtol=1e-6, atol=1e-12)
    # the particle box lies inside the geometric cell (up to the fp32 rounding of the key quantisation, R4)
    assert (t.lside <= geo_l * (1 + 1e-6)).all()
    # single-particle cells are points
    one = t.count == 1
    assert one.any() and (t.lside[one] == 0).all() and (t.delta[one] == 0).all()
    # the COM lies inside the box, so delta_t <= half the box diagonal
    assert (t.delta <= 0.5 * np.sqrt(3.0) * t.lside * (1 + 1e-6) + 1e-12).all()
    assert not np.array_equal(geo_delta, t.delta)


def test_tight_mac_accepts_a_superset_at_equal_theta():
    """l_t <= l and |COM - c_t| differs from |COM - g| by at most the centre shift, which the shrinkage of l pays for:
    on a Plummer sphere the tight MAC's interaction lists are SHORTER for every group, and every cell the geometric
    MAC accepts is covered by accepted cells of the tight MAC (it never opens something the geometric one accepts,
    except where delta grew -- counted, must be rare)."""
    n, theta = 8000, 0.75
    pm = W.plummer(n)
    sg = O.build(pm, mac_mode=0)
    st = O.build(pm, mac_mode=1)
    assert np.array_equal(sg.perm, st.perm) and sg.tree.n_cells == st.tree.n_cells
    wg = O.walk(theta, 0.01, sg.sorted_pos_mass, sg.tree, sg.groups)
    wt = O.walk(theta, 0.01, st.sorted_pos_mass, st.tree, st.groups)
    cost_g = wg.n_pp.astype(np.int64) + wg.n_pc
    cost_t = wt.n_pp.astype(np.int64) + wt.n_pc
    assert cost_t.sum() < 0.9 * cost_g.sum()
    assert (cost_t <= cost_g).mean() > 0.99


@pytest.mark.parametrize("mac_mode", [0, 1])
@pytest.mark.parametrize("order", [1, 2])
def test_theta_zero_is_direct_for_every_variant(mac_mode, order):
    n, eps = 2000, 0.01
    pm = W.plummer(n)
    s = O.full_step(pm, 0.0, eps, mac_mode=mac_mode, order=order)
    acc, pot = O.direct(s.sorted_pos_mass, eps)
    assert (s.walk.n_pc == 0).all() and (s.walk.n_pp == n - 1).all()
    assert np.allclose(s.walk.acc, acc, rtol=1e-11, atol=1e-12) and np.allclose(s.walk.pot, pot, rtol=1e-12)


def _cluster_error(order, d, s_half=0.05, n_src=12):
    """One accepted cell (a tight cluster of n_src unequal masses about the origin, asymmetric so that its quadrupole
    does not vanish) seen by one far sink at distance d: relative error of the walk's acceleration and potential
    against direct summation."""
    rng = np.random.default_rng(3)
    src = np.zeros((n_src, 4), np.float32)
    src[:, :3] = (rng.uniform(-1, 1, size=(n_src, 3)) * np.array([1.0, 0.6, 0.3]) * s_half).astype(np.float32)
    src[:, 3] = rng.uniform(0.5, 1.5, size=n_src).astype(np.float32)
    sink = np.array([[d * 0.6, d * 0.64, d * 0.48, 1e-3]], np.float32)
    pm = np.concatenate([src, sink])
    # nleaf = n_src: the root (n_src + 1 particles) is internal, the cluster is one leaf cell; tight MAC: accepted
    step = O.full_step(pm, 1.0, 0.0, nleaf=n_src, ncrit=1, group_mode=0, mac_mode=1, order=order)
    i = int(np.nonzero(step.perm == n_src)[0][0])       # the sink in sorted order
    assert step.walk.n_pc[i] >= 1 and step.walk.n_pp[i] == 0, "the cluster must be seen as cells only"
    acc, pot = O.direct(step.sorted_pos_mass, 0.0, np.array([i], np.uint32))
    ea = np.linalg.norm(step.walk.acc[i] - acc[0]) / np.linalg.norm(acc[0])
    ep = abs((step.walk.pot[i] - pot[0]) / pot[0])
    return ea, ep


def test_monopole_and_quadrupole_convergence_orders():
    """A multipole expansion about the COM truncated after the monopole has relative error ~ (s/d)^2 (the dipole
    vanishes), after the quadrupole ~ (s/d)^3: doubling d must cut the error by ~4 and ~8."""
    # cluster half-size 0.2: the truncation errors stay far above the fp32 rounding of the stored M, COM, Q (~6e-8)
    e1 = [_cluster_error(1, d, s_half=0.2) for d in (2.0, 4.0, 8.0)]
    e2 = [_cluster_error(2, d, s_half=0.2) for d in (2.0, 4.0, 8.0)]
    for k in range(2):
        r1a, r1p = e1[k][0] / e1[k + 1][0], e1[k][1] / e1[k + 1][1]
        r2a, r2p = e2[k][0] / e2[k + 1][0], e2[k][1] / e2[k + 1][1]
        assert 3.3 < r1a < 4.8 and 3.3 < r1p < 5.8, (r1a, r1p)     # the potential mixes in the next order sooner
        assert 6.2 < r2a < 9.8 and 6.2 < r2p < 9.8, (r2a, r2p)
    assert all(e2[k][0] < 0.2 * e1[k][0] for k in range(3))


def test_error_cost_curves_against_direct():
    """N = 4096 against oracle_direct: for each of the four variants the median force error falls monotonically
    with theta while the cost rises; at equal theta monopole-only is less accurate than quadrupole on the same
    lists, and the tight MAC is cheaper than the geometric one."""
    n, eps = 4096, 0.01
    pm = W.plummer(n)
    thetas = (1.0, 0.75, 0.5, 0.3)
    res = {}
    for mac_mode in (0, 1):
        b = O.build(pm, mac_mode=mac_mode)
        acc_d, pot_d = O.direct(b.sorted_pos_mass, eps)
        for order in (1, 2):
            rows = []
            for theta in thetas:
                w = O.walk(theta, eps, b.sorted_pos_mass, b.tree, b.groups, order=order)
                err = np.linalg.norm(w.acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
                rows.append((float(np.median(err)), float((w.n_pp.astype(np.int64) + w.n_pc).mean())))
            res[(mac_mode, order)] = rows
            assert all(rows[k + 1][0] < rows[k][0] for k in range(3)), (mac_mode, order, rows)
            assert all(rows[k + 1][1] > rows[k][1] for k in range(3)), (mac_mode, order, rows)
    for mac_mode in (0, 1):
        for k in range(4):
            assert res[(mac_mode, 2)][k][0] < res[(mac_mode, 1)][k][0]          # quadrupole beats monopole
            assert res[(mac_mode, 2)][k][1] == res[(mac_mode, 1)][k][1]         # ... on identical lists
    for order in (1, 2):
        for k in range(4):
            assert res[(1, order)][k][1] < res[(0, order)][k][1]                # tight MAC is cheaper


def test_lists_account_for_all_mass_with_the_tight_mac():
    n, theta = 5000, 0.75
    s = O.build(W.plummer(n), mac_mode=1)
    t, g = s.tree, s.groups
    for G in range(0, g.n_groups, max(1, g.n_groups // 25)):
        pc, pp = O.walk_lists(theta, t, g.bmin[G], g.bmax[G])
        cover = np.zeros(n, np.int32)
        for c in np.concatenate([pc, pp]):
            cover[t.first[c]:t.first[c] + t.count[c]] += 1
        assert (cover == 1).all()
        mine = g.active_list[g.first[G]:g.first[G] + g.count[G]]
        for c in pc:  # a group's own particles are never inside an accepted cell (self-term removal, R11)
            assert not ((mine >= t.first[c]) & (mine < t.first[c] + t.count[c])).any()


def test_refreshed_tree_with_the_tight_mac_equals_a_tight_mac_on_the_moved_particles():
    """R28 + R25: with the tight MAC a refreshed tree needs no grown cell side -- the boxes are simply those of the
    new positions.  theta = 0 is still direct summation; the structure is the frozen one."""
    n, eps = 3000, 0.01
    pm, vel = W.plummer(n, with_velocities=True)
    prev = O.build(pm, mac_mode=1)
    pm2 = pm.copy()
    pm2[:, :3] += (vel * np.float32(0.05)).astype(np.float32)
    s = O.refresh(prev, pm2, mac_mode=1)
    assert np.array_equal(s.perm, prev.perm) and np.array_equal(s.tree.first, prev.tree.first)
    box = O.tight_mac(s.sorted_pos_mass, s.tree)   # idempotent: recomputing changes nothing
    x = s.sorted_pos_mass[:, :3]
    for c in range(0, s.tree.n_cells, 7):
        xs = x[s.tree.first[c]:s.tree.first[c] + s.tree.count[c]]
        assert np.array_equal(box[c, :3], xs.min(axis=0)) and np.array_equal(box[c, 3:], xs.max(axis=0))
    w = O.walk(0.0, eps, s.sorted_pos_mass, s.tree, s.groups)
    acc, pot = O.direct(s.sorted_pos_mass, eps)
    assert np.allclose(w.acc, acc, rtol=1e-11, atol=1e-12)
