"""Pins for oracle_tree / oracle_groups / oracle_multipoles (CPU only): invariants, hand cases,
brute-force numpy sums and closed forms -- never the oracle against itself."""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W


def _big(k):
    return (int(k[0]) << 60) | (int(k[1]) << 30) | int(k[2])


def _key_from_digits(digits):
    """90-bit key (three 30-bit words) from a list of leading octal digits (rest zero)."""
    d = list(digits) + [0] * (30 - len(digits))
    v = 0
    for x in d:
        v = v * 8 + x
    return [(v >> 60) & 0x3FFFFFFF, (v >> 30) & 0x3FFFFFFF, v & 0x3FFFFFFF]


@pytest.fixture(scope="module")
def step():
    return O.build(W.plummer(20000), nleaf=16, ncrit=64, group_mode=1)


def test_tree_invariants(step):
    t, sk, n = step.tree, step.sorted_keys, 20000
    big = [_big(k) for k in sk]
    assert t.level[0] == 0 and t.first[0] == 0 and t.count[0] == n and t.parent[0] == 0xFFFFFFFF
    leaf = t.n_child == 0
    # leaf <=> count <= NLEAF or level 30
    assert ((t.count <= 16) | (t.level == 30))[leaf].all()
    assert ((t.count > 16) & (t.level < 30))[~leaf].all()
    # leaves tile [0, n) in order; every particle in exactly one leaf
    cover = np.zeros(n, np.int32)
    for c in np.nonzero(leaf)[0]:
        cover[t.first[c]:t.first[c] + t.count[c]] += 1
    assert (cover == 1).all()
    lf = np.nonzero(leaf)[0]
    order = np.argsort(t.first[lf], kind="stable")
    assert (t.first[lf][order][1:] == (t.first[lf] + t.count[lf])[order][:-1]).all()
    # breadth-first numbering: levels non-decreasing, level_offsets consistent, children consecutive
    assert (np.diff(t.level.astype(np.int64)) >= 0).all()
    for L in range(31):
        a, b = t.level_offsets[L], t.level_offsets[L + 1] if L < 30 else t.level_offsets[31]
        assert (t.level[a:b] == L).all()
    assert t.level_offsets[31] == t.n_cells
    nxt = 1
    for c in range(t.n_cells):
        if leaf[c]:
            assert t.first_child[c] == 0
            continue
        assert t.first_child[c] == nxt  # children allocated in parent order
        nxt += t.n_child[c]
        ch = np.arange(t.first_child[c], t.first_child[c] + t.n_child[c])
        assert (t.parent[ch] == c).all() and (t.level[ch] == t.level[c] + 1).all()
        # children tile the parent's range, ascending digit, each child shares a (L+1)-digit prefix
        assert t.first[ch[0]] == t.first[c]
        assert (t.first[ch][1:] == (t.first[ch] + t.count[ch])[:-1]).all()
        assert t.first[ch[-1]] + t.count[ch[-1]] == t.first[c] + t.count[c]
        L1 = int(t.level[c]) + 1
        digs = []
        for k in ch:
            pre = {big[i] >> (3 * (30 - L1)) for i in range(t.first[k], t.first[k] + t.count[k])}
            assert len(pre) == 1
            digs.append(pre.pop())
        assert digs == sorted(set(digs))
    assert nxt == t.n_cells


def test_tree_hand_cases():
    # two particles in different octants, NLEAF = 1 -> root + 2 leaves
    sk = np.array([_key_from_digits([2]), _key_from_digits([5])], np.uint32)
    t = O.tree(sk, nleaf=1)
    assert t.n_cells == 3 and t.n_child.tolist() == [2, 0, 0]
    assert t.first.tolist() == [0, 0, 1] and t.count.tolist() == [2, 1, 1] and t.level.tolist() == [0, 1, 1]
    # two particles sharing k leading digits -> chain of k single-child cells, then a split
    for k in (1, 4, 11, 29):
        a = _key_from_digits([3] * k + [1])
        b = _key_from_digits([3] * k + [6])
        t = O.tree(np.array([a, b], np.uint32), nleaf=1)
        assert t.n_cells == 1 + k + 2
        assert t.n_child.tolist() == [1] * k + [2, 0, 0]
        assert t.level.tolist() == list(range(k + 1)) + [k + 1, k + 1]
    # identical keys: chain down to level 30, where the leaf holds both (more than NLEAF)
    a = _key_from_digits([7] * 30)
    t = O.tree(np.array([a, a, a], np.uint32), nleaf=2)
    assert t.n_cells == 31 and t.level[-1] == 30 and t.count[-1] == 3 and t.n_child[-1] == 0
    # n <= NLEAF: the root is the only cell
    t = O.tree(np.array([_key_from_digits([1]), _key_from_digits([2])], np.uint32), nleaf=16)
    assert t.n_cells == 1 and t.n_child[0] == 0
    # nine particles, one per octant except octant 4 which has two deeper ones, NLEAF = 1
    ks = [_key_from_digits([d]) for d in (0, 1, 2, 3)] + [_key_from_digits([4, 1]), _key_from_digits([4, 6])] + \
         [_key_from_digits([d]) for d in (5, 6, 7)]
    t = O.tree(np.array(ks, np.uint32), nleaf=1)
    assert t.n_cells == 1 + 8 + 2
    assert t.n_child.tolist() == [8, 0, 0, 0, 0, 2, 0, 0, 0, 0, 0]
    assert t.first_child[5] == 9 and t.first.tolist()[9:] == [4, 5]
    # capacity overflow is reported
    with pytest.raises(OverflowError):
        O.tree(np.array([a, a, a], np.uint32), nleaf=2, cap_cells=30)


@pytest.mark.parametrize("mode,ncrit", [(1, 64), (1, 32), (0, 64), (0, 16)])
def test_groups_partition_and_boxes(step, mode, ncrit):
    spm, t = step.sorted_pos_mass, step.tree
    n = spm.shape[0]
    for act in (None, (W.uniform(3, np.arange(n, dtype=np.uint64), 0) < 0.1).astype(np.uint8)):
        g = O.groups(mode, ncrit, spm, t, act)
        want_list = np.arange(n) if act is None else np.nonzero(act)[0]
        assert g.n_active == want_list.size and (g.active_list == want_list).all()
        # groups tile the active list in order
        assert g.first[0] == 0 and (g.first[1:] == (g.first + g.count)[:-1]).all()
        assert g.first[-1] + g.count[-1] == g.n_active and (g.count > 0).all()
        if mode == 1:
            assert (g.count[:-1] == ncrit).all() and g.count[-1] <= ncrit
        else:
            assert (g.count <= ncrit).all()
            if act is None:
                # each group is exactly a tree cell with count <= ncrit whose parent has count > ncrit
                cells = {(int(f), int(c)): i for i, (f, c) in enumerate(zip(t.first, t.count))}
                starts = {}
                for i in range(t.n_cells):
                    p = t.parent[i]
                    if t.count[i] <= ncrit and p != 0xFFFFFFFF and t.count[p] > ncrit:
                        starts[(int(t.first[i]), int(t.count[i]))] = i
                got = {(int(f), int(c)) for f, c in zip(g.first, g.count)}
                assert got == set(starts.keys())
        for k in range(0, g.n_groups, max(1, g.n_groups // 50)):
            mem = g.active_list[g.first[k]:g.first[k] + g.count[k]]
            assert (g.bmin[k] == spm[mem, :3].min(axis=0)).all()
            assert (g.bmax[k] == spm[mem, :3].max(axis=0)).all()


@pytest.mark.parametrize("ncrit,group_cell", [(32, 512), (64, 1024), (16, 16), (32, 1 << 30)])
def test_groups_cell_chunk_mode(step, ncrit, group_cell):
    """mode 2 (R13): chunks of ncrit inside the container cells (count <= group_cell, parent count > group_cell)."""
    spm, t = step.sorted_pos_mass, step.tree
    n = spm.shape[0]
    # containers from the definition, by brute force over all cells
    cont = sorted((int(t.first[i]), int(t.count[i])) for i in range(t.n_cells)
                  if (t.count[i] <= group_cell or t.n_child[i] == 0)
                  and (t.parent[i] == 0xFFFFFFFF or t.count[t.parent[i]] > group_cell))
    cont = sorted(set(cont))
    assert cont[0][0] == 0 and sum(c for _, c in cont) == n          # containers tile [0, n)
    for act in (None, (W.uniform(5, np.arange(n, dtype=np.uint64), 0) < 0.07).astype(np.uint8)):
        g = O.groups(2, ncrit, spm, t, act, group_cell)
        flag = np.ones(n, bool) if act is None else act.astype(bool)
        rank = np.concatenate([[0], np.cumsum(flag)])
        want_first, want_count = [], []
        for f, c in cont:
            r0, a = rank[f], rank[f + c] - rank[f]
            for o in range(0, a, ncrit):
                want_first.append(r0 + o)
                want_count.append(min(ncrit, a - o))
        assert g.n_groups == len(want_first)
        assert (g.first == np.array(want_first)).all() and (g.count == np.array(want_count)).all()
        assert (g.active_list == np.nonzero(flag)[0]).all()
        for k in range(0, g.n_groups, max(1, g.n_groups // 50)):
            mem = g.active_list[g.first[k]:g.first[k] + g.count[k]]
            assert (g.bmin[k] == spm[mem, :3].min(axis=0)).all()
            assert (g.bmax[k] == spm[mem, :3].max(axis=0)).all()
    # limits: group_cell = ncrit reproduces mode 0, group_cell >= n reproduces mode 1
    if group_cell == ncrit:
        g0, g2 = O.groups(0, ncrit, spm, t), O.groups(2, ncrit, spm, t, None, group_cell)
        assert (g0.first == g2.first).all() and (g0.count == g2.count).all()
    if group_cell >= n:
        g1, g2 = O.groups(1, ncrit, spm, t), O.groups(2, ncrit, spm, t, None, group_cell)
        assert (g1.first == g2.first).all() and (g1.count == g2.count).all()


def _brute(spm, b, e):
    x = spm[b:e, :3].astype(np.float64)
    m = spm[b:e, 3].astype(np.float64)
    M = m.sum()
    com = (m[:, None] * x).sum(axis=0) / M
    d = x - com
    Q = np.einsum("i,ia,ib->ab", m, d, d)
    return M, com, Q


def test_multipoles_brute_force(step):
    t, spm = step.tree, step.sorted_pos_mass
    rng = np.random.default_rng(0)
    pick = np.unique(np.concatenate([[0], rng.integers(0, t.n_cells, 400)]))
    for c in pick:
        M, com, Q = _brute(spm, t.first[c], t.first[c] + t.count[c])
        assert np.float32(M) == t.com_m[c, 3]
        assert np.allclose(t.com_m[c, :3], com, rtol=1.2e-7, atol=0)
        want = np.array([Q[0, 0], Q[1, 1], Q[2, 2], Q[0, 1], Q[0, 2], Q[1, 2]])
        scale = M * float(t.lside[c]) ** 2
        assert np.all(np.abs(t.quad[c] - want) <= 1.2e-7 * np.abs(want) + 1e-12 * scale)
        # Q positive semi-definite
        assert np.linalg.eigvalsh(Q).min() >= -1e-12 * scale
        # geometric centre and delta from integer cell coordinates
        L = int(t.level[c])
        q = O.decode_key(step.sorted_keys[t.first[c]]).astype(np.int64)
        l = step.side / 2.0 ** L
        g = step.lo.astype(np.float64) + ((q >> (30 - L) if L else q * 0) + 0.5) * l
        assert t.lside[c] == np.float32(l)
        assert abs(t.delta[c] - np.linalg.norm(com - g)) <= 1.2e-7 * np.linalg.norm(com - g) + 1e-12 * l
        # every particle of the cell lies inside its geometric cube (up to the fp32 quantisation ulp)
        x = spm[t.first[c]:t.first[c] + t.count[c], :3].astype(np.float64)
        assert (np.abs(x - g) <= 0.5 * l * (1 + 1e-5) + 1e-5).all()
    # root: total mass 1, global centre of mass, direct-sum quadrupole (BASELINE.json north_star)
    M, com, Q = _brute(spm, 0, spm.shape[0])
    assert abs(M - 1.0) < 1e-6 and abs(t.com_m[0, 3] - 1.0) < 1e-6
    assert np.allclose(t.com_m[0, :3], com, rtol=1.2e-7)


def test_multipoles_parallel_axis(step):
    """parent = sum of children shifted to the parent's COM (independent route to the same numbers)."""
    t = step.tree
    for c in np.nonzero(t.n_child > 0)[0][:300]:
        ch = np.arange(t.first_child[c], t.first_child[c] + t.n_child[c])
        m = t.com_m[ch, 3].astype(np.float64)
        x = t.com_m[ch, :3].astype(np.float64)
        M = m.sum()
        com = (m[:, None] * x).sum(axis=0) / M
        d = x - com
        q = t.quad[ch].astype(np.float64)
        Q = np.zeros(6)
        Q[:3] = q[:, :3].sum(axis=0) + (m[:, None] * d * d).sum(axis=0)
        Q[3] = q[:, 3].sum() + (m * d[:, 0] * d[:, 1]).sum()
        Q[4] = q[:, 4].sum() + (m * d[:, 0] * d[:, 2]).sum()
        Q[5] = q[:, 5].sum() + (m * d[:, 1] * d[:, 2]).sum()
        scale = M * float(t.lside[c]) ** 2
        assert abs(M - t.com_m[c, 3]) <= 3e-7 * M
        assert np.allclose(com, t.com_m[c, :3], rtol=1e-6, atol=1e-6 * t.lside[c])
        assert np.all(np.abs(Q - t.quad[c]) <= 2e-6 * scale)


def _single_cell(pm):
    s = O.build(np.asarray(pm, np.float32), nleaf=16)
    assert s.tree.n_cells == 1
    return s


def test_multipoles_closed_forms():
    # 8 equal masses on the corners of a cube with half-edge s: Q = M s^2 I, COM = centre
    s_, m = 0.25, 0.125
    corners = [[1 + sx * s_, 2 + sy * s_, -1 + sz * s_, m] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    st = _single_cell(corners)
    assert st.tree.com_m[0].tolist() == [1.0, 2.0, -1.0, 1.0]
    assert st.tree.quad[0].tolist() == [s_ * s_, s_ * s_, s_ * s_, 0, 0, 0]
    # dumbbell +-s on x: Qxx = M s^2, the rest 0
    st = _single_cell([[0.5, 0, 0, 0.5], [-0.5, 0, 0, 0.5]])
    assert st.tree.com_m[0].tolist() == [0, 0, 0, 1.0]
    assert st.tree.quad[0].tolist() == [0.25, 0, 0, 0, 0, 0]
    # off-diagonal sign/index check: masses at (1,1,0) and (-1,-1,0) -> Qxy = +M, (1,0,-1),(-1,0,1) -> Qxz = -M
    st = _single_cell([[1, 1, 0, 1], [-1, -1, 0, 1]])
    assert st.tree.quad[0].tolist() == [2, 2, 0, 2, 0, 0]
    st = _single_cell([[1, 0, -1, 1], [-1, 0, 1, 1]])
    assert st.tree.quad[0].tolist() == [2, 0, 2, 0, -2, 0]
    st = _single_cell([[0, 1, 1, 1], [0, -1, -1, 1]])
    assert st.tree.quad[0].tolist() == [0, 2, 2, 0, 0, 2]
    # unequal masses: COM at the mass-weighted mean
    st = _single_cell([[0, 0, 0, 3], [4, 0, 0, 1]])
    assert st.tree.com_m[0].tolist() == [1, 0, 0, 4]
    assert st.tree.quad[0].tolist() == [3 * 1 + 1 * 9, 0, 0, 0, 0, 0]
    # delta: root geometric centre = lo + side/2
    assert st.side == 8.0 and st.tree.lside[0] == 8.0
    assert st.tree.delta[0] == np.float32(np.sqrt(3.0 ** 2 + 4.0 ** 2 + 4.0 ** 2))
