"""Pins for oracle_box / oracle_keys / oracle_sort / oracle_reorder (CPU only).

Nothing here compares the oracle with itself: the expected values are the hand-worked
fixture tests/golden/morton_keys.txt, mathematical invariants, and numpy library routines.
"""
import os

import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W

TWO30 = float(1 << 30)


def _read_golden(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "morton_keys.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            lhs, rhs = line.split("->")
            kind, *vals = lhs.split()
            rows.append((kind, vals, [int(v) for v in rhs.split()]))
    return rows


def test_hand_worked_keys(golden_dir):
    rows = _read_golden(golden_dir)
    assert len(rows) >= 15
    for kind, vals, want in rows:
        if kind == "I":
            q = [int(v) for v in vals]
            # i / 2^30 is exact in fp32 for these; 2^30-1 is reached through the clamp at x = side
            x = [1.0 if v == (1 << 30) - 1 else v / TWO30 for v in q]
            for v, xv in zip(q, x):
                if v != (1 << 30) - 1:
                    assert float(np.float32(xv)) * TWO30 == v
        else:
            x = [float(v) for v in vals]
        pm = np.array([[x[0], x[1], x[2], 1.0]], np.float32)
        k = O.keys(pm, np.zeros(3, np.float32), 1.0)
        assert k[0].tolist() == want, (kind, vals, k[0].tolist(), want)


def test_box_power_of_two_strictly_greater():
    # extent exactly 1 -> side 2; extent 0.75 -> side 1; extent 0 -> side 1 (R3)
    pm = np.array([[0, 0, 0, 1], [1, 0.5, 0.25, 1]], np.float32)
    lo, side = O.box(pm)
    assert side == 2.0 and lo.tolist() == [0, 0, 0]
    pm = np.array([[-0.25, 3, 0, 1], [0.5, 3.5, 0.1, 1]], np.float32)
    lo, side = O.box(pm)
    assert side == 1.0 and lo.tolist() == [-0.25, 3.0, 0.0]
    pm = np.array([[7, 7, 7, 1]] * 3, np.float32)
    lo, side = O.box(pm)
    assert side == 1.0 and lo.tolist() == [7, 7, 7]
    pm = np.array([[0, 0, 0, 1], [0, 0, 33.0, 1]], np.float32)
    assert O.box(pm)[1] == 64.0
    pm = np.array([[0, 0, 0, 1], [0, 2.0 ** -20, 0, 1]], np.float32)
    assert O.box(pm)[1] == 2.0 ** -19


def _interleave_ref(q):
    """Independent restatement with Python big integers: 90-bit key value."""
    key = 0
    for L in range(1, 31):
        b = 30 - L
        d = 4 * ((int(q[0]) >> b) & 1) + 2 * ((int(q[1]) >> b) & 1) + ((int(q[2]) >> b) & 1)
        key = key * 8 + d
    return key


def test_decode_encode_identity_and_bigint():
    rng = np.random.default_rng(1)
    # fp32-representable multiples of 2^-24 in [0,1): i = k * 64
    kk = rng.integers(0, 1 << 24, size=(2000, 3))
    pm = np.zeros((2000, 4), np.float32)
    pm[:, :3] = kk / float(1 << 24)
    keys = O.keys(pm, np.zeros(3, np.float32), 1.0)
    for i in range(0, 2000, 7):
        q = O.decode_key(keys[i])
        assert q.tolist() == (kk[i] * 64).tolist()
        big = (int(keys[i, 0]) << 60) | (int(keys[i, 1]) << 30) | int(keys[i, 2])
        assert big == _interleave_ref(kk[i] * 64)
    assert keys.max() < (1 << 30)


def test_key_monotone_in_each_coordinate():
    # raising one coordinate (others fixed) never lowers the key
    base = np.array([0.3, 0.6, 0.1], np.float32)
    for a in range(3):
        xs = np.sort(np.random.default_rng(a).random(500).astype(np.float32))
        pm = np.zeros((500, 4), np.float32)
        pm[:, :3] = base
        pm[:, a] = xs
        k = O.keys(pm, np.zeros(3, np.float32), 1.0)
        big = [(int(r[0]) << 60) | (int(r[1]) << 30) | int(r[2]) for r in k]
        assert all(b1 <= b2 for b1, b2 in zip(big, big[1:]))


def test_prefix_iff_same_cell():
    # top 3L bits equal <=> all three integer coordinates agree in their top L bits
    pm = W.plummer(4096)
    lo, side = O.box(pm)
    k = O.keys(pm, lo, side)
    q = np.array([O.decode_key(r) for r in k[:512]], dtype=np.int64)
    big = [(int(r[0]) << 60) | (int(r[1]) << 30) | int(r[2]) for r in k[:512]]
    for L in (1, 3, 7, 12):
        cell = q >> (30 - L)
        for i in range(0, 512, 5):
            for j in range(i + 1, 512, 37):
                same_cell = bool((cell[i] == cell[j]).all())
                same_prefix = (big[i] >> (3 * (30 - L))) == (big[j] >> (3 * (30 - L)))
                assert same_cell == same_prefix


def test_quantisation_is_fp32_as_written():
    # R4: t = x - lo (fp32, RN), u = t * scale (fp32), trunc.  Check against numpy float32 arithmetic.
    pm = W.plummer(5000)
    lo, side = O.box(pm)
    k = O.keys(pm, lo, side)
    scale = np.float32(TWO30 / side)
    t = (pm[:, :3] - lo[None, :]).astype(np.float32)
    u = (t * scale).astype(np.float32)
    q = np.minimum(np.trunc(u.astype(np.float64)), TWO30 - 1).astype(np.int64)
    dec = np.array([O.decode_key(r) for r in k], dtype=np.int64)
    assert (dec == q).all()


def test_sort_is_stable_lexsort():
    rng = np.random.default_rng(5)
    # many duplicate keys to exercise stability
    keys = rng.integers(0, 4, size=(3000, 3)).astype(np.uint32)
    perm = O.sort(keys)
    assert sorted(perm.tolist()) == list(range(3000))  # bijection
    want = np.lexsort((np.arange(3000), keys[:, 2], keys[:, 1], keys[:, 0]))
    assert (perm == want).all()
    sk = keys[perm]
    big = [(int(r[0]) << 60) | (int(r[1]) << 30) | int(r[2]) for r in sk]
    assert all(a <= b for a, b in zip(big, big[1:]))
    for i in range(2999):
        if big[i] == big[i + 1]:
            assert perm[i] < perm[i + 1]


def test_sort_brute_force_tiny():
    keys = np.array([[1, 0, 0], [0, 5, 9], [0, 5, 9], [0, 0, 7], [1, 0, 0], [0, 5, 8]], np.uint32)
    assert O.sort(keys).tolist() == [3, 5, 1, 2, 0, 4]


def test_sort_plummer_and_reorder():
    pm = W.plummer(20000)
    lo, side = O.box(pm)
    k = O.keys(pm, lo, side)
    perm = O.sort(k)
    want = np.lexsort((np.arange(20000), k[:, 2], k[:, 1], k[:, 0]))
    assert (perm == want).all()
    spm, sk = O.reorder(pm, k, perm)
    assert (spm == pm[perm]).all() and (sk == k[perm]).all()


@pytest.mark.parametrize("n", [1, 2, 17])
def test_tiny_inputs(n):
    pm = W.plummer(n)
    lo, side = O.box(pm)
    k = O.keys(pm, lo, side)
    perm = O.sort(k)
    assert sorted(perm.tolist()) == list(range(n))
