"""Randomised cross-checks of the kernel choices that must not change any result:
the number of sort passes (params.sort_passes: the permutation, the sorted keys and the tree are the same bit for
bit whether 4, 5 or 6 passes run) and the two multipole kernels (params.mult_kernel: same cell records bit for bit).
Inputs are seeded mixtures of a Plummer sphere and Gaussian clumps whose width is drawn log-uniformly between 1e-1 and
1e-7 of the sphere -- from harmless to far below the cells any pass count resolves -- plus exact duplicates.  Every
case is also compared with the oracle in full (structure, multipoles, groups)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from test_gpu_parity import _dev, check_groups, check_structure  # noqa: E402


def _clumpy(seed: int):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(1, 120_000)) if seed % 4 else int(rng.integers(1, 3000))
    pm = W.plummer(n, seed=seed + 1)
    n_clumps = int(rng.integers(0, 6))
    for _ in range(n_clumps):
        if n < 4:
            break
        size = int(min(n // 2, rng.integers(2, 5000)))
        at = int(rng.integers(0, n - size + 1))
        width = 10.0 ** (-rng.uniform(1.0, 7.0))
        centre = pm[int(rng.integers(0, n)), :3].astype(np.float64)
        pm[at:at + size, :3] = (centre + rng.normal(size=(size, 3)) * width).astype(np.float32)
        if rng.random() < 0.3:  # exact duplicates inside the clump
            k = max(1, size // 3)
            pm[at:at + k, :3] = pm[at, :3]
    return pm[rng.permutation(n)]


def _build(pm, **kw):
    b = Bonsai(pm.shape[0], **kw)
    b.load(_dev(pm)); b.build_tree(); b.compute_multipoles(); b.sync()
    c = b.cells()
    g = b.groups()
    return b, dict(perm=b.perm(), keys=b.keys(), pos=b.sorted_pos().view(np.uint32), n_cells=c.n_cells,
                links=np.stack([c.level, c.first, c.count, c.first_child, c.n_child, c.parent]),
                mac=np.concatenate([c.com_m.view(np.uint32).ravel(), c.delta.view(np.uint32), c.lside.view(np.uint32)]),
                quad=c.walk_quad.view(np.uint32), g_first=g.first, g_count=g.count,
                g_box=np.concatenate([g.bmin.view(np.uint32).ravel(), g.bmax.view(np.uint32).ravel()]))


def _same(a, b, what):
    for k in a:
        assert np.array_equal(a[k], b[k]), f"{what}: {k} differs"


@pytest.mark.parametrize("seed", range(40))
def test_sort_pass_count_and_multipole_kernel_do_not_change_the_result(seed):
    pm = _clumpy(seed)
    b, ref = _build(pm, sort_passes=6, mult_kernel=1)
    _same(ref, _build(pm, sort_passes=4, mult_kernel=2)[1], "4 passes + tiles")
    _same(ref, _build(pm, sort_passes=5, mult_kernel=2 if seed % 2 else 1)[1], "5 passes")
    # and every case against the oracle in full: box, keys, permutation, sorted particles, all link arrays and level
    # offsets bit-exact, multipoles <= 1 ulp, groups and their boxes bit-exact
    o = O.build(pm)
    check_structure(b, o)
    check_groups(b, o)
