"""Both multipole kernels (stage a5) against the oracle at sizes where the size rule would not
pick them: `mult_kernel = 2` (tiles of cells handed out deepest first, parents wait for their children; the default
from n = 2^21) on small and degenerate trees, on a refreshed tree (R25) and with the tight MAC (R28); `mult_kernel = 1`
(the last child to arrive climbs; the default below 2^21) at 2^21.  The two share the leaf sums and the combine of the
children, so their cell records must agree to the last bit."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from test_gpu_mac import check_tight_cells  # noqa: E402
from test_gpu_parity import _dev, check_groups, check_structure, check_walk, run_gpu  # noqa: E402

TILES, CLIMB = 2, 1


@pytest.mark.parametrize("n", [1, 2, 16, 17, 33, 100, 1000, 4097, 50_003])
def test_tiles_kernel_small_and_ragged_sizes(n):
    pm = W.plummer(n)
    ref = O.full_step(pm, 0.75, 0.01)
    b, out = run_gpu(pm, 0.75, 0.01, mult_kernel=TILES)
    check_structure(b, ref)
    check_groups(b, ref)
    if n > 1:
        check_walk(b, out, ref, count_frac=0.99 if n < 5000 else 0.999, eps=0.01, pm=pm)


def test_tiles_kernel_coincident_particles_and_deep_chain():
    """A level-30 leaf larger than nleaf and a single-child chain of ~20 levels: parents and children share a tile."""
    rng = np.random.default_rng(5)
    pm = W.plummer(500)
    pm[100:140, :3] = pm[100, :3]
    pm[200, :3] = pm[201, :3] + np.float32(1e-6)
    pm = pm[rng.permutation(500)]
    ref = O.full_step(pm, 0.75, 0.01)
    b, out = run_gpu(pm, 0.75, 0.01, mult_kernel=TILES)
    check_structure(b, ref)
    check_walk(b, out, ref, count_frac=0.98, eps=0.01, pm=pm)
    pm = np.zeros((20_000, 4), np.float32)
    pm[:, :3] = (1.0, 2.0, 3.0)
    pm[:, 3] = 1.0 / 20_000
    ref = O.build(pm)
    b = Bonsai(20_000, mult_kernel=TILES)
    for _ in range(2):  # twice: the tile scheduler must be back at zero after a pass
        b.load(_dev(pm)); b.build_tree(); b.compute_multipoles(); b.sync()
        check_structure(b, ref)


def test_tiles_kernel_repeated_steps_of_different_sizes():
    """The ticket and the arrival counters are reset by the pass itself: one context, sizes going up and down."""
    b = Bonsai(30_000, mult_kernel=TILES)
    for n in (30_000, 700, 12_345, 30_000):
        pm = W.plummer(n, seed=n)
        ref = O.full_step(pm, 0.75, 0.01)
        out = b.step(_dev(pm), 0.75, 0.01).cpu().numpy()
        b.sync()
        check_structure(b, ref)
        check_walk(b, out, ref, count_frac=0.99 if n < 5000 else 0.999, eps=0.01, pm=pm)


def test_tiles_kernel_on_a_refreshed_tree_and_with_the_tight_mac():
    n, theta, eps, dt = 20_000, 0.75, 0.01, 0.05
    pm, vel = W.plummer(n, with_velocities=True)
    for mac_mode in (0, 1):
        prev = O.build(pm, mac_mode=mac_mode)
        b = Bonsai(n, mac_mode=mac_mode, mult_kernel=TILES)
        d_pm, v4 = _dev(pm), _dev(O._vel4(vel))
        out = b.step(d_pm, theta, eps)
        b.sync()
        if mac_mode == 1:
            check_tight_cells(b, O.full_step(pm, theta, eps, mac_mode=1))
        b.drift(d_pm, v4, dt)
        pm2 = d_pm.cpu().numpy()
        b.load(d_pm)
        b.refresh_tree()
        b.compute_multipoles()
        out = b.walk(theta, eps, out=out).cpu().numpy()
        b.sync()
        ref = O.refreshed_step(prev, pm2, theta, eps, mac_mode=mac_mode)
        if mac_mode == 1:
            check_tight_cells(b, ref)
        else:
            check_structure(b, ref)
        check_groups(b, ref)
        check_walk(b, out, ref, eps=eps, pm=pm2)


@pytest.mark.parametrize("n", [60_001, 1 << 21])
def test_the_two_kernels_agree_to_the_last_bit(n):
    pm = W.plummer(n)
    recs = []
    for kernel in (CLIMB, TILES):
        b = Bonsai(n, mult_kernel=kernel)
        b.load(_dev(pm)); b.build_tree(); b.compute_multipoles(); b.sync()
        c = b.cells()
        recs.append((c.com_m.view(np.uint32), c.delta.view(np.uint32), c.lside.view(np.uint32), c.quad.view(np.uint32),
                     c.walk_quad.view(np.uint32)))
        del b
    for x, y in zip(*recs):
        assert np.array_equal(x, y)
