"""Parity of bonsai_refresh_tree (row f1, R25) against oracle.refresh: the permutation, keys and
cells of the last build are kept bit for bit, the re-gathered particles, group boxes and grown cell sides are
bit-exact, the multipoles within 1 ulp, the walk within the usual gates."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai, BonsaiError  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from paper_1204_2280_b200.bonsai import ESTATE  # noqa: E402
from test_gpu_parity import _dev, check_groups, check_structure, check_walk  # noqa: E402


def _drift_oracle(pm, vel, dt):
    out = pm.copy()
    O.drift(out, O._vel4(vel), np.float32(dt))
    return out


@pytest.mark.parametrize("n,mode,dt", [(32768, 2, 0.02), (32768, 2, 0.0), (20001, 0, 0.05), (4097, 1, 0.2)])
def test_refresh_matches_oracle(n, mode, dt):
    theta, eps = 0.75, 0.01
    pm, vel = W.plummer(n, with_velocities=True)
    ref0 = O.build(pm, group_mode=mode)
    b = Bonsai(n, group_mode=mode)
    pm_d, v_d = _dev(pm), _dev(O._vel4(vel))
    out = b.step(pm_d, theta, eps)
    b.drift(pm_d, v_d, dt)
    pm2 = _drift_oracle(pm, vel, dt)
    assert np.array_equal(pm_d.cpu().numpy().view(np.uint32), pm2.view(np.uint32))
    b.refresh_tree()
    b.compute_multipoles()
    out = b.walk(theta, eps, out=out)
    b.sync()
    ref = O.refreshed_step(ref0, pm2, theta, eps, group_mode=mode)
    check_structure(b, ref)
    check_groups(b, ref)
    stats = check_walk(b, out.cpu().numpy(), ref, eps=eps, pm=pm2)
    assert stats["count_frac"] >= 0.999
    if dt > 0:
        assert (ref.tree.lside > ref0.tree.level * 0 + ref.side / 2.0 ** ref0.tree.level).mean() > 0.05


def test_refresh_then_masked_walk_block_step():
    """Block time-step use (BASELINE.json configs[4]): no rebuild, only the active subset is walked."""
    n, theta, eps, dt = 32768, 0.75, 0.01, 0.01
    pm, vel = W.plummer(n, with_velocities=True)
    mask = W.active_mask(pm, n // 16, "clustered")
    ref0 = O.build(pm)
    b = Bonsai(n)
    pm_d, v_d = _dev(pm), _dev(O._vel4(vel))
    out = b.step(pm_d, theta, eps)
    before = out.clone()
    b.drift(pm_d, v_d, dt)
    b.refresh_tree(); b.compute_multipoles()
    out = b.walk(theta, eps, _dev(mask), out=out)
    b.sync()
    pm2 = _drift_oracle(pm, vel, dt)
    ref = O.refreshed_step(ref0, pm2, theta, eps, active_mask=mask)
    check_groups(b, ref)
    got = out.cpu().numpy()
    check_walk(b, got, ref, active=mask, eps=eps, pm=pm2)
    assert np.array_equal(got[mask == 0], before.cpu().numpy()[mask == 0])      # inactive outputs untouched (R19)


def test_interactions_grow_with_drift_and_rebuild_restores():
    n, theta, eps = 262144, 0.75, 0.005
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    pm_d, v_d = _dev(pm), _dev(O._vel4(vel))
    out = b.step(pm_d, theta, eps)
    base = sum(b.interaction_totals())
    seen = []
    for _ in range(3):
        b.drift(pm_d, v_d, 0.02)
        b.refresh_tree(); b.compute_multipoles(); b.walk(theta, eps, out=out)
        seen.append(sum(b.interaction_totals()))
    assert base < seen[0] < seen[1] < seen[2]                 # the count rises as the cells grow
    b.build_tree(); b.compute_multipoles(); b.walk(theta, eps, out=out)
    assert sum(b.interaction_totals()) < 1.05 * base          # a rebuild brings it back


def test_refresh_state_errors():
    n = 1000
    pm = W.plummer(n)
    b = Bonsai(2 * n)
    with pytest.raises(BonsaiError) as e:
        b.refresh_tree()
    assert e.value.code == ESTATE
    pm_d = _dev(pm)
    b.load(pm_d)
    with pytest.raises(BonsaiError) as e:
        b.refresh_tree()                                      # loaded, but no tree yet
    assert e.value.code == ESTATE
    b.build_tree()
    b.refresh_tree()                                          # same n: fine
    big = _dev(W.plummer(2 * n))
    b.load(big)
    with pytest.raises(BonsaiError) as e:
        b.refresh_tree()                                      # the tree on the device is for another n
    assert e.value.code == ESTATE
    b.sync()
