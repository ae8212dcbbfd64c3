"""Row f3 on the GPU: the MAC / accuracy variants (R28 tight particle-box MAC, R29 monopole-only walk)
through the C-ABI against the oracle (oracle/mac_oracle.cpp, oracle_walk order = 1).  Gates as for the default
variant: structure bit-exact, (l, delta) and moments <= 1 ulp, counts identical (mismatches only in borderline
groups), acc / pot within 1e-4 max, 1e-6 median; plus the theta-error-cost ordering against the oracle's direct sum."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from test_gpu_parity import _dev, _ulp_diff, check_groups, check_structure, check_walk, check_walk_sampled, record  # noqa: E402


def check_tight_cells(b: Bonsai, ref: O.Step):
    """check_structure with the tight MAC: lside is no longer the exact power of two, it is a rounded fp64 difference
    of exact fp32 bounds -- identical on both sides; delta follows the COM (<= 1 ulp above the fp64 noise floor)."""
    c = b.cells(True)
    t = ref.tree
    assert c.n_cells == t.n_cells
    for name in ("level", "first", "count", "first_child", "n_child", "parent"):
        assert np.array_equal(getattr(c, name), getattr(t, name)), name
    assert np.array_equal(c.lside.view(np.uint32), t.lside.view(np.uint32))
    d = _ulp_diff(c.delta, t.delta)
    bad = (d > 1) & (np.abs(c.delta.astype(np.float64) - t.delta) > 1e-14 * ref.side)
    assert not bad.any(), (int(bad.sum()), int(d.max()))
    assert (_ulp_diff(c.com_m, t.com_m) <= 1).all()
    return c


@pytest.mark.parametrize("mac_mode,order", [(1, 2), (0, 1), (1, 1)])
@pytest.mark.parametrize("group_mode", [2, 0])
def test_variants_config0_32k(mac_mode, order, group_mode):
    cfg = W.CONFIGS["plummer_32k"]
    pm = W.plummer(cfg["n"])
    ref = O.full_step(pm, cfg["theta"], cfg["eps"], group_mode=group_mode, mac_mode=mac_mode, order=order)
    b = Bonsai(cfg["n"], group_mode=group_mode, mac_mode=mac_mode, order=order)
    out = b.step(_dev(pm), cfg["theta"], cfg["eps"]).cpu().numpy()
    b.sync()
    if mac_mode == 1:
        check_tight_cells(b, ref)
    else:
        check_structure(b, ref)
    check_groups(b, ref)
    check_walk(b, out, ref, tag=f"f3 mac_mode {mac_mode} order {order} groups {group_mode} 32k")


@pytest.mark.parametrize("mac_mode,order", [(1, 2), (1, 1), (0, 1)])
def test_variants_ragged_sizes_masks_eps0(mac_mode, order):
    for n, eps, theta in ((17, 0.01, 0.75), (1000, 0.0, 0.6), (50_003, 0.005, 1.0)):
        pm = W.plummer(n)
        mask = W.active_mask(pm, max(1, n // 9), "scattered") if n > 100 else None
        ref = O.full_step(pm, theta, eps, active_mask=mask, mac_mode=mac_mode, order=order)
        b = Bonsai(n, mac_mode=mac_mode, order=order)
        sentinel = torch.full((n, 4), 7.0, dtype=torch.float32, device="cuda")
        out = b.step(_dev(pm), theta, eps, None if mask is None else _dev(mask), sentinel).cpu().numpy()
        b.sync()
        check_groups(b, ref)
        check_walk(b, out, ref, active=mask, count_frac=0.98, eps=eps, pm=pm)
        if mask is not None:
            assert np.all(out[mask == 0] == 7.0)


def test_theta_zero_is_direct_for_every_variant():
    n = 2048
    pm = W.plummer(n)
    acc, pot = O.direct(pm, 0.01)
    for mac_mode in (0, 1):
        for order in (1, 2):
            b = Bonsai(n, mac_mode=mac_mode, order=order)
            out = b.step(_dev(pm), 0.0, 0.01).cpu().numpy().astype(np.float64)
            b.sync()
            ea = np.linalg.norm(out[:, :3] - acc, axis=1) / np.linalg.norm(acc, axis=1)
            assert ea.max() < 1e-5 and np.abs((out[:, 3] - pot) / pot).max() < 1e-5
            n_pp, n_pc = b.counts()
            assert np.all(n_pp == n - 1) and np.all(n_pc == 0)


def test_tight_mac_on_a_refreshed_tree():
    """R28 + R25: bonsai_refresh_tree with mac_mode = 1 recomputes the particle boxes at the new positions."""
    n, theta, eps = 20_000, 0.75, 0.01
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n, mac_mode=1)
    d_pm = _dev(pm)
    b.step(d_pm, theta, eps)
    prev = O.build(pm, mac_mode=1)
    v4 = _dev(O._vel4(vel))
    b.drift(d_pm, v4, 0.05)
    pm2 = d_pm.cpu().numpy()
    b.load(d_pm)
    b.refresh_tree()
    b.compute_multipoles()
    out = b.walk(theta, eps).cpu().numpy()
    b.sync()
    ref = O.refreshed_step(prev, pm2, theta, eps, mac_mode=1)
    check_tight_cells(b, ref)
    check_groups(b, ref)
    check_walk(b, out, ref, eps=eps, pm=pm2, tag="f3 tight MAC on a refreshed tree")


def test_full_size_256k_tight_mac_sampled():
    cfg = W.CONFIGS["plummer_256k"]
    n, eps, theta = cfg["n"], cfg["eps"], cfg["theta"]
    pm = W.plummer(n)
    ref = O.build(pm, mac_mode=1)
    b = Bonsai(n, mac_mode=1)
    out = b.step(_dev(pm), theta, eps, None, torch.full((n, 4), float("nan"), dtype=torch.float32, device="cuda")).cpu().numpy()
    b.sync()
    check_tight_cells(b, ref)
    check_groups(b, ref)
    check_walk_sampled(b, out, ref, theta, eps, stride=4, tag="f3 tight MAC plummer_256k")


def test_error_cost_table_against_the_oracles_direct_sum():
    """theta "sets the trade-off between speed and accuracy".  N = 2^18 (extends configs[1]): for the four
    variants, GPU force error against oracle_direct on 512 sinks and GPU interaction counts: error falls and cost
    rises as theta falls; quadrupole beats monopole on identical lists; the tight MAC is cheaper at equal theta."""
    cfg = W.CONFIGS["plummer_256k"]
    n, eps = cfg["n"], cfg["eps"]
    pm = W.plummer(n)
    sinks = np.arange(0, n, n // 512, dtype=np.uint32)[:512]
    acc_d, pot_d = O.direct(pm, eps, sinks)
    d_pm = _dev(pm)
    res = {}
    for mac_mode in (0, 1):
        for order in (2, 1):
            b = Bonsai(n, mac_mode=mac_mode, order=order)
            rows = []
            for theta in cfg["theta_sweep"]:
                got = b.step(d_pm, theta, eps).cpu().numpy()[sinks].astype(np.float64)
                b.sync()
                ea = np.linalg.norm(got[:, :3] - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
                pp, pc = b.interaction_totals()
                rows.append((float(np.median(ea)), float(np.quantile(ea, 0.99)), pp / n, pc / n))
                record("f3 error-cost", mac_mode=mac_mode, order=order, theta=theta, acc_err_median=rows[-1][0],
                       acc_err_p99=rows[-1][1], pp_per_particle=pp / n, pc_per_particle=pc / n)
            res[(mac_mode, order)] = rows
            assert all(rows[k][0] < rows[k + 1][0] for k in range(3)), rows     # theta ascending: error rises
            assert all(rows[k][2] + rows[k][3] > rows[k + 1][2] + rows[k + 1][3] for k in range(3)), rows
    for mac_mode in (0, 1):
        for k in range(4):
            assert res[(mac_mode, 2)][k][0] < res[(mac_mode, 1)][k][0]
            assert res[(mac_mode, 2)][k][2:] == res[(mac_mode, 1)][k][2:]       # identical lists
    for k in range(4):
        assert sum(res[(1, 2)][k][2:]) < sum(res[(0, 2)][k][2:])
