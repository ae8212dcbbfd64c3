"""BASELINE.json configs[1]: theta sweep {0.3, 0.5, 0.75, 1.0} at N = 2^18 on the GPU, judged against the oracle's
DIRECT summation (not its tree walk): "the multipole acceptance criteria (theta) sets the trade-off between speed
and accuracy".  Error must fall and cost must rise as theta falls."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402


def test_theta_sweep_error_vs_direct_and_cost():
    cfg = W.CONFIGS["plummer_256k"]
    n, eps = cfg["n"], cfg["eps"]
    pm = W.plummer(n)
    sinks = np.arange(0, n, n // 512, dtype=np.uint32)[:512]          # evenly spaced in load order = random in space
    acc_d, pot_d = O.direct(pm, eps, sinks)
    b = Bonsai(n)
    d_pm = torch.from_numpy(pm).cuda()
    med, p99, cost = [], [], []
    for theta in cfg["theta_sweep"]:
        out = b.step(d_pm, theta, eps)
        b.sync()
        got = out.cpu().numpy()[sinks].astype(np.float64)
        ea = np.linalg.norm(got[:, :3] - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
        ep = np.abs((got[:, 3] - pot_d) / pot_d)
        med.append(np.median(ea)); p99.append(np.quantile(ea, 0.99))
        pp, pc = b.interaction_totals()
        cost.append((pp + pc) / n)
        assert np.median(ep) < np.median(ea)                          # the potential converges faster than the force
    # theta_sweep is ascending: error rises, cost falls
    assert all(med[i] < med[i + 1] for i in range(3)), med
    assert all(cost[i] > cost[i + 1] for i in range(3)), cost
    # survey-time probe (SURVEY.md appendix C, N = 2^22, theta = 0.75): median 7.5e-4, 99th percentile 3.4e-3
    assert med[2] < 2e-3 and p99[2] < 1e-2
    assert med[0] < 1e-4                                              # theta = 0.3
    assert cost[0] / cost[3] > 5
