"""Driver for compute-sanitizer (not a pytest file): one small pass over every kernel family of libbonsai.

    compute-sanitizer --tool memcheck|racecheck|synccheck python tests/sanitizer_case.py [quick]

Covers: the full step at N = 2^15 (staged calls and the captured CUDA graph), a masked walk that takes the team
kernel, the short-run repair and the long-run sort of the tie handling (clumps below the 20th level, coincident
particles), the refreshed tree, the tight MAC and the monopole walk, one block tick with the device-side rebuild
decision, the integrator kernels and bonsai_step_host.  Prints "sanitizer case done" on success; results are only
checked for finiteness here (parity is the job of tests/test_gpu_*.py).
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402


def main(quick: bool) -> None:
    n = 1 << (13 if quick else 15)
    theta, eps = 0.75, 0.01
    pm, vel = W.plummer(n, with_velocities=True)
    d_pm = torch.from_numpy(pm).cuda()
    v4 = np.zeros((n, 4), np.float32)
    v4[:, :3] = vel
    d_v = torch.from_numpy(v4).cuda()

    b = Bonsai(n, use_graph=False)
    out = b.step(d_pm, theta, eps)                                   # staged kernels, one by one
    b.sync()
    assert torch.isfinite(out).all()
    mask = torch.from_numpy(W.active_mask(pm, n // 256, "clustered")).cuda()
    out2 = b.walk(theta, eps, mask)                                  # few groups: team kernel
    b.sync()
    assert torch.isfinite(out2).all()

    g = Bonsai(n)                                                    # captured graph, replayed
    out3 = torch.zeros_like(out)
    for _ in range(3):
        g.step(d_pm, theta, eps, None, out3)
    g.sync()
    assert g.graph_replays() >= 2 and torch.equal(out3, out)

    # ties of the two-word sort: short runs repaired in place, long runs radix-sorted, all-coincident particles
    rng = np.random.default_rng(1)
    clump = W.plummer(4000)
    clump[0, :3] = (900.0, -700.0, 800.0)
    at = 100
    for sz in (5, 40, 700):
        off = (rng.integers(-40, 41, size=(sz, 3)) * np.float32(2.0 ** -22)).astype(np.float32)
        clump[at:at + sz, :3] = clump[at, :3] + off
        at += sz + 20
    clump[3000:3200, :3] = clump[3000, :3]
    bc = Bonsai(4000, use_graph=False)
    oc = bc.step(torch.from_numpy(clump).cuda(), theta, eps)
    bc.sync()
    assert torch.isfinite(oc).all()

    # MAC variants, refreshed tree
    for mac_mode, order in ((1, 2), (0, 1)):
        bv = Bonsai(n, mac_mode=mac_mode, order=order, use_graph=False)
        ov = bv.step(d_pm, theta, eps)
        bv.drift(d_pm, d_v, 1e-3)
        bv.load(d_pm)
        bv.refresh_tree()
        bv.compute_multipoles()
        ov = bv.walk(theta, eps)
        bv.sync()
        assert torch.isfinite(ov).all()

    # integrator, diagnostics, block ticks (rebuild, refresh, device-side decision)
    bi = Bonsai(n, rebuild_factor=1.02)
    acc = bi.step(d_pm, theta, eps).clone()
    bi.leapfrog_step(d_pm, d_v, acc, theta, eps, 1.0 / 1024)
    bi.leapfrog_step(d_pm, d_v, acc, theta, eps, 1.0 / 1024)
    diag = bi.diagnostics(d_pm, d_v, acc)
    rung = bi.timestep_rungs(acc, 0.3, eps, 1.0 / 4, 2)
    for tick, rebuild in enumerate((True, False, -1, -1, -1)):
        bi.block_tick(d_pm, d_v, acc, rung, tick, theta, eps, 0.3, 1.0 / 4, 2, rebuild=rebuild)
    bi.sync()
    assert torch.isfinite(acc).all() and torch.isfinite(diag).all()

    # host-buffer call (pinned and pageable)
    h_out = bi.step_host(torch.from_numpy(pm).pin_memory(), theta, eps)
    h_out2 = bi.step_host(torch.from_numpy(pm.copy()), theta, eps, None, torch.zeros((n, 4), dtype=torch.float32))
    assert torch.isfinite(h_out).all() and torch.equal(h_out, h_out2)
    print("sanitizer case done", "quick" if quick else "full", "n =", n)


if __name__ == "__main__":
    main(len(sys.argv) > 1 and sys.argv[1] == "quick")
