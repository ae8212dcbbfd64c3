"""Parity of the block time-step calls (integrate.cu / bonsai_block_tick through the C-ABI binding) against the
oracle (oracle/integrator_oracle.cpp R26-R27, oracle.block_tick).

Gates: rungs, active masks and rung kicks BIT-EXACT; a run of 8 block ticks (tree rebuilt, then refreshed), the two
sides running independently from the same initial state, ends with rung arrays that differ for < 1 % of the
particles and trajectories within the walk's tolerance; one rung reproduces bonsai_leapfrog_step bit for bit."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai, BonsaiError  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from paper_1204_2280_b200.bonsai import EINVAL, ESTATE  # noqa: E402


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [1, 257, 40001])
def test_rungs_masks_kicks_bit_exact(n):
    rng = np.random.default_rng(n)
    ap = (rng.normal(size=(n, 4)) * np.exp(rng.normal(size=(n, 1)) * 3)).astype(np.float32)
    ap[0, :3] = 0                                          # |a| = 0 -> rung 0
    v = rng.normal(size=(n, 4)).astype(np.float32)
    eta, eps, dt_max, kmax = 0.05, 0.01, 1 / 32, 6
    b = Bonsai(n)
    ap_d = _dev(ap)
    r_d = b.timestep_rungs(ap_d, eta, eps, dt_max, kmax)
    r = O.rungs(ap, eta, eps, dt_max, kmax)
    assert np.array_equal(r_d.cpu().numpy(), r)
    if n > 1:
        assert len(np.unique(r)) >= 4
    for tick in (0, 1, 2, 3, 8, 24, 64):
        m = O.active_at(r, kmax, tick)
        m_d = b.active_mask(r_d, kmax, tick)
        assert np.array_equal(m_d.cpu().numpy(), m)
        v_d = _dev(v)
        b.kick_rungs(v_d, ap_d, r_d, m_d, dt_max)
        v_ref = v.copy(); O.kick_rungs(v_ref, ap, r, m, np.float32(dt_max))
        assert np.array_equal(v_d.cpu().numpy().view(np.uint32), v_ref.view(np.uint32))
        # end-of-tick update with different accelerations
        ap2 = (ap * np.float32(0.05 + 3.0 * ((tick + 1) % 3))).astype(np.float32)
        r2 = r.copy(); O.rungs(ap2, eta, eps, dt_max, kmax, rung=r2, mask=m, tick=tick)
        r2_d = r_d.clone(); b.timestep_rungs(_dev(ap2), eta, eps, dt_max, kmax, rung=r2_d, active_mask=m_d, tick=tick)
        assert np.array_equal(r2_d.cpu().numpy(), r2)


def test_one_rung_is_leapfrog_step_bit_for_bit():
    n, theta, eps, dt = 5000, 0.6, 0.02, 1 / 256
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    pa, va = _dev(pm), _dev(O._vel4(vel))
    aa = b.step(pa, theta, eps).clone()
    pb, vb, ab = pa.clone(), va.clone(), aa.clone()
    rung = torch.zeros(n, dtype=torch.uint8, device="cuda")
    for t in range(3):
        b.leapfrog_step(pa, va, aa, theta, eps, dt)
        b.block_tick(pb, vb, ab, rung, t, theta, eps, 1e9, dt, 0, rebuild=True)
    b.sync()
    for x, y in ((pa, pb), (va, vb), (aa, ab)):
        assert np.array_equal(x.cpu().numpy().view(np.uint32), y.cpu().numpy().view(np.uint32))
    assert int(rung.max()) == 0


@pytest.mark.parametrize("rebuild_every", [1, 4])
def test_block_ticks_follow_the_oracle(rebuild_every):
    n, theta, eps, eta, dt_max, kmax = 8192, 0.75, 0.01, 0.1, 1 / 32, 3
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    p_d, v_d = _dev(pm), _dev(O._vel4(vel))
    a_d = b.step(p_d, theta, eps).clone()
    r_d = b.timestep_rungs(a_d, eta, eps, dt_max, kmax)
    p, v = pm.copy(), O._vel4(vel)
    ap = O.force_f32(p, theta, eps)
    r = O.rungs(ap, eta, eps, dt_max, kmax)
    flips0 = float((r_d.cpu().numpy() != r).mean())
    assert flips0 < 1e-3                                  # |a| on a rung boundary within the walk's tolerance
    # From here on the two sides run INDEPENDENTLY (nothing of the GPU's state is copied into the oracle's): a particle
    # whose rung flipped on one side steps with a different dt from then on, so divergence accumulates over the 8
    # ticks and is bounded at the end -- rung arrays differ for < 1 % of the particles, trajectories agree to the
    # walk's tolerance for the bulk and to the size of one kick for the flipped few.
    prev = None
    walked = 0
    for tick in range(8):
        rebuild = tick % rebuild_every == 0
        b.block_tick(p_d, v_d, a_d, r_d, tick, theta, eps, eta, dt_max, kmax, rebuild=rebuild)
        s, na = O.block_tick(p, v, ap, r, tick, theta, eps, eta, dt_max, kmax, prev=None if rebuild else prev)
        prev = s
        walked += na
    b.sync()
    flips = float((r_d.cpu().numpy() != r).mean())
    assert flips < 1e-2, flips
    assert walked < 0.7 * 8 * n                           # a real block scheme: not everybody every tick
    pg, vg = p_d.cpu().numpy(), v_d.cpu().numpy()
    assert np.array_equal(pg[:, 3], pm[:, 3])
    dx = np.abs(pg[:, :3].astype(np.float64) - p[:, :3]).max(axis=1)
    dv = np.abs(vg[:, :3].astype(np.float64) - v[:, :3]).max(axis=1)
    vrms = np.sqrt(np.mean(vel.astype(np.float64) ** 2))
    amax = np.abs(ap[:, :3]).max()
    assert np.median(dx) <= 2e-7 and np.quantile(dx, 0.97) <= 1e-5
    assert np.median(dv) <= 1e-6 * vrms and np.quantile(dv, 0.97) <= 1e-3 * vrms
    # nobody is further off than a few kicks of the coarsest step
    assert dv.max() <= 4 * amax * dt_max and dx.max() <= 4 * amax * dt_max * (8 * dt_max / 2 ** kmax) + 8 * dv.max() * dt_max
    from test_gpu_parity import record
    record("block_ticks", rebuild_every=rebuild_every, rung_flips_initial=flips0, rung_flips_after_8_ticks=flips,
           dx_median=float(np.median(dx)), dx_q97=float(np.quantile(dx, 0.97)), dx_max=float(dx.max()),
           dv_median_over_vrms=float(np.median(dv) / vrms), dv_max_over_vrms=float(dv.max() / vrms))


def test_device_side_rebuild_decision_follows_the_oracle_policy():
    """R30: bonsai_block_tick(rebuild = -1) decides on the device, from the interaction totals of the last
    walk, whether the tick rebuilds or refreshes the tree -- no host read-back.  Tick by tick the number of rebuilds
    and the recorded interactions per walked sink must equal those of oracle.block_tick(policy=RebuildPolicy), and the
    run must contain both kinds of tick."""
    n, theta, eps, eta, dt_max, kmax, factor = 8192, 0.75, 0.01, 0.3, 1 / 4, 2, 1.02
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n, rebuild_factor=factor)
    p_d, v_d = _dev(pm), _dev(O._vel4(vel))
    a_d = b.step(p_d, theta, eps).clone()
    r_d = b.timestep_rungs(a_d, eta, eps, dt_max, kmax)
    p, v = pm.copy(), O._vel4(vel)
    ap = O.force_f32(p, theta, eps)
    r = O.rungs(ap, eta, eps, dt_max, kmax)
    assert (r_d.cpu().numpy() != r).mean() < 1e-3
    # the context already holds a tree for p_d (built by b.step): the first tick decides; without a reference it refreshes
    pol = O.RebuildPolicy(factor)
    prev = O.build(pm)
    for tick in range(12):
        b.block_tick(p_d, v_d, a_d, r_d, tick, theta, eps, eta, dt_max, kmax, rebuild=-1)
        s, na = O.block_tick(p, v, ap, r, tick, theta, eps, eta, dt_max, kmax, prev=prev, policy=pol)
        prev = s
        st = b.rebuild_stats()
        assert st["n_decisions"] == len(pol.decisions) and st["n_rebuilds"] == sum(pol.decisions), (tick, st, pol.decisions)
        assert np.isclose(st["ipp_last"], pol.last, rtol=2e-3) and np.isclose(st["ipp_ref"], pol.ref, rtol=2e-3)
        # the tree on the device is the oracle's: rebuilt (new permutation) or frozen (old one)
        assert np.array_equal(b.perm(), s.perm), tick
    assert any(pol.decisions) and not all(pol.decisions), pol.decisions
    b.sync()
    assert (r_d.cpu().numpy() != r).mean() < 1e-2
    dx = np.abs(p_d.cpu().numpy()[:, :3].astype(np.float64) - p[:, :3]).max(axis=1)
    assert np.median(dx) <= 2e-7 and np.quantile(dx, 0.97) <= 1e-5
    from test_gpu_parity import record
    record("device-side rebuild decision", ticks=12, rebuilds=int(sum(pol.decisions)), decisions=[int(d) for d in pol.decisions],
           ipp_ref=float(pol.ref), ipp_last=float(pol.last))


def test_auto_ticks_recover_from_a_capacity_overflow():
    """bonsai.h: a build clears the sticky status.  With rebuild = -1 the library must therefore rebuild on the tick
    after an overflow (a refreshed tick would find the status set, and multipoles and walk return at once on it):
    the tick after the overflow has to give what a fresh context gives for the same state with rebuild = 1."""
    n, theta, eps, eta, dt_max, kmax = 5000, 0.75, 0.01, 0.3, 1 / 64, 2
    pm, vel = W.plummer(n, with_velocities=True)
    small = pm.copy()
    small[1000:, :3] = np.float32(np.abs(pm[:, :3]).max() * 1.5)     # 4000 coincident particles: ~270 cells
    assert O.build(small).tree.n_cells < 700 < O.build(pm).tree.n_cells
    b = Bonsai(n, cap_cells=700)
    p_d, v_d = _dev(pm), _dev(O._vel4(vel))
    a_d = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    r_d = torch.zeros(n, dtype=torch.uint8, device="cuda")
    b.block_tick(p_d, v_d, a_d, r_d, 0, theta, eps, eta, dt_max, kmax, rebuild=True)   # ~1200 cells: overflow
    with pytest.raises(BonsaiError) as e:
        b.sync()
    assert e.value.code == -3
    # the caller repairs its state in the same arrays (the context still "has a tree" for them) and lets the device decide
    p_d.copy_(_dev(small)); v_d.zero_(); a_d.zero_(); r_d.zero_()
    fresh = Bonsai(n)
    p2, v2, a2, r2 = p_d.clone(), v_d.clone(), a_d.clone(), r_d.clone()
    for tick in (3, 4, 5):                     # tick 3 walks every particle (all on rung 0), 4 and 5 the deeper rungs
        b.block_tick(p_d, v_d, a_d, r_d, tick, theta, eps, eta, dt_max, kmax, rebuild=-1)
        b.sync()                                                                      # status cleared by the rebuild
        fresh.block_tick(p2, v2, a2, r2, tick, theta, eps, eta, dt_max, kmax, rebuild=(tick == 3))
        fresh.sync()
        if tick == 3:
            assert b.rebuild_stats()["n_rebuilds"] == 1
        for x, y in ((p_d, p2), (v_d, v2), (a_d, a2), (r_d, r2)):
            assert torch.equal(x, y), tick
        assert float(a_d[:, :3].abs().max()) > 0


def test_block_ticks_at_config2_size_follow_the_oracle_tick_by_tick():
    """One rebuilt and one refreshed bonsai_block_tick at N = 2^20 (BASELINE configs[2] / [4] size: tiled multipole
    kernel, plain and team walk kernels, 4-pass sort), each against oracle.block_tick started from the state the GPU
    had before the tick (stage isolation): opening kick + drift are single fp32 FMAs on identical inputs
    -> positions bit-exact, hence the same permutation and tree; the walked particles' counts identical for >= 99.9 %,
    acc / pot within 1e-4 max / 1e-6 median; rows of particles that were not walked untouched; new rungs equal except
    where |a| sits on a rung boundary.  The oracle's walk is fanned out over the host's cores (walk_threads)."""
    import os
    threads = max(1, min(16, os.cpu_count() or 1))
    cfg = W.CONFIGS["plummer_1m"]
    n, theta, eps = cfg["n"], cfg["theta"], cfg["eps"]
    eta, dt_max, kmax = 0.3, 1 / 32, 2
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    p_d, v_d = _dev(pm), _dev(O._vel4(vel))
    a_d = b.step(p_d, theta, eps).clone()
    r_d = b.timestep_rungs(a_d, eta, eps, dt_max, kmax)
    prev = None
    u = lambda x: np.ascontiguousarray(x).view(np.uint32)
    for tick, rebuild in ((0, True), (1, False)):
        p, v, ap, r = (x.cpu().numpy().copy() for x in (p_d, v_d, a_d, r_d))
        a_before, v_before = ap.copy(), v.copy()
        m0, m1 = O.active_at(r, kmax, tick).astype(bool), O.active_at(r, kmax, tick + 1).astype(bool)
        b.block_tick(p_d, v_d, a_d, r_d, tick, theta, eps, eta, dt_max, kmax, rebuild=rebuild)
        b.sync()
        s, na = O.block_tick(p, v, ap, r, tick, theta, eps, eta, dt_max, kmax, prev=None if rebuild else prev,
                             threads=threads)
        prev = s
        assert n // 20 < na < n and na == int(m1.sum())
        pg, vg, ag, rg = (x.cpu().numpy() for x in (p_d, v_d, a_d, r_d))
        assert np.array_equal(u(pg), u(p))                                 # kick + drift: bit-exact
        assert np.array_equal(b.perm(), s.perm)                            # same tree (rebuilt or frozen)
        n_pp, n_pc = b.counts()
        w = s.walk
        same = (n_pp[s.perm] == w.n_pp) & (n_pc[s.perm] == w.n_pc)
        assert same[m1[s.perm]].mean() >= 0.999
        ea = np.linalg.norm(ag[m1, :3].astype(np.float64) - ap[m1, :3], axis=1) / np.linalg.norm(ap[m1, :3].astype(np.float64), axis=1)
        ep = np.abs((ag[m1, 3].astype(np.float64) - ap[m1, 3]) / ap[m1, 3])
        assert ea.max() <= 1e-4 and np.median(ea) <= 1e-6 and ep.max() <= 1e-4, (ea.max(), np.median(ea), ep.max())
        assert np.array_equal(u(ag[~m1]), u(a_before[~m1]))                # not walked: force row untouched
        idle = ~m0 & ~m1
        assert np.array_equal(u(vg[idle]), u(v_before[idle]))              # neither kick touched them
        only_open = m0 & ~m1
        assert np.array_equal(u(vg[only_open]), u(v[only_open]))           # opening kick only: bit-exact
        dv = np.abs(vg[m1, :3].astype(np.float64) - v[m1, :3]).max(axis=1)
        assert dv.max() <= 2e-4 * np.abs(ap[m1, :3]).max() * dt_max        # closing kick: the force tolerance times dt
        flips = float((rg != r).mean())
        assert flips < 1e-3, flips
        from test_gpu_parity import record
        record("block tick at 2^20", tick=tick, rebuilt=bool(rebuild), walked=int(na), count_frac=float(same[m1[s.perm]].mean()),
               n=int(n), n_checked=int(na), n_borderline_mismatch=int((~same[m1[s.perm]]).sum()), acc_max=float(ea.max()),
               acc_med=float(np.median(ea)), pot_max=float(ep.max()), pot_med=float(np.median(ep)), rung_flips=flips)


def test_block_tick_errors():
    n = 1000
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    p_d, v_d = _dev(pm), _dev(O._vel4(vel))
    a_d = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    r_d = torch.zeros(n, dtype=torch.uint8, device="cuda")
    with pytest.raises(BonsaiError) as e:                 # no tree yet: a refresh is impossible
        b.block_tick(p_d, v_d, a_d, r_d, 0, 0.75, 0.01, 0.1, 1 / 32, 2, rebuild=False)
    assert e.value.code == ESTATE
    with pytest.raises(BonsaiError) as e:
        b.block_tick(p_d, v_d, a_d, r_d, 0, 0.75, 0.01, 0.1, 1 / 32, 31, rebuild=True)
    assert e.value.code == EINVAL
    b.block_tick(p_d, v_d, a_d, r_d, 0, 0.75, 0.01, 0.1, 1 / 32, 2, rebuild=True)
    b.block_tick(p_d, v_d, a_d, r_d, 1, 0.75, 0.01, 0.1, 1 / 32, 2, rebuild=False)
    b.sync()
