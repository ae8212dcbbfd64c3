"""Parity of the CUDA integrator and diagnostics (row f2; integrate.cu through the C-ABI binding) against
oracle/integrator_oracle.cpp.

Gates:
  * kick, drift, fused kick+drift: BIT-EXACT (the update is defined as one fp32 fma per component, R23);
  * diagnostics: fp64 sums in a different order -> |diff| <= 1e-12 * sum |terms|;
  * an 8-step KDK run (BASELINE.json configs[2] at a size the oracle finishes in seconds): the forces that enter
    differ within the walk's tolerance (<= 1e-4 max, <= 1e-6 median), so positions agree to a few fp32 ulps and
    velocities to a few 1e-7; energy is conserved on both sides.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1204_2280_b200 import Bonsai, BonsaiError  # noqa: E402
from paper_1204_2280_b200 import workloads as W  # noqa: E402
from paper_1204_2280_b200.bonsai import DIAG_FIELDS, EINVAL, ESTATE  # noqa: E402


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _state(n, seed=11):
    rng = np.random.default_rng(seed)
    pm = rng.normal(size=(n, 4)).astype(np.float32)
    pm[:, 3] = rng.random(n).astype(np.float32) / n
    v = rng.normal(size=(n, 4)).astype(np.float32)
    a = (rng.normal(size=(n, 4)) * 5).astype(np.float32)
    return pm, v, a


@pytest.mark.parametrize("n", [1, 31, 256, 257, 100003])
def test_kick_drift_bit_exact(n):
    pm, v, a = _state(n)
    b = Bonsai(n)
    h = np.float32(1 / 1024) * np.float32(0.5)
    v_d, pm_d, a_d = _dev(v), _dev(pm), _dev(a)
    b.kick(v_d, a_d, float(h))
    v_ref = v.copy(); O.kick(v_ref, a, h)
    assert np.array_equal(v_d.cpu().numpy().view(np.uint32), v_ref.view(np.uint32))
    b.drift(pm_d, v_d, 1 / 1024)
    pm_ref = pm.copy(); O.drift(pm_ref, v_ref, np.float32(1 / 1024))
    assert np.array_equal(pm_d.cpu().numpy().view(np.uint32), pm_ref.view(np.uint32))


def test_kick_mask_bit_exact():
    n = 5000
    pm, v, a = _state(n, 5)
    mask = W.active_mask(pm, n // 16, "scattered")
    b = Bonsai(n)
    v_d = _dev(v)
    b.kick(v_d, _dev(a), 0.125, _dev(mask))
    v_ref = v.copy(); O.kick(v_ref, a, np.float32(0.125), mask)
    got = v_d.cpu().numpy()
    assert np.array_equal(got.view(np.uint32), v_ref.view(np.uint32))
    assert np.array_equal(got[mask == 0], v[mask == 0])


@pytest.mark.parametrize("n", [1, 1000, 262144 + 17])
def test_diagnostics(n):
    pm, v, a = _state(n, 2)
    b = Bonsai(n)
    got = b.diagnostics(_dev(pm), _dev(v), _dev(a)).cpu().numpy()
    want = O.diagnostics(pm, v, a)
    m = np.abs(pm[:, 3].astype(np.float64))
    x = pm[:, :3].astype(np.float64); vv = v[:, :3].astype(np.float64)
    scale = {"K": np.sum(0.5 * m * np.sum(vv * vv, axis=1)), "W": np.sum(0.5 * m * np.abs(a[:, 3].astype(np.float64))),
             "M": np.sum(m)}
    for i, k in enumerate(DIAG_FIELDS):
        if k[0] == "P":
            s = np.sum(m * np.abs(vv[:, "xyz".index(k[1])]))
        elif k[0] == "C":
            s = np.sum(m * np.abs(x[:, "xyz".index(k[1])]))
        elif k[0] == "L":
            s = np.sum(m * np.linalg.norm(x, axis=1) * np.linalg.norm(vv, axis=1))
        else:
            s = scale[k]
        assert abs(got[i] - want[i]) <= 1e-12 * s + 1e-300, (k, got[i], want[i])
    # a second call gives the same bits (fixed reduction tree, self-resetting ticket)
    again = b.diagnostics(_dev(pm), _dev(v), _dev(a)).cpu().numpy()
    assert np.array_equal(got, again)


def test_leapfrog_8_steps_config2_scaled():
    """BASELINE.json configs[2] (8 KDK steps, dt = 1/1024, shared step, tree rebuilt every step) at N = 2^15."""
    n, theta, eps, dt = 32768, 0.75, 0.01, 1.0 / 1024
    pm, vel = W.plummer(n, with_velocities=True)
    v4 = O._vel4(vel)
    b = Bonsai(n)
    pm_d, v_d = _dev(pm), _dev(v4)
    ap_d = b.step(pm_d, theta, eps).clone()
    d0 = b.diagnostics(pm_d, v_d, ap_d).cpu().numpy()
    for _ in range(8):
        b.leapfrog_step(pm_d, v_d, ap_d, theta, eps, dt)
    b.sync()
    d1 = b.diagnostics(pm_d, v_d, ap_d).cpu().numpy()
    p_ref, v_ref, a_ref = O.leapfrog(pm, vel, theta, eps, np.float32(dt), 8)
    p_g, v_g = pm_d.cpu().numpy(), v_d.cpu().numpy()
    assert np.array_equal(p_g[:, 3], pm[:, 3])
    dx = np.abs(p_g[:, :3].astype(np.float64) - p_ref[:, :3])
    dv = np.abs(v_g[:, :3].astype(np.float64) - v_ref[:, :3])
    vrms = np.sqrt(np.mean(vel.astype(np.float64) ** 2))
    # per step a force difference da moves x by da dt^2 / 2 and v by da dt; |a| ~ 1, da/a <= 1e-4 (typically 1e-7)
    assert dx.max() <= 4 * np.spacing(np.float32(np.abs(p_ref[:, :3]).max())) + 8 * 1e-4 * 30 * dt * dt
    assert np.median(dx) <= 2e-7
    assert dv.max() <= 1e-4 * vrms
    assert np.median(dv) <= 1e-6 * vrms
    e0, e1 = d0[0] + d0[1], d1[0] + d1[1]
    assert abs((e1 - e0) / e0) < 5e-5                       # tree forces at theta = 0.75: small, not exact
    dref = O.diagnostics(p_ref, v_ref, a_ref)
    assert d1[0] == pytest.approx(dref[0], rel=1e-6)       # K
    assert d1[1] == pytest.approx(dref[1], rel=1e-5)       # W (tree potential)
    assert np.allclose(d1[2:5], dref[2:5], atol=1e-7)      # P


def test_fused_step_equals_separate_calls():
    n, theta, eps, dt = 4097, 0.5, 0.02, 1.0 / 256
    pm, vel = W.plummer(n, with_velocities=True)
    v4 = O._vel4(vel)
    b = Bonsai(n)
    pa, va = _dev(pm), _dev(v4)
    aa = b.step(pa, theta, eps).clone()
    pb, vb, ab = pa.clone(), va.clone(), aa.clone()
    b.leapfrog_step(pa, va, aa, theta, eps, dt)
    b.sync()
    half = float(np.float32(0.5) * np.float32(dt))
    b.kick(vb, ab, half)
    b.drift(pb, vb, dt)
    ab = b.step(pb, theta, eps, out=ab)
    b.kick(vb, ab, half)
    b.sync()
    for x, y in ((pa, pb), (va, vb), (aa, ab)):
        assert np.array_equal(x.cpu().numpy().view(np.uint32), y.cpu().numpy().view(np.uint32))


def test_drift_invalidates_tree_and_errors():
    n = 1000
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    pm_d, v_d = _dev(pm), _dev(O._vel4(vel))
    ap = b.step(pm_d, 0.75, 0.01)
    b.drift(pm_d, v_d, 1e-3)
    with pytest.raises(BonsaiError) as e:
        b.walk(0.75, 0.01)
    assert e.value.code == ESTATE
    b.build_tree(); b.compute_multipoles(); b.walk(0.75, 0.01, out=ap)
    b.sync()
    with pytest.raises(BonsaiError) as e:
        b.kick(v_d, ap, float("nan"))
    assert e.value.code == EINVAL


@pytest.mark.parametrize("theta", [0.5, 0.75])
def test_config2_full_size_1m_properties(theta):
    """BASELINE.json configs[2] at full size (N = 2^20, eps = 0.0025, 8 steps of dt = 1/1024): the oracle cannot
    follow in seconds, so check what holds at any size -- masses untouched, energy and momentum conserved to the
    accuracy of the tree force, every particle moved by v dt to first order."""
    n, eps, dt = 1 << 20, 0.0025, 1.0 / 1024
    pm, vel = W.plummer(n, with_velocities=True)
    b = Bonsai(n)
    pm_d, v_d = _dev(pm), _dev(O._vel4(vel))
    ap_d = b.step(pm_d, theta, eps).clone()
    d0 = b.diagnostics(pm_d, v_d, ap_d).cpu().numpy()
    for _ in range(8):
        b.leapfrog_step(pm_d, v_d, ap_d, theta, eps, dt)
    b.sync()
    d1 = b.diagnostics(pm_d, v_d, ap_d).cpu().numpy()
    e0, e1 = d0[0] + d0[1], d1[0] + d1[1]
    assert d0[0] == pytest.approx(0.25, rel=0.01) and d0[1] == pytest.approx(-0.5, rel=0.01)   # virial, Henon units
    assert abs((e1 - e0) / e0) < 2e-5
    assert np.abs(d1[2:5] - d0[2:5]).max() < 2e-6          # tree forces are not exactly pairwise antisymmetric
    assert d1[8] == d0[8]
    p1 = pm_d.cpu().numpy()
    assert np.array_equal(p1[:, 3], pm[:, 3])
    moved = p1[:, :3].astype(np.float64) - pm[:, :3]
    first_order = vel.astype(np.float64) * (8 * dt)
    assert np.abs(moved - first_order).max() < 0.5 * 400.0 * (8 * dt) ** 2   # |a| stays below a few hundred at this eps
