"""Pins for the seeded Plummer generator (paper_1204_2280_b200/workloads.py): closed forms of the
Plummer model (P:L32 Results "Plummer spheres"; BASELINE.json configs: Henon units, 99.9 % mass cut)."""
import numpy as np
import pytest

import oracle as O
from paper_1204_2280_b200 import workloads as W


def test_stream_independent_of_n_and_chunking():
    a = W.plummer(1000)
    b = W.plummer(4000)
    assert (a[:, :3] == b[:1000, :3]).all()
    c = W.plummer(300, first=700)
    assert (c[:, :3] == b[700:1000, :3]).all()
    assert (a[:, 3] == np.float32(1e-3)).all()
    assert not (W.plummer(1000, seed=1)[:, :3] == a[:, :3]).any()


def test_radial_profile_closed_forms():
    n = 200000
    pm = W.plummer(n)
    r = np.linalg.norm(pm[:, :3].astype(np.float64), axis=1)
    a = W.PLUMMER_A
    # enclosed mass m(r) = (r/a)^3 (1 + r^2/a^2)^(-3/2), truncated at m = 0.999
    r_cut = a / np.sqrt(0.999 ** (-2.0 / 3.0) - 1.0)
    assert abs(r_cut - 22.804) < 2e-3
    assert r.max() <= r_cut * (1 + 1e-6)
    # half of the (cut) mass: m = 0.4995
    r_half = a / np.sqrt(0.4995 ** (-2.0 / 3.0) - 1.0)
    assert abs(np.median(r) - r_half) < 0.006 and abs(r_half - 0.768) < 1e-3
    # fraction inside r = a: 2^(-3/2) / 0.999
    frac = (r < a).mean()
    assert abs(frac - 2 ** -1.5 / 0.999) < 4e-3
    # isotropy
    u = pm[:, :3].astype(np.float64) / r[:, None]
    assert np.abs(u.mean(axis=0)).max() < 6e-3
    assert np.abs((u * u).mean(axis=0) - 1.0 / 3.0).max() < 4e-3


def test_virial_and_energy():
    n, eps = 4096, 0.002
    pm, vel = W.plummer(n, with_velocities=True)
    _, pot = O.direct(pm, eps)
    m = pm[:, 3].astype(np.float64)
    pe = 0.5 * (m * pot).sum()
    ke = 0.5 * (m * (vel.astype(np.float64) ** 2).sum(axis=1)).sum()
    # Henon units: PE -> -1/2, KE -> 1/4, E -> -1/4 (sampling noise + cut + softening ~ few %)
    assert abs(pe + 0.5) < 0.03
    assert abs(ke - 0.25) < 0.02
    assert abs(2 * ke / abs(pe) - 1.0) < 0.06
    assert abs(ke + pe + 0.25) < 0.03


def test_active_masks():
    pm = W.plummer(4096)
    for pat in ("scattered", "clustered"):
        mk = W.active_mask(pm, 256, pat)
        assert mk.dtype == np.uint8 and mk.sum() == 256
        assert (W.active_mask(pm, 256, pat) == mk).all()
    r2 = (pm[:, :3].astype(np.float64) ** 2).sum(axis=1)
    mk = W.active_mask(pm, 256, "clustered")
    assert r2[mk == 1].max() <= r2[mk == 0].min()
    assert W.active_mask(pm, 0).sum() == 0 and W.active_mask(pm, 4096).sum() == 4096


def test_no_duplicate_keys_at_config0():
    pm = W.plummer(1 << 15)
    lo, side = O.box(pm)
    assert side == 64.0
    k = O.keys(pm, lo, side)
    big = (k[:, 0].astype(object) << 60) | (k[:, 1].astype(object) << 30) | k[:, 2].astype(object)
    assert len(set(big.tolist())) == 1 << 15


def test_merger_workload_structure():
    pm, vel = W.merger(40000)
    m = pm[:, 3].astype(np.float64)
    assert m.sum() == pytest.approx(1.0, rel=1e-6)
    com = (m[:, None] * pm[:, :3]).sum(axis=0)
    assert np.abs(com).max() < 0.02                                   # sampling noise of two finite spheres
    mom = (m[:, None] * vel.astype(np.float64)).sum(axis=0)
    assert np.abs(mom).max() < 0.01
    a, b = pm[:30000], pm[30000:]
    assert a[:, 0].mean() == pytest.approx(-1.5, abs=0.05) and b[:, 0].mean() == pytest.approx(4.5, abs=0.05)
    ra = np.median(np.linalg.norm(a[:, :3] - a[:, :3].mean(axis=0), axis=1))
    rb = np.median(np.linalg.norm(b[:, :3] - b[:, :3].mean(axis=0), axis=1))
    assert rb / ra == pytest.approx(np.sqrt(1 / 3), rel=0.05)         # B is the smaller sphere
    assert vel[:30000, 0].mean() > 0 > vel[30000:, 0].mean()          # approaching
    pm2, _ = W.merger(40000)
    assert np.array_equal(pm, pm2)                                    # seeded
