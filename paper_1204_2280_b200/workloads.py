"""Seeded synthetic inputs: Plummer spheres and active-subset masks.

This module is the ONLY code shared by the oracle's tests and the CUDA path's
tests/bench.  It holds none of the method's arithmetic (no keys, no tree, no
forces): it only draws initial conditions.  It imports neither ``oracle`` nor
the CUDA binding.

Workload: the paper measures on Plummer spheres with N = 2^15 .. 2^22
(Results, "we execute simulations using Plummer spheres (Plummer
(1915))"); BASELINE.json ``configs`` fixes equal masses 1/N, G = 1, Henon
units, the Aarseth-Henon-Wielen sampling and a radius cut at 99.9 % of the
mass.  The recipe:

* every particle ``i`` owns an independent counter-based uniform stream keyed by
  ``(seed, i, c)`` (a 64-bit mixing hash), so particle ``i`` is the same for every
  N, every chunking and every thread count;
* enclosed-mass fraction ``m = 0.999 (1 - u1)`` in (0, 0.999]  (this IS the
  99.9 % mass cut), model radius ``r = (m^(-2/3) - 1)^(-1/2)``;
* direction: ``z = (1 - 2 u2) r``, ``phi = 2 pi u3``;
* speed: von Neumann rejection ``0.1 u5 < q^2 (1 - q^2)^(7/2)`` with ``q = u4``,
  ``v = q sqrt(2) (1 + r^2)^(-1/4)``, isotropic direction from two more uniforms;
* scale to Henon units (G = M = 1, E = -1/4): positions by ``a = 3 pi / 16``,
  velocities by ``a^(-1/2)``;
* computed in fp64, stored fp32, no re-centring.
"""
from __future__ import annotations

import numpy as np

SEED_PARTICLES = 12042280
SEED_ACTIVE = 2280

PLUMMER_A = 3.0 * np.pi / 16.0
MASS_CUT = 0.999

_M1 = np.uint64(0x9E3779B97F4A7C15)
_M2 = np.uint64(0xBF58476D1CE4E5B9)
_M3 = np.uint64(0x94D049BB133111EB)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wraps modulo 2^64)."""
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= _M2
    z ^= z >> np.uint64(27)
    z *= _M3
    z ^= z >> np.uint64(31)
    return z


def uniform(seed: int, index: np.ndarray, counter) -> np.ndarray:
    """Counter-based uniform in the open interval (0, 1), fp64, 53 random bits.

    ``index`` is a uint64 array of particle numbers, ``counter`` a scalar or an
    array of the same shape (the position of the draw in that particle's stream).
    """
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        ctr = np.asarray(counter, dtype=np.uint64)
        z = _mix64(np.uint64(seed) * _M1 + idx)
        z = _mix64(z ^ (ctr * _M2 + _M3))
        z = _mix64(z + _M1)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def plummer(n: int, seed: int = SEED_PARTICLES, with_velocities: bool = False,
            first: int = 0):
    """Return ``pos_mass`` float32[n, 4] (x, y, z, m) and optionally ``vel`` float32[n, 3].

    ``first`` lets a caller generate particles ``first .. first+n-1`` of the same
    infinite sequence (used to check that the stream is independent of N); the
    mass is always ``1 / n`` of THIS call.
    """
    if n <= 0:
        raise ValueError("n must be positive")
    i = np.arange(first, first + n, dtype=np.uint64)
    u1 = uniform(seed, i, 1)
    u2 = uniform(seed, i, 2)
    u3 = uniform(seed, i, 3)
    m_enc = MASS_CUT * (1.0 - u1)
    r = 1.0 / np.sqrt(m_enc ** (-2.0 / 3.0) - 1.0)
    z = (1.0 - 2.0 * u2) * r
    phi = 2.0 * np.pi * u3
    rho = np.sqrt(np.maximum(r * r - z * z, 0.0))
    pos = np.empty((n, 4), dtype=np.float64)
    pos[:, 0] = rho * np.cos(phi) * PLUMMER_A
    pos[:, 1] = rho * np.sin(phi) * PLUMMER_A
    pos[:, 2] = z * PLUMMER_A
    pos[:, 3] = 1.0 / n
    pos_mass = np.ascontiguousarray(pos.astype(np.float32))
    if not with_velocities:
        return pos_mass

    # speed by rejection; draws 4,5 then 8,9 then 10,11 ... of the particle's stream
    q = np.zeros(n, dtype=np.float64)
    todo = np.arange(n)
    rnd = 0
    while todo.size:
        c0 = 4 if rnd == 0 else 8 + 2 * (rnd - 1)
        u4 = uniform(seed, i[todo], c0)
        u5 = uniform(seed, i[todo], c0 + 1)
        ok = 0.1 * u5 < u4 * u4 * (1.0 - u4 * u4) ** 3.5
        q[todo[ok]] = u4[ok]
        todo = todo[~ok]
        rnd += 1
    speed = q * np.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    u6 = uniform(seed, i, 6)
    u7 = uniform(seed, i, 7)
    vz = (1.0 - 2.0 * u6) * speed
    vphi = 2.0 * np.pi * u7
    vrho = np.sqrt(np.maximum(speed * speed - vz * vz, 0.0))
    vel = np.empty((n, 3), dtype=np.float64)
    s = PLUMMER_A ** -0.5
    vel[:, 0] = vrho * np.cos(vphi) * s
    vel[:, 1] = vrho * np.sin(vphi) * s
    vel[:, 2] = vz * s
    return pos_mass, np.ascontiguousarray(vel.astype(np.float32))


def merger(n: int, separation: float = 6.0, mass_ratio: float = 3.0, approach_speed: float = 0.4,
           seed: int = SEED_PARTICLES):
    """Second workload (DESIGN.md row f4; P:L56 lists other uses of the tree): two Plummer spheres
    on a head-on approach -- an asymmetric, two-centred system that stresses group quality and the root cube.

    Sphere A holds mass_ratio / (1 + mass_ratio) of the particles and of the mass, sphere B the rest, scaled to
    sqrt(mass fraction) of A's radius; centres at -+ separation / 2 along x weighted so the centre of mass is at the
    origin, relative speed ``approach_speed`` along x.  Particles of B continue A's counter stream (index n_a ...).
    Returns (pos_mass float32[n, 4], vel float32[n, 3]); total mass 1.
    """
    if n < 2:
        raise ValueError("n must be at least 2")
    fa = mass_ratio / (1.0 + mass_ratio)
    n_a = min(max(int(round(n * fa)), 1), n - 1)
    n_b = n - n_a
    pa, va = plummer(n_a, seed, with_velocities=True)
    pb, vb = plummer(n_b, seed, with_velocities=True, first=n_a)
    ma, mb = n_a / n, n_b / n
    pa = pa.astype(np.float64); pb = pb.astype(np.float64)
    va = va.astype(np.float64); vb = vb.astype(np.float64)
    pa[:, 3] = 1.0 / n
    pb[:, 3] = 1.0 / n
    # a Plummer sphere of mass M and radius scale R has velocities ~ sqrt(M / R); B is smaller by sqrt(mb / ma) in radius
    sb = np.sqrt(mb / ma)
    pa[:, :3] *= 1.0                       # A keeps the Henon-unit scale of the generator (mass rescaled below)
    va *= np.sqrt(ma)
    pb[:, :3] *= sb
    vb *= np.sqrt(mb / sb)
    xa, xb = -separation * mb, separation * ma          # centre of mass at the origin
    pa[:, 0] += xa
    pb[:, 0] += xb
    va[:, 0] += approach_speed * mb
    vb[:, 0] -= approach_speed * ma
    pos = np.concatenate([pa, pb]).astype(np.float32)
    vel = np.concatenate([va, vb]).astype(np.float32)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel)


def active_mask(pos_mass: np.ndarray, n_active: int, pattern: str = "scattered",
                seed: int = SEED_ACTIVE) -> np.ndarray:
    """uint8[n] mask in LOAD order with exactly ``n_active`` ones (BASELINE.json configs[4]).

    ``scattered``: a uniform random subset chosen by ``seed`` (the n_active particles
    with the smallest hash draw).  ``clustered``: the n_active particles closest to
    the origin (what block time-steps produce: short steps live in the core).
    """
    n = pos_mass.shape[0]
    if not 0 <= n_active <= n:
        raise ValueError("n_active out of range")
    if pattern == "scattered":
        score = uniform(seed, np.arange(n, dtype=np.uint64), 0)
    elif pattern == "clustered":
        p = pos_mass[:, :3].astype(np.float64)
        score = (p * p).sum(axis=1)
    else:
        raise ValueError("pattern must be 'scattered' or 'clustered'")
    mask = np.zeros(n, dtype=np.uint8)
    if n_active:
        order = np.argsort(score, kind="stable")
        mask[order[:n_active]] = 1
    return mask


# BASELINE.json configs, as data.  eps and theta as the paper's/BASELINE's values.
CONFIGS = {
    "plummer_32k": dict(n=1 << 15, eps=0.01, theta=0.75),
    "plummer_256k": dict(n=1 << 18, eps=0.005, theta=0.75, theta_sweep=(0.3, 0.5, 0.75, 1.0)),
    "plummer_1m": dict(n=1 << 20, eps=0.0025, theta=0.75),
    "plummer_4m": dict(n=1 << 22, eps=0.00125, theta=0.75),
}
