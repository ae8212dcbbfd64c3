"""ctypes front-end of the CPU oracle (oracle/bonsai_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_1204_2280_b200 (inputs are passed in).
Each function is a thin marshalling layer over the C++ routine of the same name; see that
file for the passage of the paper / the DESIGN.md reading each one follows.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_tree.restype = C.c_uint32
        _lib.oracle_groups.restype = C.c_uint32
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


def box(pos_mass):
    pm = _f32(pos_mass)
    lo = np.zeros(3, np.float32)
    side = C.c_double(0)
    lib().oracle_box(_p(pm, C.c_float), C.c_uint32(pm.shape[0]), _p(lo, C.c_float), C.byref(side))
    return lo, side.value


def keys(pos_mass, lo, side):
    pm = _f32(pos_mass)
    lo = _f32(lo)
    out = np.zeros((pm.shape[0], 3), np.uint32)
    lib().oracle_keys(_p(pm, C.c_float), C.c_uint32(pm.shape[0]), _p(lo, C.c_float), C.c_double(side),
                      _p(out, C.c_uint32))
    return out


def decode_key(key):
    k = np.ascontiguousarray(key, dtype=np.uint32)
    q = np.zeros(3, np.uint32)
    lib().oracle_decode_key(_p(k, C.c_uint32), _p(q, C.c_uint32))
    return q


def sort(keys_):
    k = np.ascontiguousarray(keys_, dtype=np.uint32)
    perm = np.zeros(k.shape[0], np.uint32)
    lib().oracle_sort(_p(k, C.c_uint32), C.c_uint32(k.shape[0]), _p(perm, C.c_uint32))
    return perm


def reorder(pos_mass, keys_, perm):
    pm = _f32(pos_mass)
    k = np.ascontiguousarray(keys_, dtype=np.uint32)
    spm = np.zeros_like(pm)
    sk = np.zeros_like(k)
    lib().oracle_reorder(_p(pm, C.c_float), _p(k, C.c_uint32), _p(perm, C.c_uint32), C.c_uint32(pm.shape[0]),
                         _p(spm, C.c_float), _p(sk, C.c_uint32))
    return spm, sk


@dataclass
class Tree:
    n_cells: int
    level: np.ndarray
    first: np.ndarray
    count: np.ndarray
    first_child: np.ndarray
    n_child: np.ndarray
    parent: np.ndarray
    level_offsets: np.ndarray
    com_m: np.ndarray = None
    quad: np.ndarray = None
    delta: np.ndarray = None
    lside: np.ndarray = None


def tree(sorted_keys, nleaf=16, cap_cells=None):
    sk = np.ascontiguousarray(sorted_keys, dtype=np.uint32)
    n = sk.shape[0]
    cap = cap_cells if cap_cells is not None else max(4096, 2 * n + 64)
    arrs = [np.zeros(cap, np.uint32) for _ in range(6)]
    lo = np.zeros(32, np.uint32)
    nc = lib().oracle_tree(_p(sk, C.c_uint32), C.c_uint32(n), C.c_uint32(nleaf), C.c_uint32(cap),
                           *[_p(a, C.c_uint32) for a in arrs], _p(lo, C.c_uint32))
    if nc == 0xFFFFFFFF:
        raise OverflowError("oracle_tree: more than cap_cells cells")
    level, first, count, first_child, n_child, parent = [a[:nc].copy() for a in arrs]
    return Tree(nc, level, first, count, first_child, n_child, parent, lo)


@dataclass
class Groups:
    n_groups: int
    n_active: int
    active_list: np.ndarray
    first: np.ndarray
    count: np.ndarray
    bmin: np.ndarray
    bmax: np.ndarray


def groups(mode, ncrit, sorted_pos_mass, t: Tree, active_sorted=None, group_cell=512):
    spm = _f32(sorted_pos_mass)
    n = spm.shape[0]
    act = None if active_sorted is None else np.ascontiguousarray(active_sorted, dtype=np.uint8)
    active_list = np.zeros(n, np.uint32)
    gfirst = np.zeros(n, np.uint32)
    gcount = np.zeros(n, np.uint32)
    bmin = np.zeros((n, 3), np.float32)
    bmax = np.zeros((n, 3), np.float32)
    na = C.c_uint32(0)
    ng = lib().oracle_groups(C.c_uint32(mode), C.c_uint32(ncrit), C.c_uint32(group_cell), C.c_uint32(n), _p(spm, C.c_float),
                             C.c_uint32(t.n_cells), _p(t.first, C.c_uint32), _p(t.count, C.c_uint32),
                             _p(t.first_child, C.c_uint32), _p(t.n_child, C.c_uint32),
                             _p(act, C.c_uint8), _p(active_list, C.c_uint32), C.byref(na),
                             _p(gfirst, C.c_uint32), _p(gcount, C.c_uint32), _p(bmin, C.c_float),
                             _p(bmax, C.c_float))
    return Groups(ng, na.value, active_list[:na.value].copy(), gfirst[:ng].copy(), gcount[:ng].copy(),
                  bmin[:ng].copy(), bmax[:ng].copy())


def multipoles(sorted_pos_mass, sorted_keys, lo, side, t: Tree):
    spm = _f32(sorted_pos_mass)
    sk = np.ascontiguousarray(sorted_keys, dtype=np.uint32)
    lo = _f32(lo)
    nc = t.n_cells
    t.com_m = np.zeros((nc, 4), np.float32)
    t.quad = np.zeros((nc, 6), np.float32)
    t.delta = np.zeros(nc, np.float32)
    t.lside = np.zeros(nc, np.float32)
    lib().oracle_multipoles(_p(spm, C.c_float), _p(sk, C.c_uint32), C.c_uint32(spm.shape[0]),
                            _p(lo, C.c_float), C.c_double(side), C.c_uint32(nc), _p(t.level, C.c_uint32),
                            _p(t.first, C.c_uint32), _p(t.count, C.c_uint32), _p(t.com_m, C.c_float),
                            _p(t.quad, C.c_float), _p(t.delta, C.c_float), _p(t.lside, C.c_float))
    return t


@dataclass
class WalkResult:
    acc: np.ndarray          # float64[n, 3], SORTED index; rows of particles not walked are NaN
    pot: np.ndarray          # float64[n]
    n_pp: np.ndarray         # uint32[n]
    n_pc: np.ndarray         # uint32[n]
    g_ntests: np.ndarray     # uint32[n_sel]
    g_borderline: np.ndarray  # uint8[n_sel]
    sel: np.ndarray = field(default=None)


def walk(theta, eps, sorted_pos_mass, t: Tree, g: Groups, sel=None, order=2):
    spm = _f32(sorted_pos_mass)
    n = spm.shape[0]
    sel_arr = None if sel is None else np.ascontiguousarray(sel, dtype=np.uint32)
    n_sel = g.n_groups if sel_arr is None else sel_arr.shape[0]
    acc = np.full((n, 3), np.nan, np.float64)
    pot = np.full(n, np.nan, np.float64)
    n_pp = np.zeros(n, np.uint32)
    n_pc = np.zeros(n, np.uint32)
    nt = np.zeros(max(n_sel, 1), np.uint32)
    bl = np.zeros(max(n_sel, 1), np.uint8)
    lib().oracle_walk(C.c_float(theta), C.c_float(eps), _p(spm, C.c_float), C.c_uint32(n),
                      _p(t.first, C.c_uint32), _p(t.count, C.c_uint32), _p(t.first_child, C.c_uint32),
                      _p(t.n_child, C.c_uint32), _p(t.com_m, C.c_float), _p(t.quad, C.c_float),
                      _p(t.delta, C.c_float), _p(t.lside, C.c_float), _p(g.active_list, C.c_uint32),
                      _p(g.first, C.c_uint32), _p(g.count, C.c_uint32), _p(g.bmin, C.c_float),
                      _p(g.bmax, C.c_float), C.c_uint32(n_sel), _p(sel_arr, C.c_uint32),
                      _p(acc, C.c_double), _p(pot, C.c_double), _p(n_pp, C.c_uint32), _p(n_pc, C.c_uint32),
                      _p(nt, C.c_uint32), _p(bl, C.c_uint8), C.c_uint32(order))
    return WalkResult(acc, pot, n_pp, n_pc, nt[:n_sel], bl[:n_sel], sel_arr)


def walk_threads(theta, eps, sorted_pos_mass, t: Tree, g: Groups, sel, threads, order=2):
    """The same oracle_walk over the groups `sel`, split into `threads` interleaved subsets walked concurrently by
    host threads (groups are independent and write disjoint rows; ctypes releases the GIL during the call).  This is
    the "outer parallel loop over groups" of the all-cores CPU baseline (bench.py); no arithmetic lives here.
    Returns the same WalkResult as walk(); g_ntests / g_borderline follow the order of `sel`."""
    import threading
    spm = _f32(sorted_pos_mass)
    n = spm.shape[0]
    sel = np.ascontiguousarray(sel, dtype=np.uint32)
    acc = np.full((n, 3), np.nan, np.float64)
    pot = np.full(n, np.nan, np.float64)
    n_pp = np.zeros(n, np.uint32)
    n_pc = np.zeros(n, np.uint32)
    parts = [np.ascontiguousarray(sel[k::threads]) for k in range(threads)]
    nts = [np.zeros(max(len(p), 1), np.uint32) for p in parts]
    bls = [np.zeros(max(len(p), 1), np.uint8) for p in parts]
    L = lib()

    def work(k):
        if len(parts[k]) == 0:
            return
        L.oracle_walk(C.c_float(theta), C.c_float(eps), _p(spm, C.c_float), C.c_uint32(n),
                      _p(t.first, C.c_uint32), _p(t.count, C.c_uint32), _p(t.first_child, C.c_uint32),
                      _p(t.n_child, C.c_uint32), _p(t.com_m, C.c_float), _p(t.quad, C.c_float),
                      _p(t.delta, C.c_float), _p(t.lside, C.c_float), _p(g.active_list, C.c_uint32),
                      _p(g.first, C.c_uint32), _p(g.count, C.c_uint32), _p(g.bmin, C.c_float),
                      _p(g.bmax, C.c_float), C.c_uint32(len(parts[k])), _p(parts[k], C.c_uint32),
                      _p(acc, C.c_double), _p(pot, C.c_double), _p(n_pp, C.c_uint32), _p(n_pc, C.c_uint32),
                      _p(nts[k], C.c_uint32), _p(bls[k], C.c_uint8), C.c_uint32(order))

    ths = [threading.Thread(target=work, args=(k,)) for k in range(threads)]
    [th.start() for th in ths]
    [th.join() for th in ths]
    nt = np.zeros(len(sel), np.uint32)
    bl = np.zeros(len(sel), np.uint8)
    for k in range(threads):
        nt[k::threads] = nts[k][:len(parts[k])]
        bl[k::threads] = bls[k][:len(parts[k])]
    return WalkResult(acc, pot, n_pp, n_pc, nt, bl, sel)


def walk_lists(theta, t: Tree, bmin, bmax, cap=None):
    cap = cap if cap is not None else t.n_cells
    pc = np.zeros(cap, np.uint32)
    pp = np.zeros(cap, np.uint32)
    npc, npp = C.c_uint32(0), C.c_uint32(0)
    bmin = _f32(bmin)
    bmax = _f32(bmax)
    lib().oracle_walk_lists(C.c_float(theta), _p(t.first_child, C.c_uint32), _p(t.n_child, C.c_uint32),
                            _p(t.com_m, C.c_float), _p(t.delta, C.c_float), _p(t.lside, C.c_float),
                            _p(bmin, C.c_float), _p(bmax, C.c_float), C.c_uint32(cap),
                            _p(pc, C.c_uint32), C.byref(npc), _p(pp, C.c_uint32), C.byref(npp))
    return pc[:npc.value].copy(), pp[:npp.value].copy()


def direct(pos_mass, eps, sinks=None):
    pm = _f32(pos_mass)
    n = pm.shape[0]
    s = None if sinks is None else np.ascontiguousarray(sinks, dtype=np.uint32)
    ns = n if s is None else s.shape[0]
    acc = np.zeros((ns, 3), np.float64)
    pot = np.zeros(ns, np.float64)
    lib().oracle_direct(_p(pm, C.c_float), C.c_uint32(n), C.c_float(eps), C.c_uint32(ns),
                        _p(s, C.c_uint32), _p(acc, C.c_double), _p(pot, C.c_double))
    return acc, pot


@dataclass
class Step:
    """Everything one force step produces, stage by stage (sorted order unless noted)."""
    lo: np.ndarray
    side: float
    keys: np.ndarray            # load order
    perm: np.ndarray
    sorted_pos_mass: np.ndarray
    sorted_keys: np.ndarray
    tree: Tree
    groups: Groups
    walk: WalkResult = None

    def to_load_order(self, a_sorted):
        out = np.empty_like(a_sorted)
        out[self.perm] = a_sorted
        return out


def tight_mac(sorted_pos_mass, t: Tree):
    """R28 (oracle/mac_oracle.cpp): replace t.lside / t.delta by the side and COM offset of each cell's exact particle
    box; returns the boxes float32[n_cells, 6] (bmin xyz, bmax xyz)."""
    spm = _f32(sorted_pos_mass)
    box = np.zeros((t.n_cells, 6), np.float32)
    lib().oracle_tight_mac(_p(spm, C.c_float), C.c_uint32(t.n_cells), _p(t.first, C.c_uint32), _p(t.count, C.c_uint32),
                           _p(t.lside, C.c_float), _p(t.delta, C.c_float), _p(box, C.c_float))
    return box


def build(pos_mass, nleaf=16, ncrit=64, group_mode=2, active_mask=None, cap_cells=None, group_cell=512,
          mac_mode=0) -> Step:
    """O1..O6: box, keys, sort, reorder, tree, groups, multipoles.  active_mask is in LOAD order.
    mac_mode = 1: the tight MAC of R28 (cell size and centre from the particle box)."""
    pm = _f32(pos_mass)
    lo, side = box(pm)
    k = keys(pm, lo, side)
    perm = sort(k)
    spm, sk = reorder(pm, k, perm)
    t = tree(sk, nleaf, cap_cells)
    act_sorted = None if active_mask is None else np.ascontiguousarray(active_mask, np.uint8)[perm]
    g = groups(group_mode, ncrit, spm, t, act_sorted, group_cell)
    multipoles(spm, sk, lo, side, t)
    if mac_mode == 1:
        tight_mac(spm, t)
    return Step(lo, side, k, perm, spm, sk, t, g)


def _walk_maybe_threaded(theta, eps, s: "Step", sel, order, threads):
    """walk(), or the same oracle_walk fanned out over host threads (walk_threads: no arithmetic of its own)."""
    if threads <= 1:
        return walk(theta, eps, s.sorted_pos_mass, s.tree, s.groups, sel, order)
    sel = np.arange(s.groups.n_groups, dtype=np.uint32) if sel is None else sel
    return walk_threads(theta, eps, s.sorted_pos_mass, s.tree, s.groups, sel, threads, order)


def full_step(pos_mass, theta, eps, nleaf=16, ncrit=64, group_mode=2, active_mask=None, sel=None,
              group_cell=512, mac_mode=0, order=2, threads=1) -> Step:
    s = build(pos_mass, nleaf, ncrit, group_mode, active_mask, None, group_cell, mac_mode)
    s.walk = _walk_maybe_threaded(theta, eps, s, sel, order, threads)
    return s


# ---- row f2: KDK leapfrog and diagnostics (oracle/integrator_oracle.cpp, R22-R24) ----------

def _vel4(vel):
    """float32[n, 4] copy of a velocity array given as [n, 3] or [n, 4]."""
    v = np.asarray(vel, dtype=np.float32)
    out = np.zeros((v.shape[0], 4), np.float32)
    out[:, :3] = v[:, :3]
    return out


def kick(vel4, acc_pot, h, mask=None):
    """In place: vel4[i, a] = fma(acc_pot[i, a], h, vel4[i, a]) for masked-in particles (R23)."""
    assert vel4.dtype == np.float32 and vel4.flags.c_contiguous and vel4.shape[1] == 4
    ap = _f32(acc_pot)
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().oracle_kick(_p(vel4, C.c_float), _p(ap, C.c_float), C.c_uint32(vel4.shape[0]), C.c_float(h), _p(m, C.c_uint8))


def drift(pos_mass, vel4, h):
    """In place: pos_mass[i, a] = fma(vel4[i, a], h, pos_mass[i, a]), a < 3 (R23)."""
    assert pos_mass.dtype == np.float32 and pos_mass.flags.c_contiguous and pos_mass.shape[1] == 4
    v = _f32(vel4)
    lib().oracle_drift(_p(pos_mass, C.c_float), _p(v, C.c_float), C.c_uint32(pos_mass.shape[0]), C.c_float(h))


DIAG_FIELDS = ("K", "W", "Px", "Py", "Pz", "Lx", "Ly", "Lz", "M", "Cx", "Cy", "Cz")


def diagnostics(pos_mass, vel4, acc_pot):
    """float64[12] in the order of DIAG_FIELDS (R24)."""
    pm, v, ap = _f32(pos_mass), _f32(vel4), _f32(acc_pot)
    out = np.zeros(12, np.float64)
    lib().oracle_diagnostics(_p(pm, C.c_float), _p(v, C.c_float), _p(ap, C.c_float), C.c_uint32(pm.shape[0]),
                             _p(out, C.c_double))
    return out


def force_f32(pos_mass, theta, eps, **kw):
    """One force step; acc/pot in LOAD order rounded to the fp32 record the library returns (ax, ay, az, phi)."""
    s = full_step(pos_mass, theta, eps, **kw)
    ap = np.empty((pos_mass.shape[0], 4), np.float64)
    ap[s.perm, :3] = s.walk.acc
    ap[s.perm, 3] = s.walk.pot
    return ap.astype(np.float32)


def leapfrog(pos_mass, vel, theta, eps, dt, n_steps, acc_pot=None, **kw):
    """n_steps KDK steps with a shared time-step and the tree rebuilt every step (R22; BASELINE.json configs[2]).

    Returns (pos_mass, vel4, acc_pot) after the last step; inputs are not modified.  acc_pot, if given, is the
    force at the initial positions (otherwise it is computed first).
    """
    pm = np.array(pos_mass, dtype=np.float32, order="C")
    v4 = _vel4(vel)
    ap = force_f32(pm, theta, eps, **kw) if acc_pot is None else _f32(acc_pot).copy()
    h = np.float32(0.5) * np.float32(dt)
    for _ in range(n_steps):
        kick(v4, ap, h)
        drift(pm, v4, np.float32(dt))
        ap = force_f32(pm, theta, eps, **kw)
        kick(v4, ap, h)
    return pm, v4, ap


# ---- row f1: refreshed tree (oracle/refresh_oracle.cpp, R25) --------------------------------

def refresh(prev: Step, pos_mass, nleaf=16, ncrit=64, group_mode=2, active_mask=None, group_cell=512,
            mac_mode=0) -> Step:
    """The structures of ``prev`` (permutation, keys, cells, group membership) carried over to moved particles.

    pos_mass is the SAME particles in the SAME load order as the build that produced ``prev``.
    """
    del nleaf  # the cells are frozen
    import copy
    pm = _f32(pos_mass)
    spm = np.ascontiguousarray(pm[prev.perm])
    t = copy.deepcopy(prev.tree)
    act_sorted = None if active_mask is None else np.ascontiguousarray(active_mask, np.uint8)[prev.perm]
    g = groups(group_mode, ncrit, spm, t, act_sorted, group_cell)
    multipoles(spm, prev.sorted_keys, prev.lo, prev.side, t)
    if mac_mode == 1:  # R28: the particle boxes are recomputed from the new positions; nothing grows (R25 not needed)
        tight_mac(spm, t)
        return Step(prev.lo, prev.side, prev.keys, prev.perm, spm, prev.sorted_keys, t, g)
    lo = _f32(prev.lo)
    sk = np.ascontiguousarray(prev.sorted_keys, dtype=np.uint32)
    lib().oracle_extent_side(_p(spm, C.c_float), _p(sk, C.c_uint32), _p(lo, C.c_float), C.c_double(prev.side),
                             C.c_uint32(t.n_cells), _p(t.level, C.c_uint32), _p(t.first, C.c_uint32),
                             _p(t.count, C.c_uint32), _p(t.lside, C.c_float))
    return Step(prev.lo, prev.side, prev.keys, prev.perm, spm, prev.sorted_keys, t, g)


def refreshed_step(prev: Step, pos_mass, theta, eps, sel=None, order=2, threads=1, **kw) -> Step:
    s = refresh(prev, pos_mass, **kw)
    s.walk = _walk_maybe_threaded(theta, eps, s, sel, order, threads)
    return s


# ---- block time-steps (oracle/integrator_oracle.cpp, R26-R27) ------------------------------

def rungs(acc_pot, eta, eps, dt_max, kmax, rung=None, mask=None, tick=0):
    """rung is None: fresh assignment (R26) -> uint8[n].  Otherwise the R27 update of `rung` in place at `tick`."""
    ap = _f32(acc_pot)
    n = ap.shape[0]
    init = rung is None
    if init:
        rung = np.zeros(n, np.uint8)
    assert rung.dtype == np.uint8 and rung.flags.c_contiguous
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().oracle_rungs(_p(ap, C.c_float), C.c_uint32(n), C.c_float(eta), C.c_float(eps), C.c_float(dt_max),
                       C.c_uint32(kmax), _p(m, C.c_uint8), C.c_uint64(tick), _p(rung, C.c_uint8), C.c_int(int(init)))
    return rung


def active_at(rung, kmax, tick):
    r = np.ascontiguousarray(rung, np.uint8)
    mask = np.zeros(r.shape[0], np.uint8)
    lib().oracle_active_mask(_p(r, C.c_uint8), C.c_uint32(r.shape[0]), C.c_uint32(kmax), C.c_uint64(tick), _p(mask, C.c_uint8))
    return mask


def kick_rungs(vel4, acc_pot, rung, mask, dt_max):
    assert vel4.dtype == np.float32 and vel4.flags.c_contiguous and vel4.shape[1] == 4
    ap = _f32(acc_pot)
    r = np.ascontiguousarray(rung, np.uint8)
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().oracle_kick_rungs(_p(vel4, C.c_float), _p(ap, C.c_float), _p(r, C.c_uint8), _p(m, C.c_uint8),
                            C.c_uint32(vel4.shape[0]), C.c_float(dt_max))


class RebuildPolicy:
    """R30 (rebuild "only when the tree-traverse shows a considerable decline in performance ... an increase of
    the average number of particle-cell and particle-particle interactions"):
        I_t   = (sum n_pp + sum n_pc over the sinks walked in tick t) / (number of sinks walked)     (fp64)
        I_ref = I of the first recorded walk after the last full build
        rebuild at the start of a tick  <=>  a reference exists  and  I_last > factor I_ref          (factor fp32)
    """

    def __init__(self, factor=1.25):
        self.factor = float(np.float32(factor))
        self.ref = 0.0
        self.last = 0.0
        self.fresh = True          # no reference yet
        self.decisions = []        # True = rebuild, one entry per decide()

    def decide(self) -> bool:
        rebuild = (not self.fresh) and self.last > self.factor * self.ref
        self.decisions.append(bool(rebuild))
        return rebuild

    def built(self):
        self.fresh = True

    def record(self, w: WalkResult, walked_sorted: np.ndarray):
        k = int(walked_sorted.sum())
        if k == 0:
            return
        total = int(w.n_pp[walked_sorted].astype(np.int64).sum() + w.n_pc[walked_sorted].astype(np.int64).sum())
        self.last = float(total) / float(k)
        if self.fresh:
            self.ref = self.last
            self.fresh = False


def block_tick(pm, v4, ap, rung, tick, theta, eps, eta, dt_max, kmax, prev: Step = None, policy: RebuildPolicy = None,
               **kw):
    """One tick of the block scheme (R27), in place on pm / v4 / ap / rung.  prev: refresh this Step's tree instead
    of rebuilding (R25).  policy: decide between the two with R30 (prev must then be the last tick's Step, or None
    when no tree exists yet).  Returns (the Step of this tick, number of active particles walked)."""
    threads = kw.pop("threads", 1)          # host threads of the walk (fan-out only)
    m0 = active_at(rung, kmax, tick)
    kick_rungs(v4, ap, rung, m0, dt_max)
    drift(pm, v4, np.float32(np.ldexp(np.float32(dt_max), -kmax)))
    m1 = active_at(rung, kmax, tick + 1)
    if policy is not None and prev is not None and policy.decide():
        prev = None
    if prev is None:
        s = full_step(pm, theta, eps, active_mask=m1, threads=threads, **kw)
        if policy is not None:
            policy.built()
    else:
        s = refreshed_step(prev, pm, theta, eps, active_mask=m1, threads=threads, **kw)
    if policy is not None:
        policy.record(s.walk, m1[s.perm].astype(bool))
    sel = m1[s.perm].astype(bool)
    new = np.empty((int(sel.sum()), 4), np.float64)
    new[:, :3] = s.walk.acc[sel]
    new[:, 3] = s.walk.pot[sel]
    ap[s.perm[sel]] = new.astype(np.float32)
    kick_rungs(v4, ap, rung, m1, dt_max)
    rungs(ap, eta, eps, dt_max, kmax, rung=rung, mask=m1, tick=tick + 1)
    return s, int(m1.sum())
