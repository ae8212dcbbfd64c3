"""Thin ctypes binding of libbonsai (include/bonsai.h): argument marshalling only.

Every step of the force path runs in the CUDA kernels behind the C-ABI; PyTorch is used here for
device memory (the workspace, the particle / output tensors) and for the CUDA stream, nothing else.
There is NO CPU fallback: importing works without a GPU (so the symbol table can be checked), but
creating a :class:`Bonsai` without CUDA raises.

Names follow the header: ``Bonsai.load / build_tree / compute_multipoles / walk`` are
``bonsai_load / bonsai_build_tree / bonsai_compute_multipoles / bonsai_walk``.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import torch

from . import build as _build

OK, EINVAL, ESTATE, ECAPACITY, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5
N_STAGES = 9
STAGES = ("bbox", "keys", "sort", "reorder", "build", "groups", "multipoles", "walk", "integrate")
DIAG_FIELDS = ("K", "W", "Px", "Py", "Pz", "Lx", "Ly", "Lz", "M", "Cx", "Cy", "Cz")

# every symbol include/bonsai.h declares (tests check the library exports exactly these)
SYMBOLS = (
    "bonsai_workspace_bytes", "bonsai_create", "bonsai_load", "bonsai_build_tree",
    "bonsai_compute_multipoles", "bonsai_walk", "bonsai_step_host", "bonsai_destroy", "bonsai_sync", "bonsai_get_box",
    "bonsai_get_keys", "bonsai_get_perm", "bonsai_get_sorted_pos", "bonsai_get_cells", "bonsai_get_groups",
    "bonsai_get_counts", "bonsai_get_interaction_totals", "bonsai_set_timing", "bonsai_get_stage_ms",
    "bonsai_get_launch_count", "bonsai_strerror",
    "bonsai_kick", "bonsai_drift", "bonsai_leapfrog_step", "bonsai_diagnostics", "bonsai_refresh_tree",
    "bonsai_timestep_rungs", "bonsai_active_mask", "bonsai_kick_rungs", "bonsai_block_tick",
    "bonsai_measure_fp32_peak", "bonsai_get_rebuild_stats", "bonsai_step", "bonsai_get_graph_replays",
    "bonsai_diagnostics_static",
)


class Params(C.Structure):
    _fields_ = [("nleaf", C.c_uint32), ("ncrit", C.c_uint32), ("group_mode", C.c_uint32),
                ("cap_cells", C.c_uint32), ("group_cell", C.c_uint32), ("mac_mode", C.c_uint32),
                ("order", C.c_uint32), ("no_graph", C.c_uint32), ("rebuild_factor", C.c_float),
                ("mult_kernel", C.c_uint32), ("sort_passes", C.c_uint32)]


class CellsView(C.Structure):
    _fields_ = [("cap_cells", C.c_uint32)] + [(k, C.c_void_p) for k in (
        "n_cells", "level_offsets", "level", "first", "count", "first_child", "n_child", "parent",
        "mac", "quad", "walk_quad")]


class GroupsView(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("n_groups", "n_active", "active_list", "first", "count",
                                          "bmin", "bmax")]


class BonsaiError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        super().__init__(f"{what}: {strerror(code)} ({code})")


_lib = None


def lib() -> C.CDLL:
    """Load (building if stale) libbonsai.so and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    vp, u32, f32 = C.c_void_p, C.c_uint32, C.c_float
    L.bonsai_workspace_bytes.restype = C.c_size_t
    L.bonsai_workspace_bytes.argtypes = [u32, C.POINTER(Params)]
    L.bonsai_create.argtypes = [u32, C.POINTER(Params), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.bonsai_load.argtypes = [vp, vp, u32]
    L.bonsai_build_tree.argtypes = [vp]
    L.bonsai_compute_multipoles.argtypes = [vp]
    L.bonsai_walk.argtypes = [vp, f32, f32, vp, vp]
    L.bonsai_step_host.argtypes = [vp, vp, u32, f32, f32, vp, vp]
    L.bonsai_step.argtypes = [vp, vp, u32, f32, f32, vp, vp]
    L.bonsai_get_graph_replays.argtypes = [vp]
    L.bonsai_get_graph_replays.restype = C.c_uint64
    L.bonsai_destroy.argtypes = [vp]
    L.bonsai_destroy.restype = None
    L.bonsai_sync.argtypes = [vp]
    L.bonsai_get_box.argtypes = [vp, C.POINTER(vp)]
    L.bonsai_get_keys.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.bonsai_get_perm.argtypes = [vp, C.POINTER(vp)]
    L.bonsai_get_sorted_pos.argtypes = [vp, C.POINTER(vp)]
    L.bonsai_get_cells.argtypes = [vp, C.POINTER(CellsView)]
    L.bonsai_get_groups.argtypes = [vp, C.POINTER(GroupsView)]
    L.bonsai_get_counts.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    L.bonsai_get_interaction_totals.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.bonsai_set_timing.argtypes = [vp, C.c_int]
    L.bonsai_get_stage_ms.argtypes = [vp, C.POINTER(f32)]
    L.bonsai_get_launch_count.argtypes = [vp]
    L.bonsai_get_launch_count.restype = C.c_uint64
    L.bonsai_refresh_tree.argtypes = [vp]
    u64 = C.c_uint64
    L.bonsai_timestep_rungs.argtypes = [vp, vp, u32, f32, f32, f32, u32, vp, u64, vp, C.c_int]
    L.bonsai_active_mask.argtypes = [vp, vp, u32, u32, u64, vp]
    L.bonsai_kick_rungs.argtypes = [vp, vp, vp, vp, vp, u32, f32]
    L.bonsai_block_tick.argtypes = [vp, vp, vp, vp, vp, u32, u64, f32, f32, f32, f32, u32, C.c_int]
    L.bonsai_kick.argtypes = [vp, vp, vp, u32, f32, vp]
    L.bonsai_drift.argtypes = [vp, vp, vp, u32, f32]
    L.bonsai_leapfrog_step.argtypes = [vp, vp, vp, vp, u32, f32, f32, f32]
    L.bonsai_diagnostics.argtypes = [vp, vp, vp, vp, u32, vp]
    L.bonsai_diagnostics_static.argtypes = [vp, vp, vp, u32, vp, vp]
    L.bonsai_get_rebuild_stats.argtypes = [vp, C.POINTER(u32), C.POINTER(u32), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.bonsai_measure_fp32_peak.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_double)]
    L.bonsai_strerror.argtypes = [C.c_int]
    L.bonsai_strerror.restype = C.c_char_p
    for name in SYMBOLS:  # fail loudly on a stale or partial library
        getattr(L, name)
    _lib = L
    return L


def strerror(code: int) -> str:
    return lib().bonsai_strerror(code).decode()


def _check(code: int, what: str) -> None:
    if code != OK:
        raise BonsaiError(code, what)


def measure_fp32_peak(packed: bool = True, iters: int = 20000, stream: "torch.cuda.Stream | None" = None) -> float:
    """bonsai_measure_fp32_peak: measured FP32 TFLOP/s of the current device (FFMA2 when packed, else FFMA)."""
    if not torch.cuda.is_available():
        raise RuntimeError("libbonsai needs a CUDA device (sm_100a); there is no CPU fallback")
    out = C.c_double(0.0)
    st = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(lib().bonsai_measure_fp32_peak(st, int(bool(packed)), int(iters), C.byref(out)), "bonsai_measure_fp32_peak")
    return float(out.value)


DIAG_STATIC_MAX_N = 1 << 30            # BONSAI_DIAG_STATIC_MAX_N
DIAG_STATIC_SCRATCH_BYTES = 113920     # BONSAI_DIAG_STATIC_SCRATCH_BYTES


def diagnostics_static(pos_mass: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor, out: torch.Tensor,
                       stream: "torch.cuda.Stream | None" = None) -> torch.Tensor:
    """bonsai_diagnostics_static: the 12 diagnostics sums (DIAG_FIELDS) without a context or a workspace.

    For code that cannot allocate device memory (a monitor inside a simulation whose memory pool is spent, a plug-in
    whose host forbids cudaMalloc, a loop that must not risk the device-wide synchronisation of cudaMalloc / cudaFree):
    the scratch is a fixed 113 920-byte array inside libbonsai, held on every GPU that loads the library.  This wrapper
    allocates nothing either, which is why ``out`` (float64[12] on the tensors' device) is a required argument.
    All calls on a device share that scratch: keep them on one stream -- calls that overlap on the GPU race.  The first
    call on a device resolves the scratch address and should come before any stream capture.  n <= DIAG_STATIC_MAX_N."""
    if not torch.cuda.is_available():
        raise RuntimeError("libbonsai needs a CUDA device (sm_100a); there is no CPU fallback")
    n = int(pos_mass.shape[0])
    if n > DIAG_STATIC_MAX_N:
        raise ValueError(f"bonsai_diagnostics_static: n = {n} exceeds BONSAI_DIAG_STATIC_MAX_N = {DIAG_STATIC_MAX_N}")
    for t in (pos_mass, vel, acc_pot):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == (n, 4)
                and t.device == pos_mass.device):
            raise ValueError("bonsai_diagnostics_static: contiguous float32 CUDA tensors of shape (n, 4) on one device")
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 12
            and out.device == pos_mass.device):
        raise ValueError("bonsai_diagnostics_static: out must be a contiguous float64[12] tensor on the same device")
    with torch.cuda.device(pos_mass.device):  # the device that owns the buffers and the stream must be current
        st = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
        _check(lib().bonsai_diagnostics_static(C.c_void_p(pos_mass.data_ptr()), C.c_void_p(vel.data_ptr()),
                                               C.c_void_p(acc_pot.data_ptr()), n, C.c_void_p(out.data_ptr()), st),
               "bonsai_diagnostics_static")
    return out


def workspace_bytes(n_max: int, nleaf: int = 16, ncrit: int = 64, group_mode: int = 2,
                    cap_cells: int = 0, group_cell: int = 0, mac_mode: int = 0, order: int = 2) -> int:
    p = Params(nleaf, ncrit, group_mode, cap_cells, group_cell, mac_mode, order, 0, 0.0)
    return int(lib().bonsai_workspace_bytes(n_max, C.byref(p)))


_DT = {torch.uint32: 4, torch.float32: 4, torch.uint8: 1, torch.int32: 4}


@dataclass
class Cells:
    """Host copies (numpy) of the cell arrays, trimmed to n_cells."""
    n_cells: int
    level_offsets: "object"
    level: "object"
    first: "object"
    count: "object"
    first_child: "object"
    n_child: "object"
    parent: "object"
    com_m: "object" = None   # float32[n_cells, 4]
    quad: "object" = None    # float32[n_cells, 6]
    delta: "object" = None
    lside: "object" = None
    walk_quad: "object" = None  # float32[n_cells, 8]: P = tr I - 3 Q (6), tr, pad


@dataclass
class Groups:
    n_groups: int
    n_active: int
    active_list: "object"
    first: "object"
    count: "object"
    bmin: "object"
    bmax: "object"


class Bonsai:
    """One libbonsai context on ``device`` for up to ``n_max`` particles.

    The workspace is one ``torch.uint8`` tensor owned by this object; all calls are enqueued on
    ``stream`` (default: the current torch stream at construction).
    """

    def __init__(self, n_max: int, nleaf: int = 16, ncrit: int = 64, group_mode: int = 2,
                 cap_cells: int = 0, group_cell: int = 0, device: str | torch.device = "cuda:0",
                 stream: "torch.cuda.Stream | None" = None, mac_mode: int = 0, order: int = 2,
                 rebuild_factor: float = 0.0, use_graph: bool = True, mult_kernel: int = 0, sort_passes: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("libbonsai needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device(device)
        self._L = lib()
        self.n_max = int(n_max)
        self.n = 0
        self.params = Params(nleaf, ncrit, group_mode, cap_cells, group_cell, mac_mode, order, 0 if use_graph else 1,
                             rebuild_factor, mult_kernel, sort_passes)
        nbytes = int(self._L.bonsai_workspace_bytes(self.n_max, C.byref(self.params)))
        if nbytes == 0:
            raise BonsaiError(EINVAL, "bonsai_workspace_bytes")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            h = C.c_void_p()
            _check(self._L.bonsai_create(self.n_max, C.byref(self.params), self._ws_ptr, nbytes,
                                         C.c_void_p(self.stream.cuda_stream), C.byref(h)), "bonsai_create")
        self._h = h
        self.workspace_bytes = nbytes
        self._keep = []  # tensors the library reads asynchronously

    # ---- the force path ------------------------------------------------------------------------
    def load(self, pos_mass: torch.Tensor) -> None:
        """pos_mass: float32[n, 4] on the device, contiguous (x, y, z, m), load order.  Not copied."""
        assert pos_mass.is_cuda and pos_mass.dtype == torch.float32 and pos_mass.is_contiguous()
        assert pos_mass.dim() == 2 and pos_mass.shape[1] == 4
        n = pos_mass.shape[0]
        _check(self._L.bonsai_load(self._h, pos_mass.data_ptr(), n), "bonsai_load")
        self.n = n
        self._keep = [pos_mass]

    def build_tree(self) -> None:
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_build_tree(self._h), "bonsai_build_tree")

    def refresh_tree(self) -> None:
        """Keep the sorted order and the cells of the last build_tree(); re-gather the moved particles (R25)."""
        _check(self._L.bonsai_refresh_tree(self._h), "bonsai_refresh_tree")

    def compute_multipoles(self) -> None:
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_compute_multipoles(self._h), "bonsai_compute_multipoles")

    def walk(self, theta: float, eps: float, active_mask: torch.Tensor | None = None,
             out: torch.Tensor | None = None) -> torch.Tensor:
        """Returns acc_pot float32[n, 4] = (ax, ay, az, phi) in load order (device tensor)."""
        if out is None:
            with torch.cuda.stream(self.stream):  # zero-filled on the stream the walk runs on
                out = torch.zeros((self.n, 4), dtype=torch.float32, device=self.device)
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.shape == (self.n, 4)
        mptr = None
        if active_mask is not None:
            assert active_mask.is_cuda and active_mask.dtype == torch.uint8 and active_mask.is_contiguous()
            assert active_mask.numel() == self.n
            mptr = active_mask.data_ptr()
            self._keep.append(active_mask)
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_walk(self._h, float(theta), float(eps), mptr, out.data_ptr()), "bonsai_walk")
        return out

    def step(self, pos_mass: torch.Tensor, theta: float, eps: float, active_mask=None, out=None) -> torch.Tensor:
        """bonsai_step: load -> build_tree -> compute_multipoles -> walk as one call (no host sync); replayed as a
        CUDA graph while the same tensors and parameters come back (unless use_graph=False or timing is on)."""
        assert pos_mass.is_cuda and pos_mass.dtype == torch.float32 and pos_mass.is_contiguous()
        assert pos_mass.dim() == 2 and pos_mass.shape[1] == 4
        n = pos_mass.shape[0]
        if out is None:
            # a fresh result tensor per call would make every call a new graph (the buffers are part of the key):
            # without a caller-owned `out` the step is enqueued kernel by kernel
            self.load(pos_mass)
            self.build_tree()
            self.compute_multipoles()
            return self.walk(theta, eps, active_mask, None)
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.shape == (n, 4)
        mptr = None
        if active_mask is not None:
            assert active_mask.is_cuda and active_mask.dtype == torch.uint8 and active_mask.is_contiguous()
            assert active_mask.numel() == n
            mptr = active_mask.data_ptr()
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_step(self._h, pos_mass.data_ptr(), n, float(theta), float(eps), mptr, out.data_ptr()),
                   "bonsai_step")
        self.n = n
        self._keep = [pos_mass] + ([active_mask] if active_mask is not None else [])
        return out

    def step_host(self, pos_mass_host: torch.Tensor, theta: float, eps: float,
                  active_mask_host: torch.Tensor | None = None, out_host: torch.Tensor | None = None) -> torch.Tensor:
        """bonsai_step_host: HOST tensors in (float32[n,4], ideally pinned), HOST float32[n,4] out; blocking."""
        assert not pos_mass_host.is_cuda and pos_mass_host.dtype == torch.float32 and pos_mass_host.is_contiguous()
        n = pos_mass_host.shape[0]
        if out_host is None:
            out_host = torch.zeros((n, 4), dtype=torch.float32).pin_memory()
        assert not out_host.is_cuda and out_host.dtype == torch.float32 and out_host.is_contiguous()
        mptr = None
        if active_mask_host is not None:
            assert not active_mask_host.is_cuda and active_mask_host.dtype == torch.uint8
            mptr = active_mask_host.data_ptr()
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_step_host(self._h, pos_mass_host.data_ptr(), n, float(theta), float(eps), mptr,
                                            out_host.data_ptr()), "bonsai_step_host")
        self.n = n
        return out_host

    # ---- row f2: integrator and diagnostics ---------------------------------------------------------
    def _f4(self, t: torch.Tensor, n: int | None = None) -> int:
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.dim() == 2 and t.shape[1] == 4
        assert n is None or t.shape[0] == n
        return t.data_ptr()

    def kick(self, vel: torch.Tensor, acc_pot: torch.Tensor, step: float, active_mask: torch.Tensor | None = None) -> None:
        """In place on the device: vel.xyz = fma(acc_pot.xyz, step, vel.xyz) for masked-in particles (float32[n,4])."""
        n = vel.shape[0]
        mptr = None
        if active_mask is not None:
            assert active_mask.is_cuda and active_mask.dtype == torch.uint8 and active_mask.numel() == n
            mptr = active_mask.data_ptr()
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_kick(self._h, self._f4(vel), self._f4(acc_pot, n), n, float(step), mptr), "bonsai_kick")

    def drift(self, pos_mass: torch.Tensor, vel: torch.Tensor, step: float) -> None:
        """In place on the device: pos_mass.xyz = fma(vel.xyz, step, pos_mass.xyz)."""
        n = pos_mass.shape[0]
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_drift(self._h, self._f4(pos_mass), self._f4(vel, n), n, float(step)), "bonsai_drift")

    def leapfrog_step(self, pos_mass: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor, theta: float,
                      eps: float, dt: float) -> None:
        """One KDK step in place (bonsai_leapfrog_step); acc_pot is the force at the current positions on entry."""
        n = pos_mass.shape[0]
        self._keep = [pos_mass]
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_leapfrog_step(self._h, self._f4(pos_mass), self._f4(vel, n), self._f4(acc_pot, n), n,
                                                float(theta), float(eps), float(dt)), "bonsai_leapfrog_step")
        self.n = n

    def diagnostics(self, pos_mass: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor,
                    out: torch.Tensor | None = None) -> torch.Tensor:
        """float64[12] device tensor in the order of DIAG_FIELDS (asynchronous)."""
        n = pos_mass.shape[0]
        if out is None:
            out = torch.zeros(12, dtype=torch.float64, device=self.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 12 and out.is_contiguous()
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_diagnostics(self._h, self._f4(pos_mass), self._f4(vel, n), self._f4(acc_pot, n), n,
                                              out.data_ptr()), "bonsai_diagnostics")
        return out

    # ---- block time-steps (R26, R27) ----------------------------------------------------------------
    @staticmethod
    def _u8(t: torch.Tensor, n: int) -> int:
        assert t.is_cuda and t.dtype == torch.uint8 and t.is_contiguous() and t.numel() == n
        return t.data_ptr()

    def timestep_rungs(self, acc_pot: torch.Tensor, eta: float, eps: float, dt_max: float, kmax: int,
                       rung: torch.Tensor | None = None, active_mask: torch.Tensor | None = None,
                       tick: int = 0) -> torch.Tensor:
        """rung is None: fresh assignment (R26) -> uint8[n] device tensor; else the end-of-tick update in place."""
        n = acc_pot.shape[0]
        init = rung is None
        if init:
            rung = torch.zeros(n, dtype=torch.uint8, device=self.device)
        mptr = None if active_mask is None else self._u8(active_mask, n)
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_timestep_rungs(self._h, self._f4(acc_pot), n, float(eta), float(eps), float(dt_max),
                                                 int(kmax), mptr, int(tick), self._u8(rung, n), int(init)),
                   "bonsai_timestep_rungs")
        return rung

    def active_mask(self, rung: torch.Tensor, kmax: int, tick: int, out: torch.Tensor | None = None) -> torch.Tensor:
        n = rung.numel()
        if out is None:
            out = torch.zeros(n, dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_active_mask(self._h, self._u8(rung, n), n, int(kmax), int(tick), self._u8(out, n)),
                   "bonsai_active_mask")
        return out

    def kick_rungs(self, vel: torch.Tensor, acc_pot: torch.Tensor, rung: torch.Tensor,
                   active_mask: torch.Tensor | None, dt_max: float) -> None:
        n = vel.shape[0]
        mptr = None if active_mask is None else self._u8(active_mask, n)
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_kick_rungs(self._h, self._f4(vel), self._f4(acc_pot, n), self._u8(rung, n), mptr, n,
                                             float(dt_max)), "bonsai_kick_rungs")

    def block_tick(self, pos_mass: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor, rung: torch.Tensor, tick: int,
                   theta: float, eps: float, eta: float, dt_max: float, kmax: int, rebuild: "bool | int" = True) -> None:
        """One tick of the block time-step scheme in place (bonsai_block_tick).  rebuild: True / False, or -1 = decided
        on the device (R30)."""
        n = pos_mass.shape[0]
        self._keep = [pos_mass]
        with torch.cuda.device(self.device):
            _check(self._L.bonsai_block_tick(self._h, self._f4(pos_mass), self._f4(vel, n), self._f4(acc_pot, n),
                                             self._u8(rung, n), n, int(tick), float(theta), float(eps), float(eta),
                                             float(dt_max), int(kmax), -1 if (rebuild is not True and rebuild is not False and int(rebuild) < 0) else int(bool(rebuild))), "bonsai_block_tick")
        self.n = n

    def rebuild_stats(self) -> dict:
        nd, nr, ref, last = C.c_uint32(0), C.c_uint32(0), C.c_double(0), C.c_double(0)
        _check(self._L.bonsai_get_rebuild_stats(self._h, C.byref(nd), C.byref(nr), C.byref(ref), C.byref(last)),
               "bonsai_get_rebuild_stats")
        return {"n_decisions": int(nd.value), "n_rebuilds": int(nr.value), "ipp_ref": float(ref.value),
                "ipp_last": float(last.value)}

    def sync(self) -> None:
        _check(self._L.bonsai_sync(self._h), "bonsai_sync")

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h:
            try:
                torch.cuda.synchronize(self.device)
            except Exception:
                pass
            self._L.bonsai_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- timing / counters ---------------------------------------------------------------------
    def set_timing(self, enable: bool) -> None:
        _check(self._L.bonsai_set_timing(self._h, int(enable)), "bonsai_set_timing")

    def stage_ms(self) -> dict:
        arr = (C.c_float * N_STAGES)()
        _check(self._L.bonsai_get_stage_ms(self._h, arr), "bonsai_get_stage_ms")
        return {k: float(arr[i]) for i, k in enumerate(STAGES)}

    def launch_count(self) -> int:
        return int(self._L.bonsai_get_launch_count(self._h))

    def graph_replays(self) -> int:
        return int(self._L.bonsai_get_graph_replays(self._h))

    def interaction_totals(self) -> tuple[int, int]:
        a, b = C.c_uint64(0), C.c_uint64(0)
        _check(self._L.bonsai_get_interaction_totals(self._h, C.byref(a), C.byref(b)),
               "bonsai_get_interaction_totals")
        return int(a.value), int(b.value)

    # ---- introspection: host copies for the parity tests ---------------------------------------
    def _view(self, ptr: int, count: int, dtype: torch.dtype) -> torch.Tensor:
        """A torch tensor aliasing ``count`` elements of workspace memory at device pointer ``ptr``."""
        off = ptr - self.workspace.data_ptr()
        assert 0 <= off and off + count * _DT[dtype] <= self.workspace.numel()
        return self.workspace[off: off + count * _DT[dtype]].view(dtype)

    def _host(self, ptr: int, count: int, dtype: torch.dtype):
        self.sync()
        if dtype == torch.uint32:  # numpy handles uint32 natively; go through int32 bits
            return self._view(ptr, count, torch.int32).cpu().numpy().view("uint32").copy()
        return self._view(ptr, count, dtype).cpu().numpy().copy()

    def box(self):
        p = C.c_void_p()
        _check(self._L.bonsai_get_box(self._h, C.byref(p)), "bonsai_get_box")
        v = self._host(p.value, 4, torch.float32)
        return v[:3].copy(), float(v[3])

    def keys(self):
        """uint32[n, 3] sorted keys (hi, mid, lo)."""
        import numpy as np
        a, b, c = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(self._L.bonsai_get_keys(self._h, C.byref(a), C.byref(b), C.byref(c)), "bonsai_get_keys")
        return np.stack([self._host(p.value, self.n, torch.uint32) for p in (a, b, c)], axis=1)

    def perm(self):
        p = C.c_void_p()
        _check(self._L.bonsai_get_perm(self._h, C.byref(p)), "bonsai_get_perm")
        return self._host(p.value, self.n, torch.uint32)

    def sorted_pos(self):
        p = C.c_void_p()
        _check(self._L.bonsai_get_sorted_pos(self._h, C.byref(p)), "bonsai_get_sorted_pos")
        return self._host(p.value, 4 * self.n, torch.float32).reshape(self.n, 4)

    def cells(self, with_multipoles: bool = True) -> Cells:
        v = CellsView()
        _check(self._L.bonsai_get_cells(self._h, C.byref(v)), "bonsai_get_cells")
        nc = int(self._host(v.n_cells, 1, torch.uint32)[0])
        if nc > v.cap_cells:
            raise BonsaiError(ECAPACITY, "bonsai_get_cells")
        u = lambda p: self._host(p, nc, torch.uint32)
        out = Cells(nc, self._host(v.level_offsets, 32, torch.uint32), u(v.level), u(v.first), u(v.count),
                    u(v.first_child), u(v.n_child), u(v.parent))
        if with_multipoles:
            mac = self._host(v.mac, 8 * nc, torch.float32).reshape(nc, 8)
            quad = self._host(v.quad, 6 * nc, torch.float32).reshape(nc, 6)
            out.com_m = mac[:, :4].copy()
            out.delta = mac[:, 4].copy()
            out.lside = mac[:, 5].copy()
            out.quad = quad
            out.walk_quad = self._host(v.walk_quad, 8 * nc, torch.float32).reshape(nc, 8)
        return out

    def groups(self) -> Groups:
        v = GroupsView()
        _check(self._L.bonsai_get_groups(self._h, C.byref(v)), "bonsai_get_groups")
        ng = int(self._host(v.n_groups, 1, torch.uint32)[0])
        na = int(self._host(v.n_active, 1, torch.uint32)[0])
        return Groups(ng, na, self._host(v.active_list, na, torch.uint32), self._host(v.first, ng, torch.uint32),
                      self._host(v.count, ng, torch.uint32),
                      self._host(v.bmin, 3 * ng, torch.float32).reshape(ng, 3),
                      self._host(v.bmax, 3 * ng, torch.float32).reshape(ng, 3))

    def counts(self):
        a, b = C.c_void_p(), C.c_void_p()
        _check(self._L.bonsai_get_counts(self._h, C.byref(a), C.byref(b)), "bonsai_get_counts")
        return self._host(a.value, self.n, torch.uint32), self._host(b.value, self.n, torch.uint32)
