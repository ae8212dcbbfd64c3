"""bonsai_diagnostics_static -- the entry point for callers that cannot allocate device memory -- against the existing
bonsai_diagnostics path.

Why the entry point exists: bonsai_diagnostics needs a context and therefore a caller-allocated workspace.  A monitor
hooked into a simulation that has already committed all of its device memory, a plug-in whose host application forbids
cudaMalloc, or a loop that cannot afford the device-wide synchronisation cudaMalloc / cudaFree may cause, has no
workspace to offer.  For them the reduction's scratch (113 920 bytes: block partials and a ticket) is a fixed
__device__ array inside libbonsai, and the call takes only the particle arrays, the 12-double result buffer and a
stream.

What is checked here: two calls in a row (the second one finds the first one's ticket and partial rows in the shared
scratch) both reproduce bonsai_diagnostics within the tolerance tests/test_gpu_integrator.py uses for that path
(|diff| <= 1e-12 * sum |terms|), at sizes below and above the grid cap and with a ragged tail; that the two calls give
the same bits; and that sizes beyond BONSAI_DIAG_STATIC_MAX_N are refused.  The test does not depend on what ran
before it in the process: it passes alone in a fresh interpreter (the first call then does the per-device set-up) and
after the rest of the suite.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide another test).
"""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1204_2280_b200 import Bonsai  # noqa: E402
from paper_1204_2280_b200 import bonsai as B  # noqa: E402


def _state(n, seed):
    rng = np.random.default_rng(seed)
    pm = rng.normal(size=(n, 4)).astype(np.float32)
    pm[:, 3] = rng.random(n).astype(np.float32) / n
    v = rng.normal(size=(n, 4)).astype(np.float32)
    a = (rng.normal(size=(n, 4)) * 5).astype(np.float32)
    return pm, v, a


def _scales(pm, v, a):
    """sum |terms| of each of the 12 sums (the yardstick of the 1e-12 gate, as in test_gpu_integrator.py)."""
    m = np.abs(pm[:, 3].astype(np.float64))
    x = pm[:, :3].astype(np.float64)
    vv = v[:, :3].astype(np.float64)
    out = []
    for k in B.DIAG_FIELDS:
        if k == "K":
            out.append(np.sum(0.5 * m * np.sum(vv * vv, axis=1)))
        elif k == "W":
            out.append(np.sum(0.5 * m * np.abs(a[:, 3].astype(np.float64))))
        elif k == "M":
            out.append(np.sum(m))
        elif k[0] == "P":
            out.append(np.sum(m * np.abs(vv[:, "xyz".index(k[1])])))
        elif k[0] == "C":
            out.append(np.sum(m * np.abs(x[:, "xyz".index(k[1])])))
        else:
            out.append(np.sum(m * np.linalg.norm(x, axis=1) * np.linalg.norm(vv, axis=1)))
    return np.array(out)


# 1: one thread; 1000: one block; 262161: 257 blocks with a ragged tail; 1300007: above the 1184-block grid cap, so the
# blocks stride and every row of the static scratch is in use
@pytest.mark.parametrize("n", [1, 1000, 262144 + 17, 1300007])
def test_static_diagnostics_match_the_context_path_twice(n):
    pm, v, a = _state(n, 7 + n % 5)
    pm_d, v_d, a_d = (torch.from_numpy(t).cuda() for t in (pm, v, a))
    want = Bonsai(n).diagnostics(pm_d, v_d, a_d).cpu().numpy()      # existing path: context + workspace
    tol = 1e-12 * _scales(pm, v, a) + 1e-300

    out = torch.full((12,), float("nan"), dtype=torch.float64, device="cuda")   # the caller's buffer
    first = B.diagnostics_static(pm_d, v_d, a_d, out).cpu().numpy().copy()
    assert np.all(np.abs(first - want) <= tol), (first, want)

    # second call on the same stream, other data in between so that the scratch is dirty with foreign partials
    pm2, v2, a2 = _state(max(n // 3, 1), 99)
    other = torch.empty(12, dtype=torch.float64, device="cuda")
    B.diagnostics_static(*(torch.from_numpy(t).cuda() for t in (pm2, v2, a2)), other)
    out.fill_(float("nan"))
    second = B.diagnostics_static(pm_d, v_d, a_d, out).cpu().numpy().copy()
    assert np.all(np.abs(second - want) <= tol), (second, want)
    assert np.array_equal(first, second)                             # fixed fold order: same bits every time


def test_static_diagnostics_rejects_sizes_beyond_the_maximum():
    """n = 0 and n > BONSAI_DIAG_STATIC_MAX_N are refused before anything is launched (the buffers are never touched,
    so small ones do); so are null and misaligned pointers.  The Python wrapper names the limit."""
    L = B.lib()
    buf = torch.zeros(64, dtype=torch.float32, device="cuda")
    out = torch.full((12,), 3.0, dtype=torch.float64, device="cuda")
    p, o = C.c_void_p(buf.data_ptr()), C.c_void_p(out.data_ptr())
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert B.DIAG_STATIC_MAX_N == 1 << 30
    assert L.bonsai_diagnostics_static(p, p, p, B.DIAG_STATIC_MAX_N + 1, o, st) == B.EINVAL
    assert L.bonsai_diagnostics_static(p, p, p, 0xFFFFFFFF, o, st) == B.EINVAL
    assert L.bonsai_diagnostics_static(p, p, p, 0, o, st) == B.EINVAL
    assert L.bonsai_diagnostics_static(None, p, p, 4, o, st) == B.EINVAL
    assert L.bonsai_diagnostics_static(C.c_void_p(buf.data_ptr() + 4), p, p, 4, o, st) == B.EINVAL
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), np.full(12, 3.0))       # nothing ran

    class _Huge:                                                     # a shape is all the wrapper looks at first
        shape = (B.DIAG_STATIC_MAX_N + 1, 4)
    with pytest.raises(ValueError, match="BONSAI_DIAG_STATIC_MAX_N"):
        B.diagnostics_static(_Huge(), None, None, out)
