"""Host-side logic that needs no GPU: the C-ABI library exports what include/bonsai.h declares, the bench's
multi-rank plumbing (replicas only) works over gloo with world_size 2, and the reference arm
prints exactly one JSON line from rank 0."""
import json
import os
import re
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_library_exports_every_declared_symbol():
    import ctypes
    from paper_1204_2280_b200 import build as B
    from paper_1204_2280_b200.bonsai import SYMBOLS
    lib = ctypes.CDLL(B.build())          # loading needs no GPU (static cudart, no kernels run)
    header = open(os.path.join(ROOT, "include", "bonsai.h")).read()
    declared = set(re.findall(r"\b(bonsai_[a-z_0-9]+)\s*\(", header))
    declared -= {"bonsai_ctx", "bonsai_params"}
    assert declared == set(SYMBOLS), declared ^ set(SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    # argument checking happens before any CUDA call
    assert lib.bonsai_workspace_bytes(0, None) == 0
    lib.bonsai_strerror.restype = ctypes.c_char_p
    assert lib.bonsai_strerror(-2) == b"call out of order"


def test_parameter_validation_needs_no_gpu():
    """bonsai_workspace_bytes resolves and checks bonsai_params on the host (0 = rejected): the defaults, the kernel
    choices added in round 2 (sort_passes in {0, 4, 5, 6}, mult_kernel in {0, 1, 2}) and the older limits."""
    import ctypes
    from paper_1204_2280_b200 import build as B
    from paper_1204_2280_b200.bonsai import Params
    lib = ctypes.CDLL(B.build())
    lib.bonsai_workspace_bytes.restype = ctypes.c_size_t
    lib.bonsai_workspace_bytes.argtypes = [ctypes.c_uint32, ctypes.POINTER(Params)]

    def nbytes(n=100_000, **kw):
        p = Params()
        for k, v in kw.items():
            setattr(p, k, v)
        return lib.bonsai_workspace_bytes(n, ctypes.byref(p))

    base = nbytes()
    assert base > 100_000 * 100 and base == lib.bonsai_workspace_bytes(100_000, None)
    for passes in (4, 5, 6):
        assert nbytes(sort_passes=passes) == base          # a launch choice, not a layout choice
    for bad in (1, 3, 7):
        assert nbytes(sort_passes=bad) == 0
    assert nbytes(mult_kernel=1) == base and nbytes(mult_kernel=2) == base and nbytes(mult_kernel=3) == 0
    assert nbytes(nleaf=65) == 0 and nbytes(ncrit=65) == 0 and nbytes(group_mode=3) == 0
    assert nbytes(mac_mode=2) == 0 and nbytes(order=3) == 0 and nbytes(rebuild_factor=0.5) == 0
    assert nbytes(n=0) == 0


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
mine = [10.0 + 5.0 * rank, 30.0 - 7.0 * rank]          # rank 0: 10, 30   rank 1: 15, 23
got = bench.max_over_ranks(mine, 2)
assert got == [15.0, 30.0], got
assert bench.aggregate_value(1000, 2, 4, got[0]) == 2 * 1000 * 4 / 15e-3
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_max_over_ranks_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=_free_port()))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    for r, p in enumerate(procs):
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        assert f"ok {r}" in out


def test_reference_arm_under_torchrun_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "plummer_32k"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "particles_per_second_full_step" and d["n_gpus"] == 2
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "plummer_32k"


def test_ours_arm_fails_loudly_without_cuda():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
