"""B200-native Barnes-Hut force step after "Bonsai: A GPU Tree-Code" (arXiv 1204.2280).

The product is the C-ABI library ``libbonsai.so`` (include/bonsai.h, sources under csrc/);
:mod:`paper_1204_2280_b200.bonsai` is its thin ctypes binding and
:mod:`paper_1204_2280_b200.workloads` the seeded input generator.
"""
from .bonsai import Bonsai, BonsaiError, lib, workspace_bytes, STAGES  # noqa: F401
