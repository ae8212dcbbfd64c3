"""Per-region instruction totals of one kernel from an Nsight Compute source-page export.

    ncu -i REPORT.ncu-rep --page source --csv --print-source cuda,sass [--kernel-name regex:NAME] > src.csv
    python -m paper_1204_2280_b200.ncu_lines src.csv --walk            # regions of csrc/walk.cu, found by its markers
    python -m paper_1204_2280_b200.ncu_lines src.csv --lines           # one row per source line

The export lists every SASS instruction under each source line of its inline stack, so the same address appears
several times; here each address is counted ONCE and attributed to the outermost (largest) line of the kernel's own
file it is listed under; instructions listed only under the inlined packed-arithmetic helpers take the region of
their predecessor in address order (the loop they sit in).  Columns: executed warp instructions, share, the same split into packed FP32 (FFMA2 / FMUL2 /
FADD2: two issue cycles each), scalar FP32, integer-ALU-pipe instructions (what FFMA2 cannot overlap with, see
`report.py --only issue_mix`), shared / global memory, MUFU, and the rest.  Needs -lineinfo (build.py sets it).
"""
from __future__ import annotations

import argparse
import collections
import csv
import os

PACKED = {"FFMA2", "FMUL2", "FADD2"}
SCALAR_FP = {"FFMA", "FMUL", "FADD", "DADD", "DFMA", "DMUL", "F2F", "I2F", "F2I", "FMNMX", "FMNMX3", "FSETP", "FSEL", "HFMA2"}
ALU = {"IADD3", "ISETP", "LOP3", "SEL", "LEA", "SHF", "MOV", "POPC", "PRMT", "P2R", "R2P", "PLOP3", "IMNMX", "VIADDMNMX",
       "VIADD", "IABS", "FLO", "BREV", "IMAD", "CS2R", "UIADD3", "UISETP", "UPLOP3", "ULOP3", "UMOV", "USEL", "UIMAD",
       "ULEA", "USHF", "R2UR", "S2R", "S2UR", "BMSK", "SGXT", "LDC", "LDCU", "ULDC"}
MEM = {"LDS", "STS", "LDG", "STG", "LDL", "STL", "ATOM", "ATOMS", "ATOMG", "RED", "LD", "ST"}

# (name, marker that starts the region in csrc/walk.cu); a region ends where the next one starts
WALK_MARKERS = [
    ("helpers: packed fp32 intrinsics (inlined into the two loops)", "__device__ __forceinline__ float rsqrt_fast"),
    ("p-p loop", "__device__ __forceinline__ void eval_pp_packed"),
    ("p-c staging (cell records -> shared memory)", "__device__ __forceinline__ void eval_pc"),
    ("p-c loop", "        const f32x2 nsx = s.nx2, nsy = s.ny2, nsz = s.nz2;\n        const f32x2 e2 = bc(a.eps2);"),
    ("team barrier / chunk set-up", "__device__ __forceinline__ void team_barrier"),
    ("pop: runs -> 32 cells", "// ---- pop as many runs as fit into 32 lanes ----"),
    ("opening test (MAC)", "// ---- opening test (R9)"),
    ("push child runs", "// ---- rejected internal cells: push their child runs ----"),
    ("accepted cells -> id ring, hand-off to the p-c loop", "// ---- accepted cells ----"),
    ("leaf expansion -> particle ring, hand-off to the p-p loop", "// ---- rejected leaves: expand into particles ----"),
    ("tails, team fold, output", "    if (!ok) return false;"),
    ("group scheduler, kernel entry", "__device__ __forceinline__ void walk_groups"),
    ("host", "using WalkKernel"),
]


def load(path: str):
    rows = list(csv.reader(open(path)))
    h_i = next(i for i, r in enumerate(rows) if r and r[0] == "Line No")
    h = rows[h_i]
    i_line, i_addr, i_inst = h.index("Line No"), h.index("Address"), h.index("Instructions Executed")
    addr, src, cur = {}, {}, None
    for r in rows[h_i + 1:]:
        if len(r) < len(h):
            continue
        if r[i_line]:
            try:
                cur = int(r[i_line])
                src[cur] = r[1]
            except ValueError:
                cur = None
            continue
        if cur is None or not r[i_addr]:
            continue
        try:
            cnt = int(r[i_inst])
        except ValueError:
            continue
        parts = r[3].split()
        op = (parts[1] if parts[0].startswith("@") else parts[0]).split(".")[0]
        a = addr.setdefault(r[i_addr], [0, cnt, op])
        a[0] = max(a[0], cur)
    return addr, src


def classify(op: str) -> str:
    if op in PACKED:
        return "packed"
    if op in SCALAR_FP:
        return "scalar_fp"
    if op in ALU:
        return "alu"
    if op in MEM:
        return "mem"
    if op == "MUFU":
        return "mufu"
    return "other"


def walk_regions(source_file: str):
    text = open(source_file).read()
    starts = []
    for name, marker in WALK_MARKERS:
        k = text.find(marker)
        if k < 0:
            raise SystemExit(f"marker not found in {source_file}: {marker[:50]!r}")
        starts.append((text.count("\n", 0, k) + 1, name))
    starts.sort()
    return [(name, lo, (starts[i + 1][0] - 1) if i + 1 < len(starts) else 10 ** 9) for i, (lo, name) in enumerate(starts)]


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("csv")
    ap.add_argument("--walk", action="store_true", help="regions of csrc/walk.cu")
    ap.add_argument("--lines", action="store_true", help="one row per source line")
    args = ap.parse_args()
    addr, src = load(args.csv)
    total = sum(a[1] for a in addr.values())
    cols = ("packed", "scalar_fp", "alu", "mem", "mufu", "other")
    agg = collections.OrderedDict()
    if args.walk:
        regions = walk_regions(os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "walk.cu"))
        for name, _, _ in regions:
            agg[name] = collections.Counter()
        agg["(other files / headers)"] = collections.Counter()
        # the packed-arithmetic helpers are inlined: an instruction listed only under a helper line belongs to the loop
        # around it -- give it the region of the nearest preceding instruction (in address order) that has one
        helper = regions[0][0]
        last = "(other files / headers)"
        for a in sorted(addr, key=lambda x: int(x, 16)):
            line, cnt, op = addr[a]
            name = next((n for n, lo, hi in regions if lo <= line <= hi), "(other files / headers)")
            if name == helper:
                name = last
            else:
                last = name
            agg[name][classify(op)] += cnt
    else:
        for line, cnt, op in sorted(addr.values()):
            agg.setdefault(f"{line}: {src.get(line, '').strip()[:70]}", collections.Counter())[classify(op)] += cnt
    print(f"{len(addr)} SASS instructions, {total} executed warp instructions\n")
    print("| region | executed | share | " + " | ".join(cols) + " |")
    print("|---|---|---|" + "---|" * len(cols))
    for name, c in agg.items():
        t = sum(c.values())
        if t:
            print(f"| {name} | {t / 1e6:.1f} M | {100 * t / total:.2f} % | " + " | ".join(f"{c[k] / 1e6:.1f}" for k in cols) + " |")
    tot = collections.Counter()
    for c in agg.values():
        tot.update(c)
    print(f"| **total** | {total / 1e6:.1f} M | 100 % | " + " | ".join(f"{tot[k] / 1e6:.1f}" for k in cols) + " |")


if __name__ == "__main__":
    main()
