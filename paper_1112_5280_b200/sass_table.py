"""Opcode table of the hot kernels in the built liblqcd.so: what the compiler made of the hand-written paths.

    python -m paper_1112_5280_b200.sass_table            # markdown table on stdout (needs cuobjdump; no GPU)

Per kernel: registers, spill bytes, static shared memory (cuobjdump --dump-resource-usage), SASS instruction count and
the counts of the opcodes DESIGN.md argues from -- packed fp32 arithmetic (FFMA2 / FADD2 / FMUL2), fp64 FMA (DFMA), the
half-operand FMA of the 16-bit path (HFMA2 with fp32 accumulate shows as FHFMA / HFMA2), 256-bit global accesses
(LDG / STG with a .256 modifier, e.g. LDG.E.ENL2.256.CONSTANT), TMA bulk copies (UBLKCP) and mbarrier waits (SYNCS), shuffles (SHFL),
MUFU (the 8-real decoder's sin / cos / rsqrt / rcp).  Reads only the library; holds none of the method's arithmetic."""
from __future__ import annotations

import re
import subprocess
import sys

from . import _build

CUOBJDUMP = "/usr/local/cuda/bin/cuobjdump"
OPCODES = ("FFMA2", "FADD2", "FMUL2", "FFMA", "DFMA", "FHFMA", "HFMA2", "LDG.256", "LDG.128", "LDG.64", "STG.256", "UBLKCP",
           "SYNCS", "SHFL", "MUFU", "LDS", "BAR")
# the kernels that carry the bench lines (name filter on the demangled signature, label)
HOT = (
    (r"dslash_kernel<float, 12, 0, false, 64>", "gather fp32 recon-12 (headline)"),
    (r"dslash_kernel<double, 12, 0, false, 64>", "gather fp64 recon-12 (headline)"),
    (r"dslash_kernel<float, 18, 0, false, 64>", "gather fp32 recon-18"),
    (r"dslash_kernel<double, 18, 0, false, 64>", "gather fp64 recon-18"),
    (r"dslash_kernel<float, 8, 0, false, 64>", "gather fp32 recon-8"),
    (r"dslash_kernel<double, 8, 0, false, 64>", "gather fp64 recon-8"),
    (r"dslash_kernel<__half, 12, 0, false, 64>", "gather 16-bit storage"),
    (r"dslash_kernel<float, 13, 0, false, 64>", "gather fp32, half links"),
    (r"dslash_kernel<float, 12, 1, false, 64>", "gather fp32 recon-12, xpay epilogue (apply_M)"),
    (r"dslash_pipe_kernel<float, 12, 0, false>", "TMA pipeline fp32 recon-12"),
    (r"dslash_pipe_kernel<double, 12, 0, false>", "TMA pipeline fp64 recon-12"),
    (r"dslash_lstage_kernel<float, 12, 0, false, 64>", "TMA-staged links fp32 recon-12"),
    (r"dslash_slab_kernel<float, 12, false", "slab boundary fp32 recon-12"),
    (r"face_project_kernel<float", "slab face projection fp32"),
    (r"cg_update_xr_kernel<float, float>", "CG x, r update fp32"),
    (r"heatbath_kernel", "SU(3) heatbath"),
)


def _demangle(names):
    out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout.splitlines()
    return dict(zip(names, out))


def table(lib=_build.LIB):
    res = subprocess.run([CUOBJDUMP, "--dump-resource-usage", lib], capture_output=True, text=True, check=True).stdout
    usage = {}
    for m in re.finditer(r"Function (\S+):\s*\n\s*REG:(\d+) STACK:(\d+) SHARED:(\d+) LOCAL:(\d+)", res):
        usage[m.group(1)] = tuple(int(x) for x in m.group(2, 3, 4, 5))
    sass = subprocess.run([CUOBJDUMP, "-sass", lib], capture_output=True, text=True, check=True).stdout
    counts, cur = {}, None
    for ln in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", ln)
        if m:
            cur = m.group(1)
            counts[cur] = dict.fromkeys(OPCODES, 0) | {"total": 0}
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", ln)
        if m and cur:
            op = m.group(1)
            counts[cur]["total"] += 1
            for o in OPCODES:
                base, _, width = o.partition(".")     # "LDG.256": any LDG whose modifiers include 256 (LDG.E.ENL2.256.CONSTANT)
                if op == base or op.startswith(base + "."):
                    if not width or width in op.split("."):
                        counts[cur][o] += 1
    dem = _demangle(list(counts))
    rows = []
    for pat, label in HOT:
        hits = [k for k, d in dem.items() if pat in d]
        if not hits:
            rows.append((label, None, None))
            continue
        k = hits[0]
        rows.append((label, usage.get(k), counts[k]))
    return rows


def main():
    rows = table()
    cols = ("total",) + OPCODES
    print("| kernel | regs | spill B | smem B | " + " | ".join(cols) + " |")
    print("|---|---|---|---|" + "---|" * len(cols))
    for label, use, cnt in rows:
        if cnt is None:
            print(f"| {label} | not in this build |")
            continue
        reg, stack, shared, local = use if use else ("?",) * 4
        print(f"| {label} | {reg} | {stack if stack == '?' else stack + local} | {shared} | " + " | ".join(str(cnt[c]) for c in cols) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
