"""Build the C-ABI shared library in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libcn_nshape.so")
SOURCES = ["cn_api.cu"]
HEADERS = ["cn_common.cuh", "cn_factor.cuh", "cn_pass_generic.cuh", "cn_pass_tiled.cuh", "cn_reduced.cuh",
           "cn_batched.cuh", "cn_onchip.cuh", "cn_shard.cuh", os.path.join("..", "..", "include", "cn_nshape.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--threads", "4", "-diag-suppress", "550"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for f in SOURCES + HEADERS:
        path = os.path.join(CSRC, f)
        if os.path.exists(path) and os.path.getmtime(path) > t:
            return True
    return False


def build_library(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [nvcc, *NVCC_FLAGS, "-o", tmp, *[os.path.join(CSRC, s) for s in SOURCES]]
        if verbose:
            cmd += ["-Xptxas", "-v"]
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


def sass_summary(match: str = "") -> str:
    """Markdown table of what is in the built library, per kernel (cuobjdump -sass / -res-usage): registers, stack
    (spills), static shared memory, and the counts of the SASS mnemonics that prove the design -- UTMALDG / UTMASTG
    (TMA tensor loads / stores), SYNCS (mbarrier), DFMA / DMUL / DADD (FP64 pipe), MUFU.RCP64H (divisions), SHFL
    (warp shuffles), LDS / STS, LDG / STG, BAR.  `match`: only kernels whose demangled name contains it."""
    import re
    lib = build_library()
    demangle = lambda names: subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout.split("\n")
    res, cur = {}, None
    for line in subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True).stdout.splitlines():
        m = re.match(r"\s*Function (\S+):", line)
        if m:
            cur = m.group(1)
        elif cur and "REG:" in line:
            res[cur] = dict(kv.split(":") for kv in line.split() if ":" in kv and "[" not in kv)
            cur = None
    keys = ["UTMALDG", "UTMASTG", "SYNCS", "DFMA", "DMUL", "DADD", "MUFU.RCP64H", "SHFL", "LDS", "STS", "LDG", "STG", "BAR"]
    counts, cur = {}, None
    for line in subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = m.group(1)
            counts[cur] = dict.fromkeys(keys + ["total"], 0)
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and cur:
            op = m.group(1)
            counts[cur]["total"] += 1
            for k in keys:
                if op == k or op.startswith(k + "."):
                    counts[cur][k] += 1
    names = sorted(counts)
    pretty = dict(zip(names, demangle(names)))
    rows = ["| kernel | REG | STACK | SHARED | instr | " + " | ".join(keys) + " |", "|---|" + "---:|" * (4 + len(keys))]
    for n in sorted(names, key=lambda x: pretty[x]):
        short = re.sub(r"\(.*", "", pretty[n])
        if match and match not in short:
            continue
        r, c = res.get(n, {}), counts[n]
        rows.append("| `%s` | %s | %s | %s | %d | " % (short, r.get("REG", "?"), r.get("STACK", "?"), r.get("SHARED", "?"), c["total"])
                    + " | ".join(str(c[k]) for k in keys) + " |")
    return "\n".join(rows)


if __name__ == "__main__":
    if "--sass-summary" in sys.argv:
        i = sys.argv.index("--sass-summary")
        print(sass_summary(sys.argv[i + 1] if i + 1 < len(sys.argv) else ""))
    else:
        print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
