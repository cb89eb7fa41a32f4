"""Builds libajt.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["ajt_api.cu", "ajt_loss.cu", "ajt_merge.cu", "ajt_blocks.cu", "ajt_pack.cu", "ajt_lmhead.cu"]
HEADERS = ["ajt_common.cuh", "ajt_token.cuh", os.path.join("..", "..", "include", "ajt.h"), os.path.join("..", "..", "include", "ajt_test.h")]
LIB = os.path.join(HERE, "libajt.so")

NVCC_FLAGS = ["-Wno-deprecated-gpu-targets", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(o)
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [nvcc, "-shared", "--cudart", "static", "-o", LIB] + objs
    subprocess.check_call(cmd)
    return LIB


SASS_MNEMONICS = ["UTCHMMA", "UTCBAR", "LDTM", "UTMALDG", "UBLKCP", "SYNCS", "UCGABAR", "ELECT", "FENCE", "REDUX", "MATCH", "MUFU.EX2",
                  "IMAD.WIDE", "LDG.E.128", "STG.E.128", "LDS.128", "STS.128", "ATOMG", "ATOMS", "BAR.SYNC", "HMMA", "LDL", "STL"]


def sass_census() -> str:
    """Per-kernel count of the SASS mnemonics that show which hardware path a kernel uses (`cuobjdump -sass libajt.so`):
    UTCHMMA / UTCBAR / LDTM = tcgen05.mma / commit / ld (TMEM), UTMALDG = TMA tensor load, UBLKCP = 1-D bulk async copy,
    SYNCS = mbarrier, UCGABAR = cluster barrier, REDUX = warp reduce, MUFU.EX2 = exp2, LDL / STL = local-memory traffic
    (spills or indexed register arrays).  Returns a markdown table."""
    import collections
    import re

    build()
    cuobjdump = os.path.join(os.path.dirname(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")), "cuobjdump")
    text = subprocess.run([cuobjdump, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    per, cur = collections.OrderedDict(), None
    for line in text.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = per.setdefault(m.group(1), collections.Counter())
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\w+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m and cur is not None:
            cur["instructions"] += 1
            for p in SASS_MNEMONICS:
                if m.group(1).startswith(p):
                    cur[p] += 1
    names = subprocess.run(["c++filt"], input="\n".join(per), capture_output=True, text=True).stdout.splitlines()
    cols = ["instructions"] + [p for p in SASS_MNEMONICS if any(c[p] for c in per.values())]
    out = ["| kernel | " + " | ".join(cols) + " |", "|---|" + "---:|" * len(cols)]
    for (_, c), n in zip(per.items(), names):
        n = re.sub(r"\(anonymous namespace\)::", "", n)
        n = re.sub(r"\(.*", "", n).replace("void ", "")
        out.append(f"| `{n}` | " + " | ".join(str(c[k]) if c[k] else "" for k in cols) + " |")
    return "\n".join(out)


if __name__ == "__main__":
    if "--sass-census" in sys.argv:
        print(sass_census())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
