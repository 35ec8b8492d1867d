"""Build step: compiles csrc/metronome.cu into paper_2607_02640_b200/libmetronome.so for sm_100a.

nvcc cross-compiles without a GPU.  The .so is kept in-tree (git-ignored) so it travels to the GPU
box with the repo snapshot.  `python -m paper_2607_02640_b200.build` rebuilds it.
"""
from __future__ import annotations

import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libmetronome.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC"]


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  [os.path.join(os.path.dirname(_HERE), "include", "metronome.h")])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _sources())


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, os.path.join(CSRC, "metronome.cu")]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return LIB


CENSUS_OPS = ("UTCHMMA", "UTCBAR", "LDTM", "STTM", "UBLKCP", "SYNCS", "HMMA", "LDSM", "LDG", "STG", "MUFU.EX2", "FFMA2",
              "ATOMG", "REDG", "ACQBULK", "LDGDEPBAR", "F2FP.F16.E4M3", "PRMT")


def sass_census() -> dict:
    """Per kernel of libmetronome.so: how often each SASS mnemonic of interest occurs (cuobjdump -sass).
    UTCHMMA / LDTM / STTM = tcgen05.mma / tcgen05.ld / tcgen05.st, UBLKCP = cp.async.bulk, HMMA = mma.sync,
    LDSM = ldmatrix, SYNCS = mbarrier operations (B200_PROFILING.md)."""
    import re
    out = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    census, name = {}, None
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip().replace("(anonymous namespace)::", "").split("(")[0]
            name = name.replace("metronome::", "").replace("void ", "")
            census[name] = {"instructions": 0}
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and name:
            census[name]["instructions"] += 1
            op = m.group(1)
            for key in CENSUS_OPS:
                if op == key or op.startswith(key + "."):
                    census[name][key] = census[name].get(key, 0) + 1
    return census


if __name__ == "__main__":
    import sys
    if "--census" in sys.argv:
        build_library()
        c = sass_census()
        cols = [k for k in CENSUS_OPS if any(k in v for v in c.values())]
        print("| kernel | instructions | " + " | ".join(cols) + " |")
        print("|---|---|" + "---|" * len(cols))
        for name in sorted(c):
            print(f"| `{name}` | {c[name]['instructions']} | " + " | ".join(str(c[name].get(k, 0)) for k in cols) + " |")
    else:
        print(build_library(force=True, verbose=True))
