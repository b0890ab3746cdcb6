"""Build csrc/ -> paper_2606_31580_b200/liblaser_probe.so with nvcc, for sm_100a only.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box in-tree.
Usage: python -m paper_2606_31580_b200.build [--force] [--verbose] [--timeline]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
SO = HERE / "liblaser_probe.so"
SOURCES = [CSRC / "laser_probe.cu", CSRC / "laser_sim.cu"]
DEPS = SOURCES + [CSRC / "probe_kernels.cuh", CSRC / "flex_kernel.cuh", CSRC / "ptx.cuh", HERE.parent / "include" / "laser_probe.h",
                  HERE.parent / "include" / "laser_sim.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",   # tcgen05 / TMEM need the 'a' target
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (cand == "nvcc" or Path(cand).exists()):
            return cand
    return "nvcc"


# Debug build with per-CTA %globaltimer stamps in the fused kernels (-DLASER_TIMELINE): never the shipped
# library; `bench.py --timeline` loads it through LASER_PROBE_LIB.
TIMELINE_SO = HERE / "liblaser_probe_timeline.so"


def build(force: bool = False, verbose: bool = False, timeline: bool = False) -> Path:
    SO = TIMELINE_SO if timeline else globals()["SO"]
    newest = max(p.stat().st_mtime for p in DEPS)
    if not force and SO.exists() and SO.stat().st_mtime >= newest:
        return SO
    tmp = SO.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc_path(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *(["-DLASER_TIMELINE"] if timeline else []),
           "-o", str(tmp), *map(str, SOURCES)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building liblaser_probe.so")
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, timeline="--timeline" in sys.argv))
