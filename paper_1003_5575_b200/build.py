"""Build libgridder.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_1003_5575_b200.build [--force]

The shared library is git-ignored but travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libgridder.so"
CHECKED_LIB = HERE / "libgridder_checked.so"
SOURCES = ["api.cu", "bin.cu", "grid.cu", "presum.cu", "scatter.cu", "image.cu", "static_ws.cu"]
HEADERS = [CSRC / "gridder_internal.cuh", CSRC / "map.cuh", HERE.parent / "include" / "gridder.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Wno-deprecated-gpu-targets",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(d).stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> Path:
    """checked: the -DGRIDDER_CHECKED variant (index checks in every kernel, counted: gridder_check_violations),
    built beside the normal library as libgridder_checked.so."""
    objs = []
    procs = []
    lib = CHECKED_LIB if checked else LIB
    for src in SOURCES:
        s = CSRC / src
        o = CSRC / (src + (".chk.o" if checked else ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = ([_nvcc()] + NVCC_FLAGS + (["-DGRIDDER_CHECKED"] if checked else []) + (["-Xptxas", "-v"] if verbose else []) +
                   ["-c", str(s), "-o", str(o)])
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if force or procs or _stale(lib, objs):
        tmp = lib.with_suffix(f".{os.getpid()}.tmp")
        cmd = [_nvcc(), "-shared", "-Wno-deprecated-gpu-targets", "-o", str(tmp)] + [str(o) for o in objs] + ["-lcudart", "-ldl"]
        subprocess.check_call(cmd)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
