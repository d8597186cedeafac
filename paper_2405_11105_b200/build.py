"""Builds liblcf.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2405_11105_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "liblcf.so"
SOURCES = ["lcf_plan.cu", "lcf_gram.cu", "lcf_gram_tc.cu", "lcf_gram_tc2.cu", "lcf_evd.cu", "lcf_evd_chol.cu", "lcf_evd_cluster.cu", "lcf_evd_top.cu", "lcf_project.cu", "lcf_project_tc.cu", "lcf_ncc.cu", "lcf_peaks.cu", "lcf_noalloc.cu"]
# no --use_fast_math: the EVD needs IEEE division and square roots
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + [CSRC / "lcf_internal.h", CSRC / "lcf_sm100.cuh", CSRC / "lcf_thresh.cuh", HERE.parent / "include" / "lcf.h", HERE.parent / "include" / "lcf_noalloc.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    objs = []
    procs = []
    for s in SOURCES:
        o = CSRC / (s[:-3] + ".o")
        cmd = [_nvcc(), *NVCC_FLAGS, "-c", str(CSRC / s), "-o", str(o)]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(str(o))
    for s, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out)
        if pr.returncode != 0:
            raise RuntimeError(f"nvcc failed on {s}")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run([_nvcc(), "-shared", "-o", str(tmp), *objs, "-Xcompiler", "-fPIC"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
