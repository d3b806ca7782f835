"""Builds libtts_b200.so (the C-ABI library of include/tts.h) in-tree with nvcc for sm_100a.

    python -m paper_2605_09329_b200.build [--force]

nvcc cross-compiles without a GPU.  The library lands next to this file so that it travels with
the repo snapshot to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtts_b200.so")
SOURCES = ["tts_api.cu", "tts_mask.cu", "tts_accept.cu", "tts_stats.cu", "tts_simt.cu", "tts_tc.cu", "tts_tc_gemm.cu", "tts_tc_fused.cu", "tts_tc_wide.cu", "tts_tc_pair.cu"]
HEADERS = ["tts_internal.h", "tts_common.cuh", "tts_tc_ptx.cuh", "tts_tc_state.h", os.path.join("..", "..", "include", "tts.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.exists(p) and os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed (exit %d); see %s" % (r.returncode, log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
