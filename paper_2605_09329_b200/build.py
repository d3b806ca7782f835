"""Builds libtts_b200.so (the C-ABI library of include/tts.h) in-tree with nvcc for sm_100a.

    python -m paper_2605_09329_b200.build [--force]

nvcc cross-compiles without a GPU.  Every translation unit is compiled to an object under build/ (in parallel,
only the stale ones) and the objects are linked into the library next to this file, so that it travels with the
repo snapshot to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libtts_b200.so")
SOURCES = ["tts_api.cu", "tts_mask.cu", "tts_static.cu", "tts_accept.cu", "tts_stats.cu", "tts_simt.cu", "tts_check.cu",
           "tts_tc.cu", "tts_tc_gemm.cu", "tts_tc_fused.cu", "tts_tc_wide.cu", "tts_tc_pair.cu"]
HEADERS = ["tts_internal.h", "tts_common.cuh", "tts_tc_ptx.cuh", "tts_tc_state.h", "tts_adam.cuh", "tts_tc_epi.cuh",
           os.path.join("..", "..", "include", "tts.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-Xptxas", "-v"] + os.environ.get("TTS_NVCC_EXTRA", "").split()   # build-time only (e.g. -DTTS_MBAR_UNBOUNDED)


def _mtime(p: str) -> float:
    return os.path.getmtime(p) if os.path.exists(p) else 0.0


def _compile(nvcc: str, src: str, obj: str):
    cmd = [nvcc] + NVCC_FLAGS + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return cmd, r


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    hdr_t = max(_mtime(os.path.join(CSRC, h)) for h in HEADERS)
    hdr_t = max(hdr_t, _mtime(os.path.abspath(__file__)))
    jobs = []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s[:-3] + ".o")
        if force or _mtime(obj) < max(_mtime(src), hdr_t):
            jobs.append((src, obj))
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in SOURCES]
    if not jobs and os.path.exists(LIB) and _mtime(LIB) >= max(_mtime(o) for o in objs):
        return LIB
    log_lines, failed = [], False
    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for cmd, r in ex.map(lambda j: _compile(nvcc, *j), jobs):
            log_lines.append(" ".join(cmd) + "\n" + r.stdout)
            if r.returncode != 0:
                failed = True
    if not failed:
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        log_lines.append(" ".join(cmd) + "\n" + r.stdout)
        failed = r.returncode != 0
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write("\n".join(log_lines))
    if verbose or failed:
        sys.stderr.write("\n".join(log_lines))
    if failed:
        raise RuntimeError("nvcc failed; see %s" % log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
