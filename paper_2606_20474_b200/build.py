"""Builds libuq.so (the C-ABI CUDA library, include/uq.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libuq.so")
SOURCES = ["uq_api.cu", "uq_append.cu", "uq_calib.cu", "uq_debug.cu", "uq_decode.cu", "uq_decode_cmp.cu", "uq_decode_prefix.cu", "uq_decode_prefix_m.cu", "uq_decode_static.cu", "uq_merge.cu", "uq_tq_append.cu"]
PTXAS_FLAGS = {"uq_decode.cu": ["-Xptxas", "-O1"], "uq_decode_cmp.cu": ["-Xptxas", "-O1"], "uq_decode_prefix_m.cu": ["-Xptxas", "-O3"], "uq_merge.cu": ["-Xptxas", "-O1"]}


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "uq.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    extra = os.environ.get("UQ_NVCC_EXTRA", "").split()      # experiments only (e.g. -DUQ_KSTAGES=2)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    # ptxas -O1 for the decode kernel only: measured, not assumed — it is bound by the serial instruction streams of
    # twelve warps sharing four schedulers, and the -O3 schedule of the same SASS-level work is 2 % slower on config 2
    # (104.7 us against 102.6 us).  The append kernels are long straight-line arithmetic and want the -O3 scheduler.
    common = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"] + (["-Xptxas", "-v"] if verbose else [])
    objs = []
    for src in SOURCES:
        obj = os.path.join(HERE, src.replace(".cu", ".o"))
        flags = PTXAS_FLAGS.get(src, [])
        if os.environ.get("UQ_PTXAS_O") and flags:
            flags = ["-Xptxas", "-O" + os.environ["UQ_PTXAS_O"]]
        cmd = common + flags + extra + ["-c", "-o", obj, os.path.join(CSRC, src)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed compiling {src}")
        objs.append(obj)
    res = subprocess.run([nvcc, "-shared", "-o", LIB] + objs, capture_output=True, text=True)
    for obj in objs:
        os.remove(obj)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libuq.so")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
