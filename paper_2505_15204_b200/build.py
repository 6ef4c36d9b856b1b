"""Builds libblinkimg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libblinkimg.so")
SOURCES = ["blink_api.cu", "blink_grid.cu", "blink_fft2d.cu", "blink_fused.cu", "blink_fused_conv.cu", "blink_image.cu", "blink_avg.cu", "blink_fftg.cu", "blink_fused_g.cu", "blink_corr.cu", "blink_noalloc.cu"]
HEADERS = ["blink_common.cuh", "blink_fft.cuh", "blink_tma.cuh", "blink_fused_kernel.cuh", "blink_fftg.cuh", "blink_sort.cuh", os.path.join("..", "..", "include", "blinkimg.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v"]


def _stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    for f in SOURCES:
        o = os.path.join(bdir, f.replace(".cu", ".o"))
        objs.append(o)
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, f), "-o", o]
        procs.append((f, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    failed = False
    for f, p in procs:
        out, _ = p.communicate()
        log.append(f"== {f}\n{out}")
        failed |= p.returncode != 0
    text = "\n".join(log)
    with open(os.path.join(bdir, "ptxas.log"), "w") as fh:
        fh.write(text)
    if failed or verbose:
        print(text, file=sys.stderr)
    if failed:
        raise RuntimeError("nvcc failed; see output above")
    tmp = SO + f".{os.getpid()}.tmp"
    subprocess.check_call([nvcc, "-shared", "-o", tmp, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(SO)
