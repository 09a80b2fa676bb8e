"""Build paper_2512_20927_b200/libqr.so (the C-ABI library of include/qr.h) in-tree with nvcc for sm_100a.

-fmad=false: the fp32 decision arithmetic (projection, alpha', transmittance, thresholds) must round exactly as
DESIGN.md states; every fused multiply-add in the kernels is written as an explicit fmaf intrinsic.
-lineinfo: ncu source pages map to the .cu files.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libqr.so")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"] + \
    (["-DQR_PROF"] if os.environ.get("QR_PROF") == "1" else []) + \
    (["-DQR_LAG=" + os.environ["QR_LAG"]] if os.environ.get("QR_LAG") else []) + \
    os.environ.get("QR_DEFS", "").split()       # QR_PROF: per-role wait counters in the blend kernel; QR_DEFS: extra -D flags for experiments


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + \
        [os.path.join(os.path.dirname(HERE), "include", "qr.h")]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: libqr.so cannot be built (there is no CPU fallback)")
    return p


def build(force: bool = False, verbose: bool = False) -> str:
    """One object per .cu (compiled in parallel, rebuilt only when the source or a header is newer), then one link."""
    if (not force) and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    headers = [d for d in _deps() if not d.endswith(".cu")]
    hdr_time = max(os.path.getmtime(h) for h in headers)
    nvcc = nvcc_path()
    cflags = [f for f in NVCC_FLAGS if f != "-shared"]
    jobs = []
    for src in sources():
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time):
            jobs.append([nvcc] + cflags + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src])
    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for r in ex.map(lambda c: subprocess.run(c), jobs):
            if r.returncode != 0:
                raise subprocess.CalledProcessError(r.returncode, r.args)
    objs = [os.path.join(objdir, os.path.basename(s)[:-3] + ".o") for s in sources()]
    subprocess.run([nvcc] + NVCC_FLAGS + ["-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
