"""Build the CUDA library of the hot path: csrc/*.cu -> paper_2210_17509_b200/libgrx.so (sm_100a).

    python -m paper_2210_17509_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is built in-tree (git-ignored, but it travels to the GPU
box with the repo snapshot).  Objects are cached under build/ and rebuilt when a source or header is newer.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgrx.so")
OBJDIR = os.path.join(ROOT, "build", "grx")
SOURCES = ["grx_api.cu", "grx_simple.cu", "grx_fused.cu", "grx_tma.cu", "grx_ct.cu", "grx_vertex.cu", "grx_support.cu"]
# bench-side measurement probes: their own library, loaded by bench.py only (not part of the product ABI)
PROBE_LIB = os.path.join(HERE, "libgrx_probe.so")
PROBE_SRC = os.path.join(CSRC, "probe", "grx_probe.cu")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--fmad=true",
         "-Xcudafe", "--diag_suppress=177"]


def _newest_header():
    t = os.path.getmtime(os.path.join(ROOT, "include", "grx.h"))
    for f in os.listdir(CSRC):
        if f.endswith((".cuh", ".h")):
            t = max(t, os.path.getmtime(os.path.join(CSRC, f)))
    return t


def _compile(src, force, verbose):
    obj = os.path.join(OBJDIR, src.replace(".cu", ".o"))
    srcp = os.path.join(CSRC, src)
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(srcp), _newest_header()):
        return obj, ""
    cmd = [NVCC, *ARCH, *FLAGS, "-c", srcp, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    with open(obj + ".ptxas.txt", "w") as f:
        f.write(r.stderr)
    return obj, r.stderr if verbose else ""


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJDIR, exist_ok=True)
    with ThreadPoolExecutor(max_workers=4) as ex:
        res = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    objs = [o for o, _ in res]
    for _, log in res:
        if log:
            print(log)
    if force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        cmd = [NVCC, *ARCH, "-shared", "-o", LIB, *objs, "-cudart", "static"]
        subprocess.run(cmd, check=True)
    return LIB


def build_probe(force: bool = False) -> str:
    """csrc/probe/grx_probe.cu -> libgrx_probe.so (the FP64 micro-benchmarks of bench.py)."""
    hdr = os.path.join(CSRC, "probe", "grx_probe.h")
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < max(os.path.getmtime(PROBE_SRC),
                                                                                   os.path.getmtime(hdr)):
        cmd = [NVCC, *ARCH, "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", PROBE_LIB, PROBE_SRC,
               "-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for grx_probe.cu:\n%s\n%s" % (r.stdout, r.stderr))
    return PROBE_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_probe(force="--force" in sys.argv))
