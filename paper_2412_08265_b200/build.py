"""Builds the C-ABI library ``librubix_b200.so`` in-tree with nvcc for sm_100a.

    python -m paper_2412_08265_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  Every ``csrc/*.cu`` is compiled to an object file of its own (in
parallel, rebuilt only when it or a header changed) and the objects are linked into the shared library.
The library links cudart statically, so it loads on a machine with no CUDA driver (the
argument-validation paths work there; compute calls return RUBIX_ERR_CUDA).
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "librubix_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          "-Xcompiler", "-fPIC"]
LDFLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]
EXTRA = os.environ.get("RUBIX_NVCC_FLAGS", "").split()      # e.g. -DRUBIX_ACC_MINB=4 for a sweep


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h"))


def _obj(src):
    return os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")


def _compile(src, verbose):
    cmd = [NVCC] + CFLAGS + EXTRA + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", _obj(src), src]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return src, r.returncode, r.stdout


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdr_time = max(os.path.getmtime(h) for h in _headers())
    todo = [s for s in sources()
            if force or EXTRA or not os.path.exists(_obj(s))
            or os.path.getmtime(_obj(s)) < max(os.path.getmtime(s), hdr_time)]
    if todo:
        with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1)) as pool:
            for src, rc, out in pool.map(lambda s: _compile(s, verbose), todo):
                if out.strip():
                    print(out, file=sys.stderr)
                if rc != 0:
                    raise subprocess.CalledProcessError(rc, f"nvcc -c {src}")
    objs = [_obj(s) for s in sources()]
    if todo or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC] + LDFLAGS + ["-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
