"""Compile libdfr.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Each csrc/*.cu is compiled to an object under csrc/build/ (in parallel, only when it or a
header changed), then linked into libdfr.so next to this file."""
from __future__ import annotations

import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
SO = os.path.join(PKG, "libdfr.so")
OBJ = os.path.join(PKG, "csrc", "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def sources():
    return sorted(glob.glob(os.path.join(PKG, "csrc", "*.cu")))


def _headers():
    return (glob.glob(os.path.join(PKG, "csrc", "*.h")) + glob.glob(os.path.join(PKG, "csrc", "*.cuh"))
            + [os.path.join(ROOT, "include", "dfr.h")])


def _obj(src):
    return os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")


def compile_command(src, extra=()):
    return [NVCC, *ARCH, "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
            "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(PKG, "csrc"),
            *extra, "-c", src, "-o", _obj(src)]


def link_command():
    return [NVCC, *ARCH, "-shared", "-o", SO, *[_obj(s) for s in sources()]]


def _run(cmd, verbose):
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdr = max(os.path.getmtime(h) for h in _headers())
    stale = [s for s in sources()
             if force or not os.path.exists(_obj(s)) or os.path.getmtime(_obj(s)) < max(os.path.getmtime(s), hdr)]
    extra = ("-Xptxas", "-v") if verbose else ()
    with ThreadPoolExecutor(max_workers=min(8, max(1, len(stale)))) as ex:
        list(ex.map(lambda s: _run(compile_command(s, extra), verbose), stale))
    objs = [_obj(s) for s in sources()]
    for stray in set(glob.glob(os.path.join(OBJ, "*.o"))) - set(objs):
        os.remove(stray)
    if stale or not os.path.exists(SO) or os.path.getmtime(SO) < max(os.path.getmtime(o) for o in objs):
        _run(link_command(), verbose)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
