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


def _obj(src, objdir=OBJ):
    return os.path.join(objdir, os.path.basename(src)[:-3] + ".o")


def compile_command(src, extra=(), objdir=OBJ):
    return [NVCC, *ARCH, "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
            "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(PKG, "csrc"),
            *extra, "-c", src, "-o", _obj(src, objdir)]


def link_command(so=SO, objdir=OBJ):
    return [NVCC, *ARCH, "-shared", "-o", so, *[_obj(s, objdir) for s in sources()]]


# The instrumented library of tests/bounds_check.py: every staged shared-memory gather checks its
# address against the box it may read (csrc/dfr_tiled_device.cuh, DFR_BOUNDS_CHECK). Never loaded
# by the package itself.
SO_CHECKED = os.path.join(PKG, "libdfr_checked.so")


def build_checked(selftest: bool = False, verbose: bool = False) -> str:
    objdir = os.path.join(PKG, "csrc", "build_checked")
    os.makedirs(objdir, exist_ok=True)
    extra = ["-DDFR_BOUNDS_CHECK"] + (["-DDFR_BOUNDS_SELFTEST"] if selftest else [])
    with ThreadPoolExecutor(max_workers=8) as ex:
        list(ex.map(lambda s: _run(compile_command(s, extra, objdir), verbose), sources()))
    _run(link_command(SO_CHECKED, objdir), verbose)
    return SO_CHECKED


# The instruction-rate probes (csrc/probe/): a measurement tool, not part of libdfr or its ABI; its own
# library, loaded only by `bench.py --mode probes`.
SO_PROBE = os.path.join(PKG, "libdfr_probe.so")


def build_probe(force: bool = False, verbose: bool = False) -> str:
    srcs = sorted(glob.glob(os.path.join(PKG, "csrc", "probe", "*.cu")))
    if force or not os.path.exists(SO_PROBE) or os.path.getmtime(SO_PROBE) < max(os.path.getmtime(s) for s in srcs):
        _run([NVCC, *ARCH, "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-shared", "-o", SO_PROBE, *srcs], verbose)
    return SO_PROBE


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
    build_probe(force, verbose)
    return SO


if __name__ == "__main__":
    import sys
    if "--checked" in sys.argv:
        print(build_checked(selftest="--selftest" in sys.argv, verbose="-v" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
