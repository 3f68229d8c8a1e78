#!/usr/bin/env python
"""The -m gpu parity tests against the BOUNDS-CHECKED build of libdfr (not a test itself).

    python -m paper_2505_03932_b200.build --checked [--selftest]
    python tests/bounds_check.py [pytest -k expression]

compute-sanitizer is closed on the GPU pool, so the packed interior loops — which gather from the
TMA-staged box with no range test and no address guard, relying on the tile record's rigorous
index bound — are verified with an instrumented build instead: compiled with -DDFR_BOUNDS_CHECK,
every staged shared-memory load compares its address with the box the warp may read (the CTA's box
in tiled_reproject_kernel, the warp's own box in tiled_stack_kernel) and with 4-byte alignment,
counts violations and redirects the load. This script runs the parity and stack tests with that
library and prints the two counters; `--selftest` builds declare a 256-byte box instead, so the same
run must then report violations (the negative control of the checker)."""
import ctypes as C
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import pytest  # noqa: E402

import paper_2505_03932_b200 as P  # noqa: E402
from paper_2505_03932_b200 import build  # noqa: E402


def main():
    if not os.path.exists(build.SO_CHECKED):
        raise SystemExit("build it first: python -m paper_2505_03932_b200.build --checked")
    P._SO = build.SO_CHECKED                     # the package loads this file instead of libdfr.so
    L = P.lib()
    L.dfr_dev_oob_main.restype = C.c_ulonglong
    L.dfr_dev_oob_stack.restype = C.c_ulonglong
    expr = sys.argv[1] if len(sys.argv) > 1 else "not many_exposures and not two_devices"
    rc = pytest.main(["-q", "-m", "gpu", os.path.join(ROOT, "tests", "test_gpu_parity.py"),
                      os.path.join(ROOT, "tests", "test_gpu_stack.py"), "-k", expr])
    print(f"pytest exit code {int(rc)}; out-of-box staged loads: reproject kernels {L.dfr_dev_oob_main()}, "
          f"stack kernels {L.dfr_dev_oob_stack()}")


if __name__ == "__main__":
    main()
