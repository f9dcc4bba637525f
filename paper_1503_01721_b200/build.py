"""Build libvmat.so (the product) and libvmat_probe.so (a measurement aid of bench.py, csrc/probe/) in-tree with nvcc
for sm_100a (B200).  `python -m paper_1503_01721_b200.build`."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvmat.so")
PROBE_LIB = os.path.join(HERE, "libvmat_probe.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def probe_sources():
    return sorted(glob.glob(os.path.join(CSRC, "probe", "*.cu")))


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PROBE_LIB))
    inc = os.path.join(os.path.dirname(HERE), "include")
    deps = sources() + probe_sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        [os.path.join(inc, "vmat.h"), os.path.join(inc, "vmat_probe.h")]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D... flags (the tuning constants of csrc/common.cuh, e.g. -DVMAT_PRICE_MINB=5, and
    -DVMAT_CHECKED: device-side asserts on every stream access and gathered index of the layout-walking kernels, see
    MatView in csrc/common.cuh); a build with any of them replaces libvmat.so until the next plain build."""
    if not force and not defines and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc] + NVCC_FLAGS + list(defines) + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + sources()
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    tmp = PROBE_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc] + NVCC_FLAGS + ["-o", tmp] + probe_sources())
    os.replace(tmp, PROBE_LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
