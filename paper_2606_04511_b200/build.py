"""Build libsparda.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsparda.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr", "-shared", "-cudart", "shared"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "sparda.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_trace(out: str) -> str:
    """Debug build with device-side timelines (-DSPARDA_TRACE): per-CTA cycle / globaltimer stamps in the select, attention,
    prefill-select and tcgen05-attention kernels, read back through the sparda_debug_set_*_trace / _log hooks that only this
    build exports.  Never the product: written to `out`, not to libsparda.so."""
    res = subprocess.run([NVCC, *FLAGS, "-DSPARDA_TRACE", "-o", out, *sources()], capture_output=True, text=True)
    if res.returncode:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building the trace library")
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        cmd = [NVCC, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB, *sources()]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode:
            raise RuntimeError("nvcc failed building libsparda.so")
    return LIB


if __name__ == "__main__":
    if "--trace" in sys.argv:       # python -m paper_2606_04511_b200.build --trace /path/to/libsparda_trace.so
        print(build_trace(sys.argv[sys.argv.index("--trace") + 1]))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
