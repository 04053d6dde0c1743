"""Build libnmf_b200.so (sm_100a) in-tree with nvcc.

    python -m paper_2309_04623_b200.build [--force]

The library is plain CUDA C++ behind the C-ABI of include/nmf.h; it links only
the CUDA runtime (statically) and the driver API loader.  nvcc cross-compiles
for sm_100a on a box without a GPU.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnmf_b200.so")
SOURCES = ["nmf_api.cu", "nmf_generic.cu", "nmf_fused.cu", "nmf_tcfit.cu", "nmf_tcsplit.cu", "nmf_stream.cu", "nmf_resident.cu", "nmf_aux.cu", "nmf_select.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _deps():
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdrs.append(os.path.join(HERE, "..", "include", "nmf.h"))
    return max(os.path.getmtime(h) for h in hdrs)


def _compile(src: str, force: bool, verbose: bool, extra=(), suffix: str = "") -> str:
    obj = os.path.join(OBJ, src.replace(".cu", suffix + ".o"))
    srcp = os.path.join(CSRC, src)
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(srcp), _deps()):
        return obj
    cmd = ["nvcc", *NVCC_FLAGS, *extra, "-c", srcp, "-o", obj]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode:
        raise RuntimeError(f"nvcc failed on {src}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        tmp = f"{LIB}.{os.getpid()}.tmp"
        subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a",
                               "-o", tmp, *objs, "-cudart", "static", "-lcuda"])
        os.replace(tmp, LIB)
    return LIB


def build_trace() -> str:
    """build/libnmf_trace.so: the same library with the timeline instrumentation of the split tensor-core kernels
    compiled in (-DNMF_TC_TRACE; exports nmf_debug_trace).  Used by `python bench.py --trace` only."""
    os.makedirs(OBJ, exist_ok=True)
    lib = os.path.join(OBJ, "libnmf_trace.so")
    with cf.ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(lambda s: _compile(s, False, False, ("-DNMF_TC_TRACE",), ".trace"), SOURCES))
    if not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(o) for o in objs):
        subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a",
                               "-o", lib, *objs, "-cudart", "static", "-lcuda"])
    return lib


def build_wait_debug() -> str:
    """build/libnmf_waitdebug.so: the same library with -DNMF_WAIT_DEBUG: an mbarrier wait that times out is logged
    (nmf_debug_wait_log) and abandoned instead of trapping.  A debugging aid for protocol errors; not used by the
    product, the tests or bench.py."""
    os.makedirs(OBJ, exist_ok=True)
    lib = os.path.join(OBJ, "libnmf_waitdebug.so")
    with cf.ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(lambda s: _compile(s, False, False, ("-DNMF_WAIT_DEBUG",), ".waitdebug"), SOURCES))
    if not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(o) for o in objs):
        subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a",
                               "-o", lib, *objs, "-cudart", "static", "-lcuda"])
    return lib


if __name__ == "__main__":
    if "--wait-debug" in sys.argv:
        print(build_wait_debug())
    elif "--trace" in sys.argv:
        print(build_trace())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
