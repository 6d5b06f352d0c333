"""Build the C-ABI shared library libwz.so from csrc/ with nvcc for sm_100a.

    python -m paper_1005_3276_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  The kernels are instantiated in csrc/wz_kmod.cu, which is
compiled once per kernel module (-DWZ_MOD=n) so that the modules build in parallel; objects
are cached under csrc/build/ (git-ignored) and only stale ones are rebuilt.  The .so is
written next to this file (git-ignored too, but it travels to the GPU box with the repo
snapshot).
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJDIR = os.path.join(CSRC, "build")
LIB = os.path.join(_HERE, "libwz.so")
NUM_KERNEL_MODULES = 8  # kNumKernelModules in csrc/wz_tables.cuh
NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC",
]


def _units():
    """(object name, source, extra flags)"""
    u = [("wz_lib.o", "wz_lib.cu", [])]
    u += [("wz_kmod_%d.o" % i, "wz_kmod.cu", ["-DWZ_MOD=%d" % i]) for i in range(NUM_KERNEL_MODULES)]
    return u


def _deps_mtime() -> float:
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "wz.h"))
    deps.append(os.path.abspath(__file__))
    return max(os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libwz.so if missing or older than its sources; return its path."""
    newest = _deps_mtime()
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJDIR, exist_ok=True)

    def compile_one(unit):
        obj, src, extra = unit
        out = os.path.join(OBJDIR, obj)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
            return out, ""
        tmp = out + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", "-o", tmp, os.path.join(CSRC, src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s %s:\n%s" % (src, " ".join(extra), r.stderr[-8000:]))
        os.replace(tmp, out)
        return out, r.stderr

    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, _units()))
    if verbose:
        for out, log in results:
            if log:
                sys.stderr.write("==== %s\n%s" % (os.path.basename(out), log))
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] +
                          [o for o, _ in results])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
