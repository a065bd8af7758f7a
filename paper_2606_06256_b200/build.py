"""Build libsegpa.so in-tree with nvcc for sm_100a (no torch extension machinery, plain C ABI)."""
from __future__ import annotations

import os
import shlex
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsegpa.so")
# test build (-DSEGPA_BRINGUP): adds the SIMT cross-check attention kernel; loaded only by tests that ask for it
BRINGUP_LIB = os.path.join(HERE, "libsegpa_bringup.so")
BRINGUP_SOURCES = ["segpa_host.cu", "segpa_misc_kernels.cu"]     # the files that look at SEGPA_BRINGUP
SOURCES = ["segpa_host.cu", "segpa_misc_kernels.cu", "segpa_attn_tc.cu", "segpa_attn_tc1.cu", "segpa_mass.cu"]
HEADERS = ["segpa_internal.h", "sm100_ptx.cuh", "segpa_attn_common.cuh", os.path.join("..", "..", "include", "segpa.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "--use_fast_math"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(BRINGUP_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(BRINGUP_LIB))
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _link(objs, lib):
    tmp = lib + ".tmp.%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-shared", "-o", tmp] + objs + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"])
    os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False) -> str:
    """libsegpa.so (the product) and libsegpa_bringup.so (test build: the two files that look at SEGPA_BRINGUP
    recompiled with it, the kernel objects shared).  Sources are compiled in parallel."""
    extra = shlex.split(os.environ.get("SEGPA_NVCC_EXTRA", ""))   # e.g. -DSEGPA_TRACE (pipeline trace hooks)
    if not force and not extra and not needs_build():
        return LIB
    jobs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        jobs.append((o, [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + extra + ["-c", os.path.join(CSRC, s), "-o", o]))
    for s in BRINGUP_SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".bringup.o"))
        jobs.append((o, [_nvcc()] + NVCC_FLAGS + extra + ["-DSEGPA_BRINGUP", "-c", os.path.join(CSRC, s), "-o", o]))
    procs = [(o, subprocess.Popen(cmd)) for o, cmd in jobs]
    bad = [o for o, p in procs if p.wait() != 0]
    if bad:
        raise RuntimeError("nvcc failed for " + ", ".join(os.path.basename(b) for b in bad))
    objs = [os.path.join(CSRC, s.replace(".cu", ".o")) for s in SOURCES]
    _link(objs, LIB)
    _link([os.path.join(CSRC, s.replace(".cu", ".bringup.o" if s in BRINGUP_SOURCES else ".o")) for s in SOURCES], BRINGUP_LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
