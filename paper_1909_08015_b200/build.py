"""Build step: compiles csrc/ into paper_1909_08015_b200/libfg.so for sm_100a (nvcc cross-compiles without a GPU).

Usage: python -m paper_1909_08015_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfg.so")
SOURCES = ["fg_kernels.cu", "fg_plan.cpp", "fg_batch.cpp"]
DEPS = SOURCES + ["fg_core.cuh", "fg_stream.cuh", "fg_dd.cuh", "fg_qd.cuh", "fg_tables.h", "fg_plan.hpp", os.path.join("..", "..", "include", "fg.h")]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    return "nvcc"


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force=False, verbose=False, defines=(), out=None):
    """defines: extra -D macros (e.g. FG_PHASE_PROF for the per-phase cycle counters); out: library path (default LIB)."""
    out = out or LIB
    if not force and out == LIB and not needs_build():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-fopenmp,-ffp-contract=off,-O2", "-shared", "-o", out] + ["-D" + d for d in defines] + SOURCES
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, cwd=CSRC, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout[-4000:])
    return out


if __name__ == "__main__":
    defs = [a[2:] for a in sys.argv[1:] if a.startswith("-D")]
    outs = [a[6:] for a in sys.argv[1:] if a.startswith("--out=")]
    print(build(force="--force" in sys.argv or bool(defs) or bool(outs), verbose="--verbose" in sys.argv, defines=defs, out=outs[0] if outs else None))
