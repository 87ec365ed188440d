"""Builds libpt.so (the C-ABI library of include/pt.h) in-tree with nvcc for sm_100a.

    python -m paper_1308_5426_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(_HERE, "libpt.so")
SOURCES = [os.path.join(CSRC, "pt_lib.cu")]
# No --use_fast_math: the acceptance thresholds and the swap test are fp64 and must not be relaxed (A8).
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "--fmad=false", "-Xcompiler", "-fPIC", "-shared", "-I", INCLUDE, "-I", CSRC]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    out = list(SOURCES) + [os.path.join(INCLUDE, "pt.h")]
    out += [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    return out


def build_variant(out_path, defines, verbose=False):
    """A development build of the same sources with extra -D flags (e.g. ["PT_PARANOID", "PT_ONLY_HEADLINE"]) at
    out_path; load it with PT_LIBPT=out_path."""
    cmd = [_nvcc()] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", out_path] + SOURCES
    subprocess.check_call(cmd)
    return out_path


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(p) for p in _deps()):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
