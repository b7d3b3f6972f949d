"""In-tree build of libcos_b200.so (CUDA sm_100a + the host DAG compiler).

    python -m paper_2507_12349_b200.build [--force]

nvcc cross-compiles without a GPU.  The shared library stays next to this file (git-ignored, but it
travels to the GPU box with the repo snapshot).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcos_b200.so")
SOURCES = ["cos_capi.cu", "cos_kernels.cu", "cos_det.cu", "cos_compile.cpp"]
HEADERS = ["cos_compile.h", "cos_kernels.cuh", os.path.join("..", "..", "include", "cos.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-O3,-Wall", "-shared", "--cudart", "static",
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force=False, verbose=False, out=None, extra=()):
    """Builds libcos_b200.so in-tree; `out` / `extra` build a variant elsewhere (e.g. extra=["-DCOS_CHECK_BOUNDS"])."""
    lib = out or LIB
    if out is None and not force and not needs_build():
        return LIB
    tmp = lib + ".%d.tmp" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra) + os.environ.get("COS_NVCC_EXTRA", "").split() + \
          (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
