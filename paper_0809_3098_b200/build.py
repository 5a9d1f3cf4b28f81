"""Builds paper_0809_3098_b200/libcavity.so in-tree from csrc/*.cu with nvcc for sm_100a.

The library links against PyTorch's c10 / c10_cuda only (caching allocator and current stream); the
kernels are plain CUDA.  -fmad=false: every fused multiply-add in the kernels is an explicit fma(), so
the arithmetic is exactly the association DESIGN.md states.  -lineinfo keeps ncu's source page usable.

    python -m paper_0809_3098_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcavity.so")
SOURCES = ["cavity_kernels.cu", "cavity_resident.cu", "cavity_noalloc.cu", "cavity_api.cu"]
HEADERS = ["cavity_kernels.cuh", "cavity_resident.cuh", "cavity_scheme.cuh", os.path.join("..", "..", "include", "cavity.h"),
           os.path.join("..", "..", "include", "cavity_debug.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _torch_dirs():
    import torch
    root = os.path.dirname(os.path.abspath(torch.__file__))
    return os.path.join(root, "include"), os.path.join(root, "lib")


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    inc, lib = _torch_dirs()
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    common = [nvcc, "-std=c++17", "-O3", "-lineinfo", "-fmad=false", "-Xcompiler", "-fPIC,-fvisibility=hidden",
              "-D_GLIBCXX_USE_CXX11_ABI=1"] + ARCH
    if verbose:
        common += ["-Xptxas", "-v"]
    common += os.environ.get("CAV_NVCC_FLAGS", "").split()      # tuning experiments (e.g. -DCAV_RECV_BATCH=8)
    for s in SOURCES:
        o = os.path.join(CSRC, s[:-3] + ".o")
        cmd = common + ["-I", inc, "-c", os.path.join(CSRC, s), "-o", o]
        subprocess.run(cmd, check=True)
        objs.append(o)
    tmp = LIB + ".tmp.%d" % os.getpid()
    link = [nvcc, "-shared", "-o", tmp] + objs + ARCH + ["-L", lib, "-lc10", "-lc10_cuda", "-Xlinker",
                                                          "-rpath," + lib]
    subprocess.run(link, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
