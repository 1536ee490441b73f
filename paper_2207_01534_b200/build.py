"""Builds paper_2207_01534_b200/liblbm_b200.so in-tree with nvcc for sm_100a.

    python -m paper_2207_01534_b200.build [--force] [--ptxas-v]

Three translation units: csrc/lbm.cu (C ABI + kernels, nvcc), csrc/geometry.cpp (host index
build, g++ through nvcc) and csrc/torch_shim.cpp (the only file that includes PyTorch headers:
caching allocator + current stream).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblbm_b200.so")
ROOT = os.path.dirname(HERE)
SOURCES = ["lbm.cu", "geometry.cpp", "torch_shim.cpp"]
DEPS = SOURCES + ["kernels.cuh", "geometry.hpp", os.path.join(ROOT, "include", "lbm.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for d in DEPS + [os.path.abspath(__file__)]:
        p = d if os.path.isabs(d) else os.path.join(CSRC, d)
        if os.path.getmtime(p) > t:
            return True
    return False


def build(force=False, verbose=False, ptxas_v=False):
    if not force and not _stale():
        return LIB
    import torch
    from torch.utils.cpp_extension import include_paths
    torch_lib = os.path.join(os.path.dirname(torch.__file__), "lib")
    abi = int(torch._C._GLIBCXX_USE_CXX11_ABI)
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    # NCCL: the header and library PyTorch bundles (the process already holds that libnccl.so.2
    # when this library is loaded), else the system's
    site = os.path.dirname(os.path.dirname(torch.__file__))
    nccl_inc = os.path.join(site, "nvidia", "nccl", "include")
    nccl_lib = os.path.join(site, "nvidia", "nccl", "lib")
    nccl_flags = ["-I", nccl_inc] if os.path.exists(os.path.join(nccl_inc, "nccl.h")) else []
    nccl_link = ([f"-L{nccl_lib}", "-l:libnccl.so.2", "-Xlinker", f"-rpath={nccl_lib}"]
                 if os.path.exists(os.path.join(nccl_lib, "libnccl.so.2")) else ["-lnccl"])
    common = ["-O3", "-std=c++17", "-Xcompiler", "-fPIC", f"-D_GLIBCXX_USE_CXX11_ABI={abi}"]
    objs = []

    def run(cmd):
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.check_call(cmd)

    o = os.path.join(objdir, "lbm.o")
    run([nvcc, "-c", os.path.join(CSRC, "lbm.cu"), "-o", o] + common + ARCH
        + nccl_flags + ["-lineinfo", "--expt-relaxed-constexpr"]
        + (["-Xptxas", "-v"] if ptxas_v else []))
    objs.append(o)
    o = os.path.join(objdir, "geometry.o")
    run(["g++", "-c", os.path.join(CSRC, "geometry.cpp"), "-o", o, "-O2", "-std=c++17", "-fPIC",
         "-fopenmp", f"-D_GLIBCXX_USE_CXX11_ABI={abi}"])
    objs.append(o)
    o = os.path.join(objdir, "torch_shim.o")
    inc = []
    for p in include_paths("cuda"):
        inc += ["-isystem", p]
    if os.path.isdir("/usr/local/cuda/include"):
        inc += ["-isystem", "/usr/local/cuda/include"]
    run(["g++", "-c", os.path.join(CSRC, "torch_shim.cpp"), "-o", o, "-O2", "-std=c++17", "-fPIC",
         f"-D_GLIBCXX_USE_CXX11_ABI={abi}"] + inc)
    objs.append(o)
    run([nvcc, "-shared", "-o", LIB] + objs + ARCH
        + ["-Xcompiler", "-fopenmp", f"-L{torch_lib}", "-lc10", "-lc10_cuda", "-lcudart",
           "-Xlinker", f"-rpath={torch_lib}"] + nccl_link)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, ptxas_v="--ptxas-v" in sys.argv))
