"""Build libsg.so in-tree: nvcc for sm_100a (kernels + C-ABI), g++ for the host generator and the
torch glue.  Used by __graft_entry__.build(); `python -m paper_1906_11195_b200.build` also works."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsg.so")
OBJ = os.path.join(HERE, "build")

CU = ["sg_kernels.cu", "sg_vb_sweep.cu", "sg_sk.cu", "sg_api.cu"]
CPP = ["sg_host.cpp", "sg_torch_glue.cpp"]


def _newest_source() -> float:
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "sg.h"), __file__]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    import torch
    from torch.utils import cpp_extension as ce

    os.makedirs(OBJ, exist_ok=True)
    cuda_home = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    nvcc = os.path.join(cuda_home, "bin", "nvcc")
    inc = ["-I" + os.path.join(ROOT, "include"), "-I" + CSRC]
    torch_inc = ["-I" + p for p in ce.include_paths()] + ["-I" + os.path.join(cuda_home, "include")]
    torch_lib = os.path.join(os.path.dirname(torch.__file__), "lib")
    abi = "-D_GLIBCXX_USE_CXX11_ABI=%d" % int(torch._C._GLIBCXX_USE_CXX11_ABI)
    objs = []
    for f in CU:
        o = os.path.join(OBJ, f + ".o")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
               "-Xcompiler", "-fPIC,-Wall", abi, "-c", os.path.join(CSRC, f), "-o", o] + inc
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        cmd += os.environ.get("SG_NVCC_FLAGS", "").split()      # e.g. -DSG_BT=128 (experiments)
        subprocess.check_call(cmd)
        objs.append(o)
    for f in CPP:
        o = os.path.join(OBJ, f + ".o")
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-Wall", abi, "-c", os.path.join(CSRC, f), "-o", o] + inc
        if f == "sg_torch_glue.cpp":
            cmd += torch_inc
        subprocess.check_call(cmd)
        objs.append(o)
    cmd = [nvcc, "-shared", "-o", LIB] + objs + [
        "-L" + torch_lib, "-lc10", "-lc10_cuda", "-Xlinker", "-rpath," + torch_lib, "-cudart", "static"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
