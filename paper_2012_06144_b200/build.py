"""Builds paper_2012_06144_b200/libacm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libacm.so")
SOURCES = [os.path.join(CSRC, "acm.cu")]
HEADERS = [os.path.join(CSRC, "lattice.cuh"), os.path.join(os.path.dirname(HERE), "include", "acm.h")]

NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
              # fp64 parity with the oracle does not need contraction switched off, keep FMA
              "-Xptxas", "-v"]


def find_nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built")


def build_lib(force: bool = False, verbose: bool = False) -> str:
    deps = SOURCES + HEADERS + [os.path.abspath(__file__)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = [find_nvcc()] + NVCC_FLAGS + SOURCES + ["-o", LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode:
        print(res.stdout)
        print(res.stderr)
    if res.returncode:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    with open(os.path.join(HERE, "libacm.ptxas.log"), "w") as f:
        f.write(res.stderr)
    return LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
