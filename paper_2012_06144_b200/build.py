"""Builds paper_2012_06144_b200/libacm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The kernels are split over several translation units (one per kernel family and precision), which
are compiled in parallel to objects under build/ and linked into one shared library.
"""
import concurrent.futures
import glob
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libacm.so")
SOURCES = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
HEADERS = sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))) + \
    [os.path.join(os.path.dirname(HERE), "include", "acm.h")]

# fp64 parity with the oracle does not need contraction switched off, keep FMA
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def find_nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built")


def _compile(nvcc, src, extra):
    obj = os.path.join(OBJ, os.path.splitext(os.path.basename(src))[0] + ".o")
    cmd = [nvcc] + NVCC_FLAGS + list(extra) + ["-c", src, "-o", obj]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return obj, cmd, res


def build_lib(force: bool = False, verbose: bool = False, extra_flags=(), out: str = LIB) -> str:
    deps = SOURCES + HEADERS + [os.path.abspath(__file__)]
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps):
        return out
    nvcc = find_nvcc()
    os.makedirs(OBJ, exist_ok=True)
    log, objs = [], []
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        for obj, cmd, res in pool.map(lambda s: _compile(nvcc, s, extra_flags), SOURCES):
            log.append("$ " + " ".join(cmd) + "\n" + res.stdout + res.stderr)
            if res.returncode:
                print(log[-1])
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
            objs.append(obj)
    link = [nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", out]
    res = subprocess.run(link, capture_output=True, text=True)
    log.append("$ " + " ".join(link) + "\n" + res.stdout + res.stderr)
    if verbose or res.returncode:
        print("\n".join(log))
    if res.returncode:
        raise RuntimeError("link failed: " + " ".join(link))
    with open(os.path.join(HERE, "libacm.ptxas.log"), "w") as f:
        f.write("\n".join(log))
    return out


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
