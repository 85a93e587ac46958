"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liboracle.so with gcc.

Flags follow SURVEY.md 8(c-3): -O2, no FMA contraction, no fast-math; OpenMP only
parallelises independent cells of a pass.

ORACLE_SANITIZE=1 builds oracle/liboracle_san.so with -fsanitize=address,undefined instead;
the sanitizer runtimes must then be preloaded into the Python process:

    ORACLE_SANITIZE=1 ASAN_OPTIONS=detect_leaks=0 LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" \
        python -m pytest tests -m "not gpu" -q
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "acm_oracle.c")
SANITIZE = os.environ.get("ORACLE_SANITIZE") == "1"
LIB = os.path.join(HERE, "liboracle_san.so" if SANITIZE else "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(os.path.abspath(__file__)))):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-Wall", "-Wextra", "-shared", "-fPIC"]
    if SANITIZE:
        cmd += ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
    cmd += [SRC, "-o", LIB, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
