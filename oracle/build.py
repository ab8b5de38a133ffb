"""Build oracle/liboracle.so (TEST INFRASTRUCTURE, see scape_oracle.cpp header).

g++ -O2 -std=c++17 -ffp-contract=off: the oracle writes every rounding out by hand
(std::fma where the pinned order says fma), so the compiler must not contract a*b+c.

ORACLE_SANITIZE=1 in the environment (or build(sanitize=True)) builds and loads
oracle/liboracle_san.so instead: the same source with -fsanitize=address,undefined
-fno-sanitize-recover=undefined (any undefined behaviour aborts), -O1 -g.  Loading it into Python
needs the ASan runtime first in the process: LD_PRELOAD=$(gcc -print-file-name=libasan.so); see
tests/test_oracle_sanitized.py, which runs the pins that way.  The CUDA side has no sanitizer on
this GPU pool (compute-sanitizer is closed), so this is the one sanitizer the project has.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "scape_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")
LIB_SAN = os.path.join(HERE, "liboracle_san.so")

BASE = ["g++", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def asan_runtime() -> str:
    """Path of the ASan runtime that has to be LD_PRELOADed before the sanitized oracle is loaded."""
    return subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()


def build(force: bool = False, sanitize=None) -> str:
    if sanitize is None:
        sanitize = os.environ.get("ORACLE_SANITIZE", "0") not in ("", "0")
    lib = LIB_SAN if sanitize else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    opt = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
           if sanitize else ["-O2"])
    cmd = BASE + opt + ["-o", lib + ".tmp", SRC]
    subprocess.check_call(cmd)
    os.replace(lib + ".tmp", lib)
    return lib


if __name__ == "__main__":
    print(build(force=True))
