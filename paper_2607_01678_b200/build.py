"""Build paper_2607_01678_b200/libscape.so in-tree with nvcc for sm_100a (B200).

nvcc cross-compiles without a GPU.  Flags: -gencode arch=compute_100a,code=sm_100a -lineinfo
(so ncu's source page maps to csrc/), IEEE defaults (no --use_fast_math: -prec-div, -prec-sqrt,
-ftz=false are what the pinned fp32 operation order relies on).

The streaming kernels are templates over (gradient type, R, mask / moment variant, clip_grad);
csrc/scape_fused_inst.cu is compiled once per (gradient type, range of R) and csrc/scape.cu holds
the host side and every other kernel, so the translation units build in parallel.  Objects go to
paper_2607_01678_b200/build/ (git-ignored); `ptxas_info.txt` collects registers / spills per kernel.
"""
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libscape.so")
DEPS = [os.path.join(CSRC, f) for f in ("scape.cu", "scape_fused_inst.cu", "scape_kernels.cuh", "scape_select_kernels.cuh")] + \
       [os.path.join(os.path.dirname(HERE), "include", "scape.h"), os.path.abspath(__file__)]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

# (object name, source, extra defines): tag, gradient type and range of R of every instantiation unit
UNITS = [("scape", "scape.cu", [])] + [
    (f"fused_{tag}", "scape_fused_inst.cu",
     [f"-DSCAPE_INST_TAG={tag}", f"-DSCAPE_INST_BF16={bf16}", f"-DSCAPE_INST_RLO={lo}", f"-DSCAPE_INST_RHI={hi}"])
    for tag, bf16, lo, hi in (("f32_lo", 0, 1, 4), ("f32_hi", 0, 5, 8), ("bf16_lo", 1, 1, 4), ("bf16_hi", 1, 5, 8))
]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def _compile(nvcc, name, src, defs):
    obj = os.path.join(OBJ, name + ".o")
    cmd = [nvcc] + NVCC_FLAGS + defs + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed ({name}):\n" + res.stdout + res.stderr)
    return obj, " ".join(cmd) + "\n" + res.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
        done = list(ex.map(lambda u: _compile(nvcc, *u), UNITS))
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-o", LIB + ".tmp"] + [o for o, _ in done]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    os.replace(LIB + ".tmp", LIB)
    log = "\n".join(l for _, l in done)
    if verbose:
        print(log)
    with open(os.path.join(HERE, "ptxas_info.txt"), "w") as f:
        f.write(log)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
