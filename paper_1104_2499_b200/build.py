"""Build the C-ABI library (include/abm.h) for sm_100a, in-tree.

    python -m paper_1104_2499_b200.build            # -> paper_1104_2499_b200/libabm_b200.so

nvcc cross-compiles without a GPU.  The CUDA runtime is linked statically so the library also
loads (for symbol checks) on a box with no driver.
"""
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libabm_b200.so")
SOURCES = [os.path.join(CSRC, "abm.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "abm_device.cuh"), os.path.join(CSRC, "abm_kernels.cuh"),
                  os.path.join(ROOT, "include", "abm.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "-shared", "-cudart", "static",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(map(os.path.getmtime, DEPS)):
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


PIPE_RATES_SRC = os.path.join(CSRC, "pipe_rates.cu")
PIPE_RATES_EXE = os.path.join(PKG, "pipe_rates")


def build_pipe_rates(force: bool = False) -> str:
    """The stand-alone issue-rate diagnostic (csrc/pipe_rates.cu): not needed by the library."""
    if not force and os.path.exists(PIPE_RATES_EXE) and \
            os.path.getmtime(PIPE_RATES_EXE) >= max(os.path.getmtime(PIPE_RATES_SRC),
                                                    os.path.getmtime(os.path.join(CSRC, "abm_device.cuh"))):
        return PIPE_RATES_EXE
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-I", CSRC,
           "-o", PIPE_RATES_EXE, PIPE_RATES_SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return PIPE_RATES_EXE


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
    if "--pipe-rates" in sys.argv:
        print(build_pipe_rates(force=True))
