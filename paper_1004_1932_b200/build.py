"""Compile the CUDA library (csrc/ds_api.cu -> libds.so) for sm_100a with nvcc, in-tree.

nvcc cross-compiles without a GPU, so this runs on the CPU build box as well as on the B200 box.
The built .so is git-ignored but travels with the working tree.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libds.so")
SOURCES = ["ds_api.cu"]
HEADERS = ["pack.cuh", "noise.cuh", "averaged.cuh", "mobility.cuh", "pipeline.cuh", "small.cuh", "cluster.cuh", "state.cuh", "peak.cuh",
           os.path.join("..", "..", "include", "ds.h"), os.path.join("..", "..", "include", "ds_dev.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--shared", "-Xcompiler", "-fPIC"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    probe = ["-DDS_ENABLE_PROBE"] if os.environ.get("DS_ENABLE_PROBE") else []   # clock64 stage probes (development)
    cmd = [_nvcc()] + NVCC_FLAGS + probe + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
          [os.path.join(CSRC, f) for f in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
