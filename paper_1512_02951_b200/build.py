"""Build libfeds.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

`python -m paper_1512_02951_b200.build` or `build()`; nvcc cross-compiles without a GPU. The .so is git-ignored
but travels to the GPU box with the gpurun snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("FEDS_LIB_PATH") or os.path.join(HERE, "libfeds.so")
SOURCES = ["feds_api.cu"]
HEADERS = ["feds_device.cuh", "feds_dct.cuh", "feds_dct_tile.cuh", "feds_hash.cuh", "feds_dwt.cuh", "feds_dwt_fast.cuh", "feds_peaks.cu", os.path.join("..", "..", "include", "feds.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
    "--expt-relaxed-constexpr",
    "-cudart", "shared",
    "-Xlinker", "-rpath=/usr/local/cuda/lib64",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    files = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(f) > t for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + ".tmp.%d" % os.getpid()
    extra = os.environ.get("FEDS_NVCC_EXTRA", "").split()
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed (see %s)" % log)
    if verbose:
        sys.stderr.write(res.stderr)
    os.replace(tmp, LIB)
    build_peaks(nvcc)
    return LIB


PEAKS = os.path.join(HERE, "feds_peaks")


def build_peaks(nvcc=None) -> str:
    """The small stand-alone tool that measures this GPU's SHA-256 integer ceiling (bench.py's ALU-roofline context)."""
    nvcc = nvcc or os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "--expt-relaxed-constexpr",
           "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64", "-o", PEAKS, os.path.join(CSRC, "feds_peaks.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed on feds_peaks.cu")
    return PEAKS


if __name__ == "__main__":
    print(build(force=True, verbose=True))
