"""Build libfeds.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

`python -m paper_1512_02951_b200.build` or `build()`; nvcc cross-compiles without a GPU. One object per kernel family,
compiled in parallel, then linked. The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.environ.get("FEDS_LIB_PATH") or os.path.join(HERE, "libfeds.so")
SOURCES = ["feds_api.cu", "feds_k_hash.cu", "feds_k_dct_tile.cu", "feds_k_dct_tma.cu", "feds_k_dct_fused.cu", "feds_k_dwt.cu", "feds_k_dct_strong.cu", "feds_k_dwt_tiles.cu", "feds_k_static.cu"]
SOURCES = [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + [
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off",
    "-Xptxas", "-v",
    "--expt-relaxed-constexpr",
]
LINK_FLAGS = ARCH + ["--shared", "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


def _deps():
    hdr = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdr += [os.path.join(ROOT, "include", f) for f in os.listdir(os.path.join(ROOT, "include"))]
    return hdr + [os.path.abspath(__file__)]


def _newer(path, deps):
    if not os.path.exists(path):
        return True
    t = os.path.getmtime(path)
    return any(os.path.getmtime(f) > t for f in deps)


def _compile(nvcc, src, extra, log):
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log.append(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed on %s:\n%s" % (src, res.stdout + res.stderr))
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    deps = _deps()
    os.makedirs(OBJ, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("FEDS_NVCC_EXTRA", "").split()
    todo = [s for s in SOURCES if force or _newer(os.path.join(OBJ, os.path.splitext(s)[0] + ".o"), deps + [os.path.join(CSRC, s)])]
    objs = [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in SOURCES]
    if not todo and not _newer(LIB, objs):
        return LIB
    log = []
    try:
        with ThreadPoolExecutor(max_workers=min(8, max(1, len(todo)))) as ex:
            list(ex.map(lambda s: _compile(nvcc, s, extra, log), todo))
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + LINK_FLAGS + ["-o", tmp] + objs
        res = subprocess.run(cmd, capture_output=True, text=True)
        log.append(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
        os.replace(tmp, LIB)
    finally:
        with open(os.path.join(HERE, "build.log"), "w") as f:
            f.write("\n".join(log))
    if verbose:
        sys.stderr.write("\n".join(log))
    return LIB


PEAKS = os.path.join(HERE, "feds_peaks")


def build_peaks(nvcc=None) -> str:
    """bench/feds_peaks.cu: the stand-alone tool that measures this GPU's SHA-256 integer ceiling (bench.py's ALU-roofline
    context; not part of the library)."""
    nvcc = nvcc or os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    src = os.path.join(ROOT, "bench", "feds_peaks.cu")
    if not _newer(PEAKS, [src, os.path.join(CSRC, "feds_device.cuh")]):
        return PEAKS
    cmd = [nvcc] + ARCH + ["-O3", "-std=c++17", "-lineinfo", "--expt-relaxed-constexpr", "-I", CSRC,
                           "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64", "-o", PEAKS, src]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed on feds_peaks.cu")
    return PEAKS


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
    print(build_peaks())
