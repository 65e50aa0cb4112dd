"""Build libpespace.so in-tree with nvcc for sm_100a (python -m paper_2602_12011_b200.build).

Every .cu under csrc/ is one translation unit; they are compiled in parallel to build/*.o and
linked into paper_2602_12011_b200/libpespace.so."""
import concurrent.futures as cf
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpespace.so")
SOURCES = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
DEPS = SOURCES + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + sorted(glob.glob(os.path.join(CSRC, "*.hpp"))) + \
    sorted(glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h")))

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v"] + os.environ.get("PESPACE_NVCC_EXTRA", "").split()


def csrc_hash() -> str:
    """sha256 over the names and contents of the CUDA sources and the public headers: the stamp that ties
    profiles/*_ops.json (ncu operation counts) to the kernels they were counted on (bench.py: roofline.stale)."""
    import hashlib
    h = hashlib.sha256()
    for path in sorted(DEPS):
        h.update(os.path.basename(path).encode())
        h.update(b"\0")
        h.update(open(path, "rb").read())
    return h.hexdigest()[:16]


def nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _compile(src: str, verbose: bool) -> str:
    obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
    newest = max(os.path.getmtime(p) for p in DEPS)
    if os.path.exists(obj) and os.path.getmtime(obj) >= newest:
        return obj
    res = subprocess.run([nvcc(), *NVCC_FLAGS, "-c", src, "-o", obj], capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed on {os.path.basename(src)}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    stale = not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(p) for p in DEPS)
    if force or stale:
        os.makedirs(OBJ, exist_ok=True)
        if force:
            for o in glob.glob(os.path.join(OBJ, "*.o")):
                os.unlink(o)
        with cf.ThreadPoolExecutor(max_workers=max(1, min(len(SOURCES), os.cpu_count() or 1))) as ex:
            objs = list(ex.map(lambda s: _compile(s, verbose), SOURCES))
        res = subprocess.run([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", LIB],
                             capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed linking libpespace.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
