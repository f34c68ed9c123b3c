"""In-tree build of the CUDA library: csrc/*.cu -> paper_1909_04504_b200/libsph_b200.so for sm_100a.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
Usage: python -m paper_1909_04504_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
# SPH_B200_LIB / SPH_B200_NVCC_FLAGS: build (and load, see binding.py) a tuning variant beside the default library
LIB = os.environ.get("SPH_B200_LIB") or os.path.join(HERE, "libsph_b200.so")
EXTRA = os.environ.get("SPH_B200_NVCC_FLAGS", "").split()
OBJ = os.path.join(HERE, "build" if not os.environ.get("SPH_B200_LIB") else
                   "build_" + hashlib.sha256(LIB.encode()).hexdigest()[:8])
# (source, extra defines, object): sph_accel.cu is compiled once per smoothing kernel (its instantiations dominate
# the build time) and once as the dispatcher
SOURCES = [("sph_api.cu", [], "sph_api.o"), ("sph_nnps.cu", [], "sph_nnps.o"), ("sph_density.cu", [], "sph_density.o"), ("sph_search.cu", [], "sph_search.o"),
           ("sph_probe.cu", [], "sph_probe.o"), ("sph_accel.cu", [], "sph_accel.o"),
           ("sph_accel.cu", ["-DSPH_ACCEL_KERNEL=0"], "sph_accel_k0.o"),
           ("sph_accel.cu", ["-DSPH_ACCEL_KERNEL=1"], "sph_accel_k1.o"),
           ("sph_accel.cu", ["-DSPH_ACCEL_KERNEL=2"], "sph_accel_k2.o")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _nvcc() -> str:
    cand = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(cand):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")
    return cand


def _digest() -> str:
    h = hashlib.sha256()
    names = sorted(os.listdir(CSRC)) + ["../../include/sph.h"]
    for n in names:
        p = os.path.normpath(os.path.join(CSRC, n))
        if os.path.isfile(p):
            h.update(n.encode()); h.update(open(p, "rb").read())
    h.update(" ".join(ARCH + FLAGS + EXTRA + [repr(SOURCES)]).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "digest.txt")
    dig = _digest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == dig:
        return LIB
    nvcc = _nvcc()

    def compile_one(item) -> str:
        src, defs, oname = item
        obj = os.path.join(OBJ, oname)
        cmd = [nvcc, *ARCH, *FLAGS, *EXTRA, *defs, "-I", INCLUDE, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, *ARCH, "-shared", "-o", tmp, *objs, "-lcudart_static", "-lpthread", "-ldl", "-lrt"])
    os.replace(tmp, LIB)
    with open(stamp, "w") as f:
        f.write(dig)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
