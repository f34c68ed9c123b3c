"""In-tree build of the CUDA library: csrc/*.cu -> paper_1909_04504_b200/libsph_b200.so for sm_100a.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
Usage: python -m paper_1909_04504_b200.build [--force] [--verbose] [--f32 | --f64]   (default: both libraries)
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
LIB_F64 = os.path.join(HERE, "libsph_b200_f64.so")      # the same sources with -DSPH_REAL_DOUBLE (sph_real = double)
EXTRA = os.environ.get("SPH_B200_NVCC_FLAGS", "").split()
OBJ = os.path.join(HERE, "build" if not os.environ.get("SPH_B200_LIB") else
                   "build_" + hashlib.sha256(LIB.encode()).hexdigest()[:8])
# (source, extra defines, object): sph_accel.cu is compiled once per smoothing kernel (its instantiations dominate
# the build time) and once as the dispatcher
SOURCES = [("sph_api.cu", [], "sph_api.o"), ("sph_nnps.cu", [], "sph_nnps.o"), ("sph_density.cu", [], "sph_density.o"), ("sph_search.cu", [], "sph_search.o"),
           ("sph_probe.cu", [], "sph_probe.o"), ("sph_static.cu", [], "sph_static.o"), ("sph_accel.cu", [], "sph_accel.o"),
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


def _digest(extra=()) -> str:
    h = hashlib.sha256()
    names = sorted(os.listdir(CSRC)) + ["../../include/sph.h"]
    for n in names:
        p = os.path.normpath(os.path.join(CSRC, n))
        if os.path.isfile(p):
            h.update(n.encode()); h.update(open(p, "rb").read())
    h.update(" ".join(ARCH + FLAGS + EXTRA + list(extra) + [repr(SOURCES)]).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False, precision: str = "f32") -> str:
    """precision "f32": libsph_b200.so (sph_real = float); "f64": libsph_b200_f64.so (-DSPH_REAL_DOUBLE)."""
    lib, objdir, extra = (LIB, OBJ, []) if precision == "f32" else (LIB_F64, OBJ + "_f64", ["-DSPH_REAL_DOUBLE"])
    return _build(lib, objdir, extra, force, verbose)


def _build(LIB: str, OBJ: str, extra, force: bool, verbose: bool) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "digest.txt")
    dig = _digest(extra)
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == dig:
        return LIB
    nvcc = _nvcc()

    def compile_one(item) -> str:
        src, defs, oname = item
        obj = os.path.join(OBJ, oname)
        cmd = [nvcc, *ARCH, *FLAGS, *EXTRA, *extra, *defs, "-I", INCLUDE, "-c", os.path.join(CSRC, src), "-o", obj]
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
    for prec in (("f64",) if "--f64" in sys.argv else ("f32",) if "--f32" in sys.argv else ("f32", "f64")):
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, precision=prec))
