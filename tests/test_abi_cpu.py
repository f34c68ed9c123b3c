"""CPU-side checks of the boundary (no compute calls): the C-ABI library builds for sm_100a, loads, and exports
every symbol include/sph.h declares; the ctypes structs match the C layout; the product fails loudly without a
GPU (no CPU fallback); oracle and product do not import one another."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sph.h")


@pytest.fixture(scope="module", params=["f32", "f64"])
def lib(request):
    """libsph_b200.so (sph_real = float) and libsph_b200_f64.so (the same sources with -DSPH_REAL_DOUBLE)"""
    from paper_1909_04504_b200 import build, binding
    build.build(precision=request.param)
    L = binding.load(request.param)
    assert L.sph_real_size() == (4 if request.param == "f32" else 8)
    return L


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_1909_04504_b200 import binding
    names = _declared()
    assert {"sph_nnps_build", "sph_summation_density", "sph_wcsph_accel", "sph_pc_step"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sph.h but not exported"
    assert sorted(binding.EXPORTS) == names
    assert lib.sph_abi_version() == 5


def test_struct_layouts_match_the_c_compiler(tmp_path):
    from paper_1909_04504_b200 import binding
    prog = tmp_path / "sz.c"
    prog.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "sph.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",'
                    'sizeof(sph_domain),sizeof(sph_params),sizeof(sph_array),sizeof(sph_stats),'
                    'offsetof(sph_array,x),offsetof(sph_params,g),offsetof(sph_stats,h_max),offsetof(sph_params,nlist_slots),offsetof(sph_stats,nlist_rows_capacity));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)])
    got = [int(v) for v in subprocess.check_output([str(exe)]).split()]
    want = [C.sizeof(binding.sph_domain), C.sizeof(binding.sph_params), C.sizeof(binding.sph_array),
            C.sizeof(binding.sph_stats), binding.sph_array.x.offset, binding.sph_params.g.offset,
            binding.sph_stats.h_max.offset, binding.sph_params.nlist_slots.offset,
            binding.sph_stats.nlist_rows_capacity.offset]
    assert got == want


def test_error_strings_and_null_handling(lib):
    assert lib.sph_strerror(0) == b"ok"
    assert b"capacity" in lib.sph_strerror(-3)
    assert lib.sph_destroy(None) == -1
    assert lib.sph_pc_step(None, 0.1, 1, 0) == -1
    assert lib.sph_create(None, None, None, 1, None, None) == -1


def test_no_cpu_fallback():
    """Without a CUDA device sph_create must fail with SPH_ERR_CUDA and the Python wrapper must raise."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1909_04504_b200 import binding, workloads
    wl = workloads.taylor_green_2d(8)
    with pytest.raises(binding.SphError):
        binding.SphContext.from_workload(wl)
    L = binding.load()
    dom = binding.sph_domain(); dom.dim = 2
    for k in range(3):
        dom.lo[k], dom.hi[k] = 0.0, 1.0
    prm = binding.sph_params(); prm.rho0 = prm.c0 = 1.0; prm.gamma = 7.0
    ctx = C.c_void_p()
    cap = (C.c_int64 * 1)(16)
    assert L.sph_create(C.byref(ctx), C.byref(prm), C.byref(dom), 1, cap, None) == -7
    assert not ctx.value


def test_oracle_and_product_are_isolated():
    pkg = os.path.join(ROOT, "paper_1909_04504_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", s, flags=re.M), f
                assert "sph_oracle" not in s and "liboracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1909_04504_b200" not in s.replace("paper_1909_04504_b200/csrc", "") or f.endswith(".cpp"), f
            assert not re.search(r"^\s*(from|import)\s+paper_1909_04504_b200", s, flags=re.M), f
            assert "#include \"../paper" not in s and "sph.h" not in s, f


def test_sources_target_sm100a_only():
    from paper_1909_04504_b200 import build
    assert build.ARCH == ["-gencode", "arch=compute_100a,code=sm_100a"]
    out = subprocess.check_output(["cuobjdump", "-lelf", build.LIB], text=True)
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out
