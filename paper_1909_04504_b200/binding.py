"""Thin Python binding over the C ABI in include/sph.h (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels of libsph_b200.so.  PyTorch supplies device memory and
streams; nothing here computes.  There is NO CPU fallback: loading fails loudly if the library is missing,
and sph_create fails with SPH_ERR_CUDA if there is no usable device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SPH_B200_LIB") or os.path.join(_HERE, "libsph_b200.so")
LIB_PATHS = {"f32": LIB_PATH, "f64": os.path.join(_HERE, "libsph_b200_f64.so")}     # sph_real = float / double

SPH_MAX_ARRAYS = 4
KERNEL_ID = {"cubic": 0, "quintic": 1, "wendland_c2": 2}
SUMMATION, CONTINUITY = 0, 1
MODE_ID = {"summation": SUMMATION, "continuity": CONTINUITY}
INTEGRATOR_ID = {"pc": 0, "euler": 1}
MEM_DEVICE, MEM_HOST = 0, 1
ARRAY_DYNAMIC, ARRAY_FIXED = 0, 1

EXPORTS = ["sph_create", "sph_destroy", "sph_set_tables", "sph_nnps_build", "sph_summation_density",
           "sph_wcsph_accel", "sph_pc_step", "sph_sync_state", "sph_get_accel", "sph_nnps_get_neighbors",
           "sph_get_stats", "sph_synchronize", "sph_strerror", "sph_last_error", "sph_abi_version",
           "sph_set_profiling", "sph_get_profile", "sph_kernel_name", "sph_fp32_probe", "sph_stencil_candidates",
           "sph_real_size", "sph_cell_offsets_static", "sph_static_last_error"]

_FP = C.POINTER(C.c_float)
FIELD_NAMES = ("x", "y", "z", "u", "v", "w", "h", "m", "rho", "p", "ax", "ay", "az", "arho")
SPH_K_COUNT = 16


class sph_domain(C.Structure):
    _fields_ = [("dim", C.c_int), ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("periodic", C.c_int * 3)]


class sph_params(C.Structure):
    _fields_ = [("kernel", C.c_int), ("rho0", C.c_double), ("c0", C.c_double), ("gamma", C.c_double),
                ("alpha", C.c_double), ("eps", C.c_double), ("g", C.c_double * 3), ("move", C.c_int),
                ("nu", C.c_double), ("eta", C.c_double), ("integrator", C.c_int),
                ("xsub", C.c_int), ("levels", C.c_int), ("nlist_slots", C.c_int)]


class sph_array(C.Structure):
    _fields_ = [("n", C.c_int64), ("flags", C.c_int), ("mem", C.c_int)] + \
               [(k, C.c_void_p) for k in FIELD_NAMES]


class sph_stats(C.Structure):
    _fields_ = [("n_cells", C.c_int32 * 3), ("cell_size", C.c_double * 3), ("n_particles", C.c_int64),
                ("pairs_density", C.c_int64), ("pairs_accel", C.c_int64), ("candidates", C.c_int64),
                ("candidates_density", C.c_int64), ("candidates_accel", C.c_int64),
                ("kernel_launches", C.c_int64), ("steps_done", C.c_int64), ("variable_h", C.c_int32),
                ("h_max", C.c_float), ("xsub", C.c_int32), ("used_rows", C.c_int32),
                ("nlist_rows_used", C.c_int64), ("nlist_rows_capacity", C.c_int64),
                ("nlist_fallback_warps", C.c_int64), ("n_levels", C.c_int32), ("n_keys", C.c_int64),
                ("candidates_search", C.c_int64)]


class sph_profile(C.Structure):
    _fields_ = [("launches", C.c_int64 * SPH_K_COUNT), ("ms", C.c_double * SPH_K_COUNT), ("dropped", C.c_int64)]


class SphError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"sph error {code}: {msg}")
        self.code = code


_libs = {}


def load(precision: str = "f32") -> C.CDLL:
    """Loads libsph_b200.so ("f32") or libsph_b200_f64.so ("f64") (build them first with
    `python -m paper_1909_04504_b200.build`)."""
    if precision not in _libs:
        path = LIB_PATHS[precision]
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: build the CUDA library "
                              "(python -m paper_1909_04504_b200.build); there is no CPU fallback")
        L = C.CDLL(path)
        vp, i32, i64, u32p = C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_uint32)
        L.sph_create.argtypes = [C.POINTER(vp), C.POINTER(sph_params), C.POINTER(sph_domain), i32, C.POINTER(i64), vp]
        L.sph_destroy.argtypes = [vp]
        L.sph_set_tables.argtypes = [vp, u32p, u32p, u32p]
        L.sph_nnps_build.argtypes = [vp, i32, C.POINTER(sph_array)]
        L.sph_summation_density.argtypes = [vp, i32, C.c_uint32, vp, vp, i32]
        L.sph_wcsph_accel.argtypes = [vp, i32, C.c_uint32, vp, vp, vp, vp, i32]
        L.sph_pc_step.argtypes = [vp, C.c_double, i32, i32]
        L.sph_sync_state.argtypes = [vp, i32, C.POINTER(sph_array)]
        L.sph_get_accel.argtypes = [vp, i32, vp, vp, vp, vp, i32]
        L.sph_nnps_get_neighbors.argtypes = [vp, i32, i32, vp, vp, i64, C.POINTER(i64), i32]
        L.sph_get_stats.argtypes = [vp, C.POINTER(sph_stats)]
        L.sph_synchronize.argtypes = [vp]
        L.sph_set_profiling.argtypes = [vp, i32]
        L.sph_get_profile.argtypes = [vp, C.POINTER(sph_profile)]
        L.sph_kernel_name.argtypes = [i32]; L.sph_kernel_name.restype = C.c_char_p
        L.sph_fp32_probe.argtypes = [vp, i32, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.sph_stencil_candidates.argtypes = [vp, C.POINTER(i64)]
        L.sph_strerror.argtypes = [i32]; L.sph_strerror.restype = C.c_char_p
        L.sph_last_error.argtypes = [vp]; L.sph_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("sph_strerror", "sph_last_error", "sph_kernel_name"):
                getattr(L, name).restype = i32
        L.sph_static_last_error.argtypes = []; L.sph_static_last_error.restype = C.c_char_p
        L.sph_cell_offsets_static.argtypes = [vp, C.c_int64, vp, vp]
        if L.sph_real_size() != (4 if precision == "f32" else 8):
            raise ImportError(f"{path}: sph_real_size() does not match precision {precision}")
        _libs[precision] = L
    return _libs[precision]


STATIC_SCAN_MAX_N = 1 << 26       # SPH_STATIC_SCAN_MAX_N of include/sph.h


def cell_offsets_static(counts, offsets, stream=None, precision: str = "f32", n: Optional[int] = None):
    """sph_cell_offsets_static (include/sph.h): offsets[0..n] = exclusive prefix sum of counts[0..n) on the GPU,
    with the scan's scratch in the library's static device array -- the call allocates nothing.  `counts` (n) and
    `offsets` (>= n + 1) are CUDA tensors of a 32-bit integer type on the current device; `stream` a torch stream
    (default: the current one).  Argument marshalling only; raises SphError (n beyond the limit -> code -3)."""
    import torch
    L = load(precision)
    n = int(counts.numel()) if n is None else int(n)
    for t in (counts, offsets):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 4 and not t.dtype.is_floating_point
    assert n > STATIC_SCAN_MAX_N or (counts.numel() >= n and offsets.numel() >= n + 1)
    st = torch.cuda.current_stream(counts.device) if stream is None else stream
    with torch.cuda.device(counts.device):
        rc = L.sph_cell_offsets_static(counts.data_ptr(), n, offsets.data_ptr(), st.cuda_stream)
    if rc != 0:
        raise SphError(rc, L.sph_static_last_error().decode())
    return offsets


def _ptr_and_mem(t, real_size=4):
    """(address, mem) of a torch tensor (cuda -> DEVICE, cpu -> HOST) or a numpy array (HOST)."""
    if t is None:
        return None, None
    if isinstance(t, np.ndarray):
        assert t.dtype == (np.float32 if real_size == 4 else np.float64) and t.flags["C_CONTIGUOUS"]
        return t.ctypes.data, MEM_HOST
    assert t.dtype.is_floating_point and t.element_size() == real_size and t.is_contiguous()
    return t.data_ptr(), (MEM_DEVICE if t.is_cuda else MEM_HOST)


def make_array(fields: Dict[str, object], fixed: bool, real_size: int = 4) -> sph_array:
    """fields: name -> torch tensor / numpy float32 array (all on the same side) for x,y,z,u,v,w,h,m,rho,p."""
    a = sph_array()
    a.flags = ARRAY_FIXED if fixed else ARRAY_DYNAMIC
    mem = None
    n = None
    for k in FIELD_NAMES:
        ptr, m = _ptr_and_mem(fields.get(k), real_size)
        setattr(a, k, ptr)
        if ptr is not None or (fields.get(k) is not None):
            t = fields[k]
            n = int(t.shape[0]) if n is None else n
            assert int(t.shape[0]) == n
            mem = m if mem is None else mem
            assert mem == m, "all fields of an array must live on the same side"
    a.n = n or 0
    a.mem = MEM_DEVICE if mem is None else mem
    return a


class SphContext:
    """Owns one sph_ctx.  Methods mirror the C calls one to one."""

    def __init__(self, *, dim: int, lo, hi, periodic, kernel: str, rho0: float, c0: float, gamma: float = 7.0,
                 alpha: float = 0.1, eps: float = 0.01, g=(0.0, 0.0, 0.0), move: bool = True,
                 capacity: Sequence[int], stream=None, xsub: int = 0, nlist_slots: int = 0, levels: int = 0,
                 nu: float = 0.0, eta: float = 0.01, integrator: str = "pc", precision: str = "f32"):
        import torch
        if not torch.cuda.is_available():
            raise SphError(-7, "no CUDA device: the SPH path has no CPU fallback")
        self.L = load(precision)
        self.torch = torch
        self.precision = precision
        self.real_size = 4 if precision == "f32" else 8
        self.dtype = torch.float32 if precision == "f32" else torch.float64
        self.stream = stream
        dom = sph_domain(); dom.dim = int(dim)
        prm = sph_params(); prm.kernel = KERNEL_ID[kernel]
        prm.rho0, prm.c0, prm.gamma, prm.alpha, prm.eps, prm.move = rho0, c0, gamma, alpha, eps, int(move)
        prm.xsub, prm.nlist_slots, prm.levels = int(xsub), int(nlist_slots), int(levels)
        prm.nu, prm.eta, prm.integrator = float(nu), float(eta), INTEGRATOR_ID[integrator]
        for k in range(3):
            dom.lo[k], dom.hi[k], dom.periodic[k] = float(lo[k]), float(hi[k]), int(bool(periodic[k]))
            prm.g[k] = float(g[k])
        self.na = len(capacity)
        cap = (C.c_int64 * self.na)(*[int(v) for v in capacity])
        self.ctx = C.c_void_p()
        s = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
        self.device = torch.device("cuda", torch.cuda.current_device())
        rc = self.L.sph_create(C.byref(self.ctx), C.byref(prm), C.byref(dom), self.na, cap, C.c_void_p(s))
        if rc:
            msg = self.L.sph_last_error(self.ctx).decode() if self.ctx else self.L.sph_strerror(rc).decode()
            if self.ctx:
                self.L.sph_destroy(self.ctx); self.ctx = C.c_void_p()
            raise SphError(rc, msg or self.L.sph_strerror(rc).decode())
        self.n = [0] * self.na
        self.dim = int(dim)

    @classmethod
    def from_workload(cls, wl, stream=None, capacity=None, **over):
        kw = dict(dim=wl.dim, lo=wl.lo, hi=wl.hi, periodic=wl.periodic, kernel=wl.kernel, rho0=wl.rho0, c0=wl.c0,
                  gamma=wl.gamma, alpha=wl.alpha, eps=wl.eps, g=wl.g, nu=wl.nu, eta=wl.eta, integrator=wl.integrator,
                  capacity=capacity or [a.n for a in wl.arrays], stream=stream)
        kw.update(over)
        return cls(**kw)

    def _check(self, rc: int):
        if rc:
            raise SphError(rc, (self.L.sph_last_error(self.ctx) or b"").decode() or self.L.sph_strerror(rc).decode())

    def close(self):
        if getattr(self, "ctx", None):
            self.L.sph_destroy(self.ctx); self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C calls --------------------------------------------------------------------------
    def set_tables(self, density=None, accel=None, arho=None):
        def arr(v):
            return None if v is None else (C.c_uint32 * self.na)(*[int(x) for x in v])
        self._check(self.L.sph_set_tables(self.ctx, arr(density), arr(accel), arr(arho)))

    def nnps_build(self, arrays: List[Dict[str, object]], fixed: Sequence[bool]):
        """arrays[a]: dict of float32 tensors (cuda or cpu) / numpy arrays keyed x,y,z,u,v,w,h,m,rho,p."""
        A = (sph_array * self.na)(*[make_array(f, fx, self.real_size) for f, fx in zip(arrays, fixed)])
        self._keep = arrays                      # keep caller buffers alive while copies are in flight
        self.n = [int(A[a].n) for a in range(self.na)]
        self._check(self.L.sph_nnps_build(self.ctx, self.na, A))

    def _out(self, n, host):
        t = self.torch
        return t.empty(n, dtype=self.dtype, pin_memory=True) if host else t.empty(n, dtype=self.dtype, device=self.device)

    def summation_density(self, dest: int, source_mask: int, want_p: bool = True, host: bool = False):
        rho = self._out(self.n[dest], host)
        p = self._out(self.n[dest], host) if want_p else None
        self._check(self.L.sph_summation_density(self.ctx, dest, source_mask, rho.data_ptr(),
                                                 p.data_ptr() if want_p else None, MEM_HOST if host else MEM_DEVICE))
        return rho, p

    def wcsph_accel(self, dest: int, source_mask: int, want_arho: bool = False, host: bool = False):
        n = self.n[dest]
        ax, ay = self._out(n, host), self._out(n, host)
        az = self._out(n, host) if self.dim == 3 else None
        ar = self._out(n, host) if want_arho else None
        self._check(self.L.sph_wcsph_accel(self.ctx, dest, source_mask, ax.data_ptr(), ay.data_ptr(),
                                           az.data_ptr() if az is not None else None,
                                           ar.data_ptr() if ar is not None else None,
                                           MEM_HOST if host else MEM_DEVICE))
        return ax, ay, az, ar

    def pc_step(self, dt: float, n_steps: int, mode):
        self._check(self.L.sph_pc_step(self.ctx, float(dt), int(n_steps), MODE_ID.get(mode, mode)))

    def sync_state(self, array: int, fields=("x", "y", "z", "u", "v", "w", "rho", "p"), host: bool = False, out=None):
        n = self.n[array]
        if out is None:
            out = {k: self._out(n, host) for k in fields if not (self.dim == 2 and k in ("z", "w", "az"))}
        a = make_array(out, False, self.real_size)
        a.n = n; a.mem = MEM_HOST if host else MEM_DEVICE
        self._check(self.L.sph_sync_state(self.ctx, array, C.byref(a)))
        return out

    def get_accel(self, array: int, host: bool = False):
        n = self.n[array]
        o = [self._out(n, host) for _ in range(4)]
        self._check(self.L.sph_get_accel(self.ctx, array, *[t.data_ptr() for t in o], MEM_HOST if host else MEM_DEVICE))
        return dict(ax=o[0], ay=o[1], az=o[2], arho=o[3])

    def nnps_get_neighbors(self, dest: int, src: int):
        """CSR (offsets int64[n+1], indices int32[total]) as numpy arrays (verification export, synchronises)."""
        n = self.n[dest]
        off = np.zeros(n + 1, dtype=np.int64)
        total = C.c_int64(0)
        self._check(self.L.sph_nnps_get_neighbors(self.ctx, dest, src, off.ctypes.data, None, 0, C.byref(total), MEM_HOST))
        idx = np.zeros(max(total.value, 1), dtype=np.int32)
        self._check(self.L.sph_nnps_get_neighbors(self.ctx, dest, src, off.ctypes.data, idx.ctypes.data,
                                                  total.value, C.byref(total), MEM_HOST))
        return off, idx[:total.value]

    def neighbor_counts(self, dest: int, src: int):
        """|N_src(i)| for every particle i of `dest` (the counting pass of the verification export only)."""
        n = self.n[dest]
        off = np.zeros(n + 1, dtype=np.int64)
        total = C.c_int64(0)
        self._check(self.L.sph_nnps_get_neighbors(self.ctx, dest, src, off.ctypes.data, None, 0, C.byref(total), MEM_HOST))
        return np.diff(off)

    def get_stats(self) -> sph_stats:
        s = sph_stats()
        self._check(self.L.sph_get_stats(self.ctx, C.byref(s)))
        return s

    def synchronize(self):
        self._check(self.L.sph_synchronize(self.ctx))

    def set_profiling(self, enable: bool):
        self._check(self.L.sph_set_profiling(self.ctx, int(bool(enable))))

    def stencil_candidates(self) -> int:
        """Candidate-set size of the paper's own cell-list search (3^d cells >= k h_max) on the current state."""
        out = C.c_int64(0)
        self._check(self.L.sph_stencil_candidates(self.ctx, C.byref(out)))
        return int(out.value)

    def fp32_probe(self, packed: bool, iters: int = 4096):
        """(TFLOP/s, ms) of the FP32 FMA issue-rate probe (diagnostic; the ALU roofline denominator)."""
        tf, ms = C.c_double(0.0), C.c_double(0.0)
        self._check(self.L.sph_fp32_probe(self.ctx, int(bool(packed)), int(iters), C.byref(tf), C.byref(ms)))
        return tf.value, ms.value

    def get_profile(self) -> Dict[str, Dict[str, float]]:
        """{kernel name: {"launches": n, "ms": summed device time}} since set_profiling(True)."""
        p = sph_profile()
        self._check(self.L.sph_get_profile(self.ctx, C.byref(p)))
        out = {}
        for k in range(SPH_K_COUNT):
            if p.launches[k]:
                out[self.L.sph_kernel_name(k).decode()] = {"launches": int(p.launches[k]), "ms": float(p.ms[k])}
        out["_dropped"] = int(p.dropped)
        return out


def device_arrays(wl, device=None, precision: str = "f32"):
    """Uploads a workload's float32 numpy arrays as torch CUDA tensors (one dict per particle array); precision
    "f64" widens them to double (the values stay the float32-representable ones the workload holds)."""
    import torch
    dev = device or torch.device("cuda", torch.cuda.current_device())
    dt = torch.float32 if precision == "f32" else torch.float64
    keys = ("x", "y", "z", "u", "v", "w", "h", "m", "rho")
    return [{k: torch.from_numpy(getattr(a, k)).to(dev).to(dt).contiguous() for k in keys} for a in wl.arrays]


def pinned_arrays(wl):
    import torch
    keys = ("x", "y", "z", "u", "v", "w", "h", "m", "rho")
    return [{k: torch.from_numpy(getattr(a, k)).pin_memory() for k in keys} for a in wl.arrays]
