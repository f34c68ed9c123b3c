"""ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  (see the header of sph_oracle.cpp)

ctypes wrapper over oracle/sph_oracle.cpp plus the parts of the path that are per-particle numpy
one-liners: the group ordering of PAPER.md Listing 3 (L363-378), the predictor-corrector
integrator, eqs. 12-14 (L148-152), and the forward-Euler integrator of the paper's worked example
(L335, Fig.2; R22).  Everything is float64.  Pins: tests/test_oracle_*.py.  PARITY UNPINNED
(DESIGN.md section 2): the choice of the artificial-viscosity form and its constants, the h_ij
convention, the READING that rho is stepped like u (R11) and the order inside the Euler step (R22) -- the paper
prints no value to hold those choices to -- and the physical fidelity of the dam breaks.  The IMPLEMENTATION of
the chosen readings is pinned: both integrators have a step written out bit-equal by hand in the tests (PC:
test_single_step_is_eqs_12_to_14, test_continuity_mode_step_written_out; Euler: test_oracle_laminar.py).
This module imports nothing from the product package and the product imports nothing from here.

Duck-typed inputs: a "workload" is any object with attributes
  dim, lo, hi, periodic, kernel ('cubic'|'quintic'|'wendland_c2'), rho0, c0, gamma, alpha, eps, g,
  [nu, eta: laminar viscosity eq.10], arrays (each with x,y,z,u,v,w,h,m,rho and .fixed), density_sources, accel_sources, arho_sources.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_oracle.cpp")
_LIB = os.path.join(_HERE, "libsph_oracle.so")
KERNEL_ID = {"cubic": 0, "quintic": 1, "wendland_c2": 2}
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off -fopenmp (the float predicate must not be contracted)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-std=c++17", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Domain(C.Structure):
    _fields_ = [("dim", C.c_int), ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("periodic", C.c_int * 3)]


_DP = C.POINTER(C.c_double)
_IP = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_support.restype = C.c_double; L.orc_support.argtypes = [C.c_int]
        for f in (L.orc_W, L.orc_dWdr):
            f.restype = C.c_double; f.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double]
        L.orc_neighbors.restype = C.c_int64
        L.orc_neighbors.argtypes = [C.POINTER(_Domain), C.c_double, C.c_int, C.c_int,
                                    C.c_int64, _DP, _DP, _DP, _DP, C.c_int64, _DP, _DP, _DP, _DP,
                                    _IP, _IP, C.c_int64]
        L.orc_density.restype = None
        L.orc_density.argtypes = [C.POINTER(_Domain), C.c_int, C.c_int, C.c_int,
                                  C.c_int64, _DP, _DP, _DP, _DP, C.c_int64, _DP, _DP, _DP, _DP, _DP,
                                  _DP, _DP, _IP]
        L.orc_eos.restype = None
        L.orc_eos.argtypes = [C.c_int64, _DP, C.c_double, C.c_double, C.c_double, _DP]
        L.orc_accel.restype = None
        L.orc_accel.argtypes = [C.POINTER(_Domain), C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                C.c_int64] + [_DP] * 9 + [C.c_int64] + [_DP] * 10 + [_DP] * 7 + [_IP]
        L.orc_visc_laminar.restype = None
        L.orc_visc_laminar.argtypes = [C.POINTER(_Domain), C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                       C.c_int64] + [_DP] * 8 + [C.c_int64] + [_DP] * 9 + [_DP] * 5
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_DP)


def _domain(wl) -> _Domain:
    d = _Domain()
    d.dim = int(wl.dim)
    for k in range(3):
        d.lo[k] = float(wl.lo[k]); d.hi[k] = float(wl.hi[k]); d.periodic[k] = int(bool(wl.periodic[k]))
    return d


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


# ------------------------------------------------------------------------------------------------
def support(kernel: str) -> float:
    return float(lib().orc_support(KERNEL_ID[kernel]))


def W(kernel: str, dim: int, r: float, h: float) -> float:
    return float(lib().orc_W(KERNEL_ID[kernel], dim, float(r), float(h)))


def dWdr(kernel: str, dim: int, r: float, h: float) -> float:
    return float(lib().orc_dWdr(KERNEL_ID[kernel], dim, float(r), float(h)))


# ------------------------------------------------------------------------------------------------
class State:
    """Mutable float64 copy of a workload's particle arrays (+ p, au, av, aw, arho once evaluated)."""

    def __init__(self, wl):
        self.arrays: List[Dict[str, np.ndarray]] = []
        for a in wl.arrays:
            d = {k: _d(getattr(a, k)).copy() for k in ("x", "y", "z", "u", "v", "w", "h", "m", "rho")}
            d["p"] = np.zeros_like(d["x"])
            d["fixed"] = bool(a.fixed)
            self.arrays.append(d)
        self.have_accel = False

    def copy(self) -> "State":
        s = State.__new__(State)
        s.arrays = [{k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in a.items()} for a in self.arrays]
        s.have_accel = self.have_accel
        return s


def _method(method: str) -> int:
    return {"brute": 0, "cell": 1}[method]


def neighbors(wl, dest: Dict[str, np.ndarray], src: Dict[str, np.ndarray], pred32: bool = True,
              method: str = "cell", k: Optional[float] = None):
    """CSR (offsets[int64 nd+1], indices[int64]) of N(i) = {j in src : r_ij < k h_ij}, rows ascending."""
    L = lib(); dom = _domain(wl)
    k = support(wl.kernel) if k is None else float(k)
    xd, yd, zd, hd = (_d(dest[c]) for c in "xyzh")
    xs, ys, zs, hs = (_d(src[c]) for c in "xyzh")
    nd, ns = len(xd), len(xs)
    off = np.zeros(nd + 1, dtype=np.int64)
    args = [C.byref(dom), k, int(pred32), _method(method), nd, _p(xd), _p(yd), _p(zd), _p(hd),
            ns, _p(xs), _p(ys), _p(zs), _p(hs), off.ctypes.data_as(_IP)]
    total = L.orc_neighbors(*args, None, 0)
    idx = np.zeros(max(int(total), 1), dtype=np.int64)
    L.orc_neighbors(*args, idx.ctypes.data_as(_IP), int(total))
    return off, idx[:int(total)]


def _dest(st: State, dest: int, subset):
    """Destination fields of array `dest`, or of the particles `subset` (index array) of it: the sums are per
    destination particle, so a subset of destinations against ALL sources gives those particles' full sums."""
    D = st.arrays[dest]
    if subset is None:
        return D
    idx = np.asarray(subset, dtype=np.int64)
    return {k: (np.ascontiguousarray(v[idx]) if isinstance(v, np.ndarray) else v) for k, v in D.items()}


def density(wl, st: State, dest: int, sources: Sequence[int], pred32: bool = True, method: str = "cell",
            subset=None):
    """eq.3: returns (rho, abs_sum, n_pairs) for array `dest` (or its particles `subset`) summed over `sources`."""
    L = lib(); dom = _domain(wl); kid = KERNEL_ID[wl.kernel]
    D = _dest(st, dest, subset); nd = len(D["x"])
    rho = np.zeros(nd); ab = np.zeros(nd); npairs = np.zeros(1, dtype=np.int64)
    for s in sources:
        S = st.arrays[s]
        L.orc_density(C.byref(dom), kid, int(pred32), _method(method),
                      nd, _p(D["x"]), _p(D["y"]), _p(D["z"]), _p(D["h"]),
                      len(S["x"]), _p(S["x"]), _p(S["y"]), _p(S["z"]), _p(S["h"]), _p(S["m"]),
                      _p(rho), _p(ab), npairs.ctypes.data_as(_IP))
    return rho, ab, int(npairs[0])


def eos(wl, rho: np.ndarray) -> np.ndarray:
    """eq.6 / Listing 4 L393-400."""
    rho = _d(rho); p = np.zeros_like(rho)
    lib().orc_eos(len(rho), _p(rho), float(wl.rho0), float(wl.c0), float(wl.gamma), _p(p))
    return p


def accel(wl, st: State, dest: int, sources: Sequence[int], pred32: bool = True, method: str = "cell",
          gravity: bool = True, alpha: Optional[float] = None, subset=None, nu: Optional[float] = None):
    """eq.8-9 + Pi_ij (+ eq.7): dict(au,av,aw,arho,abs_a,abs_arho,visc_power,n_pairs) for array `dest`.
    The accumulators start at g (Listing 4: gravity is the initial value) and arho at 0 (L402-403)."""
    L = lib(); dom = _domain(wl); kid = KERNEL_ID[wl.kernel]
    D = _dest(st, dest, subset); nd = len(D["x"])
    g = wl.g if gravity else (0.0, 0.0, 0.0)
    out = {k: np.full(nd, float(g[i])) for i, k in enumerate(("au", "av", "aw"))}
    for k in ("arho", "abs_a", "abs_arho", "visc_power"):
        out[k] = np.zeros(nd)
    npairs = np.zeros(1, dtype=np.int64)
    al = float(wl.alpha if alpha is None else alpha)
    for s in sources:
        S = st.arrays[s]
        L.orc_accel(C.byref(dom), kid, al, float(wl.eps), float(wl.c0), int(pred32), _method(method),
                    nd, *(_p(D[c]) for c in ("x", "y", "z", "u", "v", "w", "h", "rho", "p")),
                    len(S["x"]), *(_p(S[c]) for c in ("x", "y", "z", "u", "v", "w", "h", "m", "rho", "p")),
                    _p(out["au"]), _p(out["av"]), _p(out["aw"]), _p(out["arho"]),
                    _p(out["abs_a"]), _p(out["abs_arho"]), _p(out["visc_power"]),
                    npairs.ctypes.data_as(_IP))
    nu_ = float(getattr(wl, "nu", 0.0) if nu is None else nu)
    out["lam_power"] = np.zeros(nd)
    if nu_ != 0.0:                                        # laminar viscosity, eq.10 (L134-136)
        for s in sources:
            S = st.arrays[s]
            L.orc_visc_laminar(C.byref(dom), kid, nu_, float(getattr(wl, "eta", 0.01)), int(pred32), _method(method),
                               nd, *(_p(D[c]) for c in ("x", "y", "z", "u", "v", "w", "h", "rho")),
                               len(S["x"]), *(_p(S[c]) for c in ("x", "y", "z", "u", "v", "w", "h", "m", "rho")),
                               _p(out["au"]), _p(out["av"]), _p(out["aw"]), _p(out["abs_a"]), _p(out["lam_power"]))
    out["n_pairs"] = int(npairs[0])
    return out


# ------------------------------------------------------------------------------------------------
# Group ordering (Listing 3; Fig.3): [density] -> EOS on ALL arrays -> barrier ->
# continuity + momentum.  Summation mode replaces the continuity ODE by eq.3 (R12/R13).
# ------------------------------------------------------------------------------------------------
def evaluate(wl, st: State, mode: str, pred32: bool = False, method: str = "cell") -> int:
    """Compute rho (summation mode), p, and the accelerations au,av,aw (dynamic arrays) / arho
    (continuity mode, every array) in place.  Returns the number of (i,j) pairs visited."""
    na = len(st.arrays); pairs = 0
    if mode == "summation":
        new_rho = []
        for d in range(na):
            r, _, c = density(wl, st, d, wl.density_sources[d], pred32, method)
            new_rho.append(r); pairs += c
        for d in range(na):
            st.arrays[d]["rho"] = new_rho[d]
    for d in range(na):                                   # Group 1: EOS(dest=fluid), EOS(dest=solid)
        st.arrays[d]["p"] = eos(wl, st.arrays[d]["rho"])
    for d in range(na):                                   # Group 2
        A = st.arrays[d]
        srcs = wl.accel_sources[d] if not A["fixed"] else []
        if srcs:
            o = accel(wl, st, d, srcs, pred32, method)
            A["au"], A["av"], A["aw"] = o["au"], o["av"], o["aw"]
            pairs += o["n_pairs"]
            if mode == "continuity":
                if list(wl.arho_sources[d]) == list(srcs):
                    A["arho"] = o["arho"]
                else:
                    A["arho"] = accel(wl, st, d, wl.arho_sources[d], pred32, method)["arho"]
        else:
            z = np.zeros_like(A["x"])
            A["au"], A["av"], A["aw"] = z, z.copy(), z.copy()
            if mode == "continuity":
                o = accel(wl, st, d, wl.arho_sources[d], pred32, method)   # ContinuityEquation(dest=solid, sources=[fluid])
                A["arho"] = o["arho"]; pairs += o["n_pairs"]
    st.have_accel = True
    return pairs


def _wrap(x: np.ndarray, lo: float, hi: float) -> np.ndarray:
    L = hi - lo
    x = np.where(x >= hi, x - L, x)
    return np.where(x < lo, x + L, x)


def pc_step(wl, st: State, dt: float, mode: str, move: bool = True, pred32: bool = False,
            method: str = "cell") -> int:
    """One predictor-corrector step, eqs. 12-14 (L148-152), R10/R11:
         u^{n+1/2} = u^n + dt/2 a^n                                  (12)
         x^{n+1}   = x^n + dt u^{n+1/2}      (+ periodic wrap, L443)  (13)
         a^{n+1}   = F(x^{n+1}, u^{n+1/2}, rho)                       (one evaluation per step)
         u^{n+1}   = u^{n+1/2} + dt/2 a^{n+1}                         (14)
       Continuity mode steps rho like u (R11); fixed arrays keep x,u (L142) but get rho/p.
       move=False (C5: "density + momentum" only) skips (13).  a^0 is evaluated on the first call."""
    pairs = 0
    if not st.have_accel:
        pairs += evaluate(wl, st, mode, pred32, method)
    comps = (("u", "au", "x"), ("v", "av", "y"), ("w", "aw", "z"))
    for A in st.arrays:
        if not A["fixed"]:
            for k, (vel, acc, pos) in enumerate(comps):
                if k >= wl.dim:
                    continue
                A[vel] = A[vel] + 0.5 * dt * A[acc]                                   # (12)
                if move:
                    A[pos] = A[pos] + dt * A[vel]                                     # (13)
                    if wl.periodic[k]:
                        A[pos] = _wrap(A[pos], float(wl.lo[k]), float(wl.hi[k]))
        if mode == "continuity":
            A["rho"] = A["rho"] + 0.5 * dt * A["arho"]
    pairs += evaluate(wl, st, mode, pred32, method)
    for A in st.arrays:
        if not A["fixed"]:
            for k, (vel, acc, _) in enumerate(comps):
                if k < wl.dim:
                    A[vel] = A[vel] + 0.5 * dt * A[acc]                               # (14)
        if mode == "continuity":
            A["rho"] = A["rho"] + 0.5 * dt * A["arho"]
    return pairs


def euler_step(wl, st: State, dt: float, mode: str, move: bool = True, pred32: bool = False,
               method: str = "cell") -> int:
    """One forward-Euler step ("a simple forward Euler integrator", Fig.2; R22):
         a^n = F(x^n, u^n, rho^n)          (evaluated on the first call, afterwards carried over)
         x^{n+1} = x^n + dt u^n ; u^{n+1} = u^n + dt a^n ; rho^{n+1} = rho^n + dt arho^n (continuity mode)
         periodic wrap (L443) ; a^{n+1} = F(x^{n+1}, u^{n+1}, rho^{n+1})
       Fixed arrays keep x,u."""
    pairs = 0
    if not st.have_accel:
        pairs += evaluate(wl, st, mode, pred32, method)
    comps = (("u", "au", "x"), ("v", "av", "y"), ("w", "aw", "z"))
    for A in st.arrays:
        if not A["fixed"]:
            for k, (vel, acc, pos) in enumerate(comps):
                if k >= wl.dim:
                    continue
                if move:
                    A[pos] = A[pos] + dt * A[vel]
                    if wl.periodic[k]:
                        A[pos] = _wrap(A[pos], float(wl.lo[k]), float(wl.hi[k]))
                A[vel] = A[vel] + dt * A[acc]
        if mode == "continuity":
            A["rho"] = A["rho"] + dt * A["arho"]
    pairs += evaluate(wl, st, mode, pred32, method)
    return pairs
