"""Seeded synthetic inputs shaped like the paper's workloads.

This module holds NO SPH arithmetic (no kernels, sums, EOS, integrator): it only lays out
particles, velocities and parameters.  It is the one module both the CUDA path's callers and
the oracle's callers (tests, bench cpu_baseline leg, smoke) take inputs from; neither the
oracle nor the CUDA library imports it.

The paper's own example scripts and outputs are not available (PAPER.md L246/L643 point to a
repository that is not in this environment), so these inputs STAND IN for them:
  C1  2-D Taylor-Green state on a jittered 64x64 periodic lattice    (eqs. for u,v)
  C2  2-D dam break: fluid block + 3-layer open-top tank             (PAPER.md L142, L295-312 geometry)
  C3  3-D periodic jittered 128^3 lattice, random velocities         ("block of water")
  C4  3-D dam break: fluid column + 3-layer open-top tank
  C5  3-D non-uniform (8 Gaussians + background), variable h         (PAPER.md L158-160 variable h)
All values are generated in float64 with numpy.random.default_rng(seed) and rounded ONCE to
float32; both sides receive the identical float32 arrays.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

KERNELS = ("cubic", "quintic", "wendland_c2")
SUMMATION, CONTINUITY = "summation", "continuity"


@dataclass
class PArray:
    """One named particle array (properties x,y,z,u,v,w,h,m,rho; p is an output)."""
    name: str
    fixed: bool
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    u: np.ndarray
    v: np.ndarray
    w: np.ndarray
    h: np.ndarray
    m: np.ndarray
    rho: np.ndarray

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def fields(self):
        return dict(x=self.x, y=self.y, z=self.z, u=self.u, v=self.v, w=self.w,
                    h=self.h, m=self.m, rho=self.rho)


@dataclass
class Workload:
    name: str
    dim: int
    lo: Tuple[float, float, float]
    hi: Tuple[float, float, float]
    periodic: Tuple[bool, bool, bool]
    kernel: str
    rho0: float
    c0: float
    gamma: float
    alpha: float
    eps: float
    g: Tuple[float, float, float]
    dt: float
    n_steps: int
    density_mode: str
    arrays: List[PArray]
    note: str = ""
    # dest/source tables, indices into `arrays`
    density_sources: Optional[List[List[int]]] = None   # per dest array
    accel_sources: Optional[List[List[int]]] = None      # per dynamic dest array ([] for fixed)
    arho_sources: Optional[List[List[int]]] = None       # continuity mode, per dest array
    nu: float = 0.0                                      # laminar kinematic viscosity of eq.10 (L134-136); 0 = term off
    eta: float = 0.01                                    # its regulariser eta (eq.10)
    integrator: str = "pc"                               # "pc" (eqs. 12-14) or "euler" (L335, Fig.2)

    @property
    def n_total(self) -> int:
        return sum(a.n for a in self.arrays)

    def __post_init__(self):
        na = len(self.arrays)
        allsrc = list(range(na))
        dyn = [i for i, a in enumerate(self.arrays) if not a.fixed]
        if self.density_sources is None:
            self.density_sources = [allsrc for _ in range(na)]
        if self.accel_sources is None:
            self.accel_sources = [allsrc if not a.fixed else [] for a in self.arrays]
        if self.arho_sources is None:
            # continuity: dynamic <- all ; fixed (solid) <- dynamic (fluid) only  (L369-374)
            self.arho_sources = [allsrc if not a.fixed else dyn for a in self.arrays]


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _wrap32(x64: np.ndarray, lo: float, hi: float) -> np.ndarray:
    """Wrap into [lo,hi) in float64, round to float32, and fold a rounded-up hi back to lo."""
    L = hi - lo
    x = lo + np.mod(x64 - lo, L)
    x32 = x.astype(np.float32)
    x32[x32 >= np.float32(hi)] = np.float32(lo)
    return np.ascontiguousarray(x32)


def _make_array(name, fixed, x, y, z, u, v, w, h, m, rho) -> PArray:
    n = len(x)

    def full(val):
        if np.isscalar(val):
            return np.full(n, val, dtype=np.float32)
        return _f32(val)
    return PArray(name, fixed, full(x), full(y), full(z), full(u), full(v), full(w),
                  full(h), full(m), full(rho))


# --------------------------------------------------------------------------------------------
# geometry helpers (layout only)
# --------------------------------------------------------------------------------------------
def block_2d_inclusive(dx: float, length: float, height: float, center=(0.0, 0.0)):
    """Endpoint-inclusive block like the paper's get_2d_block (PAPER.md L299-302, L319-324:
    dx=0.1, length=1, height=2 -> 231 particles, x from -1.9 to -0.9 for center x=-1.5+dx)."""
    nx = int(round(length / dx)) + 1
    ny = int(round(height / dx)) + 1
    xs = center[0] - 0.5 * length + dx * np.arange(nx)
    ys = center[1] - 0.5 * height + dx * np.arange(ny)
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    return X.ravel(), Y.ravel()


def _cell_centred(n: Sequence[int], dx: float, origin: Sequence[float]):
    axes = [origin[k] + (np.arange(n[k]) + 0.5) * dx for k in range(len(n))]
    grids = np.meshgrid(*axes, indexing="ij")
    return [g.ravel() for g in grids]


def tank_2d_open_top(dx: float, length: float, height: float, layers: int = 3):
    """3 layers of wall particles outside left/right/bottom of [0,length]x[0,height], open top."""
    nx = int(round(length / dx))
    ny = int(round(height / dx))
    xs, ys = [], []
    ycol = (np.arange(-layers, ny) + 0.5) * dx
    for l in range(layers):
        xs.append(np.full(ycol.shape, -(l + 0.5) * dx)); ys.append(ycol)            # left
        xs.append(np.full(ycol.shape, length + (l + 0.5) * dx)); ys.append(ycol)    # right
    xrow = (np.arange(nx) + 0.5) * dx
    for l in range(layers):
        xs.append(xrow); ys.append(np.full(xrow.shape, -(l + 0.5) * dx))            # bottom
    return np.concatenate(xs), np.concatenate(ys)


def tank_3d_open_top(dx: float, lx: float, ly: float, lz: float, layers: int = 3):
    """3 layers outside floor + 4 walls of [0,lx]x[0,ly]x[0,lz], open top."""
    nx, ny, nz = (int(round(v / dx)) for v in (lx, ly, lz))
    ix = np.arange(-layers, nx + layers)
    iy = np.arange(-layers, ny + layers)
    iz = np.arange(-layers, nz)
    IX, IY, IZ = np.meshgrid(ix, iy, iz, indexing="ij")
    inside = (IX >= 0) & (IX < nx) & (IY >= 0) & (IY < ny) & (IZ >= 0)
    keep = ~inside
    return ((IX[keep] + 0.5) * dx, (IY[keep] + 0.5) * dx, (IZ[keep] + 0.5) * dx)


# --------------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------------
def taylor_green_2d(n: int = 64, seed: int = 0, jitter: float = 0.1, hdx: float = 1.3,
                    kernel: str = "cubic", n_steps: int = 1) -> Workload:
    """C1. Periodic unit box, n x n cell-centred lattice jittered by U(-jitter*dx, jitter*dx);
    velocities are the t=0 Taylor-Green field (PAPER.md L649-652 with U=1) at the jittered points."""
    dx = 1.0 / n
    rng = np.random.default_rng(seed)
    X, Y = _cell_centred((n, n), dx, (0.0, 0.0))
    jit = rng.uniform(-jitter * dx, jitter * dx, size=(n * n, 2))
    x = _wrap32(X + jit[:, 0], 0.0, 1.0)
    y = _wrap32(Y + jit[:, 1], 0.0, 1.0)
    xd, yd = x.astype(np.float64), y.astype(np.float64)
    u = -np.cos(2 * np.pi * xd) * np.sin(2 * np.pi * yd)
    v = np.sin(2 * np.pi * xd) * np.cos(2 * np.pi * yd)
    rho0, c0 = 1.0, 10.0
    h = hdx * dx
    arr = _make_array("fluid", False, x, y, 0.0, u, v, 0.0, h, rho0 * dx * dx, rho0)
    return Workload(f"C1_taylor_green_2d_{n}x{n}", 2, (0, 0, 0), (1, 1, 1), (True, True, False),
                    kernel, rho0, c0, 7.0, 0.1, 0.01, (0, 0, 0), 0.25 * h / c0, n_steps,
                    SUMMATION, [arr], note="BASELINE.json configs[0]")


def dam_break_2d(dx: float = 0.01, n_steps: int = 1000, density_mode: str = CONTINUITY,
                 kernel: str = "quintic", hdx: float = 1.0) -> Workload:
    """C2. Fluid block 1x2 (cell-centred, 100x200 = 20,000 at dx=0.01) in a 4x4 tank with 3 wall layers.
    dt = 0.125 h/c0 (R24: BASELINE gives no time step for the dam breaks; 0.25 h/c0 is unstable here)."""
    fx, fy = _cell_centred((int(round(1.0 / dx)), int(round(2.0 / dx))), dx, (0.0, 0.0))
    sx, sy = tank_2d_open_top(dx, 4.0, 4.0, 3)
    rho0 = 1000.0
    c0 = 10.0 * np.sqrt(2 * 9.81 * 2.0)
    h = hdx * dx
    m = rho0 * dx * dx
    fluid = _make_array("fluid", False, fx, fy, 0.0, 0.0, 0.0, 0.0, h, m, rho0)
    solid = _make_array("solid", True, sx, sy, 0.0, 0.0, 0.0, 0.0, h, m, rho0)
    pad = 4 * dx
    lo = (-3 * dx - pad, -3 * dx - pad, 0.0)
    hi = (4.0 + 3 * dx + pad, 4.0 + pad, 1.0)
    return Workload(f"C2_dam_break_2d_dx{dx:g}", 2, lo, hi, (False, False, False), kernel,
                    rho0, float(c0), 7.0, 0.1, 0.01, (0.0, -9.81, 0.0), 0.125 * h / float(c0),
                    n_steps, density_mode, [fluid, solid], note="BASELINE.json configs[1]")


def periodic_box_3d(n: Sequence[int] = (128, 128, 128), seed: int = 1, jitter: float = 0.1,
                    hdx: float = 1.2, kernel: str = "wendland_c2", n_steps: int = 100,
                    dx: Optional[float] = None) -> Workload:
    """C3. Periodic box of n[0] x n[1] x n[2] cell-centred lattice points (dx = 1/n[0] unless given),
    jittered, velocities U[-1,1]^3 drawn AFTER the positions from the same generator."""
    n = tuple(int(v) for v in n)
    dx = 1.0 / n[0] if dx is None else dx
    N = n[0] * n[1] * n[2]
    hi = tuple(n[k] * dx for k in range(3))
    rng = np.random.default_rng(seed)
    X, Y, Z = _cell_centred(n, dx, (0.0, 0.0, 0.0))
    jit = rng.uniform(-jitter * dx, jitter * dx, size=(N, 3))
    vel = rng.uniform(-1.0, 1.0, size=(N, 3))
    x = _wrap32(X + jit[:, 0], 0.0, hi[0])
    y = _wrap32(Y + jit[:, 1], 0.0, hi[1])
    z = _wrap32(Z + jit[:, 2], 0.0, hi[2])
    rho0, c0 = 1.0, 10.0
    h = hdx * dx
    arr = _make_array("fluid", False, x, y, z, vel[:, 0], vel[:, 1], vel[:, 2], h, rho0 * dx ** 3, rho0)
    return Workload(f"C3_periodic_3d_{n[0]}x{n[1]}x{n[2]}", 3, (0, 0, 0), hi, (True, True, True),
                    kernel, rho0, c0, 7.0, 0.1, 0.01, (0, 0, 0), 0.25 * h / c0, n_steps,
                    SUMMATION, [arr], note="BASELINE.json configs[2]")


def dam_break_3d(dx: float = 0.005, n_steps: int = 50, density_mode: str = CONTINUITY,
                 kernel: str = "cubic", hdx: float = 1.3) -> Workload:
    """C4. Fluid column 0.6x0.6x1.2 (cell-centred) in a 1.6x0.6x1.2 open-top tank, 3 wall layers."""
    nf = (int(round(0.6 / dx)), int(round(0.6 / dx)), int(round(1.2 / dx)))
    fx, fy, fz = _cell_centred(nf, dx, (0.0, 0.0, 0.0))
    sx, sy, sz = tank_3d_open_top(dx, 1.6, 0.6, 1.2, 3)
    rho0 = 1000.0
    c0 = 10.0 * np.sqrt(2 * 9.81 * 1.2)
    h = hdx * dx
    m = rho0 * dx ** 3
    fluid = _make_array("fluid", False, fx, fy, fz, 0.0, 0.0, 0.0, h, m, rho0)
    solid = _make_array("solid", True, sx, sy, sz, 0.0, 0.0, 0.0, h, m, rho0)
    pad = 4 * dx
    lo = (-3 * dx - pad, -3 * dx - pad, -3 * dx - pad)
    hi = (1.6 + 3 * dx + pad, 0.6 + 3 * dx + pad, 1.2 + pad)
    return Workload(f"C4_dam_break_3d_dx{dx:g}", 3, lo, hi, (False, False, False), kernel,
                    rho0, float(c0), 7.0, 0.1, 0.01, (0.0, 0.0, -9.81), 0.125 * h / float(c0),
                    n_steps, density_mode, [fluid, solid], note="BASELINE.json configs[3]")


_C5_CENTRES = np.array([[a, b, c] for a in (0.25, 0.75) for b in (0.25, 0.75) for c in (0.25, 0.75)])


def gaussian_mixture_pdf(pos: np.ndarray, sigma: float = 0.05, f_bg: float = 0.5) -> np.ndarray:
    """Analytic density of the C5 sampling distribution (nearest periodic image of each centre).
    Used only to assign the per-particle smoothing length of the INPUT (h = 1.2 (m/rho)^(1/3))."""
    pdf = np.full(pos.shape[0], f_bg, dtype=np.float64)
    norm = (1.0 - f_bg) / 8.0 / ((2 * np.pi) ** 1.5 * sigma ** 3)
    for c in _C5_CENTRES:
        d = pos - c
        d -= np.rint(d)
        pdf += norm * np.exp(-0.5 * np.einsum("ij,ij->i", d, d) / sigma ** 2)
    return pdf


def gaussian_mixture_3d(N: int = 1 << 24, seed: int = 2, sigma: float = 0.05, f_bg: float = 0.5,
                        hdx: float = 1.2, kernel: str = "wendland_c2", n_steps: int = 10) -> Workload:
    """C5. Periodic unit cube; each particle is uniform with probability f_bg, else drawn from one of
    8 isotropic Gaussians (sigma) centred at {1/4,3/4}^3; m = 1/N; rho_i = analytic mixture density;
    h_i = hdx (m/rho_i)^(1/3); velocities U[-1,1]^3.  No position update (density + momentum only)."""
    rng = np.random.default_rng(seed)
    is_bg = rng.random(N) < f_bg
    which = rng.integers(0, 8, size=N)
    pos = rng.random((N, 3))
    gauss = rng.standard_normal((N, 3)) * sigma
    vel = rng.uniform(-1.0, 1.0, size=(N, 3))
    pos = np.where(is_bg[:, None], pos, _C5_CENTRES[which] + gauss)
    del gauss, which, is_bg
    x = _wrap32(pos[:, 0], 0.0, 1.0)
    y = _wrap32(pos[:, 1], 0.0, 1.0)
    z = _wrap32(pos[:, 2], 0.0, 1.0)
    p32 = np.stack([x, y, z], axis=1).astype(np.float64)
    pdf = np.empty(N)
    step = 1 << 21
    for s in range(0, N, step):
        pdf[s:s + step] = gaussian_mixture_pdf(p32[s:s + step], sigma, f_bg)
    del p32, pos
    m = 1.0 / N
    rho = pdf                      # m * N * pdf
    h = hdx * (m / rho) ** (1.0 / 3.0)
    rho0, c0 = 1.0, 10.0
    arr = _make_array("fluid", False, x, y, z, vel[:, 0], vel[:, 1], vel[:, 2], h, m, rho)
    hmin = float(arr.h.min())
    return Workload(f"C5_gaussian_mixture_3d_{N}", 3, (0, 0, 0), (1, 1, 1), (True, True, True),
                    kernel, rho0, c0, 7.0, 0.1, 0.01, (0, 0, 0), 0.25 * hmin / c0, n_steps,
                    SUMMATION, [arr], note="BASELINE.json configs[4]; no position update")


# --------------------------------------------------------------------------------------------
# small cases for brute-force / edge tests
# --------------------------------------------------------------------------------------------
def random_box(n: int, dim: int, periodic: bool, seed: int, kernel: str = "cubic",
               variable_h: bool = False, h_mean: Optional[float] = None, two_arrays: bool = False,
               box: Sequence[float] = (1.0, 1.0, 1.0), density_mode: str = SUMMATION,
               g=(0.0, 0.0, 0.0)) -> Workload:
    """Uniform random points (worst case for cells: empty cells, ragged occupancy, near-coincident pairs)."""
    rng = np.random.default_rng(seed)
    box = tuple(float(b) for b in box)
    vol = float(np.prod(box[:dim]))
    if h_mean is None:
        h_mean = 1.3 * (vol / max(n, 1)) ** (1.0 / dim)
    pos = rng.random((n, 3)) * np.array(box)
    vel = rng.uniform(-1.0, 1.0, size=(n, 3))
    if dim == 2:
        pos[:, 2] = 0.0
        vel[:, 2] = 0.0
    h = h_mean * (rng.uniform(0.7, 1.4, size=n) if variable_h else np.ones(n))
    rho0 = 1.0
    m = rho0 * vol / max(n, 1) * rng.uniform(0.8, 1.2, size=n)
    rho = rho0 * rng.uniform(0.95, 1.05, size=n)
    per = (periodic, periodic, periodic and dim == 3)
    xs = [(_wrap32(pos[:, k], 0.0, box[k]) if per[k] else _f32(pos[:, k])) for k in range(3)]
    if periodic:
        lo, hi = (0.0, 0.0, 0.0), box
    else:
        pad = 0.05
        lo = (-pad, -pad, -pad if dim == 3 else 0.0)
        hi = (box[0] + pad, box[1] + pad, box[2] + pad if dim == 3 else 1.0)
    if two_arrays:
        cut = (2 * n) // 3
        idx = [np.arange(0, cut), np.arange(cut, n)]
        names, fixed = ["fluid", "solid"], [False, True]
    else:
        idx, names, fixed = [np.arange(n)], ["fluid"], [False]
    arrays = []
    for ii, nm, fx in zip(idx, names, fixed):
        vv = vel[ii] * (0.0 if fx else 1.0)
        arrays.append(_make_array(nm, fx, xs[0][ii], xs[1][ii], xs[2][ii], vv[:, 0], vv[:, 1], vv[:, 2],
                                  h[ii], m[ii], rho[ii]))
    c0 = 10.0
    return Workload(f"random_{dim}d_n{n}_{'per' if periodic else 'open'}_s{seed}", dim, lo, hi, per, kernel,
                    rho0, c0, 7.0, 0.1, 0.01, tuple(g), 0.25 * float(h.min() if n else h_mean) / c0, 1,
                    density_mode, arrays)


def lattice(n: Sequence[int], dim: int, hdx: float, kernel: str, rho0: float = 1.0) -> Workload:
    """Unjittered periodic cell-centred lattice with dx = 1/n[0] (exactly representable for powers of 2)."""
    n = tuple(int(v) for v in n[:dim])
    dx = 1.0 / n[0]
    coords = _cell_centred(n, dx, (0.0,) * dim)
    while len(coords) < 3:
        coords.append(np.zeros_like(coords[0]))
    hi = tuple(n[k] * dx if k < dim else 1.0 for k in range(3))
    per = tuple(k < dim for k in range(3))
    arr = _make_array("fluid", False, coords[0], coords[1], coords[2], 0.0, 0.0, 0.0,
                      hdx * dx, rho0 * dx ** dim, rho0)
    return Workload(f"lattice_{dim}d_{'x'.join(map(str, n))}_{kernel}", dim, (0, 0, 0), hi, per, kernel,
                    rho0, 10.0, 7.0, 0.1, 0.01, (0, 0, 0), 0.25 * hdx * dx / 10.0, 1, SUMMATION, [arr])


def by_name(name: str, **kw) -> Workload:
    table = {"C1": taylor_green_2d, "C2": dam_break_2d, "C3": periodic_box_3d,
             "C4": dam_break_3d, "C5": gaussian_mixture_3d}
    return table[name](**kw)
