"""Pins of the oracle's laminar viscosity (eq.10) and forward-Euler step (L335, Fig.2) against
what the paper and the mathematics fix: a two-particle case written out by hand from eq.10, antisymmetry (total
momentum), dissipation, Galilean invariance, the continuum limit nu * laplacian(u) on a sinusoidal shear flow, and
closed forms of the Euler step (free fall, one step written out)."""
import numpy as np
import pytest


def _accel_lam_only(O, wl, st, d, srcs, nu):
    """eq.10 contribution alone: accel with nu minus accel without (alpha = 0, p = 0 make the rest vanish too)."""
    a1 = O.accel(wl, st, d, srcs, pred32=False, alpha=0.0, gravity=False, nu=nu)
    a0 = O.accel(wl, st, d, srcs, pred32=False, alpha=0.0, gravity=False, nu=0.0)
    return {k: a1[k] - a0[k] for k in ("au", "av", "aw")}, a1


def test_two_particles_by_hand(O, WL):
    wl = WL.random_box(n=2, dim=2, periodic=False, seed=1, kernel="cubic", h_mean=0.1)
    A = wl.arrays[0]
    A.x[:] = [0.40, 0.47]; A.y[:] = [0.50, 0.52]; A.h[:] = 0.1
    A.u[:] = [0.3, -0.2]; A.v[:] = [0.1, 0.4]; A.m[:] = [2.0e-3, 3.0e-3]; A.rho[:] = [1.0, 1.1]
    st = O.State(wl)
    nu, eta = 0.05, 0.01
    wl.eta = eta
    lam, _ = _accel_lam_only(O, wl, st, 0, [0], nu)
    x = A.x.astype(np.float64); y = A.y.astype(np.float64); h = float(A.h[0])
    dx, dy = x[0] - x[1], y[0] - y[1]
    r = np.hypot(dx, dy)
    dwdr = O.dWdr("cubic", 2, r, h)
    rho = A.rho.astype(np.float64); m = A.m.astype(np.float64)
    c = 4 * nu / (rho[0] + rho[1]) * (dwdr * r) / (r * r + eta * h * h)     # eq.10 with r.gradW = dW/dr r
    uij = np.float64(A.u[0]) - np.float64(A.u[1]); vij = np.float64(A.v[0]) - np.float64(A.v[1])
    assert lam["au"][0] == pytest.approx(m[1] * c * uij, rel=1e-12)
    assert lam["av"][0] == pytest.approx(m[1] * c * vij, rel=1e-12)
    assert lam["au"][1] == pytest.approx(-m[0] * c * uij, rel=1e-12)          # u_ji = -u_ij, the rest is symmetric


@pytest.mark.parametrize("dim,varh", [(2, False), (3, True)])
def test_antisymmetric_dissipative_galilean(O, WL, dim, varh):
    wl = WL.random_box(n=500, dim=dim, periodic=True, seed=7, kernel="wendland_c2", variable_h=varh)
    st = O.State(wl)
    lam, a1 = _accel_lam_only(O, wl, st, 0, [0], 0.02)
    m = st.arrays[0]["m"]
    for k in ("au", "av", "aw"):
        assert abs((m * lam[k]).sum()) <= 1e-13 * (m * np.abs(lam[k])).sum() + 1e-300     # total momentum
    assert (m * a1["lam_power"]).sum() < 0                                                 # sum m u.a_visc < 0
    st2 = O.State(wl)
    for k, c in (("u", 0.7), ("v", -1.3), ("w", 0.4)):
        st2.arrays[0][k] = st2.arrays[0][k] + c
    lam2, _ = _accel_lam_only(O, wl, st2, 0, [0], 0.02)
    for k in ("au", "av", "aw"):
        assert np.allclose(lam2[k], lam[k], rtol=0, atol=1e-12 * np.abs(lam[k]).max())


def test_continuum_limit_is_nu_laplacian(O, WL):
    """u = sin(2 pi y) ex on a 2-D periodic lattice: eq.10 -> nu d2u/dy2 = -nu (2 pi)^2 sin(2 pi y) (Morris-type
    operator [30]); the kernel-sum error at h = 1.3 dx, 64 x 64 is a few per cent."""
    wl = WL.lattice((64, 64), 2, 1.3, "cubic")
    A = wl.arrays[0]
    A.u[:] = np.sin(2 * np.pi * A.y.astype(np.float64)).astype(np.float32); A.v[:] = 0
    st = O.State(wl)
    nu = 0.01
    lam, _ = _accel_lam_only(O, wl, st, 0, [0], nu)
    want = -nu * (2 * np.pi) ** 2 * np.sin(2 * np.pi * st.arrays[0]["y"])
    assert np.abs(lam["au"] - want).max() <= 0.05 * np.abs(want).max()
    assert np.abs(lam["av"]).max() <= 1e-10 * np.abs(want).max()


def test_euler_free_fall_and_one_step_written_out(O, WL):
    # no neighbours (h tiny), gravity: x_n = x0 + n dt u0 + g dt^2 n(n-1)/2 exactly for forward Euler
    wl = WL.random_box(n=5, dim=2, periodic=False, seed=3, kernel="cubic", h_mean=1e-4, box=(50.0, 50.0, 1.0),
                       g=(0.0, -9.81, 0.0))
    st = O.State(wl)
    y0 = st.arrays[0]["y"].copy(); v0 = st.arrays[0]["v"].copy()
    dt, n = 1e-3, 7
    for _ in range(n):
        O.euler_step(wl, st, dt, "summation")
    assert np.allclose(st.arrays[0]["y"], y0 + n * dt * v0 - 9.81 * dt * dt * n * (n - 1) / 2, rtol=0, atol=1e-13)
    assert np.allclose(st.arrays[0]["v"], v0 - 9.81 * n * dt, rtol=0, atol=1e-13)
    # one step written out: x1 = x0 + dt u0 ; u1 = u0 + dt a(x0,u0) ; rho1 = rho0 + dt arho0 (continuity)
    wl = WL.dam_break_2d(dx=0.05)
    rng = np.random.default_rng(5)
    wl.arrays[0].u[:] = rng.uniform(-0.3, 0.3, wl.arrays[0].n).astype(np.float32)
    st = O.State(wl); ref = O.State(wl)
    O.evaluate(wl, ref, "continuity")
    O.euler_step(wl, st, wl.dt, "continuity")
    F, R = st.arrays[0], ref.arrays[0]
    assert np.array_equal(F["x"], R["x"] + wl.dt * R["u"])
    assert np.array_equal(F["u"], R["u"] + wl.dt * R["au"])
    assert np.array_equal(F["rho"], R["rho"] + wl.dt * R["arho"])
    S, RS = st.arrays[1], ref.arrays[1]
    assert np.array_equal(S["x"], RS["x"]) and np.array_equal(S["rho"], RS["rho"] + wl.dt * RS["arho"])
