"""Pins for the oracle's predictor-corrector step (eqs. 12-14; R10/R11).
Closed forms and invariants: constant acceleration is integrated exactly; the kick-drift-kick form is
time reversible and second order; fixed arrays do not move; the periodic wrap keeps x in [lo,hi)."""
import numpy as np
import pytest


def test_free_fall_is_an_exact_parabola(O, WL):
    """No neighbours + gravity: eqs. 12-14 give x0 + u0 t + g t^2/2 for ANY dt (KDK is exact for constant a)."""
    wl = WL.random_box(n=3, dim=2, periodic=False, seed=1, g=(0.0, -9.81, 0.0))
    st = O.State(wl); A = st.arrays[0]
    A["x"][:] = [0.1, 0.5, 0.9]; A["y"][:] = [0.9, 0.5, 0.1]; A["h"][:] = 1e-3
    A["u"][:] = [1.0, 0.0, -1.0]; A["v"][:] = [0.0, 2.0, 0.5]
    x0, y0, u0, v0 = (A[k].copy() for k in "xyuv")
    dt, n = 0.013, 7
    for _ in range(n):
        O.pc_step(wl, st, dt, "summation")
    t = n * dt
    assert np.allclose(A["x"], x0 + u0 * t, rtol=0, atol=1e-14)
    assert np.allclose(A["y"], y0 + v0 * t - 0.5 * 9.81 * t * t, rtol=0, atol=1e-13)
    assert np.allclose(A["v"], v0 - 9.81 * t, rtol=0, atol=1e-13)
    assert np.array_equal(A["u"], u0)


def test_single_step_is_eqs_12_to_14(O, WL):
    """One step from a state with known a^n: recompute eqs. 12-14 by hand around the oracle's own F."""
    wl = WL.random_box(n=400, dim=2, periodic=True, seed=41, variable_h=True)
    st = O.State(wl)
    O.evaluate(wl, st, "summation")
    s0 = st.copy(); A0 = s0.arrays[0]
    dt = wl.dt
    O.pc_step(wl, st, dt, "summation")
    A1 = st.arrays[0]
    uh = A0["u"] + 0.5 * dt * A0["au"]                        # (12)
    x1 = A0["x"] + dt * uh                                    # (13)
    x1 = np.where(x1 >= 1.0, x1 - 1.0, np.where(x1 < 0.0, x1 + 1.0, x1))
    assert np.array_equal(A1["x"], x1)
    assert np.allclose(A1["u"], uh + 0.5 * dt * A1["au"], rtol=0, atol=1e-15)   # (14) with a^{n+1}
    assert (A1["x"] >= 0).all() and (A1["x"] < 1.0).all()
    # a^{n+1} was evaluated at (x^{n+1}, u^{n+1/2}) (R10)
    chk = s0.copy(); C = chk.arrays[0]
    C["x"] = x1; C["y"] = A1["y"]; C["u"] = uh; C["v"] = A0["v"] + 0.5 * dt * A0["av"]
    O.evaluate(wl, chk, "summation")
    assert np.allclose(chk.arrays[0]["au"], A1["au"], rtol=0, atol=1e-12 * np.abs(A1["au"]).max())


def test_time_reversibility(O, WL):
    """KDK with alpha = 0 in summation mode: a step dt followed by a step -dt returns to the start."""
    wl = WL.random_box(n=500, dim=2, periodic=True, seed=42)
    wl.alpha = 0.0
    st = O.State(wl)
    A = st.arrays[0]
    A["u"] *= 0.05; A["v"] *= 0.05
    s0 = st.copy()
    dt = wl.dt
    for _ in range(3):
        O.pc_step(wl, st, dt, "summation")
    moved = np.abs(st.arrays[0]["x"] - s0.arrays[0]["x"]).max()
    for _ in range(3):
        O.pc_step(wl, st, -dt, "summation")
    for k in "xyuv":
        assert np.abs(st.arrays[0][k] - s0.arrays[0][k]).max() < 1e-9 * max(1.0, moved / dt)
    assert moved > 1e-6


def test_second_order_convergence(O, WL):
    """Halving dt divides the error against a fine reference by about 4 (2nd-order scheme, L146)."""
    wl = WL.lattice((16, 16), 2, 1.3, "cubic")
    wl.alpha = 0.0
    base = O.State(wl); A = base.arrays[0]
    A["u"] = 0.2 * np.sin(2 * np.pi * A["y"]); A["v"] = 0.2 * np.sin(2 * np.pi * A["x"])
    T = 16 * wl.dt

    def run(nsteps):
        st = base.copy()
        for _ in range(nsteps):
            O.pc_step(wl, st, T / nsteps, "summation")
        return np.concatenate([st.arrays[0]["u"], st.arrays[0]["v"]])
    ref = run(128)
    e1 = np.abs(run(8) - ref).max()
    e2 = np.abs(run(16) - ref).max()
    assert 3.0 < e1 / e2 < 5.5


def test_fixed_arrays_and_continuity_mode(O, WL):
    """L142: the tank particles are fixed, but the continuity equation is solved on them and p set by the EOS."""
    wl = WL.dam_break_2d(dx=0.05)
    st = O.State(wl)
    S0 = {k: st.arrays[1][k].copy() for k in "xyuv"}
    for _ in range(5):
        O.pc_step(wl, st, wl.dt, "continuity")
    F, S = st.arrays
    for k in "xyuv":
        assert np.array_equal(S[k], S0[k])
    assert (F["v"] < 0).all()                                 # everything is falling
    assert F["v"].min() == pytest.approx(-9.81 * 5 * wl.dt, rel=0.3)
    assert S["rho"].max() > wl.rho0 and (S["p"][S["rho"] > wl.rho0] > 0).all()
    assert np.abs(F["rho"] / wl.rho0 - 1).max() < 0.02        # weakly compressible


def test_continuity_mode_step_written_out(O, WL):
    """Continuity-mode predictor-corrector step written out by hand around the oracle's own F (eqs. 12-14
    L148-152 for u, x; L142 "the continuity equation is solved on the tank particles too"; R11: rho is
    stepped like u):   rho^{n+1/2} = rho^n + dt/2 arho^n ;  F evaluated at (x^{n+1}, u^{n+1/2}, rho^{n+1/2}) ;
    rho^{n+1} = rho^{n+1/2} + dt/2 arho^{n+1}, on BOTH arrays, bit-equal.  A full-dt kick, a dropped kick or a
    kick with the wrong arho fails this."""
    wl = WL.dam_break_2d(dx=0.05)
    rng = np.random.default_rng(11)
    wl.arrays[0].u[:] = rng.uniform(-0.3, 0.3, wl.arrays[0].n).astype(np.float32)
    wl.arrays[0].v[:] = rng.uniform(-0.3, 0.3, wl.arrays[0].n).astype(np.float32)
    dt = wl.dt
    st = O.State(wl)
    O.evaluate(wl, st, "continuity")                       # a^n, arho^n
    s0 = st.copy()
    O.pc_step(wl, st, dt, "continuity")
    # the half-step state, by hand
    mid = s0.copy()
    F0, S0 = s0.arrays
    Fm, Sm = mid.arrays
    Fm["u"] = F0["u"] + 0.5 * dt * F0["au"]; Fm["v"] = F0["v"] + 0.5 * dt * F0["av"]          # (12)
    Fm["x"] = F0["x"] + dt * Fm["u"]; Fm["y"] = F0["y"] + dt * Fm["v"]                         # (13)
    Fm["rho"] = F0["rho"] + 0.5 * dt * F0["arho"]
    Sm["rho"] = S0["rho"] + 0.5 * dt * S0["arho"]
    O.evaluate(wl, mid, "continuity")                      # a^{n+1}, arho^{n+1} from (x^{n+1}, u^{n+1/2}, rho^{n+1/2})
    F1, S1 = st.arrays
    assert np.array_equal(F1["x"], Fm["x"]) and np.array_equal(F1["y"], Fm["y"])
    assert np.array_equal(F1["u"], Fm["u"] + 0.5 * dt * Fm["au"])                              # (14)
    assert np.array_equal(F1["v"], Fm["v"] + 0.5 * dt * Fm["av"])
    assert np.array_equal(F1["rho"], Fm["rho"] + 0.5 * dt * Fm["arho"])
    assert np.array_equal(S1["rho"], Sm["rho"] + 0.5 * dt * Sm["arho"])
    assert np.array_equal(S1["x"], S0["x"]) and np.array_equal(S1["u"], S0["u"])               # fixed array (L142)
    # the kicks are not degenerate: both halves move rho, and differently (so a doubled first kick is told apart)
    k1 = 0.5 * dt * F0["arho"]; k2 = 0.5 * dt * Fm["arho"]
    assert np.abs(k1).max() > 1e-9 * wl.rho0 and np.abs(k2 - k1).max() > 1e-3 * np.abs(k1).max()
    assert np.abs(0.5 * dt * S0["arho"]).max() > 1e-9 * wl.rho0
    # p of the result is the EOS of the rho the evaluation saw (group order L364-378): rho^{n+1/2}
    assert np.array_equal(F1["p"], O.eos(wl, Fm["rho"])) and np.array_equal(S1["p"], O.eos(wl, Sm["rho"]))


def test_continuity_mode_rho_follows_the_closed_form_of_a_uniform_compression(O, WL):
    """A pin with a value the mathematics fixes: particles on a periodic lattice with the velocity field u = -c (x - 1/2)
    frozen in time (fixed array: x,u never change) have a constant arho = rho div-free term  sum_j m_j u_ij . grad W
    ~ +c rho0 (eq.7, tr A = -c), so n continuity steps give rho_n = rho_0 + n dt arho exactly (two half kicks
    per step = one full kick), and arho is within the kernel-sum error of c rho0 d."""
    wl = WL.lattice((16, 16), 2, 1.3, "cubic")
    A = wl.arrays[0]
    c = 0.7
    A.u[:] = (-c * (A.x - 0.5)).astype(np.float32); A.v[:] = (-c * (A.y - 0.5)).astype(np.float32)
    A.fixed = True
    wl.arho_sources = [[0]]
    st = O.State(wl)
    O.evaluate(wl, st, "continuity")
    arho0 = st.arrays[0]["arho"].copy(); rho0 = st.arrays[0]["rho"].copy()
    n = 4
    for _ in range(n):
        O.pc_step(wl, st, wl.dt, "continuity")
    assert np.allclose(st.arrays[0]["rho"], rho0 + n * wl.dt * arho0, rtol=0, atol=1e-12 * wl.rho0)
    inner = (np.abs(A.x - 0.5) < 0.2) & (np.abs(A.y - 0.5) < 0.2)
    assert np.allclose(arho0[inner], 2 * c * wl.rho0, rtol=2e-2)     # measured 1.06 % at h = 1.3 dx


def test_no_move_option(O, WL):
    wl = WL.random_box(n=300, dim=3, periodic=True, seed=43, variable_h=True)
    st = O.State(wl); x0 = st.arrays[0]["x"].copy(); u0 = st.arrays[0]["u"].copy()
    O.pc_step(wl, st, wl.dt, "summation", move=False)
    assert np.array_equal(st.arrays[0]["x"], x0) and not np.array_equal(st.arrays[0]["u"], u0)


def test_taylor_green_run_follows_the_analytic_decay_trend(O, WL):
    """north_star pin: the 2-D Taylor-Green state decays like exp(b t), b = -8 pi^2 nu.  With
    Monaghan's viscosity the continuum-limit nu of the scheme is alpha h c0 / 8 (all pairs; R9), so the
    kinetic energy of a run of the C1 state must fall like exp(2 b t) with b near -8 pi^2 alpha h c0 / 8 = -0.20/s.
    The first 0.1 s is an acoustic transient (rho starts uniform: O(Mach^2) = 1e-2 sloshing), so the rate is
    fitted over t in [0.1, 0.6]: 1,200 steps of the oracle (4 s)."""
    wl = WL.taylor_green_2d()
    st = O.State(wl)
    m = st.arrays[0]["m"]
    n = 1200
    ke = np.zeros(n + 1)
    for s in range(n + 1):
        A = st.arrays[0]
        ke[s] = 0.5 * float((m * (A["u"] ** 2 + A["v"] ** 2)).sum())
        if s < n:
            O.pc_step(wl, st, wl.dt, "summation")
    t = np.arange(n + 1) * wl.dt
    sel = t >= 0.1
    b = np.polyfit(t[sel], np.log(ke[sel] / ke[0]), 1)[0] / 2.0
    h = float(wl.arrays[0].h[0])
    b_ref = -8.0 * np.pi ** 2 * wl.alpha * h * wl.c0 / 8.0
    assert 0.6 * abs(b_ref) <= -b <= 1.5 * abs(b_ref), (b, b_ref)
    assert ke[-1] < 0.85 * ke[0] and np.all(ke[sel] < 1.001 * ke[np.argmax(sel)])      # it decays, monotonically on the fit window
    # the flow stays a Taylor-Green vortex: the velocities still point along the analytic field (L649-652) at the
    # particles' current positions
    A = st.arrays[0]
    ua = -np.cos(2 * np.pi * A["x"]) * np.sin(2 * np.pi * A["y"])
    va = np.sin(2 * np.pi * A["x"]) * np.cos(2 * np.pi * A["y"])
    corr = float((A["u"] * ua + A["v"] * va).sum() / np.sqrt((A["u"] ** 2 + A["v"] ** 2).sum() * (ua ** 2 + va ** 2).sum()))
    assert corr > 0.95
