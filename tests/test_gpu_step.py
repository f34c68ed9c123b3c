"""-m gpu parity of sph_pc_step (eqs. 12-14) against the oracle's step, one step from the same state
(R15: float32 trajectories drift from float64 ones, so multi-step runs are gated by
"one more step from the GPU's own state", with the GPU's a^n handed to the oracle)."""
import numpy as np
import pytest

from gpu_helpers import TOL, assert_close, make_ctx, min_image_diff

pytestmark = pytest.mark.gpu


def _compare_state(wl, ctx, st, tag, tol=TOL):
    for d, A in enumerate(st.arrays):
        if wl.arrays[d].n == 0:
            continue
        out = {k: v.cpu().numpy() for k, v in ctx.sync_state(d).items()}
        for k, axis in (("x", 0), ("y", 1), ("z", 2)):
            if axis >= wl.dim:
                continue
            diff = min_image_diff(out[k], A[k], wl.lo[axis], wl.hi[axis], wl.periodic[axis])
            scale = max(abs(wl.lo[axis]), abs(wl.hi[axis]))
            assert np.abs(diff).max() <= tol * scale, f"{tag} {k}[{d}]: {np.abs(diff).max() / scale:.3e}"
        vmax = max(np.abs(A["u"]).max(), np.abs(A["v"]).max(), np.abs(A["w"]).max())
        for k, axis in (("u", 0), ("v", 1), ("w", 2)):
            if axis >= wl.dim or vmax == 0:
                continue
            err = np.abs(out[k].astype(np.float64) - A[k]).max() / vmax
            assert err <= tol, f"{tag} {k}[{d}]: {err:.3e} of max|u|"
        assert_close(out["rho"], A["rho"], f"{tag} rho[{d}]", tol)


def _step_cases(WL):
    return [
        ("C1", WL.taylor_green_2d(), "summation"),
        ("3d_per", WL.periodic_box_3d((16, 16, 16), seed=1), "summation"),
        ("3d_varh", WL.random_box(n=4000, dim=3, periodic=True, seed=61, kernel="cubic", variable_h=True), "summation"),
        ("dam2d_cont", WL.dam_break_2d(dx=0.04), "continuity"),
        ("dam2d_summ", WL.dam_break_2d(dx=0.04), "summation"),
        ("dam3d_cont", WL.dam_break_3d(dx=0.05), "continuity"),
    ]


STEP_IDS = ["C1", "3d_per", "3d_varh", "dam2d_cont", "dam2d_summ", "dam3d_cont"]


@pytest.mark.parametrize("idx", range(len(STEP_IDS)), ids=STEP_IDS)
def test_one_step_from_the_same_state(O, WL, idx):
    """a^0 evaluation + one full step (what BASELINE config 1 calls 'one step')."""
    _, wl, mode = _step_cases(WL)[idx]
    ctx, _ = make_ctx(wl)
    ctx.pc_step(wl.dt, 1, mode)
    st = O.State(wl)
    O.pc_step(wl, st, wl.dt, mode)
    _compare_state(wl, ctx, st, "step1")
    ctx.synchronize()
    ctx.close()


def test_restart_from_synced_state_continues_the_run(WL):
    """sph_sync_state (incl. ax..arho) -> sph_nnps_build with those accelerations -> the next step reuses a^n
    (no re-evaluation): two steps in one call == step, sync out, rebuild, step."""
    for wl, mode in ((WL.periodic_box_3d((16, 16, 16), seed=3), "summation"), (WL.dam_break_2d(dx=0.04), "continuity")):
        ctx, _ = make_ctx(wl)
        ctx.pc_step(wl.dt, 2, mode)
        ref = [ctx.sync_state(d) for d in range(len(wl.arrays))]
        ctx2, arrays = make_ctx(wl)
        ctx2.pc_step(wl.dt, 1, mode)
        keys = ("x", "y", "z", "u", "v", "w", "rho", "p", "ax", "ay", "az", "arho")
        mid = [ctx2.sync_state(d, fields=keys) for d in range(len(wl.arrays))]
        l0 = ctx2.get_stats().kernel_launches
        for d, a in enumerate(arrays):
            mid[d]["h"], mid[d]["m"] = a["h"], a["m"]
        ctx2.nnps_build(mid, [a.fixed for a in wl.arrays])
        ctx2.pc_step(wl.dt, 1, mode)
        for d in range(len(wl.arrays)):
            got = ctx2.sync_state(d)
            for k in ("x", "y", "u", "v", "rho"):
                w_ = ref[d][k].cpu().numpy().astype(np.float64); g_ = got[k].cpu().numpy().astype(np.float64)
                scale = max(np.abs(w_).max(), 1e-30)
                assert np.abs(g_ - w_).max() <= TOL * scale, f"{wl.name} {k}[{d}]"
        ctx.close(); ctx2.close()


def test_record_pool_overflow_falls_back_to_searching(WL):
    """A record pool too small for the density pass's hit masks: the warps that did not fit search again in the
    momentum pass (no error, same pairs, same result as with the default pool or with no pool at all)."""
    wl = WL.periodic_box_3d((24, 24, 24), seed=5)
    res = []
    for slots in (0, 2, -1):                       # default pool, a pool of 2 rows per warp, no pool
        ctx, _ = make_ctx(wl, nlist_slots=slots)
        ctx.pc_step(wl.dt, 2, "summation")
        ctx.synchronize()
        s = ctx.get_stats()
        out = {k: v.cpu().numpy() for k, v in ctx.sync_state(0).items()}
        res.append((s.pairs_density, s.pairs_accel, s.nlist_fallback_warps, s.candidates_accel, out))
        ctx.close()
    (pd0, pa0, fb0, ca0, o0), (pd1, pa1, fb1, ca1, o1), (pd2, pa2, fb2, ca2, o2) = res
    assert pd0 == pa0 == pd1 == pa1 == pd2 == pa2
    assert fb0 == 0 and ca0 == 0                    # everything replayed
    assert fb1 > 0 and 0 < ca1 <= ca2               # some warps searched again
    assert fb2 == 0 and ca2 > 0                     # no pool: the whole momentum pass searched
    for k in ("x", "u", "v", "w", "rho"):
        for o in (o1, o2):
            scale = np.abs(o0[k]).max()
            assert np.abs(o[k].astype(np.float64) - o0[k]).max() <= 2e-6 * scale, k


@pytest.mark.parametrize("name", ["dam2d_euler_laminar", "3d_per_euler_laminar", "3d_varh_pc_laminar"])
def test_laminar_viscosity_and_euler_steps(O, WL, name):
    """eq.10 in the pair loop (nu > 0) and the forward-Euler integrator of the paper's worked example (L335,
    Fig.2): a^0 + ONE step on the GPU == the oracle's, from the same state (steps from an evolved state:
    test_gpu_evolved.py)."""
    if name == "dam2d_euler_laminar":
        wl, mode = WL.dam_break_2d(dx=0.04), "continuity"
        wl.integrator, wl.nu = "euler", 1.0e-3
        wl.arrays[0].u[:] = np.random.default_rng(9).uniform(-0.5, 0.5, wl.arrays[0].n).astype(np.float32)
    elif name == "3d_per_euler_laminar":
        wl, mode = WL.periodic_box_3d((16, 16, 16), seed=4), "summation"
        wl.integrator, wl.nu = "euler", 5.0e-3
    else:
        wl, mode = WL.random_box(n=4000, dim=3, periodic=True, seed=62, kernel="cubic", variable_h=True), "summation"
        wl.nu = 2.0e-3
    step = O.euler_step if wl.integrator == "euler" else O.pc_step
    ctx, _ = make_ctx(wl)
    ctx.pc_step(wl.dt, 1, mode)
    st = O.State(wl)
    step(wl, st, wl.dt, mode)
    _compare_state(wl, ctx, st, name + " step1")
    # the viscous term must be there: the same step with nu = 0 differs by far more than the tolerance
    nu = wl.nu; wl.nu = 0.0
    st0 = O.State(wl); step(wl, st0, wl.dt, mode); wl.nu = nu
    d = np.abs(st0.arrays[0]["u"] - st.arrays[0]["u"]).max() / np.abs(st.arrays[0]["u"]).max()
    assert d > 20 * TOL, f"nu has no visible effect in this case ({d:.2e})"
    ctx.synchronize()
    ctx.close()


def test_dense_cells_span_several_record_blocks(O, WL):
    """~100 particles per cell: a warp's candidate stream is > 30 batches, so the mask store is drained and
    recorded in several blocks per warp and the momentum pass replays a chain of blocks.  Same pairs and the same
    step as with no record pool, and parity with the oracle."""
    wl = WL.random_box(n=12000, dim=3, periodic=True, seed=71, kernel="cubic", h_mean=0.1)
    outs = []
    for slots in (0, -1):
        ctx, _ = make_ctx(wl, nlist_slots=slots)
        ctx.pc_step(wl.dt, 1, "summation")
        ctx.synchronize()
        s = ctx.get_stats()
        outs.append((s, {k: v.cpu().numpy() for k, v in ctx.sync_state(0).items()}))
        if slots == 0:
            assert s.used_rows == 1 and s.nlist_fallback_warps == 0
            assert s.nlist_rows_used > 2 * 32 * ((wl.arrays[0].n + 31) // 32)      # > 2 blocks of 30 per warp
            st = O.State(wl)
            O.pc_step(wl, st, wl.dt, "summation")
            _compare_state(wl, ctx, st, "dense step1")
        ctx.close()
    (s0, o0), (s1, o1) = outs
    assert s0.pairs_density == s0.pairs_accel == s1.pairs_density == s1.pairs_accel
    for k in ("x", "u", "v", "w", "rho"):
        assert np.abs(o1[k].astype(np.float64) - o0[k]).max() <= 2e-6 * np.abs(o0[k]).max(), k


def test_taylor_green_run_decays_like_the_oracle(O, WL):
    """Multi-step behaviour (trajectories are not gated element-wise, R15): 1,200 steps of C1 on the GPU
    lose kinetic energy at the same fitted rate as the fp64 oracle's run, which is pinned to the analytic
    Taylor-Green decay (test_oracle_step.py)."""
    wl = WL.taylor_green_2d()
    m = wl.arrays[0].m.astype(np.float64)
    n, every = 1200, 50

    def fit(ke):
        t = np.arange(len(ke)) * every * wl.dt
        sel = t >= 0.1
        return np.polyfit(t[sel], np.log(ke[sel] / ke[0]), 1)[0] / 2.0

    ctx, _ = make_ctx(wl)
    ke_g = []
    for s in range(n // every + 1):
        out = ctx.sync_state(0, fields=("u", "v"))
        ke_g.append(0.5 * float((m * (out["u"].cpu().numpy().astype(np.float64) ** 2 + out["v"].cpu().numpy().astype(np.float64) ** 2)).sum()))
        if s < n // every:
            ctx.pc_step(wl.dt, every, "summation")
    ctx.synchronize()
    ctx.close()
    st = O.State(wl)
    ke_o = []
    for s in range(n + 1):
        if s % every == 0:
            A = st.arrays[0]
            ke_o.append(0.5 * float((m * (A["u"] ** 2 + A["v"] ** 2)).sum()))
        if s < n:
            O.pc_step(wl, st, wl.dt, "summation")
    bg, bo = fit(np.array(ke_g)), fit(np.array(ke_o))
    assert abs(bg - bo) <= 0.05 * abs(bo), (bg, bo)
    assert abs(ke_g[-1] / ke_g[0] - ke_o[-1] / ke_o[0]) < 5e-3
