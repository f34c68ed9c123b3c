"""-m gpu parity from an EVOLVED state (R15): after N steps on the GPU the particles
have left their lattice, cells are ragged and the sorted order has been rebuilt N times -- the state bench.py times.
At steps {10, 100} the GPU state (x, u, rho, p AND the accelerations a^n, arho^n of its last evaluation) is copied
out, the fp64 oracle takes ONE step from it, the GPU takes its next step, and x, u, rho are compared at 1e-5.
The 10- and 100-step runs go through the captured two-step CUDA graph of sph_pc_step (n_steps - 1 >= 8), so this
is also the parity gate of that path.  Other tests of the module: accelerations of arrays that are no destination
(stale rows), a one-cell-thick non-periodic axis next to a periodic one, forced level counts."""
import numpy as np
import pytest

from gpu_helpers import TOL, assert_close, make_ctx, mask_of, min_image_diff

pytestmark = pytest.mark.gpu

KEYS = ("x", "y", "z", "u", "v", "w", "rho", "p", "ax", "ay", "az", "arho")


def _oracle_state_from_gpu(O, wl, ctx):
    """oracle State holding the GPU's float32 state and its a^n (no re-evaluation: R10/R15)"""
    st = O.State(wl)
    for d, A in enumerate(st.arrays):
        if wl.arrays[d].n == 0:
            continue
        out = {k: v.cpu().numpy().astype(np.float64) for k, v in ctx.sync_state(d, fields=KEYS).items()}
        for k in ("x", "y", "z", "u", "v", "w", "rho", "p"):
            if k in out:
                A[k] = out[k]
        A["au"], A["av"] = out["ax"], out["ay"]
        A["aw"] = out["az"] if "az" in out else np.zeros_like(out["ax"])
        A["arho"] = out["arho"]
    st.have_accel = True
    return st


def _compare(wl, ctx, st, tag, dt):
    """x, rho: 1e-5 of the per-property max magnitude (north_star).  u = u^n + dt/2 (a^n + a^{n+1}) carries the 1e-5
    relative error of BOTH terms, so its scale is max|u| + dt max|a| (near rest, e.g. a dam break that has just
    started, dt |a| exceeds |u| and max|u| alone is not the magnitude of what was computed)."""
    for d, A in enumerate(st.arrays):
        if wl.arrays[d].n == 0:
            continue
        out = {k: v.cpu().numpy() for k, v in ctx.sync_state(d).items()}
        for k, axis in (("x", 0), ("y", 1), ("z", 2)):
            if axis >= wl.dim:
                continue
            diff = min_image_diff(out[k], A[k], wl.lo[axis], wl.hi[axis], wl.periodic[axis])
            scale = max(abs(wl.lo[axis]), abs(wl.hi[axis]))
            assert np.abs(diff).max() <= TOL * scale, f"{tag} {k}[{d}]: {np.abs(diff).max() / scale:.3e}"
        vmax = max(np.abs(A["u"]).max(), np.abs(A["v"]).max(), np.abs(A["w"]).max())
        vmax += dt * max(np.abs(A["au"]).max(), np.abs(A["av"]).max(), np.abs(A["aw"]).max())
        for k, axis in (("u", 0), ("v", 1), ("w", 2)):
            if axis < wl.dim and vmax > 0:
                err = np.abs(out[k].astype(np.float64) - A[k]).max() / vmax
                assert err <= TOL, f"{tag} {k}[{d}]: {err:.3e} of max|u| + dt max|a|"
        assert_close(out["rho"], A["rho"], f"{tag} rho[{d}]")


def _cases(WL):
    return {
        "c3_24": (WL.periodic_box_3d((24, 24, 24), seed=1), "summation"),
        "dam2d_cont": (WL.dam_break_2d(dx=0.04), "continuity"),
        "varh_4k": (WL.random_box(n=4000, dim=3, periodic=True, seed=63, kernel="wendland_c2", variable_h=True), "summation"),
    }


@pytest.mark.parametrize("nsteps", [10, 100])
@pytest.mark.parametrize("name", ["c3_24", "dam2d_cont", "varh_4k"])
def test_one_oracle_step_from_the_gpu_state_after_n_steps(O, WL, name, nsteps):
    wl, mode = _cases(WL)[name]
    ctx, _ = make_ctx(wl)
    ctx.pc_step(wl.dt, nsteps, mode)
    ctx.synchronize()                                   # raises on out-of-domain / non-finite
    s = ctx.get_stats()
    assert s.steps_done == nsteps
    st = _oracle_state_from_gpu(O, wl, ctx)
    x0 = st.arrays[0]["x"].copy()
    moved = np.abs(min_image_diff(x0, wl.arrays[0].x, wl.lo[0], wl.hi[0], wl.periodic[0])).max()
    assert moved > 0.0                                  # the state has left its initial layout
    O.pc_step(wl, st, wl.dt, mode)                      # ONE oracle step from the GPU's state and a^n
    ctx.pc_step(wl.dt, 1, mode)                         # the GPU's next step
    _compare(wl, ctx, st, f"{name} step {nsteps}+1", wl.dt)
    ctx.synchronize()
    ctx.close()


def test_graph_replay_matches_step_by_step(WL):
    """sph_pc_step(dt, 21) (1 + 10 replays of the captured pair of steps) against 21 calls of sph_pc_step(dt, 1):
    same kernels, same arguments -- the runs differ only by the order of the atomics of the counting sort."""
    wl = WL.periodic_box_3d((16, 16, 16), seed=2)
    outs = []
    for chunks in ((21,), (1,) * 21):
        ctx, _ = make_ctx(wl)
        for n in chunks:
            ctx.pc_step(wl.dt, n, "summation")
        ctx.synchronize()
        assert ctx.get_stats().steps_done == 21
        outs.append({k: v.cpu().numpy().astype(np.float64) for k, v in ctx.sync_state(0).items()})
        ctx.close()
    for k in ("x", "y", "z", "u", "v", "w", "rho"):
        assert np.abs(outs[0][k] - outs[1][k]).max() <= 2e-5 * max(np.abs(outs[1][k]).max(), 1e-30), k


def test_arrays_that_are_no_destination_get_zero_accelerations(O, WL):
    """The sort does not carry acc along; rows of arrays that no launch of an evaluation writes must read zero (the
    oracle's value), not another particle's acceleration: the solids' ax, ay in both density modes, and everything
    of an array whose tables are cleared with sph_set_tables."""
    for mode in ("continuity", "summation"):
        wl = WL.dam_break_2d(dx=0.04)
        wl.arrays[0].u[:] = np.random.default_rng(3).uniform(-0.5, 0.5, wl.arrays[0].n).astype(np.float32)
        ctx, _ = make_ctx(wl)
        ctx.pc_step(wl.dt, 3, mode)
        st = O.State(wl)
        for _ in range(3):
            O.pc_step(wl, st, wl.dt, mode)
        solid = {k: v.cpu().numpy() for k, v in ctx.get_accel(1).items()}
        assert not solid["ax"].any() and not solid["ay"].any()
        if mode == "continuity":
            want = st.arrays[1]["arho"]
            assert np.abs(solid["arho"] - want).max() <= 2e-5 * np.abs(want).max()
        else:
            assert not solid["arho"].any()
        ctx.close()
    # custom tables: the solid array is no destination at all -> its rho must not move in continuity mode
    wl = WL.dam_break_2d(dx=0.04)
    wl.arrays[0].u[:] = np.random.default_rng(4).uniform(-0.5, 0.5, wl.arrays[0].n).astype(np.float32)
    ctx, _ = make_ctx(wl)
    ctx.set_tables(accel=[3, 0], arho=[3, 0])
    ctx.pc_step(wl.dt, 3, "continuity")
    out = ctx.sync_state(1, fields=("rho", "arho"))
    assert np.array_equal(out["rho"].cpu().numpy(), wl.arrays[1].rho) and not out["arho"].cpu().numpy().any()
    ctx.synchronize()
    ctx.close()


def test_thin_nonperiodic_axis_next_to_a_periodic_one(O, WL):
    """A channel periodic in x whose y extent is a single cell (L_y < 2 k h): no minimum image may be applied on the
    non-periodic axis.  Sets bit-exact, rho and a at 1e-5."""
    wl = WL.random_box(n=1500, dim=2, periodic=True, seed=81, kernel="cubic", h_mean=0.03, box=(1.0, 0.1, 1.0))
    wl.periodic = (True, False, False)
    wl.lo = (0.0, -0.005, 0.0); wl.hi = (1.0, 0.105, 1.0)
    ctx, _ = make_ctx(wl)
    A = wl.arrays[0]
    f = {c: getattr(A, c) for c in "xyzh"}
    off, idx = ctx.nnps_get_neighbors(0, 0)
    ooff, oidx = O.neighbors(wl, f, f, pred32=True)
    assert np.array_equal(off, ooff) and np.array_equal(idx.astype(np.int64), oidx)
    st = O.State(wl)
    rho, _ = ctx.summation_density(0, 1)
    orho, _, _ = O.density(wl, st, 0, [0], pred32=True)
    assert_close(rho.cpu().numpy(), orho, "rho thin axis")
    st.arrays[0]["rho"] = rho.cpu().numpy().astype(np.float64)
    st.arrays[0]["p"] = O.eos(wl, st.arrays[0]["rho"])
    ax, ay, _, _ = ctx.wcsph_accel(0, 1)
    o = O.accel(wl, st, 0, [0], pred32=True)
    scale = max(np.abs(o["au"]).max(), np.abs(o["av"]).max())
    assert np.abs(ax.cpu().numpy() - o["au"]).max() <= TOL * scale and np.abs(ay.cpu().numpy() - o["av"]).max() <= TOL * scale
    ctx.synchronize()
    ctx.close()


@pytest.mark.parametrize("levels", [1, 2, 5, 8])
def test_variable_h_sets_do_not_depend_on_the_number_of_levels(O, WL, levels):
    """f3: the h classes / level grids are a search structure only -- neighbour sets stay bit-exact and rho within
    1e-5 for any number of levels (1 = the paper's single grid sized by h_max), h ratio 6 here."""
    wl = WL.random_box(n=3000, dim=3, periodic=True, seed=91, kernel="wendland_c2", variable_h=True)
    rng = np.random.default_rng(92)
    wl.arrays[0].h[:] = (wl.arrays[0].h.mean() * np.exp(rng.uniform(np.log(0.2), np.log(1.2), wl.arrays[0].n))).astype(np.float32)
    ctx, _ = make_ctx(wl, levels=levels)
    s = ctx.get_stats()
    assert s.variable_h == 1 and 1 <= s.n_levels <= levels and (levels == 1) == (s.n_levels == 1)
    A = wl.arrays[0]
    f = {c: getattr(A, c) for c in "xyzh"}
    off, idx = ctx.nnps_get_neighbors(0, 0)
    ooff, oidx = O.neighbors(wl, f, f, pred32=True)
    assert np.array_equal(off, ooff) and np.array_equal(idx.astype(np.int64), oidx)
    rho, _ = ctx.summation_density(0, 1)
    orho, _, _ = O.density(wl, O.State(wl), 0, [0], pred32=True)
    assert_close(rho.cpu().numpy(), orho, f"rho levels={levels}")
    ctx.synchronize()
    ctx.close()


@pytest.mark.parametrize("offset", [0.0, 1000.0])
def test_filter_has_no_false_negatives_at_the_cutoff(O, WL, offset):
    """Stress of the conservative tensor-core filter: many pairs at r = cut (1 +- 1e-6 ... 1e-3) in random directions,
    constant and variable h, in a box far from the origin (coordinates ~1000: the float rounding unit of positions is
    6e-5, a third of a per cent of h).  Sets must stay bit-exact with the oracle's float predicate."""
    rng = np.random.default_rng(123 + int(offset))
    for variable_h in (False, True):
        n_pairs = 1500
        wl = WL.random_box(n=2 * n_pairs, dim=3, periodic=True, seed=97, kernel="wendland_c2", variable_h=variable_h, h_mean=0.04)
        A = wl.arrays[0]
        h = A.h.astype(np.float64)
        ctr = rng.random((n_pairs, 3))
        d = rng.standard_normal((n_pairs, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
        cut = (h[0::2] + h[1::2])                                   # k/2 = 1 for Wendland-C2
        rel = 1.0 + rng.choice([-1.0, 1.0], n_pairs) * 10.0 ** rng.uniform(-6.5, -3.0, n_pairs)
        p0 = ctr - 0.5 * d * (cut * rel)[:, None]; p1 = ctr + 0.5 * d * (cut * rel)[:, None]
        pos = np.empty((2 * n_pairs, 3)); pos[0::2] = p0; pos[1::2] = p1
        pos = np.mod(pos, 1.0) + offset
        for k, c in enumerate("xyz"):
            v = pos[:, k].astype(np.float32)
            v[v >= np.float32(offset + 1.0)] = np.float32(offset)
            setattr(A, c, np.ascontiguousarray(v))
        wl.lo = (offset, offset, offset); wl.hi = (offset + 1.0, offset + 1.0, offset + 1.0)
        ctx, _ = make_ctx(wl)
        f = {c: getattr(A, c) for c in "xyzh"}
        off, idx = ctx.nnps_get_neighbors(0, 0)
        ooff, oidx = O.neighbors(wl, f, f, pred32=True)
        assert np.array_equal(off, ooff) and np.array_equal(idx.astype(np.int64), oidx), (offset, variable_h)
        near = np.diff(ooff).sum() - len(ooff) + 1
        assert near > n_pairs // 4                                   # a good share of the constructed pairs are neighbours
        rho, _ = ctx.summation_density(0, 1)
        assert ctx.get_stats().pairs_density == int(ooff[-1])
        ctx.synchronize()
        ctx.close()


def test_c5_pair_totals_do_not_depend_on_the_tiling(WL):
    """Full-size consistency of the filter: different level counts / x sub-cells give different groups, tile origins and
    margins; a false negative of the filter would have to repeat in all of them for the totals to agree."""
    wl = WL.gaussian_mixture_3d()
    totals = []
    for over in (dict(), dict(levels=2, xsub=8), dict(levels=5, xsub=2)):
        ctx, _ = make_ctx(wl, **over)
        ctx.summation_density(0, 1, want_p=False)
        ctx.synchronize()
        totals.append(int(ctx.get_stats().pairs_density))
        ctx.close()
    assert totals[0] == totals[1] == totals[2], totals
