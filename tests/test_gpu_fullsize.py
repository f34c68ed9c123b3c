"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (one context, device
arrays, default tuning: default record pool, default levels; C5 additionally with no pool), on SAMPLED destination particles the oracle computes one by one (full
runs of the fp64 oracle take minutes to hours at these sizes), plus properties that hold at any size.

For every config the oracle evaluates eq.3 / eq.8-9 (+ eq.7) for a seeded sample of destination particles
against ALL source particles (its own cell list over the sources), from the same float32 inputs the GPU has;
for the acceleration both sides start from the GPU's own rho and p (R15: each call is compared from
identical inputs).  Gates as in test_gpu_parity.py: 1e-5 of the per-property max magnitude over the sample;
the neighbour COUNT of every sampled particle is compared exactly (same sets => same counts; the full sets are
compared bit-exactly on the small cases).  C5 is gated on the sum-of-|terms| scale as well (R14).
"""
import numpy as np
import pytest

from gpu_helpers import TOL, make_ctx, mask_of

pytestmark = pytest.mark.gpu

N_SAMPLE = 4096


def min_image(d, L=1.0):
    return d - L * np.rint(d / L)


def _sample(n, k, seed):
    return np.sort(np.random.default_rng(seed).choice(n, size=min(k, n), replace=False))


def _rows_count(O, wl, st, d, srcs, sub):
    """neighbour count per sampled destination (float predicate, R7), summed over the source arrays"""
    D = {c: st.arrays[d][c][sub] for c in "xyzh"}
    cnt = np.zeros(len(sub), dtype=np.int64)
    for s in srcs:
        S = {c: st.arrays[s][c] for c in "xyzh"}
        off, _ = O.neighbors(wl, D, S, pred32=True, method="cell")
        cnt += np.diff(off)
    return cnt


def _gpu_state_into(O, wl, ctx):
    """oracle State holding the GPU's current float32 rho and p (and the workload's x,u,h,m)"""
    st = O.State(wl)
    for d, A in enumerate(st.arrays):
        if wl.arrays[d].n == 0:
            continue
        out = ctx.sync_state(d, fields=("rho", "p"))
        A["rho"] = out["rho"].cpu().numpy().astype(np.float64)
        A["p"] = out["p"].cpu().numpy().astype(np.float64)
    return st


def _check_density(O, wl, ctx, st, seed, abs_gate=False):
    na = len(wl.arrays)
    all_src = list(range(na))
    for d in range(na):
        n = wl.arrays[d].n
        if n == 0:
            continue
        rho, p = ctx.summation_density(d, mask_of(all_src))
        rho, p = rho.cpu().numpy(), p.cpu().numpy()
        assert np.isfinite(rho).all() and (rho > 0).all()
        sub = _sample(n, N_SAMPLE, seed + d)
        orho, oabs, opairs = O.density(wl, st, d, all_src, pred32=True, subset=sub)
        err = np.abs(rho[sub].astype(np.float64) - orho)
        assert err.max() <= TOL * np.abs(orho).max(), f"rho[{d}]: {err.max() / np.abs(orho).max():.3e}"
        if abs_gate:
            assert (err / oabs).max() <= TOL, f"rho[{d}] per-particle: {(err / oabs).max():.3e} of sum|terms|"
        peos = O.eos(wl, rho[sub].astype(np.float64))
        assert np.abs(p[sub] - peos).max() <= TOL * max(np.abs(peos).max(), 1e-30), f"p=EOS(rho_gpu)[{d}]"


def _check_accel(O, wl, ctx, st, d, srcs, seed, want_arho, abs_gate=False):
    n = wl.arrays[d].n
    ax, ay, az, ar = ctx.wcsph_accel(d, mask_of(srcs), want_arho=want_arho)
    sub = _sample(n, N_SAMPLE, seed)
    o = O.accel(wl, st, d, srcs, pred32=True, subset=sub)
    scale = max(np.abs(o["au"]).max(), np.abs(o["av"]).max(), np.abs(o["aw"]).max())
    for name, g_, w_ in (("ax", ax, o["au"]), ("ay", ay, o["av"]), ("az", az, o["aw"])):
        if g_ is None:
            continue
        g_ = g_.cpu().numpy()
        assert np.isfinite(g_).all()
        err = np.abs(g_[sub].astype(np.float64) - w_)
        assert err.max() <= TOL * scale, f"{name}[{d}<-{srcs}]: {err.max() / scale:.3e} of max|a|"
        if abs_gate:
            e2 = (err / np.maximum(o["abs_a"], 1e-300)).max()
            assert e2 <= TOL, f"{name}[{d}<-{srcs}] per-particle: {e2:.3e} of sum|terms|"
    if want_arho:
        g_ = ar.cpu().numpy()
        err = np.abs(g_[sub].astype(np.float64) - o["arho"])
        sc = np.abs(o["arho"]).max()
        assert err.max() <= TOL * sc, f"arho[{d}<-{srcs}]: {err.max() / sc:.3e}"
    return o["n_pairs"]


def _perturb(wl, seed, du, drho):
    """seeded non-trivial state for the dam breaks (their t = 0 state has u = 0, rho = rho0: every term is 0)"""
    rng = np.random.default_rng(seed)
    for a in wl.arrays:
        if not a.fixed:
            for k in ("u", "v", "w")[:wl.dim]:
                setattr(a, k, rng.uniform(-du, du, a.n).astype(np.float32))
        a.rho = (wl.rho0 * (1.0 + rng.uniform(-drho, drho, a.n))).astype(np.float32)


# ------------------------------------------------------------------------------------------------
def test_c3_full_density_accel_and_counts(O, WL):
    wl = WL.periodic_box_3d((128, 128, 128), seed=1, dx=1.0 / 128)
    ctx, _ = make_ctx(wl)
    st = O.State(wl)
    _check_density(O, wl, ctx, st, seed=100)
    pairs_gpu = ctx.get_stats().pairs_density
    st2 = _gpu_state_into(O, wl, ctx)
    _check_accel(O, wl, ctx, st2, 0, [0], seed=101, want_arho=False)
    s = ctx.get_stats()
    assert s.used_rows == 1                       # the momentum pass replayed the records of the one search
    assert s.pairs_accel == pairs_gpu             # ... and saw exactly the same pairs
    # every sampled particle has exactly the oracle's neighbour count (exact sets are gated on the small cases)
    sub = _sample(wl.arrays[0].n, N_SAMPLE, 102)
    cnt = _rows_count(O, wl, st, 0, [0], sub)
    gcnt = ctx.neighbor_counts(0, 0)
    assert np.array_equal(gcnt[sub], cnt)
    assert int(gcnt.sum()) == pairs_gpu
    # property at any size: sum_i m_i a_i = 0 (periodic, one dynamic array) up to float32 round-off
    acc = ctx.get_accel(0)
    m = wl.arrays[0].m.astype(np.float64)
    for k in ("ax", "ay", "az"):
        a = acc[k].cpu().numpy().astype(np.float64)
        assert abs((m * a).sum()) < 2e-6 * (m * np.abs(a)).sum()
    # mean neighbour count of the sample vs the GPU's total pair count (57.8 on this lattice)
    assert abs(cnt.mean() - pairs_gpu / wl.arrays[0].n) < 0.5
    ctx.synchronize()
    ctx.close()


def test_c3_full_pc_steps_stay_finite_and_conserve_momentum(WL):
    """bench.py's timed configuration: sph_pc_step on C3.  Total momentum is conserved by the symmetric pair
    terms (periodic box, no gravity): after the config's 100 steps it equals the initial one to float32 round-off."""
    wl = WL.periodic_box_3d((128, 128, 128), seed=1, dx=1.0 / 128)
    ctx, _ = make_ctx(wl)
    A = wl.arrays[0]
    m = A.m.astype(np.float64)
    p0 = np.array([(m * getattr(A, k).astype(np.float64)).sum() for k in ("u", "v", "w")])
    ctx.pc_step(wl.dt, wl.n_steps, "summation")
    ctx.synchronize()
    out = ctx.sync_state(0)
    p1 = np.array([(m * out[k].cpu().numpy().astype(np.float64)).sum() for k in ("u", "v", "w")])
    scale = (m * np.abs(A.u.astype(np.float64))).sum()
    assert np.abs(p1 - p0).max() < 1e-5 * scale
    for k in ("x", "y", "z"):
        x = out[k].cpu().numpy()
        assert np.isfinite(x).all() and x.min() >= 0.0 and x.max() <= 1.0
    s = ctx.get_stats()
    assert wl.n_steps == 100 and s.steps_done == 100 and s.used_rows == 1
    assert np.abs(out["rho"].cpu().numpy() / wl.rho0 - 1.0).max() < 0.2
    ctx.close()


def test_c2_full_two_arrays_continuity_tables(O, WL):
    wl = WL.dam_break_2d()
    _perturb(wl, 7, du=0.5, drho=0.01)
    ctx, _ = make_ctx(wl)
    st = O.State(wl)
    for A in st.arrays:
        A["p"] = O.eos(wl, A["rho"])
    # Listing 3: fluid <- {fluid, solid} momentum + continuity in one pass; solid <- {fluid} continuity only
    _check_accel(O, wl, ctx, st, 0, [0, 1], seed=110, want_arho=True)
    ax, ay, az, ar = ctx.wcsph_accel(1, mask_of([0]), want_arho=True)
    sub = _sample(wl.arrays[1].n, N_SAMPLE, 111)
    o = O.accel(wl, st, 1, [0], pred32=True, subset=sub)
    err = np.abs(ar.cpu().numpy()[sub].astype(np.float64) - o["arho"]).max()
    assert err <= TOL * np.abs(o["arho"]).max()
    _check_density(O, wl, ctx, st, seed=112)
    ctx.synchronize()
    ctx.close()


def test_c4_full_two_arrays(O, WL):
    wl = WL.dam_break_3d()
    assert wl.arrays[0].n == 3_456_000 and wl.arrays[1].n == 765_468
    _perturb(wl, 8, du=0.5, drho=0.01)
    ctx, _ = make_ctx(wl)
    st = O.State(wl)
    for A in st.arrays:
        A["p"] = O.eos(wl, A["rho"])
    _check_accel(O, wl, ctx, st, 0, [0, 1], seed=120, want_arho=True)
    ax, ay, az, ar = ctx.wcsph_accel(1, mask_of([0]), want_arho=True)
    sub = _sample(wl.arrays[1].n, N_SAMPLE, 121)
    o = O.accel(wl, st, 1, [0], pred32=True, subset=sub)
    err = np.abs(ar.cpu().numpy()[sub].astype(np.float64) - o["arho"]).max()
    assert err <= TOL * np.abs(o["arho"]).max()
    _check_density(O, wl, ctx, st, seed=122)
    # the timed configuration: continuity-mode steps, NNPS rebuilt every step
    ctx2, _ = make_ctx(wl)
    ctx2.pc_step(wl.dt, 2, "continuity")
    ctx2.synchronize()
    assert ctx2.get_stats().steps_done == 2
    ctx.close(); ctx2.close()


@pytest.mark.parametrize("pool", ["default_pool", "no_pool"])
def test_c5_full_variable_h(O, WL, pool):
    """C5 in the configuration bench.py times (default record pool: one search, both pair passes replay; level
    grids) and with no pool (every pair pass searches itself)."""
    wl = WL.gaussian_mixture_3d()
    assert wl.arrays[0].n == 1 << 24
    ctx, _ = make_ctx(wl, nlist_slots=(0 if pool == "default_pool" else -1))
    st = O.State(wl)
    _check_density(O, wl, ctx, st, seed=130, abs_gate=True)
    st2 = _gpu_state_into(O, wl, ctx)
    _check_accel(O, wl, ctx, st2, 0, [0], seed=131, want_arho=False, abs_gate=True)
    s = ctx.get_stats()
    assert s.variable_h == 1 and s.n_levels >= 2
    if pool == "default_pool":
        assert s.used_rows == 1 and s.nlist_fallback_warps == 0 and s.candidates_accel == 0
        assert s.candidates_search / wl.arrays[0].n <= 1000.0          # f3: not the ~2,650 (r1) / ~4,800 (one grid) per particle
        print(f"C5 default pool: {s.candidates_search / wl.arrays[0].n:.0f} candidates per particle, "
              f"{s.nlist_rows_used} of {s.nlist_rows_capacity} record rows, fallback warps {s.nlist_fallback_warps}, levels {s.n_levels}")
    else:
        assert s.used_rows == 0 and s.candidates_accel > 0
    assert s.pairs_accel == s.pairs_density
    sub = _sample(wl.arrays[0].n, N_SAMPLE, 132)
    assert np.array_equal(ctx.neighbor_counts(0, 0)[sub], _rows_count(O, wl, st, 0, [0], sub))
    ctx.synchronize()
    ctx.close()


def test_c3_full_state_after_100_steps(O, WL):
    """A15 at full size: the C3 state after its 100 steps (ragged cells, the state bench.py times) goes back through
    the C ABI as a new build; density, momentum and neighbour counts of sampled particles against the oracle."""
    import copy
    wl = WL.periodic_box_3d((128, 128, 128), seed=1, dx=1.0 / 128)
    ctx, _ = make_ctx(wl)
    ctx.pc_step(wl.dt, 100, "summation")
    ctx.synchronize()
    out = {k: v.cpu().numpy() for k, v in ctx.sync_state(0).items()}
    ctx.close()
    wl2 = copy.deepcopy(wl)
    for k in ("x", "y", "z", "u", "v", "w", "rho"):
        setattr(wl2.arrays[0], k, np.ascontiguousarray(out[k], dtype=np.float32))
    moved = np.abs(min_image(out["x"] - wl.arrays[0].x)).max() * 128
    assert moved > 0.3, moved                                     # in units of dx
    ctx, _ = make_ctx(wl2)
    st = O.State(wl2)
    _check_density(O, wl2, ctx, st, seed=140)
    pairs = ctx.get_stats().pairs_density
    st2 = _gpu_state_into(O, wl2, ctx)
    _check_accel(O, wl2, ctx, st2, 0, [0], seed=141, want_arho=False)
    s = ctx.get_stats()
    assert s.used_rows == 1 and s.pairs_accel == pairs
    sub = _sample(wl2.arrays[0].n, N_SAMPLE, 142)
    assert np.array_equal(ctx.neighbor_counts(0, 0)[sub], _rows_count(O, wl2, st, 0, [0], sub))
    ctx.synchronize()
    ctx.close()


def test_c2_full_run_of_1000_steps_stays_sane(WL):
    """BASELINE configs[1] as stated: the 2-D dam break for its 1,000 predictor-corrector steps, NNPS rebuilt every
    step.  No particle leaves the box, nothing non-finite (sph_synchronize raises otherwise), and the weakly
    compressible density stays within a few per cent of rho0 (R24: with dt = 0.25 h/c0 this run
    explodes near step 550, in the oracle as well)."""
    wl = WL.dam_break_2d()
    ctx, _ = make_ctx(wl)
    ctx.pc_step(wl.dt, wl.n_steps, "continuity")
    ctx.synchronize()
    s = ctx.get_stats()
    assert s.steps_done == 1000
    for d in range(2):
        out = {k: v.cpu().numpy() for k, v in ctx.sync_state(d).items()}
        assert all(np.isfinite(v).all() for v in out.values())
        assert np.abs(out["rho"] / wl.rho0 - 1.0).max() < 0.05
    fluid = ctx.sync_state(0)
    assert float(fluid["y"].min()) > 0.0 and float(fluid["x"].min()) > 0.0      # nobody went through the walls
    assert float(fluid["x"].max()) > 1.0                                         # ... and the dam has started to collapse
    ctx.close()
