"""-m gpu parity tests: the CUDA path (through the C-ABI binding) against the fp64 oracle on the same seeded
float32 inputs.  Gates (north_star / DESIGN.md "Tolerances"):
  neighbour sets      bit-exact (sorted CSR rows equal), both sides deciding membership with the R7 float predicate
  rho, ax, ay, az, arho, and x,u,rho after a step    max|gpu-oracle| <= 1e-5 * max|oracle| per property
  p                   against the oracle's EOS applied to the GPU's own rho (the EOS arithmetic), because
                      dp = c0^2 drho amplifies the allowed 1e-5 density error beyond 1e-5 of max|p|
Each call is compared FROM IDENTICAL INPUTS (accelerations are fed the same float32 rho and p on both sides).
"""
import numpy as np
import pytest

from gpu_helpers import TOL, assert_close, fields_of, make_ctx, mask_of, min_image_diff, oracle_state_with_p, rows

pytestmark = pytest.mark.gpu


def _small_cases(WL):
    return [
        WL.random_box(n=600, dim=2, periodic=True, seed=11, kernel="cubic"),
        WL.random_box(n=700, dim=2, periodic=False, seed=12, kernel="quintic", variable_h=True),
        WL.random_box(n=3000, dim=3, periodic=True, seed=13, kernel="wendland_c2", variable_h=True),
        WL.random_box(n=3000, dim=3, periodic=False, seed=14, kernel="cubic", two_arrays=True),
        WL.random_box(n=200, dim=3, periodic=True, seed=15, kernel="cubic", h_mean=0.16),      # exactly 3 cells / axis
        WL.random_box(n=2500, dim=2, periodic=True, seed=16, kernel="quintic", two_arrays=True, variable_h=True),
        WL.random_box(n=1, dim=2, periodic=True, seed=17, kernel="cubic", h_mean=0.05),
        WL.random_box(n=33, dim=3, periodic=False, seed=18, kernel="wendland_c2", h_mean=2.0),   # everything in one cell
        WL.lattice((32, 32), 2, 1.0, "quintic"),          # r = 3 dx = k h exactly on the lattice: strict '<' (R4)
        WL.lattice((16, 16, 16), 3, 1.3, "cubic"),
        WL.taylor_green_2d(),                              # C1
        WL.random_box(n=900, dim=2, periodic=True, seed=19, kernel="wendland_c2"),              # 2-D Wendland-C2 (sigma_2, h^-4)
    ]


CASE_IDS = ["2d_per", "2d_open_varh", "3d_per_varh", "3d_open_two", "3cells", "2d_per_two_varh", "single",
            "one_cell", "lattice2d_quintic", "lattice3d_cubic", "C1", "2d_per_wendland"]


@pytest.fixture(scope="module", params=list(range(len(CASE_IDS))), ids=CASE_IDS)
def case(request, WL):
    return _small_cases(WL)[request.param]


# ------------------------------------------------------------------------------------------------ sets
def test_neighbor_sets_bit_exact(O, case):
    wl = case
    ctx, _ = make_ctx(wl)
    for d, D in enumerate(wl.arrays):
        for s, S in enumerate(wl.arrays):
            off, idx = ctx.nnps_get_neighbors(d, s)
            ooff, oidx = O.neighbors(wl, fields_of(D), fields_of(S), pred32=True, method="cell")
            assert np.array_equal(off, ooff), f"neighbour counts differ for dest {d} src {s}"
            assert np.array_equal(idx.astype(np.int64), oidx), f"neighbour sets differ for dest {d} src {s}"
    ctx.synchronize()
    ctx.close()


def test_neighbor_sets_after_shuffle_are_the_same_sets(O, WL):
    """Permutation invariance through the GPU sort: shuffle the input, un-permute the lists."""
    wl = WL.random_box(n=2000, dim=3, periodic=True, seed=51, variable_h=True)
    ctx, _ = make_ctx(wl)
    off1, idx1 = ctx.nnps_get_neighbors(0, 0)
    perm = np.random.default_rng(9).permutation(wl.arrays[0].n)
    A = wl.arrays[0]
    for k in ("x", "y", "z", "u", "v", "w", "h", "m", "rho"):
        setattr(A, k, np.ascontiguousarray(getattr(A, k)[perm]))
    ctx2, _ = make_ctx(wl)
    off2, idx2 = ctx2.nnps_get_neighbors(0, 0)
    r1, r2 = rows(off1, idx1), rows(off2, idx2)
    for newi, oldi in enumerate(perm):
        assert np.array_equal(np.sort(perm[r2[newi]]), r1[oldi])
    ctx.close(); ctx2.close()


# ------------------------------------------------------------------------------------------------ density
def test_density_and_eos_parity(O, case):
    wl = case
    ctx, _ = make_ctx(wl)
    st = O.State(wl)
    for d in range(len(wl.arrays)):
        if wl.arrays[d].n == 0:
            continue
        for srcs in ([s for s in range(len(wl.arrays))], [0]):
            rho, p = ctx.summation_density(d, mask_of(srcs))
            rho, p = rho.cpu().numpy(), p.cpu().numpy()
            orho, _, opairs = O.density(wl, st, d, srcs, pred32=True)
            if not orho.any():
                continue
            assert_close(rho, orho, f"rho[{d}<-{srcs}]")
            assert_close(p, O.eos(wl, rho.astype(np.float64)), f"p=EOS(rho_gpu)[{d}]")
            assert ctx.get_stats().pairs_density == opairs       # same sets => same pair count
    ctx.close()


# ------------------------------------------------------------------------------------------------ accel
def _with_pressure(O, wl):
    """float32 p = EOS(float32 rho) from the oracle; both sides then start from the same rho and p."""
    return [O.eos(wl, a.rho.astype(np.float64)).astype(np.float32) for a in wl.arrays]


def test_accel_and_continuity_parity(O, case):
    from paper_1909_04504_b200 import binding
    import torch
    wl = case
    p32 = _with_pressure(O, wl)
    arrays = binding.device_arrays(wl)
    for d, a in enumerate(arrays):
        a["p"] = torch.from_numpy(p32[d]).cuda()
    ctx, _ = make_ctx(wl, arrays)
    st = oracle_state_with_p(O, wl, p32)
    for d in range(len(wl.arrays)):
        if wl.arrays[d].n == 0:
            continue
        for srcs in ([s for s in range(len(wl.arrays))], [0]):
            ax, ay, az, ar = ctx.wcsph_accel(d, mask_of(srcs), want_arho=True)
            o = O.accel(wl, st, d, srcs, pred32=True)
            if o["n_pairs"] <= wl.arrays[d].n and d in srcs:       # only self pairs: a == g exactly
                assert np.array_equal(ax.cpu().numpy(), np.full(wl.arrays[d].n, wl.g[0], dtype=np.float32))
                continue
            scale = max(np.abs(o["au"]).max(), np.abs(o["av"]).max(), np.abs(o["aw"]).max())
            if scale < 1e-6 * o["abs_a"].max():        # exact cancellation (uniform lattice, uniform p: a = 0):
                scale = o["abs_a"].max()               # the forward-error scale of the sum is sum_j |term|
            for name, g_, w_ in (("ax", ax, o["au"]), ("ay", ay, o["av"]), ("az", az, o["aw"])):
                if g_ is None:
                    continue
                if scale == 0.0:                       # every pair term is exactly 0 (p = 0, u = 0): so must the GPU's be
                    assert not g_.cpu().numpy().any(), f"{name}[{d}<-{srcs}]: non-zero where every term is 0"
                    continue
                err = np.abs(g_.cpu().numpy().astype(np.float64) - w_).max() / scale
                assert err <= TOL, f"{name}[{d}<-{srcs}]: {err:.3e} of max|a|"
            if np.abs(o["arho"]).max() > 0:
                assert_close(ar.cpu().numpy(), o["arho"], f"arho[{d}<-{srcs}]")
            assert ctx.get_stats().pairs_accel == o["n_pairs"]
    ctx.synchronize()
    ctx.close()


def test_momentum_conservation_on_gpu(O, WL):
    """Property that holds at any size: sum_i m_i a_i = 0 up to float32 round-off of the pair terms."""
    wl = WL.random_box(n=20000, dim=3, periodic=True, seed=52, kernel="wendland_c2", variable_h=True)
    ctx, _ = make_ctx(wl)
    ax, ay, az, _ = ctx.wcsph_accel(0, 1)
    m = wl.arrays[0].m.astype(np.float64)
    for a in (ax, ay, az):
        a = a.cpu().numpy().astype(np.float64)
        assert abs((m * a).sum()) < 2e-6 * (m * np.abs(a)).sum()
    ctx.close()


@pytest.mark.parametrize("dim,varh", [(2, False), (3, False), (3, True)], ids=["2d", "3d", "3d_varh"])
def test_coincident_particles_and_uniform_mass_wendland(O, WL, dim, varh):
    """R18: grad W := 0 at r = 0.  Every tenth particle sits exactly on its predecessor (different velocity, density
    and h), all masses are equal and no p is supplied, so the momentum pass runs its uniform-mass layouts (UM / VU: the
    Wendland-C2 gradient from the polynomial f'(q)/q with the mass in its constant, p/rho^2 recomputed when h varies):
    sets bit-exact, rho and a within 1e-5, the coincident pair adds m W(0) to rho and nothing to a."""
    wl = WL.random_box(n=1500, dim=dim, periodic=True, seed=60 + dim, kernel="wendland_c2", variable_h=varh)
    A = wl.arrays[0]
    A.m[:] = A.m[0]
    for k in "xyz":
        c = getattr(A, k)
        c[1::10] = c[0::10][:len(c[1::10])]
    ctx, _ = make_ctx(wl)
    off, idx = ctx.nnps_get_neighbors(0, 0)
    ooff, oidx = O.neighbors(wl, fields_of(A), fields_of(A), pred32=True, method="cell")
    assert np.array_equal(off, ooff) and np.array_equal(idx.astype(np.int64), oidx)
    r = rows(off, idx)
    assert all(i - 1 in r[i] for i in range(1, A.n, 10))          # the coincident partner is a neighbour
    st = oracle_state_with_p(O, wl)
    rho, _ = ctx.summation_density(0, 1)
    orho, _, opairs = O.density(wl, st, 0, [0], pred32=True)
    assert_close(rho.cpu().numpy(), orho, "rho")
    assert ctx.get_stats().pairs_density == opairs
    ctx.close()
    ctx, _ = make_ctx(wl)                     # a fresh build: rho as given, p = EOS(rho) on both sides
    ax, ay, az, ar = ctx.wcsph_accel(0, 1, want_arho=True)
    o = O.accel(wl, st, 0, [0], pred32=True)
    scale = max(np.abs(o["au"]).max(), np.abs(o["av"]).max(), np.abs(o["aw"]).max())
    for name, g_, w_ in (("ax", ax, o["au"]), ("ay", ay, o["av"]), ("az", az, o["aw"])):
        if g_ is None:
            continue
        g = g_.cpu().numpy().astype(np.float64)
        assert np.isfinite(g).all(), f"{name}: non-finite"
        err = np.abs(g - w_).max() / scale
        assert err <= TOL, f"{name}: {err:.3e} of max|a|"
    assert_close(ar.cpu().numpy(), o["arho"], "arho")
    assert ctx.get_stats().pairs_accel == o["n_pairs"]
    ctx.synchronize()
    ctx.close()
