"""-m gpu parity of the fp64 build (libsph_b200_f64.so: the same sources with -DSPH_REAL_DOUBLE, sph_real = double;
north_star: "1e-12 for an fp64 build flag") on the small cases and the step cases of the float suite.
Gates: neighbour sets bit-exact against the oracle's DOUBLE predicate (pred32 = False: the double build evaluates the
same expression, products and sums rounded one by one); rho, a, arho and x, u, rho after a step within 1e-12 of the
per-property max magnitude.  Inputs are the workloads' float32 values widened to double on both sides."""
import numpy as np
import pytest

from gpu_helpers import fields_of, make_ctx, mask_of, min_image_diff
from test_gpu_parity import CASE_IDS, _small_cases
from test_gpu_step import STEP_IDS, _step_cases

pytestmark = pytest.mark.gpu
TOL64 = 1e-12
F64 = dict(precision="f64")


def _close(got, want, name, scale=None):
    want = np.asarray(want, dtype=np.float64); got = np.asarray(got, dtype=np.float64)
    sc = np.abs(want).max() if scale is None else scale
    if want.size and sc > 0:
        err = np.abs(got - want).max() / sc
        assert err <= TOL64, f"{name}: {err:.3e} > {TOL64:g}"


@pytest.fixture(scope="module", params=list(range(len(CASE_IDS))), ids=CASE_IDS)
def case(request, WL):
    return _small_cases(WL)[request.param]


def test_f64_sets_density_accel(O, case):
    import torch
    from paper_1909_04504_b200 import binding
    wl = case
    # p = EOS(rho) in double on both sides (handed in, so that both start from the identical rho and p)
    p64 = [O.eos(wl, a.rho.astype(np.float64)) for a in wl.arrays]
    arrays = binding.device_arrays(wl, precision="f64")
    for d, a in enumerate(arrays):
        a["p"] = torch.from_numpy(p64[d]).cuda()
    ctx, _ = make_ctx(wl, arrays, **F64)
    assert ctx.real_size == 8
    for d, D in enumerate(wl.arrays):
        for s, S in enumerate(wl.arrays):
            off, idx = ctx.nnps_get_neighbors(d, s)
            ooff, oidx = O.neighbors(wl, fields_of(D), fields_of(S), pred32=False, method="cell")
            assert np.array_equal(off, ooff) and np.array_equal(idx.astype(np.int64), oidx), f"sets differ for dest {d} src {s}"
    st = O.State(wl)
    for d, A in enumerate(st.arrays):
        A["p"] = p64[d]
    na = len(wl.arrays)
    for d in range(na):
        if wl.arrays[d].n == 0:
            continue
        for srcs in (list(range(na)), [0]):
            ax, ay, az, ar = ctx.wcsph_accel(d, mask_of(srcs), want_arho=True)
            o = O.accel(wl, st, d, srcs, pred32=False)
            scale = max(np.abs(o["au"]).max(), np.abs(o["av"]).max(), np.abs(o["aw"]).max())
            if scale < 1e-6 * o["abs_a"].max():
                scale = o["abs_a"].max()
            if scale > 0:
                for name, g_, w_ in (("ax", ax, o["au"]), ("ay", ay, o["av"]), ("az", az, o["aw"])):
                    if g_ is not None:
                        _close(g_.cpu().numpy(), w_, f"{name}[{d}<-{srcs}]", scale)
            _close(ar.cpu().numpy(), o["arho"], f"arho[{d}<-{srcs}]", max(np.abs(o["arho"]).max(), o["abs_arho"].max() * 1e-6))
            assert ctx.get_stats().pairs_accel == o["n_pairs"]
    for d in range(na):
        if wl.arrays[d].n == 0:
            continue
        for srcs in (list(range(na)), [0]):
            rho, p = ctx.summation_density(d, mask_of(srcs))
            orho, _, opairs = O.density(wl, st, d, srcs, pred32=False)
            if orho.any():
                _close(rho.cpu().numpy(), orho, f"rho[{d}<-{srcs}]")
                _close(p.cpu().numpy(), O.eos(wl, rho.cpu().numpy()), f"p[{d}]", max(np.abs(O.eos(wl, orho)).max(), wl.rho0 * wl.c0 ** 2 * 1e-3))
                assert ctx.get_stats().pairs_density == opairs
    ctx.synchronize()
    ctx.close()


@pytest.mark.parametrize("idx", range(len(STEP_IDS)), ids=STEP_IDS)
def test_f64_one_step(O, WL, idx):
    _, wl, mode = _step_cases(WL)[idx]
    ctx, _ = make_ctx(wl, **F64)
    ctx.pc_step(wl.dt, 1, mode)
    st = O.State(wl)
    O.pc_step(wl, st, wl.dt, mode)
    for d, A in enumerate(st.arrays):
        if wl.arrays[d].n == 0:
            continue
        out = {k: v.cpu().numpy() for k, v in ctx.sync_state(d).items()}
        for k, axis in (("x", 0), ("y", 1), ("z", 2)):
            if axis < wl.dim:
                diff = min_image_diff(out[k], A[k], wl.lo[axis], wl.hi[axis], wl.periodic[axis])
                assert np.abs(diff).max() <= TOL64 * max(abs(wl.lo[axis]), abs(wl.hi[axis])), f"{k}[{d}]"
        amax = max(np.abs(A["au"]).max(), np.abs(A["av"]).max(), np.abs(A["aw"]).max())
        vmax = max(np.abs(A["u"]).max(), np.abs(A["v"]).max(), np.abs(A["w"]).max()) + wl.dt * amax
        for k, axis in (("u", 0), ("v", 1), ("w", 2)):
            if axis < wl.dim and vmax > 0:
                _close(out[k], A[k], f"{k}[{d}]", vmax)
        _close(out["rho"], A["rho"], f"rho[{d}]")
    ctx.synchronize()
    ctx.close()
