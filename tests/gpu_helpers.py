"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding and the oracle on the same
seeded float32 inputs.  (Test infrastructure; the product never imports this.)"""
import numpy as np

TOL = 1e-5          # north_star: fp32 fields within 1e-5 of the per-property max magnitude


def rel_max_err(got, want):
    want = np.asarray(want, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    scale = np.abs(want).max() if want.size else 1.0
    return float(np.abs(got - want).max() / scale) if want.size and scale > 0 else float(np.abs(got - want).max() if want.size else 0.0)


def assert_close(got, want, name, tol=TOL):
    err = rel_max_err(got, want)
    assert err <= tol, f"{name}: max|gpu-oracle| / max|oracle| = {err:.3e} > {tol:g}"
    return err


def make_ctx(wl, arrays=None, **over):
    from paper_1909_04504_b200 import binding
    ctx = binding.SphContext.from_workload(wl, **over)
    arrays = arrays if arrays is not None else binding.device_arrays(wl, precision=over.get("precision", "f32"))
    ctx.nnps_build(arrays, [a.fixed for a in wl.arrays])
    return ctx, arrays


def rows(off, idx):
    return [idx[off[i]:off[i + 1]] for i in range(len(off) - 1)]


def fields_of(a):
    return {c: getattr(a, c) for c in "xyzh"}


def mask_of(srcs):
    m = 0
    for s in srcs:
        m |= 1 << s
    return m


def min_image_diff(a, b, lo, hi, periodic):
    d = np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)
    if periodic:
        L = hi - lo
        d -= L * np.rint(d / L)
    return d


def oracle_state_with_p(O, wl, p_arrays=None):
    """Oracle state from the workload's float32 arrays; p = given float32 arrays or EOS(rho)."""
    st = O.State(wl)
    for d, A in enumerate(st.arrays):
        A["p"] = (np.asarray(p_arrays[d], dtype=np.float64) if p_arrays is not None else O.eos(wl, A["rho"]))
    return st
