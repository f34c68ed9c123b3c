"""Pins for the oracle's neighbour sets (Sec.2.2, Fig.1):
the linked-list cell grid must return exactly the brute-force O(N^2) sets; an independent dense numpy
evaluation of |x_i-x_j| < k h_ij written here must agree; sets are symmetric and permutation invariant;
lattice counts equal the known stencil counts; the float predicate differs from the double one only on
pairs within rounding of the cut-off."""
import numpy as np
import pytest

from conftest import golden_path


def _rows(off, idx):
    return [tuple(idx[off[i]:off[i + 1]]) for i in range(len(off) - 1)]


def _cat(wl):
    return {c: np.concatenate([getattr(a, c) for a in wl.arrays]) for c in "xyzh"}


def _dense_sets(wl, P, k):
    """Independent dense O(N^2) numpy evaluation in float64 (minimum image via rint)."""
    pos = np.stack([P["x"], P["y"], P["z"]], axis=1).astype(np.float64)
    d = pos[:, None, :] - pos[None, :, :]
    for a in range(3):
        if a >= wl.dim:
            d[:, :, a] = 0.0
        elif wl.periodic[a]:
            L = wl.hi[a] - wl.lo[a]
            d[:, :, a] -= L * np.rint(d[:, :, a] / L)
    r = np.sqrt((d ** 2).sum(-1))
    h = P["h"].astype(np.float64)
    cut = k * 0.5 * (h[:, None] + h[None, :])
    return r, cut


CASES = [
    dict(n=600, dim=2, periodic=True, seed=11, variable_h=False),
    dict(n=600, dim=2, periodic=False, seed=12, variable_h=True),
    dict(n=1500, dim=3, periodic=True, seed=13, variable_h=True),
    dict(n=1500, dim=3, periodic=False, seed=14, variable_h=False, two_arrays=True),
    dict(n=200, dim=3, periodic=True, seed=15, variable_h=False, h_mean=0.16),   # exactly 3 cells per axis
    dict(n=60, dim=3, periodic=True, seed=16, variable_h=False, h_mean=0.3),     # < 3 cells: one-cell fallback
    dict(n=1, dim=2, periodic=True, seed=17),
    dict(n=0, dim=3, periodic=False, seed=18),
]


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("kernel", ["cubic", "quintic"])
@pytest.mark.parametrize("pred32", [True, False])
def test_cell_list_equals_brute_force(O, WL, case, kernel, pred32):
    wl = WL.random_box(kernel=kernel, **case)
    P = _cat(wl)
    ob, ib = O.neighbors(wl, P, P, pred32=pred32, method="brute")
    oc, ic = O.neighbors(wl, P, P, pred32=pred32, method="cell")
    assert np.array_equal(ob, oc) and np.array_equal(ib, ic)
    if case["n"]:
        rows = _rows(ob, ib)
        assert all(i in rows[i] for i in range(case["n"]))            # self pair included (R5)


@pytest.mark.parametrize("case", CASES[:5])
def test_brute_force_equals_dense_numpy(O, WL, case):
    wl = WL.random_box(kernel="cubic", **case)
    P = _cat(wl)
    k = O.support("cubic")
    off, idx = O.neighbors(wl, P, P, pred32=False, method="brute")
    r, cut = _dense_sets(wl, P, k)
    got = np.zeros_like(r, dtype=bool)
    for i, row in enumerate(_rows(off, idx)):
        got[i, list(row)] = True
    want = r < cut
    border = np.abs(r - cut) < 1e-12 * cut
    assert np.array_equal(got | border, want | border)
    assert np.array_equal(got, got.T)                                 # j in N(i) <=> i in N(j)


def test_float_predicate_differs_only_at_the_cutoff(O, WL):
    wl = WL.random_box(n=3000, dim=3, periodic=True, seed=21, variable_h=True)
    P = _cat(wl)
    o32, i32 = O.neighbors(wl, P, P, pred32=True)
    o64, i64 = O.neighbors(wl, P, P, pred32=False)
    r, cut = _dense_sets(wl, P, 2.0)
    a = np.zeros_like(r, dtype=bool); b = np.zeros_like(r, dtype=bool)
    for i, row in enumerate(_rows(o32, i32)):
        a[i, list(row)] = True
    for i, row in enumerate(_rows(o64, i64)):
        b[i, list(row)] = True
    diff = a ^ b
    assert (np.abs(r[diff] / cut[diff] - 1.0) < 1e-6).all()
    assert np.array_equal(a, a.T)                                     # the float predicate is symmetric too


def test_permutation_invariance(O, WL):
    wl = WL.random_box(n=800, dim=2, periodic=True, seed=22, variable_h=True)
    P = _cat(wl)
    perm = np.random.default_rng(5).permutation(800)
    Q = {c: P[c][perm] for c in P}
    o1, i1 = O.neighbors(wl, P, P)
    o2, i2 = O.neighbors(wl, Q, Q)
    rows1, rows2 = _rows(o1, i1), _rows(o2, i2)
    for newi, oldi in enumerate(perm):
        assert tuple(sorted(perm[list(rows2[newi])])) == rows1[oldi]


def test_two_array_sets(O, WL):
    """dest != source: no self pair is implied; counts add up to the merged-array counts."""
    wl = WL.random_box(n=900, dim=2, periodic=False, seed=23, two_arrays=True)
    f, s = ({c: getattr(a, c) for c in "xyzh"} for a in wl.arrays)
    P = _cat(wl)
    off_all, _ = O.neighbors(wl, P, P)
    off_ff, _ = O.neighbors(wl, f, f)
    off_fs, idx_fs = O.neighbors(wl, f, s)
    off_sf, idx_sf = O.neighbors(wl, s, f)
    nf = wl.arrays[0].n
    assert np.array_equal(np.diff(off_all)[:nf], np.diff(off_ff) + np.diff(off_fs))
    pairs_fs = {(i, j) for i, row in enumerate(_rows(off_fs, idx_fs)) for j in row}
    pairs_sf = {(j, i) for i, row in enumerate(_rows(off_sf, idx_sf)) for j in row}
    assert pairs_fs == pairs_sf


def test_lattice_counts_match_golden(O, WL):
    for line in open(golden_path("lattice_sums.txt")):
        if line.startswith("#") or not line.strip():
            continue
        dim, kernel, hdx, _, count = line.split()
        dim, count = int(dim), int(count)
        n = (32, 32) if dim == 2 else (16, 16, 16)
        wl = WL.lattice(n, dim, float(hdx), kernel)
        P = _cat(wl)
        for pred32 in (True, False):
            off, _ = O.neighbors(wl, P, P, pred32=pred32)
            assert (np.diff(off) == count).all()


def test_neighbours_lie_in_the_3d_boxes(O, WL):
    """Fig.1 (L177): with cells of size = support radius every neighbour is in the 9 (27) boxes around q."""
    wl = WL.random_box(n=2000, dim=2, periodic=True, seed=24)
    P = _cat(wl)
    cell = 2.0 * float(P["h"].max())
    ncell = int(np.floor(1.0 / cell))
    cs = 1.0 / ncell
    cx = np.floor(P["x"].astype(np.float64) / cs).astype(int)
    cy = np.floor(P["y"].astype(np.float64) / cs).astype(int)
    off, idx = O.neighbors(wl, P, P, pred32=False)
    for i, row in enumerate(_rows(off, idx)):
        for j in row:
            ddx = (cx[j] - cx[i] + ncell) % ncell
            ddy = (cy[j] - cy[i] + ncell) % ncell
            assert ddx in (0, 1, ncell - 1) and ddy in (0, 1, ncell - 1)


def test_block_generator_matches_paper_listing(WL):
    """get_2d_block(dx=0.1, length=1, height=2, center=[-1.5+dx, 1+dx])
    -> 231 particles, fluid.x from -1.9 to -0.9."""
    x, y = WL.block_2d_inclusive(0.1, 1.0, 2.0, (-1.5 + 0.1, 1 + 0.1))
    assert len(x) == 231
    assert x.min() == pytest.approx(-1.9) and x.max() == pytest.approx(-0.9)
    wl = WL.dam_break_2d()
    assert [a.n for a in wl.arrays] == [20000, 3618]


def test_neighbour_relation_is_symmetric(O, WL):
    """The predicate r_ij < k (h_i + h_j)/2 is symmetric in i and j (R3): j in N(i) <=> i in N(j), also
    with variable h and across the periodic seam."""
    for dim in (2, 3):
        wl = WL.random_box(n=900, dim=dim, periodic=True, seed=41 + dim, variable_h=True)
        A = wl.arrays[0]
        f = {c: getattr(A, c) for c in "xyzh"}
        for pred32 in (True, False):
            off, idx = O.neighbors(wl, f, f, pred32=pred32, method="cell")
            pairs = {(i, int(j)) for i in range(A.n) for j in idx[off[i]:off[i + 1]]}
            assert all((j, i) in pairs for (i, j) in pairs)
            assert all((i, i) in pairs for i in range(A.n))          # self pair included (R5)
