"""-m gpu: sph_cell_offsets_static (include/sph.h), the allocation-free variant of the sort's look-back scan whose
scratch is a static device array of the library, against the EXISTING path: the context's k_scan, reached through
sph_nnps_get_neighbors (its offsets[] are k_scan's exclusive prefix sum of the per-particle neighbour counts).
Integer work: bit-exact.  The file sorts last on purpose (the suite runs with pytest -x)."""
import ctypes as C

import numpy as np
import pytest

from gpu_helpers import make_ctx

pytestmark = pytest.mark.gpu


def _existing_offsets(ctx, dest=0, src=0):
    """offsets[n+1] of the context path (count pass + k_scan in context-owned scratch), as uint32"""
    n = ctx.n[dest]
    off = np.zeros(n + 1, dtype=np.int64)
    total = C.c_int64(0)
    ctx._check(ctx.L.sph_nnps_get_neighbors(ctx.ctx, dest, src, off.ctypes.data, None, 0, C.byref(total), 1))
    assert off[-1] == total.value and 0 < total.value < 2 ** 32
    return off.astype(np.uint32)


def _cases(WL):
    return [WL.periodic_box_3d((56, 56, 56), seed=5),                                  # 175,616 counts: 43 tiles, look-back past 32
            WL.random_box(n=64001, dim=2, periodic=False, seed=6, kernel="cubic"),    # 16 tiles, ragged tail of 1, zero counts
            WL.random_box(n=777, dim=2, periodic=True, seed=7, kernel="quintic")]     # less than one tile


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_static_cell_offsets_match_the_context_scan_on_calls_in_a_row(WL, precision):
    import torch
    from paper_1909_04504_b200 import binding
    dev = torch.device("cuda", 0)
    want, counts = [], []
    for wl in _cases(WL):
        ctx, _ = make_ctx(wl, precision=precision)
        off = _existing_offsets(ctx)
        ctx.close()
        want.append(off)
        counts.append(torch.from_numpy(np.diff(off.astype(np.int64)).astype(np.uint32).view(np.int32)).to(dev))
    nmax = max(c.numel() for c in counts)
    outs = [torch.full((nmax + 1,), -1, dtype=torch.int32, device=dev) for _ in counts]
    binding.cell_offsets_static(counts[0][:0], torch.empty(1, dtype=torch.int32, device=dev), precision=precision)   # set-up call
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(dev)[0]
    # the calls follow one another on one stream with no synchronisation in between and share one output buffer
    # per round, so each call starts from the scratch (and, in round 2, the output) the call before it left behind
    for rnd in range(2):
        order = (0, 1, 2) if rnd == 0 else (2, 0, 1)
        for k in order:
            binding.cell_offsets_static(counts[k], outs[k], precision=precision)
        torch.cuda.synchronize()
        for k in order:
            n = counts[k].numel()
            got = outs[k].cpu().numpy().view(np.uint32)
            assert np.array_equal(got[:n + 1], want[k]), f"round {rnd} case {k}: offsets differ from the context path"
            assert (got[n + 1:] == 0xffffffff).all(), "wrote past offsets[n]"
    assert torch.cuda.mem_get_info(dev)[0] == free0, "device memory was allocated by the call"


def test_static_cell_offsets_two_calls_same_input_and_unaligned_views(WL):
    """The same input twice gives the same output (the scratch of call 1 does not leak into call 2), also for
    pointers that are not 16-byte aligned (scalar path) and on a side stream."""
    import torch
    from paper_1909_04504_b200 import binding
    dev = torch.device("cuda", 0)
    ctx, _ = make_ctx(WL.periodic_box_3d((40, 40, 40), seed=8))
    off = _existing_offsets(ctx)
    ctx.close()
    n = off.size - 1
    buf = torch.zeros(n + 3, dtype=torch.int32, device=dev)
    buf[1:n + 1] = torch.from_numpy(np.diff(off.astype(np.int64)).astype(np.uint32).view(np.int32)).to(dev)
    cnt = buf[1:n + 1]                                     # 4-byte aligned only
    o1 = torch.empty(n + 2, dtype=torch.int32, device=dev)
    o2 = torch.empty(n + 2, dtype=torch.int32, device=dev)
    side = torch.cuda.Stream(dev)
    side.wait_stream(torch.cuda.current_stream(dev))
    binding.cell_offsets_static(cnt, o1, stream=side)
    binding.cell_offsets_static(cnt, o2[1:], stream=side)
    side.synchronize()
    assert np.array_equal(o1[:n + 1].cpu().numpy().view(np.uint32), off)
    assert np.array_equal(o2[1:].cpu().numpy().view(np.uint32), off)


def test_static_cell_offsets_limits_and_empty_input():
    import torch
    from paper_1909_04504_b200 import binding
    dev = torch.device("cuda", 0)
    one = torch.full((1,), 7, dtype=torch.int32, device=dev)
    binding.cell_offsets_static(one[:0], one)              # n == 0: offsets[0] = 0
    torch.cuda.synchronize()
    assert int(one.item()) == 0
    with pytest.raises(binding.SphError) as e:             # beyond the static array: refused before anything is launched
        binding.cell_offsets_static(one, one, n=binding.STATIC_SCAN_MAX_N + 1)
    assert e.value.code == -3 and "SPH_STATIC_SCAN_MAX_N" in str(e.value) and str(binding.STATIC_SCAN_MAX_N) in str(e.value)
    L = binding.load()
    assert L.sph_cell_offsets_static(None, 5, None, None) == -1
    assert L.sph_cell_offsets_static(one.data_ptr(), -1, one.data_ptr(), None) == -2
    torch.cuda.synchronize()


def test_static_cell_offsets_at_the_maximum_size():
    """n = SPH_STATIC_SCAN_MAX_N (16,384 tiles, every word of the static table in use), counts with a known closed
    form: counts[i] = i mod 3  ->  offsets[i] = 3 (i div 3) + {0, 0, 1}[i mod 3]."""
    import torch
    from paper_1909_04504_b200 import binding
    dev = torch.device("cuda", 0)
    n = binding.STATIC_SCAN_MAX_N
    i = torch.arange(n + 1, dtype=torch.int64, device=dev)
    cnt = (i[:n] % 3).to(torch.int32)
    want = (3 * (i // 3) + (i % 3 == 2).to(torch.int64)).to(torch.int32)
    out = torch.empty(n + 1, dtype=torch.int32, device=dev)
    for _ in range(2):
        out.fill_(-1)
        binding.cell_offsets_static(cnt, out)
        torch.cuda.synchronize()
        assert torch.equal(out, want)
