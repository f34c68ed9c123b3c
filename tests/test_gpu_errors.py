"""-m gpu: the error behaviour include/sph.h states for the boundary: argument errors are reported synchronously by
the call, device-side conditions (a particle outside a non-periodic box, a non-finite result) by the next [sync]
call; n == 0 arrays are legal; nothing falls back to a CPU path."""
import numpy as np
import pytest

from gpu_helpers import make_ctx

pytestmark = pytest.mark.gpu

ERR_NULL, ERR_BAD_ARG, ERR_CAPACITY, ERR_STALE, ERR_OOD, ERR_NONFINITE = -1, -2, -3, -4, -5, -6


def _ctx(wl, **over):
    from paper_1909_04504_b200 import binding
    return binding.SphContext.from_workload(wl, **over)


def test_calls_before_a_build_are_stale(WL):
    from paper_1909_04504_b200 import binding
    wl = WL.random_box(n=600, dim=2, periodic=True, seed=1)
    ctx = _ctx(wl)
    for call in (lambda: ctx.pc_step(wl.dt, 1, "summation"), lambda: ctx.summation_density(0, 1),
                 lambda: ctx.wcsph_accel(0, 1)):
        with pytest.raises(binding.SphError) as e:
            call()
        assert e.value.code == ERR_STALE
    ctx.close()


def test_argument_errors_are_synchronous(WL):
    from paper_1909_04504_b200 import binding
    wl = WL.random_box(n=3000, dim=3, periodic=True, seed=2)
    ctx = _ctx(wl, capacity=[50])
    with pytest.raises(binding.SphError) as e:                      # more particles than the capacity given at creation
        ctx.nnps_build(binding.device_arrays(wl), [False])
    assert e.value.code == ERR_CAPACITY
    ctx.close()
    ctx, arrays = make_ctx(wl)
    for call, code in ((lambda: ctx.summation_density(0, 0), ERR_BAD_ARG),        # empty source mask
                       (lambda: ctx.summation_density(0, 2), ERR_BAD_ARG),        # names array 1 of a 1-array context
                       (lambda: ctx.pc_step(wl.dt, -1, "summation"), ERR_BAD_ARG),
                       (lambda: ctx.pc_step(float("nan"), 1, "summation"), ERR_BAD_ARG)):
        with pytest.raises(binding.SphError) as e:
            call()
        assert e.value.code == code
    assert ctx.L.sph_wcsph_accel(ctx.ctx, 3, 1, None, None, None, None, 0) == ERR_BAD_ARG      # no such destination (C call)
    assert ctx.L.sph_summation_density(None, 0, 1, None, None, 0) == ERR_NULL                   # no context
    bad = dict(arrays[0]); bad["x"] = None
    with pytest.raises(binding.SphError) as e:                      # a required pointer is missing
        ctx.nnps_build([bad], [False])
    assert e.value.code == ERR_NULL
    ctx.close()
    with pytest.raises(binding.SphError) as e:                      # bad creation parameters
        binding.SphContext(dim=4, lo=(0, 0, 0), hi=(1, 1, 1), periodic=(0, 0, 0), kernel="cubic", rho0=1.0, c0=10.0, capacity=[8])
    assert e.value.code == ERR_BAD_ARG


def test_periodic_axis_needs_three_cells(WL):
    from paper_1909_04504_b200 import binding
    wl = WL.random_box(n=50, dim=2, periodic=True, seed=3, kernel="cubic", h_mean=0.2)      # 2 h = 0.4: 2 cells per axis
    ctx = _ctx(wl)
    with pytest.raises(binding.SphError) as e:
        ctx.nnps_build(binding.device_arrays(wl), [False])
    assert e.value.code == ERR_BAD_ARG and "3 cells" in str(e.value)
    ctx.close()


def test_out_of_domain_and_nonfinite_are_reported_by_the_next_sync(WL):
    from paper_1909_04504_b200 import binding
    wl = WL.random_box(n=500, dim=2, periodic=False, seed=4)
    wl.arrays[0].x[7] = np.float32(wl.hi[0] + 0.5)                  # outside the non-periodic box
    ctx = _ctx(wl)
    ctx.nnps_build(binding.device_arrays(wl), [False])              # enqueued: the condition is a device flag
    with pytest.raises(binding.SphError) as e:
        ctx.synchronize()
    assert e.value.code == ERR_OOD
    ctx.close()
    wl = WL.random_box(n=500, dim=2, periodic=True, seed=5)
    wl.arrays[0].m[:] = 0.0                                         # rho = 0 everywhere -> p/rho^2 is not finite
    ctx = _ctx(wl)
    ctx.nnps_build(binding.device_arrays(wl), [False])
    ctx.summation_density(0, 1)
    with pytest.raises(binding.SphError) as e:
        ctx.synchronize()
    assert e.value.code == ERR_NONFINITE
    ctx.close()


def test_empty_arrays_are_legal(WL):
    from paper_1909_04504_b200 import binding
    import torch
    wl = WL.random_box(n=3000, dim=3, periodic=True, seed=6, two_arrays=True)
    full = binding.device_arrays(wl)
    empty = {k: torch.empty(0, dtype=torch.float32, device="cuda") for k in full[1]}
    ctx = _ctx(wl)
    ctx.nnps_build([full[0], empty], [False, True])                 # second array has no particles
    rho, _ = ctx.summation_density(0, 3)
    assert np.isfinite(rho.cpu().numpy()).all()
    ctx.pc_step(wl.dt, 2, "summation")
    ctx.synchronize()
    assert ctx.get_stats().n_particles == wl.arrays[0].n
    ctx.nnps_build([{k: v[:0] for k, v in full[0].items()}, empty], [False, True])   # everything empty
    ctx.pc_step(wl.dt, 1, "summation")
    ctx.synchronize()
    ctx.close()
