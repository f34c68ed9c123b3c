"""Pins for the oracle's SPH kernels (compact support W=0 for |r|>kh; L104: the kernel
approximates a delta function, i.e. integrates to 1).  The paper prints no kernel formula (L209, L435),
so what is pinned is what the mathematics fixes: unit integral in each dimension, compact support,
smoothness at the knots, gradient = derivative of W, and the h-scaling law."""
import math

import numpy as np
import pytest
from scipy import integrate

KERNELS = ["cubic", "quintic", "wendland_c2"]
DIMS = [1, 2, 3]
KNOTS = {"cubic": [1.0, 2.0], "quintic": [1.0, 2.0, 3.0], "wendland_c2": [2.0]}
SUPPORT = {"cubic": 2.0, "quintic": 3.0, "wendland_c2": 2.0}


def _shell(dim, r):
    return {1: 2.0, 2: 2.0 * math.pi * r, 3: 4.0 * math.pi * r * r}[dim]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", DIMS)
@pytest.mark.parametrize("h", [1.0, 0.37])
def test_unit_integral(O, kernel, dim, h):
    k = O.support(kernel)
    assert k == SUPPORT[kernel]
    pts = [q * h for q in KNOTS[kernel]]
    val, _ = integrate.quad(lambda r: O.W(kernel, dim, r, h) * _shell(dim, r), 0.0, k * h,
                            points=pts[:-1] or None, epsabs=1e-14, epsrel=1e-13, limit=200)
    assert abs(val - 1.0) < 1e-12


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", DIMS)
def test_compact_support_and_positivity(O, kernel, dim):
    k, h = O.support(kernel), 0.8
    for q in (k, k + 1e-12, k + 0.5, 10.0):
        assert O.W(kernel, dim, q * h, h) == 0.0
        assert O.dWdr(kernel, dim, q * h, h) == 0.0
    qs = np.linspace(0.0, k - 1e-9, 400)
    w = np.array([O.W(kernel, dim, q * h, h) for q in qs])
    dw = np.array([O.dWdr(kernel, dim, q * h, h) for q in qs])
    assert (w > 0).all() and (np.diff(w) < 0).all()      # positive and monotonically decreasing
    assert (dw[1:] < 0).all() and dw[0] == 0.0             # W'(0) = 0
    # W -> 0 and W' -> 0 continuously at the edge of the support
    assert abs(O.W(kernel, dim, (k - 1e-7) * h, h)) < 1e-12
    assert abs(O.dWdr(kernel, dim, (k - 1e-7) * h, h)) < 1e-5


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", DIMS)
def test_continuity_at_knots(O, kernel, dim):
    h, e = 1.3, 1e-9
    for q in KNOTS[kernel]:
        for f in (O.W, O.dWdr):
            a, b = f(kernel, dim, (q - e) * h, h), f(kernel, dim, (q + e) * h, h)
            scale = abs(f(kernel, dim, 0.5 * h, h))
            assert abs(a - b) < 1e-7 * scale


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", DIMS)
def test_gradient_is_derivative(O, kernel, dim):
    h = 0.9
    k = O.support(kernel)
    for q in np.linspace(0.05, k - 0.05, 41):
        r, d = q * h, 1e-5 * h
        fd = (O.W(kernel, dim, r + d, h) - O.W(kernel, dim, r - d, h)) / (2 * d)
        an = O.dWdr(kernel, dim, r, h)
        assert abs(fd - an) < 1e-7 * abs(O.dWdr(kernel, dim, 0.7 * h, h))


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", DIMS)
def test_h_scaling(O, kernel, dim):
    """W(r,h) = h^-d W(r/h,1) and dW/dr(r,h) = h^-(d+1) dW/dr(r/h,1)."""
    for h in (0.01, 2.5):
        for q in (0.0, 0.3, 1.0, 1.7, 2.4):
            assert O.W(kernel, dim, q * h, h) == pytest.approx(O.W(kernel, dim, q, 1.0) / h ** dim, rel=1e-13)
            assert O.dWdr(kernel, dim, q * h, h) == pytest.approx(O.dWdr(kernel, dim, q, 1.0) / h ** (dim + 1), rel=1e-13)


def test_central_values_closed_form(O):
    """W(0) = sigma_d / h^d with the textbook normalisations (R1)."""
    pi = math.pi
    sig = {("cubic", 1): 2 / 3, ("cubic", 2): 10 / (7 * pi), ("cubic", 3): 1 / pi,
           ("quintic", 1): 66 / 120, ("quintic", 2): 66 * 7 / (478 * pi), ("quintic", 3): 66 / (120 * pi),
           ("wendland_c2", 1): 5 / 8, ("wendland_c2", 2): 7 / (4 * pi), ("wendland_c2", 3): 21 / (16 * pi)}
    for (kernel, dim), s in sig.items():
        assert O.W(kernel, dim, 0.0, 0.5) == pytest.approx(s / 0.5 ** dim, rel=1e-14)


@pytest.mark.parametrize("kernel", KERNELS)
def test_second_moment_isotropy_2d(O, kernel):
    """int W x x^T dV is isotropic and > 0: checked through the radial moment (sanity of the profile)."""
    h = 1.0
    k = O.support(kernel)
    m2, _ = integrate.quad(lambda r: O.W(kernel, 2, r, h) * r * r * _shell(2, r), 0, k * h, epsabs=1e-13)
    assert 0.1 < m2 < 2.0
