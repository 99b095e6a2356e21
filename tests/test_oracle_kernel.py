"""Pins for the oracle's smoothing kernel (oracle/sph_oracle.c: orc_W, orc_dWdr, orc_dWdh).

What fixes them, other than the oracle itself: the normalisation integral (quadrature), the
integration-by-parts identities int x.grad W = -3 and int dW/dh = 0, finite differences, and
hand-evaluated rationals of the Wendland C2 shape polynomial (tests/golden/wendland_c2.txt).
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as O


@pytest.mark.parametrize("h,kappa", [(1.0, 2.0), (0.013, 2.0), (209.6, 2.0), (0.7, 1.87)])
def test_normalisation_by_quadrature(h, kappa):
    H = kappa * h
    val, _ = integrate.quad(lambda r: 4.0 * math.pi * r * r * O.W(r, h, kappa), 0.0, H, epsabs=0, epsrel=1e-12)
    assert abs(val - 1.0) < 1e-10


@pytest.mark.parametrize("h,kappa", [(1.0, 2.0), (0.013, 2.0), (0.7, 1.87)])
def test_gradient_and_dh_integral_identities(h, kappa):
    H = kappa * h
    # int x . grad W d^3x = int r dW/dr 4 pi r^2 dr = -3 int W = -3
    val, _ = integrate.quad(lambda r: 4.0 * math.pi * r ** 3 * O.dWdr(r, h, kappa), 0.0, H, epsrel=1e-12)
    assert abs(val + 3.0) < 1e-9
    # int W = 1 for every h  =>  int dW/dh = 0
    val, _ = integrate.quad(lambda r: 4.0 * math.pi * r * r * O.dWdh(r, h, kappa), 0.0, H, epsrel=1e-12)
    assert abs(val) * h < 1e-9


def test_compact_support_and_smoothness():
    h, k = 0.9, 2.0
    H = k * h
    assert O.W(H, h, k) == 0.0 and O.dWdr(H, h, k) == 0.0
    assert O.W(1.5 * H, h, k) == 0.0 and O.dWdr(1.5 * H, h, k) == 0.0 and O.dWdh(1.5 * H, h, k) == 0.0
    assert O.dWdr(0.0, h, k) == 0.0
    # C2 at the edge: W, W', W'' -> 0 like (1-q)^4, (1-q)^3, (1-q)^2
    e = 1e-4
    assert abs(O.W(H * (1 - e), h, k)) < 1e-14 / H ** 3 * 1e1
    assert abs(O.dWdr(H * (1 - e), h, k)) < 1e-9
    rs = np.linspace(0.0, H, 200)
    w = np.array([O.W(r, h, k) for r in rs])
    assert np.all(np.diff(w) <= 0.0) and np.all(w >= 0.0)
    # dW/dh at r = 0 is -3 W(0)/h (self term of Eq. 3, reading Q5)
    assert abs(O.dWdh(0.0, h, k) + 3.0 * O.W(0.0, h, k) / h) < 1e-15


@pytest.mark.parametrize("q", [0.05, 0.3, 0.5, 0.8, 0.97])
def test_derivatives_match_finite_differences(q):
    h, k = 1.3, 2.0
    r = q * k * h
    d = 1e-6
    fd_r = (O.W(r + d, h, k) - O.W(r - d, h, k)) / (2 * d)
    fd_h = (O.W(r, h + d, k) - O.W(r, h - d, k)) / (2 * d)
    assert abs(fd_r - O.dWdr(r, h, k)) < 1e-8 * abs(O.dWdr(r, h, k)) + 1e-12
    assert abs(fd_h - O.dWdh(r, h, k)) < 1e-7 * abs(O.dWdh(r, h, k)) + 1e-11


def test_golden_rationals(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "wendland_c2.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 5
    h, k = 0.8, 2.0
    H = k * h
    for qn, qd, sn, sd, dn, dd in rows:
        q = int(qn) / int(qd)
        shape = int(sn) / int(sd)
        dshape = int(dn) / int(dd)
        assert abs(O.W(q * H, h, k) - 21.0 / (2 * math.pi * H ** 3) * shape) < 1e-15 / H ** 3 * 10
        assert abs(O.dWdr(q * H, h, k) - 21.0 / (2 * math.pi * H ** 4) * dshape) < 1e-14 / H ** 4 * 10
