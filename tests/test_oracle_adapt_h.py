"""Pins of the oracle's adaptive smoothing-length iteration (Eq. 2): the iteration must
solve the paper's equation M_tot(h) = (4/3) pi (kappa h)^3 rho(h) = const, and it must be Newton's method
(a wrong slope still converges, but only linearly)."""
import numpy as np

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W


def _block(n_side=10, h_factor=1.3, seed=7):
    wl = W.elastic_block(n_side, seed=W.SEED_BASE + seed)
    A = {k: v.astype(np.float64) for k, v in wl.arrays.items()}
    A["h"] = A["h"] * (h_factor / 1.3)
    return wl, A


def _residual(A, h, kappa, n_target):
    """|M_tot / (n_target m) - 1| from an independent density evaluation at h."""
    _, off, lst = O.neighbors(A["x"], A["y"], A["z"], h, kappa, O.GATHER)
    rho, _ = O.density(A["x"], A["y"], A["z"], A["m"], h, kappa, off, lst)
    return np.abs(4.0 / 3.0 * np.pi * (kappa * h) ** 3 * rho / (n_target * A["m"]) - 1.0)


def test_fixed_point_solves_eq2():
    wl, A = _block(10, 1.1)
    n_target = 60.0
    h, _, _, hist = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, n_target, 12)
    res = _residual(A, h, 2.0, n_target)
    # h lives in fp32 between iterations: the residual floor is a few fp32 ulps times d ln M / d ln h ~ 3
    assert res.max() < 5e-6
    assert hist[-1] < 2e-6 and hist[0] > 1e-2


def test_convergence_is_quadratic():
    """Newton's method squares the error; with a wrong slope (e.g. Omega dropped or the factor 3
    missing) the error ratio stays constant.  Interior particles only (smooth rho(h))."""
    wl, A = _block(12, 1.2)
    n_target = 70.0
    r = np.sqrt(sum((A[k] - A[k].mean()) ** 2 for k in ("x", "y", "z")))
    inner = r < 0.25 * r.max()
    res = []
    for it in (1, 2, 3):
        h, *_ = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, n_target, it)
        res.append(_residual(A, h, 2.0, n_target)[inner].max())
    assert res[0] < 0.1
    assert res[1] < 4.0 * res[0] ** 2 + 1e-6          # quadratic: e1 ~ C e0^2 with C = O(1)
    assert res[2] < 4.0 * res[1] ** 2 + 2e-6


def test_continuum_value_on_a_dense_lattice():
    """rho ~ rho0 inside a uniform lattice, so Eq. 2 gives h* = (n m / ((4/3) pi kappa^3 rho0))^(1/3)."""
    wl, A = _block(14, 1.3)
    n_target = 65.0
    h, rho, _, _ = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, n_target, 8)
    r = np.sqrt(sum((A[k] - A[k].mean()) ** 2 for k in ("x", "y", "z")))
    inner = r < 0.2 * r.max()
    rho0 = wl.params.materials[0].rho0
    h_star = (n_target * A["m"][inner] / (4.0 / 3.0 * np.pi * 8.0 * rho0)) ** (1.0 / 3.0)
    assert np.abs(h[inner] / h_star - 1.0).max() < 0.02


def test_more_mass_in_the_kernel_means_larger_h_and_scaling():
    wl, A = _block(8, 1.3)
    a, *_ = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, 50.0, 8)
    b, *_ = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, 80.0, 8)
    assert np.all(b > a)
    # similarity: lengths x s, masses x s^3  =>  h x s, rho unchanged
    s = 4.0      # a power of two: the fp32 roundings of the scaled problem are the same
    c, rho_c, *_ = O.adapt_h(s * A["x"], s * A["y"], s * A["z"], s ** 3 * A["m"], s * A["h"], 2.0, 50.0, 8)
    a2, rho_a, *_ = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, 50.0, 8)
    assert np.allclose(c, s * a2, rtol=1e-6)
    assert np.allclose(rho_c, rho_a, rtol=1e-9)


def test_step_limits_and_zero_iterations():
    wl, A = _block(6, 1.3)
    h0 = A["h"].astype(np.float32).astype(np.float64)
    h, rho, om, hist = O.adapt_h(A["x"], A["y"], A["z"], A["m"], 0.4 * A["h"], 2.0, 60.0, 1)
    assert np.all(h <= 1.25 * 0.4 * h0 * (1 + 1e-6)) and hist[0] == 0.25     # far too small: limited growth
    h, rho, om, hist = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], 2.0, 60.0, 0)
    assert np.array_equal(h, h0) and rho is None and hist == []
