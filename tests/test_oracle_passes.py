"""Pins for the oracle's pair passes O2 (density), O4 (gradients), O5 (forces).

None of these re-types an oracle formula.  They use what the paper and the mathematics fix:
the continuum statements rho dv/dt = d sigma/dx (Eq. 16) and
rho du/dt = sigma : eps_dot (Eq. 17) on a regular lattice interior; exact
antisymmetry identities (linear momentum, angular momentum for central forces, total energy);
exactness of G = F.C for linear velocity fields; one hand-evaluated
two-particle viscosity case (tests/golden/av_pair.txt).
"""
import os
from types import SimpleNamespace

import numpy as np
import pytest

from oracle import oracle as O


def lattice(n, dx=1.0, jitter=0.0, seed=0):
    g = (np.arange(n) + 0.5) * dx
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), z.ravel()])
    if jitter:
        p = p + jitter * dx * (2 * np.random.default_rng(seed).random(p.shape) - 1)
    return p.astype(np.float32).astype(np.float64)


def params(**kw):
    d = dict(kappa=2.0, alpha=1.0, beta=2.0, eps_av=0.01, eta_C=0.3, eta_a=0.0,
             flags=O.FLAG_STRENGTH | O.FLAG_CORRECTION_TENSOR, materials=[])
    d.update(kw)
    return SimpleNamespace(**d)


def interior(p, n, dx, margin):
    lo, hi = margin * dx, (n - margin) * dx
    return np.all((p > lo) & (p < hi), axis=0)


# ------------------------------------------------------------------ density
def test_density_continuum_limit():
    # sum_j m W -> int rho W = rho0 and Omega -> 1 as h/dx grows (kernel sum -> integral)
    n, dx, rho0 = 16, 1.0, 1000.0
    p = lattice(n, dx)
    N = p.shape[1]
    m = np.full(N, rho0 * dx ** 3)
    errs = []
    for eta in (1.3, 2.0, 3.0):
        h = np.full(N, eta * dx)
        c, o, l = O.neighbors(p[0], p[1], p[2], h, 2.0, O.GATHER, "grid")
        rho, om = O.density(p[0], p[1], p[2], m, h, 2.0, o, l)
        i = np.argmin(((p - p.mean(axis=1, keepdims=True)) ** 2).sum(axis=0))
        errs.append((abs(rho[i] / rho0 - 1.0), abs(om[i] - 1.0)))
    assert errs[0][0] < 2e-2 and errs[1][0] < 2e-3 and errs[2][0] < 2e-4
    assert errs[0][0] > errs[1][0] > errs[2][0]
    assert errs[2][1] < 1e-3


def test_density_uses_h_i_and_includes_self():
    p = np.array([[0.0, 1.0], [0.0, 0.0], [0.0, 0.0]])
    m = np.array([2.0, 3.0])
    h_small = np.array([0.4, 5.0])           # H_0 = 0.8 < r = 1: particle 0 sees only itself
    c, o, l = O.neighbors(p[0], p[1], p[2], h_small, 2.0, O.GATHER)
    rho, om = O.density(p[0], p[1], p[2], m, h_small, 2.0, o, l)
    assert c.tolist() == [1, 2]
    assert rho[0] == pytest.approx(m[0] * O.W(0.0, 0.4))                 # self term only, own h
    assert om[0] == pytest.approx(0.0, abs=1e-14)                        # 1 + h/(3 rho) m (-3 W(0)/h)
    assert rho[1] == pytest.approx(m[1] * O.W(0.0, 5.0) + m[0] * O.W(1.0, 5.0))


# ------------------------------------------------------------------ forces: exact identities
def _random_state(n=7, jitter=0.2, seed=3, strength=True):
    rng = np.random.default_rng(seed)
    p = lattice(n, 1.0, jitter, seed)
    N = p.shape[1]
    st = dict(
        m=1.0 + rng.random(N), h=0.9 + 0.6 * rng.random(N),
        v=rng.standard_normal((3, N)), rho=1.0 + rng.random(N), omega=0.8 + 0.4 * rng.random(N),
        P=rng.standard_normal(N), cs=1.0 + rng.random(N),
        S=(rng.standard_normal((5, N)) if strength else np.zeros((5, N))))
    return p, st


def _forces(p, st, prm, g=None):
    c, o, l = O.neighbors(p[0], p[1], p[2], st["h"], prm.kappa, O.SYMMETRIC)
    return O.forces(prm, p[0], p[1], p[2], st["m"], st["h"], st["v"][0], st["v"][1], st["v"][2],
                    st["rho"], st["omega"], st["P"], st["cs"], st["S"], g, o, l)


def test_linear_momentum_is_conserved_exactly():
    p, st = _random_state()
    a, dudt, mumax = _forces(p, st, params())
    tot = (st["m"][None] * a).sum(axis=1)
    scale = np.abs(st["m"][None] * a).sum(axis=1)
    assert np.all(np.abs(tot) < 1e-13 * scale)
    assert mumax.max() > 0.0                                    # AV was active


def test_angular_momentum_conserved_for_central_part_only():
    p, st = _random_state(strength=False)
    a, _, _ = _forces(p, st, params(flags=O.FLAG_CORRECTION_TENSOR))
    L = (st["m"][None] * np.cross(p.T, a.T).T).sum(axis=1)
    scale = np.abs(st["m"][None] * np.cross(p.T, a.T).T).sum(axis=1)
    assert np.all(np.abs(L) < 1e-12 * scale)
    # with deviatoric stress the pair force is not central: torque != 0
    p, st = _random_state(strength=True)
    a, _, _ = _forces(p, st, params())
    L = (st["m"][None] * np.cross(p.T, a.T).T).sum(axis=1)
    assert np.abs(L).max() > 1e-6 * scale.max()


def test_strength_flag_off_ignores_S():
    p, st = _random_state(strength=True)
    a1, du1, _ = _forces(p, st, params(flags=0))
    st2 = dict(st); st2["S"] = np.zeros_like(st["S"])
    a2, du2, _ = _forces(p, st2, params())
    assert np.array_equal(a1, a2) and np.array_equal(du1, du2)


def test_total_energy_identity():
    # sum_i m_i (v_i . a_i + du_i/dt) = 0 for hydro + S + AV: pins the relative signs of
    # Eq. 18 vs 19 and Eq. 7 vs 8 and reading Q7 (hydro du/dt = Eq. 19 with S -> -P delta)
    p, st = _random_state()
    a, dudt, _ = _forces(p, st, params())
    e = st["m"] * ((st["v"] * a).sum(axis=0) + dudt)
    assert abs(e.sum()) < 1e-12 * np.abs(e).sum()
    # and separately without viscosity
    a, dudt, _ = _forces(p, st, params(alpha=0.0, beta=0.0))
    e = st["m"] * ((st["v"] * a).sum(axis=0) + dudt)
    assert abs(e.sum()) < 1e-12 * np.abs(e).sum()


def test_external_acceleration_is_added():
    p, st = _random_state()
    N = p.shape[1]
    g = np.random.default_rng(5).standard_normal((3, N))
    a0, _, _ = _forces(p, st, params())
    a1, _, _ = _forces(p, st, params(), g)
    assert np.allclose(a1 - a0, g, rtol=0, atol=1e-12 * np.abs(a0).max())


# ------------------------------------------------------------------ forces: continuum limits
def _uniform_lattice_state(n=14, eta=1.6):
    p = lattice(n, 1.0)
    N = p.shape[1]
    rho0 = 3.0
    st = dict(m=np.full(N, rho0), h=np.full(N, eta), v=np.zeros((3, N)), rho=np.full(N, rho0),
              omega=np.ones(N), P=np.zeros(N), cs=np.ones(N), S=np.zeros((5, N)))
    return p, st, rho0, interior(p, n, 1.0, 2 * eta + 0.6)


def test_pressure_gradient_gives_minus_gradP_over_rho():
    # Eq. 16 with sigma = -P delta: dv/dt = -grad P / rho
    p, st, rho0, inner = _uniform_lattice_state()
    k = np.array([0.7, -0.3, 0.2])
    st["P"] = 5.0 + k @ p
    a, _, _ = _forces(p, st, params(alpha=0.0, beta=0.0))
    expect = -k / rho0
    assert inner.sum() > 20
    assert np.allclose(a[:, inner], expect[:, None], rtol=0, atol=0.01 * np.abs(expect).max())


def test_shear_stress_gradient_gives_plus_divS_over_rho():
    # Eq. 16: rho dv^x/dt = d S^{xy}/dy ; rho dv^y/dt = d S^{xy}/dx ; rho dv^z/dt = d S^{zz}/dz
    p, st, rho0, inner = _uniform_lattice_state()
    st["S"][2] = 0.4 * p[1] - 0.9 * p[0]            # S^{xy} = 0.4 y - 0.9 x
    st["S"][0] = 0.25 * p[2]                         # S^{xx} = 0.25 z  => S^{zz} = -0.25 z
    a, _, _ = _forces(p, st, params(alpha=0.0, beta=0.0))
    expect = np.array([0.4, -0.9, -0.25]) / rho0
    assert np.allclose(a[:, inner], expect[:, None], rtol=0, atol=0.01 * np.abs(expect).max())


def test_energy_rate_is_sigma_contract_strain_rate():
    # Eq. 17: rho du/dt = sigma^{ab} eps_dot^{ab} for uniform sigma and v = A x
    p, st, rho0, inner = _uniform_lattice_state()
    A = np.array([[0.3, 0.5, -0.2], [0.1, -0.4, 0.6], [0.7, 0.2, 0.15]])
    st["v"] = A @ p
    P0 = 2.0
    S5 = np.array([0.3, -0.5, 0.8, -0.2, 0.4])
    st["P"][:] = P0
    st["S"] = np.repeat(S5[:, None], p.shape[1], axis=1)
    S3 = np.array([[S5[0], S5[2], S5[3]], [S5[2], S5[1], S5[4]], [S5[3], S5[4], -S5[0] - S5[1]]])
    sigma = -P0 * np.eye(3) + S3
    eps = 0.5 * (A + A.T)
    expect = (sigma * eps).sum() / rho0
    _, dudt, _ = _forces(p, st, params(alpha=0.0, beta=0.0))
    assert np.allclose(dudt[inner], expect, rtol=0, atol=0.01 * abs(expect))


# ------------------------------------------------------------------ artificial viscosity
def test_av_hand_evaluated_pair(golden_dir):
    gold = dict((l.split()[0], float(l.split()[1])) for l in open(os.path.join(golden_dir, "av_pair.txt"))
                if l.strip() and l[0] != "#")
    p = np.array([[1.0, 0.0], [0.0, 0.0], [0.0, 0.0]])
    st = dict(m=np.ones(2), h=np.ones(2), v=np.array([[-1.0, 0.0], [0.0, 0.0], [0.0, 0.0]]),
              rho=np.ones(2), omega=np.ones(2), P=np.zeros(2), cs=np.ones(2), S=np.zeros((5, 2)))
    a, dudt, mumax = _forces(p, st, params())
    assert a[0, 0] == pytest.approx(gold["ax_i"], rel=1e-12)
    assert a[0, 1] == pytest.approx(-gold["ax_i"], rel=1e-12)
    assert dudt[0] == pytest.approx(gold["dudt_i"], rel=1e-12) and dudt[1] == pytest.approx(gold["dudt_i"], rel=1e-12)
    assert mumax[0] == pytest.approx(gold["mu_abs"], rel=1e-12)
    # receding pair: no viscosity at all
    st["v"] = -st["v"]
    a, dudt, mumax = _forces(p, st, params())
    assert np.all(a == 0.0) and np.all(dudt == 0.0) and np.all(mumax == 0.0)


# ------------------------------------------------------------------ gradients
def _grad(p, st, prm):
    c, o, l = O.neighbors(p[0], p[1], p[2], st["h"], prm.kappa, O.SYMMETRIC)
    return O.gradients(p[0], p[1], p[2], st["m"], st["h"], st["v"][0], st["v"][1], st["v"][2],
                       st["rho"], st["omega"], prm.kappa, o, l)


def test_linear_field_is_reproduced_exactly_everywhere():
    # v = A x + b on jittered particles with random m, h, rho, Omega, including the free surface:
    # F = A . C^-1 exactly, so G = F . C = A to rounding (pins the -1/2, the sign of v_ij and
    # x_ij, and F.C rather than C.F)
    p, st = _random_state(n=7, jitter=0.25, seed=11)
    A = np.array([[0.3, 1.5, -0.2], [-0.1, -0.4, 0.6], [0.7, 0.2, 0.15]])
    st["v"] = A @ p + np.array([[3.0], [-2.0], [1.0]])
    F, Cinv = _grad(p, st, params())
    G, cflag = O.correct_gradient(F, Cinv, O.FLAG_CORRECTION_TENSOR)
    assert cflag.sum() == 0
    assert np.abs(G - A.reshape(9, 1)).max() < 1e-10
    # C.F would NOT reproduce A (A and C^-1 do not commute)
    n = p.shape[1]
    Fm = F.T.reshape(n, 3, 3); Cm = np.linalg.inv(Cinv.T.reshape(n, 3, 3))
    wrong = np.einsum("nag,ngb->nab", Cm, Fm)
    assert np.abs(wrong - A[None]).max() > 1e-3
    # rigid translation: G = 0; rigid rotation: eps_dot = 0
    st["v"] = np.repeat(np.array([[3.0], [-2.0], [1.0]]), n, axis=1)
    F, Cinv = _grad(p, st, params())
    assert np.abs(F).max() < 1e-12
    Wm = np.array([[0.0, -0.7, 0.2], [0.7, 0.0, -0.5], [-0.2, 0.5, 0.0]])
    st["v"] = Wm @ p
    F, Cinv = _grad(p, st, params())
    G, _ = O.correct_gradient(F, Cinv, O.FLAG_CORRECTION_TENSOR)
    eps, R = O.strain_and_rotation(G)
    assert np.abs(eps).max() < 1e-11 and np.abs(R - Wm[None]).max() < 1e-11


def test_correction_tensor_is_identity_in_the_continuum_and_off_means_G_equals_F():
    p, st, rho0, inner = _uniform_lattice_state(n=14, eta=1.6)
    A = np.array([[0.0, 100.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    st["v"] = A @ p
    F, Cinv = _grad(p, st, params())
    I9 = np.eye(3).reshape(9, 1)
    assert np.abs(Cinv[:, inner] - I9).max() < 0.01          # Eq. 21 -> d x^a / d x^b = delta
    assert np.abs(F[:, inner] - A.reshape(9, 1)).max() < 0.01 * 100.0
    G, cflag = O.correct_gradient(F, Cinv, 0)
    assert np.array_equal(G, F) and cflag.all()


def test_singular_correction_falls_back_to_identity():
    # coplanar particles: C^-1 has a zero row/column
    g = np.arange(5, dtype=np.float64)
    x, y = np.meshgrid(g, g, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), np.zeros(25)])
    st = dict(m=np.ones(25), h=np.full(25, 1.3), v=np.stack([p[1], np.zeros(25), np.zeros(25)]),
              rho=np.ones(25), omega=np.ones(25))
    F, Cinv = _grad(p, st, params())
    G, cflag = O.correct_gradient(F, Cinv, O.FLAG_CORRECTION_TENSOR)
    assert cflag.all() and np.array_equal(G, F)
    # an isolated particle: everything zero, flagged
    F0 = np.zeros((9, 1)); G0, f0 = O.correct_gradient(F0, F0.copy(), O.FLAG_CORRECTION_TENSOR)
    assert f0.tolist() == [1] and np.all(G0 == 0)


# ------------------------------------------------------------------ two particles: Eq. 1, 3, 18, 19 by hand
def test_two_particle_closed_forms():
    """Two particles on the x axis, different m, h, rho, Omega, P and a full S: every sum has one term, so
    Eq. 1, 3 and Eq. 18, 19 can be written out with the scalar kernel
    functions (pinned in test_oracle_kernel.py).  A wrong sign, a swapped h_i / h_j, a missing Omega or a
    transposed stress index fails here.  No artificial viscosity (receding pair)."""
    r = 0.7
    p = np.array([[0.0, r], [0.0, 0.0], [0.0, 0.0]])
    m = np.array([2.0, 3.0]); h = np.array([0.5, 0.6]); kap = 2.0
    # density and Omega
    c, o, l = O.neighbors(p[0], p[1], p[2], h, kap, O.GATHER)
    rho, om = O.density(p[0], p[1], p[2], m, h, kap, o, l)
    for i, j in ((0, 1), (1, 0)):
        rho_i = m[i] * O.W(0.0, h[i], kap) + m[j] * O.W(r, h[i], kap)
        dh = m[i] * O.dWdh(0.0, h[i], kap) + m[j] * O.dWdh(r, h[i], kap)
        assert rho[i] == pytest.approx(rho_i, rel=1e-13)
        assert om[i] == pytest.approx(1.0 + h[i] / (3.0 * rho_i) * dh, rel=1e-12)
    # forces with prescribed rho, Omega, P, S (five stored components xx, yy, xy, xz, yz; zz = -xx - yy)
    rho_in = np.array([1.3, 0.9]); om_in = np.array([0.95, 1.1]); P = np.array([0.4, -0.2])
    S = np.array([[0.3, -0.1], [0.2, 0.25], [0.15, -0.05], [-0.2, 0.1], [0.05, 0.3]])
    v = np.array([[-0.5, 0.5], [0.2, -0.1], [0.0, 0.3]])              # v_ij . x_ij > 0: receding, Pi = 0
    prm = params()
    cs_, os_, ls_ = O.neighbors(p[0], p[1], p[2], h, kap, O.SYMMETRIC)
    a, dudt, mumax = O.forces(prm, p[0], p[1], p[2], m, h, v[0], v[1], v[2], rho_in, om_in, P,
                              np.array([1.0, 1.0]), S, None, os_, ls_)

    def sigma(k):
        sxx, syy, sxy, sxz, syz = S[:, k]
        return np.array([[sxx, sxy, sxz], [sxy, syy, syz], [sxz, syz, -sxx - syy]]) - P[k] * np.eye(3)
    for i, j in ((0, 1), (1, 0)):
        xij = p[:, i] - p[:, j]
        e = xij / r                                                      # grad_i W_ij(h) = W'(r, h) x_ij / r
        gi = O.dWdr(r, h[i], kap) * e
        gj = O.dWdr(r, h[j], kap) * e
        a_i = m[j] * (sigma(i) @ gi / (om_in[i] * rho_in[i] ** 2) + sigma(j) @ gj / (om_in[j] * rho_in[j] ** 2))
        vij = v[:, i] - v[:, j]
        du_i = -m[j] * vij @ (sigma(i) @ gi) / (om_in[i] * rho_in[i] ** 2)
        assert np.allclose(a[:, i], a_i, rtol=1e-12, atol=1e-14)
        assert dudt[i] == pytest.approx(du_i, rel=1e-12)
    assert np.all(mumax == 0.0)
    assert np.allclose(m[0] * a[:, 0] + m[1] * a[:, 1], 0.0, atol=1e-13)
