"""Pins for the oracle's per-particle steps: EOS stand-in, shear modulus (Eq. 30), yield
strength (Eq. 34-37), plastic projection (Eq. 31-33), stress rate (Eq. 13 / 25-29)."""
import math
from types import SimpleNamespace

import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200.workloads import Material


def P_(mats, flags=O.FLAG_STRENGTH | O.FLAG_CORRECTION_TENSOR):
    return SimpleNamespace(kappa=2.0, alpha=1.0, beta=2.0, eps_av=0.01, eta_C=0.3, eta_a=0.0,
                           flags=flags, materials=mats)


Z = np.zeros(1, dtype=np.int32)


def Y_of(P, T, mat=Material(), **kw):
    prm = P_([mat])
    P = np.atleast_1d(np.asarray(P, dtype=np.float64))
    T = np.broadcast_to(np.asarray(T, dtype=np.float64), P.shape)
    return O.yield_strength(prm, P, T, np.zeros(P.shape[0], np.int32))


def test_yield_limits_eq34():
    m = Material(Y0=10e6, Ym=3.5e9, mu_i=1.5)
    cold = 1e-6                                   # T -> 0: softening factor -> tanh(inf) = 1
    assert Y_of(0.0, cold, m)[0] == pytest.approx(10e6, rel=1e-12)          # Y_i(P=0) = Y0
    assert Y_of(1e16, cold, m)[0] == pytest.approx(3.5e9, rel=1e-5)         # Y_i(P->inf) = Ym
    dP = 1.0
    slope = (Y_of(dP, cold, m)[0] - Y_of(0.0, cold, m)[0]) / dP
    assert slope == pytest.approx(1.5, rel=1e-6)                            # dY_i/dP(0) = mu_i
    # negative pressures are clipped to zero
    assert Y_of(-5e8, cold, m)[0] == pytest.approx(10e6, rel=1e-12)
    # monotone and bounded
    Ps = np.logspace(3, 12, 50)
    Ys = Y_of(Ps, cold, m)
    assert np.all(np.diff(Ys) > 0) and np.all(Ys < 3.5e9) and np.all(Ys > 10e6)


def test_yield_min_rule_eq36():
    m = Material(Y0=0.0, Ym=3.5e9, mu_i=2.0, mu_d=0.8)
    cold = 1e-6
    P = np.array([0.0, 1e6, 1e9, 1e12])
    Y = Y_of(P, cold, m)
    Yi = Y_of(P, cold, Material(Y0=0.0, Ym=3.5e9, mu_i=2.0))
    assert np.allclose(Y, np.minimum(Yi, 0.8 * P), rtol=1e-14)
    assert Y[0] == 0.0 and Y[1] == pytest.approx(0.8e6) and Y[3] == pytest.approx(Yi[3])
    # with cohesion and a finite mu_d, Eq. 36 verbatim kills the cohesion at P = 0 (reading Q10)
    assert Y_of(0.0, cold, Material(Y0=1e7, mu_d=0.8))[0] == 0.0


def test_thermal_softening_limits_eq37():
    m = Material(Y0=10e6, xi=1.2, Tmelt=1500.0)
    base = Y_of(2e8, 1e-9, m)[0]
    assert Y_of(2e8, 0.0, m)[0] == base                       # T = 0: factor 1 (reading Q11)
    assert Y_of(2e8, 1500.0, m)[0] == 0.0                     # T = T_melt: 0
    assert Y_of(2e8, 1600.0, m)[0] == 0.0                     # above: clamped, not negative
    assert Y_of(2e8, 750.0, m)[0] == pytest.approx(base * math.tanh(1.2), rel=1e-14)
    Ts = np.linspace(100.0, 1500.0, 30)
    assert np.all(np.diff(Y_of(np.full(30, 2e8), Ts, m)) < 0)


def test_shear_modulus_eq30():
    rho = np.array([2700.0]); cs = np.array([3000.0])
    g = O.shear_modulus(P_([Material(Gamma=0.0, nu=0.25)]), rho, cs, Z)
    assert g[0] == pytest.approx(0.6 * 2700.0 * 9e6, rel=1e-14)           # nu = 1/4 => Gamma = 0.6 K
    g = O.shear_modulus(P_([Material(Gamma=0.0, nu=0.5)]), rho, cs, Z)
    assert g[0] == 0.0                                                     # incompressible limit
    g = O.shear_modulus(P_([Material(Gamma=22.7e9)]), rho, cs, Z)
    assert g[0] == 22.7e9


def test_eos_standin_and_pclip():
    mats = [Material(rho0=2700.0, c0=3000.0, cv=1000.0), Material(rho0=1000.0, c0=1500.0, cv=4000.0)]
    rho = np.array([2800.0, 900.0]); u = np.array([3e5, 8e5]); mat = np.array([0, 1], np.int32)
    P, c, T = O.eos(P_(mats), rho, u, mat)
    assert P.tolist() == [9e6 * 100.0, 1500.0 ** 2 * -100.0] and c.tolist() == [3000.0, 1500.0]
    assert T.tolist() == [300.0, 200.0]
    P, _, _ = O.eos(P_(mats, flags=O.FLAG_PCLIP_GLOBAL), rho, u, mat)
    assert P.tolist() == [9e8, 0.0]


def test_projection_invariants():
    rng = np.random.default_rng(0)
    S = rng.standard_normal((5, 200)) * 3.0
    Y = np.abs(rng.standard_normal(200)) * 2.0
    Y[:5] = 0.0
    Sp, f = O.project(S, Y)
    sj = np.sqrt(O.J2(Sp))
    assert np.all(sj <= Y * (1 + 1e-12))
    below = np.sqrt(O.J2(S)) <= Y
    assert below.any() and (~below).any()
    assert np.array_equal(Sp[:, below], S[:, below]) and np.all(f[below] == 1.0)
    assert np.allclose(sj[~below], Y[~below], rtol=1e-12)
    # direction unchanged, idempotent, Y = 0 -> S = 0 exactly
    nz = ~below & (Y > 0)
    assert np.allclose(Sp[:, nz] / np.sqrt(O.J2(Sp))[nz], S[:, nz] / np.sqrt(O.J2(S))[nz], rtol=1e-12)
    Sp2, f2 = O.project(Sp, Y)
    assert np.allclose(Sp2, Sp, rtol=1e-12, atol=0)
    assert np.all(Sp[:, :5] == 0.0)
    # J2 = 0: f = 1, no NaN (reading Q12)
    S0, f0 = O.project(np.zeros((5, 3)), np.array([0.0, 1.0, 2.0]))
    assert np.all(S0 == 0) and np.all(f0 == 1.0)
    # J2 from five components == 1/2 S:S of the full tensor
    S3 = O._S3(S)
    assert np.allclose(O.J2(S), 0.5 * (S3 * S3).sum(axis=(1, 2)), rtol=1e-14)
    assert np.allclose(np.trace(S3, axis1=1, axis2=2), 0.0, atol=1e-15)


def test_stress_rate_component_form_equals_eq13():
    rng = np.random.default_rng(1)
    n = 50
    G = rng.standard_normal((9, n)); S = rng.standard_normal((5, n)); Gam = 1.0 + rng.random(n)
    for flags in (0, O.FLAG_JAUMANN_AS_PRINTED):
        dS, dS3, eps2 = O.stress_rate(G, S, Gam, flags)
        comp = O.stress_rate_components(G, S, Gam, flags)
        assert np.allclose(dS, comp, rtol=1e-13, atol=1e-13)
        assert np.allclose(np.trace(dS3, axis1=1, axis2=2), 0.0, atol=1e-13)       # traceless
        assert np.allclose(dS3, np.transpose(dS3, (0, 2, 1)), atol=1e-14)          # symmetric
        # rotation terms do no work on S: S : dS_rot = 0
        rot, _, _ = O.stress_rate(G, S, np.zeros(n), flags)
        rot3 = O._S3(rot)
        assert np.allclose((O._S3(S) * rot3).sum(axis=(1, 2)), 0.0, atol=1e-12)
    eps, _ = O.strain_and_rotation(G)
    assert np.allclose(eps2, 0.5 * (eps * eps).sum(axis=(1, 2)))


def test_hooke_pure_shear_and_special_cases():
    n = 1
    Gam = np.array([22.7e9])
    G = np.zeros((9, n)); G[1] = 100.0                       # dv^x/dy = 100 1/s (configs[0] shear)
    dS, _, eps2 = O.stress_rate(G, np.zeros((5, n)), Gam, 0)
    # Hooke (Eq. 12): S^{xy} = 2 Gamma eps^{xy}, eps^{xy} = gamma/2  =>  dS^{xy}/dt = Gamma * 100
    assert dS[:, 0].tolist() == [0.0, 0.0, 22.7e9 * 100.0, 0.0, 0.0]
    assert eps2[0] == pytest.approx(0.5 * 2 * 50.0 ** 2)
    # hydrostatic compression G = lambda I, S = 0: no deviatoric growth
    G = np.zeros((9, n)); G[0] = G[4] = G[8] = -3.0
    dS, _, _ = O.stress_rate(G, np.zeros((5, n)), Gam, 0)
    assert np.all(dS == 0.0)
    # rigid rotation: the elastic (Hooke) part vanishes identically
    Wm = np.array([[0.0, -0.7, 0.2], [0.7, 0.0, -0.5], [-0.2, 0.5, 0.0]])
    dS, _, eps2 = O.stress_rate(Wm.reshape(9, 1), np.zeros((5, n)), Gam, 0)
    assert np.all(dS == 0.0) and eps2[0] == 0.0
    # uniaxial strain rate G^{xx} = e: dS^{xx} = 2 Gamma (e - e/3) = 4/3 Gamma e
    G = np.zeros((9, n)); G[0] = 2.0
    dS, _, _ = O.stress_rate(G, np.zeros((5, n)), Gam, 0)
    assert dS[0, 0] == pytest.approx(4.0 / 3.0 * 22.7e9 * 2.0) and dS[1, 0] == pytest.approx(-2.0 / 3.0 * 22.7e9 * 2.0)


def test_rotation_term_sign_documented():
    """Reading Q1.  Under a rigid rotation Q(t) about z with angular velocity w, a stress carried
    with the body is S(t) = Q S Q^T.  Its time derivative is W S - S W (W = spin = R of Eq. 15).
    The default is that objective rate (the paper: "we adopt the Jaumann rate to obtain an objective
    stress rate"); Eq. 13 with the index order AS PRINTED gives S.R + (S.R)^T = S R - R S,
    the opposite sign, kept behind JAUMANN_AS_PRINTED.  Both are tested so a silent change fails."""
    w = 0.3
    S5 = np.array([1.0, -0.4, 0.25, 0.6, -0.8])
    S3 = O._S3(S5[:, None])[0]
    Wm = np.array([[0.0, -w, 0.0], [w, 0.0, 0.0], [0.0, 0.0, 0.0]])          # v = w e_z x r
    dt = 1e-6
    def Q(t):
        c, s = math.cos(w * t), math.sin(w * t)
        return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])
    fd = (Q(dt) @ S3 @ Q(dt).T - Q(-dt) @ S3 @ Q(-dt).T) / (2 * dt)
    G = Wm.reshape(9, 1)
    _, corot, _ = O.stress_rate(G, S5[:, None], np.zeros(1), 0)
    _, printed, _ = O.stress_rate(G, S5[:, None], np.zeros(1), O.FLAG_JAUMANN_AS_PRINTED)
    assert np.allclose(corot[0], fd, atol=1e-8)
    assert np.allclose(printed[0], -fd, atol=1e-8)
    # the printed xx component, Eq. 25: S^{xy}(G^{yx}-G^{xy}) + S^{xz}(G^{zx}-G^{xz})
    assert printed[0][0, 0] == pytest.approx(S5[2] * (w - (-w)) + S5[3] * 0.0)
