"""Pins for the oracle's step sequence (Eq. 40-42)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W


def small_block(n_side=8, **kw):
    return W.elastic_block(n_side, **kw)


def test_constant_stress_rate_integrates_to_dt_times_rate():
    # uniform shear, S = 0, no yielding (huge Y0), no noise: dS^{xy}/dt = Gamma * 100 for every
    # particle (G = A exactly by the correction tensor), so after k steps S^{xy} = k dt Gamma 100:
    # the opening (Eq. 42) and closing (Eq. 41) half kicks must add up to one dt.
    wl = small_block(7)
    A = wl.arrays
    A["vx"][:] = (100.0 * A["y"].astype(np.float64)).astype(np.float32)
    A["vy"][:] = 0; A["vz"][:] = 0
    for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz"):
        A[k][:] = 0
    A["u"][:] = 1.0                                    # T ~ 0: no softening
    wl.params.materials[0].Y0 = 1e30
    wl.params.materials[0].Ym = 2e30
    wl.params.materials[0].c0 = 1e-3                   # no pressure forces ...
    wl.params.alpha = wl.params.beta = 0.0             # ... and no viscosity: the flow stays a pure shear
    st = O.Stepper(wl, mode="brute")
    dt = 1e-9                                           # tiny: particles barely move
    for _ in range(3):
        st.step(dt)
    Gam = wl.params.materials[0].Gamma
    assert np.allclose(st.S[2], 3 * dt * Gam * 100.0, rtol=1e-6)
    assert np.abs(st.S[[0, 1, 3, 4]]).max() < 1e-6 * 3 * dt * Gam * 100.0 + 1e-3
    assert np.allclose(st.e_acc, 3 * dt * 0.5 * 2 * 50.0 ** 2, rtol=1e-5)


def test_galilean_invariance_and_momentum():
    wl = small_block(6)
    V = np.array([250.0, -125.0, 500.0])                # fp32-exact shifts
    wl2 = small_block(6)
    for a, k in enumerate(("vx", "vy", "vz")):
        wl2.arrays[k] = (wl2.arrays[k].astype(np.float64) + V[a])
    s1 = O.Stepper(wl, mode="brute"); s2 = O.Stepper(wl2, mode="brute")
    s2.v = s1.v + V[:, None]
    dt = 2e-7
    p0 = (s1.m[None] * s1.v).sum(axis=1)
    for _ in range(2):
        s1.step(dt); s2.step(dt)
    # positions differ by exactly V t up to the neighbour-set flips that motion can cause
    assert np.allclose(s2.x - 2 * dt * V[:, None], s1.x, rtol=0, atol=1e-9)
    assert np.allclose(s2.v - V[:, None], s1.v, rtol=0, atol=1e-6 * np.abs(s1.v).max())
    assert np.allclose(s2.S, s1.S, rtol=1e-6, atol=1e-3)
    assert np.allclose(s2.u, s1.u, rtol=1e-9)
    # linear momentum conserved by the step (no external acceleration in configs[0])
    p1 = (s1.m[None] * s1.v).sum(axis=1)
    assert np.all(np.abs(p1 - p0) < 1e-12 * np.abs(s1.m[None] * s1.v).sum(axis=1))


def test_yielded_state_is_bounded_after_every_step():
    wl = small_block(6)
    st = O.Stepper(wl, mode="brute")
    for _ in range(3):
        st.step(0.0)                                    # CFL step
        assert np.all(np.sqrt(O.J2(st.S)) <= st.d["Y"] * (1 + 1e-12) + 1e-9)
    assert st.dt_next > 0 and np.isfinite(st.dt_next)


def test_fixed_particles_do_not_move_and_step_matches_single_pass():
    wl = small_block(6)
    wl.fixed[:40] = 1
    for k in ("vx", "vy", "vz"):
        wl.arrays[k][:40] = 0
    x0 = np.stack([wl.arrays[k] for k in ("x", "y", "z")]).astype(np.float64)
    st = O.Stepper(wl, mode="brute")
    st.step(3e-7)
    assert np.array_equal(st.x[:, :40], x0[:, :40]) and np.all(st.v[:, :40] == 0.0)
    assert np.abs(st.x[:, 40:] - x0[:, 40:]).max() > 0
    # single_pass == the closing half of a step started from rest derivatives:
    d = O.single_pass(wl, dt=3e-7)
    assert np.all(d["v_close"][:, :40] == 0.0)
    sj = np.sqrt(O.J2(d["S_close"]))
    assert np.all(sj <= d["Y"] * (1 + 1e-12) + 1e-9)


def test_cfl_timestep_eq39():
    wl = small_block(6)
    d = O.single_pass(wl)
    p = wl.params
    h = wl.arrays["h"].astype(np.float64)
    # mu_max = 0 particle: dt = eta_C h / ((1 + 0.6 alpha) c)
    i = int(np.argmin(d["mumax"]))
    lo = p.eta_C * h[i] / ((1 + 0.6 * p.alpha) * 3000.0 + 0.6 * p.beta * d["mumax"][i])
    assert d["dt_i"][i] == pytest.approx(lo, rel=1e-14)
    assert np.all(d["dt_i"] <= p.eta_C * h / (1.6 * 3000.0) * (1 + 1e-14))


def test_grid_mode_gives_the_same_step_as_brute():
    wl = small_block(7)
    a = O.Stepper(wl, mode="brute"); b = O.Stepper(wl, mode="grid")
    a.step(0.0); b.step(0.0)
    assert np.array_equal(a.x, b.x) and np.array_equal(a.S, b.S) and np.array_equal(a.u, b.u)
