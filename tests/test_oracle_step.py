"""Pins for the oracle's step sequence (Eq. 40-42)."""
import os

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


def _golden_rows(golden_dir, name):
    rows = []
    for l in open(os.path.join(golden_dir, name)):
        if l.strip() and not l.startswith("#"):
            f = l.split()
            rows.append((f[0], [float(q) for q in f[1:]]))
    return rows


def test_timestep_eq38_eq39_hand_evaluated(golden_dir):
    """Eq. 38-39 against hand-evaluated numbers (tests/golden/timestep.txt): the CFL
    branch, the acceleration branch with epsilon = h_i (reading Q22), both orders of the minimum, and
    |a| = 0."""
    p = W.Params(eta_C=0.3, eta_a=0.25, alpha=1.0, beta=2.0)
    rows = _golden_rows(golden_dir, "timestep.txt")
    assert [r[0] for r in rows] == ["A", "B", "C", "D", "E"]
    v = np.array([r[1] for r in rows])
    h, c, mu, a, want = v[:, 0], v[:, 1], v[:, 2], v[:, 3:6].T.copy(), v[:, 6]
    got = O.timestep(p, h, c, mu, a)
    assert np.allclose(got, want, rtol=1e-14, atol=0)
    # eta_a <= 0 disables Eq. 38: rows B and E fall back to their CFL values 1.35/0.8 and 12/11
    p0 = W.Params(eta_C=0.3, eta_a=0.0, alpha=1.0, beta=2.0)
    got0 = O.timestep(p0, h, c, mu, a)
    assert got0[1] == pytest.approx(1.6875, rel=1e-14) and got0[4] == pytest.approx(12.0 / 11.0, rel=1e-14)
    assert np.array_equal(got0[[0, 2, 3]], got[[0, 2, 3]])


def test_derivatives_apply_eq38_to_the_full_acceleration():
    """derivatives() must hand the acceleration INCLUDING a_ext to Eq. 38: a block at rest in a strong
    uniform external field has dt_i = eta_a sqrt(h/|g|) wherever the internal forces are negligible
    (PAPER.md:227, 234), and the same call with eta_a = 0 gives the CFL value instead."""
    wl = small_block(5)
    A = wl.arrays
    for k in ("vx", "vy", "vz", "Sxx", "Syy", "Sxy", "Sxz", "Syz"):
        A[k][:] = 0
    A["gy"][:] = -4.0e12                                       # |g| >> any internal acceleration here
    wl.params.eta_a = 0.25
    S = np.zeros((5, wl.n)); g = np.stack([A["gx"], A["gy"], A["gz"]]).astype(np.float64)
    d = O.derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"], A["u"], S,
                      wl.mat, g)
    h = A["h"].astype(np.float64)
    an = np.sqrt((d["a"] ** 2).sum(axis=0))
    assert np.allclose(an, 4.0e12, rtol=1e-2)
    assert np.allclose(d["dt_i"], 0.25 * np.sqrt(h / an), rtol=1e-14)
    assert np.allclose(d["dt_i"], 0.25 * np.sqrt(0.013 / 4.0e12), rtol=1e-2)      # h = 1.3 cm
    wl.params.eta_a = 0.0
    d0 = O.derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"], A["u"], S,
                       wl.mat, g)
    assert np.all(d0["dt_i"] > 50.0 * d["dt_i"])
    assert np.allclose(d0["dt_i"], 0.3 * h / (1.6 * 3000.0 + 1.2 * d0["mumax"]), rtol=1e-14)


def test_forces_see_the_rescaled_predicted_stress():
    """"The predicted deviatoric stress tensor is then rescaled according to Equation (31),
    after which the updated time derivatives are computed from the predicted values."  Far above yield the
    projected tensor Y S/sqrt(J2) does not depend on the magnitude of the input S (Y depends on P and T
    only), so a, du/dt and dS/dt must be the same for S and 1000 S; had the force or the stress-rate pass
    been fed the un-rescaled tensor they would differ by orders of magnitude."""
    wl = small_block(5)
    A = {k: v.astype(np.float64) for k, v in wl.arrays.items()}
    A["u"][:] = 1000.0 * 400.0                                  # T = 400 K: Y > 0 everywhere
    S1 = 3.0e4 * np.stack([A["Sxx"], A["Syy"], A["Sxy"], A["Sxz"], A["Syz"]])     # |S| ~ 1e11 >> Y <= Ym = 3.5e9
    out = []
    for lam in (1.0, 1000.0):
        out.append(O.derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"], A["u"],
                                 lam * S1, wl.mat, None))
    d1, d2 = out
    assert np.all(d1["f_pred"] < 0.9) and np.all(d2["f_pred"] < 0.9e-3)         # every particle is far above yield
    assert np.allclose(np.sqrt(O.J2(d1["S_pred"])), d1["Y"], rtol=1e-12)
    for k in ("a", "dudt", "dS", "S_pred"):
        assert np.allclose(d1[k], d2[k], rtol=1e-9, atol=1e-9 * np.abs(d1[k]).max()), k
    # and S does enter the forces: with the stress switched off the acceleration is different
    wl.params.flags &= ~O.FLAG_STRENGTH
    d3 = O.derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"], A["u"],
                       S1, wl.mat, None)
    wl.params.flags |= O.FLAG_STRENGTH
    assert np.abs(d3["a"] - d1["a"]).max() > 1e-3 * np.abs(d1["a"]).max()


def test_stepper_fp32_storage_mode_rounds_state_once_per_store():
    """Stepper(store_fp32=True): every stored quantity is an fp32 value, the arithmetic is unchanged --
    the trajectories of the two modes agree to fp32 rounding, and x of the fp32 mode is exactly what
    rounding x + dt v_half of its own (stored) operands gives."""
    wl = small_block(6)
    a = O.Stepper(wl, mode="brute"); b = O.Stepper(wl, mode="brute", store_fp32=True)
    dt = 3e-7
    for _ in range(2):
        a.step(dt); b.step(dt)
    for q in ("x", "v", "u", "S", "e_acc"):
        vb = getattr(b, q)
        assert np.array_equal(vb, vb.astype(np.float32).astype(np.float64)), q
        va = getattr(a, q)
        # S feels fp32 positions through rho -> P -> Y (an ulp of x moves rho by ~3e-7 here, P = c0^2 (rho - rho0)
        # by ~5e3 Pa and the yield-limited S with it): the reason the multi-step GPU comparison uses this mode
        assert np.abs(va - vb).max() <= (1e-4 if q == "S" else 1e-6) * np.abs(va).max(), q
    assert not np.array_equal(a.x, b.x)
    for q in ("a", "dudt", "dS"):
        assert np.array_equal(b.d[q], b.d[q].astype(np.float32).astype(np.float64)), q


def test_grid_mode_gives_the_same_step_as_brute():
    wl = small_block(7)
    a = O.Stepper(wl, mode="brute"); b = O.Stepper(wl, mode="grid")
    a.step(0.0); b.step(0.0)
    assert np.array_equal(a.x, b.x) and np.array_equal(a.S, b.S) and np.array_equal(a.u, b.u)


def test_single_pass_closing_half_kick_is_pinned_by_closed_forms():
    """Pin of oracle.single_pass()'s closing half kick (Eq. 41: v, u, S advance by HALF a step with the
    new derivatives, then S is rescaled again), by values that do not come from single_pass's own formula:

    (1) pure shear v = (g y, 0, 0) of an unstressed block, constant shear modulus: the corrected gradient is exact for a
        linear field, so G_xy = g, eps_xy = g/2 and, with S = 0, dS_xy/dt = 2 Gamma eps_xy = Gamma g
        with every other component 0 (Eq. 13).  Below yield the closed S_xy is therefore Gamma g dt / 2 -- a full-step
        kick would give twice that;
    (2) the same with a step so long that Gamma g dt / 2 is beyond the yield strength: the second rescale
         puts the state ON the yield surface, sqrt(J2) = |S_xy| = Y, direction kept;
    (3) a uniform external acceleration on an isolated particle (no neighbour within reach: a = a_ext exactly, du/dt = 0):
        g_y = -10, dt = 0.2 gives v_y - 1, not - 2; a fixed particle keeps its velocity;
    (4) the special value dt = 2, where half a step is exactly one unit: u_close - u = du/dt and v_close - v = a,
        bit for bit (a full-step kick would double them), and dt = 0 returns the input state."""
    gdot, Gam = 100.0, 22.7e9
    wl = W.elastic_block(9)
    A = wl.arrays
    assert wl.params.materials[0].Gamma == Gam
    A["vx"] = (gdot * A["y"].astype(np.float64)).astype(np.float32)
    A["vy"][:] = 0.0; A["vz"][:] = 0.0
    for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz"):
        A[k][:] = 0.0
    A["u"][:] = 300.0 * wl.params.materials[0].cv          # cold: no thermal softening to speak of (Eq. 37)
    # the velocity field the oracle sees is the fp32 array: linear up to its rounding (1e-7 relative)
    dt1 = 1.0e-7                                   # Gamma g dt / 2 = 1.135e5 Pa, far below Y0 = 1e7 Pa
    d = O.single_pass(wl, dt=dt1)
    Y = d["Y"]
    assert Y.min() > 1.0e6
    want = 0.5 * Gam * gdot * dt1
    S = d["S_close"]
    assert np.allclose(S[2], want, rtol=2e-6, atol=0.0)                     # (1): half a step
    assert np.abs(S[[0, 1, 3, 4]]).max() <= 2e-6 * want
    assert np.all(d["f_close"] == 1.0)
    dt2 = 4.0e-5                                   # Gamma g dt / 2 = 4.54e7 Pa: beyond Y for many particles
    d2 = O.single_pass(wl, dt=dt2)
    S2, Y2 = d2["S_close"], d2["Y"]
    over = 0.5 * Gam * gdot * dt2 > Y2
    assert over.sum() > 50 and (~over).sum() > 0                            # both branches of the rescale are taken
    assert np.allclose(np.abs(S2[2][over]), Y2[over], rtol=1e-9)            # (2): on the yield surface
    assert np.allclose(np.sqrt(O.J2(S2))[over], Y2[over], rtol=1e-12)
    assert np.all(S2[2][over] > 0.0)
    assert np.allclose(S2[2][~over], 0.5 * Gam * gdot * dt2, rtol=2e-6)     # below yield: untouched by the rescale
    assert np.all((d2["f_close"] < 1.0) == over)

    # (3) isolated particles under a uniform external acceleration
    far = W.elastic_block(2)
    far.arrays["x"] = (np.arange(far.n) * 1.0).astype(np.float32)           # one metre apart, h = 1.3 cm
    far.arrays["y"][:] = 0.0; far.arrays["z"][:] = 0.0
    far.arrays["gy"] = np.full(far.n, -10.0, np.float32)
    far.arrays["vx"][:] = 3.0; far.arrays["vy"][:] = 0.5; far.arrays["vz"][:] = 0.0
    far.fixed[0] = 1
    df = O.single_pass(far, dt=0.2)
    assert np.array_equal(df["a"], np.stack([np.zeros(far.n), np.full(far.n, -10.0), np.zeros(far.n)]))
    assert np.all(df["dudt"] == 0.0)
    assert np.array_equal(df["v_close"][:, 1:], np.stack([np.full(far.n - 1, 3.0), np.full(far.n - 1, -0.5),
                                                          np.zeros(far.n - 1)]))
    assert np.array_equal(df["v_close"][:, 0], [3.0, 0.5, 0.0])             # fixed: no kick
    assert np.array_equal(df["u_close"], far.arrays["u"].astype(np.float64))

    # (4) dt = 2 and dt = 0 on the generic block (random S, thermal spread, shear + noise)
    gen = W.elastic_block(8)
    g0 = O.single_pass(gen, dt=0.0)
    gA = {k: v.astype(np.float64) for k, v in gen.arrays.items()}
    v_in = np.stack([gA["vx"], gA["vy"], gA["vz"]])
    assert np.array_equal(g0["v_close"], v_in) and np.array_equal(g0["u_close"], gA["u"])
    g2 = O.single_pass(gen, dt=2.0)
    assert np.abs(g2["dudt"]).min() > 0.0
    assert np.allclose(g2["u_close"] - gA["u"], g2["dudt"], rtol=1e-9, atol=0.0)
    assert np.allclose(g2["v_close"] - v_in, g2["a"], rtol=1e-9, atol=1e-9 * np.abs(g2["a"]).max())
    assert not np.allclose(g2["u_close"] - gA["u"], 2.0 * g2["dudt"], rtol=0.2)
