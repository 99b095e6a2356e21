"""Pins for the oracle's individual-time-step stepper (NEXT-4; reading Q23 in DESIGN.md)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W


def test_rung_assignment_and_transitions_by_hand():
    dT = 1.0
    #            dt_i:  2.0  1.0  0.6  0.5  0.3  0.25  0.1   0.01
    dt = np.array([2.0, 1.0, 0.6, 0.5, 0.3, 0.25, 0.1, 0.01])
    assert O.rung_for(dt, dT, 4).tolist() == [0, 0, 1, 1, 2, 2, 4, 4]        # 1/2^r <= dt_i, clamped to max_rung
    assert O.rung_for(np.array([0.0, np.inf]), dT, 3).tolist() == [3, 0]
    # max_rung = 2: four substeps.  A particle that ends a step after 1 substep (n_done = 1) can only stay on rung 2;
    # after 2 substeps it may drop to rung 1, not to rung 0; after 4 (the end of the big step) to rung 0.
    want = np.array([0, 0, 0, 2])
    assert O.next_rung(want, np.array([2, 2, 2, 2]), 1, 2).tolist() == [2, 2, 2, 2]
    assert O.next_rung(want, np.array([2, 2, 1, 1]), 2, 2).tolist() == [1, 1, 1, 2]
    assert O.next_rung(want, np.array([2, 1, 0, 0]), 4, 2).tolist() == [0, 0, 0, 2]
    # moving to a finer rung is always allowed
    assert O.next_rung(np.array([2]), np.array([0]), 4, 2).tolist() == [2]


def test_single_rung_is_the_global_stepper_bit_for_bit():
    wl = W.elastic_block(6)
    a = O.Stepper(wl, mode="brute"); b = O.RungStepper(wl, mode="brute")
    dt = 3e-7
    for _ in range(2):
        a.step(dt); b.big_step(dt, 0)
    for q in ("x", "v", "u", "S", "e_acc"):
        assert np.array_equal(getattr(a, q), getattr(b, q)), q
    assert np.array_equal(a.d["a"], b.d["a"]) and a.dt_next == b.dt_next
    assert np.all(b.kicks == 1) and np.all(b.rung == 0)
    # ... and with every particle forced onto rung 2 the big step is four global steps of dt / 4
    c = O.Stepper(wl, mode="brute"); e = O.RungStepper(wl, mode="brute")
    for _ in range(4):
        c.step(dt / 4)
    e.big_step(dt, 2, rungs=np.full(wl.n, 2))
    for q in ("x", "v", "u", "S"):
        assert np.allclose(getattr(c, q), getattr(e, q), rtol=1e-13, atol=1e-13 * np.abs(getattr(c, q)).max()), q
    assert np.all(e.kicks == 4)


def test_free_particles_on_different_rungs_follow_their_parabolas():
    """Two particles far apart (no neighbours), constant external acceleration: kick-drift-kick is exact for a
    constant acceleration whatever the step, so after the big step x = x0 + v0 T + g T^2 / 2 and v = v0 + g T for
    both, although Eq. 38 (eta_a sqrt(h / |g|), reading Q22) puts them on rungs 0 and 2: the second one gets four
    closing kicks, the first one."""
    wl = W.elastic_block(4).subset(np.array([0, 1]))
    A = wl.arrays
    A["x"][:] = [0.0, 100.0]; A["y"][:] = 0.0; A["z"][:] = 0.0
    A["h"][:] = [16.0, 1.0]                               # dt_a = eta_a sqrt(h / g): 4 : 1
    for q in ("vx", "vy", "vz", "Sxx", "Syy", "Sxy", "Sxz", "Syz"):
        A[q][:] = 0.0
    A["vx"][:] = [3.0, -2.0]
    A["gx"][:] = 0.0; A["gy"][:] = -4.0; A["gz"][:] = 0.0
    wl.params.eta_a = 0.5                                  # dt_a = 0.5 sqrt(16/4) = 1.0 and 0.5 sqrt(1/4) = 0.25
    wl.params.materials[0].c0 = 1.0e-3                     # the CFL limit (0.3 h / 1.6 c) is far above
    s = O.RungStepper(wl, mode="brute")
    T = 1.0
    s.big_step(T, 3)
    assert s.kicks.tolist() == [1, 4]
    assert s.trace[0]["rung"].tolist() == [0, 2]
    x0 = np.array([[0.0, 100.0], [0.0, 0.0], [0.0, 0.0]]); v0 = np.array([[3.0, -2.0], [0.0, 0.0], [0.0, 0.0]])
    g = np.array([[0.0], [-4.0], [0.0]])
    assert np.allclose(s.x, x0 + v0 * T + 0.5 * g * T * T, rtol=0, atol=1e-13)
    assert np.allclose(s.v, v0 + g * T, rtol=0, atol=1e-13)


def test_inactive_neighbours_lend_predicted_values_and_kicks_add_up():
    """Uniform shear, no yielding, no pressure forces: dS^{xy}/dt = Gamma * 100 for every particle, constant in time.
    With the particles scattered over rungs 0..2 by hand, (i) the S handed to every derivative evaluation is
    S0 + t dS/dt for EVERY particle, active or not (the prediction of the inactive ones is exact for a constant rate),
    and (ii) after the big step S = S0 + T dS/dt for every particle: each particle's opening and closing half kicks
    add up to T whatever its rung."""
    wl = W.elastic_block(6)
    A = wl.arrays
    A["vx"][:] = (100.0 * A["y"].astype(np.float64)).astype(np.float32)
    A["vy"][:] = 0; A["vz"][:] = 0
    for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz"):
        A[k][:] = 0
    A["u"][:] = 1.0
    m = wl.params.materials[0]
    m.Y0 = 1e30; m.Ym = 2e30; m.c0 = 1e-3
    wl.params.alpha = wl.params.beta = 0.0
    s = O.RungStepper(wl, mode="brute")
    rungs = (np.arange(wl.n) * 7) % 3
    T = 4e-9
    s.big_step(T, 2, rungs=rungs)
    rate = m.Gamma * 100.0
    assert s.kicks.tolist() == (1 << rungs).tolist()
    for k, tr in enumerate(s.trace):
        t = (k + 1) * T / 4
        assert np.allclose(tr["S_pred_in"][2], t * rate, rtol=1e-6), k
        assert 0 < tr["active"].sum() <= wl.n
    assert s.trace[-1]["active"].all() and not s.trace[0]["active"].all()
    assert np.allclose(s.S[2], T * rate, rtol=1e-6)
    assert np.allclose(s.e_acc, T * 0.5 * 2 * 50.0 ** 2, rtol=1e-5)


def test_rungs_follow_the_time_step_limit():
    """A body with smoothly varying h (the configs[3] construction, small): the rung of every particle is the
    coarsest one its limit allows (dT / 2^r <= dt_i < dT / 2^(r-1)), particles on coarse rungs take fewer steps,
    every particle ends a step at the end of the big step, and the yielded state stays bounded."""
    wl = W.impact_pair(3000, W.SEED_BASE + 3, 30.0, 1.214)
    rs = O.RungStepper(wl, mode="grid")
    rs.bootstrap()
    dt0 = rs.d["dt_i"].copy()
    dT = float(np.percentile(dt0, 99))
    R = 3
    rs.big_step(dT, R)
    r0 = rs.trace[0]["rung"]
    step = dT / (1 << r0)
    assert np.all((step <= dt0) | (r0 == R))
    assert np.all((2.0 * step > dt0) | (r0 == 0))
    assert len(np.unique(r0)) >= 3
    assert rs.trace[-1]["active"].all()
    assert rs.kicks.min() == 1 and rs.kicks.max() <= (1 << R)        # (a particle may also move to a coarser rung)
    assert np.corrcoef(rs.kicks, r0)[0, 1] > 0.9
    assert rs.kicks.sum() < 0.6 * wl.n * (1 << R)               # far fewer force evaluations than a global fine step
    assert np.all(np.sqrt(O.J2(rs.S)) <= rs.d["Y"] * (1 + 1e-12) + 1e-9)
    assert np.all(np.isfinite(rs.x)) and np.all(np.isfinite(rs.S))
