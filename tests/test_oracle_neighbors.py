"""Pins for pass O1 (neighbour sets): hand cases, strictness at r = H, symmetry of the
symmetric relation, and cell-list == brute force on tiny inputs."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W


def _sets(x, y, z, h, kappa, which, mode="brute"):
    c, o, l = O.neighbors(x, y, z, h, kappa, which, mode)
    return [set(l[o[i]:o[i + 1]].tolist()) for i in range(len(c))], c


def test_hand_case_three_on_a_line():
    # H = 2h: particle 0 (h=1, H=2) at 0; particle 1 (h=0.25, H=0.5) at 1.5; particle 2 (h=1) at 4.5
    x = np.array([0.0, 1.5, 4.5]); y = np.zeros(3); z = np.zeros(3)
    h = np.array([1.0, 0.25, 1.0])
    g, cg = _sets(x, y, z, h, 2.0, O.GATHER)
    s, cs = _sets(x, y, z, h, 2.0, O.SYMMETRIC)
    assert g == [{0, 1}, {1}, {2}]          # gather uses H_i only and contains i
    assert s == [{1}, {0}, set()]           # symmetric uses max(H_i, H_j) and excludes i
    assert cg.tolist() == [2, 1, 1] and cs.tolist() == [1, 1, 0]


def test_strict_inequality_at_the_edge():
    # fp32-exact numbers: H = 2 * 0.5 = 1; r = 1 exactly -> r2 = 1 is NOT < H^2 = 1
    x = np.array([0.0, 1.0, np.nextafter(np.float32(1.0), np.float32(0.0))], dtype=np.float64)
    y = np.zeros(3); z = np.zeros(3); h = np.full(3, 0.5)
    g, _ = _sets(x, y, z, h, 2.0, O.GATHER)
    assert 1 not in g[0] and 2 in g[0]


def test_predicate_is_fp32():
    # two points whose fp64 distance is below H but whose fp32-rounded r2 is not (and vice versa)
    # are classified by the fp32 value: build r just inside H in fp64 that rounds to H in fp32.
    H = np.float32(1.0)
    r64 = 1.0 - 1e-9                       # < 1 in fp64, == 1.0f after the cast to fp32
    x = np.array([0.0, r64]); y = np.zeros(2); z = np.zeros(2); h = np.full(2, 0.5)
    g, _ = _sets(x, y, z, h, 2.0, O.GATHER)
    assert g[0] == {0}


@pytest.mark.parametrize("seed", [1, 2])
def test_symmetric_relation_and_grid_equals_brute(seed):
    rng = np.random.default_rng(seed)
    n = 3000
    x, y, z = (rng.random(n).astype(np.float32).astype(np.float64) for _ in range(3))
    h = (0.03 + 0.05 * rng.random(n)).astype(np.float32).astype(np.float64)
    for which in (O.GATHER, O.SYMMETRIC):
        cb, ob, lb = O.neighbors(x, y, z, h, 2.0, which, "brute")
        cg, og, lg = O.neighbors(x, y, z, h, 2.0, which, "grid")
        assert np.array_equal(cb, cg) and np.array_equal(ob, og) and np.array_equal(lb, lg)
    s, _ = _sets(x, y, z, h, 2.0, O.SYMMETRIC)
    g, _ = _sets(x, y, z, h, 2.0, O.GATHER)
    for i in range(0, n, 7):
        assert i in g[i] and i not in s[i]
        assert (g[i] - {i}) <= s[i]
        for j in s[i]:
            assert i in s[j]


def test_grid_equals_brute_on_config0():
    wl = W.config(0)
    A = wl.arrays
    for which in (O.GATHER, O.SYMMETRIC):
        b = O.neighbors(A["x"], A["y"], A["z"], A["h"], 2.0, which, "brute")
        g = O.neighbors(A["x"], A["y"], A["z"], A["h"], 2.0, which, "grid")
        for u, v in zip(b, g):
            assert np.array_equal(u, v)
    # lattice interior with kappa = 2, h = 1.3 dx: 80 neighbours + self
    assert b[0].max() == 80


def test_empty_and_single():
    e = np.zeros(0)
    c, o, l = O.neighbors(e, e, e, e, 2.0, O.GATHER, "grid")
    assert c.size == 0 and o.tolist() == [0]
    one = np.array([0.5])
    c, o, l = O.neighbors(one, one, one, np.array([0.1]), 2.0, O.GATHER, "grid")
    assert c.tolist() == [1] and l[:1].tolist() == [0]
    c, o, l = O.neighbors(one, one, one, np.array([0.1]), 2.0, O.SYMMETRIC, "brute")
    assert c.tolist() == [0]


def test_dependency_closed_sample_reproduces_the_full_run():
    """The sampling used by the full-size GPU comparisons (tests/parity_util.py): the oracle on the
    dependency-closed sample gives, for the sampled particles, what the oracle on the whole set gives."""
    from tests import parity_util as U
    wl = W.impact_pair(30000, W.SEED_BASE + 3, 100.0, 1.214)
    full = O.single_pass(wl, dt=1e-3, mode="grid")
    for centre in ((0.0, 0.0, 0.0), (5.0e4 / np.sqrt(2.0), 5.0e4 / np.sqrt(2.0), 0.0)):
        idx, pos, V = U.dependency_closed_sample(wl, centre, 1500)
        assert idx.size < wl.n
        part = U.restrict(O.single_pass(wl.subset(idx), dt=1e-3, mode="grid"), pos)
        ref = U.restrict(full, V)
        assert np.array_equal(part["n_gather"], ref["n_gather"])
        assert np.array_equal(part["n_symmetric"], ref["n_symmetric"])
        for k in ("rho", "a", "dudt", "dS", "S_close", "G"):
            assert np.allclose(part[k], ref[k], rtol=1e-12, atol=0.0), k
