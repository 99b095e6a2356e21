"""Pins of the oracle's tabulated-EOS path (NEXT-3; "tabulated function", reading Q21)."""
import numpy as np

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W


def test_bilinear_function_is_reproduced_exactly():
    """a + b x + c y + d x y is bilinear in every cell: a wrong index, weight or a transposed table fails."""
    nx, ny = 7, 5
    xg = np.linspace(2.0, 5.0, nx); yg = np.linspace(-1.0, 3.0, ny)
    X, Y = np.meshgrid(xg, yg, indexing="ij")
    f = lambda x, y: 1.5 - 2.0 * x + 0.75 * y + 0.3 * x * y
    rng = np.random.default_rng(3)
    x = rng.uniform(2.0, 5.0, 200); y = rng.uniform(-1.0, 3.0, 200)
    got = O.table_lookup(f(X, Y), 2.0, 5.0, x, -1.0, 3.0, y)
    assert np.allclose(got, f(x, y), rtol=1e-13, atol=1e-13)
    g = lambda x: 4.0 - 0.5 * x
    assert np.allclose(O.table_lookup(g(xg), 2.0, 5.0, x), g(x), rtol=1e-13)


def test_nodes_and_clamping():
    tab = np.arange(12, dtype=np.float64).reshape(4, 3) ** 2
    xs = np.array([0.0, 1.0, 2.0, 3.0]); ys = np.array([10.0, 20.0, 30.0])
    for i, x in enumerate(xs):
        for j, y in enumerate(ys):
            assert O.table_lookup(tab, 0.0, 3.0, np.array([x]), 10.0, 30.0, np.array([y]))[0] == tab[i, j]
    # outside the grid: the edge value (no extrapolation)
    assert O.table_lookup(tab, 0.0, 3.0, np.array([-5.0]), 10.0, 30.0, np.array([99.0]))[0] == tab[0, 2]
    assert O.table_lookup(tab, 0.0, 3.0, np.array([7.0]), 10.0, 30.0, np.array([-1.0]))[0] == tab[3, 0]
    # a curved function: the interpolant lies between the cell's corner values
    v = O.table_lookup(tab, 0.0, 3.0, np.array([1.4]), 10.0, 30.0, np.array([14.0]))[0]
    assert tab[1, 0] < v < tab[2, 1]


def test_linear_table_reproduces_the_analytic_eos_and_the_whole_pass():
    """The analytic stand-in is linear in rho and in u: sampled on a grid and looked up bilinearly it must
    give the same P, c, T -- and so the same single pass -- up to the fp32 storage of the table."""
    wl_a = W.elastic_block(8, two_materials=True)
    wl_t = W.elastic_block(8, two_materials=True, eos_table="linear")
    a = O.single_pass(wl_a)
    t = O.single_pass(wl_t)
    scale = 2700.0 * 3000.0 ** 2
    assert np.abs(t["P"] - a["P"]).max() < 2e-7 * scale          # fp32 table values of size ~ rho0 c0^2 * 0.25
    assert np.allclose(t["T"], a["T"], rtol=1e-6) and np.allclose(t["cs"], a["cs"], rtol=1e-7)
    assert np.abs(t["a"] - a["a"]).max() < 1e-4 * np.abs(a["a"]).max()
    assert np.abs(t["S_close"] - a["S_close"]).max() < 1e-3 * np.abs(a["S_close"]).max()


def test_curved_table_changes_the_state_and_melt_curve_is_used():
    wl = W.elastic_block(6, eos_table="curved")
    d = O.single_pass(wl)
    tab = wl.params.materials[0].table
    rho = d["rho"]
    Tm = O.melt_temperature(wl.params, rho, wl.mat)
    assert np.ptp(Tm) > 0.0 and np.all(Tm >= tab.Tmelt.min()) and np.all(Tm <= tab.Tmelt.max())
    # Eq. 37 limits with the tabulated melt temperature: Y = 0 at and above T_melt(rho)
    hot = d["T"] >= Tm
    assert hot.any() and np.all(d["Y"][hot] == 0.0) and np.all(d["Y"][~hot & (d["P"] > 0)] > 0.0)
    ref = O.single_pass(W.elastic_block(6))
    assert np.abs(d["P"] - ref["P"]).max() > 1e-2 * np.abs(ref["P"]).max()
