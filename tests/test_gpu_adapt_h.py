"""GPU parity of sph_adapt_h (NEXT-1; Eq. 2) against oracle.adapt_h, and of the pass
sequence that follows it (the lists, boxes and tree must have been rebuilt for the new h)."""
import copy

import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W
from tests import parity_util as U

pytestmark = pytest.mark.gpu

TOL_H = 2e-6        # h is fp32 on both sides; the GPU's Omega is fp32: the factor differs by ~1e-7 per iteration


def _cases():
    wl = W.elastic_block(12, h_spread=0.2)
    wl.arrays["h"] = (wl.arrays["h"] * np.float32(0.85)).astype(np.float32)
    yield "block_h_too_small", wl, 60.0
    wl = W.impact_pair(20000, W.SEED_BASE + 3, 100.0, 1.0)          # generator h ~ 35 neighbours
    yield "impact_pair_variable_h", wl, 60.0


@pytest.mark.parametrize("name,wl,n_target", list(_cases()), ids=lambda v: v if isinstance(v, str) else "")
def test_adapt_h_matches_oracle_and_passes_follow(name, wl, n_target):
    import torch
    from paper_2603_19764_b200 import binding as B
    A = wl.arrays
    mode = "grid" if wl.n > 5000 else "brute"
    for iters in (1, 3):
        s = B.Sph(wl.params, wl.n)
        t = s.upload(wl)
        s.build_neighbors(t, wl.n)
        chg = torch.zeros(1, dtype=torch.float32, device="cuda")
        s.adapt_h(n_target, iters, chg)
        h_gpu = s.get_field("H").cpu().numpy()
        h_o, _, _, hist = O.adapt_h(A["x"], A["y"], A["z"], A["m"], A["h"], wl.params.kappa, n_target, iters, mode)
        assert np.abs(h_gpu / h_o - 1.0).max() <= TOL_H
        assert float(chg.item()) == pytest.approx(hist[-1], rel=1e-4, abs=1e-7)
    # the passes after the iteration, against the oracle run on the GPU's own h (bit-exact neighbour sets)
    wl2 = copy.copy(wl)
    wl2.arrays = dict(wl.arrays)
    wl2.arrays["h"] = h_gpu.astype(np.float32)
    dt = 1e-7 if name.startswith("block") else 1e-3
    s.density(); s.strength_update(B.PREDICT); s.gradients(); s.forces(); s.strength_update(B.CLOSE, dt)
    g = {}
    for nm in ("RHO", "OMEGA", "P", "CS", "T", "GAMMA", "Y", "MUMAX", "DUDT", "DT", "EPS2", "U", "CFLAG",
               "NGATHER", "NSYMMETRIC"):
        g[nm.lower()] = s.get_field(nm).cpu().numpy()
    for nm, nc in (("A", 3), ("V", 3), ("X", 3), ("SPRED", 5), ("S", 5), ("DSDT", 5), ("F", 9), ("CINV", 9), ("G", 9)):
        g[nm.lower()] = s.get_fields(nm, nc).cpu().numpy()
    d = O.single_pass(wl2, dt=dt, mode=mode)
    errs = U.compare_single_pass(g, d, wl2)
    # Eq. 2 holds after three iterations from a 15 % / 18 % error
    mtot = 4.0 / 3.0 * np.pi * (wl.params.kappa * h_gpu.astype(np.float64)) ** 3 * d["rho"]
    res = np.abs(mtot / (n_target * A["m"].astype(np.float64)) - 1.0)
    assert np.median(res) < 1e-3, np.median(res)
    print(name, "errors", {k: float(f"{v:.3g}") for k, v in errs.items()}, "median Eq.2 residual", float(np.median(res)))


def test_adapt_h_argument_checks():
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(4)
    s = B.Sph(wl.params, wl.n)
    with pytest.raises(B.SphError) as e:
        s.adapt_h(60.0, 1)
    assert e.value.code == B.EORDER
    t = s.upload(wl)
    s.build_neighbors(t, wl.n)
    with pytest.raises(B.SphError) as e:
        s.adapt_h(0.0, 1)
    assert e.value.code == B.EINVAL
    h0 = s.get_field("H").cpu().numpy()
    s.adapt_h(60.0, 0)
    assert np.array_equal(s.get_field("H").cpu().numpy(), h0) and np.array_equal(h0, wl.arrays["h"])
