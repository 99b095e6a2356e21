"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

configs[1] and configs[2] are compared element by element over every particle (the oracle in `grid`
mode finishes them in seconds).  configs[3] and configs[4] are too large for that: the CUDA path runs
the whole set and the oracle recomputes a dependency-closed sample (parity_util.dependency_closed_sample)
around a point of interest, one in the dense core (smallest h) and one at the contact surface (largest h,
both materials); the sampled particles' fields are compared with the same tolerances."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W
from tests import parity_util as U

pytestmark = pytest.mark.gpu


def _free_gpu_bytes():
    import torch
    return torch.cuda.mem_get_info()[0]


@pytest.mark.parametrize("k,dt", [(1, 1e-4), (2, 1e-3)])
def test_full_config_every_particle(k, dt):
    wl = W.config(k)
    g = U.gpu_single_pass(wl, dt=dt)
    d = O.single_pass(wl, dt=dt, mode="grid")
    errs = U.compare_single_pass(g, d, wl)
    c = g["counters"]
    assert c["pairs_gather"] == int(d["n_gather"].sum()) and c["pairs_symmetric"] == int(d["n_symmetric"].sum())
    U.neighbor_sets_equal(g["_sph"], wl, mode="grid")          # sorted id lists of every particle
    print(f"config{k} n={wl.n}", {q: float(f"{v:.3g}") for q, v in errs.items()})


def _sampled(wl, centre, n_valid, dt):
    idx, pos, V = U.dependency_closed_sample(wl, centre, n_valid)
    # tiles over a list capacity are served by the tree-walk kernels (slower, never wrong): allowed here,
    # counted in the printed line
    g = U.gpu_single_pass(wl, dt=dt, select=V, allow_fallback=True)
    d = U.restrict(O.single_pass(wl.subset(idx), dt=dt, mode="grid"), pos)
    sub = wl.subset(V)
    errs = U.compare_single_pass(g, d, sub)
    U.neighbor_sets_equal(g["_sph"], wl, mode="grid", select=V, oracle_sample=(idx, pos))    # ids of the sampled particles
    return errs, idx.size, g["counters"]["list_overflow"]


@pytest.mark.parametrize("k,where", [(3, "core"), (3, "contact"), (4, "core"), (4, "contact")])
def test_full_config_sampled(k, where):
    need = {3: 8e9, 4: 60e9}[k]
    if _free_gpu_bytes() < need:
        pytest.skip("not enough free device memory for configs[%d]" % k)
    wl = W.config(k)
    centre = (0.0, 0.0, 0.0) if where == "core" else (5.0e4 / np.sqrt(2.0), 5.0e4 / np.sqrt(2.0), 0.0)
    errs, ns, nfb = _sampled(wl, centre, 60000, 1e-3)
    print(f"config{k} {where}: n={wl.n}, oracle sample {ns}, fallback tiles {nfb} of {(wl.n + 255) // 256}", {q: float(f"{v:.3g}") for q, v in errs.items()})


@pytest.mark.parametrize("k,steps", [(1, 4), (2, 2)])
def test_full_config_steps_in_bench_configuration(k, steps):
    """sph_step as bench.py runs it -- resident state, fused gradient + force pass, CFL time step, a capturable
    stream so that the step is captured into a CUDA graph and (configs[1]) replayed -- against the oracle's
    stepper, every particle.

    Tolerances after SEVERAL steps (BASELINE.json states its 1e-4 for one step): x, v, u keep the one-step
    tolerances.  S does not, in the max norm: the CUDA path stores positions in fp32 (BASELINE.json: "particle
    SoA storage in fp32"), the oracle carries fp64 state, and half an ulp of a position (4e-6 of a particle
    spacing at |x| / dx = 60) moves rho by ~1e-7..1e-6 relative, P = c0^2 (rho - rho0) by 1e3..1e4 Pa and the
    yield-limited S (|S| = Y ~ mu P) with it, for the particles whose drift crosses a rounding boundary.  So:
    rms and 99.9th percentile of |dS| stay within 1e-4 / 1e-3 of max |S|, the maximum within 1e-2."""
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.config(k)
    st = O.Stepper(wl, mode="grid")
    with torch.cuda.stream(torch.cuda.Stream()):
        s = B.Sph(wl.params, wl.n)
        t = s.upload(wl)
        dtu = torch.zeros(1, dtype=torch.float32, device="cuda")
        s.step(t, wl.n, 0.0, dtu)                       # ingest + bootstrap + step (kernel by kernel)
        dts = [float(dtu.item())]
        for _ in range(steps - 1):
            s.step(None, 0, 0.0, dtu)                   # captured (twice), then replayed
            dts.append(float(dtu.item()))
        s.download_state(t)
        eacc = s.get_field("EACC")
        torch.cuda.synchronize()
        got = {q: t[q].cpu().numpy() for q in ("x", "y", "z", "vx", "vy", "vz", "u", "Sxx", "Syy", "Sxy", "Sxz", "Syz")}
        eacc = eacc.cpu().numpy()
        assert s.get_counters()["list_overflow"] == 0
    for n in range(steps):
        assert dts[n] == pytest.approx(st.step(0.0), rel=2e-5)
    x = np.stack([got["x"], got["y"], got["z"]]); v = np.stack([got["vx"], got["vy"], got["vz"]])
    S = np.stack([got[q] for q in ("Sxx", "Syy", "Sxy", "Sxz", "Syz")])
    smax = np.abs(st.S).max()
    errs = {"x": U.maxnorm_err(x, st.x), "v": U.maxnorm_err(v, st.v), "u": U.maxnorm_err(got["u"], st.u),
            "S_max": U.maxnorm_err(S, st.S), "S_rms": float(np.sqrt(((S - st.S) ** 2).mean()) / smax),
            "S_p999": float(np.percentile(np.abs(S - st.S), 99.9) / smax), "eacc": U.maxnorm_err(eacc, st.e_acc)}
    print(f"config{k} n={wl.n} {steps} steps", {q: float(f"{e:.3g}") for q, e in errs.items()})
    assert errs["x"] <= 1e-6 and errs["v"] <= U.TOL_STATE and errs["u"] <= U.TOL_STATE
    assert errs["S_rms"] <= U.TOL_STATE and errs["S_p999"] <= 1e-3 and errs["S_max"] <= 1e-2
    assert errs["eacc"] <= 1e-3
