"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element,
on the same seeded inputs.  Sizes span several chunks, tree levels and a ragged tail."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_19764_b200 import workloads as W
from tests import parity_util as U

pytestmark = pytest.mark.gpu

F = W.FLAG_STRENGTH | W.FLAG_CORRECTION_TENSOR


def test_config0_single_pass_all_fields():
    wl = W.config(0)
    g = U.gpu_single_pass(wl)
    d = O.single_pass(wl)
    errs = U.compare_single_pass(g, d, wl)
    U.neighbor_sets_equal(g["_sph"], wl, mode="brute")
    c = g["counters"]
    assert c["pairs_gather"] == int(d["n_gather"].sum()) and c["pairs_symmetric"] == int(d["n_symmetric"].sum())
    assert c["cfallback"] == 0
    print("config0 errors", {k: float(f"{v:.3g}") for k, v in errs.items()})


@pytest.mark.parametrize("case", ["ragged_11", "h_spread", "two_materials", "hydro_only", "no_correction",
                                  "as_printed", "pclip_global", "block_24", "eta_a", "fused", "fused_hydro"])
def test_variants(case):
    kw = dict(n_side=12)
    if case == "ragged_11":
        kw = dict(n_side=11)                                  # 1331 = 41 chunks + 19 particles
    elif case == "h_spread":
        kw = dict(n_side=12, h_spread=0.3)                    # h_i != h_j: symmetric set > gather set
    elif case == "two_materials":
        kw = dict(n_side=12, two_materials=True)
    elif case == "hydro_only":
        kw = dict(n_side=12, flags=W.FLAG_CORRECTION_TENSOR)
    elif case == "no_correction":
        kw = dict(n_side=12, flags=W.FLAG_STRENGTH)
    elif case == "as_printed":
        kw = dict(n_side=12, flags=F | W.FLAG_JAUMANN_AS_PRINTED)
    elif case == "pclip_global":
        kw = dict(n_side=12, flags=F | W.FLAG_PCLIP_GLOBAL)
    elif case == "block_24":
        kw = dict(n_side=24)                                  # 432 chunks: two tree levels
    elif case == "fused":
        kw = dict(n_side=12, h_spread=0.3, two_materials=True)            # S4 + S5 in one pass, h_i != h_j
    elif case == "fused_hydro":
        kw = dict(n_side=12, h_spread=0.3, flags=W.FLAG_CORRECTION_TENSOR)
    elif case == "eta_a":
        kw = dict(n_side=12)
    wl = W.elastic_block(**kw)
    if case == "eta_a":
        wl.params.eta_a = 8.0e-2          # Eq. 38 (reading Q22) limits some particles, Eq. 39 the others
    g = U.gpu_single_pass(wl, split=not case.startswith("fused"))
    d = O.single_pass(wl, mode="grid" if wl.n > 5000 else "brute")
    U.compare_single_pass(g, d, wl)
    if case == "eta_a":
        wl.params.eta_a = 0.0
        d0 = O.single_pass(wl)
        lim = d["dt_i"] < d0["dt_i"] * (1 - 1e-12)
        assert 0.05 < lim.mean() < 0.95, lim.mean()        # both branches of the minimum are exercised
    U.neighbor_sets_equal(g["_sph"], wl, mode="grid")


def test_three_tree_levels_and_neighbour_ids():
    wl = W.elastic_block(40, h_spread=0.2)                    # 64000 particles, 2000 chunks, 3 levels
    g = U.gpu_single_pass(wl)
    d = O.single_pass(wl, mode="grid")
    U.compare_single_pass(g, d, wl)
    U.neighbor_sets_equal(g["_sph"], wl, mode="grid")         # sorted id lists, every particle


def test_empty_and_tiny_inputs():
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(4)
    e = wl.subset(np.arange(0))
    s = B.Sph(e.params, 16)
    t = s.upload(e)
    s.build_neighbors(t, 0)
    s.density(); s.strength_update(B.PREDICT); s.gradients(); s.forces(); s.strength_update(B.CLOSE, 1e-7)
    assert s.get_counters()["pairs_gather"] == 0
    one = wl.subset(np.array([5]))
    g = U.gpu_single_pass(one)
    d = O.single_pass(one)
    assert g["ngather"].tolist() == [1.0] and g["nsymmetric"].tolist() == [0.0]
    assert np.all(g["a"] == 0.0) and np.all(np.isfinite(g["s"]))
    assert g["cflag"].tolist() == [1.0] and d["cflag"].tolist() == [1]
    assert g["rho"][0] == pytest.approx(d["rho"][0], rel=1e-6)


def test_pass_order_is_enforced():
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(4)
    s = B.Sph(wl.params, wl.n)
    with pytest.raises(B.SphError) as e:
        s.density()
    assert e.value.code == B.EORDER
    t = s.upload(wl)
    s.build_neighbors(t, wl.n)
    with pytest.raises(B.SphError):
        s.forces()
    with pytest.raises(B.SphError) as e:
        s.build_neighbors(t, wl.n + 1)
    assert e.value.code == B.ECAPACITY


def test_results_are_bitwise_repeatable():
    wl = W.elastic_block(12, h_spread=0.2)
    a = U.gpu_single_pass(wl)
    b = U.gpu_single_pass(wl)
    for k in ("rho", "a", "dudt", "dsdt", "s", "f", "cinv"):
        assert np.array_equal(a[k], b[k]), k


def test_full_step_matches_oracle():
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(12)
    s = B.Sph(wl.params, wl.n)
    t = s.upload(wl)
    dt_used = torch.zeros(1, dtype=torch.float32, device="cuda")
    st = O.Stepper(wl, mode="brute")
    for step in range(2):
        s.step(t, wl.n, 0.0, dt_used)
        dt_o = st.step(0.0)
        torch.cuda.synchronize()
        assert float(dt_used.item()) == pytest.approx(dt_o, rel=1e-5)
        x = np.stack([t[k].cpu().numpy() for k in ("x", "y", "z")])
        v = np.stack([t[k].cpu().numpy() for k in ("vx", "vy", "vz")])
        S = np.stack([t[k].cpu().numpy() for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz")])
        u = t["u"].cpu().numpy()
        assert U.maxnorm_err(x, st.x) <= 1e-6
        assert U.maxnorm_err(v, st.v) <= U.TOL_STATE
        assert U.maxnorm_err(S, st.S) <= U.TOL_STATE
        assert U.maxnorm_err(u, st.u) <= U.TOL_STATE
        eacc = s.get_field("EACC").cpu().numpy()
        assert U.maxnorm_err(eacc, st.e_acc) <= U.TOL_STATE


def test_step_host_roundtrip_equals_device_step():
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(10)
    s1 = B.Sph(wl.params, wl.n)
    t = s1.upload(wl)
    s1.step(t, wl.n, 2e-7)
    s1.step(t, wl.n, 2e-7)
    torch.cuda.synchronize()
    host = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in wl.arrays.items()}
    host["mat"] = torch.from_numpy(wl.mat.copy()).pin_memory()
    host["fixed"] = torch.from_numpy(wl.fixed.copy()).pin_memory()
    s2 = B.Sph(wl.params, wl.n)
    assert s2.step_host(host, wl.n, 2e-7) == pytest.approx(2e-7)
    s2.step_host(host, wl.n, 2e-7)
    for k in ("x", "vx", "u", "Sxy"):
        assert np.array_equal(host[k].numpy(), t[k].cpu().numpy()), k


def test_tree_walk_kernels_still_match():
    """SPH_NO_LISTS selects the round-1 v0 kernels (pair passes walk the chunk tree)."""
    wl = W.elastic_block(12, h_spread=0.25, flags=F | W.FLAG_NO_LISTS)
    g = U.gpu_single_pass(wl)
    d = O.single_pass(wl)
    U.compare_single_pass(g, d, wl)
    U.neighbor_sets_equal(g["_sph"], wl, mode="brute")


def test_variable_h_impact_pair_scaled():
    """configs[3] construction at parity size: two bodies, two materials, h varying ~5x."""
    wl = W.impact_pair(30000, W.SEED_BASE + 3, 100.0, 1.214)
    assert wl.arrays["h"].max() / wl.arrays["h"].min() > 3.0
    g = U.gpu_single_pass(wl, dt=1e-3)
    d = O.single_pass(wl, dt=1e-3, mode="grid")
    errs = U.compare_single_pass(g, d, wl)
    assert g["counters"]["list_overflow"] == 0
    U.neighbor_sets_equal(g["_sph"], wl, mode="grid")         # multi-level walk, variable h: ids, not only counts
    print("impact pair errors", {k: float(f"{v:.3g}") for k, v in errs.items()})
    gf = U.gpu_single_pass(wl, dt=1e-3, split=False)          # the fused S4 + S5 kernel on the same set
    U.compare_single_pass(gf, d, wl)


def test_fused_step_on_variable_h_two_materials_matches_oracle_stepper():
    """sph_step (fused gradient + force kernel, CUDA-graph replay on a capturable stream) for two steps on the
    configs[3] construction at parity size -- variable h, two materials -- against the oracle's stepper."""
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.impact_pair(30000, W.SEED_BASE + 3, 100.0, 1.214)
    st = O.Stepper(wl, mode="grid")
    with torch.cuda.stream(torch.cuda.Stream()):
        s = B.Sph(wl.params, wl.n)
        t = s.upload(wl)
        dtu = torch.zeros(1, dtype=torch.float32, device="cuda")
        s.step(t, wl.n, 0.0, dtu)
        dts = [float(dtu.item())]
        s.step(None, 0, 0.0, dtu)
        dts.append(float(dtu.item()))
        s.download_state(t)
        torch.cuda.synchronize()
        assert s.get_counters()["list_overflow"] == 0
    for k in range(2):
        assert dts[k] == pytest.approx(st.step(0.0), rel=2e-5)
    x = np.stack([t[k].cpu().numpy() for k in ("x", "y", "z")])
    v = np.stack([t[k].cpu().numpy() for k in ("vx", "vy", "vz")])
    S = np.stack([t[k].cpu().numpy() for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz")])
    assert U.maxnorm_err(x, st.x) <= 1e-6
    assert U.maxnorm_err(v, st.v) <= U.TOL_STATE
    assert U.maxnorm_err(t["u"].cpu().numpy(), st.u) <= U.TOL_STATE
    assert U.maxnorm_err(S, st.S) <= U.TOL_STATE


def test_coincident_particles_and_bad_material_index():
    """Two particles at the same position (r = 0, i != j): members of each other's sets, zero pair force
    (x_ij = 0), no NaN.  A material index outside 0..n_materials-1 is replaced and counted."""
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(8, h_spread=0.2)
    for k in ("x", "y", "z"):
        wl.arrays[k][17] = wl.arrays[k][200]
    g = U.gpu_single_pass(wl)
    d = O.single_pass(wl)
    U.compare_single_pass(g, d, wl)
    U.neighbor_sets_equal(g["_sph"], wl, mode="brute")
    for k in ("a", "dudt", "dsdt", "s", "rho"):
        assert np.all(np.isfinite(g[k])), k
    assert g["counters"]["bad_material"] == 0 and g["counters"]["nonfinite"] == 0
    wl.mat[5] = 7; wl.mat[6] = -1                        # one material defined
    g2 = U.gpu_single_pass(wl)
    assert g2["counters"]["bad_material"] == 2
    assert np.array_equal(g2["s"], g["s"])               # both were given material n_materials - 1 = 0


def test_granular_column_scaled_with_fixed_floor():
    """configs[1] construction at parity size: fixed floor layers, Y0 = 0, mu_d = 0.8, gravity."""
    wl = W.granular_column(0.35)
    g = U.gpu_single_pass(wl, dt=1e-4)
    d = O.single_pass(wl, dt=1e-4, mode="grid")
    U.compare_single_pass(g, d, wl)
    fx = wl.fixed.astype(bool)
    assert np.all(g["v"][:, fx] == 0.0)


def test_tiles_over_list_capacity_fall_back_to_the_tree_walk():
    """A tile whose lists do not fit is flagged (counter) and served by the tree-walk kernels:
    slower, never wrong."""
    wl = W.elastic_block(12, h_spread=0.2)
    wl.params.list_budget = 4             # 16 neighbours per lane; this block needs ~80
    g = U.gpu_single_pass(wl, allow_fallback=True)
    assert g["counters"]["list_overflow"] > 0
    d = O.single_pass(wl)
    U.compare_single_pass(g, d, wl)
    U.neighbor_sets_equal(g["_sph"], wl, mode="brute")


def test_diagnostics_match_fp64_sums_and_momentum_is_conserved():
    """S8: device reductions in fp64 against numpy sums of the same fp32 state; linear momentum of the
    internal forces is conserved over steps (no external acceleration in configs[0])."""
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(12)
    s = B.Sph(wl.params, wl.n)
    t = s.upload(wl)
    s.build_neighbors(t, wl.n)
    d0 = s.get_diagnostics().cpu().numpy()
    A = {k: v.astype(np.float64) for k, v in wl.arrays.items()}
    m = A["m"]; x = np.stack([A["x"], A["y"], A["z"]]); v = np.stack([A["vx"], A["vy"], A["vz"]])
    ref = np.concatenate([[m.sum()], (m * v).sum(axis=1), (m * np.cross(x.T, v.T).T).sum(axis=1),
                          [(m * (0.5 * (v * v).sum(axis=0) + A["u"])).sum()]])
    assert np.allclose(d0, ref, rtol=1e-12, atol=1e-12 * np.abs(ref).max())
    assert np.array_equal(d0, s.get_diagnostics().cpu().numpy())          # fixed order: bitwise repeatable
    for _ in range(3):
        s.step(t, wl.n, 0.0)
    d1 = s.get_diagnostics().cpu().numpy()
    pscale = (m * np.abs(v)).sum()
    assert np.abs(d1[1:4] - d0[1:4]).max() <= 1e-5 * pscale                # fp32 pair sums, antisymmetric terms
    assert d1[0] == d0[0]


@pytest.mark.parametrize("kind", ["linear", "curved"])
def test_tabulated_eos_matches_oracle(kind):
    """NEXT-3: P, T, c_s from (rho, u) tables and T_melt(rho), two materials."""
    wl = W.elastic_block(12, two_materials=True, eos_table=kind)
    g = U.gpu_single_pass(wl)
    d = O.single_pass(wl)
    errs = U.compare_single_pass(g, d, wl)
    assert U.maxnorm_err(g["cs"], d["cs"]) <= 1e-6
    if kind == "curved":
        assert np.ptp(d["cs"]) > 0.0 and (d["Y"] == 0.0).any()
    print("table", kind, {k: float(f"{v:.3g}") for k, v in errs.items()})


def test_eos_table_argument_checks_and_reset():
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(6, eos_table="curved")
    ref = U.gpu_single_pass(W.elastic_block(6))
    s = B.Sph(wl.params, wl.n)
    with pytest.raises(B.SphError) as e:
        s.set_eos_table(3, wl.params.materials[0].table)
    assert e.value.code == B.EINVAL
    s.set_eos_table(0, None)                       # back to the analytic EOS
    t = s.upload(wl)
    s.build_neighbors(t, wl.n); s.density(); s.strength_update(B.PREDICT)
    assert np.array_equal(s.get_field("P").cpu().numpy(), ref["p"])


def test_graph_replay_equals_kernel_by_kernel_step():
    """The resident step replayed from its CUDA graph (a capturable stream) against the same steps
    launched kernel by kernel: bitwise equal state, timings and launch counts still reported."""
    import torch
    from paper_2603_19764_b200 import binding as B
    out = []
    for no_graph in (False, True):
        wl = W.elastic_block(12, h_spread=0.2, flags=F | (W.FLAG_NO_GRAPH if no_graph else 0))
        with torch.cuda.stream(torch.cuda.Stream()):          # torch ops and the library on one capturable stream
            s = B.Sph(wl.params, wl.n)
            t = s.upload(wl)
            s.build_neighbors(t, wl.n)
            dtu = torch.zeros(1, dtype=torch.float32, device="cuda")
            for _ in range(6):                    # bootstrap, two captures, three replays
                s.step(None, 0, 0.0, dtu)
            tm = s.get_timings()
            assert tm["step"] > 0.0 and tm["force"] > 0.0 and tm["build"] > 0.0
            s.download_state(t)
            torch.cuda.synchronize()
            out.append(({k: t[k].cpu().numpy().copy() for k in ("x", "vx", "u", "Sxy")}, float(dtu.item()),
                        s.launch_count(), s.get_field("RHO").cpu().numpy()))
    for k in out[0][0]:
        assert np.array_equal(out[0][0][k], out[1][0][k]), k
    assert out[0][1] == out[1][1] and out[0][2] == out[1][2]
    assert np.array_equal(out[0][3], out[1][3])


# ---- list reuse (sph_params.skin > 0): same neighbour sets, same numbers --------------------------------------
def test_skin_lists_give_the_same_single_pass():
    """With skin > 0 the lists hold the pairs within (1 + skin) of the cut-off and the pair passes evaluate the
    exact predicate themselves: a pair of the skin contributes exactly zero, so the neighbour sets and counts are
    those of the exact lists, and the fields differ only by the order of summation (reused lists are ordered by
    shared-memory bank class)."""
    out = []
    for skin in (0.0, 0.12):
        wl = W.elastic_block(12, h_spread=0.3, two_materials=True)
        wl.params.skin = skin
        g = U.gpu_single_pass(wl, split=False)
        out.append(g)
        U.compare_single_pass(g, O.single_pass(wl), wl)
        U.neighbor_sets_equal(g["_sph"], wl, mode="brute")
    assert out[1]["counters"]["candidates"] > out[0]["counters"]["candidates"]
    for k in ("ngather", "nsymmetric", "cflag"):
        assert np.array_equal(out[0][k], out[1][k]), k
    for k in ("rho", "a", "dudt", "dsdt", "s", "f", "cinv"):
        assert U.maxnorm_err(out[1][k], out[0][k]) <= 2e-6, k


# measured (B200, round 3): S_max 3.0e-6 (block), 5.8e-6 (impact); v 2.9e-6 / 1.7e-7; S_rms 8e-8 / 3e-8
REUSE_S_MAX_TOL = {"block": 6e-5, "impact": 6e-5}


@pytest.mark.parametrize("case", ["block", "impact"])
def test_reused_lists_keep_the_exact_neighbour_sets_over_steps(case):
    """sph_step with list reuse (full build every 5 steps, skin 5 %): after every step the neighbour sets the
    passes used are the exact sets of the CURRENT positions (oracle on the downloaded positions), dirty tiles
    included (the impact pair has a contact surface moving at 3 km/s), and the state follows the oracle's
    stepper like the step without reuse does: the stepper keeps its state in fp32 as the GPU does
    (Stepper(store_fp32=True), all arithmetic fp64) and takes the GPU's time steps, each checked against its own
    CFL step first -- x, v, u, S parity of these steps is conditional on that 1e-4 agreement of dt."""
    import torch
    from paper_2603_19764_b200 import binding as B
    if case == "block":
        wl = W.elastic_block(14, h_spread=0.2)
        for q in ("vx", "vy", "vz"):                          # a violent velocity field: lists go stale quickly
            wl.arrays[q] *= 30.0
    else:
        wl = W.impact_pair(20000, W.SEED_BASE + 3, 100.0, 1.214)
    wl.params.skin = 0.05
    wl.params.rebuild_every = 5
    st = O.Stepper(wl, mode="grid", store_fp32=True)
    st.bootstrap()
    dirty_seen = 0
    with torch.cuda.stream(torch.cuda.Stream()):
        s = B.Sph(wl.params, wl.n)
        t = s.upload(wl)
        dtu = torch.zeros(1, dtype=torch.float32, device="cuda")
        s.build_neighbors(t, wl.n)
        for step in range(12):
            s.step(None, 0, 0.0, dtu)
            assert float(dtu.item()) == pytest.approx(st.dt_next, rel=1e-4)     # the oracle's own CFL step
            st.step(float(dtu.item()))                                          # ... then the GPU's fp32 value of it
            c = s.get_counters()
            dirty_seen = max(dirty_seen, c["tiles_dirty"])
            assert c["list_overflow"] == 0 and c["nonfinite"] == 0
            if step in (2, 3, 4, 8, 11):
                s.download_state(t)
                cur = W.Workload(wl.name, wl.params, {k: t[k].cpu().numpy() for k in W.FIELDS}, wl.mat, wl.fixed, 0.0)
                U.neighbor_sets_equal(s, cur, mode="grid")
        s.download_state(t)
        torch.cuda.synchronize()
    x = np.stack([t[k].cpu().numpy() for k in ("x", "y", "z")])
    v = np.stack([t[k].cpu().numpy() for k in ("vx", "vy", "vz")])
    S = np.stack([t[k].cpu().numpy() for k in ("Sxx", "Syy", "Sxy", "Sxz", "Syz")])
    errs = U.state_errors(x, v, t["u"].cpu().numpy(), S, st)
    print(case, "dirty tiles seen", dirty_seen, {k: float(f"{e:.3g}") for k, e in errs.items()})
    # 12 steps against like storage (the fp64-state stepper needed v 1e-3, S 1e-2 here)
    assert errs["x"] <= 1e-6 and errs["v"] <= 3e-5 and errs["u"] <= 3e-5
    assert errs["S_rms"] <= 1e-6 and errs["S_p999"] <= 1e-5 and errs["S_max"] <= REUSE_S_MAX_TOL[case]
    if case == "impact":
        assert dirty_seen > 0


def test_device_step_after_a_host_buffer_step_does_not_reuse_its_lists():
    """sph_step_host builds exact lists (no skin: its positions come from the caller every step).  A resident step
    right after it must start from a full build instead of reusing them."""
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(12, h_spread=0.2)
    for q in ("vx", "vy", "vz"):
        wl.arrays[q] *= 30.0
    wl.params.skin = 0.05
    wl.params.rebuild_every = 8
    host = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in wl.arrays.items()}
    host["mat"] = torch.from_numpy(wl.mat.copy()).pin_memory()
    host["fixed"] = torch.from_numpy(wl.fixed.copy()).pin_memory()
    with torch.cuda.stream(torch.cuda.Stream()):
        s = B.Sph(wl.params, wl.n)
        s.step_host(host, wl.n, 0.0)
        s.step_host(host, wl.n, 0.0)
        t = {k: v.cuda() for k, v in host.items()}
        for _ in range(3):
            s.step(None, 0, 0.0)
        s.download_state(t)
        cur = W.Workload(wl.name, wl.params, {k: t[k].cpu().numpy() for k in W.FIELDS}, wl.mat, wl.fixed, 0.0)
        U.neighbor_sets_equal(s, cur, mode="grid")


def test_host_buffer_loop_reuses_lists_and_notices_moved_particles():
    """sph_step_host in a loop that hands back what it received: the lists are reused exactly as in the resident
    loop (bitwise the same state after 7 steps).  When the caller moves particles between two calls the library
    must notice (x, y, z, h are compared with the resident values) and start from a full build: the neighbour sets of
    the next step are the oracle's at the moved positions."""
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(12, h_spread=0.2)
    wl.params.skin = 0.06
    wl.params.rebuild_every = 4
    # an external acceleration that matters: on the steps that reuse the lists it reaches the device while the pair pass
    # runs and is added by CLOSE instead (one rounding either way: the states must still agree bit for bit)
    wl.arrays["gy"] = (-2.0e6 * (1.0 + 5.0 * wl.arrays["x"])).astype(np.float32)
    wl.arrays["gx"] = (1.0e6 * np.sin(40.0 * wl.arrays["z"])).astype(np.float32)

    def pinned():
        h = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in wl.arrays.items()}
        h["mat"] = torch.from_numpy(wl.mat.copy()).pin_memory()
        h["fixed"] = torch.from_numpy(wl.fixed.copy()).pin_memory()
        return h
    with torch.cuda.stream(torch.cuda.Stream()):
        s1 = B.Sph(wl.params, wl.n)
        t = s1.upload(wl)
        s1.build_neighbors(t, wl.n)
        for _ in range(7):
            s1.step(None, 0, 0.0)
        s1.download_state(t)
        host = pinned()
        s2 = B.Sph(wl.params, wl.n)
        for _ in range(7):
            s2.step_host(host, wl.n, 0.0)
        torch.cuda.synchronize()
        for k in ("x", "y", "vx", "u", "Sxy", "Syz"):
            assert np.array_equal(host[k].numpy(), t[k].cpu().numpy()), k
        # the caller moves a block of particles by a third of a spacing and hands the state back
        host["x"][:200] += 0.003
        s2.step_host(host, wl.n, 0.0)
        cur = W.Workload(wl.name, wl.params, {k: host[k].numpy().copy() for k in W.FIELDS}, wl.mat, wl.fixed, 0.0)
        U.neighbor_sets_equal(s2, cur, mode="grid")
        assert all(np.isfinite(host[k].numpy()).all() for k in ("x", "vx", "u", "Sxx"))


def test_host_buffer_loop_keeps_the_adapted_smoothing_lengths():
    """sph_params.adapt_h_every > 0 through sph_step_host: the h that a step adapted goes back to the
    caller with the rest of the state, so the next call finds its h equal to the resident one -- the adaptation lasts,
    and the host loop is bit for bit the resident loop (same full builds, same reuse steps)."""
    import dataclasses
    import torch
    from paper_2603_19764_b200 import binding as B
    wl = W.elastic_block(12, h_spread=0.2)
    wl.params = dataclasses.replace(wl.params, skin=0.06, rebuild_every=4, adapt_h_every=3, adapt_h_target=60.0)
    h0 = wl.arrays["h"].copy()
    with torch.cuda.stream(torch.cuda.Stream()):
        s1 = B.Sph(wl.params, wl.n)
        t = s1.upload(wl)
        s1.build_neighbors(t, wl.n)
        for _ in range(7):
            s1.step(None, 0, 0.0)
        s1.download_state(t)
        h1 = s1.get_field("H").cpu().numpy()
        host = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in wl.arrays.items()}
        host["mat"] = torch.from_numpy(wl.mat.copy()).pin_memory()
        host["fixed"] = torch.from_numpy(wl.fixed.copy()).pin_memory()
        s2 = B.Sph(wl.params, wl.n)
        for _ in range(7):
            s2.step_host(host, wl.n, 0.0)
        torch.cuda.synchronize()
        assert np.abs(h1 / h0 - 1.0).max() > 1e-3                       # two adaptation steps did change h
        assert np.array_equal(host["h"].numpy(), h1)                    # ... and the caller has the adapted values
        assert np.array_equal(s2.get_field("H").cpu().numpy(), h1)
        for k in ("x", "y", "vx", "u", "Sxy", "Syz"):
            assert np.array_equal(host[k].numpy(), t[k].cpu().numpy()), k
