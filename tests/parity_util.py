"""GPU-vs-oracle comparison helpers (tests only).  Tolerances are BASELINE.json north_star's:
neighbour sets identical; rho 1e-5 relative; a, du/dt, dS/dt max|gpu - oracle| <= 1e-4 max|oracle|
per field; yielded state (S, v, u after the closing kick) 1e-4 relative in the same max norm."""
import numpy as np

TOL_RHO = 1e-5
TOL_RATE = 1e-4
TOL_STATE = 1e-4


def maxnorm_err(gpu, ref):
    ref = np.asarray(ref, dtype=np.float64)
    gpu = np.asarray(gpu, dtype=np.float64)
    scale = np.abs(ref).max()
    if scale == 0.0:
        return np.abs(gpu).max()
    return np.abs(gpu - ref).max() / scale


def rows(counts, offsets, lst):
    counts = np.asarray(counts); offsets = np.asarray(offsets); lst = np.asarray(lst)
    return [np.sort(lst[offsets[i]:offsets[i + 1]]) for i in range(counts.shape[0])]


def sorted_rows_key(counts, lst, n_ids):
    """One int64 per list entry, row-major with every row sorted: row * n_ids + id, sorted.  Two CSR lists with
    equal counts hold the same SETS row by row iff these arrays are equal (vectorised: usable at 1e6 rows)."""
    counts = np.asarray(counts, dtype=np.int64)
    row = np.repeat(np.arange(counts.shape[0], dtype=np.int64), counts)
    key = row * np.int64(n_ids) + np.asarray(lst, dtype=np.int64)[: row.shape[0]]
    return np.sort(key)


def neighbor_sets_equal(s, wl, mode="grid", select=None, oracle_sample=None):
    """Neighbour sets of the CUDA path (sph_get_neighbors, original ids) against the oracle's, as SETS per
    particle, gather and symmetric.  select: caller-order indices of the particles to compare (full-size cases);
    oracle_sample = (idx, pos): the oracle runs on wl.subset(idx) and select == idx[pos] (dependency-closed
    sample, see dependency_closed_sample)."""
    from oracle import oracle as O
    from paper_2603_19764_b200 import binding as B
    for which_g, which_o in ((B.GATHER, O.GATHER), (B.SYMMETRIC, O.SYMMETRIC)):
        c, o, l = s.get_neighbors(which_g, select=select)
        c = c.cpu().numpy(); l = l.cpu().numpy()
        if oracle_sample is None:
            A = wl.arrays
            co, oo, lo = O.neighbors(A["x"], A["y"], A["z"], A["h"], wl.params.kappa, which_o, mode)
            if select is not None:
                sel = np.asarray(select)
                lo = np.concatenate([lo[oo[i]:oo[i + 1]] for i in sel]) if sel.size else lo[:0]
                co = co[sel]
        else:
            idx, pos = oracle_sample
            sub = wl.subset(idx).arrays
            cs, os_, ls = O.neighbors(sub["x"], sub["y"], sub["z"], sub["h"], wl.params.kappa, which_o, mode)
            co = cs[pos]
            lo = idx[np.concatenate([ls[os_[i]:os_[i + 1]] for i in pos])]       # back to ids of the whole set
        assert np.array_equal(c, co), "neighbour counts differ"
        assert np.array_equal(sorted_rows_key(c, l, wl.n), sorted_rows_key(co, lo, wl.n)), "neighbour ids differ"


def gpu_single_pass(wl, dt=None, split=True, allow_fallback=False, select=None):
    """Run the BASELINE.json configs[0] pass sequence through the C ABI; returns numpy fields
    (of the particles ``select`` -- caller-order indices -- when given: full-size cases)."""
    import torch
    from paper_2603_19764_b200 import binding as B
    s = B.Sph(wl.params, max(wl.n, 1))
    t = s.upload(wl)
    dt = wl.dt if dt is None else dt
    s.build_neighbors(t, wl.n)
    s.density()
    s.strength_update(B.PREDICT)
    strength = bool(wl.params.flags & B.STRENGTH)
    if split:
        if strength:
            s.gradients()
        s.forces()
        s.strength_update(B.CLOSE, dt)
    else:
        s.gradients_forces()                    # S4 + S5 in one pass: the kernel sph_step runs
        s.strength_update(B.CLOSE, dt)
    sel = None if select is None else torch.as_tensor(np.asarray(select), dtype=torch.long, device="cuda")
    pick = (lambda t: t) if sel is None else (lambda t: t[..., sel])
    out = {}
    for name in ("RHO", "OMEGA", "P", "CS", "T", "GAMMA", "Y", "MUMAX", "DUDT", "DT", "EPS2", "U", "CFLAG",
                 "NGATHER", "NSYMMETRIC"):
        out[name.lower()] = pick(s.get_field(name)).cpu().numpy()
    for name, nc in (("A", 3), ("V", 3), ("X", 3), ("SPRED", 5), ("S", 5), ("DSDT", 5), ("F", 9), ("CINV", 9), ("G", 9)):
        out[name.lower()] = pick(s.get_fields(name, nc)).cpu().numpy()
    out["counters"] = s.get_counters()
    assert allow_fallback or out["counters"]["list_overflow"] == 0, "tiles fell back to the tree-walk kernels"
    out["timings"] = s.get_timings()
    out["_sph"] = s
    torch.cuda.synchronize()
    return out


def compare_single_pass(g, d, wl, check_sets=None):
    """g: gpu_single_pass output, d: oracle.single_pass output.  Returns dict of errors; asserts."""
    from paper_2603_19764_b200 import binding as B
    errs = {}
    assert np.array_equal(g["ngather"].astype(np.int64), d["n_gather"].astype(np.int64)), "gather counts differ"
    assert np.array_equal(g["nsymmetric"].astype(np.int64), d["n_symmetric"].astype(np.int64)), "symmetric counts differ"
    errs["rho"] = np.abs(g["rho"] / d["rho"] - 1.0).max() if wl.n else 0.0
    assert errs["rho"] <= TOL_RHO, errs
    errs["omega"] = maxnorm_err(g["omega"], d["omega"])
    assert errs["omega"] <= 1e-5, errs
    for k, ref in (("p", d["P"]), ("y", d["Y"]), ("t", d["T"]), ("gamma", d["Gamma"])):
        errs[k] = maxnorm_err(g[k], ref)
        assert errs[k] <= TOL_RATE, errs
    errs["a"] = maxnorm_err(g["a"], d["a"])
    errs["dudt"] = maxnorm_err(g["dudt"], d["dudt"])
    errs["mumax"] = maxnorm_err(g["mumax"], d["mumax"])
    errs["dt"] = maxnorm_err(g["dt"], d["dt_i"])
    for k in ("a", "dudt", "mumax", "dt"):
        assert errs[k] <= TOL_RATE, errs
    if wl.params.flags & B.STRENGTH:
        errs["spred"] = maxnorm_err(g["spred"], d["S_pred"])
        errs["F"] = maxnorm_err(g["f"], d["F"])
        errs["Cinv"] = maxnorm_err(g["cinv"], d["Cinv"])
        errs["G"] = maxnorm_err(g["g"], d["G"])
        errs["dsdt"] = maxnorm_err(g["dsdt"], d["dS"])
        errs["eps2"] = maxnorm_err(g["eps2"], d["eps2"])
        assert np.array_equal(g["cflag"].astype(np.int64), d["cflag"].astype(np.int64)), "C fallback flags differ"
        for k in ("spred", "F", "Cinv", "G", "dsdt", "eps2"):
            assert errs[k] <= TOL_RATE, errs
    errs["S_close"] = maxnorm_err(g["s"], d["S_close"])
    errs["v_close"] = maxnorm_err(g["v"], d["v_close"])
    errs["u_close"] = maxnorm_err(g["u"], d["u_close"])
    for k in ("S_close", "v_close", "u_close"):
        assert errs[k] <= TOL_STATE, errs
    return errs


def dependency_closed_sample(wl, centre, n_valid):
    """Indices for a SAMPLED full-size comparison.  V = the n_valid particles nearest to ``centre`` in
    the max norm (a cube); N1 = every particle that can be a symmetric neighbour of a particle in V
    (distance to V's box < max(H_j, max H in V)); N2 = every particle that can be a gather neighbour
    of a particle in N1.  The oracle run on N2 alone reproduces rho, Omega, P, Y of all of N1 and hence
    every field of V exactly as the run on the whole set would.  Pure geometry: no method arithmetic.
    Returns (sample indices N2 ascending, positions of V inside the sample, V indices)."""
    A = wl.arrays
    p = np.stack([A["x"], A["y"], A["z"]]).astype(np.float64)
    H = float(wl.params.kappa) * A["h"].astype(np.float64)
    c = np.asarray(centre, dtype=np.float64)[:, None]
    d = np.abs(p - c).max(axis=0)
    V = np.sort(np.argpartition(d, n_valid)[:n_valid])

    def box_dist(idx):
        lo = p[:, idx].min(axis=1, keepdims=True); hi = p[:, idx].max(axis=1, keepdims=True)
        g = np.maximum(0.0, np.maximum(lo - p, p - hi))
        return np.sqrt((g * g).sum(axis=0))
    slack = 1.0 + 1e-6
    N1 = np.nonzero(box_dist(V) < slack * np.maximum(H, H[V].max()))[0]
    N2 = np.nonzero(box_dist(N1) < slack * H[N1].max())[0]
    pos = np.searchsorted(N2, V)
    assert np.array_equal(N2[pos], V)
    return N2, pos, V


def restrict(fields, idx):
    """Every array of a field dict whose last axis is the particle axis, restricted to idx."""
    out = {}
    for k, v in fields.items():
        out[k] = v[..., idx] if isinstance(v, np.ndarray) and v.ndim >= 1 else v
    return out


def state_errors(x, v, u, S, st):
    """Errors of a GPU state against an oracle stepper after several steps: max norm per field, and for S also the rms
    and the 99.9th percentile (both relative to max|S|) -- after many steps a handful of particles whose fp32 drift
    rounded the other way carry the maximum, the bulk statistic is the sharper check."""
    smax = np.abs(st.S).max()
    dS = np.abs(np.asarray(S, dtype=np.float64) - st.S)
    return {"x": maxnorm_err(x, st.x), "v": maxnorm_err(v, st.v), "u": maxnorm_err(u, st.u),
            "S_max": float(dS.max() / smax), "S_rms": float(np.sqrt((dS ** 2).mean()) / smax),
            "S_p999": float(np.percentile(dS, 99.9) / smax)}
