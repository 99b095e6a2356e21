#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract: see DESIGN.md section 7).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c0|c1|c2|c3|c4] [--impl ours|reference]

A "step" is one pass of the whole hot path (sph_step: opening kick, drift, prediction, Morton
re-sort + chunk tree, density, predict/EOS/yield, fused gradient+force, close, dt reduction) over
one seeded synthetic particle set shaped like BASELINE.json's configs.  value = true neighbour pair
evaluations per second (sum_i |gather set| + sum_i |symmetric set| per step) over all ranks, inputs
resident in HBM; e2e = the same through sph_step_host (pinned host buffers, H2D + D2H inside the
timed region).  N > 1 runs N independent replicas ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Algorithmic flops per TRUE pair evaluation, hand-counted from the equations as the kernels
# evaluate them (FMA = 2, rsqrt / div / min / max / compare = 1); DESIGN.md section 6.
FLOPS_PAIR_FUSED = 147      # Eq. 18-21 + 5-8, gradient and force in one pass, with S (DESIGN.md section 5 has the breakdown)
FLOPS_PAIR_HYDRO = 78       # force pass with S == 0 (no gradient sums; forms m_j K_j itself)
FLOPS_PAIR_DENSITY = 44     # Eq. 1 + 3: 20 fp32 + 12 fp64 (counted as 2 each)
FP32_LANES_PER_SM = 128


def fp32_peak_tflops(n_sm: int, mhz: float) -> float:
    """SMs x 128 FP32 lanes x 2 flop (FMA) x clock: the CUDA-core peak (guide's unit counts)."""
    return n_sm * FP32_LANES_PER_SM * 2 * mhz * 1e6 / 1e12


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [c.strip() for c in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}



def rank_reduce(ms: float, units: float, device):
    """The N > 1 reduction of the contract: time = MAX over ranks, units = SUM over ranks (each rank
    steps its own replica; there is no data-path collective).  Works on any initialised backend."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(units)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def make_workload(name: str):
    from paper_2603_19764_b200 import workloads as W
    k = int(name[1])
    return W.config(k)


ORACLE_SAMPLE_N = 1_000_000     # particles in the oracle's bounded sample (about 2 s per evaluation on 16 cores)
ORACLE_BUDGET_S = 12.0          # the cpu_baseline leg repeats the evaluation until this much CPU time is spent


def oracle_sample(wl, target_n: int = ORACLE_SAMPLE_N):
    """A bounded sample of the workload for the CPU oracle: the particles inside a cube around the
    median position that holds about target_n of them (complete neighbourhoods inside, cut faces)."""
    import numpy as np
    A = wl.arrays
    if wl.n <= target_n:
        return wl, "all %d particles" % wl.n
    p = np.stack([A["x"], A["y"], A["z"]]).astype(np.float64)
    c = np.median(p, axis=1, keepdims=True)
    d = np.abs(p - c).max(axis=0)
    half = np.partition(d, target_n)[target_n]
    idx = np.nonzero(d <= half)[0]
    return wl.subset(idx), "cube of %d particles around the median position (of %d)" % (idx.size, wl.n)


def time_oracle(wl, budget_s: float = 0.0, max_evals: int = 16):
    """Derivative evaluations (the pair work of one step) of the oracle, as it stands: one, or as
    many as fit in budget_s.  Returns (pairs per evaluation, mean seconds, threads, evaluations)."""
    from oracle import oracle as O
    import numpy as np
    A = {k: np.ascontiguousarray(v, dtype=np.float64) for k, v in wl.arrays.items()}
    S = np.stack([A["Sxx"], A["Syy"], A["Sxy"], A["Sxz"], A["Syz"]])
    g = np.stack([A["gx"], A["gy"], A["gz"]])
    O.lib()
    times = []
    pairs = 0
    while True:
        t0 = time.perf_counter()
        d = O.derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"],
                          A["u"], S, wl.mat, g, "grid")
        times.append(time.perf_counter() - t0)
        pairs = int(d["n_gather"].sum()) + int(d["n_symmetric"].sum())
        if sum(times) >= budget_s or len(times) >= max_evals:
            break
    return pairs, sum(times) / len(times), O.lib().orc_max_threads(), len(times)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.workload)
    sample, what = oracle_sample(wl)
    for _ in range(max(args.warmup, 0) and 1):
        time_oracle(sample)
    times = []
    pairs = 0
    for _ in range(args.steps):
        pairs, dt, cores, _n = time_oracle(sample)
        times.append(dt)
    total = sum(times)
    val = pairs * len(times) / total
    line = {
        "impl": "reference", "metric": "pair_interactions_per_s", "value": val, "unit": "pairs/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "n_particles": wl.n, "sample": what},
        "cpu_baseline": {"value": val, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": val, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "particle_steps_per_s": sample.n * len(times) / total,
    }
    print(json.dumps(line), flush=True)


# Algorithmic HBM bytes per particle of the HBM-bound passes
BYTES_PER_PARTICLE = {"predict": 128, "close": 230, "kickdrift": 160,
                      # S1 with a full build: keys 12 r + 12 w, radix sort 4-5 digit passes x 24, reorder 116 r + 116 w
                      "build_full": 24 + 5 * 24 + 232}

# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch, from the committed `ncu --set full` captures of this
# command (profiles/r02_*.md); None where no capture exists for the workload.
NCU_TRAFFIC_BYTES = {}
try:
    with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as _f:
        NCU_TRAFFIC_BYTES = json.load(_f)
except OSError:
    pass


def _respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun around it: start the N replica ranks ourselves
    (one process per GPU, NCCL only for the barrier and the max / sum over ranks)."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        sys.stderr.write("bench.py: --gpus %d asked, %d visible: refusing to time fewer GPUs than asked\n" % (args.gpus, have))
        return 2
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2603_19764_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    props = torch.cuda.get_device_properties(dev)
    # everything (torch fills, copies, the library's kernels, the timing events) on one non-default stream:
    # the library replays the resident step from a CUDA graph, and the default stream cannot be captured
    torch.cuda.set_stream(torch.cuda.Stream(dev))

    wl = make_workload(args.workload)
    if args.no_graph:
        wl.params.flags |= 64          # SPH_NO_GRAPH
    if args.skin is not None:
        wl.params.skin = args.skin
    if args.rebuild_every is not None:
        wl.params.rebuild_every = args.rebuild_every
    elif wl.params.skin > 0.0 and 0 < args.steps < wl.params.rebuild_every:
        # fewer timed steps than the list-reuse cycle: shorten the cycle so that the timed steps still hold one full
        # neighbour build (never time a window without the build it lives on)
        wl.params.rebuild_every = args.steps
    n = wl.n
    strength = bool(wl.params.flags & B.STRENGTH)
    reuse = wl.params.skin > 0.0
    every = (wl.params.rebuild_every if wl.params.rebuild_every > 0 else 8) if reuse else 1
    s = B.Sph(wl.params, n, device=dev)
    t = s.upload(wl)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB of L2
    working_set = s.workspace_bytes

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    # ---- the FP32 CUDA-core rate this device sustains (FFMA chains) ----------------------
    peak_measured = s.fp32_peak(5)

    # ---- device-resident timing -----------------------------------------------------------
    s.build_neighbors(t, n)
    for _ in range(args.warmup):
        s.step(None, 0, 0.0)
    barrier()
    launches0 = s.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    pass_ms = {k: 0.0 for k in B.T_SLOTS}
    pass_full = {k: 0.0 for k in B.T_SLOTS}
    pass_reuse = {k: 0.0 for k in B.T_SLOTS}
    n_full = n_reuse = 0
    pairs_g = pairs_s = entries = tests_cull = tests_cull_steps = dirty_max = 0
    barrier()
    for k in range(args.steps):
        flush.fill_(k & 0xff)
        ev[k][0].record(s.stream)
        s.step(None, 0, 0.0)
        ev[k][1].record(s.stream)
        tm = s.get_timings()                 # synchronises; outside the event pair of the next step
        c = s.get_counters()
        is_full = c["steps_since_full"] == 0         # what the library did, not a prediction of its schedule
        for q in B.T_SLOTS:
            pass_ms[q] += tm[q]
            (pass_full if is_full else pass_reuse)[q] += tm[q]
        n_full += 1 if is_full else 0
        n_reuse += 0 if is_full else 1
        pairs_g += c["pairs_gather"]; pairs_s += c["pairs_symmetric"]
        entries += c["tests_density"] + c["tests_force"]
        if is_full:
            tests_cull += c["tests_cull"]; tests_cull_steps += 1
        dirty_max = max(dirty_max, c["tiles_dirty"])
    barrier()
    launches = s.launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    pairs = pairs_g + pairs_s
    total_ms_max, pairs_all = rank_reduce(total_ms, pairs, dev)
    value = pairs_all / (total_ms_max * 1e-3)

    # ---- NEXT-4 (optional): big steps on 2^R rungs, the finest rung at the CFL step of the global stepper -------------
    rungs = None
    if args.rungs > 0:
        R = args.rungs
        dtu = torch.zeros(1, dtype=torch.float32, device=dev)
        s.step(None, 0, 0.0, dtu)
        dT = float(dtu.item()) * (1 << R)
        s.step_rungs(dT, R)                                   # warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nbig = 3
        upd = tiles = 0
        barrier()
        e0.record(s.stream)
        for _ in range(nbig):
            s.step_rungs(dT, R)
            c = s.get_counters()
            upd += c["active_updates"]; tiles += c["active_tiles"]
        e1.record(s.stream)
        barrier()
        big_ms = e0.elapsed_time(e1) / nbig
        rg = s.get_field("RUNG")
        rungs = {"max_rung": R, "dT": dT, "ms_per_big_step": big_ms,
                 "ms_of_the_same_span_on_one_rung": (total_ms / args.steps) * (1 << R),
                 "closing_kicks_per_big_step": upd / nbig, "of_global": upd / nbig / (n * (1 << R)),
                 "active_tiles_per_big_step": tiles / nbig, "of_all_tiles": tiles / nbig / (((n + 255) // 256) * (1 << R)),
                 "rung_histogram": torch.bincount(rg.to(torch.int64), minlength=R + 1).tolist(),
                 "particle_updates_per_s": upd / nbig / (big_ms * 1e-3)}

    # ---- the same step with strength off (S == 0, hydro only): BASELINE.json's "<= 30 % over hydro-only"
    hydro = None
    if strength and not args.no_hydro_only:
        import dataclasses
        wl_h = dataclasses.replace(wl, params=dataclasses.replace(wl.params, flags=wl.params.flags & ~B.STRENGTH))
        sh = B.Sph(wl_h.params, n, device=dev)
        th = sh.upload(wl_h)
        sh.build_neighbors(th, n)
        for _ in range(args.warmup):
            sh.step(None, 0, 0.0)
        barrier()
        hev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        hpass = {k: 0.0 for k in B.T_SLOTS}
        for k in range(args.steps):
            flush.fill_(k & 0xff)
            hev[k][0].record(sh.stream)
            sh.step(None, 0, 0.0)
            hev[k][1].record(sh.stream)
            tmh = sh.get_timings()
            for q in B.T_SLOTS:
                hpass[q] += tmh[q]
        barrier()
        h_ms = sum(a.elapsed_time(b) for a, b in hev) / args.steps
        hydro = {"ms_per_step": h_ms, "pass_ms": {k: v / args.steps for k, v in hpass.items()},
                 "strength_overhead": (total_ms / args.steps) / h_ms - 1.0}
        del sh, th

    # ---- end to end through the host-buffer entry point -----------------------------------
    del s, t
    torch.cuda.empty_cache()
    e2e_steps = max(1, min(args.steps, 32))      # like the device-timed leg: whole cycles of the list reuse
    e2e_s, e2e_pairs = 1.0, 0
    if not args.no_e2e:
        host = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in wl.arrays.items()}
        host["mat"] = torch.from_numpy(wl.mat.copy()).pin_memory()
        host["fixed"] = torch.from_numpy(wl.fixed.copy()).pin_memory()
        s2 = B.Sph(wl.params, n, device=dev)
        s2.step_host(host, n, 0.0)                                   # warm-up (also the bootstrap)
        s2.step_host(host, n, 0.0)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            s2.step_host(host, n, 0.0)
            c = s2.get_counters()
            e2e_pairs += c["pairs_gather"] + c["pairs_symmetric"]
        torch.cuda.synchronize(dev)
        e2e_s = time.perf_counter() - t0
    clocks = sampler.stop()          # sampled from the start of the device-timed steps to the end of the e2e steps
    e2e_s_max, e2e_pairs_all = rank_reduce(e2e_s, e2e_pairs, dev)
    e2e_value = e2e_pairs_all / e2e_s_max
    h2d = n * 17 * 4               # 17 float arrays per step (material and fixed flags travel with the first call only)
    d2h = n * 12 * 4 + 4

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines ------------------------------------------------------------------------------
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_nominal = fp32_peak_tflops(props.multi_processor_count, sm_max)
    peak = peak_measured if peak_measured > 0 else peak_nominal
    hbm_peak, hbm_src = measured_hbm_gbs()
    K = args.steps
    step_avg = total_ms / K
    traffic = NCU_TRAFFIC_BYTES.get(args.workload, {})

    def alu_entry(kernel, pass_key, units, flops_per_unit, what):
        ms = pass_ms[pass_key] / K
        ach = units / K * flops_per_unit / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        prof = traffic.get(kernel, {})
        ex = prof.get("executed_fp32_flop")
        out = {"kernel": kernel, "bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
               "frac_of_nominal": ach / peak_nominal, "kernel_ms": ms, "share_of_step": ms / step_avg,
               "work": what, "traffic": prof.get("traffic_bytes"), "traffic_unit": "bytes per launch"}
        if prof.get("traffic_bytes") and ms > 0:
            out["dram_gbs"] = prof["traffic_bytes"] / (ms * 1e-3) / 1e9       # measured DRAM bytes of a launch over this run's time
        if ex and ms > 0:
            # executed FP32 flop of one launch (2 ffma + fmul + fadd, ncu capture in profiles/) over THIS run's kernel time
            out["executed_achieved"] = ex / (ms * 1e-3) / 1e12
            out["executed_frac"] = out["executed_achieved"] / peak
            out["executed_frac_of_nominal"] = out["executed_achieved"] / peak_nominal
        return out

    flops_pair = FLOPS_PAIR_FUSED if strength else FLOPS_PAIR_HYDRO
    k_pair = alu_entry("k_pair_l", "force", pairs_s, flops_pair,
                       "%d flop per TRUE pair (gather counts exclude self), %.0f true pairs per launch"
                       % (flops_pair, pairs_s / K))
    k_dens = alu_entry("k_density_l", "density", pairs_g, FLOPS_PAIR_DENSITY,
                       "%d flop-equivalents per gather pair incl. self (20 fp32 + 12 fp64 x 2)" % FLOPS_PAIR_DENSITY)
    kernels = [k_pair, k_dens]
    if n_full:
        ms = pass_full["build"] / n_full
        by = BYTES_PER_PARTICLE["build_full"] * n
        kernels.append({"kernel": "S1 full build (keys, radix sort, k_permute, tree, k_cull, k_list_sort)", "bound": "hbm",
                        "achieved": by / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": by / (ms * 1e-3) / 1e9 / hbm_peak, "kernel_ms": ms,
                        "share_of_step": pass_ms["build"] / K / step_avg, "steps_per_full_build": every,
                        "work": "%d B per particle (SURVEY.md section 8d, S1)" % BYTES_PER_PARTICLE["build_full"],
                        "traffic": traffic.get("k_cull", {}).get("traffic_bytes"),
                        "traffic_unit": "bytes per launch of k_cull (full build)"})
    for key in ("predict", "close", "kickdrift"):
        ms = pass_ms[key] / K
        by = BYTES_PER_PARTICLE[key] * n
        kernels.append({"kernel": "k_" + ("kick_drift" if key == "kickdrift" else key), "bound": "hbm",
                        "achieved": by / (ms * 1e-3) / 1e9 if ms > 0 else 0.0, "peak": hbm_peak, "unit": "GB/s",
                        "frac": (by / (ms * 1e-3) / 1e9 / hbm_peak) if ms > 0 else 0.0, "kernel_ms": ms,
                        "share_of_step": ms / step_avg, "work": "%d B per particle" % BYTES_PER_PARTICLE[key]})
    roofline = dict(k_pair)
    roofline.update({"kernel": "k_pair_l<1,1,1> (fused Eq. 18-21 + 5-8)" if strength else "k_pair_l<0,1,0>",
                     "peak_source": "sph_fp32_peak: FFMA chains measured in this run (nominal %d SMs x 128 lanes x 2 x %.0f MHz = %.1f)"
                                    % (props.multi_processor_count, sm_max, peak_nominal),
                     "peak_nominal": peak_nominal, "peak_measured": peak_measured, "hbm_peak_source": hbm_src,
                     "flops_per_pair": flops_pair, "pairs_per_launch": pairs_s / K,
                     "list_entries_per_true_pair": entries / pairs if pairs else None,
                     "cull_tests_per_true_pair": (tests_cull / tests_cull_steps) / (pairs_s / K) if tests_cull_steps and pairs_s else None,
                     "candidate_hit_rate": (pairs_s / K) / (tests_cull / tests_cull_steps) if tests_cull else None,
                     "kernels": kernels})

    # ---- the oracle beside it ------------------------------------------------------------------
    cpu = None
    if not args.no_cpu_baseline:
        sample, what = oracle_sample(wl)
        op, ot, cores, nev = time_oracle(sample, ORACLE_BUDGET_S)
        cpu = {"value": op / ot, "unit": "pairs/s", "cores": cores, "kind": "oracle",
               "sample": "%s, %d evaluations of the step's derivatives" % (what, nev),
               "seconds": ot * nev, "particle_steps_per_s": sample.n / ot}

    line = {
        "metric": "pair_interactions_per_s", "value": value, "unit": "pairs/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": wl.name, "n_particles": n, "strength": strength,
                   # reading Q1: which rotation sign of Eq. 13 was timed (the cost is the same)
                   "jaumann": "as_printed" if (wl.params.flags & B.JAUMANN_AS_PRINTED) else "objective",
                   "mean_neighbours": pairs_s / args.steps / max(n, 1),
                   "pair_count": "value = gather pairs (Eq. 1, 3; the particle itself included: the self term is evaluated) "
                                 "+ symmetric pairs (Eq. 18-21; self excluded) per second",
                   "l2": "flushed between steps (256 MiB fill outside the timed events)",
                   "working_set_bytes": working_set, "parallelism": "replicas x%d" % world,
                   "cuda_graph": not args.no_graph,
                   "list_reuse": {"skin": wl.params.skin, "full_build_every": every, "full_steps_timed": n_full,
                                  "reuse_steps_timed": n_reuse, "dirty_tiles_max": dirty_max,
                                  "tiles": (n + 255) // 256} if reuse else None},
        "particle_steps_per_s": world * n * args.steps / (total_ms_max * 1e-3),
        "pass_ms": {k: v / args.steps for k, v in pass_ms.items()},
        "pass_ms_full_step": {k: v / n_full for k, v in pass_full.items()} if n_full else None,
        "pass_ms_reuse_step": {k: v / n_reuse for k, v in pass_reuse.items()} if n_reuse else None,
        "ms_per_step_min_max": [min(step_ms), max(step_ms)],
        "gpu_launches": launches,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "pairs/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s_max / e2e_steps,
                "note": "host buffers in and out every step; the loop hands back the state it received, so the library "
                        "finds x, y, z, h unchanged and keeps reusing its neighbour lists; on such steps u and S arrive while "
                        "the list check and the density pass run, a_ext and the outgoing x, y, z travel during the pair pass"},
        "roofline": roofline,
        "cpu_baseline": cpu,
        "hydro_only": hydro,
        "rungs": rungs,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def measured_hbm_gbs():
    """MEASURED_PEAKS.json (driver-written) if present, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, KeyError, ValueError):
        return 6650.0, "of fallback (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=32,
                    help="timed steps; the default covers one whole cycle of the list reuse of configs[4] (a full build every 32 steps)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=["c0", "c1", "c2", "c3", "c4"],
                    help="BASELINE.json configs[k]; default: the largest single-GPU configuration")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-hydro-only", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--rungs", type=int, default=0, help="NEXT-4: also time big steps on 2^R rungs (sph_step_rungs)")
    ap.add_argument("--no-graph", action="store_true", help="launch the step kernel by kernel (A/B of the CUDA graph)")
    ap.add_argument("--skin", type=float, default=None, help="list reuse: skin as a fraction of H (0 = off; A/B)")
    ap.add_argument("--rebuild-every", type=int, default=None, help="list reuse: steps between full builds (A/B)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(_respawn_under_torchrun(args))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
