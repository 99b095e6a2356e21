"""Thin ctypes binding of libsph.so (include/sph.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used here for device
memory (the workspace and the particle arrays are torch tensors) and for the CUDA stream.  There
is NO CPU fallback: load() raises if libsph.so is missing or a symbol is absent.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import sys
from typing import Dict, Optional

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsph.so")

MAX_MATERIALS = 8
STRENGTH, CORRECTION_TENSOR, PCLIP_GLOBAL, JAUMANN_AS_PRINTED, NO_LISTS = 1, 2, 4, 512, 16
OK, EINVAL, ENOMEM, ECUDA, EORDER, ECAPACITY = 0, -1, -2, -3, -4, -5
PREDICT, CLOSE, DERIVATIVES = 0, 1, 2
GATHER, SYMMETRIC = 0, 1

F = dict(RHO=0, OMEGA=1, P=2, CS=3, T=4, GAMMA=5, Y=6, MUMAX=7, DUDT=8, DT=9, EACC=10, EPS2=11, U=12,
         CFLAG=13, NGATHER=14, NSYMMETRIC=15, H=16, RUNG=17, TILE=18, A=32, V=36, X=40, SPRED=48, S=56, DSDT=64, F=80, CINV=96, G=112)
T_SLOTS = ("build", "density", "predict", "gradient", "force", "close", "kickdrift", "step")
C_SLOTS = ("pairs_gather", "pairs_symmetric", "tests_density", "tests_force", "cfallback", "tests_cull",
           "candidates", "list_overflow", "bad_material", "omega_small", "nonfinite", "tiles_dirty", "active_updates", "active_tiles", "pairs_intile", "list_slots",
           "rung_clamped", "steps_since_full")

FLOAT_FIELDS = ("x", "y", "z", "m", "h", "vx", "vy", "vz", "u", "Sxx", "Syy", "Sxy", "Sxz", "Syz")
OPT_FIELDS = ("gx", "gy", "gz")

# every symbol include/sph.h declares (tests check the library exports all of them)
SYMBOLS = ("sph_workspace_bytes", "sph_init", "sph_build_neighbors", "sph_density", "sph_strength_update",
           "sph_gradients", "sph_forces", "sph_gradients_forces", "sph_fp32_peak", "sph_fp32_rate", "sph_step_rungs", "sph_adapt_h", "sph_set_eos_table", "sph_step", "sph_step_host", "sph_download_state", "sph_get_field",
           "sph_get_neighbors", "sph_get_timings", "sph_get_counters", "sph_get_tile_stats", "sph_get_tile_dirty", "sph_get_diagnostics",
           "sph_diagnostics_noalloc", "sph_launch_count",
           "sph_last_cuda_error", "sph_strerror", "sph_destroy")


class sph_eos_table(C.Structure):
    _fields_ = [("n_rho", C.c_int), ("n_u", C.c_int), ("n_melt", C.c_int),
                ("rho_min", C.c_float), ("rho_max", C.c_float), ("u_min", C.c_float), ("u_max", C.c_float),
                ("P", C.c_void_p), ("T", C.c_void_p), ("cs", C.c_void_p), ("Tmelt", C.c_void_p)]


class sph_material(C.Structure):
    _fields_ = [(k, C.c_float) for k in
                ("rho0", "c0", "cv", "Gamma", "nu", "Y0", "Ym", "mu_i", "mu_d", "xi", "Tmelt")]


class sph_params(C.Structure):
    _fields_ = [("kappa", C.c_float), ("alpha", C.c_float), ("beta", C.c_float), ("eps_av", C.c_float),
                ("eta_C", C.c_float), ("eta_a", C.c_float), ("n_materials", C.c_int), ("flags", C.c_uint),
                ("mat", sph_material * MAX_MATERIALS), ("list_budget", C.c_int),
                ("skin", C.c_float), ("rebuild_every", C.c_int), ("adapt_h_every", C.c_int), ("adapt_h_target", C.c_float)]


class sph_state(C.Structure):
    _fields_ = ([(k, C.c_void_p) for k in FLOAT_FIELDS] + [(k, C.c_void_p) for k in OPT_FIELDS]
                + [("mat", C.c_void_p), ("fixed", C.c_void_p)])


class SphError(RuntimeError):
    def __init__(self, code: int, what: str, msg: str):
        super().__init__(f"{what}: {msg} ({code})")
        self.code = code


_lib = None


def _ensure_built():
    """Compile libsph.so when it is missing or older than its sources (nvcc is in the image; this is a
    build step, not a fallback).  Under torchrun only local rank 0 compiles; the others wait for the file."""
    import time
    from . import build as _build
    if os.environ.get("LOCAL_RANK", "0") == "0":
        try:
            _build.build()                          # compiles to a temporary file and renames it into place
        except Exception as e:
            # a failed rebuild must not run a stale binary silently
            raise RuntimeError(f"building {LIB_PATH} failed: {e} (there is no CPU fallback)") from e
        return
    t0 = time.time()
    while _build.stale() and time.time() - t0 < 600.0:        # until rank 0 has renamed a current library into place
        time.sleep(1.0)


def load():
    """dlopen libsph.so and declare the prototypes.  Fails loudly; never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.environ.get("SPH_LIB")             # another build of the same sources (build.build(out=..., defines=...))
    if not path:
        path = LIB_PATH
        _ensure_built()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2603_19764_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    for s in SYMBOLS:
        getattr(lib, s)                      # AttributeError if a declared symbol is not exported
    vp, ll, fl, i = C.c_void_p, C.c_longlong, C.c_float, C.c_int
    lib.sph_workspace_bytes.restype = C.c_size_t
    lib.sph_workspace_bytes.argtypes = [C.POINTER(sph_params), ll]
    lib.sph_init.argtypes = [C.POINTER(vp), C.POINTER(sph_params), ll, vp, C.c_size_t, vp]
    lib.sph_build_neighbors.argtypes = [vp, C.POINTER(sph_state), ll]
    lib.sph_density.argtypes = [vp]
    lib.sph_strength_update.argtypes = [vp, i, fl]
    lib.sph_gradients.argtypes = [vp]
    lib.sph_forces.argtypes = [vp]
    lib.sph_gradients_forces.argtypes = [vp]
    lib.sph_gradients_forces.restype = i
    lib.sph_fp32_peak.argtypes = [vp, i, C.POINTER(C.c_double)]
    lib.sph_fp32_peak.restype = i
    lib.sph_fp32_rate.argtypes = [vp, i, i, C.POINTER(C.c_double)]
    lib.sph_fp32_rate.restype = i
    lib.sph_step_rungs.argtypes = [vp, fl, i, vp]
    lib.sph_step_rungs.restype = i
    lib.sph_step.argtypes = [vp, C.POINTER(sph_state), ll, fl, vp]
    lib.sph_step_host.argtypes = [vp, C.POINTER(sph_state), ll, fl, vp]
    lib.sph_download_state.argtypes = [vp, C.POINTER(sph_state)]
    lib.sph_get_field.argtypes = [vp, i, vp]
    lib.sph_get_neighbors.argtypes = [vp, i, vp, vp, vp]
    lib.sph_get_timings.argtypes = [vp, C.POINTER(fl), i]
    lib.sph_get_counters.argtypes = [vp, C.POINTER(ll), i]
    lib.sph_get_tile_stats.argtypes = [vp, vp, vp, vp, i]
    lib.sph_get_tile_dirty.argtypes = [vp, vp, i]
    lib.sph_get_tile_dirty.restype = i
    lib.sph_set_eos_table.argtypes = [vp, i, vp]
    lib.sph_set_eos_table.restype = i
    lib.sph_get_diagnostics.argtypes = [vp, vp]
    lib.sph_get_diagnostics.restype = i
    lib.sph_diagnostics_noalloc.argtypes = [C.POINTER(sph_state), ll, vp, vp, C.POINTER(i)]
    lib.sph_diagnostics_noalloc.restype = i
    lib.sph_adapt_h.argtypes = [vp, fl, i, vp]
    lib.sph_adapt_h.restype = i
    lib.sph_launch_count.restype = ll
    lib.sph_launch_count.argtypes = [vp]
    lib.sph_last_cuda_error.argtypes = [vp]
    lib.sph_strerror.restype = C.c_char_p
    lib.sph_strerror.argtypes = [i]
    lib.sph_destroy.restype = None
    lib.sph_destroy.argtypes = [vp]
    for s in ("sph_init", "sph_build_neighbors", "sph_density", "sph_strength_update", "sph_gradients",
              "sph_forces", "sph_step", "sph_step_host", "sph_download_state", "sph_get_field",
              "sph_get_neighbors", "sph_get_timings", "sph_get_counters", "sph_get_tile_stats",
              "sph_last_cuda_error"):
        getattr(lib, s).restype = i
    _lib = lib
    return lib


def make_params(p) -> sph_params:
    """Marshal a workloads.Params-like record (duck-typed) into the C struct."""
    out = sph_params()
    out.kappa, out.alpha, out.beta, out.eps_av = p.kappa, p.alpha, p.beta, p.eps_av
    out.eta_C, out.eta_a = p.eta_C, p.eta_a
    out.flags = int(p.flags)
    out.list_budget = int(getattr(p, "list_budget", 0))
    out.skin = float(getattr(p, "skin", 0.0))
    out.rebuild_every = int(getattr(p, "rebuild_every", 0))
    out.adapt_h_every = int(getattr(p, "adapt_h_every", 0))
    out.adapt_h_target = float(getattr(p, "adapt_h_target", 0.0))
    out.n_materials = len(p.materials)
    for k, m in enumerate(p.materials):
        for name, _ in sph_material._fields_:
            setattr(out.mat[k], name, float(getattr(m, name)))
    return out


def _ptr(t) -> Optional[int]:
    return None if t is None else int(t.data_ptr())


DIAG_NOALLOC_MAX_N = 1 << 25       # SPH_DIAG_NOALLOC_MAX_N of include/sph.h


def diagnostics_noalloc(tensors: Dict[str, object], n: int, out, stream=None):
    """sph_diagnostics_noalloc: the eight S8 sums (M, P, L, E) of the caller's own device arrays, written to `out`
    (float64 device tensor [8], supplied by the caller).  For programs that cannot allocate on the GPU -- all of
    its memory already belongs to their own pool, or an allocation's device-wide synchronisation would stall their
    loop: neither the library nor this wrapper allocates anything; the partial sums live in a static array inside
    libsph.so, which limits n to DIAG_NOALLOC_MAX_N.  tensors: x, y, z, m, vx, vy, vz, u (float32, on out's
    device, which must be the current one).  Calls on different streams of one device must not overlap."""
    import torch
    lib = load()
    st = sph_state()
    for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u"):
        setattr(st, k, _ptr(tensors.get(k)))
    if stream is None:
        stream = torch.cuda.current_stream(out.device)
    err = C.c_int(0)
    rc = lib.sph_diagnostics_noalloc(C.byref(st), int(n), _ptr(out), stream.cuda_stream, C.byref(err))
    if rc == ECAPACITY:
        raise SphError(rc, "sph_diagnostics_noalloc", f"n = {n} is more than the static scratch array holds "
                                                      f"(SPH_DIAG_NOALLOC_MAX_N = {DIAG_NOALLOC_MAX_N})")
    if rc != 0:
        raise SphError(rc, "sph_diagnostics_noalloc", lib.sph_strerror(rc).decode() + (f" cudaError={err.value}" if rc == ECUDA else ""))
    return out


class Sph:
    """One sph_ctx plus the torch tensors that back it.  Method names follow include/sph.h."""

    def __init__(self, params, n_max: int, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.lib = load()
        self.device = torch.device(device)
        self.cparams = make_params(params)
        self.n_max = int(n_max)
        need = self.lib.sph_workspace_bytes(C.byref(self.cparams), self.n_max)
        if need == 0:
            raise SphError(EINVAL, "sph_workspace_bytes", "invalid parameters")
        self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
        self.workspace_bytes = need
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.ctx = C.c_void_p()
        self._check(self.lib.sph_init(C.byref(self.ctx), C.byref(self.cparams), self.n_max,
                                      self.workspace.data_ptr(), need, self.stream.cuda_stream), "sph_init")
        self.n = 0
        self._dev_state: Dict[str, object] = {}
        self._tables: Dict[int, object] = {}
        for k, m in enumerate(params.materials):          # NEXT-3: materials that carry an EOS table
            if getattr(m, "table", None) is not None:
                self.set_eos_table(k, m.table)

    # ---- plumbing ---------------------------------------------------------------------------
    def _check(self, rc: int, what: str):
        if rc != 0:
            msg = self.lib.sph_strerror(rc).decode()
            if rc == ECUDA and self.ctx:
                msg += f" cudaError={self.lib.sph_last_cuda_error(self.ctx)}"
            raise SphError(rc, what, msg)

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.sph_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def state_struct(self, tensors: Dict[str, object]) -> sph_state:
        st = sph_state()
        for k in FLOAT_FIELDS:
            setattr(st, k, _ptr(tensors[k]))
        for k in OPT_FIELDS + ("mat", "fixed"):
            setattr(st, k, _ptr(tensors.get(k)))
        return st

    def upload(self, wl) -> Dict[str, object]:
        """Copy a workloads.Workload to device tensors (plumbing; not part of the C ABI)."""
        torch = self.torch
        t = {k: torch.from_numpy(v).to(self.device) for k, v in wl.arrays.items()}
        t["mat"] = torch.from_numpy(wl.mat).to(self.device)
        t["fixed"] = torch.from_numpy(wl.fixed).to(self.device)
        self._dev_state = t
        return t

    # ---- the C ABI, one method per entry point -----------------------------------------------
    def build_neighbors(self, tensors: Optional[Dict[str, object]] = None, n: int = 0):
        if tensors is None:
            self._check(self.lib.sph_build_neighbors(self.ctx, None, 0), "sph_build_neighbors")
        else:
            st = self.state_struct(tensors)
            self._check(self.lib.sph_build_neighbors(self.ctx, C.byref(st), n), "sph_build_neighbors")
            self.n = n

    def density(self):
        self._check(self.lib.sph_density(self.ctx), "sph_density")

    def strength_update(self, phase: int, dt: float = 0.0):
        self._check(self.lib.sph_strength_update(self.ctx, phase, dt), "sph_strength_update")

    def gradients(self):
        self._check(self.lib.sph_gradients(self.ctx), "sph_gradients")

    def forces(self):
        self._check(self.lib.sph_forces(self.ctx), "sph_forces")

    def gradients_forces(self):
        self._check(self.lib.sph_gradients_forces(self.ctx), "sph_gradients_forces")

    def fp32_peak(self, repeats: int = 5) -> float:
        """sph_fp32_peak: TFLOP/s of independent FFMA chains on this device (measurement aid)."""
        out = C.c_double(0.0)
        self._check(self.lib.sph_fp32_peak(self.stream.cuda_stream, int(repeats), C.byref(out)), "sph_fp32_peak")
        return float(out.value)

    def fp32_rate(self, variant: int, repeats: int = 5) -> float:
        """sph_fp32_rate: TFLOP/s of FFMA chains in another instruction form (see include/sph.h)."""
        out = C.c_double(0.0)
        self._check(self.lib.sph_fp32_rate(self.stream.cuda_stream, int(variant), int(repeats), C.byref(out)), "sph_fp32_rate")
        return float(out.value)

    def step(self, tensors: Optional[Dict[str, object]] = None, n: int = 0, dt: float = 0.0, dt_used=None):
        st = C.byref(self.state_struct(tensors)) if tensors is not None else None
        if tensors is not None:
            self.n = n
        self._check(self.lib.sph_step(self.ctx, st, n, dt, _ptr(dt_used)), "sph_step")

    def step_rungs(self, dT: float, max_rung: int, rungs=None):
        """sph_step_rungs; rungs: optional uint8 device tensor [n] in caller order (fixed rungs)."""
        self._check(self.lib.sph_step_rungs(self.ctx, float(dT), int(max_rung), _ptr(rungs)), "sph_step_rungs")

    def step_host(self, host: Dict[str, object], n: int, dt: float = 0.0) -> float:
        """host: dict of (pinned) CPU torch tensors / numpy arrays keyed like sph_state."""
        st = sph_state()
        for k in FLOAT_FIELDS + OPT_FIELDS + ("mat", "fixed"):
            v = host.get(k)
            if v is None:
                setattr(st, k, None)
            elif hasattr(v, "data_ptr"):
                setattr(st, k, int(v.data_ptr()))
            else:
                setattr(st, k, int(v.ctypes.data))
        used = C.c_float(0.0)
        self._check(self.lib.sph_step_host(self.ctx, C.byref(st), n, dt, C.addressof(used)), "sph_step_host")
        self.n = n
        return float(used.value)

    def download_state(self, tensors: Dict[str, object]):
        st = self.state_struct(tensors)
        self._check(self.lib.sph_download_state(self.ctx, C.byref(st)), "sph_download_state")

    def get_field(self, name: str, comp: int = 0):
        out = self.torch.empty(max(self.n, 1), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.sph_get_field(self.ctx, F[name] + comp, out.data_ptr()), "sph_get_field")
        return out[: self.n]

    def get_fields(self, name: str, ncomp: int):
        return self.torch.stack([self.get_field(name, c) for c in range(ncomp)], dim=0)

    def get_neighbors(self, which: int, select=None):
        """(counts[n], offsets[n+1], list) on the device; list holds ORIGINAL ids, rows unordered.
        select (caller-order indices): only these particles' ids are written (offsets = -1 elsewhere)."""
        torch = self.torch
        counts = torch.zeros(max(self.n, 1), dtype=torch.int32, device=self.device)
        self._check(self.lib.sph_get_neighbors(self.ctx, which, counts.data_ptr(), None, None), "sph_get_neighbors")
        counts = counts[: self.n]
        if select is not None:
            sel = torch.as_tensor(select, dtype=torch.long, device=self.device)
            csel = counts[sel].to(torch.int64)
            offsets = torch.full((self.n + 1,), -1, dtype=torch.int64, device=self.device)
            starts = torch.cumsum(csel, dim=0) - csel
            offsets[sel] = starts
            total = int(csel.sum().item())
            lst = torch.zeros(max(total, 1), dtype=torch.int32, device=self.device)
            self._check(self.lib.sph_get_neighbors(self.ctx, which, counts.data_ptr(), offsets.data_ptr(), lst.data_ptr()),
                        "sph_get_neighbors")
            so = torch.zeros(sel.numel() + 1, dtype=torch.int64, device=self.device)
            so[1:] = torch.cumsum(csel, dim=0)
            return counts[sel], so, lst[:total]
        offsets = torch.zeros(self.n + 1, dtype=torch.int64, device=self.device)
        if self.n:
            offsets[1:] = torch.cumsum(counts.to(torch.int64), dim=0)
        total = int(offsets[-1].item()) if self.n else 0
        lst = torch.zeros(max(total, 1), dtype=torch.int32, device=self.device)
        self._check(self.lib.sph_get_neighbors(self.ctx, which, counts.data_ptr() if self.n else lst.data_ptr(),
                                               offsets.data_ptr(), lst.data_ptr()), "sph_get_neighbors")
        return counts, offsets, lst[:total]

    def get_timings(self) -> Dict[str, float]:
        ms = (C.c_float * len(T_SLOTS))()
        self._check(self.lib.sph_get_timings(self.ctx, ms, len(T_SLOTS)), "sph_get_timings")
        return {k: float(ms[i]) for i, k in enumerate(T_SLOTS)}

    def get_counters(self) -> Dict[str, int]:
        cs = (C.c_longlong * len(C_SLOTS))()
        self._check(self.lib.sph_get_counters(self.ctx, cs, len(C_SLOTS)), "sph_get_counters")
        return {k: int(cs[i]) for i, k in enumerate(C_SLOTS)}

    def set_eos_table(self, material: int, table):
        """sph_set_eos_table; table: a workloads.EosTable-like record (numpy arrays) or None."""
        if table is None:
            self._check(self.lib.sph_set_eos_table(self.ctx, int(material), None), "sph_set_eos_table")
            self._tables.pop(material, None)
            return
        torch = self.torch
        dev = {k: torch.as_tensor(getattr(table, k), dtype=torch.float32, device=self.device).contiguous()
               for k in ("P", "T", "cs")}
        tm = None if table.Tmelt is None else torch.as_tensor(table.Tmelt, dtype=torch.float32, device=self.device).contiguous()
        t = sph_eos_table()
        t.n_rho, t.n_u = dev["P"].shape
        t.n_melt = 0 if tm is None else tm.shape[0]
        t.rho_min, t.rho_max, t.u_min, t.u_max = table.rho_min, table.rho_max, table.u_min, table.u_max
        t.P, t.T, t.cs = dev["P"].data_ptr(), dev["T"].data_ptr(), dev["cs"].data_ptr()
        t.Tmelt = None if tm is None else tm.data_ptr()
        self._check(self.lib.sph_set_eos_table(self.ctx, int(material), C.byref(t)), "sph_set_eos_table")
        self._tables[material] = (dev, tm)              # keep the device arrays alive

    def adapt_h(self, n_target: float, iterations: int, max_change=None):
        """sph_adapt_h; max_change: optional 1-element float32 device tensor."""
        ptr = max_change.data_ptr() if max_change is not None else None
        self._check(self.lib.sph_adapt_h(self.ctx, float(n_target), int(iterations), ptr), "sph_adapt_h")

    def get_diagnostics(self):
        """float64 device tensor [8]: M, P (3), L (3), E = sum m (v^2/2 + u)."""
        out = self.torch.zeros(8, dtype=self.torch.float64, device=self.device)
        self._check(self.lib.sph_get_diagnostics(self.ctx, out.data_ptr()), "sph_get_diagnostics")
        return out

    def get_tile_stats(self):
        """(candidates, cycles, fell_back) per tile of the last neighbour build, as numpy arrays (host)."""
        import numpy as np
        nt = self.lib.sph_get_tile_stats(self.ctx, None, None, None, 0)
        self._check(min(nt, 0), "sph_get_tile_stats")
        nc = np.zeros(nt, np.int32); cy = np.zeros(nt, np.uint32); fl = np.zeros(nt, np.uint8)
        rc = self.lib.sph_get_tile_stats(self.ctx, nc.ctypes.data, cy.ctypes.data, fl.ctypes.data, nt)
        self._check(min(rc, 0), "sph_get_tile_stats")
        return nc, cy, fl

    def get_tile_dirty(self):
        """sph_get_tile_dirty: uint8 numpy array, 1 for tiles whose lists are rebuilt in every step (host)."""
        import numpy as np
        nt = self.lib.sph_get_tile_dirty(self.ctx, None, 0)
        self._check(min(nt, 0), "sph_get_tile_dirty")
        out = np.zeros(nt, np.uint8)
        self._check(min(self.lib.sph_get_tile_dirty(self.ctx, out.ctypes.data, nt), 0), "sph_get_tile_dirty")
        return out

    def launch_count(self) -> int:
        return int(self.lib.sph_launch_count(self.ctx))

    # ---- convenience: BASELINE.json configs[0] single pass -------
    def single_pass(self, tensors, n: int, dt: float, fused: bool = False):
        """fused: S4 + S5 in one pass (sph_gradients_forces, the kernel sph_step runs) instead of two."""
        self.build_neighbors(tensors, n)
        self.density()
        self.strength_update(PREDICT)
        if fused:
            self.gradients_forces()
        else:
            if self.cparams.flags & STRENGTH:
                self.gradients()
            self.forces()
        self.strength_update(CLOSE, dt)
