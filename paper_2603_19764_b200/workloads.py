"""Seeded synthetic particle sets shaped like the paper's workloads.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path, so it
holds none of the method's arithmetic: no kernel function, no EOS, no yield
law.  It only lays particles out (lattices, spheres, a column on a floor), draws
jitter / noise from a stateless counter-based generator and writes the material
constants of BASELINE.json's configs into plain records.  The synthetic EOS tables
(``synthetic_eos_table``) are input DATA in the same sense: smooth surfaces sampled on a grid,
standing in for the paper's M-ANEOS tables; how a table is looked up is the method's business and
lives in oracle/ and in the CUDA path, separately.

Recipe: everything is generated in
fp64 from splitmix64(seed + GOLDEN*(16*i + stream)) and cast ONCE to fp32; the
oracle and the GPU read the same fp32 arrays.  seed = 260319764 + config index.

The paper's own initial conditions (relaxed BCC quartz bodies, M-ANEOS states;
PAPER.md:258, 299, 363) are not available; these sets stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

SEED_BASE = 260319764

# flag bits of sph_params.flags (mirrored in include/sph.h and oracle/oracle.py;
# plain constants, no arithmetic)
FLAG_STRENGTH = 1
FLAG_CORRECTION_TENSOR = 2
FLAG_PCLIP_GLOBAL = 4
FLAG_JAUMANN_AS_PRINTED = 512
FLAG_NO_LISTS = 16
FLAG_NO_GRAPH = 64

G_NEWTON = 6.674e-11

FIELDS = ("x", "y", "z", "m", "h", "vx", "vy", "vz", "u",
          "Sxx", "Syy", "Sxy", "Sxz", "Syz", "gx", "gy", "gz")


@dataclass
class EosTable:
    """Tabulated EOS of one material on a uniform (rho, u) grid (P and T come from
    EOSlib as functions of rho and u; T_melt is "a tabulated function of density").  Values are fp32;
    P, T, cs have shape (n_rho, n_u); Tmelt has shape (n_melt,) over the same rho range, or is None
    (constant T_melt of the material).  How the values are looked up is the method's business
    (oracle / CUDA), not this module's."""
    rho_min: float
    rho_max: float
    u_min: float
    u_max: float
    P: np.ndarray
    T: np.ndarray
    cs: np.ndarray
    Tmelt: Optional[np.ndarray] = None


@dataclass
class Material:
    """Per-material constants (BASELINE.json configs[0])."""
    rho0: float = 2700.0
    c0: float = 3000.0
    cv: float = 1000.0
    Gamma: float = 22.7e9      # > 0: constant shear modulus; <= 0: Eq. 30 with nu
    nu: float = 0.25
    Y0: float = 10.0e6
    Ym: float = 3.5e9
    mu_i: float = 1.5
    mu_d: float = math.inf     # +inf disables Eq. 35-36
    xi: float = 1.2
    Tmelt: float = 1500.0
    table: Optional[EosTable] = None   # NEXT-3: tabulated EOS instead of the analytic stand-in


@dataclass
class Params:
    kappa: float = 2.0
    alpha: float = 1.0
    beta: float = 2.0
    eps_av: float = 0.01
    eta_C: float = 0.3
    eta_a: float = 0.0
    flags: int = FLAG_STRENGTH | FLAG_CORRECTION_TENSOR
    list_budget: int = 0       # neighbour-list rows per particle of the CUDA path (0 = library default)
    skin: float = 0.0          # CUDA path: list reuse between full neighbour builds (sph_params.skin); no effect on results
    rebuild_every: int = 0     # CUDA path: steps between full builds when skin > 0 (0 = library default)
    adapt_h_every: int = 0     # sph_step: one smoothing-length iteration every so many steps (0 = never)
    adapt_h_target: float = 0.0
    materials: List[Material] = field(default_factory=lambda: [Material()])


@dataclass
class Workload:
    name: str
    params: Params
    arrays: Dict[str, np.ndarray]          # fp32, length n, keys = FIELDS
    mat: np.ndarray                        # int32
    fixed: np.ndarray                      # uint8
    dt: float                              # a fixed step for single-pass parity
    notes: str = ""

    @property
    def n(self) -> int:
        return int(self.arrays["x"].shape[0])

    def subset(self, idx: np.ndarray, name: Optional[str] = None) -> "Workload":
        idx = np.asarray(idx)
        return Workload(name or (self.name + "_subset"), self.params,
                        {k: np.ascontiguousarray(v[idx]) for k, v in self.arrays.items()},
                        np.ascontiguousarray(self.mat[idx]),
                        np.ascontiguousarray(self.fixed[idx]), self.dt, self.notes)


# ----------------------------------------------------------------------------
# counter-based generator (ours, nothing in the paper)
# ----------------------------------------------------------------------------
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.uint64, copy=True)
    z ^= z >> np.uint64(30)
    z *= np.uint64(0xBF58476D1CE4E5B9)
    z ^= z >> np.uint64(27)
    z *= np.uint64(0x94D049BB133111EB)
    z ^= z >> np.uint64(31)
    return z


def uniform01(seed: int, index: np.ndarray, stream: int) -> np.ndarray:
    """U[0,1) for particle ``index`` and ``stream`` (0..15); stateless."""
    with np.errstate(over="ignore"):
        ctr = index.astype(np.uint64) * np.uint64(16) + np.uint64(stream)
        z = np.uint64(seed) + _GOLDEN * ctr
        r = _splitmix64(z)
    return (r >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, index: np.ndarray, stream_a: int, stream_b: int) -> np.ndarray:
    """N(0,1) by Box-Muller from two streams."""
    u1 = uniform01(seed, index, stream_a)
    u2 = uniform01(seed, index, stream_b)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _finish(name, params, cols, mat, fixed, dt, notes) -> Workload:
    n = cols["x"].shape[0]
    arrays = {}
    for k in FIELDS:
        arrays[k] = _f32(cols[k]) if k in cols else np.zeros(n, dtype=np.float32)
    return Workload(name, params, arrays,
                    np.ascontiguousarray(mat, dtype=np.int32),
                    np.ascontiguousarray(fixed, dtype=np.uint8), float(dt), notes)


def _lattice_block(nx, ny, nz, dx, seed, jitter=0.05, origin=(0.0, 0.0, 0.0), first_index=0):
    i, j, k = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    i = i.ravel(); j = j.ravel(); k = k.ravel()
    idx = np.arange(i.size, dtype=np.int64) + first_index
    x = origin[0] + (i + 0.5) * dx + (2.0 * uniform01(seed, idx, 0) - 1.0) * jitter * dx
    y = origin[1] + (j + 0.5) * dx + (2.0 * uniform01(seed, idx, 1) - 1.0) * jitter * dx
    z = origin[2] + (k + 0.5) * dx + (2.0 * uniform01(seed, idx, 2) - 1.0) * jitter * dx
    return x, y, z, idx


# ----------------------------------------------------------------------------
# configs[0]: tiny elastic block (also used, scaled, for parity at other sizes)
# ----------------------------------------------------------------------------
def elastic_block(n_side: int = 16, seed: int = SEED_BASE, dx: float = 0.01,
                  flags: int = FLAG_STRENGTH | FLAG_CORRECTION_TENSOR,
                  h_spread: float = 0.0, two_materials: bool = False,
                  eos_table: Optional[str] = None) -> Workload:
    """BASELINE.json configs[0]: jittered n_side^3 lattice, shear flow, random S, T in [300,1600] K.

    ``h_spread`` > 0 multiplies h by U(1-h_spread, 1+h_spread) per particle (a parity
    case for the symmetric neighbour set with h_i != h_j); ``two_materials`` gives the
    upper half (y > mid) material 1 (configs[3] second material); ``eos_table`` ("linear" |
    "curved") attaches a synthetic EOS table to every material (NEXT-3).
    """
    mat0 = Material()
    mats = [mat0]
    if two_materials:
        mats.append(Material(Y0=1.0e6, mu_i=1.0))
    if eos_table:
        for mm in mats:
            mm.table = synthetic_eos_table(mm, eos_table)
    x, y, z, idx = _lattice_block(n_side, n_side, n_side, dx, seed)
    n = idx.size
    h = np.full(n, 1.3 * dx)
    if h_spread > 0.0:
        h = h * (1.0 + h_spread * (2.0 * uniform01(seed, idx, 15) - 1.0))
    m = np.full(n, mat0.rho0 * dx ** 3)
    vx = 100.0 * y + 0.01 * normal(seed, idx, 3, 4)
    vy = 0.01 * normal(seed, idx, 5, 6)
    vz = 0.01 * normal(seed, idx, 7, 8)
    s_amp = mat0.Y0 / 3.0
    S = [s_amp * (2.0 * uniform01(seed, idx, 9 + c) - 1.0) for c in range(5)]
    T = 300.0 + 1300.0 * uniform01(seed, idx, 14)
    u = mat0.cv * T
    mat = np.zeros(n, dtype=np.int32)
    if two_materials:
        mat[y > 0.5 * n_side * dx] = 1
    cols = dict(x=x, y=y, z=z, m=m, h=h, vx=vx, vy=vy, vz=vz, u=u,
                Sxx=S[0], Syy=S[1], Sxy=S[2], Sxz=S[3], Syz=S[4])
    params = Params(flags=flags, materials=mats)
    return _finish(f"elastic_block_{n_side}^3", params, cols, mat, np.zeros(n, np.uint8), 5.0e-7,
                   "BASELINE.json configs[0]; free surfaces; dt fixed at 5e-7 s for the single pass")


# ----------------------------------------------------------------------------
# configs[1]: granular column on a fixed floor
# ----------------------------------------------------------------------------
def granular_column(scale: float = 1.0, seed: int = SEED_BASE + 1) -> Workload:
    """BASELINE.json configs[1]: 46 x 92 x 46 column + 4 fixed floor layers (92 x 4 x 92).

    Shape after PAPER.md:268-270 (fixed floor layers, material released under gravity).
    ``scale`` < 1 shrinks every edge for parity-sized cases.
    """
    dx = 1.0
    cx = max(4, int(round(46 * scale))); cy = 2 * cx; fl = 2 * cx
    mat0 = Material(rho0=2700.0, c0=300.0, Gamma=0.0,   # Eq. 30 mode (nu = 0.25)
                    Y0=0.0, Ym=3.5e9, mu_i=2.0, mu_d=0.8)
    xc, yc, zc, idc = _lattice_block(cx, cy, cx, dx, seed, origin=((fl - cx) // 2 * dx, 0.0, (fl - cx) // 2 * dx))
    xf, yf, zf, idf = _lattice_block(fl, 4, fl, dx, seed, origin=(0.0, -4.0 * dx, 0.0), first_index=idc.size)
    x = np.concatenate([xc, xf]); y = np.concatenate([yc, yf]); z = np.concatenate([zc, zf])
    n = x.size
    fixed = np.concatenate([np.zeros(idc.size, np.uint8), np.ones(idf.size, np.uint8)])
    cols = dict(x=x, y=y, z=z, m=np.full(n, mat0.rho0 * dx ** 3), h=np.full(n, 1.3 * dx),
                vx=np.zeros(n), vy=np.zeros(n), vz=np.zeros(n), u=np.full(n, mat0.cv * 300.0),
                gx=np.zeros(n), gy=np.full(n, -9.81), gz=np.zeros(n))
    params = Params(flags=FLAG_STRENGTH | FLAG_CORRECTION_TENSOR | FLAG_PCLIP_GLOBAL, materials=[mat0])
    return _finish(f"granular_column_{cx}x{cy}x{cx}", params, cols, np.zeros(n, np.int32), fixed, 0.0,
                   "BASELINE.json configs[1]; Y0=0, mu_d=0.8, g=9.81 as a_ext; PCLIP_GLOBAL")


# ----------------------------------------------------------------------------
# spheres (configs[2..4])
# ----------------------------------------------------------------------------
def _unit_ball_lattice(n_target: int, seed: int, first_index: int = 0, jitter: float = 0.05):
    """Cubic lattice cut to |xi| < 1 with about n_target points; returns xi (n,3), spacing, index."""
    delta = (4.0 * math.pi / 3.0 / n_target) ** (1.0 / 3.0)
    nside = int(math.ceil(2.0 / delta)) + 1
    g = (np.arange(nside) - 0.5 * (nside - 1)) * delta
    # build per-slab to bound memory at 3e7 particles
    out = []
    g2 = g * g
    for gx in g:
        r2 = gx * gx + g2[:, None] + g2[None, :]
        jj, kk = np.nonzero(r2 < 1.0)
        if jj.size:
            out.append(np.stack([np.full(jj.size, gx), g[jj], g[kk]], axis=1))
    xi = np.concatenate(out, axis=0)
    idx = np.arange(xi.shape[0], dtype=np.int64) + first_index
    for a in range(3):
        xi[:, a] += (2.0 * uniform01(seed, idx, a) - 1.0) * jitter * delta
    return xi, delta, idx


def gravitating_sphere(n_target: int = 1_000_000, seed: int = SEED_BASE + 2) -> Workload:
    """BASELINE.json configs[2]: R = 10 km sphere at rest, rho(r) = rho0 (1 + 0.1 (1 - r^2/R^2)),
    uniform-sphere gravity supplied as a_ext, T = 200 K."""
    R = 1.0e4
    mat0 = Material()
    xi, delta, idx = _unit_ball_lattice(n_target, seed)
    n = idx.size
    dx = R * delta
    pos = xi * R
    r2 = (xi * xi).sum(axis=1)
    m = mat0.rho0 * (1.0 + 0.1 * (1.0 - r2)) * dx ** 3
    M = m.sum()
    gfac = -G_NEWTON * M / R ** 3
    cols = dict(x=pos[:, 0], y=pos[:, 1], z=pos[:, 2], m=m, h=np.full(n, 1.3 * dx),
                vx=np.zeros(n), vy=np.zeros(n), vz=np.zeros(n), u=np.full(n, mat0.cv * 200.0),
                gx=gfac * pos[:, 0], gy=gfac * pos[:, 1], gz=gfac * pos[:, 2])
    params = Params(flags=FLAG_STRENGTH | FLAG_CORRECTION_TENSOR | FLAG_PCLIP_GLOBAL, materials=[mat0])
    return _finish(f"gravitating_sphere_{n}", params, cols, np.zeros(n, np.int32), np.zeros(n, np.uint8), 0.0,
                   "BASELINE.json configs[2]; a_ext = uniform-sphere field; PCLIP_GLOBAL")


def _stretched_body(n_target, R, contrast, eta_h, rho0, seed, first_index):
    """Lattice ball with a smooth radial stretch r = R (xi + b xi^3)/(1+b): number density
    falls by ``contrast`` from centre to surface; m = rho0 / n(x) keeps mass density ~ rho0;
    h = eta_h * n^(-1/3)."""
    # solve (1+b)^2 (1+3b) = contrast by bisection
    lo, hi = 0.0, 100.0
    for _ in range(200):
        b = 0.5 * (lo + hi)
        if (1 + b) ** 2 * (1 + 3 * b) < contrast:
            lo = b
        else:
            hi = b
    xi, delta, idx = _unit_ball_lattice(n_target, seed, first_index)
    s = np.sqrt((xi * xi).sum(axis=1))
    stretch = R * (1.0 + b * s * s) / (1.0 + b)
    pos = xi * stretch[:, None]
    n0 = 1.0 / delta ** 3                                   # per unit xi-volume
    ndens = n0 * (1 + b) ** 3 / (R ** 3 * (1 + b * s * s) ** 2 * (1 + 3 * b * s * s))
    m = rho0 / ndens
    h = eta_h * ndens ** (-1.0 / 3.0)
    return pos, m, h, idx


def impact_pair(n_total: int = 4_400_000, seed: int = SEED_BASE + 3, contrast: float = 100.0,
                eta_h: float = 1.214, R_target: float = 5.0e4, R_impactor: float = 2.3e4,
                v_impact: float = 3000.0, name: str = "impact_pair") -> Workload:
    """BASELINE.json configs[3] (defaults) and configs[4] (n_total=3.2e7, contrast=1e3, eta_h=1.530).

    Two lattice spheres (materials 0/1), just touching along the line at 45 degrees, relative
    speed ``v_impact`` split in the centre-of-mass frame; h adaptive (eta_h = 1.214 -> ~60
    neighbours, 1.530 -> ~120, with kappa = 2); own-body uniform-sphere gravity as a_ext.
    """
    mats = [Material(), Material(Y0=1.0e6, mu_i=1.0)]
    n_t = int(round(n_total * 10.0 / 11.0)); n_i = n_total - n_t
    pt, mt, ht, it = _stretched_body(n_t, R_target, contrast, eta_h, mats[0].rho0, seed, 0)
    pi_, mi, hi_, ii = _stretched_body(n_i, R_impactor, contrast, eta_h, mats[1].rho0, seed, it.size)
    d = R_target + R_impactor
    ctr_i = np.array([d * math.cos(math.pi / 4), d * math.sin(math.pi / 4), 0.0])
    Mt, Mi = mt.sum(), mi.sum()
    v_t = np.array([v_impact * Mi / (Mt + Mi), 0.0, 0.0])
    v_i = np.array([-v_impact * Mt / (Mt + Mi), 0.0, 0.0])
    gt = -G_NEWTON * Mt / R_target ** 3 * pt
    gi = -G_NEWTON * Mi / R_impactor ** 3 * pi_
    pos = np.concatenate([pt, pi_ + ctr_i[None, :]], axis=0)
    g = np.concatenate([gt, gi], axis=0)
    n = pos.shape[0]
    vel = np.concatenate([np.tile(v_t, (it.size, 1)), np.tile(v_i, (ii.size, 1))], axis=0)
    mat = np.concatenate([np.zeros(it.size, np.int32), np.ones(ii.size, np.int32)])
    cols = dict(x=pos[:, 0], y=pos[:, 1], z=pos[:, 2], m=np.concatenate([mt, mi]),
                h=np.concatenate([ht, hi_]), vx=vel[:, 0], vy=vel[:, 1], vz=vel[:, 2],
                u=np.full(n, mats[0].cv * 200.0), gx=g[:, 0], gy=g[:, 1], gz=g[:, 2])
    params = Params(flags=FLAG_STRENGTH | FLAG_CORRECTION_TENSOR | FLAG_PCLIP_GLOBAL, materials=mats)
    return _finish(f"{name}_{n}", params, cols, mat, np.zeros(n, np.uint8), 0.0,
                   f"number-density contrast {contrast:g}, eta_h {eta_h}; PCLIP_GLOBAL")


def synthetic_eos_table(mat: Material, kind: str = "curved", n_rho: int = 97, n_u: int = 33,
                        n_melt: int = 49) -> EosTable:
    """A synthetic table standing in for the paper's M-ANEOS quartz tables and SiO2 melt curve
    (PAPER.md:221, 258), which are not available.  kind = "linear": the analytic stand-in of
    BASELINE.json configs[0] sampled on the grid (P = c0^2 (rho - rho0), T = u / cv, c = c0, constant
    T_melt) -- a bilinear lookup reproduces it; kind = "curved": a Tillotson-like smooth surface with
    a density-dependent melt curve (coefficients arbitrary, fixed)."""
    rho = np.linspace(0.1 * mat.rho0, 1.3 * mat.rho0, n_rho)      # free-surface particles sit near rho0 / 4
    u = np.linspace(0.0, 2.5e6, n_u)
    R, U = np.meshgrid(rho, u, indexing="ij")
    mu = R / mat.rho0 - 1.0
    if kind == "linear":
        P = mat.c0 ** 2 * (R - mat.rho0)
        T = U / mat.cv
        cs = np.full_like(R, mat.c0)
        tm = None
    else:
        P = mat.c0 ** 2 * mat.rho0 * (mu + 1.5 * mu * mu) + 0.5 * R * U * (1.0 + mu)
        T = U / mat.cv * (1.0 + 0.3 * mu) + 40.0 * mu
        cs = mat.c0 * np.sqrt(np.maximum(0.25, 1.0 + 1.5 * mu + 0.5 * U / mat.c0 ** 2))
        rm = np.linspace(rho[0], rho[-1], n_melt)
        tm = _f32(mat.Tmelt * np.maximum(0.2, 1.0 + 2.0 * (rm / mat.rho0 - 1.0)) ** 1.5)
    return EosTable(float(rho[0]), float(rho[-1]), float(u[0]), float(u[-1]), _f32(P), _f32(T), _f32(cs), tm)


def oblique_impact(n_total: int = 30_000, v_impact: float = 100.0, seed: int = SEED_BASE + 7) -> Workload:
    """Stand-in for the paper's angular-momentum experiment (Fig. 7: oblique impact at
    100 m/s and 45 degrees): two uniform lattice spheres (R = 50 km and 23 km, materials 0/1), just
    touching, no external acceleration (self-gravity is not built here), h = 1.3 dx."""
    wl = impact_pair(n_total, seed, 1.0, 1.3, v_impact=v_impact, name="oblique_impact")
    for k in ("gx", "gy", "gz"):
        wl.arrays[k][:] = 0.0
    wl.notes = "uniform bodies, a_ext = 0, v = %g m/s at 45 degrees; PCLIP_GLOBAL" % v_impact
    return wl


# list reuse of the CUDA path per config (skin as a fraction of H, steps between full builds): measured choices,
# DESIGN.md section 7; they change how often the neighbour lists are rebuilt, never a result
LIST_REUSE = {1: (0.05, 16), 2: (0.05, 16), 3: (0.04, 16), 4: (0.025, 32)}


def config(k: int, scale: float = 1.0) -> Workload:
    """BASELINE.json configs[k]; ``scale`` < 1 shrinks particle counts (parity-sized cases)."""
    if k == 0:
        return elastic_block(16 if scale >= 1.0 else max(4, int(round(16 * scale))))
    if k == 1:
        wl = granular_column(scale)
    elif k == 2:
        wl = gravitating_sphere(int(1_000_000 * scale ** 3) if scale < 1.0 else 1_000_000)
    elif k == 3:
        wl = impact_pair(int(4_400_000 * (scale ** 3 if scale < 1.0 else 1.0)), SEED_BASE + 3, 100.0, 1.214,
                         name="impact_pair_c3")
    elif k == 4:
        wl = impact_pair(int(32_000_000 * (scale ** 3 if scale < 1.0 else 1.0)), SEED_BASE + 4, 1000.0, 1.530,
                         name="impact_pair_c4")
        wl.params.list_budget = 96        # ~120 neighbours: room for 384 list entries per particle (default 256)
    else:
        raise ValueError(f"no config {k}")
    wl.params.skin, wl.params.rebuild_every = LIST_REUSE[k]
    return wl
