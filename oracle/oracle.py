"""CPU oracle for one SPH + shear-strength step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64: the pair passes call oracle/sph_oracle.c (straight loops over brute-force or
cell-list neighbour sets); every per-particle step is written here in numpy, in the paper's
order and notation, each function citing the passage of /root/reference/PAPER.md it follows
(line numbers as PAPER.md:<line>; "reading Qn" = DESIGN.md section 3 / SURVEY.md section 8c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares no code with paper_2603_19764_b200/csrc or binding.py and
imports neither; parameter records are duck-typed (attributes kappa, alpha, ..., materials).

Parity-unpinned choices (no authority in PAPER.md; listed in DESIGN.md): the kernel's
functional form and kappa (Q3), AV constants (Q6), the analytic EOS stand-in (Q13), the
singular-C fallback rule (Q9), the fixed-particle rule (Q16), the target mass and the
safeguards of the smoothing-length iteration (Q20).  Everything else is pinned by
tests/test_oracle_*.py.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np

from . import build as _build

FLAG_STRENGTH = 1
FLAG_CORRECTION_TENSOR = 2
FLAG_PCLIP_GLOBAL = 4
FLAG_JAUMANN_AS_PRINTED = 512

GATHER, SYMMETRIC = 0, 1
CTOL = 1.0e-4          # reading Q9: C = I unless |det C^-1| > CTOL * ||C^-1||_F^3

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lp = C.POINTER(C.c_longlong)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        for name in ("orc_W", "orc_dWdr", "orc_dWdh"):
            f = getattr(_lib, name)
            f.restype = C.c_double
            f.argtypes = [C.c_double, C.c_double, C.c_double]
        _lib.orc_max_threads.restype = C.c_int
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---------------------------------------------------------------------------
# kernel (reading Q3) -- scalar entry points for the pin tests
# ---------------------------------------------------------------------------
def W(r, h, kappa=2.0):
    return lib().orc_W(float(r), float(h), float(kappa))


def dWdr(r, h, kappa=2.0):
    return lib().orc_dWdr(float(r), float(h), float(kappa))


def dWdh(r, h, kappa=2.0):
    return lib().orc_dWdh(float(r), float(h), float(kappa))


# ---------------------------------------------------------------------------
# Pass O1 -- neighbour sets
# ---------------------------------------------------------------------------
def neighbors(x, y, z, h, kappa, which, mode="brute"):
    """CSR neighbour lists (counts, offsets[n+1], list), ascending j, fp32 predicate (reading Q4).

    which = GATHER: {j : r2 < H_i^2} (contains i);
    which = SYMMETRIC: {j != i : r2 < max(H_i^2, H_j^2)}.
    """
    x, y, z, h = map(_f64, (x, y, z, h))
    n = x.shape[0]
    fn = lib().orc_neighbors_brute if mode == "brute" else lib().orc_neighbors_grid
    counts = np.zeros(n, dtype=np.int32)
    fn(C.c_longlong(n), _d(x), _d(y), _d(z), _d(h), C.c_double(kappa), C.c_int(which),
       counts.ctypes.data_as(_ip), None, None)
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    lst = np.zeros(max(int(offsets[-1]), 1), dtype=np.int32)
    fn(C.c_longlong(n), _d(x), _d(y), _d(z), _d(h), C.c_double(kappa), C.c_int(which),
       counts.ctypes.data_as(_ip), offsets.ctypes.data_as(_lp), lst.ctypes.data_as(_ip))
    return counts, offsets, lst


# ---------------------------------------------------------------------------
# Pass O2 -- density, Omega (PAPER.md:57 Eq. 1, :66 Eq. 3)
# ---------------------------------------------------------------------------
def density(x, y, z, m, h, kappa, offsets, lst):
    x, y, z, m, h = map(_f64, (x, y, z, m, h))
    n = x.shape[0]
    rho = np.zeros(n); omega = np.zeros(n)
    lib().orc_density(C.c_longlong(n), _d(x), _d(y), _d(z), _d(m), _d(h), C.c_double(kappa),
                      offsets.ctypes.data_as(_lp), lst.ctypes.data_as(_ip), _d(rho), _d(omega))
    return rho, omega


# ---------------------------------------------------------------------------
# NEXT-1 -- adaptive smoothing length (Eq. 2)
# ---------------------------------------------------------------------------
H_OMEGA_FLOOR = 0.1        # reading Q20: the Newton slope uses max(Omega, 0.1)
H_STEP_LIMITS = (0.8, 1.25)  # reading Q20: h changes by at most this factor per iteration


def kernel_mass(rho, h, kappa):
    """M_tot = (4/3) pi R_kernel(h)^3 rho with R_kernel = kappa h (Eq. 2)."""
    return 4.0 / 3.0 * np.pi * (kappa * h) ** 3 * rho


def adapt_h(x, y, z, m, h, kappa, n_target, iterations, mode="brute"):
    """Newton-Raphson iterations on h_i towards a constant effective kernel mass:
    solve f(h_i) = M_tot^i(h_i) - n_target m_i = 0, M_tot of Eq. 2 with rho_i(h_i) of Eq. 1.
    "The density and its derivative with respect to h_i are computed and used": with Eq. 3,
    d(h^3 rho)/dh = 3 h^2 rho + h^3 drho/dh = 3 h^2 rho Omega, hence
        h <- h [1 - (1 - n_target m / M_tot) / (3 Omega)].
    Readings (Q20, ours: the paper gives neither the target mass nor safeguards): the target is
    n_target particle masses; the slope uses max(Omega, H_OMEGA_FLOOR); the factor is limited to
    H_STEP_LIMITS; h is stored in fp32 between iterations (the neighbour predicate is defined on
    fp32 h, reading Q4).  Returns (h [fp32 values as fp64], rho, Omega of the last density pass
    -- taken at the h BEFORE the last update --, history of max |factor - 1|)."""
    x, y, z, m = map(_f64, (x, y, z, m))
    h = _f64(np.asarray(h, dtype=np.float32))
    hist = []
    rho = omega = None
    for _ in range(iterations):
        _, off, lst = neighbors(x, y, z, h, kappa, GATHER, mode)
        rho, omega = density(x, y, z, m, h, kappa, off, lst)
        ratio = n_target * m / kernel_mass(rho, h, kappa)
        fac = 1.0 - (1.0 - ratio) / (3.0 * np.maximum(omega, H_OMEGA_FLOOR))
        fac = np.clip(fac, H_STEP_LIMITS[0], H_STEP_LIMITS[1])
        hist.append(float(np.abs(fac - 1.0).max()))
        h = _f64((h * fac).astype(np.float32))
    return h, rho, omega, hist


# ---------------------------------------------------------------------------
# Pass O3 -- EOS, shear modulus, yield strength, plastic projection (per particle)
# ---------------------------------------------------------------------------
def _matcol(params, mat, name):
    return np.array([getattr(mm, name) for mm in params.materials], dtype=np.float64)[mat]


def table_lookup(f, x_min, x_max, x, y_min=None, y_max=None, y=None):
    """Piecewise-linear (1-D) or bilinear (2-D) interpolation on a uniform grid, clamped to the grid's
    edges (reading Q21: the paper says "tabulated", not how it interpolates).
    f[i] sits at x_min + i (x_max - x_min)/(n_x - 1); f[i, j] likewise in y."""
    f = np.asarray(f, dtype=np.float64)
    nx = f.shape[0]
    fx = np.clip((x - x_min) / (x_max - x_min) * (nx - 1), 0.0, nx - 1.0)
    i = np.minimum(np.floor(fx).astype(np.int64), nx - 2)
    tx = fx - i
    if f.ndim == 1:
        return (1.0 - tx) * f[i] + tx * f[i + 1]
    ny = f.shape[1]
    fy = np.clip((y - y_min) / (y_max - y_min) * (ny - 1), 0.0, ny - 1.0)
    j = np.minimum(np.floor(fy).astype(np.int64), ny - 2)
    ty = fy - j
    return ((1.0 - tx) * (1.0 - ty) * f[i, j] + tx * (1.0 - ty) * f[i + 1, j]
            + (1.0 - tx) * ty * f[i, j + 1] + tx * ty * f[i + 1, j + 1])


def eos(params, rho, u, mat):
    """P, c, T from (rho, u).  Materials without a table: the analytic stand-in for
    EOSlib (reading Q13, BASELINE.json configs[0]): P = c0^2 (rho - rho0), c = c0, T = u / cv.
    Materials with a table (NEXT-3): bilinear lookups (table_lookup).  PCLIP_GLOBAL clips P >= 0
    everywhere (Q8)."""
    rho0 = _matcol(params, mat, "rho0"); c0 = _matcol(params, mat, "c0"); cv = _matcol(params, mat, "cv")
    P = c0 * c0 * (rho - rho0)
    cs = c0.copy()
    T = u / cv
    for k, mm in enumerate(params.materials):
        tab = getattr(mm, "table", None)
        if tab is None:
            continue
        sel = mat == k
        a = (tab.rho_min, tab.rho_max, rho[sel], tab.u_min, tab.u_max, u[sel])
        P[sel] = table_lookup(tab.P, *a)
        T[sel] = table_lookup(tab.T, *a)
        cs[sel] = table_lookup(tab.cs, *a)
    if params.flags & FLAG_PCLIP_GLOBAL:
        P = np.maximum(P, 0.0)
    return P, cs, T


def melt_temperature(params, rho, mat):
    """T_melt: the material's constant, or "a tabulated function of density"."""
    Tm = _matcol(params, mat, "Tmelt").copy()
    for k, mm in enumerate(params.materials):
        tab = getattr(mm, "table", None)
        if tab is not None and tab.Tmelt is not None:
            sel = mat == k
            Tm[sel] = table_lookup(tab.Tmelt, tab.rho_min, tab.rho_max, rho[sel])
    return Tm


def shear_modulus(params, rho, cs, mat):
    """Gamma = 3(1-2nu)/(2(1+nu)) K, K = rho c_s^2 (Eq. 30), or the runtime
    constant per material when one is given."""
    Gc = _matcol(params, mat, "Gamma"); nu = _matcol(params, mat, "nu")
    G30 = 3.0 * (1.0 - 2.0 * nu) / (2.0 * (1.0 + nu)) * rho * cs * cs
    return np.where(Gc > 0.0, Gc, G30)


def yield_strength(params, P, T, mat, rho=None):
    """Y_i = Y0 + mu_i P/(1 + mu_i P/(Ym - Y0)) (Eq. 34) with P < 0 clipped to 0
    (PAPER.md:202); Y_d = mu_d P (Eq. 35); Y = min(Y_i, Y_d) when mu_d is finite (Eq. 36,
    reading Q10); Y -> Y tanh(xi (T_melt/T - 1)) (Eq. 37), clamped to >= 0 above
    the melting point and equal to Y for T <= 0 (reading Q11)."""
    Y0 = _matcol(params, mat, "Y0"); Ym = _matcol(params, mat, "Ym")
    mu_i = _matcol(params, mat, "mu_i"); mu_d = _matcol(params, mat, "mu_d")
    xi = _matcol(params, mat, "xi")
    Tm = _matcol(params, mat, "Tmelt") if rho is None else melt_temperature(params, rho, mat)
    Pp = np.maximum(P, 0.0)
    span = Ym - Y0
    with np.errstate(divide="ignore", invalid="ignore"):
        Yi = np.where(span > 0.0, Y0 + mu_i * Pp / (1.0 + mu_i * Pp / np.where(span > 0.0, span, 1.0)), Y0)
        Y = np.where(np.isfinite(mu_d), np.minimum(Yi, np.where(np.isfinite(mu_d), mu_d, 0.0) * Pp), Yi)
        soft = np.where(T > 0.0, np.maximum(0.0, np.tanh(xi * (Tm / np.where(T > 0.0, T, 1.0) - 1.0))), 1.0)
    return Y * soft


def J2(S):
    """J2 = 1/2 S:S (Eq. 33) from the five stored components, S_zz = -S_xx - S_yy."""
    sxx, syy, sxy, sxz, syz = S
    szz = -sxx - syy
    return 0.5 * (sxx * sxx + syy * syy + szz * szz) + sxy * sxy + sxz * sxz + syz * syz


def project(S, Y):
    """S -> f S, f = min(Y / sqrt(J2), 1) (Eq. 31-32); f = 1 if J2 = 0 (Q12)."""
    sj = np.sqrt(J2(S))
    with np.errstate(divide="ignore", invalid="ignore"):
        f = np.where(sj > Y, Y / np.where(sj > 0.0, sj, 1.0), 1.0)
    return S * f[None, :], f


# ---------------------------------------------------------------------------
# Pass O4 -- velocity gradient (Eq. 20-24)
# ---------------------------------------------------------------------------
def gradients(x, y, z, m, h, vx, vy, vz, rho, omega, kappa, offsets, lst):
    """F (Eq. 20) and C^-1 (Eq. 21) as [9][n], component 3*alpha + beta."""
    args = list(map(_f64, (x, y, z, m, h, vx, vy, vz, rho, omega)))
    n = args[0].shape[0]
    F = np.zeros((9, n)); Cinv = np.zeros((9, n))
    lib().orc_gradients(C.c_longlong(n), *[_d(a) for a in args], C.c_double(kappa),
                        offsets.ctypes.data_as(_lp), lst.ctypes.data_as(_ip), _d(F), _d(Cinv))
    return F, Cinv


def correct_gradient(F, Cinv, flags):
    """G = F . C (Eq. 22).  C = (C^-1)^-1 by a 3x3 inverse; C = 1 when the correction
    tensor is switched off or C^-1 is singular (reading Q9).  Returns G [9][n] and
    the per-particle fallback flag."""
    n = F.shape[1]
    Fm = F.T.reshape(n, 3, 3)
    Cm = Cinv.T.reshape(n, 3, 3)
    det = np.linalg.det(Cm)
    fro = np.sqrt((Cm * Cm).sum(axis=(1, 2)))
    ok = np.abs(det) > CTOL * fro ** 3
    if not (flags & FLAG_CORRECTION_TENSOR):
        ok[:] = False
    Cfull = np.tile(np.eye(3), (n, 1, 1))
    if ok.any():
        Cfull[ok] = np.linalg.inv(Cm[ok])
    G = np.einsum("nag,ngb->nab", Fm, Cfull)
    return np.ascontiguousarray(G.reshape(n, 9).T), (~ok).astype(np.int32)


def strain_and_rotation(G):
    """eps_dot = (G + G^T)/2 (Eq. 24), R = (G - G^T)/2 (Eq. 23)."""
    n = G.shape[1]
    Gm = G.T.reshape(n, 3, 3)
    GT = np.transpose(Gm, (0, 2, 1))
    return 0.5 * (Gm + GT), 0.5 * (Gm - GT)


def _S3(S):
    sxx, syy, sxy, sxz, syz = S
    szz = -sxx - syy
    return np.stack([np.stack([sxx, sxy, sxz], axis=1),
                     np.stack([sxy, syy, syz], axis=1),
                     np.stack([sxz, syz, szz], axis=1)], axis=1)


def stress_rate(G, S, Gamma, flags):
    """dS/dt = 2 Gamma (eps_dot - tr(eps_dot)/3 delta) + rotation terms (Eq. 13).
    Reading Q1: the paper "adopt[s] the Jaumann rate to obtain an objective stress rate"
     after Benz & Asphaug, whose rotation terms are S^{ag} R^{bg} + S^{gb} R^{ag}
    = R.S - S.R with R of Eq. 15: the rate that turns S with the body.  The index order AS PRINTED,
    S^{ag} R^{gb} + S^{bg} R^{ga} = S.R + (S.R)^T = S.R - R.S, is the negative of that and is not
    objective, so the text is at odds with itself; the default follows the words ("objective"),
    JAUMANN_AS_PRINTED follows the indices.  Evaluated as a full 3x3; returns the five stored
    components [5][n], the full tensor and 1/2 eps_dot:eps_dot (Eq. 43)."""
    eps, R = strain_and_rotation(G)
    S3 = _S3(S)
    tr = np.trace(eps, axis1=1, axis2=2)
    elastic = 2.0 * Gamma[:, None, None] * (eps - tr[:, None, None] / 3.0 * np.eye(3)[None])
    SR = np.einsum("nag,ngb->nab", S3, R)
    sgn = 1.0 if (flags & FLAG_JAUMANN_AS_PRINTED) else -1.0
    dS3 = elastic + sgn * (SR + np.transpose(SR, (0, 2, 1)))
    dS = np.stack([dS3[:, 0, 0], dS3[:, 1, 1], dS3[:, 0, 1], dS3[:, 0, 2], dS3[:, 1, 2]], axis=0)
    eps2 = 0.5 * (eps * eps).sum(axis=(1, 2))
    return np.ascontiguousarray(dS), dS3, eps2


def stress_rate_components(G, S, Gamma, flags):
    """The component form Eq. 25-29 (garbled in the extraction, reconstructed from
    Eq. 13 in SURVEY.md Appendix A / DESIGN.md reading Q2).  Used by the tests as a cross-check
    of stress_rate(); G component index 3*alpha + beta."""
    Gxx, Gxy, Gxz, Gyx, Gyy, Gyz, Gzx, Gzy, Gzz = G
    Sxx, Syy, Sxy, Sxz, Syz = S
    s = 1.0 if (flags & FLAG_JAUMANN_AS_PRINTED) else -1.0
    dSxx = s * (Sxy * (Gyx - Gxy) + Sxz * (Gzx - Gxz)) - (2.0 / 3.0) * Gamma * (Gyy + Gzz - 2.0 * Gxx)
    dSyy = s * (Sxy * (Gxy - Gyx) + Syz * (Gzy - Gyz)) - (2.0 / 3.0) * Gamma * (Gxx + Gzz - 2.0 * Gyy)
    dSxy = Gamma * (Gxy + Gyx) + s * 0.5 * (Sxx * (Gxy - Gyx) + Syy * (Gyx - Gxy)
                                            + Syz * (Gzx - Gxz) + Sxz * (Gzy - Gyz))
    dSxz = Gamma * (Gxz + Gzx) + s * 0.5 * ((Sxx + Syy) * (Gxz - Gzx) + Sxx * (Gxz - Gzx)
                                            + Sxy * (Gyz - Gzy) + Syz * (Gyx - Gxy))
    dSyz = Gamma * (Gyz + Gzy) + s * 0.5 * ((Sxx + Syy) * (Gyz - Gzy) + Syy * (Gyz - Gzy)
                                            + Sxz * (Gxy - Gyx) + Sxy * (Gxz - Gzx))
    return np.stack([dSxx, dSyy, dSxy, dSxz, dSyz], axis=0)


# ---------------------------------------------------------------------------
# Pass O5 -- forces (PAPER.md:71 Eq. 4, :76-93 Eq. 5-8, :140-144 Eq. 18-19)
# ---------------------------------------------------------------------------
def forces(params, x, y, z, m, h, vx, vy, vz, rho, omega, P, cs, S, g, offsets, lst):
    args = list(map(_f64, (x, y, z, m, h, vx, vy, vz, rho, omega, P, cs)))
    n = args[0].shape[0]
    S = _f64(S)
    strength = 1 if (params.flags & FLAG_STRENGTH) else 0
    a = np.zeros((3, n)); dudt = np.zeros(n); mumax = np.zeros(n)
    if g is None:
        gp = [None, None, None]
    else:
        g = _f64(g)
        gp = [_d(g[0]), _d(g[1]), _d(g[2])]
    lib().orc_forces(C.c_longlong(n), *[_d(q) for q in args], _d(S), C.c_int(strength),
                     gp[0], gp[1], gp[2],
                     C.c_double(params.kappa), C.c_double(params.alpha), C.c_double(params.beta),
                     C.c_double(params.eps_av),
                     offsets.ctypes.data_as(_lp), lst.ctypes.data_as(_ip), _d(a), _d(dudt), _d(mumax))
    return a, dudt, mumax


def timestep(params, h, cs, mumax, a=None):
    """dt_i,CFL = eta_C h_i / ((1 + 0.6 alpha) c_i + 0.6 beta max_j |min(0, mu_ij)|)
    (Eq. 39); when eta_a > 0 also dt_i,a = eta_a sqrt(epsilon/|a_i|) (PAPER.md:227,
    Eq. 38) with epsilon = h_i (reading Q22: PAPER.md:234 offers "the gravitational softening length
    or SPH kernel size"; gravity is not built here, so the SPH length it is) and a_i the full
    acceleration of Eq. 18 including a_ext; "the minimum of these criteria".
    |a_i| = 0 leaves Eq. 39 alone."""
    dt = params.eta_C * h / ((1.0 + 0.6 * params.alpha) * cs + 0.6 * params.beta * mumax)
    if params.eta_a > 0.0 and a is not None:
        an = np.sqrt((a * a).sum(axis=0))
        dt_a = np.where(an > 0.0, params.eta_a * np.sqrt(h / np.where(an > 0.0, an, 1.0)), np.inf)
        dt = np.minimum(dt, dt_a)
    return dt


# ---------------------------------------------------------------------------
# O1..O6 for one set of predicted values
# ---------------------------------------------------------------------------
def derivatives(params, x, y, z, m, h, vx, vy, vz, u, S, mat, g=None, mode="brute") -> Dict[str, np.ndarray]:
    """Everything the step needs at one time level, from PREDICTED v, u, S (PAPER.md:240,
    reading Q14): neighbour sets -> rho, Omega -> P, c, T, Gamma, Y -> S_pred rescaled (Eq. 31)
    -> F, C^-1, G -> a, du/dt, mu_max -> dS/dt, 1/2 eps:eps, dt_i."""
    kap = params.kappa
    out: Dict[str, np.ndarray] = {}
    cg, og, lg = neighbors(x, y, z, h, kap, GATHER, mode)
    cs_, os_, ls_ = neighbors(x, y, z, h, kap, SYMMETRIC, mode)
    out["n_gather"], out["n_symmetric"] = cg, cs_
    rho, omega = density(x, y, z, m, h, kap, og, lg)
    P, cs, T = eos(params, rho, _f64(u), mat)
    Gamma = shear_modulus(params, rho, cs, mat)
    Y = yield_strength(params, P, T, mat, rho)
    strength = bool(params.flags & FLAG_STRENGTH)
    S = _f64(S)
    if strength:
        Sp, f = project(S, Y)
    else:
        Sp, f = np.zeros_like(S), np.ones_like(rho)
    out.update(rho=rho, omega=omega, P=P, cs=cs, T=T, Gamma=Gamma, Y=Y, S_pred=Sp, f_pred=f)
    a, dudt, mumax = forces(params, x, y, z, m, h, vx, vy, vz, rho, omega, P, cs, Sp, g, os_, ls_)
    out.update(a=a, dudt=dudt, mumax=mumax)
    if strength:
        F, Cinv = gradients(x, y, z, m, h, vx, vy, vz, rho, omega, kap, os_, ls_)
        G, cflag = correct_gradient(F, Cinv, params.flags)
        dS, _, eps2 = stress_rate(G, Sp, Gamma, params.flags)
    else:
        n = rho.shape[0]
        F = np.zeros((9, n)); Cinv = np.zeros((9, n)); G = np.zeros((9, n))
        cflag = np.zeros(n, np.int32); dS = np.zeros((5, n)); eps2 = np.zeros(n)
    out.update(F=F, Cinv=Cinv, G=G, cflag=cflag, dS=dS, eps2=eps2)
    out["dt_i"] = timestep(params, _f64(h), cs, mumax, a)
    return out


def single_pass(wl, dt: Optional[float] = None, mode="brute") -> Dict[str, np.ndarray]:
    """BASELINE.json configs[0]: one density + gradient + force + strength-update pass, i.e.
    steps 4-7 of the step sequence with S_half = S_pred = S_in, v_pred = v_in, u_pred = u_in
    (SURVEY.md Appendix B).  Adds the closed S, v, u (Eq. 41 + rescale)."""
    A = {k: _f64(v) for k, v in wl.arrays.items()}
    dt = wl.dt if dt is None else dt
    S = np.stack([A["Sxx"], A["Syy"], A["Sxy"], A["Sxz"], A["Syz"]], axis=0)
    g = np.stack([A["gx"], A["gy"], A["gz"]], axis=0)
    d = derivatives(wl.params, A["x"], A["y"], A["z"], A["m"], A["h"], A["vx"], A["vy"], A["vz"],
                    A["u"], S, wl.mat, g, mode)
    free = (wl.fixed == 0)
    v = np.stack([A["vx"], A["vy"], A["vz"]], axis=0)
    d["v_close"] = v + 0.5 * dt * d["a"] * free[None, :]
    d["u_close"] = A["u"] + 0.5 * dt * d["dudt"]
    if wl.params.flags & FLAG_STRENGTH:
        Sc = S + 0.5 * dt * d["dS"]
        d["S_close"], d["f_close"] = project(Sc, d["Y"])
    else:
        d["S_close"], d["f_close"] = np.zeros_like(S), np.ones(S.shape[1])
    return d


# ---------------------------------------------------------------------------
# the full step (Eq. 40-42)
# ---------------------------------------------------------------------------
class Stepper:
    """Global-dt kick-drift-kick with predictor-corrector for u and S (reading Q17).

    store_fp32: BASELINE.json's north_star fixes the STORAGE of the particle state as fp32.  With this
    switch every quantity that is kept between two passes of a step (x after the drift; v, u, S at the
    half step, predicted and at the full step; the carried derivatives a, du/dt, dS/dt; e_acc) is rounded
    to fp32 once, where it would be stored; all arithmetic stays fp64.  The default carries fp64 state."""

    def __init__(self, wl, mode="grid", store_fp32=False):
        A = {k: _f64(v) for k, v in wl.arrays.items()}
        self.params = wl.params
        self.mode = mode
        self.x = np.stack([A["x"], A["y"], A["z"]], axis=0)
        self.v = np.stack([A["vx"], A["vy"], A["vz"]], axis=0)
        self.u = A["u"].copy()
        self.S = np.stack([A["Sxx"], A["Syy"], A["Sxy"], A["Sxz"], A["Syz"]], axis=0)
        self.m, self.h = A["m"], A["h"]
        self.g = np.stack([A["gx"], A["gy"], A["gz"]], axis=0)
        self.mat = wl.mat
        self.store_fp32 = bool(store_fp32)
        self.free = (wl.fixed == 0).astype(np.float64)
        self.e_acc = np.zeros_like(self.u)
        self.d = None              # derivatives at the current full step
        self.dt_next = None
        self.strength = bool(wl.params.flags & FLAG_STRENGTH)

    def _st(self, a):
        """what the stored copy of ``a`` holds"""
        return a.astype(np.float32).astype(np.float64) if self.store_fp32 else a

    def _derivs(self, v, u, S):
        d = derivatives(self.params, self.x[0], self.x[1], self.x[2], self.m, self.h,
                        v[0], v[1], v[2], u, S, self.mat, self.g, self.mode)
        if self.store_fp32:
            for k in ("a", "dudt", "dS", "Y", "S_pred", "eps2"):
                d[k] = self._st(d[k])
        return d

    def bootstrap(self):
        """First step: a_0, du_0, dS_0 from the current state (pred = current, dt = 0)."""
        self.d = self._derivs(self.v, self.u, self.S)
        self.dt_next = float(self.d["dt_i"].min())

    def step(self, dt: float = 0.0) -> float:
        if self.d is None:
            self.bootstrap()
        if dt <= 0.0:
            dt = self.dt_next
        a, dudt, dS = self.d["a"], self.d["dudt"], self.d["dS"]
        fr = self.free[None, :]
        # 1. opening kick (Eq. 42); fixed particles keep x, v (reading Q16)
        st = self._st
        v_half = st(self.v + 0.5 * dt * a * fr)
        u_half = st(self.u + 0.5 * dt * dudt)
        S_half = st(self.S + 0.5 * dt * dS)
        # 2. drift
        self.x = st(self.x + dt * v_half * fr)
        # 3. prediction from the derivatives of the previous step (Eq. 40)
        v_pred = st(v_half + 0.5 * dt * a * fr)
        u_pred = st(u_half + 0.5 * dt * dudt)
        S_pred = st(S_half + 0.5 * dt * dS)
        # 4-6. new derivatives from the predicted (and rescaled, Eq. 31) values
        d = self._derivs(v_pred, u_pred, S_pred)
        # 7. closing kick (Eq. 41) and rescale again
        self.v = st(v_half + 0.5 * dt * d["a"] * fr)
        self.u = st(u_half + 0.5 * dt * d["dudt"])
        if self.strength:
            self.S = st(project(S_half + 0.5 * dt * d["dS"], d["Y"])[0])
        # 8. carried derivatives, accumulated strain-rate invariant (Eq. 43)
        self.e_acc = st(self.e_acc + dt * d["eps2"])
        self.d = d
        self.dt_next = float(d["dt_i"].min())
        return dt


# ---------------------------------------------------------------------------
# NEXT-4: individual (hierarchical) time steps on power-of-two rungs ("the hierarchical individual
# timestep scheme described in Paper I"; "8 substeps").  Paper I is not available: reading Q23.
# ---------------------------------------------------------------------------
def rung_for(dt_i, dT, max_rung):
    """Smallest rung r in [0, max_rung] with dT / 2^r <= dt_i (rung 0 takes the whole big step dT; a particle
    whose limit is below dT / 2^max_rung sits on max_rung: the caller chose dT too large for it)."""
    with np.errstate(divide="ignore"):
        r = np.ceil(np.log2(dT / dt_i))
    r = np.where(np.isnan(r), 0.0, r)                     # dt_i = 0 -> +inf -> max_rung; dt_i = inf -> -inf -> 0
    return np.clip(r, 0, max_rung).astype(np.int64)


def next_rung(wanted, current, n_done, max_rung):
    """Rung of a particle that has just finished a step at the end of substep n_done - 1 (n_done substeps of the
    big step are done).  It may always move to a FINER rung; to a coarser one only as far as that rung's step
    boundaries line up with the present time: rung r has steps of 2^(max_rung - r) substeps, so it may start at
    n_done only if n_done is a multiple of that."""
    out = np.maximum(wanted, 0).copy()
    for r in range(max_rung + 1):                         # coarsest admissible rung at this time
        ok = (n_done % (1 << (max_rung - r))) == 0
        if ok:
            coarsest = r
            break
    out = np.maximum(out, coarsest)
    return np.minimum(out, max_rung)


class RungStepper(Stepper):
    """Kick-drift-kick on block time steps (reading Q23).  One BIG step dT = 2^R substeps of delta = dT / 2^R.
    A particle on rung r takes steps of dt_r = dT / 2^r.  In every substep
      * particles that START a step get the opening kick with their own dt_r (Eq. 42),
      * EVERY particle drifts by delta with its half-step velocity,
      * the values of every particle are PREDICTED to the new time from its last derivatives
        (Eq. 40 generalised: q_pred = q_half + (t - t_mid) dq/dt, t_mid the middle of the particle's step),
      * the derivatives are evaluated from the predicted values; particles that END a step here (the ACTIVE ones)
        take them, get the closing kick with their own dt_r (Eq. 41) and the rescale, and choose their next rung
        from their new limit (Eq. 38-39); the others keep their old derivatives and only lend their predicted
        values to their active neighbours.
    rho, P, Y, ... of every particle are evaluated at the current positions in every substep (they depend on
    positions and predicted u only; nothing is extrapolated).  With every particle on rung 0 and R = 0 this is
    Stepper.step(dT), operation for operation."""

    def __init__(self, wl, mode="grid", store_fp32=False):
        super().__init__(wl, mode, store_fp32)
        self.rung = None
        self.kicks = None           # closing kicks each particle received in the last big step
        self.trace = []             # per substep: predicted S handed to the derivative evaluation (pins)

    def big_step(self, dT, max_rung, rungs=None):
        if self.d is None:
            self.bootstrap()
        R = int(max_rung)
        nsubs = 1 << R
        delta = dT / nsubs
        n = self.u.shape[0]
        fr = self.free[None, :]
        st = self._st
        self.rung = rung_for(self.d["dt_i"], dT, R) if rungs is None else np.asarray(rungs, dtype=np.int64).copy()
        self.kicks = np.zeros(n, dtype=np.int64)
        self.trace = []
        a, dudt, dS = self.d["a"].copy(), self.d["dudt"].copy(), self.d["dS"].copy()
        dt_i = self.d["dt_i"].copy()
        v_half = self.v.copy(); u_half = self.u.copy(); S_half = self.S.copy()
        last = None
        for k in range(nsubs):
            per = 1 << (R - self.rung)                      # substeps per step of each particle's rung
            dtr = dT / (1 << self.rung)                     # its step
            start = (k % per) == 0
            # opening kick (Eq. 42) of the particles that start a step now
            v_half = np.where(start[None, :], st(self.v + 0.5 * dtr * a * fr), v_half)
            u_half = np.where(start, st(self.u + 0.5 * dtr * dudt), u_half)
            S_half = np.where(start[None, :], st(self.S + 0.5 * dtr * dS), S_half)
            # drift of every particle
            self.x = st(self.x + delta * v_half * fr)
            # prediction to the new time from each particle's own last derivatives (Eq. 40 generalised)
            tau = ((k % per) + 1) * delta - 0.5 * dtr         # t_new - t_mid
            v_pred = st(v_half + tau * a * fr)
            u_pred = st(u_half + tau * dudt)
            S_pred = st(S_half + tau * dS)
            d = self._derivs(v_pred, u_pred, S_pred)
            act = ((k + 1) % per) == 0
            self.trace.append({"S_pred_in": S_pred.copy(), "active": act.copy(), "rung": self.rung.copy()})
            # closing kick (Eq. 41) and rescale of the active particles, with their own step
            self.v = np.where(act[None, :], st(v_half + 0.5 * dtr * d["a"] * fr), self.v)
            self.u = np.where(act, st(u_half + 0.5 * dtr * d["dudt"]), self.u)
            if self.strength:
                Sc = st(project(S_half + 0.5 * dtr * d["dS"], d["Y"])[0])
                self.S = np.where(act[None, :], Sc, self.S)
            self.e_acc = np.where(act, st(self.e_acc + dtr * d["eps2"]), self.e_acc)
            a = np.where(act[None, :], d["a"], a)
            dudt = np.where(act, d["dudt"], dudt)
            dS = np.where(act[None, :], d["dS"], dS)
            dt_i = np.where(act, d["dt_i"], dt_i)
            self.kicks += act
            if rungs is None:
                nr = next_rung(rung_for(dt_i, dT, R), self.rung, k + 1, R)
                self.rung = np.where(act, nr, self.rung)
            last = d
        # every particle has finished a step at the end of the big step: the state is synchronised
        self.d = dict(last)
        self.d.update(a=a, dudt=dudt, dS=dS, dt_i=dt_i)
        self.dt_next = float(dt_i.min())
        return dT
