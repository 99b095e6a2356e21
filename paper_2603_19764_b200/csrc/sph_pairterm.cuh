// sph_pairterm.cuh -- the arithmetic of one (i, j) pair of the gradient (S4) and force (S5) passes,
// shared by the list-driven kernel (sph_lists.cu) and the tree-walk kernel (sph_pair.cu).
//
// With D(h) = -(dW/dr)/r = K t^3, t = max(0, 1 - r/H), K = 20 SIGMA / H^5 (Wendland C2, reading Q3),
// grad_i W_ij(h) = -D x_ij, and st = sigma/(Omega rho^2) = (-P delta + S)/(Omega rho^2), w = 1/(Omega rho):
//   F^{ab}    = +1/2 sum_j m_j (w_i D_i + w_j D_j) v_ij^a x_ij^b                         (Eq. 20)
//   Cinv^{ab} = +1/2 sum_j m_j (w_i D_i + w_j D_j) x_ij^a x_ij^b                         (Eq. 21)
//   a_i       = - sum_j m_j [ D_i st_i + D_j st_j ] x_ij + sum_j 1/2 m_j Pi_ij (D_i + D_j) x_ij   (Eq. 4, 7, 18)
//   du_i/dt   = + sum_j m_j D_i (st_i x_ij).v_ij - sum_j 1/4 m_j Pi_ij (D_i + D_j) v_ij.x_ij      (Eq. 8, 19)
//   mu_ij     = hbar v_ij.x_ij / (r^2 + eps hbar^2),  Pi_ij = (-alpha cbar mu + beta mu^2)/rhobar  if v_ij.x_ij < 0
// (Eq. 5-6; means are arithmetic).  The accumulators F and C hold TWICE the sums of
// Eq. 20-21; the caller halves them once at the end.
#pragma once

#define SPH_WC2_SIGMA 3.3422538049298023f     // 21 / (2 pi)
#define SPH_WC2_K20 66.845076098596046f       // 20 * 21 / (2 pi)

// x / y and 1 / y by one MUFU.RCP and no range checks (__fdividef adds an FSETP and two scaling FMULs
// per call); every operand here is far from the 2^126 limit of rcp.approx.
__device__ __forceinline__ float sph_rcp(float y)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y));
    return r;
}

// 1 / sqrt(y) by one MUFU.RSQ (rsqrtf() adds a denormal-range rescue: three more instructions per call);
// callers clamp y away from zero.
__device__ __forceinline__ float sph_rsqrt(float y)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y));
    return r;
}

// m K with K = 20 SIGMA / H^5: -(dW/dr)/r = K (1 - r/H)^3 for Wendland C2 (reading Q3); invH = 1 / H
__device__ __forceinline__ float sph_mK(float m, float invH)
{
    const float g2 = invH * invH;
    return m * ((SPH_WC2_K20 * invH) * (g2 * g2));
}

// sqrt(y) by one MUFU.SQRT (max relative error 2^-23; sqrt(0) = 0, so no clamp and no multiply as with rsqrt)
__device__ __forceinline__ float sph_sqrt(float y)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y));
    return r;
}

// ---- S2: one term of Eq. 1 and Eq. 3 (Wendland C2, reading Q3) ---------------------------------------------
//   W = SIGMA/H^3 t^4 (1 + 4q),  dW/dh = -SIGMA/(H^3 h) t^3 (3 + 9q - 32 q^2),  q = r/H, t = 1 - q
// rho is evaluated and accumulated in fp64: P = c0^2 (rho - rho0) amplifies the relative error of rho by
// rho/(rho - rho0) ~ 100 on a lattice, and a yielding particle (Y small against rho0 c0^2) passes the error of P
// on to the rescaled S: BASELINE.json configs[0] needs rho to ~2e-8 for its 1e-4 on the yielded state, which is
// below what fp32 geometry can give (measured in round 2: fp32 terms with an fp64 accumulator leave 1.4e-7 in rho
// and 1.02e-4 in S_pred).  The Omega sum (Eq. 3) uses the same fp64 q and t.  r = sqrt(r2) by one Newton step, in fp64, on the
// fp32 rsqrt.  ex, ey, ez: x_i - x_j in fp64 (exact: both are fp32 values); md = m_j.
struct DensAcc {
    double sum;     // sum_j m_j t^4 (1 + 4q)
    double sh;      // sum_j m_j t^3 (3 + 9q - 32 q^2)
    int n;          // |gather set|
};

__device__ __forceinline__ void density_term(DensAcc &A, float r2, double ex, double ey, double ez, double md,
                                             double invHd);

// fp32 -> fp64 of a POSITIVE NORMAL float by integer operations (exact): the conversion instruction runs on the XU
// pipe (16 per clock and SM), which bounds the density kernel; three ALU instructions do not.  Zero becomes 2^-127.
__device__ __forceinline__ double sph_widen_pos(float f)
{
    const unsigned b = __float_as_uint(f);
    return __hiloint2double((int)((b >> 3) + 0x38000000u), (int)(b << 29));
}

// Eq. 5-6 with hbar = hk (H_i + H_j), hk = 1 / (2 kappa), and mu = hk mu', mu' = (H_i + H_j) v.x / (r^2 + eps hbar^2):
// the factor hk is folded into the constants, and the kernels carry max(-mu') (pair_store scales it back)
struct PairConst {
    float beta_h2;    // beta hk^2
    float alpha2_h;   // alpha / 2 * hk: alpha cbar mu = alpha2_h (c_i + c_j) mu'
    float eps_h2;     // eps hk^2
    float hk;         // 1 / (2 kappa)
};
__device__ __forceinline__ PairConst pair_const(float alpha, float beta, float eps_av, float kappa)
{
    PairConst k;
    k.hk = 0.5f / kappa;
    k.beta_h2 = beta * k.hk * k.hk;
    k.alpha2_h = 0.5f * alpha * k.hk;
    k.eps_h2 = eps_av * k.hk * k.hk;
    return k;
}

// per-target operands, constant over the neighbour loop
struct PairTarget {
    float x, y, z;
    float vx, vy, vz;
    float H, invH;    // support radius kappa h_i and its reciprocal
    float K;          // 20 SIGMA / H_i^5
    float wK;         // w_i K_i
    float rho, c;
    float kxx, kyy, kzz, kxy, kxz, kyz;   // K_i st_i
};

struct PairAcc {
    float F[9], C[6];
    float ax, ay, az, du, mumax;     // mumax: max(-mu') (see PairConst)
    float duv;                       // sum_j 1/2 m_j Pi_ij (D_i + D_j) v_ij.x_ij: du/dt gets -1/2 of it (Eq. 8)
};

__device__ __forceinline__ void pair_acc_zero(PairAcc &A)
{
#pragma unroll
    for (int k = 0; k < 9; ++k) A.F[k] = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) A.C[k] = 0.f;
    A.ax = A.ay = A.az = A.du = A.mumax = A.duv = 0.f;
}

// Membership band of the list-driven kernel (SELFMASK): u = max(1 - r/H_i, 1 - r/H_j) computed here differs from the
// exact value by < 5e-7 (r2 by FMA 2.4e-7 hence r 1.2e-7, sqrt.approx 1.2e-7, the reciprocals 1.2e-7, roundings), and the fp32
// predicate of reading Q4 from the real-number boundary by 1e-7: outside |u| <= SPH_UBAND the sign of u IS the predicate.
#ifndef SPH_UBAND
#define SPH_UBAND 2.0e-6f
#endif

// the geometry both the pair term and the re-walk of the ambiguous entries evaluate, operation for operation
struct PairGeom {
    float dx, dy, dz, r2, r, invHj, ui, uj;
};
__device__ __forceinline__ PairGeom pair_geom(const PairTarget &t, float4 q1, float Hj)
{
    PairGeom g;
    g.dx = __fsub_rn(t.x, q1.x); g.dy = __fsub_rn(t.y, q1.y); g.dz = __fsub_rn(t.z, q1.z);
    g.r2 = __fmaf_rn(g.dz, g.dz, __fmaf_rn(g.dy, g.dy, __fmul_rn(g.dx, g.dx)));
    g.r = sph_sqrt(g.r2);
    g.invHj = sph_rcp(Hj);
    g.ui = __fmaf_rn(-g.r, t.invH, 1.f);
    g.uj = __fmaf_rn(-g.r, g.invHj, 1.f);
    return g;
}

// q1 = {x, y, z, m}_j   q2 = {vx, vy, vz, H}_j   q3 = {rho, c, w, st_xx}_j   q4 = {st_yy, st_zz, st_xy, st_xz}_j
// q5 = {st_yz, m K}_j with K_j = 20 SIGMA / H_j^5 (TENSOR only; the hydro-only pass forms m_j K_j itself).
// SELFMASK == false: valid == false means the entry contributes nothing (list padding).
// SELFMASK == true (list-driven kernel; lists with a skin, padding entries pointing at a far dummy source of mass 0):
// nothing is masked by hand -- outside both supports t_i = t_j = 0 and every sum gets an exact zero -- except mu_max
// and the viscosity, which take v = (u > SPH_UBAND); v is returned in `valid` and u in `um`: an entry with
// |u| <= SPH_UBAND is decided by the caller with the exact predicate (its weight is < 1e-17 of a neighbour's either way).
// TENSOR == false (hydro only, S == 0): st is the scalar -P/(Omega rho^2) held in t.kxx / q3.w.
template <bool GRAD, bool FORCE, bool TENSOR = true, bool SELFMASK = false>
__device__ __forceinline__ void pair_term(const PairTarget &t, const PairConst &k, PairAcc &A, float4 q1, float4 q2,
                                          float4 q3, float4 q4, float2 q5, bool &valid, float &um)
{
    const PairGeom g = pair_geom(t, q1, q2.w);
    const float dx = g.dx, dy = g.dy, dz = g.dz, r2 = g.r2, invHj = g.invHj;
    if (SELFMASK) {
        um = fmaxf(g.ui, g.uj);
        valid = um > SPH_UBAND;
    }
    const float ti = fmaxf(0.f, g.ui);
    const float tj = fmaxf(0.f, g.uj);
    const float ti3 = ti * ti * ti, tj3 = tj * tj * tj;
    float mKj;
    if (TENSOR) {
        mKj = q5.y;
    } else {
        mKj = sph_mK(q1.w, invHj);
    }
    const bool on = SELFMASK || valid;
    const float di = (on ? q1.w : 0.f) * ti3;        // m_j t_i^3       (D_i = K_i t_i^3)
    const float dj = (on ? mKj : 0.f) * tj3;         // m_j D_j
    const float dvx = t.vx - q2.x, dvy = t.vy - q2.y, dvz = t.vz - q2.z;
    if (GRAD) {
        const float s = fmaf(di, t.wK, dj * q3.z);   // m_j (w_i D_i + w_j D_j)
        const float sx = s * dx, sy = s * dy, sz = s * dz;
        A.F[0] = fmaf(dvx, sx, A.F[0]); A.F[1] = fmaf(dvx, sy, A.F[1]); A.F[2] = fmaf(dvx, sz, A.F[2]);
        A.F[3] = fmaf(dvy, sx, A.F[3]); A.F[4] = fmaf(dvy, sy, A.F[4]); A.F[5] = fmaf(dvy, sz, A.F[5]);
        A.F[6] = fmaf(dvz, sx, A.F[6]); A.F[7] = fmaf(dvz, sy, A.F[7]); A.F[8] = fmaf(dvz, sz, A.F[8]);
        A.C[0] = fmaf(dx, sx, A.C[0]); A.C[1] = fmaf(dx, sy, A.C[1]); A.C[2] = fmaf(dx, sz, A.C[2]);
        A.C[3] = fmaf(dy, sy, A.C[3]); A.C[4] = fmaf(dy, sz, A.C[4]); A.C[5] = fmaf(dz, sz, A.C[5]);
    }
    if (FORCE) {
        const float vx_ = fmaf(dvx, dx, fmaf(dvy, dy, dvz * dz));          // v_ij . x_ij
        if (TENSOR) {
            // i side: z = K_i st_i x_ij
            const float zx = fmaf(t.kxx, dx, fmaf(t.kxy, dy, t.kxz * dz));
            const float zy = fmaf(t.kxy, dx, fmaf(t.kyy, dy, t.kyz * dz));
            const float zz = fmaf(t.kxz, dx, fmaf(t.kyz, dy, t.kzz * dz));
            A.ax = fmaf(-di, zx, A.ax); A.ay = fmaf(-di, zy, A.ay); A.az = fmaf(-di, zz, A.az);
            A.du = fmaf(di, fmaf(zx, dvx, fmaf(zy, dvy, zz * dvz)), A.du);
            // j side: y = st_j x_ij
            const float yx = fmaf(q3.w, dx, fmaf(q4.z, dy, q4.w * dz));
            const float yy = fmaf(q4.z, dx, fmaf(q4.x, dy, q5.x * dz));
            const float yz = fmaf(q4.w, dx, fmaf(q5.x, dy, q4.y * dz));
            A.ax = fmaf(-dj, yx, A.ax); A.ay = fmaf(-dj, yy, A.ay); A.az = fmaf(-dj, yz, A.az);
        } else {
            const float si = di * t.kxx;                                     // m_j D_i st_i
            const float sc = fmaf(dj, q3.w, si);                             // m_j (D_i st_i + D_j st_j)
            A.ax = fmaf(-sc, dx, A.ax); A.ay = fmaf(-sc, dy, A.ay); A.az = fmaf(-sc, dz, A.az);
            A.du = fmaf(si, vx_, A.du);
        }
        // artificial viscosity (only approaching pairs: min(v.x, 0))
        float vr = fminf(vx_, 0.f);
        vr = valid ? vr : 0.f;
        const float hs = t.H + q2.w;
        const float mu = (hs * vr) * sph_rcp(fmaf(k.eps_h2 * hs, hs, r2));                              // mu'
        const float P2 = (mu * fmaf(k.beta_h2, mu, -k.alpha2_h * (t.c + q3.y))) * sph_rcp(t.rho + q3.x);   // Pi_ij / 2
        const float kk = P2 * fmaf(t.K, di, dj);     // 1/2 m_j Pi_ij (D_i + D_j)
        A.ax = fmaf(kk, dx, A.ax); A.ay = fmaf(kk, dy, A.ay); A.az = fmaf(kk, dz, A.az);
        A.duv = fmaf(kk, vr, A.duv);
        A.mumax = fmaxf(A.mumax, -mu);
    }
}

template <bool GRAD, bool FORCE, bool TENSOR = true>
__device__ __forceinline__ void pair_term(const PairTarget &t, const PairConst &k, PairAcc &A, float4 q1, float4 q2,
                                          float4 q3, float4 q4, float2 q5, bool valid)
{
    float um = 0.f;
    pair_term<GRAD, FORCE, TENSOR, false>(t, k, A, q1, q2, q3, q4, q5, valid, um);
}

// -mu' (>= 0) of one pair: the entries of the list-driven kernel that the exact predicate decides
__device__ __forceinline__ float pair_neg_mu(const PairTarget &t, const PairConst &k, const PairGeom &g, float4 q2)
{
    const float dvx = t.vx - q2.x, dvy = t.vy - q2.y, dvz = t.vz - q2.z;
    const float vr = fminf(fmaf(dvx, g.dx, fmaf(dvy, g.dy, dvz * g.dz)), 0.f);
    const float hs = t.H + q2.w;
    return -(hs * vr) * sph_rcp(fmaf(k.eps_h2 * hs, hs, g.r2));
}

__device__ __forceinline__ void density_term(DensAcc &A, float r2, double ex, double ey, double ez, double md,
                                             double invHd)
{
    const float rinv = sph_rsqrt(fmaxf(r2, 1.0e-37f));
    const double r2d = fma(ex, ex, fma(ey, ey, ez * ez));
    const double yd = sph_widen_pos(rinv), td0 = r2d * yd;
    const double rd = fma(0.5 * td0, fma(-td0, yd, 1.0), td0);
    const double qd = rd * invHd;
    // no clamp at 0: membership (r2 < H_i^2 in fp32) already says q < 1 up to rounding, and (1 - q)^4 of a q that
    // exceeds 1 by 1e-7 is 1e-28
    const double td = 1.0 - qd, a = md * (td * td);
    // both sums from the fp64 q and t: four more fp64 operations instead of nine fp32 ones (the kernel is bound by
    // instruction issue: configs[4] 10.08 -> 9.91 ms)
    A.sh = fma(a * td, fma(qd, fma(-32.0, qd, 9.0), 3.0), A.sh);
    A.sum = fma(a * (td * td), fma(4.0, qd, 1.0), A.sum);
    A.n++;
}

// rho (fp64 and fp32) and Omega from the sums; invH = 1 / (kappa h_i) in fp32 (the Omega terms), invHd in fp64
__device__ __forceinline__ void density_finish(const DensAcc &A, float invH, double invHd, double &rhod, float &rho,
                                               float &omega)
{
    rhod = 3.3422538049298023 * invHd * invHd * invHd * A.sum;
    rho = (float)rhod;
    const float kw = SPH_WC2_SIGMA * invH * invH * invH;
    omega = 1.f - kw * (float)A.sh / (3.f * rho);
}

// loads the per-target operands (resident arrays of sph_internal.cuh's Dev)
__device__ __forceinline__ PairTarget pair_target_load(const Dev &d, long long i, float kappa)
{
    const float4 pi = d.r.pm[i], vi = d.r.vh[i], b3 = d.B3[i], b4 = d.B4[i];
    const float b5 = d.B5[i].x;
    PairTarget t;
    t.x = pi.x; t.y = pi.y; t.z = pi.z;
    t.vx = vi.x; t.vy = vi.y; t.vz = vi.z;
    t.H = sph_H(kappa, vi.w);
    t.invH = 1.f / t.H;
    const float g2 = t.invH * t.invH;
    t.K = (SPH_WC2_K20 * t.invH) * (g2 * g2);
    t.wK = b3.z * t.K;
    t.rho = b3.x; t.c = b3.y;
    t.kxx = t.K * b3.w; t.kyy = t.K * b4.x; t.kzz = t.K * b4.y;
    t.kxy = t.K * b4.z; t.kxz = t.K * b4.w; t.kyz = t.K * b5;
    return t;
}

// add_aext == false: a_ext is added by CLOSE instead (SPH_INT_DEFER_AEXT)
template <bool GRAD, bool FORCE>
__device__ __forceinline__ void pair_store(const Dev &d, long long i, const PairAcc &A, const PairConst &k, bool add_aext)
{
    if (GRAD) {
#pragma unroll
        for (int c = 0; c < 9; ++c) d.F[c][i] = 0.5f * A.F[c];
        const float c0 = 0.5f * A.C[0], c1 = 0.5f * A.C[1], c2 = 0.5f * A.C[2], c3 = 0.5f * A.C[3], c4 = 0.5f * A.C[4],
                    c5 = 0.5f * A.C[5];
        d.Cinv[0][i] = c0; d.Cinv[1][i] = c1; d.Cinv[2][i] = c2;
        d.Cinv[3][i] = c1; d.Cinv[4][i] = c3; d.Cinv[5][i] = c4;
        d.Cinv[6][i] = c2; d.Cinv[7][i] = c4; d.Cinv[8][i] = c5;
    }
    if (FORCE) {
        float gx = 0.f, gy = 0.f, gz = 0.f;
        if (add_aext) { gx = d.r.s[PP_G + 0][i]; gy = d.r.s[PP_G + 1][i]; gz = d.r.s[PP_G + 2][i]; }
        d.a[0][i] = A.ax + gx;
        d.a[1][i] = A.ay + gy;
        d.a[2][i] = A.az + gz;
        d.dudt[i] = fmaf(-0.5f, A.duv, A.du);
        d.mumax[i] = k.hk * A.mumax;
    }
}
