// sph_particle.cu -- the per-particle (HBM-bound) kernels: S3 predict / EOS / yield, S6 close,
// S7 kick-drift-predict, S8 time-step reduction, and the caller-order scatter helpers.
#include "sph_internal.cuh"

#define WC2_SIGMA 3.3422538049298023f     // 21 / (2 pi), Wendland C2 in 3-D (reading Q3)
#define SPH_CTOL 1.0e-4f                  // reading Q9: C = 1 unless |det C^-1| > CTOL ||C^-1||_F^3

// ------------------------------------------------------------------------------------------
// material laws
// ------------------------------------------------------------------------------------------
// Y_i = Y0 + mu_i P/(1 + mu_i P/(Ym - Y0)) with P < 0 clipped (Eq. 34);
// Y = min(Y_i, mu_d P) for finite mu_d (Eq. 35-36); Y *= max(0, tanh(xi (Tm/T - 1))) (Eq. 37).
__device__ __forceinline__ float yield_strength(const sph_material &m, float P, float T, float Tmelt)
{
    float Pp = fmaxf(P, 0.f);
    float span = m.Ym - m.Y0;
    float Y = m.Y0;
    if (span > 0.f) Y = m.Y0 + m.mu_i * Pp / (1.f + m.mu_i * Pp / span);
    if (isfinite(m.mu_d)) Y = fminf(Y, m.mu_d * Pp);
    float soft = 1.f;
    if (T > 0.f) soft = fmaxf(0.f, tanhf(m.xi * (Tmelt / T - 1.f)));
    return Y * soft;
}

// NEXT-3 (P and T from (rho, u) tables, T_melt "a tabulated function of density"): piecewise-
// linear / bilinear lookup on a uniform grid, clamped to the grid's edges (reading Q21).  Index and weights
// in fp64 from the fp64 density: (rho - rho_k) cancels like (rho - rho0) does in the analytic EOS.
__device__ __forceinline__ void table_cell(double x, float x_min, float x_max, int n, int &i, double &t)
{
    double f = (x - (double)x_min) / ((double)x_max - (double)x_min) * (double)(n - 1);
    f = fmin(fmax(f, 0.0), (double)(n - 1));
    i = min((int)f, n - 2);
    t = f - (double)i;
}
__device__ __forceinline__ float table_2d(const float *__restrict__ f, int n_u, int i, int j, double tx, double ty)
{
    const float *r0 = f + (size_t)i * n_u + j, *r1 = r0 + n_u;
    return (float)((1.0 - tx) * (1.0 - ty) * (double)r0[0] + tx * (1.0 - ty) * (double)r1[0]
                   + (1.0 - tx) * ty * (double)r0[1] + tx * ty * (double)r1[1]);
}

// f = min(Y / sqrt(J2), 1) (Eq. 31-33); J2 from the five stored components
__device__ __forceinline__ float plastic_factor(const float S[5], float Y)
{
    float szz = -S[0] - S[1];
    float J2 = 0.5f * (S[0] * S[0] + S[1] * S[1] + szz * szz) + S[2] * S[2] + S[3] * S[3] + S[4] * S[4];
    float sj = sqrtf(J2);
    return sj > Y ? Y / sj : 1.f;
}

// ------------------------------------------------------------------------------------------
// S3 PREDICT: EOS (reading Q13), Gamma (Eq. 30), Y (Eq. 34-37), S_pred <- f S_pred (Eq. 31,
// PAPER.md:240), and the packed operands of the pair pass (sph_pairterm.cuh):
//   B3 = {rho, c, w, st_xx}, B4 = {st_yy, st_zz, st_xy, st_xz}, B5 = st_yz
//   w = 1/(Omega rho), st = (-P delta + S_pred)/(Omega rho^2)
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_predict(Dev d, DevParams p, DevTabs tabs, RungCtl rc)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    if (rc.on && !rc.tile_need[i / SPH_TILE]) return;        // NEXT-4: nobody reads this particle in this substep
    unsigned mf = ((const unsigned *)d.r.s[PP_MATFIX])[i];
    const sph_material &m = p.mat[mf & 0xffu];
    float rho = d.rho[i], om = d.omega[i], u = d.r.s[PP_UPRED][i];
    const DevTab &tb = tabs.t[mf & 0xffu];
    float P, cs, T, Tmelt = m.Tmelt;
    if (tb.P) {
        int ir, iu;
        double tr, tu;
        table_cell(d.rho64[i], tb.rho_min, tb.rho_max, tb.n_rho, ir, tr);
        table_cell((double)u, tb.u_min, tb.u_max, tb.n_u, iu, tu);
        P = table_2d(tb.P, tb.n_u, ir, iu, tr, tu);
        T = table_2d(tb.T, tb.n_u, ir, iu, tr, tu);
        cs = table_2d(tb.cs, tb.n_u, ir, iu, tr, tu);
        if (tb.Tmelt) {
            table_cell(d.rho64[i], tb.rho_min, tb.rho_max, tb.n_melt, ir, tr);
            Tmelt = (float)((1.0 - tr) * (double)tb.Tmelt[ir] + tr * (double)tb.Tmelt[ir + 1]);
        }
    } else {
        // the subtraction rho - rho0 in fp64 (see k_density)
        P = (float)((double)m.c0 * (double)m.c0 * (d.rho64[i] - (double)m.rho0));
        cs = m.c0;
        T = u / m.cv;
    }
    if (p.flags & SPH_PCLIP_GLOBAL) P = fmaxf(P, 0.f);
    float Gam = m.Gamma > 0.f ? m.Gamma : 3.f * (1.f - 2.f * m.nu) / (2.f * (1.f + m.nu)) * rho * cs * cs;
    float Y = yield_strength(m, P, T, Tmelt);
    float S[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (p.flags & SPH_STRENGTH) {
#pragma unroll
        for (int c = 0; c < 5; ++c) S[c] = d.r.s[PP_SPRED + c][i];
        float f = plastic_factor(S, Y);
#pragma unroll
        for (int c = 0; c < 5; ++c) { S[c] *= f; d.r.s[PP_SPRED + c][i] = S[c]; }
    }
    d.P[i] = P; d.cs[i] = cs; d.T[i] = T; d.Gamma[i] = Gam; d.Y[i] = Y;

    float w = 1.f / (om * rho);
    float g = w / rho;                                // 1 / (Omega rho^2)
    d.B3[i] = make_float4(rho, cs, w, g * (S[0] - P));
    d.B4[i] = make_float4(g * (S[1] - P), g * (-S[0] - S[1] - P), g * S[2], g * S[3]);
    d.B5[i] = make_float2(g * S[4], d.mK[i]);
}

// ------------------------------------------------------------------------------------------
// S6 CLOSE: C = (C^-1)^-1, G = F.C (Eq. 22), eps_dot, R (Eq. 23-24), dS/dt (Eq. 25-29 as
// reconstructed from Eq. 13, reading Q2), closing kick (Eq. 41) + rescale,
// strain-rate invariant (Eq. 43), per-particle time-step limit (Eq. 38-39).
// phase == SPH_DERIVATIVES leaves v, u, S, e_acc untouched (bootstrap of the first step).
// ------------------------------------------------------------------------------------------
// Also S8: the block's minimum of dt_i goes into dt_next with one atomicMin (positive floats order like
// unsigned ints; k_dt_select / k_dt_reset set dt_next to +inf before), and the robustness counters.
// NEXT-4 (rc.on): only the active particles; the step of the closing kick is the particle's own, dT / 2^rung, and
// the particle chooses its next rung from its new limit (reading Q23).
__global__ void __launch_bounds__(256, 6) k_close(Dev d, DevParams p, int phase, float dt_arg, int dt_from_device, RungCtl rc)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    float dti = __int_as_float(0x7f800000);
    unsigned nfall = 0u, nbad = 0u, nact = 0u;
    if (i < d.n && sph_active(rc, i)) {
    float dt = dt_from_device ? *d.dt_cur : dt_arg;
    if (rc.on) { dt = rc.dT / (float)(1 << (int)d.rung[i]); nact = 1u; }
    const bool strength = (p.flags & SPH_STRENGTH) != 0;
    unsigned mf = ((const unsigned *)d.r.s[PP_MATFIX])[i];
    const bool fixed = (mf >> 8) & 1u;
    float dS[5] = {0.f, 0.f, 0.f, 0.f, 0.f}, eps2 = 0.f, cflag = 0.f;
    if (strength) {
        float F[9], Ci[9], C[9], G[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) { F[k] = d.F[k][i]; Ci[k] = d.Cinv[k][i]; }
        // cofactors / determinant of C^-1
        float c00 = Ci[4] * Ci[8] - Ci[5] * Ci[7], c01 = Ci[5] * Ci[6] - Ci[3] * Ci[8], c02 = Ci[3] * Ci[7] - Ci[4] * Ci[6];
        float det = Ci[0] * c00 + Ci[1] * c01 + Ci[2] * c02;
        float fro2 = 0.f;
#pragma unroll
        for (int k = 0; k < 9; ++k) fro2 = fmaf(Ci[k], Ci[k], fro2);
        float fro = sqrtf(fro2);
        bool ok = (p.flags & SPH_CORRECTION_TENSOR) && (fabsf(det) > SPH_CTOL * fro * fro * fro);
        if (ok) {
            float id = 1.f / det;
            C[0] = c00 * id;
            C[1] = (Ci[2] * Ci[7] - Ci[1] * Ci[8]) * id;
            C[2] = (Ci[1] * Ci[5] - Ci[2] * Ci[4]) * id;
            C[3] = c01 * id;
            C[4] = (Ci[0] * Ci[8] - Ci[2] * Ci[6]) * id;
            C[5] = (Ci[2] * Ci[3] - Ci[0] * Ci[5]) * id;
            C[6] = c02 * id;
            C[7] = (Ci[1] * Ci[6] - Ci[0] * Ci[7]) * id;
            C[8] = (Ci[0] * Ci[4] - Ci[1] * Ci[3]) * id;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    G[3 * a + b] = F[3 * a] * C[b] + F[3 * a + 1] * C[3 + b] + F[3 * a + 2] * C[6 + b];
        } else {
            cflag = 1.f;
            nfall = 1u;
#pragma unroll
            for (int k = 0; k < 9; ++k) G[k] = F[k];
        }
#pragma unroll
        for (int k = 0; k < 9; ++k) d.G[k][i] = G[k];
        const float Gxx = G[0], Gxy = G[1], Gxz = G[2], Gyx = G[3], Gyy = G[4], Gyz = G[5], Gzx = G[6], Gzy = G[7], Gzz = G[8];
        const float Sxx = d.r.s[PP_SPRED + 0][i], Syy = d.r.s[PP_SPRED + 1][i], Sxy = d.r.s[PP_SPRED + 2][i],
                    Sxz = d.r.s[PP_SPRED + 3][i], Syz = d.r.s[PP_SPRED + 4][i];
        const float Gam = d.Gamma[i];
        // reading Q1: the objective (co-rotational) Jaumann rate R.S - S.R by default; the index order as printed is its negative
        const float s = (p.flags & SPH_JAUMANN_AS_PRINTED) ? 1.f : -1.f;
        const float rxy = Gxy - Gyx, rxz = Gxz - Gzx, ryz = Gyz - Gzy;       // 2 R^{xy}, 2 R^{xz}, 2 R^{yz}
        dS[0] = s * (-Sxy * rxy - Sxz * rxz) - (2.f / 3.f) * Gam * (Gyy + Gzz - 2.f * Gxx);
        dS[1] = s * (Sxy * rxy - Syz * ryz) - (2.f / 3.f) * Gam * (Gxx + Gzz - 2.f * Gyy);
        dS[2] = Gam * (Gxy + Gyx) + s * 0.5f * (Sxx * rxy - Syy * rxy - Syz * rxz - Sxz * ryz);
        dS[3] = Gam * (Gxz + Gzx) + s * 0.5f * ((Sxx + Syy) * rxz + Sxx * rxz + Sxy * ryz - Syz * rxy);
        dS[4] = Gam * (Gyz + Gzy) + s * 0.5f * ((Sxx + Syy) * ryz + Syy * ryz + Sxz * rxy + Sxy * rxz);
        // 1/2 eps_dot : eps_dot with eps_dot = (G + G^T)/2
        float exy = 0.5f * (Gxy + Gyx), exz = 0.5f * (Gxz + Gzx), eyz = 0.5f * (Gyz + Gzy);
        eps2 = 0.5f * (Gxx * Gxx + Gyy * Gyy + Gzz * Gzz) + exy * exy + exz * exz + eyz * eyz;
        d.cflag[i] = cflag;
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) d.dS[c][i] = dS[c];
    d.eps2[i] = eps2;

    // time-step limit, Eq. 39 (and Eq. 38 with epsilon = h when eta_a > 0)
    float h = d.r.vh[i].w;
    float ax = d.a[0][i], ay = d.a[1][i], az = d.a[2][i];
    if (p.flags & SPH_INT_DEFER_AEXT) {               // the pair pass left a_ext out (sph_step_host): a = a_int + a_ext
        ax += d.r.s[PP_G + 0][i]; ay += d.r.s[PP_G + 1][i]; az += d.r.s[PP_G + 2][i];
        d.a[0][i] = ax; d.a[1][i] = ay; d.a[2][i] = az;
    }
    dti = p.eta_C * h / ((1.f + 0.6f * p.alpha) * d.cs[i] + 0.6f * p.beta * d.mumax[i]);
    if (p.eta_a > 0.f) {
        float an = sqrtf(ax * ax + ay * ay + az * az);
        if (an > 0.f) dti = fminf(dti, p.eta_a * sqrtf(h / an));
    }
    d.dti[i] = dti;
    const float du_ = d.dudt[i];
    if (!(isfinite(ax) && isfinite(ay) && isfinite(az) && isfinite(du_) && isfinite(dS[0] + dS[1] + dS[2] + dS[3] + dS[4])))
        nbad = 1u;

    if (phase == SPH_CLOSE) {
        float hdt = 0.5f * dt;
        float vx = d.r.s[PP_VHALF + 0][i], vy = d.r.s[PP_VHALF + 1][i], vz = d.r.s[PP_VHALF + 2][i];
        if (!fixed) { vx = fmaf(hdt, ax, vx); vy = fmaf(hdt, ay, vy); vz = fmaf(hdt, az, vz); }
        d.vfull[0][i] = vx; d.vfull[1][i] = vy; d.vfull[2][i] = vz;
        d.ufull[i] = fmaf(hdt, du_, d.r.s[PP_UHALF][i]);
        float S[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
        if (strength) {
#pragma unroll
            for (int c = 0; c < 5; ++c) S[c] = fmaf(hdt, dS[c], d.r.s[PP_SHALF + c][i]);
            float f = plastic_factor(S, d.Y[i]);
#pragma unroll
            for (int c = 0; c < 5; ++c) S[c] *= f;
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) d.Sfull[c][i] = S[c];
        d.r.s[PP_EACC][i] = fmaf(dt, eps2, d.r.s[PP_EACC][i]);
    }
    if (rc.on && !rc.fixed_rungs) {
        // next rung: the smallest one whose step is within the new limit, but no coarser than the rungs whose
        // steps line up with the present time (n1 substeps of 2^R done)
        // (a limit that is not a number sends the particle to the finest rung; a limit below the finest step is counted)
        int want = 0;
        while (want < rc.R && !(rc.dT / (float)(1 << want) <= dti)) ++want;
        if (!(rc.dT / (float)(1 << rc.R) <= dti)) atomicAdd(&d.counters[SPH_C_RUNG_CLAMPED], 1ull);     // rare
        const int tz = rc.n1 >= (1 << rc.R) ? rc.R : (__ffs(rc.n1) - 1);
        d.rung[i] = (unsigned char)min(rc.R, max(want, rc.R - tz));
    }
    }   // i < d.n and active
    // S8 and the counters: one atomic per block
    __shared__ float s_dt[8];
    __shared__ unsigned s_cnt[8];
    unsigned packed = nfall | (nbad << 16);
    if (rc.on) {
        const unsigned na = __popc(__ballot_sync(0xffffffffu, nact != 0u));
        if ((threadIdx.x & 31) == 0 && na) atomicAdd(&d.counters[SPH_C_ACTIVE_UPDATES], (unsigned long long)na);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dti = fminf(dti, __shfl_xor_sync(0xffffffffu, dti, o));
        packed += __shfl_xor_sync(0xffffffffu, packed, o);
    }
    if ((threadIdx.x & 31) == 0) { s_dt[threadIdx.x >> 5] = dti; s_cnt[threadIdx.x >> 5] = packed; }
    __syncthreads();
    if (threadIdx.x == 0) {
        float m = s_dt[0];
        unsigned c = s_cnt[0];
#pragma unroll
        for (int w = 1; w < 8; ++w) { m = fminf(m, s_dt[w]); c += s_cnt[w]; }
        if (m > 0.f) atomicMin((unsigned *)d.dt_next, __float_as_uint(m));
        if (c & 0xffffu) atomicAdd(&d.counters[SPH_C_CFALLBACK], (unsigned long long)(c & 0xffffu));
        if (c >> 16) atomicAdd(&d.counters[SPH_C_NONFINITE], (unsigned long long)(c >> 16));
    }
}

// ------------------------------------------------------------------------------------------
// S8: dt_next = min_i dt_i is accumulated by k_close; these set it up
// ------------------------------------------------------------------------------------------
__global__ void k_dt_reset(float *dt_next) { *(unsigned *)dt_next = 0x7f800000u; }

// head of a step: the step in use (dt_arg, or the CFL step the last CLOSE left in dt_next), and dt_next
// reset to +inf for this step's CLOSE
__global__ void k_dt_select(float dt_arg, float *dt_cur, float *dt_next, float *dt_used)
{
    float dt = dt_arg > 0.f ? dt_arg : *dt_next;
    *dt_cur = dt;
    if (dt_used) *dt_used = dt;
    *(unsigned *)dt_next = 0x7f800000u;
}

// ------------------------------------------------------------------------------------------
// S7 opening kick (Eq. 42), drift, prediction (Eq. 40); fixed particles keep x and v
// ------------------------------------------------------------------------------------------
// PARTS: 1 = x and v, 2 = u and S, 3 = both.  The two halves are independent; sph_step_host runs the second one after
// the list check and the density pass, while u, S and a_ext are still on their way from the host.
template <int PARTS>
__global__ void __launch_bounds__(256) k_kick_drift(Dev d, DevParams p)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const float dt = *d.dt_cur, hdt = 0.5f * dt;
    if (PARTS & 1) {
        unsigned mf = ((const unsigned *)d.r.s[PP_MATFIX])[i];
        const bool fixed = (mf >> 8) & 1u;
        float4 pm = d.r.pm[i];
        float h = d.r.vh[i].w;
        float v[3] = {d.vfull[0][i], d.vfull[1][i], d.vfull[2][i]};
        float a[3] = {d.a[0][i], d.a[1][i], d.a[2][i]};
        float vh[3], vp[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            vh[k] = fixed ? v[k] : fmaf(hdt, a[k], v[k]);
            vp[k] = fixed ? v[k] : fmaf(hdt, a[k], vh[k]);
            d.r.s[PP_VHALF + k][i] = vh[k];
        }
        if (!fixed) { pm.x = fmaf(dt, vh[0], pm.x); pm.y = fmaf(dt, vh[1], pm.y); pm.z = fmaf(dt, vh[2], pm.z); }
        d.r.pm[i] = pm;
        d.r.vh[i] = make_float4(vp[0], vp[1], vp[2], h);
    }
    if (PARTS & 2) {
        float du = d.dudt[i];
        float uh = fmaf(hdt, du, d.ufull[i]);
        d.r.s[PP_UHALF][i] = uh;
        d.r.s[PP_UPRED][i] = fmaf(hdt, du, uh);
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            float ds = d.dS[c][i];
            float sh = fmaf(hdt, ds, d.Sfull[c][i]);
            d.r.s[PP_SHALF + c][i] = sh;
            d.r.s[PP_SPRED + c][i] = fmaf(hdt, ds, sh);
        }
    }
}

// ------------------------------------------------------------------------------------------
// NEXT-4: rungs (reading Q23).  k_rung_assign: at the start of a big step, from the limits of the last CLOSE (or the
// caller's fixed rungs).  k_kick_drift_rung: substep n of 2^R: opening kick (Eq. 42, own step) of the particles that
// start a step, drift of all by delta, prediction of all to the new time (Eq. 40 generalised), and the tiles that
// hold a particle which ends a step now.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_rung_assign(Dev d, float dT, int R, const unsigned char *__restrict__ fixed_rungs)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    int r = 0;
    if (fixed_rungs) r = min((int)fixed_rungs[((const unsigned *)d.r.s[PP_ORIG])[i]], R);
    else {
        const float dti = d.dti[i];
        while (r < R && !(dT / (float)(1 << r) <= dti)) ++r;         // NaN limit: the finest rung, not the coarsest
        if (!(dT / (float)(1 << R) <= dti)) atomicAdd(&d.counters[SPH_C_RUNG_CLAMPED], 1ull);   // beyond its limit even there
    }
    d.rung[i] = (unsigned char)r;
}

__global__ void __launch_bounds__(256) k_kick_drift_rung(Dev d, DevParams p, int n, int R, float dT)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const int r = (int)d.rung[i], per = 1 << (R - r), kk = n & (per - 1);
    const float dtr = dT / (float)(1 << r), delta = dT / (float)(1 << R), hdt = 0.5f * dtr;
    const float tau = (float)(kk + 1) * delta - hdt;                 // new time minus the middle of the particle's step
    unsigned mf = ((const unsigned *)d.r.s[PP_MATFIX])[i];
    const bool fixed = (mf >> 8) & 1u;
    const bool start = kk == 0;
    float4 pm = d.r.pm[i];
    const float h = d.r.vh[i].w;
    const float a[3] = {d.a[0][i], d.a[1][i], d.a[2][i]};
    float vh[3], vp[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        if (start) {
            const float v = d.vfull[k][i];
            vh[k] = fixed ? v : fmaf(hdt, a[k], v);
            d.r.s[PP_VHALF + k][i] = vh[k];
        } else {
            vh[k] = d.r.s[PP_VHALF + k][i];
        }
        vp[k] = fixed ? vh[k] : fmaf(tau, a[k], vh[k]);
    }
    if (!fixed) { pm.x = fmaf(delta, vh[0], pm.x); pm.y = fmaf(delta, vh[1], pm.y); pm.z = fmaf(delta, vh[2], pm.z); }
    d.r.pm[i] = pm;
    d.r.vh[i] = make_float4(vp[0], vp[1], vp[2], h);
    const float du = d.dudt[i];
    float uh;
    if (start) { uh = fmaf(hdt, du, d.ufull[i]); d.r.s[PP_UHALF][i] = uh; }
    else uh = d.r.s[PP_UHALF][i];
    d.r.s[PP_UPRED][i] = fmaf(tau, du, uh);
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        const float ds = d.dS[c][i];
        float sh;
        if (start) { sh = fmaf(hdt, ds, d.Sfull[c][i]); d.r.s[PP_SHALF + c][i] = sh; }
        else sh = d.r.s[PP_SHALF + c][i];
        d.r.s[PP_SPRED + c][i] = fmaf(tau, ds, sh);
    }
    if (((n + 1) & (per - 1)) == 0) d.tile_act[i / SPH_TILE] = 1;    // ends a step now: active (same value from all)
}

// tiles that hold a candidate neighbour of an active tile need their density and PREDICT in this substep
// lists == 0 (SPH_NO_LISTS): there are no candidate lists to follow (tile_flag, tile_ncand, tile_off, cand are never
// written), and the tree-walk pair pass works on every tile: every tile is needed.
__global__ void __launch_bounds__(256) k_mark_need(Dev d, int ntile, int lists)
{
    const int tile = blockIdx.x;
    if (tile >= ntile) return;
    if (!lists) {
        if (threadIdx.x == 0) {
            d.tile_need[tile] = 1;
            atomicAdd(&d.counters[SPH_C_ACTIVE_TILES], 1ull);
        }
        return;
    }
    if (!d.tile_act[tile]) return;
    if (threadIdx.x == 0) {
        d.tile_need[tile] = 1;
        atomicAdd(&d.counters[SPH_C_ACTIVE_TILES], 1ull);
    }
    if (d.tile_flag[tile]) {                              // no candidate list (served by the tree walk): everything
        for (int t = threadIdx.x; t < ntile; t += blockDim.x) d.tile_need[t] = 1;
        return;
    }
    const int nc = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    for (int s = threadIdx.x; s < nc; s += blockDim.x) d.tile_need[cand[s] / SPH_TILE] = 1;
}

int sph_launch_rung_assign(sph_ctx *c, float dT, int R, const unsigned char *rungs)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_rung_assign<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, dT, R, rungs);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_kick_drift_rung(sph_ctx *c, int n, int R, float dT)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    const size_t ntile = (size_t)sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    SPH_CUDA(c, cudaMemsetAsync(d.tile_act, 0, ntile, c->stream));
    SPH_CUDA(c, cudaMemsetAsync(d.tile_need, 0, ntile, c->stream));
    k_kick_drift_rung<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, c->p, n, R, dT);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_mark_need(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    const int ntile = sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    k_mark_need<<<ntile, 256, 0, c->stream>>>(d, ntile, c->use_lists ? 1 : 0);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------
// caller-order scatter helpers
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_scatter(const float *__restrict__ src, const unsigned *__restrict__ orig,
                                                 long long n, float *__restrict__ dst, int as_int)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    dst[orig[i]] = as_int == 2 ? (float)((const unsigned char *)src)[i] : (as_int ? (float)((const int *)src)[i] : src[i]);
}

__global__ void __launch_bounds__(256) k_scatter_pos(const float4 *__restrict__ pm, const unsigned *__restrict__ orig,
                                                     long long n, float *__restrict__ dst, int comp)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 q = pm[i];
    dst[orig[i]] = comp == 0 ? q.x : (comp == 1 ? q.y : q.z);
}

// part: 0 everything, 1 the positions only (final once the drift is done), 2 everything but the positions
__global__ void __launch_bounds__(256) k_download(Dev d, sph_state st, int part)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    unsigned o = ((const unsigned *)d.r.s[PP_ORIG])[i];
    if (part != 2) {
        float4 pm = d.r.pm[i];
        st.x[o] = pm.x; st.y[o] = pm.y; st.z[o] = pm.z;
    }
    if (part == 1) return;
    st.vx[o] = d.vfull[0][i]; st.vy[o] = d.vfull[1][i]; st.vz[o] = d.vfull[2][i];
    st.u[o] = d.ufull[i];
    st.Sxx[o] = d.Sfull[0][i]; st.Syy[o] = d.Sfull[1][i]; st.Sxy[o] = d.Sfull[2][i];
    st.Sxz[o] = d.Sfull[3][i]; st.Syz[o] = d.Sfull[4][i];
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
int sph_launch_predict(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_predict<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, c->p, c->tabs, c->rc);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_close(sph_ctx *c, int phase, float dt, bool dt_from_device)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_CFALLBACK], 0, sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_NONFINITE], 0, sizeof(unsigned long long), c->stream));
    if (!dt_from_device) {                 // inside sph_step k_dt_select has already reset dt_next
        k_dt_reset<<<1, 1, 0, c->stream>>>(d.dt_next);
        c->launches++;
    }
    if (d.n > 0) {
        k_close<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, c->p, phase, dt, dt_from_device ? 1 : 0, c->rc);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// parts: 1 = x and v (selects the time step first), 2 = u and S (with the step already selected), 3 = everything
int sph_launch_kick_drift(sph_ctx *c, float dt, int parts)
{
    Dev &d = c->d;
    if (parts & 1) {
        k_dt_select<<<1, 1, 0, c->stream>>>(dt, d.dt_cur, d.dt_next, nullptr);
        c->launches++;
    }
    if (d.n > 0) {
        const int nb = sph_div_up(d.n, 256);
        if (parts == 3) k_kick_drift<3><<<nb, 256, 0, c->stream>>>(d, c->p);
        else if (parts == 1) k_kick_drift<1><<<nb, 256, 0, c->stream>>>(d, c->p);
        else k_kick_drift<2><<<nb, 256, 0, c->stream>>>(d, c->p);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------
// NEXT-1: one Newton-Raphson update of h_i towards a constant kernel mass (Eq. 2):
//   M_tot = (4/3) pi (kappa h)^3 rho(h),  d(h^3 rho)/dh = 3 h^2 rho Omega (Eq. 3)
//   h <- h [1 - (1 - n_target m / M_tot) / (3 max(Omega, 0.1))], factor limited to [0.8, 1.25] (reading Q20)
// Per particle, in fp64 from the fp64 density; h is stored back in fp32.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_h_update(Dev d, float kappa, float n_target, float *hchange)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    float change = 0.f;
    if (i < d.n) {
        float4 vh = d.r.vh[i];
        const double h = (double)vh.w, H = (double)kappa * h;
        const double mtot = 4.0 / 3.0 * 3.14159265358979323846 * H * H * H * d.rho64[i];
        const double ratio = (double)n_target * (double)d.r.pm[i].w / mtot;
        double fac = 1.0 - (1.0 - ratio) / (3.0 * fmax((double)d.omega[i], 0.1));
        fac = fmin(fmax(fac, 0.8), 1.25);
        vh.w = (float)(h * fac);
        d.r.vh[i] = vh;
        change = (float)fabs(fac - 1.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) change = fmaxf(change, __shfl_xor_sync(0xffffffffu, change, o));
    if ((threadIdx.x & 31) == 0 && change > 0.f) atomicMax((unsigned *)hchange, __float_as_uint(change));
}

int sph_launch_h_update(sph_ctx *c, float n_target)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(d.hchange, 0, sizeof(float), c->stream));
    if (d.n > 0) {
        k_h_update<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, c->p.kappa, n_target, d.hchange);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------
// S8 diagnostics (the conservation checks): M, sum m v, sum m x cross v, sum m (v^2/2 + u)
// of the state at the full step, in fp64, in a fixed order (per-block partials, then one block):
// bitwise repeatable.
// ------------------------------------------------------------------------------------------
#define DIAG_BLOCKS 592
__global__ void __launch_bounds__(256) k_diag_partial(Dev d, double *__restrict__ part)
{
    double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < d.n; i += (long long)gridDim.x * blockDim.x) {
        const float4 pm = d.r.pm[i];
        const double m = pm.w, x = pm.x, y = pm.y, z = pm.z;
        const double vx = d.vfull[0][i], vy = d.vfull[1][i], vz = d.vfull[2][i], u = d.ufull[i];
        s[0] += m;
        s[1] += m * vx; s[2] += m * vy; s[3] += m * vz;
        s[4] += m * (y * vz - z * vy); s[5] += m * (z * vx - x * vz); s[6] += m * (x * vy - y * vx);
        s[7] += m * (0.5 * (vx * vx + vy * vy + vz * vz) + u);
    }
    __shared__ double sh[8][8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < 8) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[w][threadIdx.x];
        part[blockIdx.x * 8 + threadIdx.x] = t;
    }
}

__global__ void k_diag_final(const double *__restrict__ part, int nblocks, double *__restrict__ out)
{
    // 8 warps, one per quantity; lanes stride over the partials, then a shuffle tree: a fixed order
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double t = 0.0;
    for (int b = lane; b < nblocks; b += 32) t += part[b * 8 + k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) out[k] = t;
}

int sph_launch_diagnostics(sph_ctx *c, double *out)
{
    Dev &d = c->d;
    int nb = sph_div_up(d.n > 0 ? d.n : 1, 256);
    if (nb > DIAG_BLOCKS) nb = DIAG_BLOCKS;
    k_diag_partial<<<nb, 256, 0, c->stream>>>(d, d.diag_part);
    k_diag_final<<<1, 256, 0, c->stream>>>(d.diag_part, nb, out);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// h in caller order (sph_get_field(SPH_F_H))
__global__ void __launch_bounds__(256) k_scatter_h(const float4 *__restrict__ vh, const unsigned *__restrict__ orig,
                                                   long long n, float *__restrict__ dst)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) dst[orig[i]] = vh[i].w;
}

// the tile (SPH_TILE curve-consecutive resident particles) each particle sits in, caller order (sph_get_field(SPH_F_TILE))
__global__ void __launch_bounds__(256) k_scatter_tile(const unsigned *__restrict__ orig, long long n, float *__restrict__ dst)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) dst[orig[i]] = (float)(i / SPH_TILE);
}

int sph_launch_get_tile(sph_ctx *c, float *dst)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_scatter_tile<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>((const unsigned *)d.r.s[PP_ORIG], d.n, dst);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_get_h(sph_ctx *c, float *dst)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_scatter_h<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d.r.vh, (const unsigned *)d.r.s[PP_ORIG], d.n, dst);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_get_field(sph_ctx *c, const float *src, float *dst, int as_int)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_scatter<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(src, (const unsigned *)d.r.s[PP_ORIG], d.n, dst, as_int);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_get_position(sph_ctx *c, int comp, float *dst)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_scatter_pos<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d.r.pm, (const unsigned *)d.r.s[PP_ORIG], d.n, dst, comp);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_download(sph_ctx *c, sph_state *st, int part)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    k_download<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d, *st, part);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}
