// sph_pair.cu -- the neighbour (pair) passes S2, S4, S5 and the neighbour-set test hook.
//
// Layout of the work: one warp owns one target chunk (32 Morton-consecutive particles, one per
// lane, all target state in registers).  The warp walks the implicit 32-ary chunk tree (one lane
// tests one child box), and for every source chunk whose box can reach the target box it stages
// the 32 source particles in shared memory with coalesced float4 loads and runs them past all 32
// targets (shared-memory broadcast reads).  Every ordered pair (i, j) is evaluated from i's side
// only (gather form): no atomics on particle data, run-to-run bit-identical results.
//
// Membership is decided by the fp32 predicate of DESIGN.md reading Q4 (sph_r2, no FMA).
#include "sph_internal.cuh"

#define PAIR_WARPS 8                      // warps (= target chunks) per CTA
#define STACK_DEPTH (SPH_ARITY * (SPH_MAX_LEVELS - 1))

// sigma of the Wendland C2 kernel in 3-D: W = SIGMA/H^3 (1-q)^4 (1+4q)   (reading Q3)
#define WC2_SIGMA 3.3422538049298023f     // 21 / (2 pi)

// ------------------------------------------------------------------------------------------
// tree walk: calls leaf(chunk) (warp-uniform) for every source chunk whose box is within reach
// ------------------------------------------------------------------------------------------
template <bool SYM>
__device__ __forceinline__ bool box_reach(float4 lo, float4 hi, float3 tlo, float3 thi, float tH)
{
    float gx = fmaxf(0.f, fmaxf(lo.x - thi.x, tlo.x - hi.x));
    float gy = fmaxf(0.f, fmaxf(lo.y - thi.y, tlo.y - hi.y));
    float gz = fmaxf(0.f, fmaxf(lo.z - thi.z, tlo.z - hi.z));
    float d2 = gx * gx + gy * gy + gz * gz;
    float R = SYM ? fmaxf(lo.w, tH) : tH;
    return d2 <= R * R * 1.00001f;        // conservative against the rounding of the exact predicate
}

template <bool SYM, class Leaf>
__device__ __forceinline__ void walk(const Tree &t, float3 tlo, float3 thi, float tH, unsigned *stack, Leaf &&leaf)
{
    const int lane = threadIdx.x & 31;
    int sp = 0;
    int L = t.nlev - 1, first = 0, cnt = t.count[L];
    while (true) {
        bool pass = false;
        if (lane < cnt) pass = box_reach<SYM>(t.lo[L][first + lane], t.hi[L][first + lane], tlo, thi, tH);
        unsigned mask = __ballot_sync(0xffffffffu, pass);
        if (L == 0) {
            while (mask) {
                int b = __ffs(mask) - 1;
                mask &= mask - 1;
                leaf(first + b);
            }
        } else {
            if (pass) stack[sp + __popc(mask & ((1u << lane) - 1u))] = ((unsigned)L << 27) | (unsigned)(first + lane);
            sp += __popc(mask);
            __syncwarp();
        }
        if (sp == 0) break;
        unsigned e = stack[--sp];
        __syncwarp();
        int pl = (int)(e >> 27);
        int idx = (int)(e & 0x7ffffffu);
        L = pl - 1;
        first = idx * SPH_ARITY;
        cnt = min(SPH_ARITY, t.count[L] - first);
    }
}

// ------------------------------------------------------------------------------------------
// S2 density: rho_i = sum_j m_j W_ij(h_i) (Eq. 1), Omega_i (Eq. 3), over r2 < H_i^2, self included.
//   W           = SIGMA/H^3 t^4 (1+4q),            t = 1-q
//   dW/dh       = -(3W + r dW/dr)/h = -SIGMA/(H^3 h) t^3 (3 + 9q - 32 q^2)
// so   rho = SIGMA/H^3 sum m t^4 (1+4q),   Omega = 1 - SIGMA/(3 rho H^3) sum m t^3 (3 + 9q - 32q^2).
// rho is evaluated and accumulated in fp64 for the TRUE neighbours only: P = c0^2 (rho - rho0)
// amplifies the relative error of rho by rho/(rho - rho0) ~ 100 on a lattice and Y = Y0 + mu_i P
// by another rho0 c0^2 / Y0 ~ 2400 (hard part 2), so even a correctly rounded
// fp32 rho misses the 1e-4 target on the yielded S.  B200 runs FP64 at half the FP32 rate, and the
// extra work is ~12 DFMA per true pair.  r comes from the fp32 rsqrt plus one Newton step in fp64.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_density(Dev d, float kappa)
{
    __shared__ float4 s_src[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = blockIdx.x * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) return;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float hi = valid ? d.r.vh[i].w : 1.f;
    float Hi = sph_H(kappa, hi);
    float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    float invH = 1.f / Hi;
    const double invHd = 1.0 / ((double)kappa * (double)hi);
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];
    double sum = 0.0;
    float sh = 0.f;
    int cnt_i = 0;
    unsigned long long tests = 0;
    const unsigned vmask = __ballot_sync(0xffffffffu, valid);

    walk<false>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_stack[warp],
                [&](int c) {
        long long j0 = (long long)c * SPH_CHUNK;
        int cnt = (int)min((long long)SPH_CHUNK, d.n - j0);
        if (lane < cnt) s_src[warp][lane] = d.r.pm[j0 + lane];
        __syncwarp();
        tests += (unsigned long long)cnt * __popc(vmask);
#pragma unroll 4
        for (int j = 0; j < cnt; ++j) {
            float4 q = s_src[warp][j];
            float dx = __fsub_rn(pi.x, q.x), dy = __fsub_rn(pi.y, q.y), dz = __fsub_rn(pi.z, q.z);
            float r2 = sph_r2(dx, dy, dz);
            if (r2 < H2i) {
                float rinv = rsqrtf(fmaxf(r2, 1.0e-37f));
                float r = r2 * rinv;
                float qq = r * invH;
                float t = fmaxf(0.f, 1.f - qq);
                float t3 = t * t * t;
                sh = fmaf(q.w * t3, fmaf(qq, fmaf(-32.f, qq, 9.f), 3.f), sh);
                // fp64 value of m_j t^4 (1 + 4q)
                double ex = (double)pi.x - (double)q.x, ey = (double)pi.y - (double)q.y, ez = (double)pi.z - (double)q.z;
                double r2d = fma(ex, ex, fma(ey, ey, ez * ez));
                double r0 = (double)r;
                double rd = fma(fma(-r0, r0, r2d), 0.5 * (double)rinv, r0);      // one Newton step for sqrt
                double qd = rd * invHd;
                double td = fmax(0.0, 1.0 - qd);
                double t2 = td * td;
                sum = fma((double)q.w * t2 * t2, fma(4.0, qd, 1.0), sum);
                ++cnt_i;
            }
        }
        __syncwarp();
    });

    if (valid) {
        float kw = WC2_SIGMA * invH * invH * invH;
        double rhod = 3.3422538049298023 * invHd * invHd * invHd * sum;
        float rho = (float)rhod;
        d.rho64[i] = rhod;
        d.rho[i] = rho;
        d.omega[i] = 1.f - kw * sh / (3.f * rho);
        d.ngather[i] = cnt_i;
    }
    // counters: true pairs and candidate tests
    unsigned long long hits = (unsigned long long)cnt_i;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, o);
    if (lane == 0) {
        atomicAdd(&d.counters[SPH_C_PAIRS_GATHER], hits);
        atomicAdd(&d.counters[SPH_C_TESTS_DENSITY], tests);
    }
}

// ------------------------------------------------------------------------------------------
// S4 + S5 fused (or either alone): over the symmetric set r2 < max(H_i^2, H_j^2), j != i.
//
// With D(h) = -(dW/dr)/r = K t^3, K = 20 SIGMA / H^5, grad_i W_ij(h) = -D x_ij:
//   F^{ab}    = +1/2 sum m_j (w_i D_i + w_j D_j) v_ij^a x_ij^b          (Eq. 20)
//   Cinv^{ab} = +1/2 sum m_j (w_i D_i + w_j D_j) x_ij^a x_ij^b          (Eq. 21, symmetric)
//   a_i       = - sum m_j D_i (st_i x_ij) - sum m_j D_j (st_j x_ij)      (Eq. 4 + 18, st = sigma/(Om rho^2))
//               + sum 1/2 m_j Pi_ij (D_i + D_j) x_ij  + a_ext            (Eq. 7)
//   du_i/dt   = + sum m_j D_i (st_i x_ij).v_ij                           (Eq. 19 + hydro analogue)
//               - sum 1/4 m_j Pi_ij (D_i + D_j) (v_ij.x_ij)              (Eq. 8)
// Per-source operands packed by k_predict:
//   A3 = {rho, c, K, 1/H}   A4 = {Sg_xx, Sg_yy, Sg_zz, Sg_xy}   A5 = {Sg_xz, Sg_yz, m w K, H^2}
// with Sg = m K st (so the j-side stress term is -t_j^3 Sg_j x_ij) and w = 1/(Omega rho).
// ------------------------------------------------------------------------------------------
template <bool GRAD, bool FORCE>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_pair(Dev d, DevParams p)
{
    __shared__ float4 s_src[PAIR_WARPS][5][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = blockIdx.x * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) return;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    const long long il = valid ? i : 0;
    const float4 pi = d.r.pm[il], vi = d.r.vh[il], a3 = d.A3[il], a4 = d.A4[il], a5 = d.A5[il];
    const float H2i = valid ? a5.w : -1.f;
    const float invHi = a3.w, Ki = a3.z, rhoi = a3.x, ci = a3.y, hi = vi.w;
    const float invm = 1.f / pi.w;
    const float wKi = a5.z * invm;                          // w_i K_i
    // K_i st_i (xx, yy, zz, xy, xz, yz)
    const float kxx = a4.x * invm, kyy = a4.y * invm, kzz = a4.z * invm, kxy = a4.w * invm, kxz = a5.x * invm,
                kyz = a5.y * invm;
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];

    float F[9], C[6];
#pragma unroll
    for (int k = 0; k < 9; ++k) F[k] = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) C[k] = 0.f;
    float ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, mumax = 0.f;
    int cnt_i = 0;
    unsigned long long tests = 0;
    const unsigned vmask = __ballot_sync(0xffffffffu, valid);

    walk<true>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_stack[warp],
               [&](int c) {
        long long j0 = (long long)c * SPH_CHUNK;
        int cnt = (int)min((long long)SPH_CHUNK, d.n - j0);
        if (lane < cnt) {
            s_src[warp][0][lane] = d.r.pm[j0 + lane];
            s_src[warp][1][lane] = d.r.vh[j0 + lane];
            s_src[warp][2][lane] = d.A3[j0 + lane];
            s_src[warp][3][lane] = d.A4[j0 + lane];
            s_src[warp][4][lane] = d.A5[j0 + lane];
        }
        __syncwarp();
        tests += (unsigned long long)cnt * __popc(vmask);
        for (int j = 0; j < cnt; ++j) {
            float4 s1 = s_src[warp][0][j];
            float4 s5 = s_src[warp][4][j];
            float dx = __fsub_rn(pi.x, s1.x), dy = __fsub_rn(pi.y, s1.y), dz = __fsub_rn(pi.z, s1.z);
            float r2 = sph_r2(dx, dy, dz);
            if (r2 < fmaxf(H2i, s5.w) && (j0 + j) != i) {
                float4 s2 = s_src[warp][1][j];
                float4 s3 = s_src[warp][2][j];
                float4 s4 = s_src[warp][3][j];
                ++cnt_i;
                float r = r2 * rsqrtf(fmaxf(r2, 1.0e-37f));
                float ti = fmaxf(0.f, 1.f - r * invHi);
                float tj = fmaxf(0.f, 1.f - r * s3.w);
                float ti3 = ti * ti * ti, tj3 = tj * tj * tj;
                float mj = s1.w;
                float dvx = vi.x - s2.x, dvy = vi.y - s2.y, dvz = vi.z - s2.z;
                float wi = mj * ti3;                                   // m_j t_i^3
                if (GRAD) {
                    float s = 0.5f * fmaf(wi, wKi, s5.z * tj3);        // 1/2 m_j (w_i D_i + w_j D_j)
                    float sx = s * dx, sy = s * dy, sz = s * dz;
                    F[0] = fmaf(dvx, sx, F[0]); F[1] = fmaf(dvx, sy, F[1]); F[2] = fmaf(dvx, sz, F[2]);
                    F[3] = fmaf(dvy, sx, F[3]); F[4] = fmaf(dvy, sy, F[4]); F[5] = fmaf(dvy, sz, F[5]);
                    F[6] = fmaf(dvz, sx, F[6]); F[7] = fmaf(dvz, sy, F[7]); F[8] = fmaf(dvz, sz, F[8]);
                    C[0] = fmaf(dx, sx, C[0]); C[1] = fmaf(dx, sy, C[1]); C[2] = fmaf(dx, sz, C[2]);
                    C[3] = fmaf(dy, sy, C[3]); C[4] = fmaf(dy, sz, C[4]); C[5] = fmaf(dz, sz, C[5]);
                }
                if (FORCE) {
                    // i side: z = K_i st_i x_ij
                    float zx = fmaf(kxx, dx, fmaf(kxy, dy, kxz * dz));
                    float zy = fmaf(kxy, dx, fmaf(kyy, dy, kyz * dz));
                    float zz = fmaf(kxz, dx, fmaf(kyz, dy, kzz * dz));
                    ax = fmaf(-wi, zx, ax); ay = fmaf(-wi, zy, ay); az = fmaf(-wi, zz, az);
                    du = fmaf(wi, fmaf(zx, dvx, fmaf(zy, dvy, zz * dvz)), du);
                    // j side: y = Sg_j x_ij
                    float yx = fmaf(s4.x, dx, fmaf(s4.w, dy, s5.x * dz));
                    float yy = fmaf(s4.w, dx, fmaf(s4.y, dy, s5.y * dz));
                    float yz = fmaf(s5.x, dx, fmaf(s5.y, dy, s4.z * dz));
                    ax = fmaf(-tj3, yx, ax); ay = fmaf(-tj3, yy, ay); az = fmaf(-tj3, yz, az);
                    // artificial viscosity, Eq. 5-8 (only approaching pairs: min(v.r, 0))
                    float vr = fminf(fmaf(dvx, dx, fmaf(dvy, dy, dvz * dz)), 0.f);
                    float hb = 0.5f * (hi + s2.w);
                    float mu = hb * vr / fmaf(p.eps_av * hb, hb, r2);
                    float Pi = mu * fmaf(p.beta, mu, -p.alpha * 0.5f * (ci + s3.y)) / (0.5f * (rhoi + s3.x));
                    float k = 0.5f * mj * Pi * fmaf(Ki, ti3, s3.z * tj3);
                    ax = fmaf(k, dx, ax); ay = fmaf(k, dy, ay); az = fmaf(k, dz, az);
                    du = fmaf(-0.5f * k, vr, du);
                    mumax = fmaxf(mumax, -mu);
                }
            }
        }
        __syncwarp();
    });

    if (valid) {
        if (GRAD) {
#pragma unroll
            for (int k = 0; k < 9; ++k) d.F[k][i] = F[k];
            d.Cinv[0][i] = C[0]; d.Cinv[1][i] = C[1]; d.Cinv[2][i] = C[2];
            d.Cinv[3][i] = C[1]; d.Cinv[4][i] = C[3]; d.Cinv[5][i] = C[4];
            d.Cinv[6][i] = C[2]; d.Cinv[7][i] = C[4]; d.Cinv[8][i] = C[5];
        }
        if (FORCE) {
            d.a[0][i] = ax + d.r.s[PP_G + 0][i];
            d.a[1][i] = ay + d.r.s[PP_G + 1][i];
            d.a[2][i] = az + d.r.s[PP_G + 2][i];
            d.dudt[i] = du;
            d.mumax[i] = mumax;
        }
        d.nsym[i] = cnt_i;
    }
    if (FORCE) {
        unsigned long long hits = (unsigned long long)cnt_i;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, o);
        if (lane == 0) {
            atomicAdd(&d.counters[SPH_C_PAIRS_SYMMETRIC], hits);
            atomicAdd(&d.counters[SPH_C_TESTS_FORCE], tests);
        }
    }
}

// ------------------------------------------------------------------------------------------
// test hook: neighbour sets as original ids
// ------------------------------------------------------------------------------------------
template <bool SYM>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_neighbors(Dev d, float kappa, int *counts,
                                                               const long long *offsets, int *list)
{
    __shared__ float4 s_src[PAIR_WARPS][SPH_CHUNK];
    __shared__ float s_H2[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_orig[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = blockIdx.x * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) return;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    const unsigned *orig = (const unsigned *)d.r.s[PP_ORIG];
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float Hi = sph_H(kappa, valid ? d.r.vh[i].w : 1.f);
    float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    unsigned oi = valid ? orig[i] : 0u;
    long long base = (valid && list) ? offsets[oi] : 0;
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];
    int cnt_i = 0;
    walk<SYM>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_stack[warp],
              [&](int c) {
        long long j0 = (long long)c * SPH_CHUNK;
        int cnt = (int)min((long long)SPH_CHUNK, d.n - j0);
        if (lane < cnt) {
            s_src[warp][lane] = d.r.pm[j0 + lane];
            float Hj = sph_H(kappa, d.r.vh[j0 + lane].w);
            s_H2[warp][lane] = __fmul_rn(Hj, Hj);
            s_orig[warp][lane] = orig[j0 + lane];
        }
        __syncwarp();
        for (int j = 0; j < cnt; ++j) {
            float4 q = s_src[warp][j];
            float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
            bool hit = SYM ? (r2 < fmaxf(H2i, s_H2[warp][j]) && (j0 + j) != i) : (r2 < H2i);
            if (hit) {
                if (list) list[base + cnt_i] = (int)s_orig[warp][j];
                ++cnt_i;
            }
        }
        __syncwarp();
    });
    if (valid) counts[oi] = cnt_i;
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
int sph_launch_density(sph_ctx *c)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_GATHER], 0, sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_DENSITY], 0, sizeof(unsigned long long), c->stream));
    if (d.n == 0) return SPH_OK;
    k_density<<<sph_div_up(d.nchunk, PAIR_WARPS), PAIR_WARPS * 32, 0, c->stream>>>(d, c->p.kappa);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_pair(sph_ctx *c, bool grad, bool force)
{
    Dev &d = c->d;
    if (force) {
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_SYMMETRIC], 0, sizeof(unsigned long long), c->stream));
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_FORCE], 0, sizeof(unsigned long long), c->stream));
    }
    if (d.n == 0) return SPH_OK;
    dim3 grid(sph_div_up(d.nchunk, PAIR_WARPS)), block(PAIR_WARPS * 32);
    if (grad && force) k_pair<true, true><<<grid, block, 0, c->stream>>>(d, c->p);
    else if (grad) k_pair<true, false><<<grid, block, 0, c->stream>>>(d, c->p);
    else k_pair<false, true><<<grid, block, 0, c->stream>>>(d, c->p);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_neighbors(sph_ctx *c, int which, int *counts, const long long *offsets, int *list)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    dim3 grid(sph_div_up(d.nchunk, PAIR_WARPS)), block(PAIR_WARPS * 32);
    if (which == SPH_SYMMETRIC) k_neighbors<true><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    else k_neighbors<false><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}
