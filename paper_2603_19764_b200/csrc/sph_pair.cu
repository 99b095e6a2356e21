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
#include "sph_pairterm.cuh"

#define PAIR_WARPS SPH_TILE_CHUNKS        // warps (= target chunks) per CTA: one CTA serves one tile
#define STACK_DEPTH (SPH_ARITY * (SPH_MAX_LEVELS - 1))

// These are the round-1 "v0" kernels.  They have no capacity limits, so they also serve the tiles
// that k_cull (sph_lists.cu) flags because a list capacity was exceeded: launched with a tile_flag
// array they visit only the flagged tiles (persistent CTAs), with tile_flag == nullptr every tile.
#define WC2_SIGMA SPH_WC2_SIGMA

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

// EXACT: a node must also be within reach of one of the warp's 32 TARGET PARTICLES (tgt[t] = {x, y, z, H},
// H < 0: no particle), not only of their bounding box.  Thirty times the work per node, which pays for the
// chunks this path exists for: a chunk that straddles a gap of the space-filling curve has a box that
// covers the gap, and the box test alone would accept every source chunk in it.
template <bool SYM, bool EXACT>
__device__ __forceinline__ bool node_reach(float4 lo, float4 hi, float3 tlo, float3 thi, float tH, const float4 *tgt)
{
    bool pass = box_reach<SYM>(lo, hi, tlo, thi, tH);
    if (!EXACT || !pass) return pass;
    for (int t = 0; t < SPH_CHUNK; ++t) {
        const float4 q = tgt[t];
        if (q.w < 0.f) continue;
        float gx = fmaxf(0.f, fmaxf(lo.x - q.x, q.x - hi.x));
        float gy = fmaxf(0.f, fmaxf(lo.y - q.y, q.y - hi.y));
        float gz = fmaxf(0.f, fmaxf(lo.z - q.z, q.z - hi.z));
        float R = SYM ? fmaxf(lo.w, q.w) : q.w;
        if (gx * gx + gy * gy + gz * gz <= R * R * 1.00001f) return true;
    }
    return false;
}

template <bool SYM, bool EXACT, class Leaf>
__device__ __forceinline__ void walk(const Tree &t, float3 tlo, float3 thi, float tH, const float4 *tgt, unsigned *stack,
                                     Leaf &&leaf)
{
    const int lane = threadIdx.x & 31;
    int sp = 0;
    int L = t.nlev - 1, first = 0, cnt = t.count[L];
    while (true) {
        bool pass = false;
        if (lane < cnt) pass = node_reach<SYM, EXACT>(t.lo[L][first + lane], t.hi[L][first + lane], tlo, thi, tH, tgt);
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
// Arithmetic: density_term (sph_pairterm.cuh), the same as in the list-driven kernel.
// ------------------------------------------------------------------------------------------
template <bool EXACT>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_density(Dev d, float kappa, const unsigned char *__restrict__ tile_flag, int ntile)
{
    __shared__ float4 s_src[PAIR_WARPS][SPH_CHUNK];
    __shared__ float4 s_tgt[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (tile_flag && d.counters[SPH_C_LIST_OVERFLOW] == 0ull) return;       // serving flagged tiles: there are none
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    if (tile_flag && !tile_flag[tile]) continue;
    const int chunk = tile * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) continue;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float hi = valid ? d.r.vh[i].w : 1.f;
    float Hi = sph_H(kappa, hi);
    float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    float invH = 1.f / Hi;
    const double invHd = 1.0 / ((double)kappa * (double)hi);
    const double pxd = (double)pi.x, pyd = (double)pi.y, pzd = (double)pi.z;
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];
    DensAcc A;
    A.sum = 0.0; A.sh = 0.0; A.n = 0;                  // the walk meets the particle itself (r2 = 0)
    unsigned long long tests = 0;
    const unsigned vmask = __ballot_sync(0xffffffffu, valid);
    if (EXACT) {
        s_tgt[warp][lane] = make_float4(pi.x, pi.y, pi.z, valid ? Hi : -1.f);
        __syncwarp();
    }

    walk<false, EXACT>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_tgt[warp],
                       s_stack[warp], [&](int c) {
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
            if (r2 < H2i)
                density_term(A, r2, pxd - (double)q.x, pyd - (double)q.y, pzd - (double)q.z, (double)q.w, invHd);
        }
        __syncwarp();
    });

    unsigned small = 0u;
    if (valid) {
        double rhod;
        float rho, om;
        density_finish(A, invH, invHd, rhod, rho, om);
        d.rho64[i] = rhod;
        d.rho[i] = rho;
        d.omega[i] = om;
        d.ngather[i] = A.n;
        d.mK[i] = sph_mK(pi.w, invH);
        small = fabsf(om) < 0.1f ? 1u : 0u;
    }
    small = __popc(__ballot_sync(0xffffffffu, small != 0u));
    // counters: true pairs and candidate tests
    unsigned long long hits = (unsigned long long)A.n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, o);
    if (lane == 0) {
        atomicAdd(&d.counters[SPH_C_PAIRS_GATHER], hits);
        atomicAdd(&d.counters[SPH_C_TESTS_DENSITY], tests);
        if (small) atomicAdd(&d.counters[SPH_C_OMEGA_SMALL], (unsigned long long)small);
    }
    }   // tile loop
}

// ------------------------------------------------------------------------------------------
// S4 + S5 fused (or either alone): over the symmetric set r2 < max(H_i^2, H_j^2), j != i.
// Equations and operand packing: sph_pairterm.cuh.
// ------------------------------------------------------------------------------------------
template <bool GRAD, bool FORCE, bool EXACT>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_pair(Dev d, DevParams p, const unsigned char *__restrict__ tile_flag, int ntile, RungCtl rc)
{
    __shared__ float4 s_src[PAIR_WARPS][4][SPH_CHUNK];
    __shared__ float2 s_src5[PAIR_WARPS][SPH_CHUNK];
    __shared__ float4 s_tgt[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const PairConst kc = pair_const(p.alpha, p.beta, p.eps_av, p.kappa);
    if (tile_flag && d.counters[SPH_C_LIST_OVERFLOW] == 0ull) return;       // serving flagged tiles: there are none
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    if (tile_flag && !tile_flag[tile]) continue;
    const int chunk = tile * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) continue;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    const long long il = valid ? i : 0;
    const PairTarget t = pair_target_load(d, il, p.kappa);
    const float H2i = valid ? __fmul_rn(t.H, t.H) : -1.f;
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];
    PairAcc A;
    pair_acc_zero(A);
    int cnt_i = 0;
    unsigned long long tests = 0;
    const unsigned vmask = __ballot_sync(0xffffffffu, valid);
    if (EXACT) {
        s_tgt[warp][lane] = make_float4(t.x, t.y, t.z, valid ? t.H : -1.f);
        __syncwarp();
    }

    walk<true, EXACT>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_tgt[warp],
                      s_stack[warp], [&](int c) {
        long long j0 = (long long)c * SPH_CHUNK;
        int cnt = (int)min((long long)SPH_CHUNK, d.n - j0);
        if (lane < cnt) {
            float4 vh = d.r.vh[j0 + lane];
            vh.w = sph_H(p.kappa, vh.w);
            s_src[warp][0][lane] = d.r.pm[j0 + lane];
            s_src[warp][1][lane] = vh;
            s_src[warp][2][lane] = d.B3[j0 + lane];
            s_src[warp][3][lane] = d.B4[j0 + lane];
            s_src5[warp][lane] = d.B5[j0 + lane];
        }
        __syncwarp();
        tests += (unsigned long long)cnt * __popc(vmask);
        for (int j = 0; j < cnt; ++j) {
            float4 q1 = s_src[warp][0][j];
            float4 q2 = s_src[warp][1][j];
            float dx = __fsub_rn(t.x, q1.x), dy = __fsub_rn(t.y, q1.y), dz = __fsub_rn(t.z, q1.z);
            float r2 = sph_r2(dx, dy, dz);
            if (r2 < fmaxf(H2i, __fmul_rn(q2.w, q2.w)) && (j0 + j) != i) {
                ++cnt_i;
                pair_term<GRAD, FORCE>(t, kc, A, q1, q2, s_src[warp][2][j], s_src[warp][3][j], s_src5[warp][j], true);
            }
        }
        __syncwarp();
    });

    const bool keep = valid && sph_active(rc, i);          // NEXT-4: an inactive particle keeps its old derivatives
    if (keep) {
        pair_store<GRAD, FORCE>(d, i, A, kc, !(p.flags & SPH_INT_DEFER_AEXT));
        d.nsym[i] = cnt_i;
    }
    if (FORCE) {
        unsigned long long hits = keep ? (unsigned long long)cnt_i : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, o);
        if (lane == 0) {
            atomicAdd(&d.counters[SPH_C_PAIRS_SYMMETRIC], hits);
            atomicAdd(&d.counters[SPH_C_TESTS_FORCE], tests);
        }
    }
    }   // tile loop
}

// ------------------------------------------------------------------------------------------
// test hook: neighbour sets as original ids
// ------------------------------------------------------------------------------------------
template <bool SYM, bool EXACT>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_neighbors(Dev d, float kappa, int *counts, const long long *offsets,
                                                               int *list, const unsigned char *__restrict__ tile_flag, int ntile)
{
    __shared__ float4 s_src[PAIR_WARPS][SPH_CHUNK];
    __shared__ float s_H2[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_orig[PAIR_WARPS][SPH_CHUNK];
    __shared__ float4 s_tgt[PAIR_WARPS][SPH_CHUNK];
    __shared__ unsigned s_stack[PAIR_WARPS][STACK_DEPTH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (tile_flag && d.counters[SPH_C_LIST_OVERFLOW] == 0ull) return;       // serving flagged tiles: there are none
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    if (tile_flag && !tile_flag[tile]) continue;
    const int chunk = tile * PAIR_WARPS + warp;
    if (chunk >= d.nchunk) continue;
    const long long i = (long long)chunk * SPH_CHUNK + lane;
    const bool valid = i < d.n;
    const unsigned *orig = (const unsigned *)d.r.s[PP_ORIG];
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float Hi = sph_H(kappa, valid ? d.r.vh[i].w : 1.f);
    float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    unsigned oi = valid ? orig[i] : 0u;
    long long base = (valid && list) ? offsets[oi] : 0;
    const bool want = list && base >= 0;                 // offsets[i] < 0: this particle's ids are not wanted
    float4 blo = d.tree.lo[0][chunk], bhi = d.tree.hi[0][chunk];
    int cnt_i = 0;
    if (EXACT) {
        s_tgt[warp][lane] = make_float4(pi.x, pi.y, pi.z, valid ? Hi : -1.f);
        __syncwarp();
    }
    walk<SYM, EXACT>(d.tree, make_float3(blo.x, blo.y, blo.z), make_float3(bhi.x, bhi.y, bhi.z), blo.w, s_tgt[warp],
                     s_stack[warp], [&](int c) {
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
                if (want) list[base + cnt_i] = (int)s_orig[warp][j];
                ++cnt_i;
            }
        }
        __syncwarp();
    });
    if (valid) counts[oi] = cnt_i;
    }   // tile loop
}

// ------------------------------------------------------------------------------------------
// launchers.  flagged_only: visit only the tiles k_cull flagged (persistent grid); the counters of
// the pass were already reset by the list-driven launcher that ran just before.
// ------------------------------------------------------------------------------------------
static inline int walk_grid_of(const Dev &d, bool flagged_only, int ntile)
{
    return flagged_only ? (ntile < d.walk_grid ? ntile : d.walk_grid) : ntile;
}

int sph_launch_density(sph_ctx *c, bool flagged_only)
{
    Dev &d = c->d;
    if (!flagged_only) {
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_GATHER], 0, sizeof(unsigned long long), c->stream));
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_DENSITY], 0, sizeof(unsigned long long), c->stream));
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_OMEGA_SMALL], 0, sizeof(unsigned long long), c->stream));
    }
    if (d.n == 0) return SPH_OK;
    const int ntile = sph_div_up(d.nchunk, PAIR_WARPS);
    if (flagged_only)
        k_density<true><<<walk_grid_of(d, true, ntile), PAIR_WARPS * 32, 0, c->stream>>>(d, c->p.kappa, d.tile_flag, ntile);
    else
        k_density<false><<<ntile, PAIR_WARPS * 32, 0, c->stream>>>(d, c->p.kappa, nullptr, ntile);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_pair(sph_ctx *c, bool grad, bool force, bool flagged_only)
{
    Dev &d = c->d;
    if (force && !flagged_only) {
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_SYMMETRIC], 0, sizeof(unsigned long long), c->stream));
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_FORCE], 0, sizeof(unsigned long long), c->stream));
    }
    if (d.n == 0) return SPH_OK;
    const int ntile = sph_div_up(d.nchunk, PAIR_WARPS);
    dim3 grid(walk_grid_of(d, flagged_only, ntile)), block(PAIR_WARPS * 32);
    const unsigned char *tf = flagged_only ? d.tile_flag : nullptr;
    if (flagged_only) {
        if (grad && force) k_pair<true, true, true><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
        else if (grad) k_pair<true, false, true><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
        else k_pair<false, true, true><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
    } else {
        if (grad && force) k_pair<true, true, false><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
        else if (grad) k_pair<true, false, false><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
        else k_pair<false, true, false><<<grid, block, 0, c->stream>>>(d, c->p, tf, ntile, c->rc);
    }
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_neighbors(sph_ctx *c, int which, int *counts, const long long *offsets, int *list, bool flagged_only)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    const int ntile = sph_div_up(d.nchunk, PAIR_WARPS);
    dim3 grid(walk_grid_of(d, flagged_only, ntile)), block(PAIR_WARPS * 32);
    const unsigned char *tf = flagged_only ? d.tile_flag : nullptr;
    if (flagged_only) {
        if (which == SPH_SYMMETRIC) k_neighbors<true, true><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list, tf, ntile);
        else k_neighbors<false, true><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list, tf, ntile);
    } else {
        if (which == SPH_SYMMETRIC) k_neighbors<true, false><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list, tf, ntile);
        else k_neighbors<false, false><<<grid, block, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list, tf, ntile);
    }
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}
