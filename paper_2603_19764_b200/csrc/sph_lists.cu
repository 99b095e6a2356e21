// sph_lists.cu -- "v1" neighbour machinery: cull ONCE per step into compact lists, then let the
// pair passes evaluate true pairs only.
//
//   tile        = 16 consecutive chunks = 512 Morton-consecutive targets = one CTA of 16 warps.
//   k_cull      : per tile, (A) walk the chunk tree with the tile box, test every particle of the
//                 accepted source chunks against the tile's 16 chunk boxes and compact the survivors
//                 into the tile CANDIDATE LIST (global indices, ascending);  (B) every warp runs the
//                 candidates flagged for its chunk past its 32 targets (exact fp32 predicate,
//                 reading Q4) and appends the hits to each target's NEIGHBOUR LIST: u16 slot numbers
//                 into the tile candidate list, the symmetric set, self excluded.
//   k_density_l : stages {x,y,z,m} of the tile's candidates in shared memory (coalesced gathers of
//                 index runs), then every lane walks its own list.  The gather set is the subset of
//                 the symmetric list with r2 < H_i^2, plus the self term.
//   k_pair_l    : same with the five float4 operand streams of the fused gradient + force pass.
//
// Evidence for this design: profiles/r01_v0_launches_and_pair_kernel.md (candidate hit rate 3.5 %,
// 18.65 of 32 threads active per instruction in the broadcast-tile kernels).
#include "sph_internal.cuh"

#define WC2_SIGMA 3.3422538049298023f
#define STACK_DEPTH (SPH_ARITY * (SPH_MAX_LEVELS - 1))
#define FULL 0xffffffffu

// ------------------------------------------------------------------------------------------
// ascending tree walk (source chunks are reported in increasing index order)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ bool box_reach_sym(float4 lo, float4 hi, float3 tlo, float3 thi, float tH)
{
    float gx = fmaxf(0.f, fmaxf(lo.x - thi.x, tlo.x - hi.x));
    float gy = fmaxf(0.f, fmaxf(lo.y - thi.y, tlo.y - hi.y));
    float gz = fmaxf(0.f, fmaxf(lo.z - thi.z, tlo.z - hi.z));
    float d2 = gx * gx + gy * gy + gz * gz;
    float R = fmaxf(lo.w, tH);
    return d2 <= R * R * 1.00001f;
}

template <class Leaf>
__device__ __forceinline__ void walk_ascending(const Tree &t, float3 tlo, float3 thi, float tH, unsigned *stack, Leaf &&leaf)
{
    const int lane = threadIdx.x & 31;
    int sp = 0;
    int L = t.nlev - 1, first = 0, cnt = t.count[L];
    while (true) {
        bool pass = false;
        if (lane < cnt) pass = box_reach_sym(t.lo[L][first + lane], t.hi[L][first + lane], tlo, thi, tH);
        unsigned mask = __ballot_sync(FULL, pass);
        if (L == 0) {
            leaf(first, mask);
        } else {
            int np = __popc(mask);
            // push in reverse so that the lowest child is popped first
            if (pass) stack[sp + np - 1 - __popc(mask & ((1u << lane) - 1u))] = ((unsigned)L << 27) | (unsigned)(first + lane);
            sp += np;
            __syncwarp();
        }
        if (sp == 0) break;
        unsigned e = stack[--sp];
        __syncwarp();
        L = (int)(e >> 27) - 1;
        first = (int)(e & 0x7ffffffu) * SPH_ARITY;
        cnt = min(SPH_ARITY, t.count[L] - first);
    }
}

// ------------------------------------------------------------------------------------------
// k_cull
// ------------------------------------------------------------------------------------------
struct CullSmem {
    float4 pos[SPH_TILE_SC];             // x, y, z, H^2 of the candidates of the current round
    unsigned idx[SPH_TILE_SC];           // their global (sorted) indices
    unsigned short flag[SPH_TILE_SC];    // bit w: within reach of chunk w of the tile
    unsigned chunks[SPH_CULL_MAXSRC];    // accepted source chunks, ascending
    unsigned mask[SPH_CULL_MAXSRC];      // surviving lanes of each source chunk
    unsigned off[SPH_CULL_MAXSRC];       // exclusive prefix of popc(mask)
    unsigned short cmask[SPH_CULL_MAXSRC];   // which chunk boxes of the tile the source chunk box reaches
    float4 blo[SPH_TILE_CHUNKS], bhi[SPH_TILE_CHUNKS];
    unsigned stack[STACK_DEPTH];
    unsigned short buf[SPH_TILE_CHUNKS][8][SPH_CHUNK];   // per-warp append buffers (8 entries per lane)
    int nsrc, ntotal;
    unsigned long long pool_off;
};

// bits w of `among` whose chunk box is within reach of the point (x,y,z) with support Hj
__device__ __forceinline__ unsigned reach_flags(const CullSmem &sm, unsigned among, float x, float y, float z, float Hj)
{
    unsigned f = 0;
    while (among) {
        int w = __ffs(among) - 1;
        among &= among - 1;
        float4 lo = sm.blo[w], hi = sm.bhi[w];
        float gx = fmaxf(0.f, fmaxf(lo.x - x, x - hi.x));
        float gy = fmaxf(0.f, fmaxf(lo.y - y, y - hi.y));
        float gz = fmaxf(0.f, fmaxf(lo.z - z, z - hi.z));
        float d2 = gx * gx + gy * gy + gz * gz;
        float R = fmaxf(lo.w, Hj);
        if (d2 <= R * R * 1.00001f) f |= 1u << w;
    }
    return f;
}

__global__ void __launch_bounds__(SPH_TILE) k_cull(Dev d, float kappa)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CullSmem &sm = *reinterpret_cast<CullSmem *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x;
    const int chunk0 = tile * SPH_TILE_CHUNKS;
    const int nch = min(SPH_TILE_CHUNKS, d.nchunk - chunk0);

    if (threadIdx.x < nch) {
        sm.blo[threadIdx.x] = d.tree.lo[0][chunk0 + threadIdx.x];
        sm.bhi[threadIdx.x] = d.tree.hi[0][chunk0 + threadIdx.x];
    }
    __syncthreads();

    // ---- A1: warp 0 walks the tree with the tile box; a source chunk is accepted only if its box
    //          reaches at least one of the tile's chunk boxes (cmask) -----------------------------
    if (warp == 0) {
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, H = 0.f;
        if (lane < nch) {
            float4 a = sm.blo[lane], b = sm.bhi[lane];
            lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; H = a.w;
            hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(FULL, lo[a], o));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(FULL, hi[a], o));
            }
            H = fmaxf(H, __shfl_xor_sync(FULL, H, o));
        }
        int nsrc = 0;
        walk_ascending(d.tree, make_float3(lo[0], lo[1], lo[2]), make_float3(hi[0], hi[1], hi[2]), H, sm.stack,
                       [&](int first, unsigned mask) {
            unsigned cm = 0;
            if ((mask >> lane) & 1u) {
                float4 clo = d.tree.lo[0][first + lane], chi = d.tree.hi[0][first + lane];
                for (int w = 0; w < nch; ++w) {
                    float4 tl = sm.blo[w], th = sm.bhi[w];
                    if (box_reach_sym(clo, chi, make_float3(tl.x, tl.y, tl.z), make_float3(th.x, th.y, th.z), tl.w))
                        cm |= 1u << w;
                }
            }
            unsigned acc = __ballot_sync(FULL, cm != 0);
            int rank = __popc(acc & ((1u << lane) - 1u));
            if (cm != 0 && nsrc + rank < SPH_CULL_MAXSRC) {
                sm.chunks[nsrc + rank] = (unsigned)(first + lane);
                sm.cmask[nsrc + rank] = (unsigned short)cm;
            }
            nsrc += __popc(acc);
        });
        if (lane == 0) {
            if (nsrc > SPH_CULL_MAXSRC) { atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull); nsrc = SPH_CULL_MAXSRC; }
            sm.nsrc = nsrc;
        }
    }
    __syncthreads();
    const int nsrc = sm.nsrc;

    // ---- A2: which particles of the accepted source chunks reach a chunk box of the tile --------
    for (int k = warp; k < nsrc; k += SPH_TILE_CHUNKS) {
        long long j = (long long)sm.chunks[k] * SPH_CHUNK + lane;
        unsigned f = 0;
        if (j < d.n) {
            float4 q = d.r.pm[j];
            f = reach_flags(sm, sm.cmask[k], q.x, q.y, q.z, sph_H(kappa, d.r.vh[j].w));
        }
        unsigned m = __ballot_sync(FULL, f != 0);
        if (lane == 0) sm.mask[k] = m;
    }
    __syncthreads();
    if (warp == 0) {                                    // exclusive scan of popc(mask[0..nsrc))
        int per = (nsrc + 31) / 32, b0 = lane * per, local = 0;
        for (int k = b0; k < min(b0 + per, nsrc); ++k) local += __popc(sm.mask[k]);
        int incl = local;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int v = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += v;
        }
        int run = incl - local;
        for (int k = b0; k < min(b0 + per, nsrc); ++k) { sm.off[k] = (unsigned)run; run += __popc(sm.mask[k]); }
        if (lane == 31) {
            int total = incl;
            if (total > 65535) { atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull); total = 65535; }   // slots are u16
            unsigned long long o = atomicAdd(d.cand_cursor, (unsigned long long)total);
            if (o + (unsigned long long)total > d.cand_cap) {                 // candidate pool exhausted
                atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull);
                total = 0; o = 0;
            }
            sm.ntotal = total;
            sm.pool_off = o;
            d.tile_ncand[tile] = total;
            d.tile_off[tile] = o;
            atomicAdd(&d.counters[SPH_C_CANDIDATES], (unsigned long long)total);
        }
    }
    __syncthreads();
    const int ntotal = sm.ntotal;
    unsigned *cand = d.cand + sm.pool_off;

    // ---- per-target state for phase B -------------------------------------------------------------
    const long long i = (long long)(chunk0 + warp) * SPH_CHUNK + lane;
    const bool valid = warp < nch && i < d.n;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float Hi = sph_H(kappa, valid ? d.r.vh[i].w : 1.f);
    const float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    const unsigned wbit = 1u << warp;
    const int kcap = d.kcap;
    unsigned short *row = d.nbr + (size_t)(valid ? i : 0) * kcap;
    int cnt = 0;
    unsigned long long tests = 0;
    const int nvalid = __popc(__ballot_sync(FULL, valid));

    for (int r0 = 0; r0 < ntotal; r0 += SPH_TILE_SC) {
        const int nr = min(SPH_TILE_SC, ntotal - r0);
        // ---- A3: compact this round's survivors into shared memory (and the global candidate list)
        for (int k = warp; k < nsrc; k += SPH_TILE_CHUNKS) {
            unsigned m = sm.mask[k];
            int o = (int)sm.off[k];
            if (o >= r0 + nr || o + 32 <= r0) continue;          // (o + popc(m) <= o + 32)
            if (!((m >> lane) & 1u)) continue;
            int slot = o + __popc(m & ((1u << lane) - 1u)) - r0;
            if (slot < 0 || slot >= nr) continue;
            long long j = (long long)sm.chunks[k] * SPH_CHUNK + lane;
            float4 q = d.r.pm[j];
            float Hj = sph_H(kappa, d.r.vh[j].w);
            sm.pos[slot] = make_float4(q.x, q.y, q.z, __fmul_rn(Hj, Hj));
            sm.idx[slot] = (unsigned)j;
            sm.flag[slot] = (unsigned short)reach_flags(sm, sm.cmask[k], q.x, q.y, q.z, Hj);
            cand[r0 + slot] = (unsigned)j;
        }
        __syncthreads();
        // ---- B: every warp runs the candidates flagged for its chunk past its 32 targets ------------
        for (int base = 0; base < nr; base += 32) {
            int s = base + lane;
            unsigned m = __ballot_sync(FULL, s < nr && (sm.flag[s] & wbit));
            tests += (unsigned long long)__popc(m) * nvalid;
            while (m) {
                int b = __ffs(m) - 1;
                m &= m - 1;
                int slot = base + b;
                float4 q = sm.pos[slot];
                float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
                if (valid && r2 < fmaxf(H2i, q.w) && sm.idx[slot] != (unsigned)i) {
                    if (cnt < kcap) {
                        sm.buf[warp][cnt & 7][lane] = (unsigned short)(r0 + slot);
                        if ((cnt & 7) == 7) {
                            uint4 v;
                            v.x = sm.buf[warp][0][lane] | ((unsigned)sm.buf[warp][1][lane] << 16);
                            v.y = sm.buf[warp][2][lane] | ((unsigned)sm.buf[warp][3][lane] << 16);
                            v.z = sm.buf[warp][4][lane] | ((unsigned)sm.buf[warp][5][lane] << 16);
                            v.w = sm.buf[warp][6][lane] | ((unsigned)sm.buf[warp][7][lane] << 16);
                            *reinterpret_cast<uint4 *>(row + (cnt - 7)) = v;
                        }
                    }
                    ++cnt;
                }
            }
        }
        __syncthreads();
    }
    if (valid) {
        int stored = min(cnt, kcap);
        if (stored & 7) {                                  // partial last group (tail is never read)
            uint4 v;
            v.x = sm.buf[warp][0][lane] | ((unsigned)sm.buf[warp][1][lane] << 16);
            v.y = sm.buf[warp][2][lane] | ((unsigned)sm.buf[warp][3][lane] << 16);
            v.z = sm.buf[warp][4][lane] | ((unsigned)sm.buf[warp][5][lane] << 16);
            v.w = sm.buf[warp][6][lane] | ((unsigned)sm.buf[warp][7][lane] << 16);
            *reinterpret_cast<uint4 *>(row + (stored & ~7)) = v;
        }
        d.nsym[i] = stored;
        if (cnt > kcap) atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull);
    }
    if (lane == 0 && warp < nch) atomicAdd(&d.counters[SPH_C_TESTS_CULL], tests);
}

// entry k (0..7) of a group of eight u16 held in a uint4
__device__ __forceinline__ unsigned list_entry(const uint4 &v, int k)
{
    unsigned w = (k & 4) ? ((k & 2) ? v.w : v.z) : ((k & 2) ? v.y : v.x);
    return (k & 1) ? (w >> 16) : (w & 0xffffu);
}

// ------------------------------------------------------------------------------------------
// S2 density from the lists (fp64 accumulation as in k_density; see sph_pair.cu for why)
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SPH_TILE) k_density_l(Dev d, float kappa)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_pm = reinterpret_cast<float4 *>(smem_raw);
    const int tile = blockIdx.x;
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    const int lane = threadIdx.x & 31;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float hi = valid ? d.r.vh[i].w : 1.f;
    float Hi = sph_H(kappa, hi);
    const float H2i = __fmul_rn(Hi, Hi);
    const float invH = 1.f / Hi;
    const double invHd = 1.0 / ((double)kappa * (double)hi);
    const int cnt = valid ? d.nsym[i] : 0;
    const uint4 *row = reinterpret_cast<const uint4 *>(d.nbr + (size_t)(valid ? i : 0) * d.kcap);
    // self term: q = 0, t = 1
    double sum = (double)pi.w;
    float sh = 3.f * pi.w;
    int ng = 1;
    int k = 0;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (cnt > 0) v = row[0];
    for (int r0 = 0; r0 < ncand || r0 == 0; r0 += SPH_TILE_SC) {
        const int nr = min(SPH_TILE_SC, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) s_pm[s] = d.r.pm[cand[r0 + s]];
        __syncthreads();
        const int lim = r0 + nr;
        while (k < cnt) {
            int slot = (int)list_entry(v, k & 7);
            if (slot >= lim) break;
            ++k;
            if ((k & 7) == 0 && k < cnt) v = row[k >> 3];
            float4 q = s_pm[slot - r0];
            float dx = __fsub_rn(pi.x, q.x), dy = __fsub_rn(pi.y, q.y), dz = __fsub_rn(pi.z, q.z);
            float r2 = sph_r2(dx, dy, dz);
            if (r2 < H2i) {
                float rinv = rsqrtf(fmaxf(r2, 1.0e-37f));
                float r = r2 * rinv;
                float qq = r * invH;
                float t = fmaxf(0.f, 1.f - qq);
                float t3 = t * t * t;
                sh = fmaf(q.w * t3, fmaf(qq, fmaf(-32.f, qq, 9.f), 3.f), sh);
                double ex = (double)pi.x - (double)q.x, ey = (double)pi.y - (double)q.y, ez = (double)pi.z - (double)q.z;
                double r2d = fma(ex, ex, fma(ey, ey, ez * ez));
                double r0d = (double)r;
                double rd = fma(fma(-r0d, r0d, r2d), 0.5 * (double)rinv, r0d);
                double qd = rd * invHd;
                double td = fmax(0.0, 1.0 - qd);
                double t2 = td * td;
                sum = fma((double)q.w * t2 * t2, fma(4.0, qd, 1.0), sum);
                ++ng;
            }
        }
        __syncthreads();
    }
    if (valid) {
        float kw = WC2_SIGMA * invH * invH * invH;
        double rhod = 3.3422538049298023 * invHd * invHd * invHd * sum;
        float rho = (float)rhod;
        d.rho64[i] = rhod;
        d.rho[i] = rho;
        d.omega[i] = 1.f - kw * sh / (3.f * rho);
        d.ngather[i] = ng;
    }
    unsigned long long hits = valid ? (unsigned long long)ng : 0ull, tests = valid ? (unsigned long long)cnt + 1ull : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        hits += __shfl_xor_sync(FULL, hits, o);
        tests += __shfl_xor_sync(FULL, tests, o);
    }
    if (lane == 0) {
        atomicAdd(&d.counters[SPH_C_PAIRS_GATHER], hits);
        atomicAdd(&d.counters[SPH_C_TESTS_DENSITY], tests);
    }
}

// ------------------------------------------------------------------------------------------
// S4 + S5 from the lists.  Equations and operand packing: see k_pair in sph_pair.cu.
// The tile's candidates are staged in rounds of SPH_PAIR_SE slots; lists are ascending in slot,
// so each lane just advances a cursor.
// ------------------------------------------------------------------------------------------
template <bool GRAD, bool FORCE>
__global__ void __launch_bounds__(SPH_TILE) k_pair_l(Dev d, DevParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s1 = reinterpret_cast<float4 *>(smem_raw);
    float4 *s2 = s1 + SPH_PAIR_SE, *s3 = s2 + SPH_PAIR_SE, *s4 = s3 + SPH_PAIR_SE, *s5 = s4 + SPH_PAIR_SE;
    const int tile = blockIdx.x;
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const int lane = threadIdx.x & 31;
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    const long long il = valid ? i : 0;
    const float4 pi = d.r.pm[il], vi = d.r.vh[il], a3 = d.A3[il], a4 = d.A4[il], a5 = d.A5[il];
    const float invHi = a3.w, Ki = a3.z, rhoi = a3.x, ci = a3.y, hi = vi.w;
    const float invm = 1.f / pi.w;
    const float wKi = a5.z * invm;
    const float kxx = a4.x * invm, kyy = a4.y * invm, kzz = a4.z * invm, kxy = a4.w * invm, kxz = a5.x * invm,
                kyz = a5.y * invm;
    const int cnt = valid ? d.nsym[i] : 0;
    const uint4 *row = reinterpret_cast<const uint4 *>(d.nbr + (size_t)il * d.kcap);

    float F[9], C[6];
#pragma unroll
    for (int k = 0; k < 9; ++k) F[k] = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) C[k] = 0.f;
    float ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, mumax = 0.f;
    int k = 0;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (cnt > 0) v = row[0];

    for (int r0 = 0; r0 < ncand || r0 == 0; r0 += SPH_PAIR_SE) {
        const int nr = min(SPH_PAIR_SE, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) {
            unsigned j = cand[r0 + s];
            s1[s] = d.r.pm[j];
            s2[s] = d.r.vh[j];
            s3[s] = d.A3[j];
            s4[s] = d.A4[j];
            s5[s] = d.A5[j];
        }
        __syncthreads();
        const int lim = r0 + nr;
        while (k < cnt) {
            int slot = (int)list_entry(v, k & 7);
            if (slot >= lim) break;
            slot -= r0;
            ++k;
            if ((k & 7) == 0 && k < cnt) v = row[k >> 3];
            const float4 q1 = s1[slot], q2 = s2[slot], q3 = s3[slot], q4 = s4[slot], q5 = s5[slot];
            float dx = __fsub_rn(pi.x, q1.x), dy = __fsub_rn(pi.y, q1.y), dz = __fsub_rn(pi.z, q1.z);
            float r2 = sph_r2(dx, dy, dz);
            float r = r2 * rsqrtf(fmaxf(r2, 1.0e-37f));
            float ti = fmaxf(0.f, 1.f - r * invHi);
            float tj = fmaxf(0.f, 1.f - r * q3.w);
            float ti3 = ti * ti * ti, tj3 = tj * tj * tj;
            float mj = q1.w;
            float dvx = vi.x - q2.x, dvy = vi.y - q2.y, dvz = vi.z - q2.z;
            float wi = mj * ti3;
            if (GRAD) {
                float s = 0.5f * fmaf(wi, wKi, q5.z * tj3);
                float sx = s * dx, sy = s * dy, sz = s * dz;
                F[0] = fmaf(dvx, sx, F[0]); F[1] = fmaf(dvx, sy, F[1]); F[2] = fmaf(dvx, sz, F[2]);
                F[3] = fmaf(dvy, sx, F[3]); F[4] = fmaf(dvy, sy, F[4]); F[5] = fmaf(dvy, sz, F[5]);
                F[6] = fmaf(dvz, sx, F[6]); F[7] = fmaf(dvz, sy, F[7]); F[8] = fmaf(dvz, sz, F[8]);
                C[0] = fmaf(dx, sx, C[0]); C[1] = fmaf(dx, sy, C[1]); C[2] = fmaf(dx, sz, C[2]);
                C[3] = fmaf(dy, sy, C[3]); C[4] = fmaf(dy, sz, C[4]); C[5] = fmaf(dz, sz, C[5]);
            }
            if (FORCE) {
                float zx = fmaf(kxx, dx, fmaf(kxy, dy, kxz * dz));
                float zy = fmaf(kxy, dx, fmaf(kyy, dy, kyz * dz));
                float zz = fmaf(kxz, dx, fmaf(kyz, dy, kzz * dz));
                ax = fmaf(-wi, zx, ax); ay = fmaf(-wi, zy, ay); az = fmaf(-wi, zz, az);
                du = fmaf(wi, fmaf(zx, dvx, fmaf(zy, dvy, zz * dvz)), du);
                float yx = fmaf(q4.x, dx, fmaf(q4.w, dy, q5.x * dz));
                float yy = fmaf(q4.w, dx, fmaf(q4.y, dy, q5.y * dz));
                float yz = fmaf(q5.x, dx, fmaf(q5.y, dy, q4.z * dz));
                ax = fmaf(-tj3, yx, ax); ay = fmaf(-tj3, yy, ay); az = fmaf(-tj3, yz, az);
                float vr = fminf(fmaf(dvx, dx, fmaf(dvy, dy, dvz * dz)), 0.f);
                float hb = 0.5f * (hi + q2.w);
                float mu = __fdividef(hb * vr, fmaf(p.eps_av * hb, hb, r2));
                float Pi = __fdividef(mu * fmaf(p.beta, mu, -p.alpha * 0.5f * (ci + q3.y)), 0.5f * (rhoi + q3.x));
                float kk = 0.5f * mj * Pi * fmaf(Ki, ti3, q3.z * tj3);
                ax = fmaf(kk, dx, ax); ay = fmaf(kk, dy, ay); az = fmaf(kk, dz, az);
                du = fmaf(-0.5f * kk, vr, du);
                mumax = fmaxf(mumax, -mu);
            }
        }
        __syncthreads();
    }

    if (valid) {
        if (GRAD) {
#pragma unroll
            for (int c = 0; c < 9; ++c) d.F[c][i] = F[c];
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
    }
    if (FORCE) {
        unsigned long long hits = (unsigned long long)cnt;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(FULL, hits, o);
        if (lane == 0) {
            atomicAdd(&d.counters[SPH_C_PAIRS_SYMMETRIC], hits);
            atomicAdd(&d.counters[SPH_C_TESTS_FORCE], hits);
        }
    }
}

// ------------------------------------------------------------------------------------------
// test hook from the lists
// ------------------------------------------------------------------------------------------
template <bool SYM>
__global__ void __launch_bounds__(256) k_neighbors_l(Dev d, float kappa, int *counts, const long long *offsets, int *list)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const unsigned *orig = (const unsigned *)d.r.s[PP_ORIG];
    const unsigned *cand = d.cand + d.tile_off[i / SPH_TILE];
    const unsigned short *row = d.nbr + (size_t)i * d.kcap;
    const int cnt = d.nsym[i];
    unsigned oi = orig[i];
    long long base = list ? offsets[oi] : 0;
    float4 pi = d.r.pm[i];
    float Hi = sph_H(kappa, d.r.vh[i].w);
    float H2i = __fmul_rn(Hi, Hi);
    int out = 0;
    if (!SYM) {
        if (list) list[base] = (int)oi;
        out = 1;
    }
    for (int k = 0; k < cnt; ++k) {
        unsigned j = cand[row[k]];
        bool hit = true;
        if (!SYM) {
            float4 q = d.r.pm[j];
            hit = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z)) < H2i;
        }
        if (hit) {
            if (list) list[base + out] = (int)orig[j];
            ++out;
        }
    }
    counts[oi] = out;
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
static int set_smem(sph_ctx *c, const void *fn, size_t bytes)
{
    SPH_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return SPH_OK;
}

int sph_launch_cull(sph_ctx *c)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_CULL], 0, 3 * sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(d.cand_cursor, 0, sizeof(unsigned long long), c->stream));
    if (d.n == 0) return SPH_OK;
    int rc = set_smem(c, (const void *)k_cull, sizeof(CullSmem));
    if (rc) return rc;
    k_cull<<<sph_div_up(d.nchunk, SPH_TILE_CHUNKS), SPH_TILE, sizeof(CullSmem), c->stream>>>(d, c->p.kappa);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_density_l(sph_ctx *c)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_GATHER], 0, sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_DENSITY], 0, sizeof(unsigned long long), c->stream));
    if (d.n == 0) return SPH_OK;
    size_t bytes = (size_t)SPH_TILE_SC * sizeof(float4);
    int rc = set_smem(c, (const void *)k_density_l, bytes);
    if (rc) return rc;
    k_density_l<<<sph_div_up(d.nchunk, SPH_TILE_CHUNKS), SPH_TILE, bytes, c->stream>>>(d, c->p.kappa);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_pair_l(sph_ctx *c, bool grad, bool force)
{
    Dev &d = c->d;
    if (force) {
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_SYMMETRIC], 0, sizeof(unsigned long long), c->stream));
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_FORCE], 0, sizeof(unsigned long long), c->stream));
    }
    if (d.n == 0) return SPH_OK;
    size_t bytes = (size_t)5 * SPH_PAIR_SE * sizeof(float4);
    dim3 grid(sph_div_up(d.nchunk, SPH_TILE_CHUNKS)), block(SPH_TILE);
    int rc;
    if (grad && force) {
        if ((rc = set_smem(c, (const void *)k_pair_l<true, true>, bytes))) return rc;
        k_pair_l<true, true><<<grid, block, bytes, c->stream>>>(d, c->p);
    } else if (grad) {
        if ((rc = set_smem(c, (const void *)k_pair_l<true, false>, bytes))) return rc;
        k_pair_l<true, false><<<grid, block, bytes, c->stream>>>(d, c->p);
    } else {
        if ((rc = set_smem(c, (const void *)k_pair_l<false, true>, bytes))) return rc;
        k_pair_l<false, true><<<grid, block, bytes, c->stream>>>(d, c->p);
    }
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_neighbors_l(sph_ctx *c, int which, int *counts, const long long *offsets, int *list)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    int nb = sph_div_up(d.n, 256);
    if (which == SPH_SYMMETRIC) k_neighbors_l<true><<<nb, 256, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    else k_neighbors_l<false><<<nb, 256, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}
