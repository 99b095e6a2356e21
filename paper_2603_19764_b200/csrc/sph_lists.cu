// sph_lists.cu -- "v1" neighbour machinery: cull ONCE per step into compact lists, then let the
// pair passes evaluate true pairs only.
//
//   tile        = 16 consecutive chunks = 512 Hilbert-consecutive targets = one CTA of 16 warps.
//   k_cull      : persistent CTAs, one tile at a time:
//                 (A) breadth-first walk of the chunk tree by all warps; every particle of the accepted
//                     source chunks is tested against the tile's 16 chunk boxes; the survivors are
//                     compacted into the tile CANDIDATE LIST (global indices, ascending) together with
//                     a 16-bit FLAG word (bit w: within reach of chunk w of the tile);
//                 (B) warp w runs the candidates flagged for its chunk, in slot order, past its 32
//                     targets (exact fp32 predicate, reading Q4).  The k-th flagged candidate is bit k
//                     of each target's NEIGHBOUR MASK: a dense bitmask (~18 % set, ~14 words per
//                     target) emitted word by word straight from the test loop -- no append, no decode,
//                     no per-particle capacity.  The symmetric set, self excluded.
//   k_density_l : stages {x,y,z,m} of the tile's candidates in shared memory (coalesced gathers of
//                 index runs); every warp rebuilds its k -> slot table from the flags, then every lane
//                 walks the set bits of its own mask.  The gather set is the subset of the symmetric
//                 set with r2 < H_i^2, plus the self term.
//   k_pair_l    : same with the five float4 operand streams of the fused gradient + force pass.
//
// Evidence for this design: profiles/r01_v0_launches_and_pair_kernel.md (candidate hit rate 3.5 %,
// 18.65 of 32 threads active per instruction in the broadcast-tile kernels) and
// profiles/r01_cull_iterations.md (append / decode variants of the list build).
#include "sph_internal.cuh"

#define WC2_SIGMA 3.3422538049298023f
#define FULL 0xffffffffu

__device__ __forceinline__ bool box_reach_sym(float4 lo, float4 hi, float3 tlo, float3 thi, float tH)
{
    float gx = fmaxf(0.f, fmaxf(lo.x - thi.x, tlo.x - hi.x));
    float gy = fmaxf(0.f, fmaxf(lo.y - thi.y, tlo.y - hi.y));
    float gz = fmaxf(0.f, fmaxf(lo.z - thi.z, tlo.z - hi.z));
    float d2 = gx * gx + gy * gy + gz * gz;
    float R = fmaxf(lo.w, tH);
    return d2 <= R * R * 1.00001f;        // conservative against the rounding of the exact predicate
}

// ------------------------------------------------------------------------------------------
// k_cull
// ------------------------------------------------------------------------------------------
struct CullSmem {
    float4 pos[SPH_TILE_SC];             // x, y, z, H^2 of the candidates of the current round
    unsigned short flag[SPH_TILE_SC];    // bit w: within reach of chunk w of the tile
    unsigned chunks[SPH_CULL_MAXSRC];    // frontier / accepted source chunks, ascending
    unsigned next[SPH_CULL_MAXSRC];      // next frontier
    unsigned mask[SPH_CULL_MAXSRC];      // surviving lanes (children / particles) of each entry
    unsigned off[SPH_CULL_MAXSRC];       // exclusive prefix of popc(mask)
    unsigned short cmask[SPH_CULL_MAXSRC];       // chunk boxes of the tile a source chunk box reaches
    unsigned short ctmp[SPH_CULL_MAXPAR][SPH_ARITY];   // per-child cmask of the leaf expansion
    float4 blo[SPH_TILE_CHUNKS], bhi[SPH_TILE_CHUNKS];
    float4 tlo, thi;                     // tile box (tlo.w = max H)
    unsigned selfslot[SPH_TILE];         // slot of each target of the tile in its own candidate list
    unsigned wcount[SPH_TILE_CHUNKS];    // candidates flagged for each chunk of the tile
    int nsrc, ntotal, nfront, overflow, nwm;
    unsigned long long cand_off, mask_off;
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

// warp 0: off[k] = exclusive prefix of popc(mask[k]), k < n; returns the total (valid in every lane)
__device__ __forceinline__ int scan_popc(const unsigned *mask, unsigned *off, int n, int lane)
{
    int per = (n + 31) / 32, b0 = lane * per, local = 0;
    for (int k = b0; k < min(b0 + per, n); ++k) local += __popc(mask[k]);
    int incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int v = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += v;
    }
    int run = incl - local;
    for (int k = b0; k < min(b0 + per, n); ++k) { off[k] = (unsigned)run; run += __popc(mask[k]); }
    return __shfl_sync(FULL, incl, 31);
}

__global__ void __launch_bounds__(SPH_TILE) k_cull(Dev d, float kappa, int ntile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CullSmem &sm = *reinterpret_cast<CullSmem *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    const int chunk0 = tile * SPH_TILE_CHUNKS;
    const int nch = min(SPH_TILE_CHUNKS, d.nchunk - chunk0);

    if (threadIdx.x < nch) {
        sm.blo[threadIdx.x] = d.tree.lo[0][chunk0 + threadIdx.x];
        sm.bhi[threadIdx.x] = d.tree.hi[0][chunk0 + threadIdx.x];
    }
    if (threadIdx.x < SPH_TILE_CHUNKS) sm.wcount[threadIdx.x] = 0u;
    if (threadIdx.x == 0) sm.overflow = 0;
    sm.selfslot[threadIdx.x] = 0xffffffffu;
    __syncthreads();
    if (warp == 0) {                                   // tile box = union of its chunk boxes
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
        if (lane == 0) {
            sm.tlo = make_float4(lo[0], lo[1], lo[2], H);
            sm.thi = make_float4(hi[0], hi[1], hi[2], 0.f);
            sm.nfront = 1;
            sm.chunks[0] = 0;                          // the virtual root: its children are the top level
        }
    }
    __syncthreads();

    // ---- A1: breadth-first walk of the chunk tree by all warps (one parent per warp, one child per
    //          lane).  A source chunk is accepted only if its box reaches one of the tile's chunk boxes.
    const float3 tlo = make_float3(sm.tlo.x, sm.tlo.y, sm.tlo.z), thi = make_float3(sm.thi.x, sm.thi.y, sm.thi.z);
    const float tH = sm.tlo.w;
    for (int L = d.tree.nlev - 1; L >= 0; --L) {
        const int nf = sm.nfront;
        for (int k = warp; k < nf; k += SPH_TILE_CHUNKS) {
            int first = (int)sm.chunks[k] * SPH_ARITY;
            int cnt = min(SPH_ARITY, d.tree.count[L] - first);
            unsigned cm = 0;
            bool pass = false;
            if (lane < cnt) {
                float4 clo = d.tree.lo[L][first + lane], chi = d.tree.hi[L][first + lane];
                pass = box_reach_sym(clo, chi, tlo, thi, tH);
                if (pass && L == 0) {
                    for (int w = 0; w < nch; ++w) {
                        float4 tl = sm.blo[w], th = sm.bhi[w];
                        if (box_reach_sym(clo, chi, make_float3(tl.x, tl.y, tl.z), make_float3(th.x, th.y, th.z), tl.w))
                            cm |= 1u << w;
                    }
                    pass = cm != 0;
                    sm.ctmp[k][lane] = (unsigned short)cm;
                }
            }
            unsigned m = __ballot_sync(FULL, pass);
            if (lane == 0) sm.mask[k] = m;
        }
        __syncthreads();
        if (warp == 0) {
            int total = scan_popc(sm.mask, sm.off, nf, lane);
            int cap = (L == 1) ? SPH_CULL_MAXPAR : SPH_CULL_MAXSRC;     // level-1 parents index ctmp
            if (total > cap) { total = cap; if (lane == 0) sm.overflow |= 1; }
            if (lane == 0) sm.nfront = total;
        }
        __syncthreads();
        const int cap = sm.nfront;
        for (int k = warp; k < nf; k += SPH_TILE_CHUNKS) {
            unsigned m = sm.mask[k];
            if ((m >> lane) & 1u) {
                int o = (int)sm.off[k] + __popc(m & ((1u << lane) - 1u));
                if (o < cap) {
                    sm.next[o] = sm.chunks[k] * SPH_ARITY + (unsigned)lane;
                    if (L == 0) sm.cmask[o] = sm.ctmp[k][lane];
                }
            }
        }
        __syncthreads();
        for (int k = threadIdx.x; k < cap; k += SPH_TILE) sm.chunks[k] = sm.next[k];
        __syncthreads();
    }
    const int nsrc = sm.nfront;

    // ---- A2: which particles of the accepted source chunks reach a chunk box of the tile, and how
    //          many candidates each chunk of the tile will see (-> length of its mask rows) ----------
    for (int k = warp; k < nsrc; k += SPH_TILE_CHUNKS) {
        long long j = (long long)sm.chunks[k] * SPH_CHUNK + lane;
        unsigned f = 0;
        unsigned cm = sm.cmask[k];
        if (j < d.n) {
            float4 q = d.r.pm[j];
            f = reach_flags(sm, cm, q.x, q.y, q.z, sph_H(kappa, d.r.vh[j].w));
        }
        unsigned m = __ballot_sync(FULL, f != 0);
        if (lane == 0) sm.mask[k] = m;
        while (cm) {
            int w = __ffs(cm) - 1;
            cm &= cm - 1;
            unsigned c = __popc(__ballot_sync(FULL, (f >> w) & 1u));
            if (lane == 0 && c) atomicAdd(&sm.wcount[w], c);
        }
    }
    __syncthreads();
    if (warp == 0) {
        int total = scan_popc(sm.mask, sm.off, nsrc, lane);
        unsigned wc = lane < SPH_TILE_CHUNKS ? sm.wcount[lane] : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) wc = max(wc, __shfl_xor_sync(FULL, wc, o));
        if (lane == 0) {
            unsigned long long nwm = (unsigned long long)((((wc + 31u) >> 5) + 3u) & ~3u);   // words per target
            unsigned long long co = atomicAdd(d.cand_cursor, (unsigned long long)total);
            unsigned long long mo = atomicAdd(d.mask_cursor, nwm * SPH_TILE);
            if (co + (unsigned long long)total > d.cand_cap) { sm.overflow |= 2; total = 0; co = 0; nwm = 0; }
            if (mo + nwm * SPH_TILE > d.mask_cap) { sm.overflow |= 4; total = 0; nwm = 0; mo = 0; }
            sm.ntotal = total;
            sm.nwm = (int)nwm;
            sm.cand_off = co;
            sm.mask_off = mo;
            d.tile_ncand[tile] = total;
            d.tile_off[tile] = co;
            d.tile_nwm[tile] = (int)nwm;
            d.tile_moff[tile] = mo;
            atomicAdd(&d.counters[SPH_C_CANDIDATES], (unsigned long long)total);
            if (sm.overflow) atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], (unsigned long long)sm.overflow);
        }
    }
    __syncthreads();
    const int ntotal = sm.ntotal;
    const int nwm = sm.nwm;
    unsigned *cand = d.cand + sm.cand_off;
    unsigned short *cflag = d.candflag + sm.cand_off;

    // ---- per-target state for phase B -------------------------------------------------------------
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = warp < nch && i < d.n;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float Hi = sph_H(kappa, valid ? d.r.vh[i].w : 1.f);
    const float H2i = valid ? __fmul_rn(Hi, Hi) : -1.f;
    const unsigned wbit = 1u << warp;
    uint4 *mrow = reinterpret_cast<uint4 *>(d.nmask + sm.mask_off + (size_t)threadIdx.x * nwm);
    unsigned long long tests = 0;
    int nsym = 0;
    int kk = 0;                           // running index of this warp's flagged candidates (uniform)
    unsigned hits = 0;
    uint4 acc = make_uint4(0, 0, 0, 0);
    const int nvalid = __popc(__ballot_sync(FULL, valid));

    for (int r0 = 0; r0 < ntotal; r0 += SPH_TILE_SC) {
        const int nr = min(SPH_TILE_SC, ntotal - r0);
        // ---- A3: compact this round's survivors into shared memory and the global candidate list
        for (int k = warp; k < nsrc; k += SPH_TILE_CHUNKS) {
            unsigned m = sm.mask[k];
            int o = (int)sm.off[k];
            if (o >= r0 + nr || o + 32 <= r0) continue;
            if (!((m >> lane) & 1u)) continue;
            int slot = o + __popc(m & ((1u << lane) - 1u)) - r0;
            if (slot < 0 || slot >= nr) continue;
            long long j = (long long)sm.chunks[k] * SPH_CHUNK + lane;
            float4 q = d.r.pm[j];
            float Hj = sph_H(kappa, d.r.vh[j].w);
            unsigned short f = (unsigned short)reach_flags(sm, sm.cmask[k], q.x, q.y, q.z, Hj);
            sm.pos[slot] = make_float4(q.x, q.y, q.z, __fmul_rn(Hj, Hj));
            sm.flag[slot] = f;
            cand[r0 + slot] = (unsigned)j;
            cflag[r0 + slot] = f;
            long long rel = j - (long long)tile * SPH_TILE;
            if (rel >= 0 && rel < SPH_TILE) sm.selfslot[rel] = (unsigned)(r0 + slot);
        }
        __syncthreads();
        // ---- B: the k-th candidate flagged for this warp's chunk is bit k of each target's mask -------
        const int self = (int)sm.selfslot[threadIdx.x] - r0;       // self exclusion (j != i)
        for (int base = 0; base < nr; base += 32) {
            int s = base + lane;
            unsigned m = __ballot_sync(FULL, s < nr && (sm.flag[s] & wbit));
            tests += (unsigned long long)__popc(m);
            while (m) {
                int b = __ffs(m) - 1;
                m &= m - 1;
                float4 q = sm.pos[base + b];
                float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
                if (r2 < fmaxf(H2i, q.w) && base + b != self) hits |= 1u << (kk & 31);
                ++kk;
                if ((kk & 31) == 0) {                                // a word is complete (uniform branch)
                    hits = valid ? hits : 0u;
                    nsym += __popc(hits);
                    int wi = ((kk - 1) >> 5) & 3;
                    if (wi == 0) acc.x = hits; else if (wi == 1) acc.y = hits; else if (wi == 2) acc.z = hits; else acc.w = hits;
                    if (wi == 3) { if (warp < nch && nwm) mrow[(kk - 1) >> 7] = acc; acc = make_uint4(0, 0, 0, 0); }
                    hits = 0;
                }
            }
        }
        __syncthreads();
    }
    if (kk & 127) {                                                  // partial last word / last group of four
        hits = valid ? hits : 0u;
        nsym += __popc(hits);
        int wi = (kk >> 5) & 3;
        if (kk & 31) { if (wi == 0) acc.x = hits; else if (wi == 1) acc.y = hits; else if (wi == 2) acc.z = hits; else acc.w = hits; }
        if (warp < nch && nwm) mrow[kk >> 7] = acc;
    }
    if (valid) d.nsym[i] = nwm ? nsym : 0;
    if (lane == 0 && warp < nch) atomicAdd(&d.counters[SPH_C_TESTS_CULL], tests * (unsigned long long)nvalid);
    __syncthreads();
    }   // tile loop
}

// ------------------------------------------------------------------------------------------
// shared by the list-driven passes: k -> slot table of one warp, and the per-lane bit walk
// ------------------------------------------------------------------------------------------
// Appends to wl[] the slots (relative to r0) of this round's candidates in [base, nr) that are flagged
// for this warp, until the table is full or the round ends; returns the new base.  Warp-uniform.
__device__ __forceinline__ int build_wl(const unsigned short *s_flag, int nr, int base,
                                        unsigned wbit, unsigned short *wl, int &nwl, int lane)
{
    nwl = 0;
    while (base < nr && nwl + 32 <= SPH_WL_CAP) {
        int s = base + lane;
        bool f = s < nr && (s_flag[s] & wbit);
        unsigned m = __ballot_sync(FULL, f);
        if (f) wl[nwl + __popc(m & ((1u << lane) - 1u))] = (unsigned short)s;
        nwl += __popc(m);
        base += 32;
    }
    __syncwarp();
    return base;
}

// Copies words [wg0, wg0 + SPH_MASK_GROUP) of this thread's mask row into its private column of the
// shared scratch msk[word][thread] (bank-conflict free, read back only by the same thread), restricted
// to bits k in [klo, khi).  Rows are multiples of four words, 16-byte aligned.
__device__ __forceinline__ void load_mask_group(const unsigned *__restrict__ mrow, int nwm, int wg0, int klo, int khi,
                                                unsigned *msk)
{
#pragma unroll
    for (int q = 0; q < SPH_MASK_GROUP / 4; ++q) {
        int w0 = wg0 + 4 * q;
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (w0 < nwm) v = *reinterpret_cast<const uint4 *>(mrow + w0);
        unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            int lo = klo - ((w0 + e) << 5), hi = khi - ((w0 + e) << 5);
            unsigned x = w[e];
            if (lo > 0) x = lo >= 32 ? 0u : (x & ~((1u << lo) - 1u));
            if (hi < 32) x = hi <= 0 ? 0u : (x & ((1u << hi) - 1u));
            msk[(4 * q + e) * SPH_TILE + threadIdx.x] = x;
        }
    }
}

// ------------------------------------------------------------------------------------------
// S2 density from the lists (fp64 accumulation as in k_density; see sph_pair.cu for why)
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SPH_TILE) k_density_l(Dev d, float kappa)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_pm = reinterpret_cast<float4 *>(smem_raw);
    unsigned short *s_wl = reinterpret_cast<unsigned short *>(s_pm + SPH_TILE_SC);
    unsigned *msk = reinterpret_cast<unsigned *>(s_wl + SPH_TILE_CHUNKS * SPH_WL_CAP);
    unsigned short *s_flag = reinterpret_cast<unsigned short *>(msk + SPH_MASK_GROUP * SPH_TILE);
    const int tile = blockIdx.x;
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const unsigned short *cflag = d.candflag + d.tile_off[tile];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    float hi = valid ? d.r.vh[i].w : 1.f;
    float Hi = sph_H(kappa, hi);
    const float H2i = __fmul_rn(Hi, Hi);
    const float invH = 1.f / Hi;
    const double invHd = 1.0 / ((double)kappa * (double)hi);
    const int nwm = d.tile_nwm[tile];
    const unsigned *mrow = d.nmask + d.tile_moff[tile] + (size_t)threadIdx.x * nwm;
    unsigned short *wl = s_wl + warp * SPH_WL_CAP;
    const unsigned wbit = 1u << warp;
    // self term: q = 0, t = 1
    double sum = (double)pi.w;
    float sh = 3.f * pi.w;
    int ng = 1, ntest = 1;
    int kstart = 0;
    for (int r0 = 0; r0 < ncand || r0 == 0; r0 += SPH_TILE_SC) {
        const int nr = min(SPH_TILE_SC, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) {
            s_pm[s] = d.r.pm[cand[r0 + s]];
            s_flag[s] = cflag[r0 + s];
        }
        __syncthreads();
        int base = 0;
        while (base < nr) {
            int nwl;
            base = build_wl(s_flag, nr, base, wbit, wl, nwl, lane);
            const int klo = kstart, khi = kstart + nwl;      // warp-uniform: the walk below votes
            // per-lane walk over the set bits of its mask words, one group of SPH_MASK_GROUP words at a
            // time: `bits` is the word in hand, `nxt` the next one (read one refill ahead from the
            // thread's shared-memory column); the refill is predicated, not a divergent branch
            for (int wg0 = (klo >> 5) & ~3; (wg0 << 5) < khi; wg0 += SPH_MASK_GROUP) {
            load_mask_group(mrow, nwm, wg0, klo, valid ? khi : klo, msk);   // padding lanes: all zero
            int wcur = wg0;
            const int wend = min(wg0 + SPH_MASK_GROUP, (khi + 31) >> 5);
            unsigned bits = msk[threadIdx.x];
            unsigned nxt = wcur + 1 < wend ? msk[SPH_TILE + threadIdx.x] : 0u;
            while (true) {
                if (bits == 0u && wcur < wend) {
                    ++wcur;
                    bits = nxt;
                    nxt = wcur + 1 < wend ? msk[(wcur + 1 - wg0) * SPH_TILE + threadIdx.x] : 0u;
                }
                if (!__any_sync(FULL, wcur < wend)) break;
                if (bits == 0u) continue;
                int b = __ffs(bits) - 1;
                bits &= bits - 1;
                float4 q = s_pm[wl[(wcur << 5) + b - klo]];
                ++ntest;
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
            }   // mask groups
            kstart += nwl;
            __syncwarp();
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
    unsigned long long hits = valid ? (unsigned long long)ng : 0ull, tests = valid ? (unsigned long long)ntest : 0ull;
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
// The tile's candidates are staged in rounds of SPH_PAIR_SE slots.
// ------------------------------------------------------------------------------------------
template <bool GRAD, bool FORCE>
__global__ void __launch_bounds__(SPH_TILE) k_pair_l(Dev d, DevParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s1 = reinterpret_cast<float4 *>(smem_raw);
    float4 *s2 = s1 + SPH_PAIR_SE, *s3 = s2 + SPH_PAIR_SE, *s4 = s3 + SPH_PAIR_SE, *s5 = s4 + SPH_PAIR_SE;
    unsigned short *s_wl = reinterpret_cast<unsigned short *>(s5 + SPH_PAIR_SE);
    unsigned *msk = reinterpret_cast<unsigned *>(s_wl + SPH_TILE_CHUNKS * SPH_WL_CAP);
    unsigned short *s_flag = reinterpret_cast<unsigned short *>(msk + SPH_MASK_GROUP * SPH_TILE);
    const int tile = blockIdx.x;
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const unsigned short *cflag = d.candflag + d.tile_off[tile];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    const long long il = valid ? i : 0;
    const float4 pi = d.r.pm[il], vi = d.r.vh[il], a3 = d.A3[il], a4 = d.A4[il], a5 = d.A5[il];
    const float invHi = a3.w, Ki = a3.z, rhoi = a3.x, ci = a3.y, hi = vi.w;
    const float invm = 1.f / pi.w;
    const float wKi = a5.z * invm;
    const float kxx = a4.x * invm, kyy = a4.y * invm, kzz = a4.z * invm, kxy = a4.w * invm, kxz = a5.x * invm,
                kyz = a5.y * invm;
    const int nwm = d.tile_nwm[tile];
    const unsigned *mrow = d.nmask + d.tile_moff[tile] + (size_t)threadIdx.x * nwm;
    unsigned short *wl = s_wl + warp * SPH_WL_CAP;
    const unsigned wbit = 1u << warp;

    float F[9], C[6];
#pragma unroll
    for (int k = 0; k < 9; ++k) F[k] = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) C[k] = 0.f;
    float ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, mumax = 0.f;
    int kstart = 0, cnt = 0;

    for (int r0 = 0; r0 < ncand || r0 == 0; r0 += SPH_PAIR_SE) {
        const int nr = min(SPH_PAIR_SE, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) {
            unsigned j = cand[r0 + s];
            s1[s] = d.r.pm[j];
            s2[s] = d.r.vh[j];
            s3[s] = d.A3[j];
            s4[s] = d.A4[j];
            s5[s] = d.A5[j];
            s_flag[s] = cflag[r0 + s];
        }
        __syncthreads();
        int base = 0;
        while (base < nr) {
            int nwl;
            base = build_wl(s_flag, nr, base, wbit, wl, nwl, lane);
            const int klo = kstart, khi = kstart + nwl;      // warp-uniform: the walk below votes
            for (int wg0 = (klo >> 5) & ~3; (wg0 << 5) < khi; wg0 += SPH_MASK_GROUP) {
            load_mask_group(mrow, nwm, wg0, klo, valid ? khi : klo, msk);   // padding lanes: all zero
            int wcur = wg0;
            const int wend = min(wg0 + SPH_MASK_GROUP, (khi + 31) >> 5);
            unsigned bits = msk[threadIdx.x];
            unsigned nxt = wcur + 1 < wend ? msk[SPH_TILE + threadIdx.x] : 0u;
            while (true) {
                if (bits == 0u && wcur < wend) {
                    ++wcur;
                    bits = nxt;
                    nxt = wcur + 1 < wend ? msk[(wcur + 1 - wg0) * SPH_TILE + threadIdx.x] : 0u;
                }
                if (!__any_sync(FULL, wcur < wend)) break;
                if (bits == 0u) continue;
                int b = __ffs(bits) - 1;
                bits &= bits - 1;
                const int slot = wl[(wcur << 5) + b - klo];
                ++cnt;
                const float4 q1 = s1[slot], q2 = s2[slot], q3 = s3[slot], q4 = s4[slot], q5 = s5[slot];
                float dx = __fsub_rn(pi.x, q1.x), dy = __fsub_rn(pi.y, q1.y), dz = __fsub_rn(pi.z, q1.z);
                float r2 = sph_r2(dx, dy, dz);
                float r = r2 * rsqrtf(fmaxf(r2, 1.0e-37f));
                float ti = fmaxf(0.f, 1.f - r * invHi);
                float tj = fmaxf(0.f, 1.f - r * q3.w);
                float ti3 = ti * ti * ti, tj3 = tj * tj * tj;
                float mj = q1.w;
                float dvx = vi.x - q2.x, dvy = vi.y - q2.y, dvz = vi.z - q2.z;
                float wi_ = mj * ti3;
                if (GRAD) {
                    float s = 0.5f * fmaf(wi_, wKi, q5.z * tj3);
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
                    ax = fmaf(-wi_, zx, ax); ay = fmaf(-wi_, zy, ay); az = fmaf(-wi_, zz, az);
                    du = fmaf(wi_, fmaf(zx, dvx, fmaf(zy, dvy, zz * dvz)), du);
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
            }   // mask groups
            kstart += nwl;
            __syncwarp();
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
// test hook from the lists (one thread per particle; slow and simple)
// ------------------------------------------------------------------------------------------
template <bool SYM>
__global__ void __launch_bounds__(256) k_neighbors_l(Dev d, float kappa, int *counts, const long long *offsets, int *list)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const unsigned *orig = (const unsigned *)d.r.s[PP_ORIG];
    const int tile = (int)(i / SPH_TILE);
    const int tid = (int)(i - (long long)tile * SPH_TILE);
    const unsigned wbit = 1u << (tid >> 5);
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const unsigned short *cflag = d.candflag + d.tile_off[tile];
    const unsigned *mrow = d.nmask + d.tile_moff[tile] + (size_t)tid * d.tile_nwm[tile];
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
    int k = 0;
    for (int s = 0; s < ncand; ++s) {
        if (!(cflag[s] & wbit)) continue;
        bool set = (mrow[k >> 5] >> (k & 31)) & 1u;
        ++k;
        if (!set) continue;
        unsigned j = cand[s];
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
    SPH_CUDA(c, cudaMemsetAsync(d.cand_cursor, 0, 2 * sizeof(unsigned long long), c->stream));
    if (d.n == 0) return SPH_OK;
    int rc = set_smem(c, (const void *)k_cull, sizeof(CullSmem));
    if (rc) return rc;
    int ntile = sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    k_cull<<<ntile < d.cull_grid ? ntile : d.cull_grid, SPH_TILE, sizeof(CullSmem), c->stream>>>(d, c->p.kappa, ntile);
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
    size_t bytes = (size_t)SPH_TILE_SC * sizeof(float4) + (size_t)SPH_TILE_CHUNKS * SPH_WL_CAP * sizeof(unsigned short) +
                   (size_t)SPH_MASK_GROUP * SPH_TILE * sizeof(unsigned) + (size_t)SPH_TILE_SC * sizeof(unsigned short);
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
    size_t bytes = (size_t)5 * SPH_PAIR_SE * sizeof(float4) + (size_t)SPH_TILE_CHUNKS * SPH_WL_CAP * sizeof(unsigned short) +
                   (size_t)SPH_MASK_GROUP * SPH_TILE * sizeof(unsigned) + (size_t)SPH_PAIR_SE * sizeof(unsigned short);
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
