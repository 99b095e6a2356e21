// sph_lists.cu -- neighbour lists: cull ONCE per step into explicit per-particle lists, then let the
// pair passes evaluate true pairs only, one lane per target, with no search work in their inner loop.
//
//   tile        = 8 consecutive chunks = 256 Hilbert-consecutive targets = one CTA of 8 warps.
//   k_tile_plan : the tiles that were expensive in the previous build are launched first (sph_tile_of_block).
//   k_cull      : one CTA per tile:
//                 (A) breadth-first walk of the chunk tree by all warps (a level that overflows its
//                     frontier is redone with per-target-particle tests); every particle of the accepted
//                     source chunks is tested against the tile's chunk boxes; the survivors form the tile
//                     CANDIDATE LIST (global indices, ascending), split into ROUNDS of SPH_SE slots, each
//                     slot with one byte of flags (bit w: within reach of the box of chunk w);
//                 (B) every warp keeps the slots that reach its chunk (one ballot per 32 slots), tests 32
//                     of them at a time against its four quarter boxes and splits them over four rings of
//                     offsets; every quarter-warp runs its ring, 32 candidates at a time, past its 8
//                     targets (exact fp32 predicate, reading Q4) and appends each hit to the target's
//                     NEIGHBOUR LIST: the symmetric set, self excluded, as 16-bit byte offsets (slot * 16)
//                     into the round's staged arrays.  A hit is one predicated store into the lane's
//                     buffer in shared memory; complete row-groups of 4 entries go to the global list,
//                     which is stored transposed ([chunk][row-group][lane]) so that a warp reads one
//                     coalesced 256-byte row-group per four pairs.  Rounds start at a common row-group
//                     (rowptr); LIST_PAD pads.
//   k_density_l : stages {x,y,z,m} of the round's candidates in shared memory (coalesced gathers of index
//                 runs) and walks the lists; the gather set is the subset with r2 < H_i^2, plus self.
//   k_pair_l    : same with the 18 floats per source of the fused gradient + force pass.
//   A tile that exceeds any capacity (tree-walk frontier, candidate pool, rounds, list rows) is FLAGGED
//   and served by the tree-walk kernels of sph_pair.cu instead: slower, never wrong.
//
// Evidence for this design: profiles/r01_v0_launches_and_pair_kernel.md (broadcast tiles: candidate hit
// rate 3.5 %, 18.65 of 32 threads active) and profiles/r01_v1_mask_lists.md (bitmask lists: 83 non-FP
// instructions per pair, half of the shared-memory wavefronts were bank conflicts); for the inside of
// k_cull: profiles/r01_v4_ring_tables_heavy_first.md and profiles/r01_v5_dense_flags_graph.md.
#include "sph_internal.cuh"
#include "sph_pairterm.cuh"

#define FULL 0xffffffffu
#define ROWPTR_STRIDE (SPH_MAXROUND + 1)
#define LIST_PAD ((unsigned)(SPH_SE << 4))         // padding entry of a list: the byte offset of slot SPH_SE, where the
                                                   // density and pair kernels keep a far dummy source of mass 0
#define LIST_PAD2 (LIST_PAD | (LIST_PAD << 16))
#define LBUF_ENTRIES 32                    // u16 entries a lane can hold between two flushes
#define LBUF_STRIDE (LBUF_ENTRIES * 2 + 8) // bytes per lane: 18 words, so lanes at the same fill level spread over banks

__device__ __forceinline__ bool box_reach_sym(float4 lo, float4 hi, float4 tlo, float4 thi)
{
    float gx = fmaxf(0.f, fmaxf(lo.x - thi.x, tlo.x - hi.x));
    float gy = fmaxf(0.f, fmaxf(lo.y - thi.y, tlo.y - hi.y));
    float gz = fmaxf(0.f, fmaxf(lo.z - thi.z, tlo.z - hi.z));
    float d2 = gx * gx + gy * gy + gz * gz;
    float R = fmaxf(lo.w, tlo.w);
    return d2 <= R * R * 1.00001f;        // conservative against the rounding of the exact predicate
}

// Point-vs-box reach test with the box as centre c and half-extent e (c.w = R^2 of the box: its largest
// support radius squared, times the slack factor): 14 instructions instead of 19 for the lo/hi form.
// H2s = H_j^2 times the slack factor.  e carries an absolute inflation that covers the rounding of c.
__device__ __forceinline__ bool point_reach(float4 c, float4 e, float x, float y, float z, float H2s)
{
    const float gx = fmaxf(fabsf(x - c.x) - e.x, 0.f);
    const float gy = fmaxf(fabsf(y - c.y) - e.y, 0.f);
    const float gz = fmaxf(fabsf(z - c.z) - e.z, 0.f);
    const float d2 = fmaf(gz, gz, fmaf(gy, gy, gx * gx));
    return d2 <= fmaxf(c.w, H2s);
}

#define SPH_REACH_SLACK 1.00001f       // conservative against the rounding of the exact predicate

__device__ __forceinline__ void box_centre_form(float4 lo, float4 hi, float4 &c, float4 &e)
{
    c = make_float4(0.5f * (lo.x + hi.x), 0.5f * (lo.y + hi.y), 0.5f * (lo.z + hi.z), lo.w * lo.w * SPH_REACH_SLACK);
    e = make_float4(0.5f * (hi.x - lo.x) + 1.0e-6f * fmaxf(fabsf(lo.x), fabsf(hi.x)),
                    0.5f * (hi.y - lo.y) + 1.0e-6f * fmaxf(fabsf(lo.y), fabsf(hi.y)),
                    0.5f * (hi.z - lo.z) + 1.0e-6f * fmaxf(fabsf(lo.z), fabsf(hi.z)), 0.f);
}

// ------------------------------------------------------------------------------------------
// k_cull
// ------------------------------------------------------------------------------------------
struct CullSmem {
    float4 pos[SPH_SE + 1];              // x, y, z, H^2 of the candidates of the current round; [SPH_SE] is a
                                         // sentinel no target can reach (pads the quarter-warp tables)
    unsigned char flag[SPH_SE];          // bit w: within reach of the box of chunk (warp) w of the tile
    unsigned chunks[SPH_CULL_MAXSRC];    // frontier / accepted source chunks, ascending
    unsigned mask[SPH_CULL_MAXSRC];      // surviving lanes (children / particles) of each entry
    unsigned short off[SPH_CULL_MAXSRC]; // exclusive prefix of popc(mask) (< SPH_MAXROUND * SPH_SE + 32 < 65536); in A2/A3: of
                                         // the survivors that are not "late"
    unsigned maskB[SPH_CULL_MAXSRC];     // A2/A3: the "late" survivors (within reach of <= SPH_CULL_LATE chunk boxes)
    unsigned short offB[SPH_CULL_MAXSRC];// A2/A3: exclusive prefix of popc(maskB)
    unsigned char cmask[SPH_CULL_MAXSRC];                // chunk boxes of the tile a source chunk box reaches
    union alignas(16) {
        struct {                                         // the tree walk (A1) only
            unsigned next[SPH_CULL_MAXSRC];              // next frontier
            unsigned char ctmp[SPH_CULL_MAXPAR][SPH_ARITY];   // per-child cmask of the leaf expansion
        } walk;
        unsigned char lbuf[SPH_TILE * LBUF_STRIDE];      // the list phase (B) only: per lane, list entries found
                                                         // and not yet written out
    } u;
    unsigned char cf[SPH_CULL_CFCACHE][SPH_CHUNK];       // per-particle chunk flags of the first source chunks
    float4 blo[SPH_TILE_CHUNKS], bhi[SPH_TILE_CHUNKS];   // chunk boxes (lo.w = max H)
    float4 bc[SPH_TILE_CHUNKS], be[SPH_TILE_CHUNKS];     // the same as centre / half-extent (box_centre_form)
    float4 gc[4 * SPH_TILE_CHUNKS], ge[4 * SPH_TILE_CHUNKS];     // quarter-warp boxes, centre / half-extent
    float4 tlo, thi;                     // tile box (tlo.w = max H)
    unsigned selfslot[SPH_TILE];         // slot of each target of the tile in its own candidate list
    unsigned short c1[SPH_TILE_CHUNKS][64];              // per warp: ring of the slots (as offsets) that reach its chunk
    alignas(16) unsigned short sentinels[32];            // a block of padding offsets (pos[SPH_SE])
    alignas(16) unsigned short gl[SPH_TILE_CHUNKS][4][SPH_GCAP];     // per quarter-warp: candidates still to test, ascending,
                                                         // as byte offsets (slot * 16) into pos[]
    int nsrc, ntotal, ntotalA, nfront, overflow;
    unsigned long long cand_off;
};

// bits w of `among` whose chunk box is within reach of the point (x,y,z) with support Hj
__device__ __forceinline__ unsigned reach_chunks(const CullSmem &sm, unsigned among, float x, float y, float z, float H2s)
{
    unsigned f = 0;
    while (among) {
        int w = __ffs(among) - 1;
        among &= among - 1;
        if (point_reach(sm.bc[w], sm.be[w], x, y, z, H2s)) f |= 1u << w;
    }
    return f;
}

// warp 0: off[k] = exclusive prefix of popc(mask[k]), k < n; returns the total (valid in every lane)
__device__ __forceinline__ int scan_popc(const unsigned *mask, unsigned short *off, int n, int lane)
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
    for (int k = b0; k < min(b0 + per, n); ++k) { off[k] = (unsigned short)min(run, 65535); run += __popc(mask[k]); }
    return __shfl_sync(FULL, incl, 31);
}

// infl2 = (1 + skin)^2 (1 with no list reuse): every support radius of this kernel -- box reaches and the exact
// test alike -- is inflated by 1 + skin, so that the lists hold every pair with r < (1 + skin) max(H_i, H_j) and
// the pair passes, which evaluate the exact predicate themselves, can go on using them while the particles move.
// dirty: only the tiles k_check marked (their candidates go to the second region of the pool).
__global__ void __launch_bounds__(SPH_TILE) k_cull(Dev d, float kappa, float infl, float infl2, int ntile, int dirty)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CullSmem &sm = *reinterpret_cast<CullSmem *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    {
    const int tile = sph_tile_of_block(d, blockIdx.x);
    if (tile < 0 || tile >= ntile) return;
    if (dirty) {
        if (!d.tile_dirty[tile]) return;
    } else if (d.skin > 0.f && threadIdx.x == 0) {
        d.tile_dirty[tile] = 0;
    }
    const long long t_begin = clock64();
    // SPH_C_LIST_OVERFLOW counts the tiles that are flagged NOW: a rebuilt dirty tile may change sides
    const int was_flagged = (dirty && d.tile_flag[tile]) ? 1 : 0;
    const int chunk0 = tile * SPH_TILE_CHUNKS;
    const int nch = min(SPH_TILE_CHUNKS, d.nchunk - chunk0);

    // ---- per-target state, chunk and quarter-warp boxes --------------------------------------------
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = warp < nch && i < d.n;
    // lanes without a particle sit where every r2 overflows to +inf (and differs from the table sentinel)
    const float4 pi = valid ? d.r.pm[i] : make_float4(-1.0e30f, -1.0e30f, -1.0e30f, 0.f);
    const float Hi = sph_H(kappa, valid ? d.r.vh[i].w : 1.f);
    const float H2i = valid ? __fmul_rn(__fmul_rn(Hi, Hi), infl2) : -1.f;
    {
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, Hm = 0.f;
        if (valid) { lo[0] = hi[0] = pi.x; lo[1] = hi[1] = pi.y; lo[2] = hi[2] = pi.z; Hm = Hi * infl; }
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(FULL, lo[a], o));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(FULL, hi[a], o));
            }
            Hm = fmaxf(Hm, __shfl_xor_sync(FULL, Hm, o));
        }
        if ((lane & 7) == 0)
            box_centre_form(make_float4(lo[0], lo[1], lo[2], Hm), make_float4(hi[0], hi[1], hi[2], 0.f),
                            sm.gc[4 * warp + (lane >> 3)], sm.ge[4 * warp + (lane >> 3)]);
    }
    if (threadIdx.x < nch) {
        float4 lo = d.tree.lo[0][chunk0 + threadIdx.x];
        const float4 hi = d.tree.hi[0][chunk0 + threadIdx.x];
        lo.w *= infl;
        sm.blo[threadIdx.x] = lo;
        sm.bhi[threadIdx.x] = hi;
        box_centre_form(lo, hi, sm.bc[threadIdx.x], sm.be[threadIdx.x]);
    }
    if (threadIdx.x == 0) {
        sm.overflow = 0;
        sm.pos[SPH_SE] = make_float4(1.0e30f, 1.0e30f, 1.0e30f, -1.f);
    }
    if (threadIdx.x < 32) sm.sentinels[threadIdx.x] = (unsigned short)(SPH_SE << 4);
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
    //          lane).  A node is kept only if its box reaches one of the tile's CHUNK boxes: a tile that
    //          straddles a gap of the space-filling curve has a huge union box but small chunk boxes.
    //          If a level still overflows its capacity (a CHUNK that straddles such a gap has a huge box
    //          too), the level is redone with the exact test: a node must be within reach of one of the
    //          target PARTICLES of the chunks it was accepted for (32 point tests per chunk and node:
    //          expensive, and needed by a few tiles in ten thousand).
    const float4 tlo = sm.tlo, thi = sm.thi;
    sm.pos[threadIdx.x] = make_float4(pi.x, pi.y, pi.z, valid ? H2i * SPH_REACH_SLACK : -1.f);   // pos[] is free until A3
    for (int L = d.tree.nlev - 1; L >= 0; --L) {
        const int nf = sm.nfront;
        const int capL = (L == 1) ? SPH_CULL_MAXPAR : SPH_CULL_MAXSRC;         // level-1 parents index ctmp
        for (int attempt = 0;; ++attempt) {
            for (int k = warp; k < nf; k += SPH_TILE_CHUNKS) {
                int first = (int)sm.chunks[k] * SPH_ARITY;
                int cnt = min(SPH_ARITY, d.tree.count[L] - first);
                unsigned cm = 0;
                if (lane < cnt) {
                    float4 clo = d.tree.lo[L][first + lane];
                    const float4 chi = d.tree.hi[L][first + lane];
                    clo.w *= infl;
                    if (box_reach_sym(clo, chi, tlo, thi)) {
                        for (int w = 0; w < nch; ++w)
                            if (box_reach_sym(clo, chi, sm.blo[w], sm.bhi[w])) cm |= 1u << w;
                        if (attempt && cm) {
                            float4 cc, ce;
                            box_centre_form(clo, chi, cc, ce);
                            unsigned left = cm;
                            cm = 0;
                            while (left) {
                                const int w = __ffs(left) - 1;
                                left &= left - 1;
                                for (int t = 0; t < SPH_CHUNK; ++t) {
                                    const float4 q = sm.pos[w * SPH_CHUNK + t];
                                    if (q.w >= 0.f && point_reach(cc, ce, q.x, q.y, q.z, q.w)) { cm |= 1u << w; break; }
                                }
                            }
                        }
                    }
                    if (L == 0 && k < SPH_CULL_MAXPAR) sm.u.walk.ctmp[k][lane] = (unsigned char)cm;
                }
                unsigned m = __ballot_sync(FULL, cm != 0);
                if (lane == 0) sm.mask[k] = m;
            }
            __syncthreads();
            if (warp == 0) {
                const int total = scan_popc(sm.mask, sm.off, nf, lane);
                if (lane == 0) sm.ntotal = total;
            }
            __syncthreads();
            if (sm.ntotal <= capL || attempt == 1) break;
            __syncthreads();                           // everyone has read ntotal before warp 0 writes it again
        }
        if (threadIdx.x == 0) {
            if (sm.ntotal > capL) sm.overflow |= 1;
            sm.nfront = min(sm.ntotal, capL);
        }
        __syncthreads();
        const int cap = sm.nfront;
        for (int k = warp; k < nf; k += SPH_TILE_CHUNKS) {
            unsigned m = sm.mask[k];
            if ((m >> lane) & 1u) {
                int o = (int)sm.off[k] + __popc(m & lt);
                if (o < cap) {
                    sm.u.walk.next[o] = sm.chunks[k] * SPH_ARITY + (unsigned)lane;
                    if (L == 0) sm.cmask[o] = sm.u.walk.ctmp[k][lane];
                }
            }
        }
        __syncthreads();
        for (int k = threadIdx.x; k < cap; k += SPH_TILE) sm.chunks[k] = sm.u.walk.next[k];
        __syncthreads();
    }
    const int nsrc = sm.nfront;

    // ---- A2: which particles of the accepted source chunks reach a chunk box of the tile ------------
    // (two source chunks per trip: both pairs of loads are in flight before the first is used -- the loop is
    //  bound by the latency of these L2 reads, not by its arithmetic)
    for (int k = warp; k < nsrc; k += 2 * SPH_TILE_CHUNKS) {
        const int k2 = k + SPH_TILE_CHUNKS;
        const bool has2 = k2 < nsrc;
        const long long j = (long long)sm.chunks[k] * SPH_CHUNK + lane;
        const long long j2 = has2 ? (long long)sm.chunks[k2] * SPH_CHUNK + lane : d.n;
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f), q2 = q;
        float h = 0.f, h2 = 0.f;
        if (j < d.n) { q = d.r.pm[j]; h = d.r.vh[j].w; }
        if (j2 < d.n) { q2 = d.r.pm[j2]; h2 = d.r.vh[j2].w; }
        unsigned f = 0, f2 = 0;
        if (j < d.n) {
            const float Hj = sph_H(kappa, h);
            f = reach_chunks(sm, sm.cmask[k], q.x, q.y, q.z, Hj * Hj * infl2 * SPH_REACH_SLACK);
        }
        if (j2 < d.n) {
            const float Hj = sph_H(kappa, h2);
            f2 = reach_chunks(sm, sm.cmask[k2], q2.x, q2.y, q2.z, Hj * Hj * infl2 * SPH_REACH_SLACK);
        }
        if (k < SPH_CULL_CFCACHE) sm.cf[k][lane] = (unsigned char)f;
        const unsigned m = __ballot_sync(FULL, f != 0);
        const unsigned mB = __ballot_sync(FULL, f != 0 && __popc(f) <= SPH_CULL_LATE);
        if (lane == 0) { sm.mask[k] = m & ~mB; sm.maskB[k] = mB; }
        if (has2) {
            if (k2 < SPH_CULL_CFCACHE) sm.cf[k2][lane] = (unsigned char)f2;
            const unsigned m2 = __ballot_sync(FULL, f2 != 0);
            const unsigned m2B = __ballot_sync(FULL, f2 != 0 && __popc(f2) <= SPH_CULL_LATE);
            if (lane == 0) { sm.mask[k2] = m2 & ~m2B; sm.maskB[k2] = m2B; }
        }
    }
    __syncthreads();
    // The candidate list of a tile that fits one round is in ascending index order.  One that needs several rounds is
    // split: first the candidates within reach of more than SPH_CULL_LATE chunk boxes, then the "late" ones, which
    // only one of the eight chunks can have as neighbours.  The last round then holds fewer entries for most warps: the
    // 32 lists of a chunk are padded to equal length in every round it has entries in, and on configs[4] (1 967
    // candidates per tile, 1 632 slots per round at the time) that padding was 30 % of the slots the pair passes step through;
    // with the late candidates last it is 14 % (SPH_CULL_LATE = 1; 2: 19 %, 3: 23 %, 4: 26 %), 49.5 -> 45.3 ms per step.
    if (warp == 0) {
        const int totalA = scan_popc(sm.mask, sm.off, nsrc, lane);
        const int totalB = scan_popc(sm.maskB, sm.offB, nsrc, lane);
        const int total = totalA + totalB;
        if (lane == 0) {
            // -1: ascending order (one round; or more than three: a tile that straddles a gap of the curve -- there the
            // split would spread a chunk's entries over more rounds and use up its list rows)
            sm.ntotalA = (total > SPH_SE && total <= 3 * SPH_SE) ? totalA : -1;
            // the pool: [0, cand_cap) for full builds, [cand_cap, cand_cap + cand_cap_dirty) for dirty tiles
            unsigned long long co = atomicAdd(d.cand_cursor + (dirty ? 1 : 0), (unsigned long long)total);
            if (co + (unsigned long long)total > (dirty ? d.cand_cap_dirty : d.cand_cap)) sm.overflow |= 2;
            if (dirty) co += d.cand_cap;
            if (total > SPH_MAXROUND * SPH_SE) sm.overflow |= 4;
            sm.ntotal = total;
            sm.cand_off = co;
        }
    }
    __syncthreads();
    if (sm.overflow) {                                 // flagged before any list was written
        if (threadIdx.x == 0) {
            d.tile_flag[tile] = (unsigned char)sm.overflow;     // which capacity: 1 walk, 2 pool, 4 rounds
            d.tile_ncand[tile] = 0;
            d.tile_off[tile] = 0;
            if (!was_flagged) atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull);
        }
        if (valid) { d.nsym[i] = 0; d.nlen[i] = 0; }
        if (threadIdx.x == 0 && !dirty) {
            const unsigned cyc = (unsigned)(clock64() - t_begin);
            d.tile_cycles[tile] = cyc;
            atomicAdd(d.cull_cycles, (unsigned long long)cyc);
        }
        return;
    }
    const int ntotal = sm.ntotal, ntotalA = sm.ntotalA;
    unsigned *cand = d.cand + sm.cand_off;
    if (threadIdx.x == 0) {
        d.tile_ncand[tile] = ntotal;
        d.tile_off[tile] = sm.cand_off;
        atomicAdd(&d.counters[SPH_C_CANDIDATES], (unsigned long long)ntotal);
    }

    // ---- per-lane list state --------------------------------------------------------------------------
    // A lane appends the byte offset of every hit to its own buffer in shared memory (one predicated
    // store per test: no bit masks, no serial extraction loop).  Complete row-groups (4 entries) go to
    // the transposed global list when some lane's buffer could overflow in the next block of tests and
    // at the end of the round, all lanes in lockstep: by then the lanes hold similar numbers of rows.
    const int chunk = chunk0 + warp;
    uint2 *lp = d.nlist + ((size_t)(warp < nch ? chunk : chunk0) * d.rows_cap) * 32 + lane;
    unsigned short *rp = d.rowptr + (size_t)(warp < nch ? chunk : chunk0) * ROWPTR_STRIDE;
    // the lane's buffer and its write position as 32-bit byte offsets into the dynamic shared memory
    const unsigned lb = (unsigned)(sm.u.lbuf - smem_raw) + threadIdx.x * LBUF_STRIDE;
    unsigned wp = lb;                     // where the next entry goes
    int G = 0;                            // row-groups of this lane in the global list so far (padding included)
    int nhit = 0;                         // true neighbours
    unsigned tests = 0, slots = 0;
    int Gstart = 0;                       // first row-group of the current round
    // write the complete row-groups of the buffer out, keep the 0..3 entries left over
#define LIST_FLUSH()                                                                        \
    do {                                                                                    \
        const int cnt_ = (int)(wp - lb) >> 1, rows_ = cnt_ >> 2;                            \
        const int rmax_ = __reduce_max_sync(FULL, rows_);                                   \
        for (int r_ = 0; r_ < rmax_; ++r_)                                                  \
            if (r_ < rows_ && G + r_ < d.rows_cap)                                          \
                lp[(size_t)(G + r_) * 32] = *reinterpret_cast<const uint2 *>(smem_raw + lb + 8 * r_);  \
        if (cnt_ & 3) *reinterpret_cast<uint2 *>(smem_raw + lb) = *reinterpret_cast<const uint2 *>(smem_raw + lb + 8 * rows_); \
        G += rows_;                                                                         \
        wp = lb + 2 * (cnt_ & 3);                                                           \
    } while (0)
    const int g = lane >> 3;
    if (warp < nch && lane == 0) rp[0] = 0;

    int round = 0;
    const int se = sph_round_size(ntotal);
    for (int r0 = 0; r0 < ntotal; r0 += se, ++round) {
        const int nr = min(se, ntotal - r0);
        // ---- A3: compact this round's survivors into shared memory and the global candidate list
        // (two source chunks per trip, as in A2: the loads of both are issued before either is used)
        for (int k = warp; k < nsrc; k += 2 * SPH_TILE_CHUNKS) {
            int slot[2];
            long long jj[2];
            float4 q[2];
            float hh[2];
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int kk = k + t * SPH_TILE_CHUNKS;
                slot[t] = -1;
                jj[t] = 0;
                if (kk < nsrc) {
                    const unsigned mA = sm.mask[kk], mB = sm.maskB[kk];
                    if (((mA | mB) >> lane) & 1u) {
                        int sl;
                        if (ntotalA < 0) sl = (int)sm.off[kk] + (int)sm.offB[kk] + __popc((mA | mB) & lt);
                        else if ((mB >> lane) & 1u) sl = ntotalA + (int)sm.offB[kk] + __popc(mB & lt);
                        else sl = (int)sm.off[kk] + __popc(mA & lt);
                        sl -= r0;
                        if (sl >= 0 && sl < nr) { slot[t] = sl; jj[t] = (long long)sm.chunks[kk] * SPH_CHUNK + lane; }
                    }
                }
            }
#pragma unroll
            for (int t = 0; t < 2; ++t)
                if (slot[t] >= 0) { q[t] = d.r.pm[jj[t]]; hh[t] = d.r.vh[jj[t]].w; }
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                if (slot[t] < 0) continue;
                const int kk = k + t * SPH_TILE_CHUNKS;
                const float Hj = sph_H(kappa, hh[t]);
                sm.pos[slot[t]] = make_float4(q[t].x, q[t].y, q[t].z, __fmul_rn(__fmul_rn(Hj, Hj), infl2));
                const float H2s = Hj * Hj * infl2 * SPH_REACH_SLACK;
                const unsigned fc = kk < SPH_CULL_CFCACHE ? (unsigned)sm.cf[kk][lane]
                                                          : reach_chunks(sm, sm.cmask[kk], q[t].x, q[t].y, q[t].z, H2s);
                sm.flag[slot[t]] = (unsigned char)fc;
                cand[r0 + slot[t]] = (unsigned)jj[t];
                const long long rel = jj[t] - (long long)tile * SPH_TILE;
                if (rel >= 0 && rel < SPH_TILE) sm.selfslot[rel] = (unsigned)(r0 + slot[t]);
            }
        }
        __syncthreads();
        if (warp < nch) {
            // ---- B: quarter g of this warp tests the candidates flagged for it, in slot order ---------
            const int selfrel = (int)sm.selfslot[threadIdx.x] - r0;    // self exclusion (j != i)
            const unsigned selfoff = (selfrel >= 0 && selfrel < nr) ? (unsigned)selfrel << 4 : 0xffffffffu;
            Gstart = G;
            unsigned short(*gl)[SPH_GCAP] = sm.gl[warp];
            const unsigned char *const posb = reinterpret_cast<const unsigned char *>(sm.pos);
            // Every quarter keeps a ring of SPH_GCAP offsets.  The rings are filled from the flag words
            // until every quarter has a block of 32 (or one ring is full, or the round is exhausted);
            // then each quarter that has a block tests it.  Quarters see different numbers of
            // candidates: this way a lane tests padding only in the last block of a round.
            int base = 0;
            int h0 = 0, h1 = 0, h2 = 0, h3 = 0;           // ring heads (entries consumed), multiples of 32
            int t0 = 0, t1 = 0, t2 = 0, t3 = 0;           // ring tails (entries produced)
            int ch = 0, ct = 0;                           // head / tail of the warp's ring of flagged slots
            unsigned short *const c1 = sm.c1[warp];
            const unsigned short sent = (unsigned short)(SPH_SE << 4);
            for (;;) {
                // Two stages.  (1) one ballot per 32 slots keeps the slots that reach this warp's chunk at
                // all (about a third); (2) 32 of those at a time are split over the four quarter rings
                // (four ballots).  Every warp scans every slot of the round: stage 1 is the cheap part.
                for (;;) {
                    const int a0 = t0 - h0, a1 = t1 - h1, a2 = t2 - h2, a3 = t3 - h3;
                    if (max(max(a0, a1), max(a2, a3)) + 32 > SPH_GCAP) break;     // a ring could overflow
                    if (min(min(a0, a1), min(a2, a3)) >= 32) break;               // every quarter has a block
                    while (ct - ch < 32 && base < nr) {
                        const int s = base + lane;
                        const bool any = s < nr && ((sm.flag[s] >> warp) & 1u) != 0u;
                        const unsigned m = __ballot_sync(FULL, any);
                        if (any) c1[(ct + __popc(m & lt)) & 63] = (unsigned short)(s << 4);
                        ct += __popc(m);
                        base += 32;
                    }
                    const int take = min(32, ct - ch);
                    if (take == 0) break;                                         // round exhausted
                    __syncwarp();
                    unsigned f = 0u;
                    unsigned short so = 0;
                    if (lane < take) {
                        // which of the warp's four quarter boxes the candidate reaches (every lane has an
                        // entry here: the quarter tests run at full width, unlike in A3)
                        so = c1[(ch + lane) & 63];
                        const float4 q = *reinterpret_cast<const float4 *>(posb + so);
                        const float H2s = q.w * SPH_REACH_SLACK;
#pragma unroll
                        for (int gq = 0; gq < 4; ++gq)
                            if (point_reach(sm.gc[4 * warp + gq], sm.ge[4 * warp + gq], q.x, q.y, q.z, H2s)) f |= 1u << gq;
                    }
                    ch += take;
                    const unsigned m0 = __ballot_sync(FULL, f & 1u), m1 = __ballot_sync(FULL, f & 2u),
                                   m2 = __ballot_sync(FULL, f & 4u), m3 = __ballot_sync(FULL, f & 8u);
                    if (f & 1u) gl[0][(t0 + __popc(m0 & lt)) & (SPH_GCAP - 1)] = so;
                    if (f & 2u) gl[1][(t1 + __popc(m1 & lt)) & (SPH_GCAP - 1)] = so;
                    if (f & 4u) gl[2][(t2 + __popc(m2 & lt)) & (SPH_GCAP - 1)] = so;
                    if (f & 8u) gl[3][(t3 + __popc(m3 & lt)) & (SPH_GCAP - 1)] = so;
                    t0 += __popc(m0); t1 += __popc(m1); t2 += __popc(m2); t3 += __popc(m3);
                }
                const bool drain = base >= nr && ct == ch;
                const int a0 = t0 - h0, a1 = t1 - h1, a2 = t2 - h2, a3 = t3 - h3;
                // entries each quarter tests now: a full block, or what is left when the round is exhausted
                const int n0 = a0 >= 32 ? 32 : (drain ? a0 : 0), n1 = a1 >= 32 ? 32 : (drain ? a1 : 0),
                          n2 = a2 >= 32 ? 32 : (drain ? a2 : 0), n3 = a3 >= 32 ? 32 : (drain ? a3 : 0);
                if ((n0 | n1 | n2 | n3) == 0) break;      // only when drained and empty
                if (lane >= n0 && n0 > 0) gl[0][(h0 + lane) & (SPH_GCAP - 1)] = sent;
                if (lane >= n1 && n1 > 0) gl[1][(h1 + lane) & (SPH_GCAP - 1)] = sent;
                if (lane >= n2 && n2 > 0) gl[2][(h2 + lane) & (SPH_GCAP - 1)] = sent;
                if (lane >= n3 && n3 > 0) gl[3][(h3 + lane) & (SPH_GCAP - 1)] = sent;
                __syncwarp();
                const int ng = g == 0 ? n0 : (g == 1 ? n1 : (g == 2 ? n2 : n3));
                const int hg = g == 0 ? h0 : (g == 1 ? h1 : (g == 2 ? h2 : h3));
                // a quarter without a block reads 32 sentinels
                const uint4 *mygl = ng ? reinterpret_cast<const uint4 *>(&gl[g][hg & (SPH_GCAP - 1)])
                                       : reinterpret_cast<const uint4 *>(sm.sentinels);
                tests += valid ? (unsigned)ng : 0u;
                // 32 candidates of the quarter's ring (8 offsets per 16-byte read), 16 between two checks of
                // the list buffer level
#pragma unroll
                for (int k8 = 0; k8 < 4; ++k8) {
                    if (k8 == 2 && __any_sync(FULL, (int)(wp - lb) > 2 * (LBUF_ENTRIES - 16))) LIST_FLUSH();
                    const uint4 tw = mygl[k8];
                    const unsigned wv[4] = {tw.x, tw.y, tw.z, tw.w};
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const unsigned off = (e & 1) ? (wv[e >> 1] >> 16) : (wv[e >> 1] & 0xffffu);
                        const float4 q = *reinterpret_cast<const float4 *>(posb + off);
                        const float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
                        if (r2 < fmaxf(H2i, q.w) && off != selfoff) {
                            *reinterpret_cast<unsigned short *>(smem_raw + wp) = (unsigned short)off;
                            wp += 2;
                        }
                    }
                }
                // room for another 16 entries in every lane?  (3 may stay behind after a flush)
                if (__any_sync(FULL, (int)(wp - lb) > 2 * (LBUF_ENTRIES - 16))) LIST_FLUSH();
                __syncwarp();
                // consumed blocks leave the rings (a partial last block leaves it empty: head = tail, aligned)
                h0 += n0 == 32 ? 32 : 0; h1 += n1 == 32 ? 32 : 0; h2 += n2 == 32 ? 32 : 0; h3 += n3 == 32 ? 32 : 0;
                if (n0 < 32 && n0 > 0) { h0 = 0; t0 = 0; }
                if (n1 < 32 && n1 > 0) { h1 = 0; t1 = 0; }
                if (n2 < 32 && n2 > 0) { h2 = 0; t2 = 0; }
                if (n3 < 32 && n3 > 0) { h3 = 0; t3 = 0; }
            }
            // ---- end of the round: pad the last row-group, flush, pad every lane to the warp's longest list
            nhit += 4 * (G - Gstart) + ((int)(wp - lb) >> 1);
            while ((int)(wp - lb) & 7) {
                *reinterpret_cast<unsigned short *>(smem_raw + wp) = (unsigned short)LIST_PAD;
                wp += 2;
            }
            LIST_FLUSH();
            const int Gmax = __reduce_max_sync(FULL, G);
            for (int gg = G; gg < Gmax; ++gg)
                if (gg < d.rows_cap) lp[(size_t)gg * 32] = make_uint2(LIST_PAD2, LIST_PAD2);
            G = Gmax;
            if (G > d.rows_cap) sm.overflow = 8;      // list rows exhausted: the tile falls back
            if (lane == 0) {
                rp[round + 1] = (unsigned short)min(Gmax, d.rows_cap);
                slots += (unsigned)(Gmax - Gstart) * 128u;
            }
        }
        __syncthreads();
    }
    if (valid) { d.nsym[i] = nhit; d.nlen[i] = nhit; }      // nlen: entries of the particle's list (pairs of the skin included)
    if (warp < nch) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tests += __shfl_xor_sync(FULL, tests, o);
        if (lane == 0) {
            atomicAdd(&d.counters[SPH_C_TESTS_CULL], (unsigned long long)tests);
            atomicAdd(&d.counters[SPH_C_LIST_SLOTS], (unsigned long long)slots);
        }
    }
#undef LIST_FLUSH
    if (threadIdx.x == 0) {
        d.tile_flag[tile] = (unsigned char)sm.overflow;         // 8: list rows
        if (!dirty) {                                           // the cost statistics are those of full builds
            const unsigned cyc = (unsigned)(clock64() - t_begin);
            d.tile_cycles[tile] = cyc;
            atomicAdd(d.cull_cycles, (unsigned long long)cyc);
        }
        const int now_flagged = sm.overflow ? 1 : 0;
        if (now_flagged > was_flagged) atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], 1ull);
        if (now_flagged < was_flagged) atomicAdd(&d.counters[SPH_C_LIST_OVERFLOW], ~0ull);      // minus one
    }
    }
}

// A point no particle can reach and that reaches no particle, from the top level of the chunk tree at the current
// positions (warp-wide): beyond the box of everything by twice its extent plus eight times the largest support radius,
// carrying that radius.  The padding entries of the neighbour lists stand for a source of mass 0 there.
__device__ __forceinline__ void sph_far_point(const Dev &d, int lane)
{
    const int L = d.tree.nlev - 1, cnt = d.tree.count[L];
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, H = 0.f;
    if (lane < cnt) {
        const float4 a = d.tree.lo[L][lane], b = d.tree.hi[L][lane];
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
        const float ext = fmaxf(hi[0] - lo[0], fmaxf(hi[1] - lo[1], hi[2] - lo[2]));
        const float off = 2.f * ext + 8.f * H;
        *d.far_point = make_float4(hi[0] + off, hi[1] + off, hi[2] + off, H);
    }
}

// Head of a list build, ONE block: which tiles go first (those that cost more than 1.5x the average in the previous
// build), and the resets the build needs (list-build counters, candidate pool cursor, cycle sum).
__global__ void __launch_bounds__(1024) k_tile_plan(Dev d, int ntile, int dirty)
{
    if (threadIdx.x < 32) sph_far_point(d, threadIdx.x);
    if (dirty) {                  // a step that reuses the lists: only the second region of the pool starts over
        if (threadIdx.x == 0) {
            d.cand_cursor[1] = 0ull;
            d.counters[SPH_C_TESTS_CULL] = 0ull;
            d.counters[SPH_C_CANDIDATES] = 0ull;
            d.counters[SPH_C_LIST_SLOTS] = 0ull;
        }
        return;
    }
    __shared__ unsigned s_n;
    if (threadIdx.x == 0) s_n = 0u;
    __syncthreads();
    const unsigned long long sum = *d.cull_cycles;
    for (int t = threadIdx.x; t < ntile; t += blockDim.x) {
        bool heavy = 2ull * (unsigned long long)d.tile_cycles[t] * (unsigned long long)ntile > 3ull * sum;
        if (heavy) {
            const unsigned k = atomicAdd(&s_n, 1u);
            if (k < (unsigned)d.heavy_cap) d.heavy_list[k] = (unsigned)t;
            else heavy = false;                // list full: the tile stays in curve order
        }
        d.heavy_mark[t] = heavy ? 1 : 0;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        *d.nheavy = min(s_n, (unsigned)d.heavy_cap);
        *d.cull_cycles = 0ull;
        d.cand_cursor[0] = 0ull;
        d.cand_cursor[1] = 0ull;
        d.counters[SPH_C_TESTS_CULL] = 0ull;
        d.counters[SPH_C_CANDIDATES] = 0ull;
        d.counters[SPH_C_LIST_OVERFLOW] = 0ull;
        d.counters[SPH_C_TILES_DIRTY] = 0ull;
        d.counters[SPH_C_LIST_SLOTS] = 0ull;
    }
}

// ------------------------------------------------------------------------------------------
// k_list_sort (after a full build when the lists are reused, sph_params.skin > 0: its cost is spread over the steps
// that reuse them -- as a pass of every step it did not pay, profiles/r01_v5): reorder every lane's list entries of a
// round so that lane l reads bank class
// (l + n) mod 8 at step n (class = slot mod 8 = which 16-byte bank group the slot's float4 sits in).  The eight
// lanes of a quarter-warp phase then hit eight different bank groups in the pair kernel's gathers instead of
// random ones (2.47 wavefronts per phase).  Per lane: count the classes, bucket the entries by class in shared
// memory (counting sort, cursors packed 8 x 8 bit), emit them round-robin over the classes starting at the
// lane's own; when the wanted class has run out, the next one in cyclic order that has entries.  One warp per
// chunk, all lanes in lockstep over the positions of the round; rounds with a lane over SORT_CAP entries stay as
// they are.  The order of a lane's entries has no meaning (a set), so results change only by summation order.
// ------------------------------------------------------------------------------------------
// entry e (0..3) of a row-group word pair
__device__ __forceinline__ unsigned list_entry(uint2 w, int e)
{
    const unsigned x = (e & 2) ? w.y : w.x;
    return (e & 1) ? (x >> 16) : (x & 0xffffu);
}

static int set_smem(sph_ctx *c, const void *fn, size_t bytes);

#define SORT_CAP 192
#define SORT_STRIDE (SORT_CAP * 2 + 4)       // bytes per lane: 97 words
#define SORT_BITW (2 * SPH_SE / 32)          // bitmap words: tiles of up to two rounds are compacted

// pass 3 of the sort: emit N buffered entries round-robin over the classes, all lanes in lockstep over 4 * rows
// positions, into the row-groups [gfirst, gfirst + rows) of the lane's column
__device__ __forceinline__ void sort_emit(uint2 *lp, const unsigned short *buf, unsigned long long tk, unsigned long long end,
                                          int N, int gfirst, int rows, int lane)
{
    unsigned w0 = 0u, w1 = 0u;
    for (int n = 0; n < rows * 4; ++n) {
        unsigned entry = LIST_PAD;
        if (n < N) {
            unsigned c8 = ((unsigned)(lane + n) & 7u) << 3;
            while (((unsigned)(tk >> c8) & 0xffu) >= ((unsigned)(end >> c8) & 0xffu)) c8 = (c8 + 8u) & 63u;
            entry = buf[(unsigned)(tk >> c8) & 0xffu];
            tk += 1ull << c8;
        }
        w0 = __byte_perm(w0, w1, 0x5432);
        w1 = __byte_perm(w1, entry, 0x5432);
        if ((n & 3) == 3) lp[(size_t)(gfirst + (n >> 2)) * 32] = make_uint2(w0, w1);
    }
}

// walk the row-groups [ga, gb) of a lane's column with SORT_INFLIGHT loads in flight (these kernels are bound by the
// latency of the list reads): f(gq, w)
#ifndef SORT_INFLIGHT
#define SORT_INFLIGHT 8
#endif
template <typename F>
__device__ __forceinline__ void for_rows(const uint2 *lp, int ga, int gb, F f)
{
    for (int gq = ga; gq < gb; gq += SORT_INFLIGHT) {
        uint2 w[SORT_INFLIGHT];
#pragma unroll
        for (int j = 0; j < SORT_INFLIGHT; ++j)
            w[j] = gq + j < gb ? lp[(size_t)(gq + j) * 32] : make_uint2(LIST_PAD2, LIST_PAD2);
#pragma unroll
        for (int j = 0; j < SORT_INFLIGHT; ++j)
            if (gq + j < gb) f(gq + j, w[j]);
    }
}

// the entries of one round of a lane's list, row-groups [g0, ge), ordered by bank class (all lanes of a warp together);
// a round with a lane over SORT_CAP entries stays as it is
__device__ __forceinline__ void sort_round(uint2 *lp, unsigned short *buf, int g0, int ge, int lane)
{
    if (ge <= g0) return;
    // pass 1: class counts
    unsigned long long cnt = 0ull;
    int N = 0;
    for_rows(lp, g0, ge, [&](int, uint2 w) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const unsigned off = list_entry(w, e);
            if (off != LIST_PAD) { cnt += 1ull << (((off >> 4) & 7u) << 3); ++N; }
        }
    });
    if (__any_sync(FULL, N > SORT_CAP)) return;
    const unsigned long long base = cnt * 0x0101010101010100ull;     // field c = entries of the classes below c
    // pass 2: bucket by class
    unsigned long long cur = base;
    for_rows(lp, g0, ge, [&](int, uint2 w) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const unsigned off = list_entry(w, e);
            if (off != LIST_PAD) {
                const unsigned c8 = ((off >> 4) & 7u) << 3;
                buf[(unsigned)(cur >> c8) & 0xffu] = (unsigned short)off;
                cur += 1ull << c8;
            }
        }
    });
    sort_emit(lp, buf, base, cur, N, g0, ge - g0, lane);
}

// One CTA per tile, one warp per chunk.
// COMPACTION (tiles of two rounds).  k_cull accepts a candidate when it is within reach of a chunk BOX of the
// tile; a fifth of them (configs[3-4]) turn out to be nobody's neighbour.  The CTA marks the candidates some list of
// the tile uses, renumbers them (order kept), compacts the tile's candidate list in place, and the sort below writes
// the entries with their new slots: entries move from the second round into the first.  configs[4]: 1 954 -> 1 577
// candidates per tile, 60 % of the tiles then need one round instead of two (2 % before): pair pass 22.2 -> 19.4 ms,
// density 9.9 -> 9.1 ms.  A two-round tile is compacted if that saves a round or an eighth of its candidates, and if the new
// row-groups are sure to fit (first round <= all old rows, second round <= its old rows) and no lane has more than
// SORT_CAP entries.
__global__ void __launch_bounds__(SPH_TILE, 2) k_list_compact_sort(Dev d)
{
    extern __shared__ __align__(16) unsigned char s_buf[];
    unsigned short *tab = reinterpret_cast<unsigned short *>(s_buf + (size_t)SPH_TILE * SORT_STRIDE);      // [2 SPH_SE] new slot
    unsigned *bits = reinterpret_cast<unsigned *>(tab + 2 * SPH_SE);                                        // [SORT_BITW]
    unsigned *pre = bits + SORT_BITW;                                                                       // [SORT_BITW + 1]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x;
    if (d.tile_flag[tile]) return;
    const int chunk = tile * SPH_TILE_CHUNKS + warp;
    const bool haschunk = chunk < d.nchunk;
    uint2 *lp = d.nlist + ((size_t)(haschunk ? chunk : 0) * d.rows_cap) * 32 + lane;
    unsigned short *rp = d.rowptr + (size_t)(haschunk ? chunk : 0) * ROWPTR_STRIDE;
    unsigned short *buf = reinterpret_cast<unsigned short *>(s_buf + (size_t)threadIdx.x * SORT_STRIDE);
    const int ncand = d.tile_ncand[tile];
    const int nround = sph_round_count(ncand);
    if (nround != 2) return;                   // k_list_sort has ordered this tile's lists
    bool compact = false;
    int nused = ncand, g1 = 0, g2 = 0;
    {
        for (int w = threadIdx.x; w < SORT_BITW; w += SPH_TILE) bits[w] = 0u;
        __syncthreads();
        int ok = 1;
        if (haschunk) {
            g1 = rp[1];
            g2 = nround > 1 ? (int)rp[2] : g1;
            for_rows(lp, 0, g2, [&](int gq, uint2 w) {
                const unsigned kb = gq < g1 ? 0u : (unsigned)SPH_SE;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const unsigned off = list_entry(w, e);
                    if (off != LIST_PAD) {
                        const unsigned k = kb + (off >> 4);
                        atomicOr(&bits[k >> 5], 1u << (k & 31u));
                    }
                }
            });
            const long long i = (long long)tile * SPH_TILE + threadIdx.x;
            const int tot = __reduce_max_sync(FULL, i < d.n ? d.nlen[i] : 0);
            ok = (2 * g2 - g1 <= d.rows_cap && tot <= SORT_CAP) ? 1 : 0;
        }
        __syncthreads();
        if (warp == 0) {                               // exclusive prefix of the popcounts
            const int per = (SORT_BITW + 31) / 32, b0 = lane * per;
            int local = 0;
            for (int w = b0; w < min(b0 + per, SORT_BITW); ++w) local += __popc(bits[w]);
            int incl = local;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += v;
            }
            int run = incl - local;
            for (int w = b0; w < min(b0 + per, SORT_BITW); ++w) { pre[w] = (unsigned)run; run += __popc(bits[w]); }
            if (lane == 31) pre[SORT_BITW] = (unsigned)incl;
        }
        ok = __syncthreads_and(ok);
        nused = (int)pre[SORT_BITW];
        compact = ok && (sph_round_count(nused) < nround || nused * 8 <= ncand * 7);
    }
    if (compact) {
        // the new slot of every candidate; the candidate list in place, order kept: a block of 256 entries is read before
        // any of it is written, and an entry never moves to a higher index
        unsigned *cand = d.cand + d.tile_off[tile];
        for (int b0 = 0; b0 < ncand; b0 += SPH_TILE) {
            const int k = b0 + threadIdx.x;
            unsigned v = 0u, ns = 0xffffu;
            if (k < ncand) {
                v = cand[k];
                if ((bits[k >> 5] >> (k & 31)) & 1u) ns = pre[k >> 5] + __popc(bits[k >> 5] & ((1u << (k & 31)) - 1u));
                tab[k] = (unsigned short)ns;
            }
            __syncthreads();
            if (ns != 0xffffu) cand[ns] = v;
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            d.tile_ncand[tile] = nused;
            atomicAdd(&d.counters[SPH_C_CANDIDATES], (unsigned long long)(long long)(nused - ncand));
        }
        if (!haschunk) return;
        // entries of both old rounds together: the new first round in [0, N0) of the buffer, the second in [N0, N0 + N1)
        unsigned long long cnt0 = 0ull, cnt1 = 0ull;
        int N0 = 0, N1 = 0;
        for_rows(lp, 0, g2, [&](int gq, uint2 w) {
            const unsigned kb = gq < g1 ? 0u : (unsigned)SPH_SE;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const unsigned off = list_entry(w, e);
                if (off != LIST_PAD) {
                    const unsigned ns = tab[kb + (off >> 4)];
                    if (ns < (unsigned)SPH_SE) { cnt0 += 1ull << ((ns & 7u) << 3); ++N0; }
                    else { cnt1 += 1ull << (((ns - SPH_SE) & 7u) << 3); ++N1; }
                }
            }
        });
        const unsigned long long base0 = cnt0 * 0x0101010101010100ull;
        const unsigned long long base1 = cnt1 * 0x0101010101010100ull + (unsigned long long)N0 * 0x0101010101010101ull;
        unsigned long long cur0 = base0, cur1 = base1;
        for_rows(lp, 0, g2, [&](int gq, uint2 w) {
            const unsigned kb = gq < g1 ? 0u : (unsigned)SPH_SE;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const unsigned off = list_entry(w, e);
                if (off != LIST_PAD) {
                    const unsigned ns = tab[kb + (off >> 4)];
                    if (ns < (unsigned)SPH_SE) {
                        const unsigned c8 = (ns & 7u) << 3;
                        buf[(unsigned)(cur0 >> c8) & 0xffu] = (unsigned short)(ns << 4);
                        cur0 += 1ull << c8;
                    } else {
                        const unsigned c8 = ((ns - SPH_SE) & 7u) << 3;
                        buf[(unsigned)(cur1 >> c8) & 0xffu] = (unsigned short)((ns - SPH_SE) << 4);
                        cur1 += 1ull << c8;
                    }
                }
            }
        });
        const int R0 = __reduce_max_sync(FULL, (N0 + 3) >> 2), R1 = __reduce_max_sync(FULL, (N1 + 3) >> 2);
        sort_emit(lp, buf, base0, cur0, N0, 0, R0, lane);
        sort_emit(lp, buf, base1, cur1, N1, R0, R1, lane);
        if (lane == 0) {
            rp[1] = (unsigned short)R0;
            rp[2] = (unsigned short)(R0 + R1);
            atomicAdd(&d.counters[SPH_C_LIST_SLOTS], (unsigned long long)(long long)((R0 + R1 - g2) * 128));
        }
        return;
    }
    if (!haschunk) return;
    for (int r = 0; r < nround; ++r) sort_round(lp, buf, rp[r], rp[r + 1], lane);
}

// The tiles of one round or of more than two: the sort alone, one warp per chunk, four chunks per CTA (five CTAs per
// SM; the compacting kernel holds two).  Runs BEFORE k_list_compact_sort, which changes tile_ncand of its tiles.
#define SORT_WARPS 4
__global__ void __launch_bounds__(SORT_WARPS * 32) k_list_sort(Dev d)
{
    extern __shared__ __align__(16) unsigned char s_buf[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = blockIdx.x * SORT_WARPS + warp;
    if (chunk >= d.nchunk) return;
    const int tile = chunk / SPH_TILE_CHUNKS;
    if (d.tile_flag[tile]) return;
    const int nround = sph_round_count(d.tile_ncand[tile]);
    if (nround == 2) return;
    uint2 *lp = d.nlist + ((size_t)chunk * d.rows_cap) * 32 + lane;
    const unsigned short *rp = d.rowptr + (size_t)chunk * ROWPTR_STRIDE;
    unsigned short *buf = reinterpret_cast<unsigned short *>(s_buf + (size_t)threadIdx.x * SORT_STRIDE);
    for (int r = 0; r < nround; ++r) sort_round(lp, buf, rp[r], rp[r + 1], lane);
}

#define SORT_SMEM ((size_t)SPH_TILE * SORT_STRIDE + 2 * SPH_SE * 2 + (2 * SORT_BITW + 1) * 4)
int sph_launch_list_sort(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    int rc = set_smem(c, (const void *)k_list_compact_sort, SORT_SMEM);
    if (rc) return rc;
    rc = set_smem(c, (const void *)k_list_sort, SORT_WARPS * 32 * SORT_STRIDE);
    if (rc) return rc;
    k_list_sort<<<sph_div_up(d.nchunk, SORT_WARPS), SORT_WARPS * 32, SORT_WARPS * 32 * SORT_STRIDE, c->stream>>>(d);
    k_list_compact_sort<<<sph_div_up(d.nchunk, SPH_TILE_CHUNKS), SPH_TILE, SORT_SMEM, c->stream>>>(d);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

// cp.async: global -> shared without a register in between (LDGSTS)
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}


// ------------------------------------------------------------------------------------------
// S2 density from the lists: the gather set is the subset of the symmetric list with r2 < H_i^2, plus self.
// Arithmetic: density_term (sph_pairterm.cuh): rho in fp64 (five fp32 -> fp64 conversions per true pair).
// Measured alternatives (round 2, configs[2], this kernel 0.222 ms): fp32 terms with an fp64 accumulator:
// 0.151 ms but rho only to 1.4e-7 and S_pred of configs[0] at 1.02e-4 (tolerance 1e-4): rejected; candidates
// staged a second time widened to fp64 (48 B per slot, no conversions in the loop): 0.39 ms with one or two
// warps per chunk -- three random LDS.128 per pair instead of one: the shared-memory pipe binds: rejected.
// What did help: (1) the register budget.  With the default budget (48 registers) ptxas re-converted the TARGET's
// x, y, z to fp64 for every pair instead of keeping three doubles alive: six conversions per pair in the SASS where
// the source has three.  __launch_bounds__(256, 4) allows 55 registers: 0.228 -> 0.207 ms (configs[2]), 11.7 ->
// 10.8 ms (configs[4]).  (2) mass and rsqrt widened by integer operations (sph_widen_pos) instead of on the XU pipe.
// XU operations per gather pair: 7 (round 1) -> 4.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SPH_TILE, 4) k_density_l(Dev d, float kappa, RungCtl rc)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_pm = reinterpret_cast<float4 *>(smem_raw);
    const int tile = sph_tile_of_block(d, blockIdx.x);
    if (tile < 0 || d.tile_flag[tile]) return;
    if (rc.on && !rc.tile_need[tile]) return;              // NEXT-4: no active particle reads this tile's density now
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = tile * SPH_TILE_CHUNKS + warp;
    const bool haschunk = chunk < d.nchunk;
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    const float4 pi = valid ? d.r.pm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    const float hi = valid ? d.r.vh[i].w : 1.f;
    const float Hi = sph_H(kappa, hi);
    const float H2i = __fmul_rn(Hi, Hi);
    const float invH = 1.f / Hi;
    const double invHd = 1.0 / ((double)kappa * (double)hi);
    const double pxd = (double)pi.x, pyd = (double)pi.y, pzd = (double)pi.z;
    const uint2 *lp = d.nlist + ((size_t)(haschunk ? chunk : 0) * d.rows_cap) * 32 + lane;
    const unsigned short *rp = d.rowptr + (size_t)(haschunk ? chunk : 0) * ROWPTR_STRIDE;
    DensAcc A;
    A.sum = (double)pi.w; A.sh = 3.0 * (double)pi.w; A.n = 1;          // self term: q = 0, t = 1
    // slot SPH_SE: the far dummy source the padding entries of the lists point at (out of everybody's reach)
    if (threadIdx.x == 0) {
        const float4 fp = *d.far_point;
        s_pm[SPH_SE] = make_float4(fp.x, fp.y, fp.z, 0.f);
    }
    int round = 0;
    const int se = sph_round_size(ncand);
    for (int r0 = 0; r0 < ncand; r0 += se, ++round) {
        const int nr = min(se, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) cp_async16(&s_pm[s], &d.r.pm[cand[r0 + s]]);
        asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (haschunk) {
            const int g0 = rp[round], g1 = rp[round + 1];
            uint2 nxt = g0 < g1 ? lp[(size_t)g0 * 32] : make_uint2(LIST_PAD2, LIST_PAD2);
            for (int gq = g0; gq < g1; ++gq) {
                const uint2 w = nxt;
                if (gq + 1 < g1) nxt = lp[(size_t)(gq + 1) * 32];      // (streaming loads + an L2 prefetch, as in k_pair_l: +2.7 % here)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const unsigned off = list_entry(w, e);               // padding (LIST_PAD): the dummy
                    const float4 q = *reinterpret_cast<const float4 *>(smem_raw + off);
                    const float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
                    if (r2 < H2i)
                        density_term(A, r2, pxd - (double)q.x, pyd - (double)q.y, pzd - (double)q.z,
                                     sph_widen_pos(q.w), invHd);
                }
            }
        }
        __syncthreads();
    }
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
    unsigned long long hits = valid ? (unsigned long long)A.n : 0ull, tests = valid ? (unsigned long long)(d.nlen[i] + 1) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        hits += __shfl_xor_sync(FULL, hits, o);
        tests += __shfl_xor_sync(FULL, tests, o);
    }
    small = __popc(__ballot_sync(FULL, small != 0u));
    if (lane == 0) {
        atomicAdd(&d.counters[SPH_C_PAIRS_GATHER], hits);
        atomicAdd(&d.counters[SPH_C_TESTS_DENSITY], tests);
        if (small) atomicAdd(&d.counters[SPH_C_OMEGA_SMALL], (unsigned long long)small);
    }
}

// ------------------------------------------------------------------------------------------
// S4 + S5 from the lists.  Equations and operand packing: sph_pairterm.cuh.
// Shared memory: four float4 arrays and one float2 array of SPH_SE + 1 slots (72 B per candidate; the
// hydro-only variant stages the first three arrays only); slot SPH_SE is the far dummy source of mass 0 that the
// padding entries of the lists point at.
// ------------------------------------------------------------------------------------------
// The candidates are staged with cp.async (measured against loads and stores through registers, round 2: force pass
// 0.452 -> 0.437 ms on configs[2], 27.9 -> 26.8 ms on configs[4]); the staged h is the raw smoothing length,
// H_j = kappa h_j is formed per list entry.  The list loop is bound by instruction issue (profiles/r02_v8_pair_diet.md):
// 112.5 instructions per entry, no test for padding, membership from u = max(1 - r/H_i, 1 - r/H_j) (pair_term).

// One list entry (staged at byte offset off) that may lie inside the band |u| <= SPH_UBAND: if it does, the exact
// predicate (reading Q4) decides whether it is a neighbour: the count and mu_max of Eq. 39.
template <bool FORCE>
__device__ __forceinline__ void pair_decide(const PairTarget &t, const PairConst &kc, PairAcc &A, int &cnt, float H2i,
                                            float kappa, const unsigned char *s1, const unsigned char *s2, unsigned off)
{
    const float4 q1 = *reinterpret_cast<const float4 *>(s1 + off);
    float4 q2 = *reinterpret_cast<const float4 *>(s2 + off);
    q2.w = sph_H(kappa, q2.w);
    const PairGeom g = pair_geom(t, q1, q2.w);
    const float um = fmaxf(g.ui, g.uj);
    if (um >= -SPH_UBAND && !(um > SPH_UBAND)) {
        const float r2x = sph_r2(g.dx, g.dy, g.dz);
        if (r2x < fmaxf(H2i, __fmul_rn(q2.w, q2.w))) {
            ++cnt;
            if (FORCE) A.mumax = fmaxf(A.mumax, pair_neg_mu(t, kc, g, q2));
        }
    }
}

template <bool GRAD, bool FORCE, bool TENSOR>
__global__ void __launch_bounds__(SPH_TILE, 2) k_pair_l(Dev d, DevParams p, RungCtl rc)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char *s1 = smem_raw, *s2 = s1 + (SPH_SE + 1) * 16, *s3 = s2 + (SPH_SE + 1) * 16, *s4 = s3 + (SPH_SE + 1) * 16,
                  *s5 = s4 + (SPH_SE + 1) * 16;
    const int tile = sph_tile_of_block(d, blockIdx.x);
    if (tile < 0 || d.tile_flag[tile]) return;
    if (rc.on && !rc.tile_act[tile]) return;               // NEXT-4: no particle of this tile ends a step now
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chunk = tile * SPH_TILE_CHUNKS + warp;
    const bool haschunk = chunk < d.nchunk;
    const long long i = (long long)tile * SPH_TILE + threadIdx.x;
    const bool valid = i < d.n;
    const PairTarget t = pair_target_load(d, valid ? i : 0, p.kappa);
    const float H2i = __fmul_rn(t.H, t.H);
    const PairConst kc = pair_const(p.alpha, p.beta, p.eps_av, p.kappa);
    const uint2 *lp = d.nlist + ((size_t)(haschunk ? chunk : 0) * d.rows_cap) * 32 + lane;
    const unsigned short *rp = d.rowptr + (size_t)(haschunk ? chunk : 0) * ROWPTR_STRIDE;
    PairAcc A;
    pair_acc_zero(A);
    int cnt = 0;
    // slot SPH_SE of the staged arrays: the far dummy source the padding entries of the lists point at (mass 0, out of
    // everybody's reach: sph_far_point), so that the inner loop needs no test for padding
    if (threadIdx.x == 0) {
        const float4 fp = *d.far_point;
        *reinterpret_cast<float4 *>(s1 + 16 * SPH_SE) = make_float4(fp.x, fp.y, fp.z, 0.f);
        *reinterpret_cast<float4 *>(s2 + 16 * SPH_SE) = make_float4(0.f, 0.f, 0.f, fp.w);
        *reinterpret_cast<float4 *>(s3 + 16 * SPH_SE) = make_float4(1.f, 0.f, 0.f, 0.f);
        if (TENSOR) {
            *reinterpret_cast<float4 *>(s4 + 16 * SPH_SE) = make_float4(0.f, 0.f, 0.f, 0.f);
            *reinterpret_cast<float2 *>(s5 + 8 * SPH_SE) = make_float2(0.f, 0.f);
        }
    }

    int round = 0;
    const int se = sph_round_size(ncand);
    for (int r0 = 0; r0 < ncand; r0 += se, ++round) {
        const int nr = min(se, ncand - r0);
        for (int s = threadIdx.x; s < nr; s += SPH_TILE) {
            const unsigned j = cand[r0 + s];
            cp_async16(s1 + 16 * s, &d.r.pm[j]);
            cp_async16(s2 + 16 * s, &d.r.vh[j]);
            cp_async16(s3 + 16 * s, &d.B3[j]);
            if (TENSOR) {
                cp_async16(s4 + 16 * s, &d.B4[j]);
                cp_async8(s5 + 8 * s, &d.B5[j]);
            }
        }
        asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (haschunk) {
            const int g0 = rp[round], g1 = rp[round + 1];
            uint2 nxt = g0 < g1 ? lp[(size_t)g0 * 32] : make_uint2(LIST_PAD2, LIST_PAD2);
            int namb = 0, ambrow = 0;              // row-groups of this lane with an entry inside the band; the last one
            for (int gq = g0; gq < g1; ++gq) {
                const uint2 w = nxt;
                // the lists stream through once per pass: read them past L1 and ask L2 for the row-group eight ahead
                // (measured: -1.3 % on configs[4]; four or sixteen ahead, or two row-groups in registers: slower)
                if (gq + 1 < g1) nxt = __ldcs(&lp[(size_t)(gq + 1) * 32]);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(&lp[(size_t)min(gq + 8, g1 - 1) * 32]));
                float umin = 3.0e38f;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const unsigned off = list_entry(w, e);               // padding (LIST_PAD): the dummy
                    const float4 q1 = *reinterpret_cast<const float4 *>(s1 + off);
                    float4 q2 = *reinterpret_cast<const float4 *>(s2 + off);
                    q2.w = sph_H(p.kappa, q2.w);
                    const float4 q3 = *reinterpret_cast<const float4 *>(s3 + off);
                    float4 q4 = make_float4(0.f, 0.f, 0.f, 0.f);
                    float2 q5 = make_float2(0.f, 0.f);
                    if (TENSOR) {
                        q4 = *reinterpret_cast<const float4 *>(s4 + off);
                        q5 = *reinterpret_cast<const float2 *>(s5 + (off >> 1));
                    }
                    // The lists may hold pairs of the skin (list reuse) and padding.  Membership is the exact predicate
                    // on the current positions (reading Q4); pair_term decides it from u = max(1 - r/H_i, 1 - r/H_j)
                    // wherever |u| > SPH_UBAND; the entries inside the band are decided below.
                    bool v;
                    float um;
                    pair_term<GRAD, FORCE, TENSOR, true>(t, kc, A, q1, q2, q3, q4, q5, v, um);
                    cnt += v ? 1 : 0;
                    umin = fminf(umin, fabsf(um));
                }
                if (umin <= SPH_UBAND) { ++namb; ambrow = gq; }
            }
            // Entries inside the band (one list entry in 10^5) are decided with the exact predicate: the count, and
            // mu_max of Eq. 39 (the sums got their < 1e-17 either way).  A lane with one such row-group looks at its
            // four entries; a lane with several walks the round's rows again.
            if (__any_sync(FULL, namb > 0)) {
                if (namb == 1) {
                    const uint2 w = lp[(size_t)ambrow * 32];
                    for (int e = 0; e < 4; ++e) pair_decide<FORCE>(t, kc, A, cnt, H2i, p.kappa, s1, s2, list_entry(w, e));
                }
                if (__any_sync(FULL, namb > 1)) {
                    for (int gq = g0; gq < g1; ++gq) {
                        const uint2 w = lp[(size_t)gq * 32];
                        for (int e = 0; e < 4; ++e)
                            if (namb > 1) pair_decide<FORCE>(t, kc, A, cnt, H2i, p.kappa, s1, s2, list_entry(w, e));
                    }
                }
            }
        }
        __syncthreads();
    }

    const bool keep = valid && sph_active(rc, i);          // NEXT-4: an inactive particle keeps its old derivatives
    if (keep) {
        pair_store<GRAD, FORCE>(d, i, A, kc, !(p.flags & SPH_INT_DEFER_AEXT));
        d.nsym[i] = cnt;
    }
    if (FORCE) {
        unsigned long long hits = keep ? (unsigned long long)cnt : 0ull, ents = valid ? (unsigned long long)d.nlen[i] : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            hits += __shfl_xor_sync(FULL, hits, o);
            ents += __shfl_xor_sync(FULL, ents, o);
        }
        if (lane == 0) {
            atomicAdd(&d.counters[SPH_C_PAIRS_SYMMETRIC], hits);
            atomicAdd(&d.counters[SPH_C_TESTS_FORCE], ents);          // list entries examined (skin pairs included)
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
    const int tile = (int)(i / SPH_TILE);
    if (d.tile_flag[tile]) return;
    const unsigned *orig = (const unsigned *)d.r.s[PP_ORIG];
    const int chunk = (int)(i / SPH_CHUNK), lane = (int)(i % SPH_CHUNK);
    const int ncand = d.tile_ncand[tile];
    const unsigned *cand = d.cand + d.tile_off[tile];
    const uint2 *lp = d.nlist + ((size_t)chunk * d.rows_cap) * 32 + lane;
    const unsigned short *rp = d.rowptr + (size_t)chunk * ROWPTR_STRIDE;
    unsigned oi = orig[i];
    long long base = list ? offsets[oi] : 0;
    if (base < 0) { base = 0; list = nullptr; }          // offsets[i] < 0: this particle's ids are not wanted
    float4 pi = d.r.pm[i];
    float Hi = sph_H(kappa, d.r.vh[i].w);
    float H2i = __fmul_rn(Hi, Hi);
    int out = 0, intile = 0;
    // the lists may hold pairs of the skin: the sets are defined by the exact predicate (reading Q4)
    if (!SYM) {
        if (list) list[base] = (int)oi;
        out = 1;
    }
    int round = 0;
    const int se = sph_round_size(ncand);
    for (int r0 = 0; r0 < ncand; r0 += se, ++round) {
        for (int gq = rp[round]; gq < rp[round + 1]; ++gq) {
            const uint2 w = lp[(size_t)gq * 32];
            for (int e = 0; e < 4; ++e) {
                const unsigned off = list_entry(w, e);
                if (off == LIST_PAD) continue;
                unsigned j = cand[r0 + (int)(off >> 4)];
                const float4 q = d.r.pm[j];
                const float r2 = sph_r2(__fsub_rn(pi.x, q.x), __fsub_rn(pi.y, q.y), __fsub_rn(pi.z, q.z));
                bool hit = r2 < H2i;
                if (SYM) {
                    const float Hj = sph_H(kappa, d.r.vh[j].w);
                    hit = r2 < fmaxf(H2i, __fmul_rn(Hj, Hj));
                }
                if (hit) {
                    if (list) list[base + out] = (int)orig[j];
                    ++out;
                    if (SYM && (long long)j / SPH_TILE == i / SPH_TILE) ++intile;
                }
            }
        }
    }
    counts[oi] = out;
    if (SYM && intile) atomicAdd(&d.counters[SPH_C_PAIRS_INTILE], (unsigned long long)intile);
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
static int set_smem(sph_ctx *c, const void *fn, size_t bytes)
{
    SPH_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return SPH_OK;
}

int sph_launch_cull(sph_ctx *c, bool dirty_only)
{
    Dev &d = c->d;
    if (d.n == 0) {
        SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_CULL], 0, 3 * sizeof(unsigned long long), c->stream));
        return SPH_OK;
    }
    int rc = set_smem(c, (const void *)k_cull, sizeof(CullSmem));
    if (rc) return rc;
    int ntile = sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    const bool reuse = d.skin > 0.f && !c->no_reuse_now;
    const float infl = 1.f + (reuse ? d.skin : 0.f);
    k_tile_plan<<<1, 1024, 0, c->stream>>>(d, ntile, dirty_only ? 1 : 0);
    k_cull<<<d.heavy_cap + ntile, SPH_TILE, sizeof(CullSmem), c->stream>>>(d, c->p.kappa, infl, infl * infl, ntile,
                                                                            dirty_only ? 1 : 0);
    c->launches += 2;
    SPH_CUDA(c, cudaGetLastError());
    if (!dirty_only && reuse) return sph_launch_list_sort(c);      // lists that will be reused: order them
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------
// k_check (list reuse): may tile T go on using the lists of the last full build?  Those lists hold every pair
// that was within (1 + skin) max(H_i, H_j) then.  A pair (t, j) that is within max(H_t, H_j) NOW and is not in
// t's list must have closed in by more than skin max(H_t, H_j) >= skin H_t:  |d_t - d_j| > skin H_t, d = x - xref.
// With D_T the centre of the box of the tile's displacements and E_T its half diagonal, that cannot happen if
//     max_{j in N} |d_j - D_T| + E_T <= 0.95 skin min_T H
// for every tree node N whose box is within reach of the tile's box now (0.95 covers the rounding of the two
// predicates).  One warp per tile walks the chunk tree: a node out of reach is skipped, a node that satisfies
// the bound is done with all its descendants, others are opened; a CHUNK that fails makes the tile DIRTY -- its
// lists are then rebuilt at the current positions in every step until the next full build (sticky).
// Rigid motion of a body costs nothing here (its displacement boxes are points); a tile at a contact surface
// gets dirty at once, and only it and its like are rebuilt.
// ------------------------------------------------------------------------------------------
#define CHECK_STACK (SPH_ARITY * (SPH_MAX_LEVELS - 1))
__global__ void __launch_bounds__(SPH_TILE) k_check(Dev d, float thr, int ntile)
{
    __shared__ unsigned s_stack[SPH_TILE_CHUNKS][CHECK_STACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x * SPH_TILE_CHUNKS + warp;
    if (tile >= ntile || d.tile_dirty[tile]) return;
    const int chunk0 = tile * SPH_TILE_CHUNKS;
    const int nch = min(SPH_TILE_CHUNKS, d.nchunk - chunk0);
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, H = 0.f;
    float dl[3] = {3.0e38f, 3.0e38f, 3.0e38f}, dh[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, Hmin = 3.0e38f;
    if (lane < nch) {
        float4 a = d.tree.lo[0][chunk0 + lane], b = d.tree.hi[0][chunk0 + lane];
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; H = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
        a = d.tree.dlo[0][chunk0 + lane]; b = d.tree.dhi[0][chunk0 + lane];
        dl[0] = a.x; dl[1] = a.y; dl[2] = a.z; Hmin = a.w;
        dh[0] = b.x; dh[1] = b.y; dh[2] = b.z;
    }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(FULL, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(FULL, hi[a], o));
            dl[a] = fminf(dl[a], __shfl_xor_sync(FULL, dl[a], o));
            dh[a] = fmaxf(dh[a], __shfl_xor_sync(FULL, dh[a], o));
        }
        H = fmaxf(H, __shfl_xor_sync(FULL, H, o));
        Hmin = fminf(Hmin, __shfl_xor_sync(FULL, Hmin, o));
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = __shfl_sync(FULL, lo[a], 0); hi[a] = __shfl_sync(FULL, hi[a], 0);
        dl[a] = __shfl_sync(FULL, dl[a], 0); dh[a] = __shfl_sync(FULL, dh[a], 0);
    }
    H = __shfl_sync(FULL, H, 0);
    Hmin = __shfl_sync(FULL, Hmin, 0);
    const float4 tlo = make_float4(lo[0], lo[1], lo[2], H), thi = make_float4(hi[0], hi[1], hi[2], 0.f);
    const float Dx = 0.5f * (dl[0] + dh[0]), Dy = 0.5f * (dl[1] + dh[1]), Dz = 0.5f * (dl[2] + dh[2]);
    const float ex = 0.5f * (dh[0] - dl[0]), ey = 0.5f * (dh[1] - dl[1]), ez = 0.5f * (dh[2] - dl[2]);
    const float E = sqrtf(ex * ex + ey * ey + ez * ez) * 1.000001f;
    const float budget = thr * Hmin - E;          // what a node's displacements may differ from D_T by
    bool dirty = !(budget > 0.f);
    const float budget2 = budget * budget;
    unsigned *stack = s_stack[warp];
    int sp = 0;
    int L = d.tree.nlev - 1, first = 0, cnt = d.tree.count[L];
    while (!dirty) {
        bool open = false;
        if (lane < cnt) {
            const float4 clo = d.tree.lo[L][first + lane], chi = d.tree.hi[L][first + lane];
            if (box_reach_sym(clo, chi, tlo, thi)) {
                const float4 a = d.tree.dlo[L][first + lane], b = d.tree.dhi[L][first + lane];
                const float fx = fmaxf(fabsf(a.x - Dx), fabsf(b.x - Dx)), fy = fmaxf(fabsf(a.y - Dy), fabsf(b.y - Dy)),
                            fz = fmaxf(fabsf(a.z - Dz), fabsf(b.z - Dz));
                open = !(fx * fx + fy * fy + fz * fz <= budget2);
            }
        }
        const unsigned mask = __ballot_sync(FULL, open);
        if (L == 0) {
            if (mask) { dirty = true; break; }
        } else {
            if (open) stack[sp + __popc(mask & ((1u << lane) - 1u))] = ((unsigned)L << 27) | (unsigned)(first + lane);
            sp += __popc(mask);
            __syncwarp();
        }
        if (sp == 0) break;
        const unsigned e = stack[--sp];
        __syncwarp();
        L = (int)(e >> 27) - 1;
        first = (int)(e & 0x7ffffffu) * SPH_ARITY;
        cnt = min(SPH_ARITY, d.tree.count[L] - first);
    }
    if (dirty && lane == 0) {
        d.tile_dirty[tile] = 1;
        atomicAdd(&d.counters[SPH_C_TILES_DIRTY], 1ull);
    }
}

int sph_launch_check(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    const int ntile = sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    k_check<<<sph_div_up(ntile, SPH_TILE_CHUNKS), SPH_TILE, 0, c->stream>>>(d, 0.95f * d.skin, ntile);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_density_l(sph_ctx *c)
{
    Dev &d = c->d;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_GATHER], 0, sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_TESTS_DENSITY], 0, sizeof(unsigned long long), c->stream));
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_OMEGA_SMALL], 0, sizeof(unsigned long long), c->stream));
    if (d.n == 0) return SPH_OK;
    size_t bytes = (size_t)(SPH_SE + 1) * sizeof(float4);
    int rc = set_smem(c, (const void *)k_density_l, bytes);
    if (rc) return rc;
    k_density_l<<<d.heavy_cap + sph_div_up(d.nchunk, SPH_TILE_CHUNKS), SPH_TILE, bytes, c->stream>>>(d, c->p.kappa, c->rc);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return sph_launch_density(c, true);               // the flagged tiles, if any
}

template <bool GRAD, bool FORCE, bool TENSOR>
static int launch_pair_l(sph_ctx *c)
{
    Dev &d = c->d;
    size_t bytes = (size_t)(SPH_SE + 1) * (TENSOR ? 72 : 48);
    const int grid = d.heavy_cap + sph_div_up(d.nchunk, SPH_TILE_CHUNKS);
    int rc = set_smem(c, (const void *)k_pair_l<GRAD, FORCE, TENSOR>, bytes);
    if (rc) return rc;
    k_pair_l<GRAD, FORCE, TENSOR><<<grid, SPH_TILE, bytes, c->stream>>>(d, c->p, c->rc);
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
    const bool tensor = (c->p.flags & SPH_STRENGTH) != 0;
    int rc;
    if (grad && force) rc = launch_pair_l<true, true, true>(c);
    else if (grad) rc = launch_pair_l<true, false, true>(c);
    else if (tensor) rc = launch_pair_l<false, true, true>(c);
    else rc = launch_pair_l<false, true, false>(c);
    if (rc) return rc;
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return sph_launch_pair(c, grad, force, true);     // the flagged tiles, if any
}

int sph_launch_neighbors_l(sph_ctx *c, int which, int *counts, const long long *offsets, int *list)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    int nb = sph_div_up(d.n, 256);
    if (which == SPH_SYMMETRIC) SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_PAIRS_INTILE], 0, sizeof(unsigned long long), c->stream));
    if (which == SPH_SYMMETRIC) k_neighbors_l<true><<<nb, 256, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    else k_neighbors_l<false><<<nb, 256, 0, c->stream>>>(d, c->p.kappa, counts, offsets, list);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return sph_launch_neighbors(c, which, counts, offsets, list, true);
}
