// sph_internal.cuh -- internal declarations of libsph.so (CUDA, sm_100a only).
// Shares nothing with oracle/.  Equation numbers refer to /root/reference/PAPER.md.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sph.h"

#define SPH_CHUNK 32          // particles per target chunk = one warp of targets
#define SPH_ARITY 32          // children per node of the implicit chunk tree (one lane each)
#define SPH_MAX_LEVELS 7      // 32^6 chunks * 32 particles >> any n that fits in HBM
#define SPH_NPP 21            // scalar (4-byte) resident arrays that are permuted at re-sort

// internal bit of DevParams.flags (never set by callers: sph_init masks it): the pair pass leaves a_ext out and CLOSE adds
// it -- sph_step_host on a step whose a_ext is still on its way from the host while the pair pass runs
#define SPH_INT_DEFER_AEXT 0x80000000u

// neighbour-list machinery (sph_lists.cu)
#define SPH_TILE_CHUNKS 8     // chunks per tile = warps per CTA of the list kernels
#define SPH_TILE (SPH_TILE_CHUNKS * SPH_CHUNK)
#ifndef SPH_SE                // (a test build with fewer slots drives the multi-round paths on every tile: tests/test_gpu_rounds.py)
#define SPH_SE 1600           // candidates staged per round; the cull, density and pair kernels agree on it
#endif
                              // (18 floats per slot plus the dummy slot, twice per SM: 1601 x 72 B <= 115 712 B)
#define SPH_MAXROUND 15       // rounds a tile may need (more: the tile falls back to the tree-walk kernels)
#define SPH_CULL_MAXSRC 768   // source chunks a tile may accept in the tree walk
#define SPH_CULL_MAXPAR 128   // level-1 nodes a tile may expand in the last level of the walk
#define SPH_GCAP 128          // entries of a quarter-warp's candidate table in k_cull (multiple of 32)
#define SPH_CULL_CFCACHE 128  // source chunks whose per-particle chunk flags are kept between the two passes
#define SPH_CULL_LATE 1       // a candidate within reach of at most this many chunk boxes of a tile that needs several
                              // rounds goes to the END of the tile's candidate list (k_cull, A2; measured 1..4 on configs[4])
#ifndef SPH_ROWS_DEFAULT
#define SPH_ROWS_DEFAULT 64   // default row-groups (4 neighbours per lane each) reserved per chunk
#endif
#ifndef SPH_POOL_PER_TILE     // candidate pool: slots per tile on average (twice the one-round capacity); half as much again
#define SPH_POOL_PER_TILE (2 * SPH_SE)   // for the dirty tiles' region.  (The small-SPH_SE test build keeps the 3 200 of the product.)
#endif

// indices into Resident::s (scalar ping-pong arrays)
enum {
    PP_UPRED = 0,
    PP_SPRED = 1,   // +0..4
    PP_VHALF = 6,   // +0..2
    PP_UHALF = 9,
    PP_SHALF = 10,  // +0..4
    PP_EACC = 15,
    PP_G = 16,      // +0..2
    PP_ORIG = 19,   // uint32 original index
    PP_MATFIX = 20  // uint32: material | fixed << 8
};

struct DevParams {
    float kappa, alpha, beta, eps_av, eta_C, eta_a;
    unsigned flags;
    int n_materials;
    sph_material mat[SPH_MAX_MATERIALS];
};

// NEXT-3: tabulated EOS per material (sph_set_eos_table); P == nullptr: the analytic stand-in
struct DevTab {
    int n_rho, n_u, n_melt;
    float rho_min, rho_max, u_min, u_max;
    const float *P, *T, *cs, *Tmelt;
};
struct DevTabs {
    DevTab t[SPH_MAX_MATERIALS];
};

// Sorted ("resident") particle data that moves with the particle at re-sort.
struct Resident {
    float4 *pm;              // x, y, z, m
    float4 *vh;              // predicted v (Eq. 40 analogue for v), h
    float *s[SPH_NPP];       // see PP_*
};

// Implicit 32-ary tree over the Morton-sorted chunk array: node k of level L covers chunks
// [k 32^L, (k+1) 32^L).  lo.w = max H of the node, hi.w unused.
// dlo / dhi (list reuse, see Dev::skin): per node the box of the DISPLACEMENTS x - xref of its particles since
// the last full list build; dlo.w = smallest support radius H in the node.
struct Tree {
    int nlev;                        // levels stored; level nlev-1 has <= 32 nodes
    int count[SPH_MAX_LEVELS];
    float4 *lo[SPH_MAX_LEVELS];
    float4 *hi[SPH_MAX_LEVELS];
    float4 *dlo[SPH_MAX_LEVELS];
    float4 *dhi[SPH_MAX_LEVELS];
};

// NEXT-4 (sph_step_rungs): which particles / tiles a pass of a substep works on.  on == 0: everything (global step).
// A particle on rung r is ACTIVE at the end of substep n (n1 = n + 1 substeps done) iff n1 is a multiple of
// 2^(R - r).  need: tiles that hold an active particle or a candidate neighbour of one (density, PREDICT);
// act: tiles that hold an active particle (pair pass).
struct RungCtl {
    int on;
    int n1, R;
    float dT;
    int fixed_rungs;                 // keep the rungs (test hook)
    const unsigned char *rung;       // per particle, current sorted order
    const unsigned char *tile_act, *tile_need;
};

// Everything the kernels need, passed by value.
struct Dev {
    long long n;       // particles resident
    int nchunk;        // ceil(n / 32)
    long long n_max;
    Resident r;        // current
    Resident alt;      // other half of the ping-pong
    Tree tree;
    // single-buffered, current sorted order
    float *vfull[3], *ufull, *Sfull[5];     // state at the full step (after CLOSE)
    float *a[3], *dudt, *dS[5];             // derivatives at the full step
    float *rho, *omega, *P, *cs, *T, *Gamma, *Y, *mumax, *dti, *eps2, *cflag;
    double *rho64;                          // fp64 density for the EOS (see k_density)
    float *mK;                              // m K, K = 20 SIGMA / H^5 (written by the density kernels, packed into B5 by k_predict)
    int *ngather, *nsym;
    float *F[9], *Cinv[9], *G[9];
    float4 *B3, *B4;                        // packed pair-pass operands (see k_predict):
    float2 *B5;                             //   B3 = {rho, c, w, st_xx}, B4 = {st_yy, st_zz, st_xy, st_xz}, B5 = {st_yz, m K},
                                            //   K = 20 SIGMA / H^5 (Wendland C2: -(dW/dr)/r = K (1 - r/H)^3)
    // neighbour lists (sph_lists.cu)
    int *tile_ncand;                        // candidates per tile
    unsigned *cand;                         // candidate pool: global indices, tile after tile, ascending per tile
    unsigned long long *tile_off;           // where each tile's candidates start in the pool
    unsigned long long *cand_cursor;        // bump allocators of the pool: [0] full builds, [1] per-step rebuilds of dirty tiles
    unsigned long long cand_cap;            // pool capacity (entries) of a full build; the entries behind it
    unsigned long long cand_cap_dirty;      //   serve the dirty tiles of the steps in between
    // list reuse (sph_params.skin > 0): the lists of a full build hold every pair within (1 + skin) of its
    // cut-off and stay in use, with the exact predicate evaluated in the pair passes, until the next full
    // build; a tile whose surroundings moved too much against it (k_check) is DIRTY: its lists are rebuilt
    // at the current positions in every step until then
    float skin;                             // 0: off (every step is a full build)
    float4 *xref;                           // positions at the last full build (current sorted order)
    unsigned char *rung;                    // NEXT-4: rung per particle (current sorted order)
    unsigned char *tile_act, *tile_need;    // NEXT-4: per tile, see RungCtl
    unsigned char *tile_dirty;              // sticky until the next full build
    uint2 *nlist;                           // [chunk][row-group][lane]: 4 x u16 per lane = byte offsets (slot * 16)
                                            // into the round's staged arrays; SPH_SE << 4 (the dummy slot) = no entry
    int rows_cap;                           // row-groups reserved per chunk
    unsigned short *rowptr;                 // [chunk][SPH_MAXROUND + 1]: first row-group of each round
    unsigned *tile_cycles;                  // SM clock cycles k_cull spent on each tile in the last build
    unsigned long long *cull_cycles;        // their sum
    // launch order of the tile kernels: the tiles that were expensive in the previous build go first
    // (a tile that straddles gaps of the space-filling curve costs up to 5x the average and would
    // otherwise finish long after everything else); see sph_tile_of_block
    unsigned *heavy_list;                   // [heavy_cap] tiles that run first
    unsigned *nheavy;                       // entries of heavy_list
    unsigned char *heavy_mark;              // [tile] != 0: in heavy_list
    int heavy_cap;                          // blocks reserved in front of the grid for heavy_list
    unsigned char *tile_flag;               // != 0: the tile exceeded a capacity; the tree-walk kernels serve it
    float4 *far_point;                      // x, y, z out of everybody's reach and the largest support radius (sph_far_point)
    int *nlen;                              // per particle: entries of its neighbour list (pairs of the skin included)
    int cull_grid;                          // persistent CTAs of k_cull
    int walk_grid;                          // persistent CTAs of the tree-walk kernels when they serve flagged tiles
    // scalars on the device
    float *bbox;                            // 6 floats as ordered ints: lo xyz, hi xyz
    float *dt_cur, *dt_next;                // step in use / CFL step from the last CLOSE
    double *diag_part;                      // [592][8] per-block partial sums of sph_get_diagnostics
    float *hchange;                         // max |factor - 1| of the last smoothing-length update
    int *refresh_changed;                   // sph_step_host: != 0 if the caller's x, y, z or h differ from the resident ones
    unsigned long long *counters;           // SPH_C_COUNT
    // sort scratch
    unsigned long long *keys, *keys_alt;
    unsigned *perm, *perm_alt;
    void *cub_tmp;
    size_t cub_tmp_bytes;
};

struct sph_ctx {
    DevParams p;
    DevTabs tabs;
    Dev d;
    cudaStream_t stream;
    int last_cuda;
    long long launches;
    bool use_lists;
    // CUDA graphs of the resident step (sph_step with state == NULL, dt <= 0): one per half of the
    // ping-pong (the kernels take the array pointers by value); see sph_step
    bool use_graph, capturing;
    int parity;                      // which half of the ping-pong is current
    // graphs of the resident step: [kind][parity], kind 0 = step with a full list build (re-sort), 1 = step that
    // reuses the lists
    // kind 2 = a full step that first runs one smoothing-length iteration (sph_params.adapt_h_every)
    cudaGraphExec_t gexec[3][2];
    long long glaunches[3][2];       // launches one replay stands for
    long long gkey_n[3][2];
    const void *gkey_dtused[3][2];
    int adapt_h_every;               // > 0: one iteration of sph_adapt_h every so many steps, inside sph_step
    float adapt_h_target;
    long long step_count;            // steps taken since the state was ingested
    RungCtl rc;                      // on only inside sph_step_rungs
    int rebuild_every;               // steps between two full list builds when skin > 0
    int steps_since_full;            // steps taken since the last full build
    bool force_full;                 // the next step must do a full build (state refreshed, h changed, ...)
    bool resident, have_density, have_predict, have_grad, have_force, have_derivs;
    cudaEvent_t ev[2 * SPH_T_COUNT];
    bool ev_used[SPH_T_COUNT];
    // sph_step_host: device staging (17 floats + 2 words per particle), a second stream that carries the positions back
    // to the host while the pair passes still run, and the state they go to
    float *stage;
    cudaStream_t copy_stream;
    cudaEvent_t ev_pos, ev_copied;
    // sph_step_host on a step that reuses the lists: u, S and a_ext travel on h2d_stream behind x, m, h, v and are taken
    // into the resident arrays (k_refresh<2>, second half of the kick) after the density pass
    cudaStream_t h2d_stream;
    cudaEvent_t ev_first, ev_second;     // the first group of copies is issued / the second group has landed
    sph_state *host_in;                  // != NULL: the staging arrays whose second group is still to be taken in
    cudaEvent_t ev_third;                // a_ext has landed (third group: taken in before CLOSE, SPH_INT_DEFER_AEXT)
    sph_state *host_in_g;                // != NULL: a_ext is still to be taken in
    sph_state *host_out;     // != NULL inside sph_step_host: {device staging arrays}; host_dst: where x, y, z go on the host
    float *host_dst[3];
    bool no_reuse_now;       // the lists of this build will not be reused (host-buffer steps): no skin, no ordering pass
    size_t ws_bytes;
};

#define SPH_CUDA(ctx, call)                                   \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) {                             \
            (ctx)->last_cuda = (int)e__;                      \
            return SPH_ECUDA;                                 \
        }                                                     \
    } while (0)

static inline int sph_div_up(long long a, long long b) { return (int)((a + b - 1) / b); }

// ---- launchers implemented in the .cu files ---------------------------------------------
size_t sph_cub_temp_bytes(long long n_max);
int sph_launch_ingest(sph_ctx *c, const sph_state *st, long long n);
int sph_launch_resort(sph_ctx *c);
int sph_launch_tree(sph_ctx *c);
int sph_launch_set_ref(sph_ctx *c);
int sph_launch_check(sph_ctx *c);
int sph_launch_density(sph_ctx *c, bool flagged_only);
int sph_launch_pair(sph_ctx *c, bool grad, bool force, bool flagged_only);
int sph_launch_predict(sph_ctx *c);
int sph_launch_close(sph_ctx *c, int phase, float dt, bool dt_from_device);
int sph_launch_kick_drift(sph_ctx *c, float dt, int parts = 3);
int sph_launch_rung_assign(sph_ctx *c, float dT, int R, const unsigned char *rungs);
int sph_launch_kick_drift_rung(sph_ctx *c, int n, int R, float dT);
int sph_launch_mark_need(sph_ctx *c);
int sph_launch_get_field(sph_ctx *c, const float *src, float *dst, int as_int);
int sph_launch_get_position(sph_ctx *c, int comp, float *dst);
int sph_launch_get_h(sph_ctx *c, float *dst);
int sph_launch_get_tile(sph_ctx *c, float *dst);
int sph_launch_diagnostics(sph_ctx *c, double *out);
int sph_launch_h_update(sph_ctx *c, float n_target);
int sph_launch_neighbors(sph_ctx *c, int which, int *counts, const long long *offsets, int *list, bool flagged_only);
int sph_launch_download(sph_ctx *c, sph_state *st, int part);      // part: 0 everything, 1 positions, 2 the rest
int sph_launch_cull(sph_ctx *c, bool dirty_only);
int sph_launch_list_sort(sph_ctx *c);
int sph_launch_density_l(sph_ctx *c);
int sph_launch_pair_l(sph_ctx *c, bool grad, bool force);
int sph_launch_neighbors_l(sph_ctx *c, int which, int *counts, const long long *offsets, int *list);

// ---- small device helpers ----------------------------------------------------------------
#ifdef __CUDACC__
// is particle i active at the end of this substep? (everything is, outside sph_step_rungs)
__device__ __forceinline__ bool sph_active(const RungCtl &rc, long long i)
{
    return !rc.on || ((rc.n1 & ((1 << (rc.R - (int)rc.rung[i])) - 1)) == 0);
}

__device__ __forceinline__ float sph_r2(float dx, float dy, float dz)
{
    // reading Q4: every multiply and add rounded separately (no FMA contraction)
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}
__device__ __forceinline__ float sph_H(float kappa, float h) { return __fmul_rn(kappa, h); }

// Block b of a tile kernel launched with grid = heavy_cap + ntile: blocks [0, heavy_cap) take the heavy
// list, the rest take the remaining tiles in curve order; -1 = nothing to do for this block.
__device__ __forceinline__ int sph_tile_of_block(const Dev &d, int b)
{
    if (b < d.heavy_cap) return b < (int)*d.nheavy ? (int)d.heavy_list[b] : -1;
    const int t = b - d.heavy_cap;
    return d.heavy_mark[t] ? -1 : t;
}

// Rounds of a tile with ncand candidates: SPH_SE slots each, the last one shorter.  (Measured on configs[4], 1967
// candidates per tile on average, i.e. 1632 + 335 with the 1632 slots of that measurement: the 32 lists of a chunk are padded to equal length in every
// round, 30 % of the slots the pair passes step through are padding; rounds of EQUAL size, 2 x 984, were tried
// and are worse, 56 % -- the candidates are in curve order, an even split cuts through every chunk's neighbourhood.)
__host__ __device__ __forceinline__ int sph_round_count(int ncand) { return (ncand + SPH_SE - 1) / SPH_SE; }
__host__ __device__ __forceinline__ int sph_round_size(int) { return SPH_SE; }

// order-preserving float <-> int map for atomicMin/atomicMax on floats
__device__ __forceinline__ int sph_f2ord(float f)
{
    int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float sph_ord2f(int i)
{
    return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff);
}
#endif
