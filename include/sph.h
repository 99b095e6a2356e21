/*
 * sph.h -- C ABI of libsph.so: one SPH time step of a solid body with pressure-dependent
 * shear strength (arxiv/paper_2603_19764, section 2), hand-written CUDA for sm_100a.
 *
 * Citations are PAPER.md:<line> (section / equation) of /root/reference/PAPER.md; "reading Qn"
 * refers to DESIGN.md section 3.  No torch types cross this boundary: plain pointers and sizes.
 *
 * Conventions
 *  - Every pointer marked DEVICE is a CUDA device pointer, HOST a host pointer.
 *  - Every call returns SPH_OK (0) or a negative SPH_E* code; nothing throws.
 *  - Every call except sph_get_timings, sph_get_counters and sph_step_host is asynchronous on
 *    the CUDA stream given to sph_init and never synchronises the device.
 *  - The caller owns every particle array and the workspace; the library owns only the small
 *    host-side context.  The workspace must stay alive and untouched until sph_destroy.
 *  - Internally particles are kept sorted along a space-filling curve (Hilbert by default, Morton with
 *    SPH_MORTON_ORDER): the "resident" state.  Outputs of
 *    sph_get_field / sph_get_neighbors / sph_download_state are in CALLER order.
 *  - Particle arrays are fp32 structure-of-arrays, length n (BASELINE.json north_star).
 */
#ifndef SPH_H_
#define SPH_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_MAX_MATERIALS 8

/* sph_params.flags */
#define SPH_STRENGTH              1u  /* evolve S, add the S terms of Eq. 18-19      */
#define SPH_CORRECTION_TENSOR     2u  /* G = F.C (Eq. 22); off: C = 1      */
#define SPH_PCLIP_GLOBAL          4u  /* clip P >= 0 in the EOS too, not only in Eq. 34 (reading Q8)    */
#define SPH_JAUMANN_AS_PRINTED  512u  /* rotation terms of Eq. 13 with the index order AS PRINTED, S.R - R.S,
                                         instead of the objective (co-rotational) Jaumann rate R.S - S.R that
                                         is the default (reading Q1: the print contradicts "objective")     */
/* Retired bits: 8 (once SPH_JAUMANN_COROTATIONAL, the opposite choice under the opposite default), 128, 256.  sph_init and
 * sph_workspace_bytes refuse them, and any other bit not listed here, with SPH_EINVAL / 0 instead of ignoring them. */
#define SPH_NO_LISTS             16u  /* pair passes walk the chunk tree themselves instead of reading
                                         the per-particle neighbour lists (the round-1 "v0" kernels: A/B
                                         measurement; they also serve tiles over a list capacity)           */
#define SPH_NO_GRAPH             64u  /* launch the resident step kernel by kernel instead of replaying its
                                         CUDA graph (A/B measurement)                                      */
#define SPH_MORTON_ORDER         32u  /* sort by Morton (Z-order) keys instead of Hilbert keys (A/B
                                         measurement; results do not depend on the order)                  */

/* error codes */
#define SPH_OK         0
#define SPH_EINVAL    (-1)  /* bad argument (NULL, n < 0, unknown id, bad material index count)        */
#define SPH_ENOMEM    (-2)  /* workspace smaller than sph_workspace_bytes()                             */
#define SPH_ECUDA     (-3)  /* a CUDA call failed; sph_last_cuda_error() has the cudaError_t            */
#define SPH_EORDER    (-4)  /* pass called before its prerequisite (e.g. sph_forces before sph_density) */
#define SPH_ECAPACITY (-5)  /* n > n_max given to sph_init                                              */

/* sph_strength_update phases */
#define SPH_PREDICT     0   /* EOS, Gamma, Y, rescale S_pred, pack pair-pass operands */
#define SPH_CLOSE       1   /* G, eps_dot, R, dS/dt, closing kick + rescale       */
#define SPH_DERIVATIVES 2   /* as SPH_CLOSE but leaves v, u, S untouched (bootstrap of the first step)       */

/* sph_get_neighbors sets (reading Q4: fp32 predicate) */
#define SPH_GATHER     0    /* { j : r2_ij < H_i^2 }, contains i            */
#define SPH_SYMMETRIC  1    /* { j != i : r2_ij < max(H_i^2, H_j^2) } */

/* sph_get_field ids; multi-component fields take id + component                                        */
enum {
    SPH_F_RHO = 0,      /* Eq. 1                                          */
    SPH_F_OMEGA,        /* Eq. 3                                          */
    SPH_F_P,            /* EOS pressure (after SPH_PCLIP_GLOBAL)          */
    SPH_F_CS,           /* sound speed                                    */
    SPH_F_T,            /* temperature u_pred / cv                        */
    SPH_F_GAMMA,        /* shear modulus, Eq. 30 or constant              */
    SPH_F_Y,            /* yield strength, Eq. 34-37                      */
    SPH_F_MUMAX,        /* max_j |min(0, mu_ij)|, Eq. 39                  */
    SPH_F_DUDT,         /* Eq. 8 + Eq. 19                                 */
    SPH_F_DT,           /* per-particle time-step limit, Eq. 38-39        */
    SPH_F_EACC,         /* accumulated 1/2 eps_dot:eps_dot dt, Eq. 43     */
    SPH_F_EPS2,         /* 1/2 eps_dot:eps_dot of the last CLOSE          */
    SPH_F_U,            /* u after the closing kick                       */
    SPH_F_CFLAG,        /* 1.0 where C fell back to 1 (reading Q9)        */
    SPH_F_NGATHER,      /* |gather set| as float                          */
    SPH_F_NSYMMETRIC,   /* |symmetric set| as float                       */
    SPH_F_H,            /* smoothing length (after sph_adapt_h)           */
    SPH_F_RUNG,         /* rung of the last sph_step_rungs, as float      */
    SPH_F_TILE,         /* tile (256 curve-consecutive resident particles) the particle sits in, as float: the
                           index into the arrays of sph_get_tile_stats / sph_get_tile_dirty (test hook)       */
    SPH_F_A = 32,       /* +0..2   acceleration, Eq. 18 (+ a_ext)         */
    SPH_F_V = 36,       /* +0..2   velocity after the closing kick        */
    SPH_F_X = 40,       /* +0..2   position                               */
    SPH_F_SPRED = 48,   /* +0..4   predicted + rescaled S (xx,yy,xy,xz,yz)*/
    SPH_F_S = 56,       /* +0..4   S after the closing kick + rescale     */
    SPH_F_DSDT = 64,    /* +0..4   dS/dt, Eq. 13 / 25-29                  */
    SPH_F_F = 80,       /* +0..8   raw velocity gradient, Eq. 20, 3*a+b   */
    SPH_F_CINV = 96,    /* +0..8   C^-1, Eq. 21                           */
    SPH_F_G = 112       /* +0..8   corrected gradient, Eq. 22             */
};

/* sph_get_timings slots (milliseconds of the last call of each pass; CUDA events) */
enum { SPH_T_BUILD = 0, SPH_T_DENSITY, SPH_T_PREDICT, SPH_T_GRADIENT, SPH_T_FORCE, SPH_T_CLOSE,
       SPH_T_KICKDRIFT, SPH_T_STEP, SPH_T_COUNT };

/* sph_get_counters slots (from the last pass of each kind) */
enum { SPH_C_PAIRS_GATHER = 0,   /* sum_i |gather set(i)|   (true pairs of the density pass)    */
       SPH_C_PAIRS_SYMMETRIC,    /* sum_i |symmetric set(i)| (true pairs of gradient/force)     */
       SPH_C_TESTS_DENSITY,      /* candidate pairs the density pass tested                     */
       SPH_C_TESTS_FORCE,        /* candidate pairs the gradient/force pass tested              */
       SPH_C_CFALLBACK,          /* particles whose C fell back to 1                             */
       SPH_C_TESTS_CULL,         /* candidate pairs the list build tested (sph_build_neighbors) */
       SPH_C_CANDIDATES,         /* sum over tiles of the tile candidate-list lengths           */
       SPH_C_LIST_OVERFLOW,      /* tiles (256 particles) that exceeded a list capacity and were served
                                    by the tree-walk kernels instead: results are complete, the step is
                                    slower; raise sph_params.list_budget if this is large           */
       SPH_C_BAD_MATERIAL,       /* particles ingested with a material index outside 0..n_materials-1 (they were
                                    given material n_materials-1; see sph_state.mat)                        */
       SPH_C_OMEGA_SMALL,        /* particles with |Omega| < 0.1 in the last density pass (Eq. 3): too few
                                    neighbours for the grad-h terms; sph_adapt_h is the method's remedy     */
       SPH_C_NONFINITE,          /* particles whose a, du/dt or dS/dt was not finite in the last CLOSE      */
       SPH_C_TILES_DIRTY,        /* sph_params.skin > 0: tiles whose lists are rebuilt in every step since the
                                    last full build (0 right after one)                                      */
       SPH_C_ACTIVE_UPDATES,     /* sph_step_rungs: closing kicks done in the last big step (n 2^max_rung if every
                                    particle sat on the finest rung)                                           */
       SPH_C_ACTIVE_TILES,       /* sph_step_rungs: tiles the pair pass worked on, summed over the substeps    */
       SPH_C_PAIRS_INTILE,       /* symmetric pairs whose two particles sit in the same tile (counted by
                                    sph_get_neighbors(SPH_SYMMETRIC): the share a tile could evaluate once)     */
       SPH_C_LIST_SLOTS,         /* list slots the pair passes step through per launch: entries plus the padding
                                    that makes the 32 lists of a chunk equally long in every round (last build) */
       SPH_C_RUNG_CLAMPED,       /* sph_step_rungs with rungs from the limits: rung choices (at the start of the big
                                    step and at every closing kick) that put a particle on max_rung although its limit
                                    (Eq. 38-39) is below dT / 2^max_rung, or is not a number: such a particle is stepped
                                    beyond its limit; raise max_rung or lower dT if this is not 0                     */
       SPH_C_STEPS_SINCE_FULL,   /* steps taken on the lists of the last full neighbour build: 0 right after a call that
                                    did a full build (re-sort + lists), k after the k-th step that reused them (kept
                                    on the host; the way to tell which kind of step the last sph_step was)            */
       SPH_C_COUNT };

typedef struct sph_ctx sph_ctx;   /* opaque, library-owned (host memory) */

/* Per-material constants.  EOS stand-in (reading Q13, BASELINE.json
 * configs[0]): P = c0^2 (rho - rho0), c = c0, T = u / cv. */
typedef struct sph_material {
    float rho0, c0, cv;
    float Gamma;   /* > 0: constant shear modulus; <= 0: Eq. 30 with nu            */
    float nu;      /* Poisson ratio of Eq. 30                                  */
    float Y0, Ym, mu_i;   /* Eq. 34                                               */
    float mu_d;    /* Eq. 35-36; +INFINITY disables the min rule (reading Q10) */
    float xi, Tmelt;      /* Eq. 37                                               */
} sph_material;

typedef struct sph_params {
    float kappa;               /* support radius H = kappa h (reading Q3; default 2)              */
    float alpha, beta, eps_av; /* Eq. 5-6                                        */
    float eta_C, eta_a;        /* Eq. 38-39; eta_a <= 0 disables Eq. 38        */
    int n_materials;           /* 1..SPH_MAX_MATERIALS                                            */
    unsigned flags;            /* SPH_STRENGTH | ...                                              */
    sph_material mat[SPH_MAX_MATERIALS];
    int list_budget;           /* neighbour-list capacity: a quarter of the longest neighbour list a
                                  particle may have (8 bytes of workspace per particle and unit);
                                  <= 0 selects 64 (256 neighbours).  Tiles that need more are served by
                                  the tree-walk kernels and counted in SPH_C_LIST_OVERFLOW.           */
    float skin;                /* list reuse inside sph_step: > 0: a full neighbour build
                                  (re-sort + lists) keeps every pair within (1 + skin) of its cut-off, and the
                                  following steps reuse those lists -- the exact fp32 predicate (reading Q4) is
                                  evaluated on the current positions inside the pair passes, so the neighbour
                                  SETS are the same as with skin = 0 -- until the next full build; tiles whose
                                  surroundings moved by more than skin * H against them are rebuilt in every
                                  step (SPH_C_TILES_DIRTY).  <= 0: every step is a full build.             */
    int rebuild_every;         /* skin > 0: steps from one full build to the next (<= 0 selects 8)          */
    int adapt_h_every;         /* > 0: sph_step runs one iteration of sph_adapt_h (Eq. 2)
                                  every adapt_h_every steps, before the neighbour build of that step, with  */
    float adapt_h_target;      /* ... this n_target (the method's remedy for Omega -> 0, SPH_C_OMEGA_SMALL)  */
} sph_params;

/* NEXT-3: a tabulated EOS for one material (P and T are computed from rho and u by the EOS
 * library; T_melt "is provided as a tabulated function of density").  Uniform grids; value k of an axis
 * sits at min + k (max - min)/(n - 1).  P, T, cs: DEVICE, row-major [n_rho][n_u].  Tmelt: DEVICE [n_melt]
 * over [rho_min, rho_max], or NULL (the material's constant Tmelt).  The arrays are caller-owned and
 * must stay valid while the table is set. */
typedef struct sph_eos_table {
    int n_rho, n_u, n_melt;
    float rho_min, rho_max, u_min, u_max;
    const float *P, *T, *cs;
    const float *Tmelt;
} sph_eos_table;

/* Caller-owned particle arrays, each of length n.  For the device entry points all pointers are
 * DEVICE pointers; for sph_step_host all are HOST pointers.  S is symmetric and traceless, five
 * stored components (Eq. 11).  gx,gy,gz (external acceleration, the "G" term of
 * Eq. 18 supplied as input), mat and fixed may be NULL (= 0, material 0, nothing fixed). */
typedef struct sph_state {
    float *x, *y, *z, *m, *h, *vx, *vy, *vz, *u;
    float *Sxx, *Syy, *Sxy, *Sxz, *Syz;
    const float *gx, *gy, *gz;
    const int *mat;              /* material index per particle, 0..n_materials-1; an index outside that
                                    range is replaced by n_materials-1 and counted (SPH_C_BAD_MATERIAL)  */
    const unsigned char *fixed;  /* 1: particle skips kick and drift (reading Q16)  */
} sph_state;

/* Bytes of DEVICE workspace sph_init needs for up to n_max particles (0 on bad arguments). */
size_t sph_workspace_bytes(const sph_params *params, long long n_max);

/* Create a context.  params: HOST.  workspace: DEVICE, >= sph_workspace_bytes(), 256-byte aligned.
 * cuda_stream: a cudaStream_t (NULL = default stream; the resident step is replayed from a CUDA graph
 * only on a stream that can be captured, i.e. not on the default stream).  Errors: EINVAL, ENOMEM, ECUDA. */
int sph_init(sph_ctx **ctx, const sph_params *params, long long n_max,
             void *workspace, size_t workspace_bytes, void *cuda_stream);

/* S1: Morton keys -> radix sort -> gather into the resident sorted arrays -> chunk bounding boxes
 * and chunk tree -> per-tile candidate lists and per-particle neighbour lists (the symmetric set)
 * that the pair passes read (stands in for the paper's tree build).
 * state != NULL: ingest the caller's arrays (DEVICE), n particles; derivatives carried between
 * steps are reset.  state == NULL: re-sort the resident particles at their current positions.
 * n = 0 is legal.  Errors: EINVAL, ECAPACITY, EORDER (state == NULL with nothing resident). */
int sph_build_neighbors(sph_ctx *ctx, const sph_state *state, long long n);

/* S2: rho_i (Eq. 1), Omega_i (Eq. 3), |gather set|.  Needs sph_build_neighbors. */
int sph_density(sph_ctx *ctx);

/* NEXT-1 (the step before the path): adaptive smoothing length.  `iterations`
 * Newton-Raphson updates of the resident h_i towards a constant effective kernel mass (Eq. 2),
 *   M_tot,i = (4/3) pi (kappa h_i)^3 rho_i(h_i) = n_target m_i,
 * with the slope from Eq. 3: h <- h [1 - (1 - n_target m / M_tot) / (3 max(Omega, 0.1))], the factor
 * limited to [0.8, 1.25] (reading Q20 in DESIGN.md).  Every iteration is one density pass (skipped when
 * a current one exists), the per-particle update, and a rebuild of the chunk boxes, tree and neighbour
 * lists for the new support radii; the particle order is kept.  Afterwards the lists are current and
 * sph_density is the next call.  max_change: DEVICE pointer to one float (max_i |factor - 1| of the last
 * iteration) or NULL.  The caller's h array is not written: read h with sph_get_field(SPH_F_H).
 * Asynchronous.  Errors: EINVAL (n_target <= 0, iterations < 0), EORDER (nothing resident). */
int sph_adapt_h(sph_ctx *ctx, float n_target, int iterations, float *max_change);

/* S3 / S6: per-particle strength update, phase = SPH_PREDICT | SPH_CLOSE | SPH_DERIVATIVES.
 * PREDICT needs sph_density; CLOSE needs sph_gradients (if SPH_STRENGTH) and sph_forces.
 * dt is the step of the closing half kick (ignored by PREDICT and DERIVATIVES). */
int sph_strength_update(sph_ctx *ctx, int phase, float dt);

/* S4: F_i (Eq. 20), C_i^-1 (Eq. 21) over the symmetric set.  Needs PREDICT. */
int sph_gradients(sph_ctx *ctx);

/* S5: a_i (Eq. 4, 7, 18 + a_ext), du_i/dt (Eq. 8, 19), mu_max (Eq. 39).  Needs PREDICT. */
int sph_forces(sph_ctx *ctx);

/* S4 + S5 in ONE pass over the neighbour lists (both are sums over the same symmetric set):
 * the kernel sph_step itself runs.  Same outputs as sph_gradients followed by sph_forces.  Without
 * SPH_STRENGTH it is sph_forces.  Needs PREDICT. */
int sph_gradients_forces(sph_ctx *ctx);

/* One full step (Eq. 40-42): opening kick, drift,
 * prediction, S1..S6 (gradient and force passes fused), next dt.  state != NULL (DEVICE arrays):
 * ingested first if nothing is resident, and written back (x, v, u, S) in caller order at the
 * end; state == NULL: everything stays resident.  dt > 0: use it; dt <= 0: use the CFL step of
 * the previous derivatives (Eq. 39).  dt_used: DEVICE pointer to one float, or NULL. */
int sph_step(sph_ctx *ctx, sph_state *state, long long n, float dt, float *dt_used);

/* NEXT-4 ("hierarchical individual timestep scheme"; reading Q23 in DESIGN.md): ONE BIG
 * STEP dT of the resident particles on power-of-two rungs.  dT is split into 2^max_rung substeps; a particle on rung r
 * takes steps dT / 2^r, r the smallest rung whose step is within the particle's limit (Eq. 38-39) from its last
 * CLOSE -- or max_rung when even dT / 2^max_rung exceeds the limit (counted in SPH_C_RUNG_CLAMPED; nothing else signals it).  Per substep: opening kick of the particles that start a step, drift of all, prediction of all to the new
 * time from their own last derivatives, neighbour lists (reused, checked, rebuilt where dirty), then density and
 * PREDICT for the tiles that hold an active particle or a neighbour of one, the fused pair pass for the tiles that
 * hold an active particle, CLOSE (own step, rescale, next rung) for the active particles only: tiles (256 particles)
 * without active particles cost nothing in the pair passes.  The particle order is kept for the whole big step.
 * rungs: DEVICE unsigned char[n] in caller order = fixed rungs for this big step (test hook), or NULL = from the
 * limits.  max_rung in [0, 16]; dT > 0.  Needs a resident state; derivatives are bootstrapped if none are carried.
 * Afterwards every particle is at t + dT; SPH_F_RUNG has the rungs, SPH_C_ACTIVE_UPDATES the closing kicks done.
 * Errors: EINVAL, EORDER. */
int sph_step_rungs(sph_ctx *ctx, float dT, int max_rung, const unsigned char *rungs);

/* The same step through HOST buffers: copies the state host->device into library-owned staging,
 * steps, copies x, v, u, S back device->host, and synchronises the stream.  dt_used: HOST.
 * If the caller's x, y, z, h equal the resident ones bit for bit (a loop that hands back what it was given) the
 * neighbour lists stay in use as in sph_step; if anything moved, the step starts from a full neighbour build.
 * mat and fixed are read at the FIRST call only (they stay with the resident particles).  Copies overlap the step
 * where the data flow allows: on a step that reuses the lists u and S arrive on a second stream while the first half
 * of the kick, the list check and the density pass run, a_ext while the pair pass runs (CLOSE adds it then, with
 * the same single rounding); x, y, z leave during the pair pass.  With
 * sph_params.adapt_h_every > 0 the smoothing lengths the step adapted are written back to host_state->h as well (the
 * host state stays the resident one, and the lists stay in use between the adaptation steps); otherwise m and h are
 * only read.  If the call fails part way it waits for every copy it issued before it returns (the host arrays are the
 * caller's again), and the next step starts from a full build.  All host
 * arrays should be pinned (pageable memory works, without the overlap) and must not be touched during the call. */
int sph_step_host(sph_ctx *ctx, sph_state *host_state, long long n, float dt, float *dt_used);

/* Write x, v, u, S of the resident particles to the caller's DEVICE arrays in caller order. */
int sph_download_state(sph_ctx *ctx, sph_state *state);

/* Copy one scalar field (enum above, id + component) to dst (DEVICE, n floats, caller order). */
int sph_get_field(sph_ctx *ctx, int field_id, float *dst);

/* Test hook: neighbour sets as the pair passes see them, as ORIGINAL particle ids.
 * counts: DEVICE int[n].  If list != NULL, offsets (DEVICE long long[n+1], exclusive prefix of
 * counts, supplied by the caller) says where each particle's ids go; order within a row is
 * unspecified; a particle with offsets[i] < 0 is skipped (its ids are not written: sampled comparisons
 * at sizes where the whole list would not fit).  The capacity of list is NOT checked on the device; the
 * caller sizes it from counts. */
int sph_get_neighbors(sph_ctx *ctx, int which, int *counts, const long long *offsets, int *list);

/* NEXT-3: use `table` (HOST struct, DEVICE arrays) for P, T, c_s (and T_melt) of `material` in
 * sph_strength_update(SPH_PREDICT) and every pass after it, instead of the analytic stand-in; NULL
 * returns to the analytic EOS.  Lookup: bilinear (T_melt: piecewise linear), clamped to the grid's edges
 * (reading Q21 in DESIGN.md); cell index and weights in fp64 from the fp64 density.  SPH_PCLIP_GLOBAL
 * still clips P >= 0 afterwards.  Host-only call (no launch); passes from PREDICT on must be redone.
 * Errors: EINVAL (material out of range, grid < 2 points, NULL arrays, empty ranges). */
int sph_set_eos_table(sph_ctx *ctx, int material, const sph_eos_table *table);

/* S8 diagnostics (the conservation checks of PAPER.md:349-357): out = DEVICE double[8] =
 * { sum m, sum m v (3), sum m x cross v (3), sum m (v.v/2 + u) } over the resident particles at the
 * full step (after the last closing kick; the ingested state before any step), accumulated in fp64
 * in a fixed order (bitwise repeatable).  Asynchronous.  Errors: EINVAL, EORDER. */
int sph_get_diagnostics(sph_ctx *ctx, double *out);

/* The same eight sums for callers that cannot allocate device memory -- no context, no workspace.
 * Meant for two kinds of caller: a host code that gave the whole GPU to its own particle pool at start-up, so
 * that any later cudaMalloc (the workspace sph_init wants) fails; and a time-step loop that cannot afford the
 * device-wide synchronisation that cudaMalloc / cudaFree bring.  This call allocates nothing: the per-block
 * partial sums sit in a static __device__ array inside libsph.so (512 KiB; every GPU that loads the library's
 * kernels holds it until the process exits).  That fixes the limit: n <= SPH_DIAG_NOALLOC_MAX_N.
 *   state: HOST struct; its x, y, z, m, vx, vy, vz, u are DEVICE float[n] (the other members are not read), in any
 *          order -- this is the caller's state as it stands, not the resident one.
 *   out:   DEVICE double[8] = { sum m, sum m v (3), sum m x cross v (3), sum m (v.v/2 + u) },
 *          fp64, summed in a fixed order that depends on n only: repeatable bit for bit, and equal to
 *          sph_get_diagnostics of the same state up to the rounding of a different order (1e-12 relative).
 *   cuda_stream: a cudaStream_t (NULL = default stream); asynchronous on it.  n = 0 writes zeros.
 *   cuda_error: HOST int receiving the cudaError_t when SPH_ECUDA is returned, or NULL.
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 * current); make that first call outside any stream capture.  All calls on a device share the one array, which
 * keeps the last call's partial sums; a call reads only rows it has just written, so nothing needs clearing.
 * Calls that can overlap on the GPU (two streams of one device) race on it and give undefined sums: keep them on
 * one stream or order them with events.  Different devices do not interfere.
 * Errors: EINVAL (NULL state / out / a needed array, n < 0), ECAPACITY (n > SPH_DIAG_NOALLOC_MAX_N; nothing is
 * launched), ECUDA. */
#define SPH_DIAG_NOALLOC_MAX_N 33554432   /* 2^25 particles */
int sph_diagnostics_noalloc(const sph_state *state, long long n, double *out, void *cuda_stream, int *cuda_error);

/* HOST outputs.  Both synchronise the stream. */
int sph_get_timings(sph_ctx *ctx, float *ms, int n);            /* SPH_T_* slots              */
int sph_get_counters(sph_ctx *ctx, long long *counters, int n); /* SPH_C_* slots              */

/* Diagnostic: per-tile statistics of the last neighbour build (tile = 256 curve-consecutive particles).
 * ncand / cycles / flag: HOST arrays of `capacity` entries, each may be NULL: candidates staged for the
 * tile, SM clock cycles the list builder spent on it, and whether it fell back to the tree-walk kernels.
 * Returns the number of tiles (nothing is copied if capacity is smaller), or a negative SPH_E* code.
 * Synchronises the stream. */
int sph_get_tile_stats(sph_ctx *ctx, int *ncand, unsigned *cycles, unsigned char *flag, int capacity);

/* Diagnostic / test hook: which tiles are "dirty" (sph_params.skin > 0): their surroundings moved by more than the skin
 * since the last full build, and their lists are rebuilt in every step until the next one (SPH_C_TILES_DIRTY is their
 * number).  dirty: HOST array of `capacity` bytes (1 = dirty).  Returns the number of tiles (nothing is copied if
 * capacity is smaller or dirty is NULL), or a negative SPH_E* code.  Synchronises the stream. */
int sph_get_tile_dirty(sph_ctx *ctx, unsigned char *dirty, int capacity);

/* Measurement aid ("measure an FMA-chain microbenchmark"): the FP32 CUDA-core rate this
 * device sustains on a kernel of independent FFMA chains (2 flop each, no memory traffic), in TFLOP/s, best of
 * `repeats` launches timed with CUDA events on `cuda_stream`.  tflops: HOST.  Synchronises the stream.
 * It is the denominator of the ALU-bound roofline entries of bench.py. */
int sph_fp32_peak(void *cuda_stream, int repeats, double *tflops);

/* The same measurement for other instruction forms (variant 0 is sph_fp32_peak): 1 = scalar FFMA with three register
 * operands, 2 = packed FFMA2 (fma.rn.f32x2) with three 64-bit register operands, 3 / 4 = variants 1 / 2 with one independent
 * integer ALU instruction per FP32 instruction.  TFLOP/s (2 flop per FFMA, 4 per FFMA2).  It answers whether packed FP32
 * arithmetic frees issue slots on this device; nothing on the step path calls it.  Synchronises. */
int sph_fp32_rate(void *cuda_stream, int variant, int repeats, double *tflops);

/* Number of this library's kernel launches since sph_init (HOST; no synchronisation). */
long long sph_launch_count(const sph_ctx *ctx);

int sph_last_cuda_error(const sph_ctx *ctx);
const char *sph_strerror(int code);
void sph_destroy(sph_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* SPH_H_ */
