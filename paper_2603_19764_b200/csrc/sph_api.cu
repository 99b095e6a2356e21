// sph_api.cu -- the C ABI of include/sph.h: workspace layout, pass sequencing, timings.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "sph_internal.cuh"

// ------------------------------------------------------------------------------------------
// workspace layout: one bump allocation, 256-byte aligned pieces
// ------------------------------------------------------------------------------------------
struct Bump {
    char *base;
    size_t off;
    template <class T> T *take(size_t count)
    {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? (T *)(base + off) : (T *)nullptr;
        off += count * sizeof(T);
        return p;
    }
};

static void tree_counts(long long n_max, int *count, int *nlev)
{
    int cnt = sph_div_up(n_max > 0 ? n_max : 1, SPH_CHUNK), L = 0;
    count[0] = cnt;
    while (cnt > SPH_ARITY && L + 1 < SPH_MAX_LEVELS) {
        cnt = sph_div_up(cnt, SPH_ARITY);
        count[++L] = cnt;
    }
    *nlev = L + 1;
}

static int kcap_of(const sph_params *p)          // row-groups of the neighbour lists reserved per chunk
{
    int r = p->list_budget > 0 ? p->list_budget : SPH_ROWS_DEFAULT;
    return r > 16000 ? 16000 : r;                 // rowptr entries are 16-bit
}

static int sm_count_cached = 0;
static int device_sm_count()
{
    if (sm_count_cached > 0) return sm_count_cached;
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
        sm_count_cached = n;
    else {
        (void)cudaGetLastError();
        return 148;                       // sizing on a box without a GPU: B200
    }
    return sm_count_cached;
}

static float skin_of(const sph_params *p)
{
    if (!(p->skin > 0.f) || (p->flags & SPH_NO_LISTS)) return 0.f;
    return p->skin > 0.5f ? 0.5f : p->skin;
}

static size_t carve(Dev *d, float **stage, char *base, long long n_max, int kcap, bool lists, float skin)
{
    const int sm_count = device_sm_count();
    Bump b{base, 0};
    size_t N = (size_t)(n_max > 0 ? n_max : 1);
    Dev tmp;
    Dev &o = d ? *d : tmp;
    o.n_max = n_max;
    for (int k = 0; k < 2; ++k) {
        Resident &r = k ? o.alt : o.r;
        r.pm = b.take<float4>(N);
        r.vh = b.take<float4>(N);
        for (int f = 0; f < SPH_NPP; ++f) r.s[f] = b.take<float>(N);
    }
    int count[SPH_MAX_LEVELS], nlev;
    tree_counts(n_max, count, &nlev);
    for (int L = 0; L < SPH_MAX_LEVELS; ++L) {
        size_t c = L < nlev ? (size_t)count[L] : 1;
        o.tree.lo[L] = b.take<float4>(c);
        o.tree.hi[L] = b.take<float4>(c);
        o.tree.dlo[L] = b.take<float4>(skin > 0.f ? c : 1);
        o.tree.dhi[L] = b.take<float4>(skin > 0.f ? c : 1);
    }
    o.skin = skin;
    o.xref = b.take<float4>(skin > 0.f ? N : 1);
    for (int k = 0; k < 3; ++k) o.vfull[k] = b.take<float>(N);
    o.ufull = b.take<float>(N);
    for (int k = 0; k < 5; ++k) o.Sfull[k] = b.take<float>(N);
    for (int k = 0; k < 3; ++k) o.a[k] = b.take<float>(N);
    o.dudt = b.take<float>(N);
    for (int k = 0; k < 5; ++k) o.dS[k] = b.take<float>(N);
    o.rho = b.take<float>(N); o.omega = b.take<float>(N); o.P = b.take<float>(N); o.cs = b.take<float>(N);
    o.T = b.take<float>(N); o.Gamma = b.take<float>(N); o.Y = b.take<float>(N); o.mumax = b.take<float>(N);
    o.dti = b.take<float>(N); o.eps2 = b.take<float>(N); o.cflag = b.take<float>(N);
    o.rho64 = b.take<double>(N);
    o.mK = b.take<float>(N);
    o.ngather = b.take<int>(N); o.nsym = b.take<int>(N);
    for (int k = 0; k < 9; ++k) o.F[k] = b.take<float>(N);
    for (int k = 0; k < 9; ++k) o.Cinv[k] = b.take<float>(N);
    for (int k = 0; k < 9; ++k) o.G[k] = b.take<float>(N);
    o.B3 = b.take<float4>(N); o.B4 = b.take<float4>(N); o.B5 = b.take<float2>(N);
    size_t ntile = (N + SPH_TILE - 1) / SPH_TILE;
    size_t nchunk = (N + SPH_CHUNK - 1) / SPH_CHUNK;
    o.tile_ncand = b.take<int>(ntile);
    o.tile_off = b.take<unsigned long long>(ntile);
    o.tile_flag = b.take<unsigned char>(ntile);
    o.tile_cycles = b.take<unsigned>(ntile);
    o.cull_cycles = b.take<unsigned long long>(1);
    o.heavy_cap = (int)(ntile / 16 < 16 ? 16 : (ntile / 16 > 2048 ? 2048 : ntile / 16));
    o.heavy_list = b.take<unsigned>(o.heavy_cap);
    o.nheavy = b.take<unsigned>(1);
    o.heavy_mark = b.take<unsigned char>(ntile);
    o.tile_dirty = b.take<unsigned char>(ntile);
    o.tile_act = b.take<unsigned char>(ntile);
    o.tile_need = b.take<unsigned char>(ntile);
    o.rung = b.take<unsigned char>(N);
    o.cand_cursor = b.take<unsigned long long>(2);
    o.cand_cap = lists ? (unsigned long long)ntile * SPH_POOL_PER_TILE : 1;   // pool: twice the one-round average
    o.cand_cap_dirty = (lists && skin > 0.f) ? (unsigned long long)ntile * (SPH_POOL_PER_TILE / 2) : 0;
    o.cand = b.take<unsigned>((size_t)(o.cand_cap + o.cand_cap_dirty));
    o.rows_cap = kcap;
    o.rowptr = b.take<unsigned short>(lists ? nchunk * (SPH_MAXROUND + 1) : 1);
    o.nlist = b.take<uint2>(lists ? nchunk * (size_t)kcap * 32 : 1);
    o.far_point = b.take<float4>(1);
    o.nlen = b.take<int>(N);
    o.cull_grid = (int)ntile;
    o.walk_grid = 2 * sm_count;
    o.bbox = b.take<float>(8);
    o.dt_cur = b.take<float>(1);
    o.dt_next = b.take<float>(1);
    o.hchange = b.take<float>(1);
    o.refresh_changed = b.take<int>(1);
    o.diag_part = b.take<double>(592 * 8);
    o.counters = b.take<unsigned long long>(SPH_C_COUNT);
    o.keys = b.take<unsigned long long>(N); o.keys_alt = b.take<unsigned long long>(N);
    o.perm = b.take<unsigned>(N); o.perm_alt = b.take<unsigned>(N);
    o.cub_tmp_bytes = sph_cub_temp_bytes(n_max);
    o.cub_tmp = b.take<char>(o.cub_tmp_bytes);
    float *st = b.take<float>(19 * N);      // sph_step_host staging: 17 float arrays + mat + fixed
    if (stage) *stage = st;
    return (b.off + 255) & ~(size_t)255;
}

static bool params_ok(const sph_params *p)
{
    if (!p) return false;
    if (p->n_materials < 1 || p->n_materials > SPH_MAX_MATERIALS) return false;
    if (!(p->kappa > 0.f)) return false;
    const unsigned known = SPH_STRENGTH | SPH_CORRECTION_TENSOR | SPH_PCLIP_GLOBAL | SPH_JAUMANN_AS_PRINTED | SPH_NO_LISTS
                           | SPH_NO_GRAPH | SPH_MORTON_ORDER;
    if (p->flags & ~known) return false;     // retired bits (8, 128, 256) and unknown ones: refused, never ignored
    for (int k = 0; k < p->n_materials; ++k)
        if (!(p->mat[k].rho0 > 0.f) || !(p->mat[k].cv > 0.f) || !(p->mat[k].c0 > 0.f)) return false;
    return true;
}

extern "C" size_t sph_workspace_bytes(const sph_params *params, long long n_max)
{
    if (!params_ok(params) || n_max < 0 || n_max > 2000000000ll) return 0;
    return carve(nullptr, nullptr, nullptr, n_max, kcap_of(params), !(params->flags & SPH_NO_LISTS), skin_of(params));
}

extern "C" int sph_init(sph_ctx **out, const sph_params *params, long long n_max, void *workspace,
                        size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return SPH_EINVAL;
    *out = nullptr;
    if (!params_ok(params) || n_max < 0 || n_max > 2000000000ll || !workspace) return SPH_EINVAL;
    if (((uintptr_t)workspace & 255u) != 0) return SPH_EINVAL;
    size_t need = carve(nullptr, nullptr, nullptr, n_max, kcap_of(params), !(params->flags & SPH_NO_LISTS), skin_of(params));
    if (workspace_bytes < need) return SPH_ENOMEM;
    sph_ctx *c = new (std::nothrow) sph_ctx();
    if (!c) return SPH_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->p.kappa = params->kappa; c->p.alpha = params->alpha; c->p.beta = params->beta;
    c->p.eps_av = params->eps_av; c->p.eta_C = params->eta_C; c->p.eta_a = params->eta_a;
    c->p.flags = params->flags & ~SPH_INT_DEFER_AEXT; c->p.n_materials = params->n_materials;
    memcpy(c->p.mat, params->mat, sizeof(params->mat));
    c->stream = (cudaStream_t)cuda_stream;
    c->use_lists = !(params->flags & SPH_NO_LISTS);
    // a capture cannot be taken on the legacy default stream
    c->use_graph = !(params->flags & SPH_NO_GRAPH) && cuda_stream != nullptr && (cudaStream_t)cuda_stream != cudaStreamLegacy
                   && (cudaStream_t)cuda_stream != cudaStreamPerThread;
    c->ws_bytes = carve(&c->d, &c->stage, (char *)workspace, n_max, kcap_of(params), c->use_lists, skin_of(params));
    c->rebuild_every = params->rebuild_every > 0 ? params->rebuild_every : 8;
    c->adapt_h_every = (params->adapt_h_every > 0 && params->adapt_h_target > 0.f) ? params->adapt_h_every : 0;
    c->adapt_h_target = params->adapt_h_target;
    c->force_full = true;
    c->d.n = 0; c->d.nchunk = 0;
    for (int k = 0; k < 2 * SPH_T_COUNT; ++k) {
        cudaError_t e = cudaEventCreate(&c->ev[k]);
        if (e != cudaSuccess) {
            for (int j = 0; j < k; ++j) cudaEventDestroy(c->ev[j]);
            delete c;
            return SPH_ECUDA;
        }
    }
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess
        || cudaEventCreateWithFlags(&c->ev_pos, cudaEventDisableTiming) != cudaSuccess
        || cudaEventCreateWithFlags(&c->ev_copied, cudaEventDisableTiming) != cudaSuccess
        || cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking) != cudaSuccess
        || cudaEventCreateWithFlags(&c->ev_first, cudaEventDisableTiming) != cudaSuccess
        || cudaEventCreateWithFlags(&c->ev_second, cudaEventDisableTiming) != cudaSuccess
        || cudaEventCreateWithFlags(&c->ev_third, cudaEventDisableTiming) != cudaSuccess) {
        sph_destroy(c);
        return SPH_ECUDA;
    }
    cudaError_t e = cudaMemsetAsync(c->d.counters, 0, SPH_C_COUNT * sizeof(unsigned long long), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d.dt_cur, 0, sizeof(float), c->stream);
    {
        const size_t ntile = ((size_t)c->d.n_max + SPH_TILE - 1) / SPH_TILE;
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.tile_cycles, 0, ntile * sizeof(unsigned), c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.cull_cycles, 0, sizeof(unsigned long long), c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.nheavy, 0, sizeof(unsigned), c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.heavy_mark, 0, ntile, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.tile_dirty, 0, ntile, c->stream);
        // never written with SPH_NO_LISTS; the workspace arrives uninitialised
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.tile_flag, 0, ntile, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.tile_ncand, 0, ntile * sizeof(int), c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->d.tile_off, 0, ntile * sizeof(unsigned long long), c->stream);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d.dt_next, 0, sizeof(float), c->stream);
    if (e != cudaSuccess) { sph_destroy(c); return SPH_ECUDA; }
    *out = c;
    return SPH_OK;
}

static void drop_graphs(sph_ctx *c)
{
    for (int k = 0; k < 3; ++k)
        for (int s = 0; s < 2; ++s)
            if (c->gexec[k][s]) { cudaGraphExecDestroy(c->gexec[k][s]); c->gexec[k][s] = nullptr; }
}

extern "C" void sph_destroy(sph_ctx *c)
{
    if (!c) return;
    drop_graphs(c);
    for (int k = 0; k < 2 * SPH_T_COUNT; ++k)
        if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    if (c->ev_pos) cudaEventDestroy(c->ev_pos);
    if (c->ev_copied) cudaEventDestroy(c->ev_copied);
    if (c->ev_first) cudaEventDestroy(c->ev_first);
    if (c->ev_second) cudaEventDestroy(c->ev_second);
    if (c->ev_third) cudaEventDestroy(c->ev_third);
    if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
}

// ------------------------------------------------------------------------------------------
// timing helpers
// ------------------------------------------------------------------------------------------
struct PassTimer {
    sph_ctx *c;
    int slot;
    // inside a stream capture the record becomes an external event-record node, so that
    // cudaEventElapsedTime still works on the events after a graph launch
    static void record(sph_ctx *c, cudaEvent_t e)
    {
        cudaEventRecordWithFlags(e, c->stream, c->capturing ? cudaEventRecordExternal : cudaEventRecordDefault);
    }
    PassTimer(sph_ctx *c_, int s) : c(c_), slot(s) { record(c, c->ev[2 * slot]); }
    ~PassTimer()
    {
        record(c, c->ev[2 * slot + 1]);
        c->ev_used[slot] = true;
    }
};

static bool state_ok(const sph_state *s)
{
    return s && s->x && s->y && s->z && s->m && s->h && s->vx && s->vy && s->vz && s->u && s->Sxx && s->Syy &&
           s->Sxy && s->Sxz && s->Syz;
}

// ------------------------------------------------------------------------------------------
// passes
// ------------------------------------------------------------------------------------------
extern "C" int sph_build_neighbors(sph_ctx *c, const sph_state *state, long long n)
{
    if (!c) return SPH_EINVAL;
    int rc;
    PassTimer t(c, SPH_T_BUILD);
    if (state) {
        if (n < 0 || (n > 0 && !state_ok(state))) return SPH_EINVAL;
        if (n > c->d.n_max) return SPH_ECAPACITY;
        rc = sph_launch_ingest(c, state, n);
        if (rc) return rc;
        drop_graphs(c);
        c->resident = true;
        c->have_derivs = false;
        c->step_count = 0;
    } else {
        if (!c->resident) return SPH_EORDER;
        rc = sph_launch_resort(c);
        if (rc) return rc;
    }
    c->have_density = c->have_predict = c->have_grad = c->have_force = false;
    if (c->use_lists) {
        rc = sph_launch_set_ref(c);          // list reuse: the positions this full build refers to
        if (rc) return rc;
        rc = sph_launch_cull(c, false);
        if (rc) return rc;
    }
    c->steps_since_full = 0;
    c->force_full = false;
    return SPH_OK;
}

// The neighbour structure of a step that REUSES the lists of the last full build (sph_params.skin > 0): chunk
// boxes and tree at the current positions (with the displacement boxes), the check of every tile, and the
// rebuild of the dirty ones.  The particle order stays.
static int reuse_neighbors(sph_ctx *c)
{
    PassTimer t(c, SPH_T_BUILD);
    int rc = sph_launch_tree(c);
    if (rc) return rc;
    rc = sph_launch_check(c);
    if (rc) return rc;
    rc = sph_launch_cull(c, true);
    if (rc) return rc;
    c->have_density = c->have_predict = c->have_grad = c->have_force = false;
    c->steps_since_full++;
    return SPH_OK;
}

extern "C" int sph_density(sph_ctx *c)
{
    if (!c) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    PassTimer t(c, SPH_T_DENSITY);
    int rc = c->use_lists ? sph_launch_density_l(c) : sph_launch_density(c, false);
    if (rc) return rc;
    c->have_density = true;
    c->have_predict = c->have_grad = c->have_force = false;
    return SPH_OK;
}

extern "C" int sph_adapt_h(sph_ctx *c, float n_target, int iterations, float *max_change)
{
    if (!c || !(n_target > 0.f) || iterations < 0) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    int rc;
    for (int it = 0; it < iterations; ++it) {
        if (!c->have_density) {
            rc = sph_density(c);
            if (rc) return rc;
        }
        rc = sph_launch_h_update(c, n_target);
        if (rc) return rc;
        // new support radii: chunk boxes, tree and lists again (the curve order stays)
        rc = sph_launch_tree(c);
        if (rc) return rc;
        if (c->use_lists) {
            rc = sph_launch_set_ref(c);
            if (rc) return rc;
            rc = sph_launch_cull(c, false);
            if (rc) return rc;
            c->steps_since_full = 0;
        }
        c->have_density = c->have_predict = c->have_grad = c->have_force = false;
    }
    if (iterations > 0 && max_change)
        SPH_CUDA(c, cudaMemcpyAsync(max_change, c->d.hchange, sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    return SPH_OK;
}

extern "C" int sph_gradients(sph_ctx *c)
{
    if (!c) return SPH_EINVAL;
    if (!c->have_predict) return SPH_EORDER;
    PassTimer t(c, SPH_T_GRADIENT);
    int rc = c->use_lists ? sph_launch_pair_l(c, true, false) : sph_launch_pair(c, true, false, false);
    if (rc) return rc;
    c->have_grad = true;
    return SPH_OK;
}

extern "C" int sph_forces(sph_ctx *c)
{
    if (!c) return SPH_EINVAL;
    if (!c->have_predict) return SPH_EORDER;
    PassTimer t(c, SPH_T_FORCE);
    int rc = c->use_lists ? sph_launch_pair_l(c, false, true) : sph_launch_pair(c, false, true, false);
    if (rc) return rc;
    c->have_force = true;
    return SPH_OK;
}

extern "C" int sph_gradients_forces(sph_ctx *c)
{
    if (!c) return SPH_EINVAL;
    if (!c->have_predict) return SPH_EORDER;
    const bool strength = (c->p.flags & SPH_STRENGTH) != 0;
    PassTimer t(c, SPH_T_FORCE);
    int rc = c->use_lists ? sph_launch_pair_l(c, strength, true) : sph_launch_pair(c, strength, true, false);
    if (rc) return rc;
    c->have_force = true;
    c->have_grad = strength;
    return SPH_OK;
}

static int take_third_group(sph_ctx *c);

static int do_close(sph_ctx *c, int phase, float dt, bool dt_from_device)
{
    const bool strength = (c->p.flags & SPH_STRENGTH) != 0;
    if (!c->have_force || (strength && !c->have_grad)) return SPH_EORDER;
    if (c->host_in_g) {               // sph_step_host: a_ext has landed by now; this CLOSE adds it (SPH_INT_DEFER_AEXT)
        int rc = take_third_group(c);
        if (rc) return rc;
    }
    PassTimer t(c, SPH_T_CLOSE);
    int rc = sph_launch_close(c, phase, dt, dt_from_device);
    if (rc) return rc;
    c->have_derivs = true;
    return SPH_OK;
}

extern "C" int sph_strength_update(sph_ctx *c, int phase, float dt)
{
    if (!c) return SPH_EINVAL;
    if (phase == SPH_PREDICT) {
        if (!c->have_density) return SPH_EORDER;
        PassTimer t(c, SPH_T_PREDICT);
        int rc = sph_launch_predict(c);
        if (rc) return rc;
        c->have_predict = true;
        c->have_grad = c->have_force = false;
        return SPH_OK;
    }
    if (phase == SPH_CLOSE || phase == SPH_DERIVATIVES) {
        if (phase == SPH_CLOSE && !(dt >= 0.f)) return SPH_EINVAL;
        return do_close(c, phase, dt, false);
    }
    return SPH_EINVAL;
}

// density -> predict -> fused gradient + force
static int take_second_group(sph_ctx *c);

static int derivative_passes(sph_ctx *c)
{
    int rc = c->have_density ? SPH_OK : sph_density(c);
    if (rc) return rc;
    if (c->host_in) {                 // sph_step_host: u, S, a_ext have landed by now; second half of the kick
        rc = take_second_group(c);
        if (rc) return rc;
    }
    rc = sph_strength_update(c, SPH_PREDICT, 0.f);
    if (rc) return rc;
    return sph_gradients_forces(c);
}

// does the next step rebuild everything (re-sort, full list build) or reuse the lists?
static bool step_adapts_h(const sph_ctx *c)
{
    return c->adapt_h_every > 0 && (c->step_count + 1) % c->adapt_h_every == 0;
}

static bool step_is_full(const sph_ctx *c)
{
    return !(c->d.skin > 0.f) || !c->use_lists || c->force_full || c->steps_since_full + 1 >= c->rebuild_every
           || step_adapts_h(c);
}

static int step_body(sph_ctx *c, sph_state *state, long long n, float dt, float *dt_used)
{
    int rc;
    PassTimer ts(c, SPH_T_STEP);
    if (!c->resident) {
        if (!state) return SPH_EORDER;
        rc = sph_build_neighbors(c, state, n);
        if (rc) return rc;
    } else if (state && n != c->d.n) {
        return SPH_EINVAL;
    }
    if (!c->have_derivs) {          // first step: a_0, du_0/dt, dS_0/dt from the current state
        rc = derivative_passes(c);
        if (rc) return rc;
        rc = do_close(c, SPH_DERIVATIVES, 0.f, false);
        if (rc) return rc;
    }
    {
        PassTimer t(c, SPH_T_KICKDRIFT);
        rc = sph_launch_kick_drift(c, dt, c->host_in ? 1 : 3);
        if (rc) return rc;
    }
    const bool adapt = step_adapts_h(c);
    rc = step_is_full(c) ? sph_build_neighbors(c, nullptr, 0) : reuse_neighbors(c);
    if (rc) return rc;
    if (c->host_out && c->d.n > 0) {
        // sph_step_host: the positions are final (drift and re-sort done): scatter them to the staging arrays and let
        // the second stream carry them to the host while the pair passes run on this one
        rc = sph_launch_download(c, c->host_out, 1);
        if (rc) return rc;
        SPH_CUDA(c, cudaEventRecord(c->ev_pos, c->stream));
        SPH_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_pos, 0));
        float *src[3] = {c->host_out->x, c->host_out->y, c->host_out->z};
        for (int k = 0; k < 3; ++k)
            SPH_CUDA(c, cudaMemcpyAsync(c->host_dst[k], src[k], (size_t)c->d.n * sizeof(float), cudaMemcpyDeviceToHost,
                                        c->copy_stream));
        SPH_CUDA(c, cudaEventRecord(c->ev_copied, c->copy_stream));
    }
    if (adapt) {
        // one Newton-Raphson update of h towards a constant kernel mass at the new positions (density
        // pass, update, tree and lists again); the method's own remedy for particles that lose their neighbours
        rc = sph_adapt_h(c, c->adapt_h_target, 1, nullptr);
        if (rc) return rc;
    }
    c->step_count++;
    rc = derivative_passes(c);
    if (rc) return rc;
    rc = do_close(c, SPH_CLOSE, 0.f, true);
    if (rc) return rc;
    if (dt_used) SPH_CUDA(c, cudaMemcpyAsync(dt_used, c->d.dt_cur, sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    if (state) {
        rc = sph_launch_download(c, state, c->host_out ? 2 : 0);
        if (rc) return rc;
    }
    return SPH_OK;
}

// The resident step (state == NULL, CFL dt, derivatives carried) is about forty dependent launches with
// fixed arguments: it is captured once per half of the ping-pong into a CUDA graph and replayed, which
// removes the launch gaps (a third of the step at 2e5 particles).  Everything a replay does not do on
// the host -- the swap of the ping-pong halves, the pass flags, the launch count -- is redone here.
extern "C" int sph_step(sph_ctx *c, sph_state *state, long long n, float dt, float *dt_used)
{
    if (!c) return SPH_EINVAL;
    const bool graphable = c->use_graph && c->resident && c->have_derivs && !state && !(dt > 0.f) && c->d.n > 0;
    if (!graphable) return step_body(c, state, n, dt, dt_used);
    // a step with a full build (re-sort), one that reuses the lists, or a full one with a smoothing-length update
    const int kind = step_adapts_h(c) ? 2 : (step_is_full(c) ? 0 : 1);
    const int s = c->parity;
    if (c->gexec[kind][s] && (c->gkey_n[kind][s] != c->d.n || c->gkey_dtused[kind][s] != (const void *)dt_used)) {
        cudaGraphExecDestroy(c->gexec[kind][s]);
        c->gexec[kind][s] = nullptr;
    }
    if (!c->gexec[kind][s]) {
        // everything step_body changes on the host, in case the capture fails half way (no kernel has run then)
        const Resident r0 = c->d.r, alt0 = c->d.alt;
        const int parity0 = c->parity, since0 = c->steps_since_full;
        const long long count0 = c->step_count;
        const bool force0 = c->force_full, hd = c->have_density, hp = c->have_predict, hg = c->have_grad,
                   hf = c->have_force, hv = c->have_derivs;
        cudaGraph_t g = nullptr;
        const long long l0 = c->launches;
        SPH_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        c->capturing = true;
        const int rc = step_body(c, nullptr, 0, dt, dt_used);         // records; runs nothing
        c->capturing = false;
        cudaError_t e = cudaStreamEndCapture(c->stream, &g);
        if (!rc && e == cudaSuccess && g) {
            e = cudaGraphInstantiate(&c->gexec[kind][s], g, 0);
            if (e != cudaSuccess) c->gexec[kind][s] = nullptr;
        }
        if (g) cudaGraphDestroy(g);
        if (rc || e != cudaSuccess || !c->gexec[kind][s]) {
            c->d.r = r0; c->d.alt = alt0; c->parity = parity0; c->steps_since_full = since0; c->force_full = force0;
            c->step_count = count0;
            c->have_density = hd; c->have_predict = hp; c->have_grad = hg; c->have_force = hf; c->have_derivs = hv;
            c->launches = l0;
            (void)cudaGetLastError();
            if (rc) return rc;
            c->last_cuda = (int)e;
            c->use_graph = false;                                     // from now on kernel by kernel
            return step_body(c, state, n, dt, dt_used);
        }
        c->glaunches[kind][s] = c->launches - l0;
        c->gkey_n[kind][s] = c->d.n;
        c->gkey_dtused[kind][s] = (const void *)dt_used;
        SPH_CUDA(c, cudaGraphLaunch(c->gexec[kind][s], c->stream));   // the host effects were applied by step_body
        return SPH_OK;
    }
    SPH_CUDA(c, cudaGraphLaunch(c->gexec[kind][s], c->stream));
    {                                                                 // what step_body does on the host
        Dev &d = c->d;
        c->step_count++;
        if (kind != 1) {
            Resident t = d.r; d.r = d.alt; d.alt = t;
            c->parity ^= 1;
            c->steps_since_full = 0;
            c->force_full = false;
        } else {
            c->steps_since_full++;
        }
        c->launches += c->glaunches[kind][s];
        c->have_density = c->have_predict = c->have_force = c->have_derivs = true;
        c->have_grad = (c->p.flags & SPH_STRENGTH) != 0;
        for (int k = 0; k < SPH_T_COUNT; ++k) c->ev_used[k] = c->ev_used[k] || k != SPH_T_GRADIENT;
    }
    return SPH_OK;
}

// NEXT-4: one big step on power-of-two rungs (reading Q23; include/sph.h).  Kernel by kernel: every substep has its
// own arguments, and most of them touch a fraction of the tiles only.
extern "C" int sph_step_rungs(sph_ctx *c, float dT, int max_rung, const unsigned char *rungs)
{
    if (!c || !(dT > 0.f) || max_rung < 0 || max_rung > 16) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    int rc;
    PassTimer ts(c, SPH_T_STEP);
    if (!c->have_derivs) {          // a_0, du_0/dt, dS_0/dt and the limits from the current state
        rc = derivative_passes(c);
        if (rc) return rc;
        rc = do_close(c, SPH_DERIVATIVES, 0.f, false);
        if (rc) return rc;
    }
    Dev &d = c->d;
    // the lists of the big step: built here at the current positions, particle order kept throughout
    if (c->use_lists) {
        PassTimer t(c, SPH_T_BUILD);
        rc = sph_launch_tree(c);
        if (rc) return rc;
        rc = sph_launch_set_ref(c);
        if (rc) return rc;
        rc = sph_launch_cull(c, false);
        if (rc) return rc;
        c->steps_since_full = 0;
        c->force_full = false;
    }
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_RUNG_CLAMPED], 0, sizeof(unsigned long long), c->stream));
    rc = sph_launch_rung_assign(c, dT, max_rung, rungs);
    if (rc) return rc;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_ACTIVE_UPDATES], 0, 2 * sizeof(unsigned long long), c->stream));
    const bool strength = (c->p.flags & SPH_STRENGTH) != 0;
    for (int n = 0; n < (1 << max_rung); ++n) {
        {
            PassTimer t(c, SPH_T_KICKDRIFT);
            rc = sph_launch_kick_drift_rung(c, n, max_rung, dT);
            if (rc) return rc;
        }
        if (c->use_lists && d.skin > 0.f) {
            rc = reuse_neighbors(c);
        } else {
            PassTimer t(c, SPH_T_BUILD);
            rc = sph_launch_tree(c);
            if (!rc && c->use_lists) rc = sph_launch_cull(c, false);
            c->have_density = c->have_predict = c->have_grad = c->have_force = false;
        }
        if (rc) return rc;
        rc = sph_launch_mark_need(c);
        if (rc) return rc;
        c->rc.on = 1; c->rc.n1 = n + 1; c->rc.R = max_rung; c->rc.dT = dT; c->rc.fixed_rungs = rungs ? 1 : 0;
        c->rc.rung = d.rung; c->rc.tile_act = d.tile_act; c->rc.tile_need = d.tile_need;
        rc = derivative_passes(c);
        if (!rc) rc = do_close(c, SPH_CLOSE, 0.f, false);
        c->rc.on = 0;
        if (rc) return rc;
        (void)strength;
    }
    c->step_count++;
    c->force_full = true;            // a global step after this starts from a full build (re-sort)
    return SPH_OK;
}

// refresh the resident state from caller-order device arrays, keeping order and derivatives.  What the neighbour lists
// depend on -- x, y, z, h -- is compared with the resident values first: a caller that hands back the state it was
// given (the usual host-buffer loop) leaves them bit for bit, and the lists (with their skin and their validity
// check) stay in use; any difference sets the flag and the step starts from a full build.
// PARTS: 1 = x, y, z, m, h, v (and the test whether the caller moved anything), 2 = u, S, 4 = a_ext
template <int PARTS>
__global__ void __launch_bounds__(256) k_refresh(Dev d, sph_state st)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    unsigned o = ((const unsigned *)d.r.s[PP_ORIG])[i];
    if (PARTS & 1) {
        const float4 np = make_float4(st.x[o], st.y[o], st.z[o], st.m[o]), op = d.r.pm[i];
        const float nh = st.h[o];
        if (!(np.x == op.x && np.y == op.y && np.z == op.z && nh == d.r.vh[i].w)) *d.refresh_changed = 1;
        d.r.pm[i] = np;
        d.r.vh[i].w = nh;
        d.vfull[0][i] = st.vx[o]; d.vfull[1][i] = st.vy[o]; d.vfull[2][i] = st.vz[o];
    }
    if (PARTS & 2) {
        d.ufull[i] = st.u[o];
        d.Sfull[0][i] = st.Sxx[o]; d.Sfull[1][i] = st.Syy[o]; d.Sfull[2][i] = st.Sxy[o];
        d.Sfull[3][i] = st.Sxz[o]; d.Sfull[4][i] = st.Syz[o];
    }
    if (PARTS & 4) {
        d.r.s[PP_G + 0][i] = st.gx ? st.gx[o] : 0.f;
        d.r.s[PP_G + 1][i] = st.gy ? st.gy[o] : 0.f;
        d.r.s[PP_G + 2][i] = st.gz ? st.gz[o] : 0.f;
    }
}

// sph_step_host, a step that reuses the lists: the second group of host arrays (u, S) has been travelling on
// h2d_stream while the first half of the kick, the list check and the density pass ran; take it in and kick u and S.
// The third group (a_ext) is still on its way: the pair pass leaves it out and CLOSE adds it (take_third_group).
static int take_second_group(sph_ctx *c)
{
    sph_state *ds = c->host_in;
    c->host_in = nullptr;
    SPH_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_second, 0));
    k_refresh<2><<<sph_div_up(c->d.n, 256), 256, 0, c->stream>>>(c->d, *ds);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    c->host_in_g = ds;
    c->p.flags |= SPH_INT_DEFER_AEXT;
    return sph_launch_kick_drift(c, 0.f, 2);
}

static int take_third_group(sph_ctx *c)
{
    sph_state *ds = c->host_in_g;
    c->host_in_g = nullptr;
    SPH_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_third, 0));
    k_refresh<4><<<sph_div_up(c->d.n, 256), 256, 0, c->stream>>>(c->d, *ds);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

static int step_host_body(sph_ctx *c, sph_state *hs, long long n, float dt, float *dt_used)
{
    size_t N = (size_t)(c->d.n_max > 0 ? c->d.n_max : 1);
    float *base = c->stage;
    float *dev[17];
    for (int k = 0; k < 17; ++k) dev[k] = base + (size_t)k * N;
    int *dmat = (int *)(base + 17 * N);
    unsigned char *dfix = (unsigned char *)(base + 18 * N);
    const float *src[17] = {hs->x, hs->y, hs->z, hs->m, hs->h, hs->vx, hs->vy, hs->vz, hs->u,
                            hs->Sxx, hs->Syy, hs->Sxy, hs->Sxz, hs->Syz, hs->gx, hs->gy, hs->gz};
    sph_state ds;
    memset(&ds, 0, sizeof(ds));
    // first group: what the first half of the kick, the list check and the density pass need (x, y, z, m, h, v);
    // second group (u, S, a_ext) on its own stream behind it when the particles are resident already
    const bool split = c->resident && n > 0;
    for (int k = 0; k < 8; ++k)
        if (n > 0) SPH_CUDA(c, cudaMemcpyAsync(dev[k], src[k], (size_t)n * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    cudaStream_t s2 = c->stream;
    if (split) {
        SPH_CUDA(c, cudaEventRecord(c->ev_first, c->stream));
        SPH_CUDA(c, cudaStreamWaitEvent(c->h2d_stream, c->ev_first, 0));
        s2 = c->h2d_stream;
    }
    for (int k = 8; k < 14; ++k)
        if (n > 0 && src[k]) SPH_CUDA(c, cudaMemcpyAsync(dev[k], src[k], (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s2));
    if (split) SPH_CUDA(c, cudaEventRecord(c->ev_second, c->h2d_stream));
    for (int k = 14; k < 17; ++k)
        if (n > 0 && src[k]) SPH_CUDA(c, cudaMemcpyAsync(dev[k], src[k], (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s2));
    if (split) SPH_CUDA(c, cudaEventRecord(c->ev_third, c->h2d_stream));
    ds.x = dev[0]; ds.y = dev[1]; ds.z = dev[2]; ds.m = dev[3]; ds.h = dev[4];
    ds.vx = dev[5]; ds.vy = dev[6]; ds.vz = dev[7]; ds.u = dev[8];
    ds.Sxx = dev[9]; ds.Syy = dev[10]; ds.Sxy = dev[11]; ds.Sxz = dev[12]; ds.Syz = dev[13];
    ds.gx = hs->gx ? dev[14] : nullptr; ds.gy = hs->gy ? dev[15] : nullptr; ds.gz = hs->gz ? dev[16] : nullptr;
    // material and fixed flags are read at the first call only (they stay with the resident particles)
    if (n > 0 && hs->mat && !c->resident) {
        SPH_CUDA(c, cudaMemcpyAsync(dmat, hs->mat, (size_t)n * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        ds.mat = dmat;
    }
    if (n > 0 && hs->fixed && !c->resident) {
        SPH_CUDA(c, cudaMemcpyAsync(dfix, hs->fixed, (size_t)n, cudaMemcpyHostToDevice, c->stream));
        ds.fixed = dfix;
    }
    int rc;
    bool changed = false;
    if (split) {
        SPH_CUDA(c, cudaMemsetAsync(c->d.refresh_changed, 0, sizeof(int), c->stream));
        k_refresh<1><<<sph_div_up(n, 256), 256, 0, c->stream>>>(c->d, ds);
        c->launches++;
        SPH_CUDA(c, cudaGetLastError());
        int h_changed = 1;
        SPH_CUDA(c, cudaMemcpyAsync(&h_changed, c->d.refresh_changed, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        SPH_CUDA(c, cudaStreamSynchronize(c->stream));     // the step cannot start before these copies have landed anyway
        changed = h_changed != 0;
        if (changed) c->force_full = true;    // the caller moved particles: nothing the lists were built on holds
        // A step that reuses the lists keeps the particle order, so u and S can be taken in and kicked after the
        // density pass (take_second_group); a step with a re-sort permutes them, so it waits for them here.
        if (c->have_derivs && !step_is_full(c)) {
            c->host_in = &ds;
        } else {
            SPH_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_third, 0));
            k_refresh<6><<<sph_div_up(n, 256), 256, 0, c->stream>>>(c->d, ds);
            c->launches++;
            SPH_CUDA(c, cudaGetLastError());
        }
    }
    // a step on positions the caller changed builds lists that serve this step only: no skin, no ordering pass.
    // x, y, z go back on the second stream as soon as the drift is done (step_body)
    c->no_reuse_now = changed;
    const bool overlap = c->resident && n > 0;          // (the very first call ingests and bootstraps first)
    if (overlap) {
        c->host_out = &ds;
        c->host_dst[0] = hs->x; c->host_dst[1] = hs->y; c->host_dst[2] = hs->z;
    }
    rc = sph_step(c, &ds, n, dt, nullptr);
    c->host_out = nullptr;
    c->host_in = nullptr;
    c->host_in_g = nullptr;
    c->p.flags &= ~SPH_INT_DEFER_AEXT;
    c->no_reuse_now = false;
    if (changed) c->force_full = true;     // those lists have no skin: whatever step comes next must not reuse them
    if (rc) return rc;
    float *dst[14] = {hs->x, hs->y, hs->z, nullptr, nullptr, hs->vx, hs->vy, hs->vz, hs->u,
                      hs->Sxx, hs->Syy, hs->Sxy, hs->Sxz, hs->Syz};
    if (c->adapt_h_every > 0 && n > 0) {
        // the step may have updated the smoothing lengths: they go back with the rest of the state, so
        // that the caller's h stays the resident one (otherwise the next call would see "the caller changed h", put its
        // stale h back over the adapted one and start from a full build every time)
        rc = sph_launch_get_h(c, dev[4]);
        if (rc) return rc;
        dst[4] = hs->h;
    }
    for (int k = overlap ? 3 : 0; k < 14; ++k) {
        if (n > 0 && dst[k])
            SPH_CUDA(c, cudaMemcpyAsync(dst[k], dev[k], (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    }
    if (dt_used) SPH_CUDA(c, cudaMemcpyAsync(dt_used, c->d.dt_cur, sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    if (overlap) SPH_CUDA(c, cudaEventSynchronize(c->ev_copied));
    return SPH_OK;
}

extern "C" int sph_step_host(sph_ctx *c, sph_state *hs, long long n, float dt, float *dt_used)
{
    if (!c || n < 0 || (n > 0 && !state_ok(hs))) return SPH_EINVAL;
    if (n > c->d.n_max) return SPH_ECAPACITY;
    if (c->resident && n != c->d.n) return SPH_EINVAL;
    const int rc = step_host_body(c, hs, n, dt, dt_used);
    if (rc) {
        // an error part way: copies into the staging arrays or into the caller's host arrays may still be in flight on
        // the three streams.  The caller is free to reuse its buffers once this returns, so wait for all of them, and
        // leave nothing of this call's per-call state behind.
        cudaStreamSynchronize(c->stream);
        cudaStreamSynchronize(c->h2d_stream);
        cudaStreamSynchronize(c->copy_stream);
        (void)cudaGetLastError();
        c->host_out = nullptr; c->host_in = nullptr; c->host_in_g = nullptr;
        c->p.flags &= ~SPH_INT_DEFER_AEXT;
        c->no_reuse_now = false;
        c->force_full = true;
    }
    return rc;
}

extern "C" int sph_download_state(sph_ctx *c, sph_state *state)
{
    if (!c || !state_ok(state)) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    return sph_launch_download(c, state, 0);
}

// ------------------------------------------------------------------------------------------
// outputs
// ------------------------------------------------------------------------------------------
extern "C" int sph_get_field(sph_ctx *c, int id, float *dst)
{
    if (!c || !dst) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    Dev &d = c->d;
    const float *src = nullptr;
    int as_int = 0;
    switch (id) {
    case SPH_F_RHO: src = d.rho; break;
    case SPH_F_OMEGA: src = d.omega; break;
    case SPH_F_P: src = d.P; break;
    case SPH_F_CS: src = d.cs; break;
    case SPH_F_T: src = d.T; break;
    case SPH_F_GAMMA: src = d.Gamma; break;
    case SPH_F_Y: src = d.Y; break;
    case SPH_F_MUMAX: src = d.mumax; break;
    case SPH_F_DUDT: src = d.dudt; break;
    case SPH_F_DT: src = d.dti; break;
    case SPH_F_EACC: src = d.r.s[PP_EACC]; break;
    case SPH_F_EPS2: src = d.eps2; break;
    case SPH_F_U: src = d.ufull; break;
    case SPH_F_CFLAG: src = d.cflag; break;
    case SPH_F_NGATHER: src = (const float *)d.ngather; as_int = 1; break;
    case SPH_F_NSYMMETRIC: src = (const float *)d.nsym; as_int = 1; break;
    case SPH_F_H: return sph_launch_get_h(c, dst);
    case SPH_F_RUNG: src = (const float *)d.rung; as_int = 2; break;
    case SPH_F_TILE: return sph_launch_get_tile(c, dst);
    default: break;
    }
    if (!src) {
        if (id >= SPH_F_A && id < SPH_F_A + 3) src = d.a[id - SPH_F_A];
        else if (id >= SPH_F_V && id < SPH_F_V + 3) src = d.vfull[id - SPH_F_V];
        else if (id >= SPH_F_X && id < SPH_F_X + 3) return sph_launch_get_position(c, id - SPH_F_X, dst);
        else if (id >= SPH_F_SPRED && id < SPH_F_SPRED + 5) src = d.r.s[PP_SPRED + id - SPH_F_SPRED];
        else if (id >= SPH_F_S && id < SPH_F_S + 5) src = d.Sfull[id - SPH_F_S];
        else if (id >= SPH_F_DSDT && id < SPH_F_DSDT + 5) src = d.dS[id - SPH_F_DSDT];
        else if (id >= SPH_F_F && id < SPH_F_F + 9) src = d.F[id - SPH_F_F];
        else if (id >= SPH_F_CINV && id < SPH_F_CINV + 9) src = d.Cinv[id - SPH_F_CINV];
        else if (id >= SPH_F_G && id < SPH_F_G + 9) src = d.G[id - SPH_F_G];
    }
    if (!src) return SPH_EINVAL;
    return sph_launch_get_field(c, src, dst, as_int);
}

extern "C" int sph_get_neighbors(sph_ctx *c, int which, int *counts, const long long *offsets, int *list)
{
    if (!c || !counts || (which != SPH_GATHER && which != SPH_SYMMETRIC) || (list && !offsets)) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    return c->use_lists ? sph_launch_neighbors_l(c, which, counts, offsets, list)
                        : sph_launch_neighbors(c, which, counts, offsets, list, false);
}

extern "C" int sph_get_timings(sph_ctx *c, float *ms, int n)
{
    if (!c || !ms || n < 0) return SPH_EINVAL;
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < n && k < SPH_T_COUNT; ++k) {
        ms[k] = 0.f;
        if (c->ev_used[k]) cudaEventElapsedTime(&ms[k], c->ev[2 * k], c->ev[2 * k + 1]);
    }
    return SPH_OK;
}

extern "C" int sph_get_counters(sph_ctx *c, long long *out, int n)
{
    if (!c || !out || n < 0) return SPH_EINVAL;
    unsigned long long h[SPH_C_COUNT];
    SPH_CUDA(c, cudaMemcpyAsync(h, c->d.counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    h[SPH_C_STEPS_SINCE_FULL] = (unsigned long long)c->steps_since_full;       // host-side
    for (int k = 0; k < n && k < SPH_C_COUNT; ++k) out[k] = (long long)h[k];
    return SPH_OK;
}

extern "C" int sph_set_eos_table(sph_ctx *c, int material, const sph_eos_table *tab)
{
    if (!c || material < 0 || material >= c->p.n_materials) return SPH_EINVAL;
    DevTab &t = c->tabs.t[material];
    drop_graphs(c);
    if (!tab) {
        t = DevTab{};
        c->have_predict = c->have_grad = c->have_force = false;
        return SPH_OK;
    }
    if (tab->n_rho < 2 || tab->n_u < 2 || !tab->P || !tab->T || !tab->cs || !(tab->rho_max > tab->rho_min)
        || !(tab->u_max > tab->u_min) || (tab->Tmelt && tab->n_melt < 2))
        return SPH_EINVAL;
    t.n_rho = tab->n_rho; t.n_u = tab->n_u; t.n_melt = tab->Tmelt ? tab->n_melt : 0;
    t.rho_min = tab->rho_min; t.rho_max = tab->rho_max; t.u_min = tab->u_min; t.u_max = tab->u_max;
    t.P = tab->P; t.T = tab->T; t.cs = tab->cs; t.Tmelt = tab->Tmelt;
    c->have_predict = c->have_grad = c->have_force = false;
    return SPH_OK;
}

extern "C" int sph_get_diagnostics(sph_ctx *c, double *out)
{
    if (!c || !out) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    return sph_launch_diagnostics(c, out);
}

extern "C" int sph_get_tile_stats(sph_ctx *c, int *ncand, unsigned *cycles, unsigned char *flag, int capacity)
{
    if (!c || capacity < 0) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    const int ntile = sph_div_up(c->d.nchunk, SPH_TILE_CHUNKS);
    if (!c->use_lists || capacity < ntile) return ntile;
    if (ncand) SPH_CUDA(c, cudaMemcpyAsync(ncand, c->d.tile_ncand, sizeof(int) * ntile, cudaMemcpyDeviceToHost, c->stream));
    if (cycles) SPH_CUDA(c, cudaMemcpyAsync(cycles, c->d.tile_cycles, sizeof(unsigned) * ntile, cudaMemcpyDeviceToHost, c->stream));
    if (flag) SPH_CUDA(c, cudaMemcpyAsync(flag, c->d.tile_flag, ntile, cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    return ntile;
}

extern "C" int sph_get_tile_dirty(sph_ctx *c, unsigned char *dirty, int capacity)
{
    if (!c || capacity < 0) return SPH_EINVAL;
    if (!c->resident) return SPH_EORDER;
    const int ntile = sph_div_up(c->d.nchunk, SPH_TILE_CHUNKS);
    if (!c->use_lists || capacity < ntile || !dirty) return ntile;
    SPH_CUDA(c, cudaMemcpyAsync(dirty, c->d.tile_dirty, ntile, cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA(c, cudaStreamSynchronize(c->stream));
    return ntile;
}

extern "C" long long sph_launch_count(const sph_ctx *c) { return c ? c->launches : 0; }
extern "C" int sph_last_cuda_error(const sph_ctx *c) { return c ? c->last_cuda : 0; }

extern "C" const char *sph_strerror(int code)
{
    switch (code) {
    case SPH_OK: return "ok";
    case SPH_EINVAL: return "invalid argument";
    case SPH_ENOMEM: return "workspace too small";
    case SPH_ECUDA: return "CUDA error (see sph_last_cuda_error)";
    case SPH_EORDER: return "pass called before its prerequisite";
    case SPH_ECAPACITY: return "n exceeds n_max";
    default: return "unknown error";
    }
}
