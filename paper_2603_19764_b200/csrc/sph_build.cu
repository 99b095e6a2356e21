// sph_build.cu -- S1: Morton keys, radix sort, gather into the resident sorted arrays, chunk
// bounding boxes and the implicit 32-ary chunk tree (stands in for the paper's tree build and
// domain decomposition; BASELINE.json north_star "Morton-key sort and reorder").
#include <cub/device/device_radix_sort.cuh>

#include "sph_internal.cuh"

// ------------------------------------------------------------------------------------------
// bounding box of all particles (ordered-int atomics; 6 words: lo xyz, hi xyz)
// ------------------------------------------------------------------------------------------
__global__ void k_bbox_init(int *bbox)
{
    if (threadIdx.x < 3) bbox[threadIdx.x] = 0x7fffffff;          // +max ordered
    else if (threadIdx.x < 6) bbox[threadIdx.x] = (int)0x80000000; // -max ordered
}

template <bool FROM_STATE>
__global__ void __launch_bounds__(256) k_bbox(const float *__restrict__ x, const float *__restrict__ y,
                                              const float *__restrict__ z, const float4 *__restrict__ pm,
                                              long long n, int *bbox)
{
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        float p[3];
        if (FROM_STATE) { p[0] = x[i]; p[1] = y[i]; p[2] = z[i]; }
        else { float4 q = pm[i]; p[0] = q.x; p[1] = q.y; p[2] = q.z; }
#pragma unroll
        for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], p[a]); hi[a] = fmaxf(hi[a], p[a]); }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
    }
    // one atomic per component per CTA: six addresses shared by every warp serialise otherwise
    __shared__ float s_lo[3][8], s_hi[3][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) { s_lo[a][warp] = lo[a]; s_hi[a][warp] = hi[a]; }
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        const int a = threadIdx.x % 3;
        if (threadIdx.x < 3) {
            float v = s_lo[a][0];
#pragma unroll
            for (int w = 1; w < 8; ++w) v = fminf(v, s_lo[a][w]);
            atomicMin(&bbox[a], sph_f2ord(v));
        } else {
            float v = s_hi[a][0];
#pragma unroll
            for (int w = 1; w < 8; ++w) v = fmaxf(v, s_hi[a][w]);
            atomicMax(&bbox[3 + a], sph_f2ord(v));
        }
    }
}

// ------------------------------------------------------------------------------------------
// space-filling-curve key (3 x B bits, B <= 21, in the low 3B bits of a 64-bit word) on a cubic grid
// spanning the bounding box.  The key only fixes the ORDER of the particles (locality of chunks and
// tiles), never a result, so B is chosen from n (key_bits below) and the radix sort runs over 3B
// bits only: 5 digit passes instead of 8 at 10^6 particles.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long expand21(unsigned long long v)
{
    v &= 0x1fffffull;
    v = (v | v << 32) & 0x1f00000000ffffull;
    v = (v | v << 16) & 0x1f0000ff0000ffull;
    v = (v | v << 8) & 0x100f00f00f00f00full;
    v = (v | v << 4) & 0x10c30c30c30c30c3ull;
    v = (v | v << 2) & 0x1249249249249249ull;
    return v;
}

// Hilbert index of a 3 x 21-bit lattice point (Skilling's transpose algorithm, AIP Conf. Proc. 707,
// 2004): unlike the Morton curve it has no jumps, so ANY run of consecutive particles is a compact
// connected blob -- which is what bounds the chunk / tile boxes of the pair passes.
__device__ __forceinline__ unsigned long long hilbert63(unsigned X0, unsigned X1, unsigned X2, int bits)
{
    unsigned X[3] = {X0, X1, X2};
    const unsigned M = 1u << (bits - 1);
    for (unsigned Q = M; Q > 1; Q >>= 1) {
        unsigned P = Q - 1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (X[a] & Q) X[0] ^= P;
            else { unsigned t = (X[0] ^ X[a]) & P; X[0] ^= t; X[a] ^= t; }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    unsigned t = 0;
    for (unsigned Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    return (expand21(X[0]) << 2) | (expand21(X[1]) << 1) | expand21(X[2]);
}

template <bool FROM_STATE>
__global__ void __launch_bounds__(256) k_keys(const float *__restrict__ x, const float *__restrict__ y,
                                              const float *__restrict__ z, const float4 *__restrict__ pm,
                                              long long n, const int *__restrict__ bbox, int morton, int bits,
                                              unsigned long long *__restrict__ keys, unsigned *__restrict__ perm)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    float lo[3], ext = 0.f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = sph_ord2f(bbox[a]);
        ext = fmaxf(ext, sph_ord2f(bbox[3 + a]) - lo[a]);
    }
    const float cmax = (float)((1u << bits) - 1u);
    float scale = ext > 0.f ? cmax / ext : 0.f;
    float p[3];
    if (FROM_STATE) { p[0] = x[i]; p[1] = y[i]; p[2] = z[i]; }
    else { float4 q = pm[i]; p[0] = q.x; p[1] = q.y; p[2] = q.z; }
    unsigned c[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float f = (p[a] - lo[a]) * scale;
        c[a] = (unsigned)fminf(fmaxf(f, 0.f), cmax);
    }
    keys[i] = morton ? (expand21(c[0]) | (expand21(c[1]) << 1) | (expand21(c[2]) << 2)) : hilbert63(c[0], c[1], c[2], bits);
    perm[i] = (unsigned)i;
}

// ------------------------------------------------------------------------------------------
// ingest: caller arrays (caller order) -> resident sorted arrays
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_ingest(sph_state st, Dev d, const unsigned *__restrict__ perm, int n_materials)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    unsigned p = perm[i];
    float vx = st.vx[p], vy = st.vy[p], vz = st.vz[p], u = st.u[p];
    float S[5] = {st.Sxx[p], st.Syy[p], st.Sxy[p], st.Sxz[p], st.Syz[p]};
    d.r.pm[i] = make_float4(st.x[p], st.y[p], st.z[p], st.m[p]);
    d.r.vh[i] = make_float4(vx, vy, vz, st.h[p]);
    d.r.s[PP_UPRED][i] = u;
    d.r.s[PP_UHALF][i] = u;
    d.ufull[i] = u;
    d.r.s[PP_VHALF + 0][i] = vx; d.r.s[PP_VHALF + 1][i] = vy; d.r.s[PP_VHALF + 2][i] = vz;
    d.vfull[0][i] = vx; d.vfull[1][i] = vy; d.vfull[2][i] = vz;
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        d.r.s[PP_SPRED + c][i] = S[c];
        d.r.s[PP_SHALF + c][i] = S[c];
        d.Sfull[c][i] = S[c];
        d.dS[c][i] = 0.f;
    }
    d.r.s[PP_EACC][i] = 0.f;
    d.r.s[PP_G + 0][i] = st.gx ? st.gx[p] : 0.f;
    d.r.s[PP_G + 1][i] = st.gy ? st.gy[p] : 0.f;
    d.r.s[PP_G + 2][i] = st.gz ? st.gz[p] : 0.f;
    ((unsigned *)d.r.s[PP_ORIG])[i] = p;
    // a material index outside 0..n_materials-1 would index past the parameter tables in k_predict / k_close
    int mi = st.mat ? st.mat[p] : 0;
    if (mi < 0 || mi >= n_materials) {
        mi = n_materials - 1;
        atomicAdd(&d.counters[SPH_C_BAD_MATERIAL], 1ull);
    }
    unsigned mf = (unsigned)mi | (st.fixed ? ((unsigned)(st.fixed[p] != 0) << 8) : 0u);
    ((unsigned *)d.r.s[PP_MATFIX])[i] = mf;
    d.a[0][i] = 0.f; d.a[1][i] = 0.f; d.a[2][i] = 0.f;
    d.dudt[i] = 0.f;
}

// re-sort: alt[i] = cur[perm[i]] for every array that moves with the particle
__global__ void __launch_bounds__(256) k_permute(Dev d, const unsigned *__restrict__ perm)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    unsigned p = perm[i];
    d.alt.pm[i] = d.r.pm[p];
    d.alt.vh[i] = d.r.vh[p];
#pragma unroll
    for (int f = 0; f < SPH_NPP; ++f) d.alt.s[f][i] = d.r.s[f][p];
}

// ------------------------------------------------------------------------------------------
// chunk boxes (level 0) and inner levels of the implicit tree.  DISP (list reuse, Dev::skin > 0): also the
// box of the displacements x - xref since the last full list build and the smallest H of the node.
// ------------------------------------------------------------------------------------------
template <bool DISP>
__global__ void __launch_bounds__(256) k_chunk_boxes(Dev d, float kappa)
{
    int chunk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (chunk >= d.nchunk) return;
    int lane = threadIdx.x & 31;
    long long i = (long long)chunk * SPH_CHUNK + lane;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, H = 0.f;
    float dl[3] = {3.0e38f, 3.0e38f, 3.0e38f}, dh[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, Hmin = 3.0e38f;
    if (i < d.n) {
        float4 q = d.r.pm[i];
        lo[0] = hi[0] = q.x; lo[1] = hi[1] = q.y; lo[2] = hi[2] = q.z;
        H = sph_H(kappa, d.r.vh[i].w);
        if (DISP) {
            const float4 r = d.xref[i];
            dl[0] = dh[0] = q.x - r.x; dl[1] = dh[1] = q.y - r.y; dl[2] = dh[2] = q.z - r.z;
            Hmin = H;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
            if (DISP) {
                dl[a] = fminf(dl[a], __shfl_xor_sync(0xffffffffu, dl[a], o));
                dh[a] = fmaxf(dh[a], __shfl_xor_sync(0xffffffffu, dh[a], o));
            }
        }
        H = fmaxf(H, __shfl_xor_sync(0xffffffffu, H, o));
        if (DISP) Hmin = fminf(Hmin, __shfl_xor_sync(0xffffffffu, Hmin, o));
    }
    if (lane == 0) {
        d.tree.lo[0][chunk] = make_float4(lo[0], lo[1], lo[2], H);
        d.tree.hi[0][chunk] = make_float4(hi[0], hi[1], hi[2], 0.f);
        if (DISP) {
            d.tree.dlo[0][chunk] = make_float4(dl[0], dl[1], dl[2], Hmin);
            d.tree.dhi[0][chunk] = make_float4(dh[0], dh[1], dh[2], 0.f);
        }
    }
}

template <bool DISP>
__global__ void __launch_bounds__(256) k_tree_level(Tree t, int L)
{
    int node = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (node >= t.count[L]) return;
    int lane = threadIdx.x & 31;
    int child = node * SPH_ARITY + lane;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, H = 0.f;
    float dl[3] = {3.0e38f, 3.0e38f, 3.0e38f}, dh[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, Hmin = 3.0e38f;
    if (child < t.count[L - 1]) {
        float4 a = t.lo[L - 1][child], b = t.hi[L - 1][child];
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; H = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
        if (DISP) {
            a = t.dlo[L - 1][child]; b = t.dhi[L - 1][child];
            dl[0] = a.x; dl[1] = a.y; dl[2] = a.z; Hmin = a.w;
            dh[0] = b.x; dh[1] = b.y; dh[2] = b.z;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
            if (DISP) {
                dl[a] = fminf(dl[a], __shfl_xor_sync(0xffffffffu, dl[a], o));
                dh[a] = fmaxf(dh[a], __shfl_xor_sync(0xffffffffu, dh[a], o));
            }
        }
        H = fmaxf(H, __shfl_xor_sync(0xffffffffu, H, o));
        if (DISP) Hmin = fminf(Hmin, __shfl_xor_sync(0xffffffffu, Hmin, o));
    }
    if (lane == 0) {
        t.lo[L][node] = make_float4(lo[0], lo[1], lo[2], H);
        t.hi[L][node] = make_float4(hi[0], hi[1], hi[2], 0.f);
        if (DISP) {
            t.dlo[L][node] = make_float4(dl[0], dl[1], dl[2], Hmin);
            t.dhi[L][node] = make_float4(dh[0], dh[1], dh[2], 0.f);
        }
    }
}

// the reference positions of the list reuse: xref = x (at a full list build)
__global__ void __launch_bounds__(256) k_set_ref(Dev d)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < d.n) d.xref[i] = d.r.pm[i];
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
size_t sph_cub_temp_bytes(long long n_max)
{
    size_t bytes = 0;
    cudaError_t e = cub::DeviceRadixSort::SortPairs(nullptr, bytes, (const unsigned long long *)nullptr,
                                                    (unsigned long long *)nullptr, (const unsigned *)nullptr,
                                                    (unsigned *)nullptr, (int)(n_max > 0 ? n_max : 1), 0, 63);
    // no device to ask (sizing on a CPU-only box): a bound well above what onesweep needs
    size_t bound = (size_t)(n_max > 0 ? n_max : 1) * 16 + ((size_t)1 << 20);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return bound; }
    return bytes > bound ? bytes : bound;
}

// bits per axis of the curve key: 2^3 cells per mean particle spacing and axis, within [10, 21].  Where the
// particle spacing is below a cell (a linear density contrast above 8) the stable sort keeps ties in their
// previous order, which is the previous step's curve order: measured on configs[3-4] (contrast 4.6 / 10) the
// list build is as fast as with 2^6 cells, and the radix sort needs one pass less (30 key bits at 1e6).
static int key_bits(long long n)
{
    int b = 0;
    while (((long long)1 << (3 * b)) < n) ++b;      // ceil(log2(n) / 3)
    b += 3;
    return b < 10 ? 10 : (b > 21 ? 21 : b);
}

static int sort_keys(sph_ctx *c, int bits)
{
    Dev &d = c->d;
    size_t bytes = d.cub_tmp_bytes;
    SPH_CUDA(c, cub::DeviceRadixSort::SortPairs(d.cub_tmp, bytes, d.keys, d.keys_alt, d.perm, d.perm_alt,
                                                (int)d.n, 0, 3 * bits, c->stream));
    c->launches += 2 + (3 * bits + 7) / 8;   // onesweep: histogram + scan + one pass per 8-bit digit
    return SPH_OK;
}

int sph_launch_tree(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    const bool disp = d.skin > 0.f;
    if (disp) k_chunk_boxes<true><<<sph_div_up(d.nchunk, 8), 256, 0, c->stream>>>(d, c->p.kappa);
    else k_chunk_boxes<false><<<sph_div_up(d.nchunk, 8), 256, 0, c->stream>>>(d, c->p.kappa);
    c->launches++;
    for (int L = 1; L < d.tree.nlev; ++L) {
        if (disp) k_tree_level<true><<<sph_div_up(d.tree.count[L], 8), 256, 0, c->stream>>>(d.tree, L);
        else k_tree_level<false><<<sph_div_up(d.tree.count[L], 8), 256, 0, c->stream>>>(d.tree, L);
        c->launches++;
    }
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

int sph_launch_set_ref(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0 || !(d.skin > 0.f)) return SPH_OK;
    k_set_ref<<<sph_div_up(d.n, 256), 256, 0, c->stream>>>(d);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return SPH_OK;
}

static void set_counts(sph_ctx *c, long long n)
{
    Dev &d = c->d;
    d.n = n;
    d.nchunk = sph_div_up(n, SPH_CHUNK);
    int cnt = d.nchunk, L = 0;
    d.tree.count[0] = cnt;
    while (cnt > SPH_ARITY && L + 1 < SPH_MAX_LEVELS) {
        cnt = sph_div_up(cnt, SPH_ARITY);
        d.tree.count[++L] = cnt;
    }
    d.tree.nlev = L + 1;
}

int sph_launch_ingest(sph_ctx *c, const sph_state *st, long long n)
{
    set_counts(c, n);
    Dev &d = c->d;
    if (n == 0) return SPH_OK;
    int nb = sph_div_up(n, 256);
    k_bbox_init<<<1, 32, 0, c->stream>>>((int *)d.bbox);
    k_bbox<true><<<nb < 592 ? nb : 592, 256, 0, c->stream>>>(st->x, st->y, st->z, nullptr, n, (int *)d.bbox);
    k_keys<true><<<nb, 256, 0, c->stream>>>(st->x, st->y, st->z, nullptr, n, (const int *)d.bbox, (c->p.flags & SPH_MORTON_ORDER) ? 1 : 0, key_bits(n), d.keys, d.perm);
    c->launches += 3;
    int rc = sort_keys(c, key_bits(n));
    if (rc) return rc;
    SPH_CUDA(c, cudaMemsetAsync(&d.counters[SPH_C_BAD_MATERIAL], 0, sizeof(unsigned long long), c->stream));
    k_ingest<<<nb, 256, 0, c->stream>>>(*st, d, d.perm_alt, c->p.n_materials);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    return sph_launch_tree(c);
}

int sph_launch_resort(sph_ctx *c)
{
    Dev &d = c->d;
    if (d.n == 0) return SPH_OK;
    int nb = sph_div_up(d.n, 256);
    k_bbox_init<<<1, 32, 0, c->stream>>>((int *)d.bbox);
    k_bbox<false><<<nb < 592 ? nb : 592, 256, 0, c->stream>>>(nullptr, nullptr, nullptr, d.r.pm, d.n, (int *)d.bbox);
    k_keys<false><<<nb, 256, 0, c->stream>>>(nullptr, nullptr, nullptr, d.r.pm, d.n, (const int *)d.bbox, (c->p.flags & SPH_MORTON_ORDER) ? 1 : 0, key_bits(d.n), d.keys, d.perm);
    c->launches += 3;
    int rc = sort_keys(c, key_bits(d.n));
    if (rc) return rc;
    k_permute<<<nb, 256, 0, c->stream>>>(d, d.perm_alt);
    c->launches++;
    SPH_CUDA(c, cudaGetLastError());
    Resident t = d.r; d.r = d.alt; d.alt = t;
    c->parity ^= 1;
    return sph_launch_tree(c);
}
