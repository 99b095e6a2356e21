/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain fp64 CPU oracle for the neighbour (pair) passes of one SPH + shear-strength
 * step of arxiv/paper_2603_19764 (section 2).  It is written from the paper's
 * equations, loop by loop, with no blocking, fusion or reordering, so that it can be
 * checked against the paper by eye.  It shares no code with the CUDA path
 * (paper_2603_19764_b200/csrc) and neither imports the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.
 *
 * The per-particle steps (EOS, yield, stress rate, projection, kicks) are in
 * oracle/oracle.py (numpy fp64); this file holds what needs loops over pairs.
 *
 * Notation: x_ij = x_i - x_j, v_ij = v_i - v_j, H = kappa*h is the
 * support radius, grad_i W_ij(h) = dW/dr(r_ij,h) * x_ij / r_ij.
 *
 * Pins: tests/test_oracle_*.py (kernel normalisation by quadrature, continuum limits of
 * Eq. 16/17, linear-field exactness of Eq. 20-22, conservation identities, grid == brute).
 * Parity-unpinned choices (ours): kernel form Q3, AV constants Q6.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).
 * -ffp-contract=off matters: the neighbour predicate is DEFINED in fp32 with separately
 * rounded multiplies and adds (reading Q4).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

#define ORC_GATHER 0
#define ORC_SYMMETRIC 1

/* ------------------------------------------------------------------------- */
/* Smoothing kernel: Wendland C2 in 3-D (PAPER.md:256 names it; the functional */
/* form is the textbook one of Dehnen & Aly 2012, reading Q3):                 */
/*   W(r,h) = 21/(2 pi H^3) (1-q)^4 (1+4q),  q = r/H < 1,  H = kappa h        */
/* ------------------------------------------------------------------------- */
double orc_W(double r, double h, double kappa)
{
    double H = kappa * h, q = r / H;
    if (q >= 1.0) return 0.0;
    double t = 1.0 - q;
    return 21.0 / (2.0 * M_PI * H * H * H) * t * t * t * t * (1.0 + 4.0 * q);
}

/* dW/dr = 21/(2 pi H^4) * (-20 q) (1-q)^3 */
double orc_dWdr(double r, double h, double kappa)
{
    double H = kappa * h, q = r / H;
    if (q >= 1.0) return 0.0;
    double t = 1.0 - q;
    return 21.0 / (2.0 * M_PI * H * H * H * H) * (-20.0 * q) * t * t * t;
}

/* dW/dh at fixed r: W = H^-3 f(r/H)  =>  dW/dh = -(3 W + r dW/dr)/h  (Eq. 3) */
double orc_dWdh(double r, double h, double kappa)
{
    return -(3.0 * orc_W(r, h, kappa) + r * orc_dWdr(r, h, kappa)) / h;
}

/* ------------------------------------------------------------------------- */
/* Pass O1 -- neighbour sets (PAPER.md:57 gather set; 140, 150, 157 use both h) */
/* Membership is defined in fp32 (reading Q4): d = fl(x_i - x_j) per axis,       */
/* r2 = fl(fl(fl(dx dx) + fl(dy dy)) + fl(dz dz)), H = fl(kappa h),              */
/* gather: r2 < fl(H_i H_i) (contains i); symmetric: j != i, r2 < max(H_i^2,H_j^2) */
/* ------------------------------------------------------------------------- */
static inline float r2_f32(float xi, float yi, float zi, float xj, float yj, float zj)
{
    float dx = xi - xj, dy = yi - yj, dz = zi - zj;
    float a = dx * dx, b = dy * dy, c = dz * dz;
    float s = a + b;
    return s + c;
}

static inline int member(int which, long long i, long long j, float r2, float H2i, float H2j)
{
    if (which == ORC_GATHER) return r2 < H2i;
    if (i == j) return 0;
    return r2 < (H2i > H2j ? H2i : H2j);
}

/* Brute force O(n^2).  counts[i] = |set(i)|; if list != NULL, offsets[] (n+1, exclusive
 * prefix of counts, filled by the caller) says where i's ascending list goes. */
void orc_neighbors_brute(long long n, const double *x, const double *y, const double *z,
                         const double *h, double kappa, int which,
                         int *counts, const long long *offsets, int *list)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (long long i = 0; i < n; ++i) {
        float Hi = (float)kappa * (float)h[i];
        float H2i = Hi * Hi;
        int c = 0;
        for (long long j = 0; j < n; ++j) {
            float Hj = (float)kappa * (float)h[j];
            float H2j = Hj * Hj;
            float r2 = r2_f32((float)x[i], (float)y[i], (float)z[i], (float)x[j], (float)y[j], (float)z[j]);
            if (member(which, i, j, r2, H2i, H2j)) {
                if (list) list[offsets[i] + c] = (int)j;
                ++c;
            }
        }
        counts[i] = c;
    }
}

/* Cell-list variant for sizes where O(n^2) is too slow: uniform grid with cell edge
 * >= max_i H_i, 27-cell stencil, SAME fp32 predicate; validated to give identical sets
 * to orc_neighbors_brute (tests/test_oracle_neighbors.py).  Lists are sorted ascending. */
static int cmp_int(const void *a, const void *b)
{
    int ia = *(const int *)a, ib = *(const int *)b;
    return (ia > ib) - (ia < ib);
}

void orc_neighbors_grid(long long n, const double *x, const double *y, const double *z,
                        const double *h, double kappa, int which,
                        int *counts, const long long *offsets, int *list)
{
    if (n <= 0) return;
    double lo[3] = {x[0], y[0], z[0]}, hi[3] = {x[0], y[0], z[0]}, Hmax = 0.0;
    for (long long i = 0; i < n; ++i) {
        double p[3] = {x[i], y[i], z[i]};
        for (int a = 0; a < 3; ++a) { if (p[a] < lo[a]) lo[a] = p[a]; if (p[a] > hi[a]) hi[a] = p[a]; }
        double H = kappa * h[i];
        if (H > Hmax) Hmax = H;
    }
    double edge = Hmax * 1.001;              /* margin over fp32 rounding of the predicate */
    if (!(edge > 0.0)) edge = 1.0;
    long long nc[3];
    double ce[3];
    for (int a = 0; a < 3; ++a) {
        nc[a] = (long long)floor((hi[a] - lo[a]) / edge);   /* cells never finer than the reach */
        if (nc[a] < 1) nc[a] = 1;
        if (nc[a] > 1024) nc[a] = 1024;                      /* bound the table; coarser stays correct */
        ce[a] = (hi[a] - lo[a]) / (double)nc[a];
        if (!(ce[a] >= edge)) ce[a] = edge;
    }
    long long ncell = nc[0] * nc[1] * nc[2];
    long long *start = (long long *)calloc((size_t)ncell + 1, sizeof(long long));
    int *cell_of = (int *)malloc((size_t)n * sizeof(int));
    int *order = (int *)malloc((size_t)n * sizeof(int));
    for (long long i = 0; i < n; ++i) {
        long long c[3];
        double p[3] = {x[i], y[i], z[i]};
        for (int a = 0; a < 3; ++a) {
            c[a] = (long long)floor((p[a] - lo[a]) / ce[a]);
            if (c[a] < 0) c[a] = 0;
            if (c[a] >= nc[a]) c[a] = nc[a] - 1;
        }
        cell_of[i] = (int)((c[0] * nc[1] + c[1]) * nc[2] + c[2]);
        start[cell_of[i] + 1]++;
    }
    for (long long c = 0; c < ncell; ++c) start[c + 1] += start[c];
    long long *fill = (long long *)malloc((size_t)ncell * sizeof(long long));
    memcpy(fill, start, (size_t)ncell * sizeof(long long));
    for (long long i = 0; i < n; ++i) order[fill[cell_of[i]]++] = (int)i;
    free(fill);

#pragma omp parallel for schedule(dynamic, 256)
    for (long long i = 0; i < n; ++i) {
        float Hi = (float)kappa * (float)h[i];
        float H2i = Hi * Hi;
        long long ci = cell_of[i];
        long long c0 = ci / (nc[1] * nc[2]), c1 = (ci / nc[2]) % nc[1], c2 = ci % nc[2];
        int c = 0;
        for (long long a0 = c0 - 1; a0 <= c0 + 1; ++a0) {
            if (a0 < 0 || a0 >= nc[0]) continue;
            for (long long a1 = c1 - 1; a1 <= c1 + 1; ++a1) {
                if (a1 < 0 || a1 >= nc[1]) continue;
                for (long long a2 = c2 - 1; a2 <= c2 + 1; ++a2) {
                    if (a2 < 0 || a2 >= nc[2]) continue;
                    long long cj = (a0 * nc[1] + a1) * nc[2] + a2;
                    for (long long k = start[cj]; k < start[cj + 1]; ++k) {
                        long long j = order[k];
                        float Hj = (float)kappa * (float)h[j];
                        float H2j = Hj * Hj;
                        float r2 = r2_f32((float)x[i], (float)y[i], (float)z[i],
                                          (float)x[j], (float)y[j], (float)z[j]);
                        if (member(which, i, j, r2, H2i, H2j)) {
                            if (list) list[offsets[i] + c] = (int)j;
                            ++c;
                        }
                    }
                }
            }
        }
        counts[i] = c;
        if (list) qsort(list + offsets[i], (size_t)c, sizeof(int), cmp_int);
    }
    free(start); free(cell_of); free(order);
}

/* ------------------------------------------------------------------------- */
/* Pass O2 -- density and grad-h term over the gather set, self term included   */
/*   rho_i   = sum_j m_j W_ij(h_i)                          (Eq. 1) */
/*   Omega_i = 1 + h_i/(3 rho_i) sum_j m_j dW_ij(h_i)/dh_i  (Eq. 3) */
/* ------------------------------------------------------------------------- */
void orc_density(long long n, const double *x, const double *y, const double *z,
                 const double *m, const double *h, double kappa,
                 const long long *off, const int *list, double *rho, double *omega)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (long long i = 0; i < n; ++i) {
        double s = 0.0, sh = 0.0;
        for (long long k = off[i]; k < off[i + 1]; ++k) {
            long long j = list[k];
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
            double r = sqrt(dx * dx + dy * dy + dz * dz);
            s += m[j] * orc_W(r, h[i], kappa);
            sh += m[j] * orc_dWdh(r, h[i], kappa);
        }
        rho[i] = s;
        omega[i] = 1.0 + h[i] / (3.0 * s) * sh;
    }
}

/* ------------------------------------------------------------------------- */
/* Pass O4 -- raw velocity gradient and correction tensor over the symmetric set */
/*   F_i^{ab}      = -1/2 sum_j m_j v_ij^a ( w_i dW_ij(h_i)/dx_i^b + w_j dW_ij(h_j)/dx_i^b ) */
/*   (C_i^-1)^{ab} = -1/2 sum_j m_j x_ij^a (            same bracket                     )  */
/*   with w = 1/(Omega rho)                          (Eq. 20, 21)         */
/* F, Cinv are [9][n], component index 3*a + b.                                            */
/* ------------------------------------------------------------------------- */
void orc_gradients(long long n, const double *x, const double *y, const double *z,
                   const double *m, const double *h,
                   const double *vx, const double *vy, const double *vz,
                   const double *rho, const double *omega, double kappa,
                   const long long *off, const int *list, double *F, double *Cinv)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (long long i = 0; i < n; ++i) {
        double f[9] = {0}, ci[9] = {0};
        double wi = 1.0 / (omega[i] * rho[i]);
        for (long long k = off[i]; k < off[i + 1]; ++k) {
            long long j = list[k];
            double xij[3] = {x[i] - x[j], y[i] - y[j], z[i] - z[j]};
            double vij[3] = {vx[i] - vx[j], vy[i] - vy[j], vz[i] - vz[j]};
            double r = sqrt(xij[0] * xij[0] + xij[1] * xij[1] + xij[2] * xij[2]);
            if (!(r > 0.0)) continue;                 /* dW/dr(0) = 0: no contribution */
            double wj = 1.0 / (omega[j] * rho[j]);
            double dWi = orc_dWdr(r, h[i], kappa), dWj = orc_dWdr(r, h[j], kappa);
            for (int b = 0; b < 3; ++b) {
                double bracket = wi * dWi * xij[b] / r + wj * dWj * xij[b] / r;
                for (int a = 0; a < 3; ++a) {
                    f[3 * a + b] += -0.5 * m[j] * vij[a] * bracket;
                    ci[3 * a + b] += -0.5 * m[j] * xij[a] * bracket;
                }
            }
        }
        for (int c = 0; c < 9; ++c) { F[c * n + i] = f[c]; Cinv[c * n + i] = ci[c]; }
    }
}

/* ------------------------------------------------------------------------- */
/* Pass O5 -- accelerations, energy rate and max |mu_ij| over the symmetric set  */
/*   sigma = -P delta + S                                     (Eq. 9) */
/*   a_i^a  = sum_j m_j [ sigma_i^{ab}/(Om_i rho_i^2) dW_ij(h_i)/dx_i^b               */
/*                      + sigma_j^{ab}/(Om_j rho_j^2) dW_ij(h_j)/dx_i^b ]            */
/*            (Eq. 4 + the S sum of Eq. 18)                         */
/*          - sum_j m_j Pi_ij dWbar_ij/dx_i^a                 (Eq. 7)     */
/*          + a_ext,i  (the "G" term of Eq. 18 is an input array; BASELINE.json)     */
/*   du_i/dt = - sigma_i^{ab}/(Om_i rho_i^2) sum_j m_j v_ij^a dW_ij(h_i)/dx_i^b       */
/*             (Eq. 19 and its hydro analogue, reading Q7)              */
/*           + 1/2 sum_j m_j Pi_ij v_ij . dWbar_ij/dx_i        (Eq. 8)    */
/*   Pi_ij, mu_ij: Eq. 5-6 with arithmetic means of c, rho, h;       */
/*   Wbar = (W(h_i) + W(h_j))/2; mu_max,i = max_j |min(0, mu_ij)| (Eq.39) */
/* S is [5][n] in the order xx, yy, xy, xz, yz (zz = -xx - yy, Eq. 11); a is [3][n].    */
/* ------------------------------------------------------------------------- */
static void sigma_tilde(double P, const double *S, long long n, long long i,
                        double omega, double rho, int strength, double st[3][3])
{
    double sxx = 0, syy = 0, sxy = 0, sxz = 0, syz = 0;
    if (strength) { sxx = S[0 * n + i]; syy = S[1 * n + i]; sxy = S[2 * n + i]; sxz = S[3 * n + i]; syz = S[4 * n + i]; }
    double szz = -sxx - syy;
    double f = 1.0 / (omega * rho * rho);
    st[0][0] = (-P + sxx) * f; st[0][1] = sxy * f;        st[0][2] = sxz * f;
    st[1][0] = sxy * f;        st[1][1] = (-P + syy) * f; st[1][2] = syz * f;
    st[2][0] = sxz * f;        st[2][1] = syz * f;        st[2][2] = (-P + szz) * f;
}

void orc_forces(long long n, const double *x, const double *y, const double *z,
                const double *m, const double *h,
                const double *vx, const double *vy, const double *vz,
                const double *rho, const double *omega, const double *P, const double *cs,
                const double *S, int strength,
                const double *gx, const double *gy, const double *gz,
                double kappa, double alpha, double beta, double eps_av,
                const long long *off, const int *list,
                double *a, double *dudt, double *mumax)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (long long i = 0; i < n; ++i) {
        double sti[3][3];
        sigma_tilde(P[i], S, n, i, omega[i], rho[i], strength, sti);
        double acc[3] = {0, 0, 0}, du = 0.0, mmax = 0.0;
        for (long long k = off[i]; k < off[i + 1]; ++k) {
            long long j = list[k];
            double xij[3] = {x[i] - x[j], y[i] - y[j], z[i] - z[j]};
            double vij[3] = {vx[i] - vx[j], vy[i] - vy[j], vz[i] - vz[j]};
            double r2 = xij[0] * xij[0] + xij[1] * xij[1] + xij[2] * xij[2];
            double r = sqrt(r2);
            double gWi[3] = {0, 0, 0}, gWj[3] = {0, 0, 0};   /* grad_i W_ij(h_i), grad_i W_ij(h_j) */
            if (r > 0.0) {
                double dWi = orc_dWdr(r, h[i], kappa), dWj = orc_dWdr(r, h[j], kappa);
                for (int b = 0; b < 3; ++b) { gWi[b] = dWi * xij[b] / r; gWj[b] = dWj * xij[b] / r; }
            }
            double stj[3][3];
            sigma_tilde(P[j], S, n, j, omega[j], rho[j], strength, stj);
            /* stress terms: Eq. 4 + Eq. 18 */
            for (int al = 0; al < 3; ++al)
                for (int b = 0; b < 3; ++b)
                    acc[al] += m[j] * (sti[al][b] * gWi[b] + stj[al][b] * gWj[b]);
            /* energy: Eq. 19 (+ hydro analogue) */
            for (int al = 0; al < 3; ++al)
                for (int b = 0; b < 3; ++b)
                    du -= sti[al][b] * m[j] * vij[al] * gWi[b];
            /* artificial viscosity: Eq. 5-8 */
            double vr = vij[0] * xij[0] + vij[1] * xij[1] + vij[2] * xij[2];
            if (vr < 0.0) {
                double hb = 0.5 * (h[i] + h[j]);
                double cb = 0.5 * (cs[i] + cs[j]);
                double rb = 0.5 * (rho[i] + rho[j]);
                double mu = hb * vr / (r2 + eps_av * hb * hb);
                double Pi = (-alpha * cb * mu + beta * mu * mu) / rb;
                double gWb[3], vdotg = 0.0;
                for (int b = 0; b < 3; ++b) { gWb[b] = 0.5 * (gWi[b] + gWj[b]); vdotg += vij[b] * gWb[b]; }
                for (int b = 0; b < 3; ++b) acc[b] -= m[j] * Pi * gWb[b];
                du += 0.5 * m[j] * Pi * vdotg;
                if (fabs(mu) > mmax) mmax = fabs(mu);
            }
        }
        a[0 * n + i] = acc[0] + (gx ? gx[i] : 0.0);
        a[1 * n + i] = acc[1] + (gy ? gy[i] : 0.0);
        a[2 * n + i] = acc[2] + (gz ? gz[i] : 0.0);
        dudt[i] = du;
        mumax[i] = mmax;
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
