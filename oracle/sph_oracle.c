/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the delta-SPH hot path computes, written from
 * /root/reference/PAPER.md (diffSPH, arXiv 2507.21684) and the readings listed in DESIGN.md
 * (taken from SURVEY.md section 8(c)).  It shares no code, header, table or helper with the CUDA
 * path under paper_2507_21684_b200/csrc/ and neither side includes or imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.
 *
 * Every function cites the passage it follows.  Nothing is blocked, fused or reordered
 * beyond what the formula says; OpenMP only distributes independent rows.
 *
 * Pins (tests/test_oracle_pins.py, all "-m not gpu"):
 *   orc_w / orc_gfac / orc_kfac : quadrature int W = 1, finite differences, values at q=0
 *   orc_wrap32                  : hand cases incl. negative / far out-of-box positions
 *   orc_neighbors               : lattice counts 45 (2D,H=4dx) / 93 (3D,H=3dx), symmetry, brute vs grid,
 *                                 pure-Python brute force on tiny inputs
 *   orc_density                 : interior lattice 1.000415750 / 1.002898240, Riemann-sum argument
 *   orc_max_displacement        : hand cases (known shift, shift by the box length, crossing a periodic face)
 *   orc_grad_sum(_vjp)          : two-particle closed form, zero on a periodic lattice with uniform weights, equals the
 *                                 own-position derivative of orc_density for a = m; central finite differences (x, a),
 *                                 sum x_bar = 0
 *   orc_density_vjp             : central finite differences of orc_density (x and m), sum x_bar = 0, two-particle
 *                                 closed form, zero on a lattice with uniform rho_bar
 *   orc_renorm_moments (+ numpy pinv in renorm_gradient): linear fields reproduced exactly on disordered / free-surface /
 *                                 varying-h particles, L M = I, M rebuilt from central differences of orc_w, M ~ I on a
 *                                 full lattice, x^2 exact on symmetric neighbourhoods, rank-1 line and isolated particle
 *   orc_renorm_moments_vjp (+ the pseudo-inverse adjoint in renorm_gradient_vjp): central differences of renorm_gradient
 *                                 w.r.t. x (random direction, single components), vol and A on 2D/3D/varying-h/wall cases and
 *                                 on a rank-1 line (constant-rank term), sum x_bar = 0, sum A_bar = 0
 *   orc_rhs                     : momentum conservation, Galilean / rigid rotation invariance, uniform
 *                                 compression, Brookshaw Laplacian of |x|^2, hydrostatic column, viscous symbol
 *   orc_rhs_vjp                 : central finite differences of orc_rhs (x, v, rho, all 10 scalars),
 *                                 sum x_bar = sum v_bar = 0, viscous self-adjointness
 *   orc_rk4_step(_vjp)          : 4th-order convergence, Taylor-Green decay, finite differences of KE
 * No function is "parity unpinned"; three READINGS (delta-term form and length scale, viscosity
 * coefficient / eps, boundary-kind rule) are pinned by internal consistency only.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC  (see oracle/build.py).
 * -ffp-contract=off matters: the neighbour predicate is defined as a fixed sequence of IEEE ops.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* kernel scales H/h of the Wendland C4 kernel */
static const double KAPPA2 = 2.171239;
static const double KAPPA3 = 2.207940;

/* ------------------------------------------------------------------------------------------
 * c-1  Wendland C4 kernel.  PAPER.md:421 Eq.25  W = C_d/H^d w(r/H);  PAPER.md:434 Eq.27
 *      w(q) = (1-q)_+^6 (1 + 6q + 35/3 q^2)   [Eq.27 prints "r" inside the polynomial: garble, q is meant]
 *      C_2 = 9/pi, C_3 = 495/(32 pi).   "h" in the paper == support radius H.
 * ------------------------------------------------------------------------------------------ */
static double Cd(int dim) { return dim == 2 ? 9.0 / M_PI : 495.0 / (32.0 * M_PI); }
static double kappa(int dim) { return dim == 2 ? KAPPA2 : KAPPA3; }

double orc_w(double r, double H, int dim)
{
    double q = r / H;
    if (q >= 1.0) return 0.0;
    double t = 1.0 - q;
    double t6 = t * t * t * t * t * t;
    return Cd(dim) / pow(H, dim) * t6 * (1.0 + 6.0 * q + 35.0 / 3.0 * q * q);
}

/* grad_i W_ij = G * d, d = x_i - x_j.  PAPER.md:444 Eq.29: grad W = rhat C_d/H^(d+1) w'(q).
 * w'(q) = -6(1-q)^5 (1+6q+35/3 q^2) + (1-q)^6 (6 + 70/3 q) = -(56/3) q (1+5q) (1-q)^5,
 * so rhat w'(q) / H = d * [w'(q)/q] / H^2 with F(q) := w'(q)/q = -(56/3)(1+5q)(1-q)^5, regular at q=0:
 *      G = C_d H^-(d+2) F(q).                                                                 */
double orc_gfac(double r, double H, int dim)
{
    double q = r / H;
    if (q >= 1.0) return 0.0;
    double t = 1.0 - q;
    double F = -(56.0 / 3.0) * (1.0 + 5.0 * q) * t * t * t * t * t;
    return Cd(dim) / pow(H, dim + 2) * F;
}

/* dG = K (d . delta d):  K = (1/r) dG/dr = C_d H^-(d+4) F'(q)/q,  F'(q) = 560 q (1-q)^4.
 * Hessian of W = G Id + K d (x) d; at r=0 it equals -(56/3) C_d H^-(d+2) Id, the q<eps branch of
 * PAPER.md:189 Eq.16 (A = Id, w''(0) = -56/3), so no epsilon is needed for Wendland C4.        */
double orc_kfac(double r, double H, int dim)
{
    double q = r / H;
    if (q >= 1.0) return 0.0;
    double t = 1.0 - q;
    return Cd(dim) / pow(H, dim + 4) * 560.0 * t * t * t * t;
}

/* ------------------------------------------------------------------------------------------
 * c-4  Wrapping ("mapped into the primary simulation domain using modulo arithmetic").
 * Reading: binary32, each operation rounded separately, in this order
 *      L = hi - lo;  xw = x - L*floor((x-lo)/L);  if (xw >= hi) xw -= L;  if (xw < lo) xw += L.
 * Bounded axes: unchanged; a position outside [lo,hi) (or non-finite) is counted in *n_oob.
 * x / xw are doubles HOLDING binary32 values (what the C ABI receives).
 * ------------------------------------------------------------------------------------------ */
void orc_wrap32(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                const double *x, double *xw, int64_t *n_oob)
{
    int64_t bad = 0;
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < dim; ++k) {
            volatile float xf = (float)x[i * dim + k], lof = (float)lo[k], hif = (float)hi[k];
            if (!isfinite(xf)) { bad++; xw[i * dim + k] = (double)xf; continue; }
            if (periodic[k]) {
                volatile float L = hif - lof;
                volatile float a = xf - lof;
                volatile float t = a / L;
                volatile float f = floorf(t);
                volatile float p = L * f;
                volatile float w = xf - p;
                if (w >= hif) w = w - L;
                if (w < lof) w = w + L;
                xw[i * dim + k] = (double)w;
            } else {
                if (xf < lof || xf >= hif) bad++;
                xw[i * dim + k] = (double)xf;
            }
        }
    if (n_oob) *n_oob = bad;
}

/* The same map in binary64, for the physics path (smooth in x, so finite differences work). */
static void wrap64(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                   const double *x, double *xw)
{
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < dim; ++k) {
            double xv = x[i * dim + k];
            if (periodic[k]) {
                volatile float l32 = (float)hi[k] - (float)lo[k];   /* same L as orc_wrap32 / box_len */
                double L = (double)l32;
                double w = xv - L * floor((xv - lo[k]) / L);
                if (w >= hi[k]) w -= L;
                if (w < lo[k]) w += L;
                xw[i * dim + k] = w;
            } else
                xw[i * dim + k] = xv;
        }
}

/* minimum image, SURVEY 8c-3 order: if d > L/2: d -= L; else if d < -L/2: d += L */
static inline void min_image(double *d, int dim, const int *periodic, const double *L)
{
    for (int k = 0; k < dim; ++k)
        if (periodic[k]) {
            if (d[k] > 0.5 * L[k]) d[k] -= L[k];
            else if (d[k] < -0.5 * L[k]) d[k] += L[k];
        }
}

static void box_len(int dim, const double *lo, const double *hi, double *L)
{
    /* L is the binary32 difference hi - lo (same L as orc_wrap32) */
    for (int k = 0; k < 3; ++k) L[k] = 0.0;
    for (int k = 0; k < dim; ++k) { volatile float l = (float)hi[k] - (float)lo[k]; L[k] = (double)l; }
}

/* ------------------------------------------------------------------------------------------
 * c-3  Neighbour set  N(i) = { j : r_ij^2 < Hs_ij^2 },  self included, strict "<".
 * Predicate evaluated in binary64 on WRAPPED binary32 positions, in this order:
 *   d_k = xw_i,k - xw_j,k ; minimum image ; r2 = fma(dz,dz, fma(dy,dy, dx*dx)) ;
 *   Hs = (float)(search_scale * max(h_i,h_j))  [one binary32 product] ;  r2 < (double)Hs*(double)Hs.
 * the search radius of a pair is max{h_i,h_j}.
 * ------------------------------------------------------------------------------------------ */
static inline int nb_pred(const double *xi, const double *xj, float hi_, float hj_, float scale,
                          int dim, const int *periodic, const double *L)
{
    double d[3] = {0, 0, 0};
    for (int k = 0; k < dim; ++k) d[k] = xi[k] - xj[k];
    min_image(d, dim, periodic, L);
    double r2 = d[0] * d[0];
    r2 = fma(d[1], d[1], r2);
    if (dim == 3) r2 = fma(d[2], d[2], r2);
    volatile float hm = hi_ > hj_ ? hi_ : hj_;
    volatile float Hs = scale * hm;
    double Hs2 = (double)Hs * (double)Hs;
    return r2 < Hs2;
}

static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* method 0: brute force O(n^2) (the definition).  method 1: the oracle's own uniform grid
 * (PAPER.md:556-558 steps 1-3: cells, map, adjacent-cell query), validated against method 0 in tests.
 * xw: wrapped positions (doubles).  h: support radii.  Two-call use: col_idx == NULL -> only row_ptr.
 * Rows are ascending in j.  Returns nnz, or -1 on allocation failure.                          */
int64_t orc_neighbors(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                      const double *xw, const double *h, double search_scale, int method,
                      int64_t *row_ptr, int32_t *col_idx)
{
    double L[3];
    box_len(dim, lo, hi, L);
    float scale = (float)search_scale;
    int64_t *cnt = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
    if (!cnt) return -1;

    if (method == 0) {
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t i = 0; i < n; ++i) {
            int64_t c = 0;
            int64_t base = col_idx ? row_ptr[i] : 0;
            for (int64_t j = 0; j < n; ++j)
                if (nb_pred(xw + i * dim, xw + j * dim, (float)h[i], (float)h[j], scale, dim, periodic, L)) {
                    if (col_idx) col_idx[base + c] = (int32_t)j;
                    c++;
                }
            cnt[i] = c;
        }
    } else {
        /* uniform grid, edge >= 1.001 * max search radius so that +-1 cell is a strict superset */
        double hmax = 0.0;
        for (int64_t i = 0; i < n; ++i) if (h[i] > hmax) hmax = h[i];
        double R = 1.001 * (double)scale * hmax;
        int nc[3] = {1, 1, 1};
        double edge[3] = {1, 1, 1}, ext[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) {
            ext[k] = periodic[k] ? L[k] : (hi[k] - lo[k]);
            int c = (int)floor(ext[k] / R);
            if (c < 1) c = 1;
            if (c > 2048) c = 2048;
            if (periodic[k] && c < 3) c = 1;
            nc[k] = c;
            edge[k] = ext[k] / c;
        }
        int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
        int64_t *cstart = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
        int32_t *order = (int32_t *)malloc((size_t)n * sizeof(int32_t));
        int32_t *cell_of = (int32_t *)malloc((size_t)n * 3 * sizeof(int32_t));
        if (!cstart || !order || !cell_of) { free(cnt); free(cstart); free(order); free(cell_of); return -1; }
        for (int64_t i = 0; i < n; ++i) {
            int64_t lin = 0, mul = 1;
            for (int k = 0; k < 3; ++k) {
                int c = 0;
                if (k < dim) {
                    c = (int)floor((xw[i * dim + k] - lo[k]) / edge[k]);
                    if (c < 0) c = 0;
                    if (c >= nc[k]) c = nc[k] - 1;
                }
                cell_of[i * 3 + k] = c;
                lin += mul * c;
                mul *= nc[k];
            }
            cstart[lin + 1]++;
        }
        for (int64_t c = 0; c < ncell; ++c) cstart[c + 1] += cstart[c];
        int64_t *fillp = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
        memcpy(fillp, cstart, (size_t)ncell * sizeof(int64_t));
        for (int64_t i = 0; i < n; ++i) {
            int64_t lin = cell_of[i * 3] + (int64_t)nc[0] * (cell_of[i * 3 + 1] + (int64_t)nc[1] * cell_of[i * 3 + 2]);
            order[fillp[lin]++] = (int32_t)i;
        }
        free(fillp);
#pragma omp parallel for schedule(dynamic, 256)
        for (int64_t i = 0; i < n; ++i) {
            int64_t c = 0;
            int64_t base = col_idx ? row_ptr[i] : 0;
            int o[3][3], no[3];
            for (int k = 0; k < 3; ++k) {
                no[k] = 0;
                int ci = cell_of[i * 3 + k];
                if (nc[k] == 1) { o[k][no[k]++] = 0; continue; }
                for (int s = -1; s <= 1; ++s) {
                    int cc = ci + s;
                    if (k < dim && periodic[k]) cc = (cc + nc[k]) % nc[k];
                    else if (cc < 0 || cc >= nc[k]) continue;
                    o[k][no[k]++] = cc;
                }
            }
            for (int a = 0; a < no[2]; ++a)
                for (int b = 0; b < no[1]; ++b)
                    for (int e = 0; e < no[0]; ++e) {
                        int64_t lin = o[0][e] + (int64_t)nc[0] * (o[1][b] + (int64_t)nc[1] * o[2][a]);
                        for (int64_t p = cstart[lin]; p < cstart[lin + 1]; ++p) {
                            int64_t j = order[p];
                            if (nb_pred(xw + i * dim, xw + j * dim, (float)h[i], (float)h[j], scale, dim, periodic, L)) {
                                if (col_idx) col_idx[base + c] = (int32_t)j;
                                c++;
                            }
                        }
                    }
            if (col_idx) qsort(col_idx + base, (size_t)c, sizeof(int32_t), cmp_i32);
            cnt[i] = c;
        }
        free(cstart); free(order); free(cell_of);
    }
    int64_t nnz = 0;
    if (!col_idx) {
        row_ptr[0] = 0;
        for (int64_t i = 0; i < n; ++i) { nnz += cnt[i]; row_ptr[i + 1] = nnz; }
    } else
        nnz = row_ptr[n];
    free(cnt);
    return nnz;
}

/* ------------------------------------------------------------------------------------------
 * NEXT-3a  Verlet-list validity: "the neighbor list needs to be updated if any particle
 *      moves more than half of the skin-width, where it is important to compute this update with respect to the
 *      positions used during the original neighborhood query".  Returns D = max_i |x_i - xb_i| with the minimum image
 *      on periodic axes ("tracking of total particle motion is significantly simplified for periodic BCs when using
 *      the minimum image convention").  The decision itself, 2 D <= skin width, is one comparison made by the caller.
 * ------------------------------------------------------------------------------------------ */
double orc_max_displacement(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                            const double *x, const double *x_build)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    double *bw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    wrap64(n, dim, periodic, lo, hi, x_build, bw);
    double D = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double d[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - bw[i * dim + k];
        min_image(d, dim, periodic, L);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (r > D) D = r;
    }
    free(xw);
    free(bw);
    return D;
}

/* ------------------------------------------------------------------------------------------
 * c-5  Summation density  rho_i = sum_{j in N(i)} m_j W(r_ij, H_ij)   PAPER.md:91 Eq.8, 476 Eq.35
 *      H_ij = max(h_i,h_j)  (BASELINE.json config 4)
 * ------------------------------------------------------------------------------------------ */
void orc_density(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                 const double *x, const double *h, const double *m,
                 const int64_t *row_ptr, const int32_t *col_idx, double *rho_out)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) {
        double acc = 0.0;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            acc += m[j] * orc_w(r, H, dim);
        }
        rho_out[i] = acc;
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-1  Adjoint of the summation density: the paper's own backward benchmark differentiates the
 *      summation density w.r.t. the particle positions, and the density-matching loss of PAPER.md:353
 *      Eq.21 needs the same product.  Given rho_bar_i = dL/d rho_i, reverse mode of the loop of orc_density, term
 *      by term, adjacency fixed, h not differentiated:
 *          rho_i = sum_j m_j W(|x_i - x_j|, H_ij)
 *          d rho_i = sum_j [ W_ij dm_j + m_j G_ij d_ij . (dx_i - dx_j) ],   grad_i W_ij = G_ij d_ij  (Eq.29)
 *      =>  x_bar_i += rho_bar_i m_j G_ij d_ij,   x_bar_j -= rho_bar_i m_j G_ij d_ij,   m_bar_j += rho_bar_i W_ij.
 *      Plain scatter, sequential (no threads): this is test infrastructure, obviously correct beats fast.
 * ------------------------------------------------------------------------------------------ */
void orc_density_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                     const double *x, const double *h, const double *m,
                     const int64_t *row_ptr, const int32_t *col_idx, const double *rho_bar,
                     double *x_bar, double *m_bar)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    for (int64_t i = 0; i < n * dim; ++i) x_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) m_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            double G = orc_gfac(r, H, dim);
            m_bar[j] += rho_bar[i] * orc_w(r, H, dim);
            for (int k = 0; k < dim; ++k) {
                double c = rho_bar[i] * m[j] * G * d[k];
                x_bar[i * dim + k] += c;
                x_bar[j * dim + k] -= c;
            }
        }
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-1, second half: the gradient term of the particle-shifting loss, Eq.24,
 *      [ sum_j m_j/rho_j grad_i W_ij ]^2.  The operator is the SPH gradient of the constant field with weights a_j
 *      (a_j = m_j/rho_j in Eq.24):
 *          g_i = sum_{j in N(i)} a_j grad_i W_ij = sum_j a_j G_ij d_ij,      d_ij = x_i - x_j   (Eq.29)
 *      and its reverse mode, term by term, adjacency fixed, with the exact Hessian of the kernel
 *      d(G d) = G dd + K (d . dd) d   (Eq.16):
 *          a_bar_j += g_bar_i . (G d),   D = a_j (G g_bar_i + K (d . g_bar_i) d),   x_bar_i += D,   x_bar_j -= D.
 * ------------------------------------------------------------------------------------------ */
void orc_grad_sum(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                  const double *x, const double *h, const double *a,
                  const int64_t *row_ptr, const int32_t *col_idx, double *g_out)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    for (int64_t i = 0; i < n; ++i) {
        double acc[3] = {0, 0, 0};
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            double G = orc_gfac(r, H, dim);
            for (int k = 0; k < dim; ++k) acc[k] += a[j] * G * d[k];
        }
        for (int k = 0; k < dim; ++k) g_out[i * dim + k] = acc[k];
    }
    free(xw);
}

void orc_grad_sum_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                      const double *x, const double *h, const double *a,
                      const int64_t *row_ptr, const int32_t *col_idx, const double *g_bar,
                      double *x_bar, double *a_bar)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    for (int64_t i = 0; i < n * dim; ++i) x_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) a_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            double G = orc_gfac(r, H, dim), K = orc_kfac(r, H, dim);
            double dg = 0.0;
            for (int k = 0; k < dim; ++k) dg += d[k] * g_bar[i * dim + k];
            a_bar[j] += G * dg;
            for (int k = 0; k < dim; ++k) {
                double D = a[j] * (G * g_bar[i * dim + k] + K * dg * d[k]);
                x_bar[i * dim + k] += D;
                x_bar[j * dim + k] -= D;
            }
        }
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-2, first part: kernel renormalisation, Eq.44, Eq.45.  With V_j = m_j/rho_j
 * passed in as `vol`, and grad_i W_ij = G_ij d_ij, d_ij = x_i - x_j (Eq.29):
 *      M_i = sum_j V_j (x_j - x_i) (x) grad_i W_ij          the matrix Eq.45 inverts,   L_i = M_i^+
 *      b_i = sum_j V_j (A_j - A_i) grad_i W_ij               so that Eq.44 reads  <grad A>_i = L_i b_i
 * This routine only accumulates the two sums (M row-major d x d, b); the pseudo-inverse of Eq.45 ("commonly performed
 * as a pseudo-inverse") is numpy.linalg.pinv in oracle/__init__.py renorm_gradient().
 * ------------------------------------------------------------------------------------------ */
void orc_renorm_moments(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                        const double *x, const double *h, const double *vol, const double *A,
                        const int64_t *row_ptr, const int32_t *col_idx, double *M_out, double *b_out)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    for (int64_t i = 0; i < n; ++i) {
        double M[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, b[3] = {0, 0, 0};
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            double G = orc_gfac(r, H, dim);
            for (int k = 0; k < dim; ++k) {
                double gw = G * d[k];                                   /* component k of grad_i W_ij */
                for (int l = 0; l < dim; ++l) M[l][k] += vol[j] * (-d[l]) * gw;   /* (x_j - x_i)_l (grad W)_k */
                b[k] += vol[j] * (A[j] - A[i]) * gw;
            }
        }
        for (int l = 0; l < dim; ++l)
            for (int k = 0; k < dim; ++k) M_out[(i * dim + l) * dim + k] = M[l][k];
        for (int k = 0; k < dim; ++k) b_out[i * dim + k] = b[k];
    }
    free(xw);
}

/* Reverse mode of orc_renorm_moments, term by term with the adjacency held fixed ("fully supports
 * backpropagation through this operation as well").  Given the cotangents Mbar_i (d x d, row-major, of
 * M_i) and bbar_i (of b_i), and with  d(G d) = G dd + K (d . dd) d  (Eq.16), every ordered pair
 * (i <- j) of the list contributes, with d = x_i - x_j, dA = A_j - A_i, a = d^T Mbar_i d, be = bbar_i . d:
 *      M_i term  -V_j G d d^T :   vol_bar_j += -G a ;   F += -V_j [ K a d + G (Mbar_i + Mbar_i^T) d ]
 *      b_i term   V_j dA G d  :   vol_bar_j += dA G be ; A_bar_j += V_j G be ; A_bar_i -= V_j G be ;
 *                                 F += V_j dA [ K be d + G bbar_i ]
 *      x_bar_i += F ,  x_bar_j -= F .
 * The adjoint of the pseudo-inverse itself is taken in oracle/__init__.py renorm_gradient_vjp(). */
void orc_renorm_moments_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                            const double *x, const double *h, const double *vol, const double *A,
                            const int64_t *row_ptr, const int32_t *col_idx, const double *Mbar, const double *bbar,
                            double *x_bar, double *vol_bar, double *A_bar)
{
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    for (int64_t i = 0; i < n * dim; ++i) x_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) vol_bar[i] = A_bar[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        const double *Mb = Mbar + i * dim * dim, *bb = bbar + i * dim;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            double G = orc_gfac(r, H, dim), K = orc_kfac(r, H, dim);
            double dA = A[j] - A[i];
            double a = 0.0, be = 0.0, Nd[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) {
                be += bb[k] * d[k];
                for (int l = 0; l < dim; ++l) {
                    a += d[k] * Mb[k * dim + l] * d[l];
                    Nd[k] += (Mb[k * dim + l] + Mb[l * dim + k]) * d[l];
                }
            }
            vol_bar[j] += -G * a + dA * G * be;
            A_bar[j] += vol[j] * G * be;
            A_bar[i] -= vol[j] * G * be;
            for (int k = 0; k < dim; ++k) {
                double F = -vol[j] * (K * a * d[k] + G * Nd[k]) + vol[j] * dA * (K * be * d[k] + G * bb[k]);
                x_bar[i * dim + k] += F;
                x_bar[j * dim + k] -= F;
            }
        }
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * c-2 / c-6  Right-hand side.  Parameters par[11] = {c0, rho0, gamma, delta, alpha, nu, eps, gx, gy, gz, form}
 *
 * Tait EOS  p = rho0 c0^2/gamma [(rho/rho0)^gamma - 1]            PAPER.md:112 Eq.12
 * ------------------------------------------------------------------------------------------ */
typedef struct { double c0, rho0, gamma, delta, alpha, nu, eps, g[3]; int form; } Par;

static Par par_load(const double *p)
{
    Par P;
    P.c0 = p[0]; P.rho0 = p[1]; P.gamma = p[2]; P.delta = p[3]; P.alpha = p[4]; P.nu = p[5]; P.eps = p[6];
    P.g[0] = p[7]; P.g[1] = p[8]; P.g[2] = p[9]; P.form = (int)p[10];
    return P;
}

static double eos_p(const Par *P, double rho)
{ return P->rho0 * P->c0 * P->c0 / P->gamma * (pow(rho / P->rho0, P->gamma) - 1.0); }
static double eos_dp_drho(const Par *P, double rho)
{ return P->c0 * P->c0 * pow(rho / P->rho0, P->gamma - 1.0); }
static double eos_dp_dc0(const Par *P, double rho) { return 2.0 * eos_p(P, rho) / P->c0; }
static double eos_dp_drho0(const Par *P, double rho)
{
    double ug = pow(rho / P->rho0, P->gamma);
    return P->c0 * P->c0 / P->gamma * (ug - 1.0) - P->c0 * P->c0 * ug;
}
static double eos_dp_dgamma(const Par *P, double rho)
{
    double u = rho / P->rho0, ug = pow(u, P->gamma), B = P->rho0 * P->c0 * P->c0;
    return -B / (P->gamma * P->gamma) * (ug - 1.0) + B / P->gamma * ug * log(u);
}

/* pressure pair factor e_ij with E_ij = -m_j e_ij:
 *   form 0 (symmetric, Eq.40 read as A_i/rho_i^2 + A_j/rho_j^2):  e = p_i/rho_i^2 + p_j/rho_j^2
 *   form 1 (summation form Eq.39 divided by rho_i, PAPER.md:85 [51]):          e = (p_i + p_j)/(rho_i rho_j) */
static double e_pair(const Par *P, double ri, double rj)
{
    double pi_ = eos_p(P, ri), pj = eos_p(P, rj);
    return P->form == 0 ? pi_ / (ri * ri) + pj / (rj * rj) : (pi_ + pj) / (ri * rj);
}
/* d e / d rho_i  (the partial w.r.t. the first argument; d e/d rho_j follows by symmetry e(ri,rj)=e(rj,ri)) */
static double e_pair_d1(const Par *P, double ri, double rj)
{
    double pi_ = eos_p(P, ri), pj = eos_p(P, rj), dpi = eos_dp_drho(P, ri);
    if (P->form == 0) return dpi / (ri * ri) - 2.0 * pi_ / (ri * ri * ri);
    return dpi / (ri * rj) - (pi_ + pj) / (ri * ri * rj);
}
/* d e / d theta for theta in {c0, rho0, gamma} through p only */
static double e_pair_dtheta(const Par *P, double ri, double rj, int which)
{
    double di, dj;
    if (which == 0) { di = eos_dp_dc0(P, ri); dj = eos_dp_dc0(P, rj); }
    else if (which == 1) { di = eos_dp_drho0(P, ri); dj = eos_dp_drho0(P, rj); }
    else { di = eos_dp_dgamma(P, ri); dj = eos_dp_dgamma(P, rj); }
    return P->form == 0 ? di / (ri * ri) + dj / (rj * rj) : (di + dj) / (ri * rj);
}

/* everything one ordered pair (i <- j) needs, in the notation of SURVEY 8c-6 */
typedef struct {
    double d[3], w[3], r2, s, R, e2, H, ell, G, K, Vj, A, D, E, Phi1, Phi, eta, kd;
    int active;
} Pair;

static Pair pair_eval(const Par *P, int dim, const int *periodic, const double *L,
                      const double *xw, const double *v, const double *rho, const double *m, const double *h,
                      int64_t i, int64_t j)
{
    Pair q;
    memset(&q, 0, sizeof q);
    for (int k = 0; k < dim; ++k) { q.d[k] = xw[i * dim + k] - xw[j * dim + k]; q.w[k] = v[i * dim + k] - v[j * dim + k]; }
    min_image(q.d, dim, periodic, L);
    q.r2 = q.d[0] * q.d[0] + q.d[1] * q.d[1] + q.d[2] * q.d[2];
    q.H = h[i] > h[j] ? h[i] : h[j];
    double r = sqrt(q.r2);
    if (r >= q.H) { q.active = 0; return q; }          /* kernel clamp: W, G, K vanish for q >= 1 */
    q.active = 1;
    q.ell = q.H / kappa(dim);                           /* smoothing scale l = H/kappa_d */
    q.G = orc_gfac(r, q.H, dim);
    q.K = orc_kfac(r, q.H, dim);
    q.s = q.w[0] * q.d[0] + q.w[1] * q.d[1] + q.w[2] * q.d[2];
    q.e2 = (P->eps * q.H) * (P->eps * q.H);             /* (eps H)^2, Eq.42 denominator */
    q.R = q.r2 + q.e2;
    q.Vj = m[j] / rho[j];
    /* continuity, Eq.9 with Omega=1 and the physical sign (Eq.9's sign is garbled, cf. Eq.43):
     *   drho_i/dt = rho_i sum_j V_j (v_i - v_j) . grad_i W_ij                                    */
    q.A = rho[i] * q.Vj * q.s * q.G;
    /* delta-SPH diffusion (PAPER.md:103 cites [43],[50]; no equation printed). Reading: Molteni-Colagrossi
     *   delta l c0 sum_j psi_ij . grad_i W_ij V_j,  psi_ij = 2 (rho_j - rho_i)(x_j - x_i)/(r^2 + (eps H)^2)
     * = the Brookshaw Laplacian of rho (Eq.42, with its missing factor 2) times delta l c0. */
    q.kd = 2.0 * P->delta * q.ell * P->c0;
    q.D = q.kd * q.Vj * (rho[i] - rho[j]) * (q.r2 / q.R) * q.G;
    /* pressure: a = -grad p / rho, symmetric form PAPER.md:497 Eq.40 */
    q.E = -m[j] * e_pair(P, rho[i], rho[j]);
    /* viscosity PAPER.md:87 Eq.7 read with |x_ij|^2 + (eps H)^2, Pi_ij of delta-SPH [43]:
     *   a_i += eta (rho0/rho_i) sum_j V_j (v_ij . x_ij)/(r^2+(eps H)^2) grad_i W_ij ,
     *   eta = alpha l c0 + 2(d+2) nu   (Monaghan relation nu = alpha l c / (2(d+2)))              */
    q.eta = P->alpha * q.ell * P->c0 + 2.0 * (dim + 2) * P->nu;
    q.Phi1 = P->rho0 * q.Vj * q.s / (rho[i] * q.R);
    q.Phi = q.eta * q.Phi1;
    return q;
}

/* drho_i/dt = sum_j (A_ij + D_ij);   a_i = sum_j (E_ij + Phi_ij) G d + g;   a_i := 0 for boundary kinds.
 * rows == NULL: all rows; else only rows[0..nrows) are written (others untouched).
 * scale_drho / scale_acc (optional): sum_j of |pair terms|, the floor of the error metric. */
void orc_rhs(int64_t n, int dim, const int *periodic, const double *lo, const double *hi, const double *par,
             const double *x, const double *v, const double *rho, const double *m, const double *h,
             const uint8_t *kind, const int64_t *row_ptr, const int32_t *col_idx,
             const int64_t *rows, int64_t nrows,
             double *drho_dt, double *acc, double *scale_drho, double *scale_acc)
{
    Par P = par_load(par);
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    int64_t cnt = rows ? nrows : n;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t t = 0; t < cnt; ++t) {
        int64_t i = rows ? rows[t] : t;
        double dr = 0.0, a[3] = {0, 0, 0}, sd = 0.0, sa = 0.0;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            Pair q = pair_eval(&P, dim, periodic, L, xw, v, rho, m, h, i, j);
            if (!q.active) continue;
            dr += q.A + q.D;
            sd += fabs(q.A) + fabs(q.D);
            double dmax = 0.0;
            for (int k = 0; k < dim; ++k) {
                a[k] += (q.E + q.Phi) * q.G * q.d[k];
                if (fabs(q.d[k]) > dmax) dmax = fabs(q.d[k]);
            }
            sa += (fabs(q.E) + fabs(q.Phi)) * fabs(q.G) * dmax;
        }
        for (int k = 0; k < dim; ++k) {
            a[k] += P.g[k];
            if (kind[i]) a[k] = 0.0;
        }
        drho_dt[i] = dr;
        for (int k = 0; k < dim; ++k) acc[i * dim + k] = a[k];
        if (scale_drho) scale_drho[i] = sd;
        if (scale_acc) scale_acc[i] = sa;
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * c-7  VJP (Jacobian-transpose times incoming gradients; recompute pair terms;
 *      adjacency is not differentiated).
 * For T_ij = lambda_i (A_ij + D_ij) + (mu_i . d)(E_ij + Phi_ij) G  the reverse sweep over one ordered
 * pair (i <- j) is written out term by term below.  It mirrors PAPER.md:198: first the gradient on the
 * kernel factor G ("Gbar"), then ONE back-propagation through the kernel (K).
 * Scatter form: each ordered pair adds to particle i (first role) and particle j (second role).
 * ------------------------------------------------------------------------------------------ */
typedef struct { double dbar[3], wbar[3], rho_first, rho_second, pbar[7]; } PairAdj;

static PairAdj pair_adjoint(const Par *P, int dim, const Pair *q, double rho_i, double rho_j, double m_j,
                            double lam, const double *mu)
{
    PairAdj o;
    memset(&o, 0, sizeof o);
    double mm = mu[0] * q->d[0] + mu[1] * q->d[1] + mu[2] * q->d[2];          /* mu_i . d */
    double B = q->E + q->Phi;
    double drho = rho_i - rho_j;
    /* T = lam [rho_i Vj s G + kd Vj drho (r2/R) G] + mm (E + eta rho0 Vj s/(rho_i R)) G */
    double sbar = lam * rho_i * q->Vj * q->G + mm * q->eta * P->rho0 * q->Vj * q->G / (rho_i * q->R);
    double r2bar = lam * q->kd * q->Vj * drho * q->G * q->e2 / (q->R * q->R) - mm * q->Phi * q->G / q->R;
    double Gbar = lam * (rho_i * q->Vj * q->s + q->kd * q->Vj * drho * q->r2 / q->R) + mm * B;
    for (int k = 0; k < dim; ++k) {
        o.dbar[k] = sbar * q->w[k] + (2.0 * r2bar + Gbar * q->K) * q->d[k] + B * q->G * mu[k];
        o.wbar[k] = sbar * q->d[k];
    }
    double de_i = e_pair_d1(P, rho_i, rho_j), de_j = e_pair_d1(P, rho_j, rho_i);
    double diffu = lam * q->kd * q->Vj * (q->r2 / q->R) * q->G;
    o.rho_first = lam * q->Vj * q->s * q->G + diffu - mm * q->G * m_j * de_i - mm * q->G * q->Phi / rho_i;
    o.rho_second = -lam * (q->A + q->D) / rho_j - diffu - mm * q->G * m_j * de_j - mm * q->G * q->Phi / rho_j;
    /* scalar parameters: c0, rho0, gamma, delta, alpha, nu, eps */
    double xphi1 = mm * q->G * q->Phi1;
    o.pbar[0] = lam * q->D / P->c0 + xphi1 * P->alpha * q->ell - mm * q->G * m_j * e_pair_dtheta(P, rho_i, rho_j, 0);
    o.pbar[1] = xphi1 * q->eta / P->rho0 - mm * q->G * m_j * e_pair_dtheta(P, rho_i, rho_j, 1);
    o.pbar[2] = -mm * q->G * m_j * e_pair_dtheta(P, rho_i, rho_j, 2);
    o.pbar[3] = lam * 2.0 * q->ell * P->c0 * q->Vj * drho * (q->r2 / q->R) * q->G;
    o.pbar[4] = xphi1 * q->ell * P->c0;
    o.pbar[5] = xphi1 * 2.0 * (dim + 2);
    o.pbar[6] = -(lam * q->D + mm * q->G * q->Phi) / q->R * 2.0 * P->eps * q->H * q->H;
    return o;
}

/* rows == NULL: full adjoint (all outputs incl. params_bar[10] = c0,rho0,gamma,delta,alpha,nu,eps,gx,gy,gz).
 * rows != NULL: only x_bar/v_bar/rho_bar of the listed rows are produced (gathering both roles of every
 * pair that touches the row, which needs the symmetric list j in N(i) <=> i in N(j)); params_bar untouched. */
void orc_rhs_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi, const double *par,
                 const double *x, const double *v, const double *rho, const double *m, const double *h,
                 const uint8_t *kind, const int64_t *row_ptr, const int32_t *col_idx,
                 const double *drho_bar, const double *acc_bar,
                 const int64_t *rows, int64_t nrows,
                 double *x_bar, double *v_bar, double *rho_bar, double *params_bar)
{
    Par P = par_load(par);
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);

    if (rows) {
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t t = 0; t < nrows; ++t) {
            int64_t i = rows[t];
            double xb[3] = {0, 0, 0}, vb[3] = {0, 0, 0}, rb = 0.0;
            double mui[3] = {0, 0, 0};
            if (!kind[i]) for (int k = 0; k < dim; ++k) mui[k] = acc_bar[i * dim + k];
            for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
                int64_t j = col_idx[p];
                if (j == i) continue;                     /* self pair: d = 0, both roles cancel exactly */
                Pair q = pair_eval(&P, dim, periodic, L, xw, v, rho, m, h, i, j);
                if (!q.active) continue;
                PairAdj a = pair_adjoint(&P, dim, &q, rho[i], rho[j], m[j], drho_bar[i], mui);
                for (int k = 0; k < dim; ++k) { xb[k] += a.dbar[k]; vb[k] += a.wbar[k]; }
                rb += a.rho_first;
                double muj[3] = {0, 0, 0};
                if (!kind[j]) for (int k = 0; k < dim; ++k) muj[k] = acc_bar[j * dim + k];
                Pair q2 = pair_eval(&P, dim, periodic, L, xw, v, rho, m, h, j, i);
                PairAdj b = pair_adjoint(&P, dim, &q2, rho[j], rho[i], m[i], drho_bar[j], muj);
                for (int k = 0; k < dim; ++k) { xb[k] -= b.dbar[k]; vb[k] -= b.wbar[k]; }
                rb += b.rho_second;
            }
            for (int k = 0; k < dim; ++k) { x_bar[i * dim + k] = xb[k]; v_bar[i * dim + k] = vb[k]; }
            rho_bar[i] = rb;
        }
        free(xw);
        return;
    }

    memset(x_bar, 0, (size_t)n * dim * sizeof(double));
    memset(v_bar, 0, (size_t)n * dim * sizeof(double));
    memset(rho_bar, 0, (size_t)n * sizeof(double));
    double pb0 = 0, pb1 = 0, pb2 = 0, pb3 = 0, pb4 = 0, pb5 = 0, pb6 = 0, g0 = 0, g1 = 0, g2 = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : pb0, pb1, pb2, pb3, pb4, pb5, pb6, g0, g1, g2)
    for (int64_t i = 0; i < n; ++i) {
        double xb[3] = {0, 0, 0}, vb[3] = {0, 0, 0}, rb = 0.0;
        double mui[3] = {0, 0, 0};
        if (!kind[i]) for (int k = 0; k < dim; ++k) mui[k] = acc_bar[i * dim + k];
        g0 += mui[0]; g1 += mui[1]; g2 += mui[2];         /* a_i = ... + g for fluid kinds */
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            Pair q = pair_eval(&P, dim, periodic, L, xw, v, rho, m, h, i, j);
            if (!q.active) continue;
            PairAdj a = pair_adjoint(&P, dim, &q, rho[i], rho[j], m[j], drho_bar[i], mui);
            for (int k = 0; k < dim; ++k) { xb[k] += a.dbar[k]; vb[k] += a.wbar[k]; }
            rb += a.rho_first;
            for (int k = 0; k < dim; ++k) {
#pragma omp atomic
                x_bar[j * dim + k] -= a.dbar[k];
#pragma omp atomic
                v_bar[j * dim + k] -= a.wbar[k];
            }
#pragma omp atomic
            rho_bar[j] += a.rho_second;
            pb0 += a.pbar[0]; pb1 += a.pbar[1]; pb2 += a.pbar[2]; pb3 += a.pbar[3];
            pb4 += a.pbar[4]; pb5 += a.pbar[5]; pb6 += a.pbar[6];
        }
        for (int k = 0; k < dim; ++k) {
#pragma omp atomic
            x_bar[i * dim + k] += xb[k];
#pragma omp atomic
            v_bar[i * dim + k] += vb[k];
        }
#pragma omp atomic
        rho_bar[i] += rb;
    }
    if (params_bar) {
        params_bar[0] = pb0; params_bar[1] = pb1; params_bar[2] = pb2; params_bar[3] = pb3; params_bar[4] = pb4;
        params_bar[5] = pb5; params_bar[6] = pb6; params_bar[7] = g0; params_bar[8] = g1; params_bar[9] = g2;
    }
    free(xw);
}

/* ------------------------------------------------------------------------------------------
 * c-8  Classic RK4 ("standard fourth-order Runge-Kutta") of
 *      y = (x, v, rho),  f(y) = (v, a, drho/dt);  boundary kinds: dx/dt = 0, a = 0.
 * Reading: exact neighbours at EVERY stage (rebuilt here from the stage positions).
 * ------------------------------------------------------------------------------------------ */
typedef struct { int64_t nnz; int64_t *row_ptr; int32_t *col_idx; } List;

static List build_list(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                       const double *x, const double *h, int method)
{
    List l;
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    l.row_ptr = (int64_t *)malloc(((size_t)n + 1) * sizeof(int64_t));
    l.nnz = orc_neighbors(n, dim, periodic, lo, hi, xw, h, 1.0, method, l.row_ptr, NULL);
    l.col_idx = (int32_t *)malloc((size_t)(l.nnz > 0 ? l.nnz : 1) * sizeof(int32_t));
    orc_neighbors(n, dim, periodic, lo, hi, xw, h, 1.0, method, l.row_ptr, l.col_idx);
    free(xw);
    return l;
}
static void free_list(List *l) { free(l->row_ptr); free(l->col_idx); }

/* k = f(Y): kx = v (0 for boundary), kv = a, kr = drho/dt */
static void f_eval(int64_t n, int dim, const int *periodic, const double *lo, const double *hi, const double *par,
                   const double *X, const double *V, const double *Rr, const double *m, const double *h,
                   const uint8_t *kind, int method, double *kx, double *kv, double *kr)
{
    List l = build_list(n, dim, periodic, lo, hi, X, h, method);
    orc_rhs(n, dim, periodic, lo, hi, par, X, V, Rr, m, h, kind, l.row_ptr, l.col_idx, NULL, 0, kr, kv, NULL, NULL);
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < dim; ++k) kx[i * dim + k] = kind[i] ? 0.0 : V[i * dim + k];
    free_list(&l);
}

void orc_rk4_step(int64_t n, int dim, const int *periodic, const double *lo, const double *hi, const double *par,
                  double dt, double *x, double *v, double *rho, const double *m, const double *h,
                  const uint8_t *kind, int method)
{
    size_t nv = (size_t)n * dim, ns = (size_t)n;
    double *kx[4], *kv[4], *kr[4];
    for (int s = 0; s < 4; ++s) {
        kx[s] = (double *)malloc(nv * sizeof(double));
        kv[s] = (double *)malloc(nv * sizeof(double));
        kr[s] = (double *)malloc(ns * sizeof(double));
    }
    double *X = (double *)malloc(nv * sizeof(double)), *V = (double *)malloc(nv * sizeof(double));
    double *R = (double *)malloc(ns * sizeof(double));
    const double c[4] = {0.0, 0.5, 0.5, 1.0};
    for (int s = 0; s < 4; ++s) {
        for (size_t t = 0; t < nv; ++t) {
            X[t] = x[t] + (s ? c[s] * dt * kx[s - 1][t] : 0.0);
            V[t] = v[t] + (s ? c[s] * dt * kv[s - 1][t] : 0.0);
        }
        for (size_t t = 0; t < ns; ++t) R[t] = rho[t] + (s ? c[s] * dt * kr[s - 1][t] : 0.0);
        f_eval(n, dim, periodic, lo, hi, par, X, V, R, m, h, kind, method, kx[s], kv[s], kr[s]);
    }
    for (size_t t = 0; t < nv; ++t) {
        x[t] += dt / 6.0 * (kx[0][t] + 2.0 * kx[1][t] + 2.0 * kx[2][t] + kx[3][t]);
        v[t] += dt / 6.0 * (kv[0][t] + 2.0 * kv[1][t] + 2.0 * kv[2][t] + kv[3][t]);
    }
    for (size_t t = 0; t < ns; ++t) rho[t] += dt / 6.0 * (kr[0][t] + 2.0 * kr[1][t] + 2.0 * kr[2][t] + kr[3][t]);
    for (int s = 0; s < 4; ++s) { free(kx[s]); free(kv[s]); free(kr[s]); }
    free(X); free(V); free(R);
}

/* Discrete adjoint of one RK4 step, stages recomputed from the stored step state
 * ("only essential particle data is retained").  In: cotangents at t+dt in x_bar/v_bar/rho_bar.
 * Out: cotangents at t (same arrays).  params_bar[10] is ACCUMULATED into.                       */
void orc_rk4_step_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi, const double *par,
                      double dt, const double *x0, const double *v0, const double *r0, const double *m,
                      const double *h, const uint8_t *kind, int method,
                      double *x_bar, double *v_bar, double *rho_bar, double *params_bar)
{
    size_t nv = (size_t)n * dim, ns = (size_t)n;
    double *Yx[4], *Yv[4], *Yr[4];
    double *kx = (double *)malloc(nv * sizeof(double)), *kv = (double *)malloc(nv * sizeof(double));
    double *kr = (double *)malloc(ns * sizeof(double));
    const double c[4] = {0.0, 0.5, 0.5, 1.0};
    for (int s = 0; s < 4; ++s) {
        Yx[s] = (double *)malloc(nv * sizeof(double));
        Yv[s] = (double *)malloc(nv * sizeof(double));
        Yr[s] = (double *)malloc(ns * sizeof(double));
        for (size_t t = 0; t < nv; ++t) {
            Yx[s][t] = x0[t] + (s ? c[s] * dt * kx[t] : 0.0);
            Yv[s][t] = v0[t] + (s ? c[s] * dt * kv[t] : 0.0);
        }
        for (size_t t = 0; t < ns; ++t) Yr[s][t] = r0[t] + (s ? c[s] * dt * kr[t] : 0.0);
        if (s < 3) f_eval(n, dim, periodic, lo, hi, par, Yx[s], Yv[s], Yr[s], m, h, kind, method, kx, kv, kr);
    }
    /* reverse sweep: kbar_4 = dt/6 ybar+ ; Ybar_s = J^T(Y_s) kbar_s ; kbar_{s-1} = b_{s-1} dt ybar+ + a_{s,s-1} dt Ybar_s */
    const double b[4] = {1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0};
    double *kbx = (double *)malloc(nv * sizeof(double)), *kbv = (double *)malloc(nv * sizeof(double));
    double *kbr = (double *)malloc(ns * sizeof(double));
    double *Ybx = (double *)calloc(nv, sizeof(double)), *Ybv = (double *)calloc(nv, sizeof(double));
    double *Ybr = (double *)calloc(ns, sizeof(double));
    double *sx = (double *)calloc(nv, sizeof(double)), *sv = (double *)calloc(nv, sizeof(double));
    double *sr = (double *)calloc(ns, sizeof(double));
    double pb[10];
    for (int s = 3; s >= 0; --s) {
        double a_next = (s == 3) ? 0.0 : c[s + 1];         /* a_{s+1,s} of the classic tableau = c_{s+1} */
        for (size_t t = 0; t < nv; ++t) {
            kbx[t] = b[s] * dt * x_bar[t] + a_next * dt * Ybx[t];
            kbv[t] = b[s] * dt * v_bar[t] + a_next * dt * Ybv[t];
        }
        for (size_t t = 0; t < ns; ++t) kbr[t] = b[s] * dt * rho_bar[t] + a_next * dt * Ybr[t];
        List l = build_list(n, dim, periodic, lo, hi, Yx[s], h, method);
        orc_rhs_vjp(n, dim, periodic, lo, hi, par, Yx[s], Yv[s], Yr[s], m, h, kind, l.row_ptr, l.col_idx,
                    kbr, kbv, NULL, 0, Ybx, Ybv, Ybr, pb);
        free_list(&l);
        for (int64_t i = 0; i < n; ++i)
            if (!kind[i]) for (int k = 0; k < dim; ++k) Ybv[i * dim + k] += kbx[i * dim + k];   /* dx/dt = v */
        for (size_t t = 0; t < nv; ++t) { sx[t] += Ybx[t]; sv[t] += Ybv[t]; }
        for (size_t t = 0; t < ns; ++t) sr[t] += Ybr[t];
        if (params_bar) for (int k = 0; k < 10; ++k) params_bar[k] += pb[k];
    }
    for (size_t t = 0; t < nv; ++t) { x_bar[t] += sx[t]; v_bar[t] += sv[t]; }
    for (size_t t = 0; t < ns; ++t) rho_bar[t] += sr[t];
    for (int s = 0; s < 4; ++s) { free(Yx[s]); free(Yv[s]); free(Yr[s]); }
    free(kx); free(kv); free(kr); free(kbx); free(kbv); free(kbr);
    free(Ybx); free(Ybv); free(Ybr); free(sx); free(sv); free(sr);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-2  delta-SPH diffusion with the renormalised density gradient (PAPER.md:103 cites [43], PAPER.md:85 [51];
 * the equation is not printed -- DESIGN.md reading R17).  The term of Antuono et al. [43]:
 *     D_i = delta l c0 sum_j psi_ij . grad_i W_ij V_j ,
 *     psi_ij = 2 (rho_j - rho_i) (x_j - x_i)/|x_ij|^2  -  [ <grad rho>^L_i + <grad rho>^L_j ] ,
 * <grad rho>^L the renormalised gradient of PAPER.md:524-528 Eq.44/45.  The first part is the Molteni-Colagrossi
 * term orc_rhs already adds (delta_form 0, with its (eps H)^2 regularisation); this function adds the second,
 *     X_ij = - delta l_ij c0 V_j (g_i + g_j) . d G ,   d = x_i - x_j ,  grad_i W_ij = G d ,
 * with g = <grad rho>^L passed in (the pseudo-inverse L_i is formed by the caller, oracle/__init__.py).
 * drho_dt is ADDED to; scale_drho (may be NULL) gets sum_j |X_ij| added.
 * ------------------------------------------------------------------------------------------ */
void orc_delta_renorm_term(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                           const double *par, const double *x, const double *rho, const double *m, const double *h,
                           const int64_t *row_ptr, const int32_t *col_idx, const double *grho,
                           const int64_t *rows, int64_t nrows, double *drho_dt, double *scale_drho)
{
    Par P = par_load(par);
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    int64_t cnt = rows ? nrows : n;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t t = 0; t < cnt; ++t) {
        int64_t i = rows ? rows[t] : t;
        double dr = 0.0, sd = 0.0;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            if (r >= H) continue;
            double G = orc_gfac(r, H, dim);
            double ell = H / kappa(dim);
            double S = 0.0;
            for (int k = 0; k < dim; ++k) S += (grho[i * dim + k] + grho[j * dim + k]) * d[k];
            double X = -P.delta * ell * P.c0 * (m[j] / rho[j]) * S * G;
            dr += X;
            sd += fabs(X);
        }
        drho_dt[i] += dr;
        if (scale_drho) scale_drho[i] += sd;
    }
    free(xw);
}

/* Adjoint of the term above for the cotangent lam = dL/d(drho_dt), scatter form over ordered pairs (serial: the
 * definition).  Direct dependences only: x (through d and G; dG = K d.dd), rho_j (through V_j = m_j/rho_j), delta, c0,
 * and the gradient field g, whose cotangent g_bar [n][dim] is returned for the caller to push through the adjoint of
 * the renormalised gradient (orc_renorm_moments_vjp + the pseudo-inverse, oracle/__init__.py).
 * x_bar, rho_bar, params_bar[10] are ADDED to; g_bar is overwritten. */
void orc_delta_renorm_term_vjp(int64_t n, int dim, const int *periodic, const double *lo, const double *hi,
                               const double *par, const double *x, const double *rho, const double *m, const double *h,
                               const int64_t *row_ptr, const int32_t *col_idx, const double *grho, const double *lam,
                               double *x_bar, double *rho_bar, double *g_bar, double *params_bar)
{
    Par P = par_load(par);
    double L[3];
    box_len(dim, lo, hi, L);
    double *xw = (double *)malloc((size_t)n * dim * sizeof(double));
    wrap64(n, dim, periodic, lo, hi, x, xw);
    memset(g_bar, 0, (size_t)n * dim * sizeof(double));
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int64_t j = col_idx[p];
            double d[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k) d[k] = xw[i * dim + k] - xw[j * dim + k];
            min_image(d, dim, periodic, L);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double H = h[i] > h[j] ? h[i] : h[j];
            if (r >= H) continue;
            double G = orc_gfac(r, H, dim), K = orc_kfac(r, H, dim);
            double ell = H / kappa(dim);
            double Vj = m[j] / rho[j];
            double c = -P.delta * ell * P.c0 * Vj;              /* X = c S G */
            double S = 0.0;
            for (int k = 0; k < dim; ++k) S += (grho[i * dim + k] + grho[j * dim + k]) * d[k];
            double X = c * S * G;
            for (int k = 0; k < dim; ++k) {
                /* dX/dd_k = c [ (g_i + g_j)_k G + S K d_k ] */
                double F = lam[i] * c * ((grho[i * dim + k] + grho[j * dim + k]) * G + S * K * d[k]);
                x_bar[i * dim + k] += F;
                x_bar[j * dim + k] -= F;
                /* dX/dg_i = dX/dg_j = c G d */
                g_bar[i * dim + k] += lam[i] * c * G * d[k];
                g_bar[j * dim + k] += lam[i] * c * G * d[k];
            }
            rho_bar[j] += -lam[i] * X / rho[j];                 /* V_j = m_j / rho_j */
            params_bar[3] += lam[i] * X / P.delta;              /* delta */
            params_bar[0] += lam[i] * X / P.c0;                 /* c0 */
        }
    }
    free(xw);
}

int orc_num_threads(void)
{
    int nt = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        nt = omp_get_num_threads();
    }
#endif
    return nt;
}
