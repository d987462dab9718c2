/*
 * jastrow_ref.c -- CPU ORACLE for the homogeneous two-body Jastrow terms u and p.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow restatement of /root/reference/PAPER.md section 2.3:
 *   Eq. 6  u(r) = sum_{l=0}^{N_u} alpha_l r^l (r - L_u)^C Theta(L_u - r)
 *   Eq. 7  p(r) = sum_{m=1}^{N_p} a_m sum_{G in star_m^+} cos(G.r)
 *   PAPER.md:151          L_u is less than half the distance to the closest lattice point (so only the minimum
 *                         image of a pair can lie inside the cut-off); "+" = one G of each +-G pair
 *   PAPER.md:142          "values and derivatives of the two-body terms": for each particle i the value
 *                         J = sum_{i<j} [u(r_ij) + p(r_ij)], the gradient grad_i J and the Laplacian lap_i J
 *   PAPER.md:94           single-particle moves: Delta J for r_k -> r'
 * Every pair is visited and every cosine is a direct cosl/sinl of G.r_ij from Cartesian G and r_ij: no
 * structure factor, no phase powers (Eq. 8 is what the fast path uses), no tables.  Sums in long double.
 * Shares nothing with the CUDA path.  Pins: tests/test_jastrow_pins.py.
 *
 * Layouts (HOST): cell[9] row-major lattice vectors (dim = 2 uses [0,1,3,4]); pos [W][n][dim];
 * g_n [n_g][3] integer coefficients of G = n1 b1 + n2 b2 + n3 b3 (one of each +-G pair), star [n_g] = index of
 * the coefficient a[star] of that G; alpha [n_u + 1].
 * Outputs: value [W]; grad [W][n][dim]; lap [W][n].  Return 0 = ok.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double real;
static const real PI_L = 3.141592653589793238462643383279502884L;

static int cell_setup(int dim, const double *cell, real a[3][3], real b[3][3])
{
    /* a: lattice rows; b: reciprocal rows with a_i . b_j = 2 pi delta_ij */
    int i, j;
    for (i = 0; i < 3; i++) for (j = 0; j < 3; j++) a[i][j] = i == j ? 1 : 0;
    if (dim == 3) { for (i = 0; i < 3; i++) for (j = 0; j < 3; j++) a[i][j] = cell[3 * i + j]; }
    else if (dim == 2) { a[0][0] = cell[0]; a[0][1] = cell[1]; a[1][0] = cell[3]; a[1][1] = cell[4]; }
    else return 1;
    real det = a[0][0] * (a[1][1] * a[2][2] - a[1][2] * a[2][1]) - a[0][1] * (a[1][0] * a[2][2] - a[1][2] * a[2][0]) +
               a[0][2] * (a[1][0] * a[2][1] - a[1][1] * a[2][0]);
    if (det == 0) return 1;
    for (i = 0; i < 3; i++) {
        const int i1 = (i + 1) % 3, i2 = (i + 2) % 3;
        b[i][0] = 2 * PI_L * (a[i1][1] * a[i2][2] - a[i1][2] * a[i2][1]) / det;
        b[i][1] = 2 * PI_L * (a[i1][2] * a[i2][0] - a[i1][0] * a[i2][2]) / det;
        b[i][2] = 2 * PI_L * (a[i1][0] * a[i2][1] - a[i1][1] * a[i2][0]) / det;
    }
    return 0;
}

/* minimum image of d: subtract the lattice vector nearest in fractional coordinates, then check the 3^dim
 * neighbours (a skewed cell's nearest image need not be the fractionally rounded one) */
static void min_image(int dim, real a[3][3], real b[3][3], real d[3])
{
    int k, x, m0, m1, m2;
    real f[3];
    for (k = 0; k < 3; k++) {
        real s = 0;
        for (x = 0; x < 3; x++) s += d[x] * b[k][x];
        f[k] = k < dim ? nearbyintl(s / (2 * PI_L)) : 0;
    }
    for (x = 0; x < 3; x++) for (k = 0; k < dim; k++) d[x] -= f[k] * a[k][x];
    real best[3] = {d[0], d[1], d[2]}, best2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    for (m0 = -1; m0 <= 1; m0++) for (m1 = -1; m1 <= 1; m1++) for (m2 = (dim == 3 ? -1 : 0); m2 <= (dim == 3 ? 1 : 0); m2++) {
        real t[3];
        for (x = 0; x < 3; x++) t[x] = d[x] - m0 * a[0][x] - m1 * a[1][x] - m2 * a[2][x];
        const real t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
        if (t2 < best2) { best2 = t2; best[0] = t[0]; best[1] = t[1]; best[2] = t[2]; }
    }
    d[0] = best[0]; d[1] = best[1]; d[2] = best[2];
}

/* Eq. 6 and its first two derivatives at r < L_u (0 beyond) */
static void u_of_r(int n_u, const double *alpha, real L_u, int C, real r, real *u, real *du, real *d2u)
{
    *u = *du = *d2u = 0;
    if (!(r < L_u)) return;
    real poly = 0, dpoly = 0, d2poly = 0, rl = 1; /* sum alpha_l r^l and derivatives, term by term */
    int l;
    for (l = 0; l <= n_u; l++) {
        poly += alpha[l] * rl;
        if (l >= 1) dpoly += alpha[l] * l * powl(r, l - 1);
        if (l >= 2) d2poly += alpha[l] * l * (l - 1) * powl(r, l - 2);
        rl *= r;
    }
    const real s = r - L_u, sc = powl(s, C), sc1 = C >= 1 ? C * powl(s, C - 1) : 0, sc2 = C >= 2 ? C * (C - 1) * powl(s, C - 2) : 0;
    *u = poly * sc;
    *du = dpoly * sc + poly * sc1;
    *d2u = d2poly * sc + 2 * dpoly * sc1 + poly * sc2;
}

/* one pair displacement d = r_i - r_j: value of u + p, gradient with respect to r_i, Laplacian */
static void pair_terms(int dim, real a[3][3], real b[3][3], int n_u, const double *alpha, real L_u, int C,
                       int n_g, const int *g_n, const int *star, const double *acoef, const real d_in[3],
                       real *val, real grad[3], real *lap)
{
    int g, x;
    *val = 0; *lap = 0; grad[0] = grad[1] = grad[2] = 0;
    if (n_u >= 0 && L_u > 0) {
        real d[3] = {d_in[0], d_in[1], d_in[2]};
        min_image(dim, a, b, d);
        const real r = sqrtl(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        real u, du, d2u;
        u_of_r(n_u, alpha, L_u, C, r, &u, &du, &d2u);
        *val += u;
        if (r > 0) {
            for (x = 0; x < dim; x++) grad[x] += du * d[x] / r;
            *lap += d2u + (dim - 1) * du / r;
        }
    }
    for (g = 0; g < n_g; g++) {
        real G[3] = {0, 0, 0}, ph = 0, g2 = 0;
        int k;
        for (k = 0; k < dim; k++) for (x = 0; x < 3; x++) G[x] += g_n[3 * g + k] * b[k][x];
        for (x = 0; x < 3; x++) { ph += G[x] * d_in[x]; g2 += G[x] * G[x]; }
        const real am = acoef[star[g]], c = cosl(ph), s = sinl(ph);
        *val += am * c;
        for (x = 0; x < dim; x++) grad[x] -= am * G[x] * s;
        *lap -= am * g2 * c;
    }
}

int jastrow_ref_batch(int dim, const double *cell, int n_u, const double *alpha, double L_u, int C,
                      int n_g, const int *g_n, const int *star, const double *acoef,
                      int n_walkers, int n, const double *pos, double *value, double *grad, double *lap)
{
    real a[3][3], b[3][3];
    if (cell_setup(dim, cell, a, b) || n <= 0 || n_walkers < 0) return 1;
    int w;
#pragma omp parallel for schedule(dynamic, 1)
    for (w = 0; w < n_walkers; w++) {
        const double *p = pos + (size_t)w * n * dim;
        real total = 0;
        int i, j, x;
        for (i = 0; i < n; i++) {
            real gi[3] = {0, 0, 0}, li = 0;
            for (j = 0; j < n; j++) {
                if (j == i) continue;
                real d[3] = {0, 0, 0}, v, gr[3], lp;
                for (x = 0; x < dim; x++) d[x] = (real)p[i * dim + x] - (real)p[j * dim + x];
                pair_terms(dim, a, b, n_u, alpha, L_u, C, n_g, g_n, star, acoef, d, &v, gr, &lp);
                if (j > i) total += v;
                for (x = 0; x < dim; x++) gi[x] += gr[x];
                li += lp;
            }
            if (grad) for (x = 0; x < dim; x++) grad[((size_t)w * n + i) * dim + x] = (double)gi[x];
            if (lap) lap[(size_t)w * n + i] = (double)li;
        }
        if (value) value[w] = (double)total;
    }
    return 0;
}

/* Delta J of one single-particle move per walker and step, applied in sequence (always committed):
 * electron [n_steps][W], new_r [n_steps][W][dim]; delta [n_steps][W]; pos_out [W][n][dim] (nullable). */
int jastrow_ref_move_chain(int dim, const double *cell, int n_u, const double *alpha, double L_u, int C,
                           int n_g, const int *g_n, const int *star, const double *acoef,
                           int n_walkers, int n, const double *pos, int n_steps, const int *electron,
                           const double *new_r, double *delta, double *pos_out)
{
    real a[3][3], b[3][3];
    if (cell_setup(dim, cell, a, b) || n <= 0) return 1;
    int w;
#pragma omp parallel for schedule(dynamic, 1)
    for (w = 0; w < n_walkers; w++) {
        double *p = (double *)malloc(sizeof(double) * n * dim);
        memcpy(p, pos + (size_t)w * n * dim, sizeof(double) * n * dim);
        int s, j, x;
        for (s = 0; s < n_steps; s++) {
            const int k = electron[(size_t)s * n_walkers + w];
            const double *rn = new_r + ((size_t)s * n_walkers + w) * dim;
            real dj = 0;
            for (j = 0; j < n; j++) {
                if (j == k) continue;
                real d0[3] = {0, 0, 0}, d1[3] = {0, 0, 0}, v0, v1, gr[3], lp;
                for (x = 0; x < dim; x++) { d0[x] = (real)p[k * dim + x] - (real)p[j * dim + x]; d1[x] = (real)rn[x] - (real)p[j * dim + x]; }
                pair_terms(dim, a, b, n_u, alpha, L_u, C, n_g, g_n, star, acoef, d0, &v0, gr, &lp);
                pair_terms(dim, a, b, n_u, alpha, L_u, C, n_g, g_n, star, acoef, d1, &v1, gr, &lp);
                dj += v1 - v0;
            }
            delta[(size_t)s * n_walkers + w] = (double)dj;
            for (x = 0; x < dim; x++) p[k * dim + x] = rn[x];
        }
        if (pos_out) memcpy(pos_out + (size_t)w * n * dim, p, sizeof(double) * n * dim);
        free(p);
    }
    return 0;
}

/* u(r), u'(r), u''(r) of Eq. 6 at one r (for the pins) */
int jastrow_ref_u(int n_u, const double *alpha, double L_u, int C, double r, double *u, double *du, double *d2u)
{
    real v, d1, d2;
    u_of_r(n_u, alpha, L_u, C, r, &v, &d1, &d2);
    *u = (double)v; *du = (double)d1; *d2u = (double)d2;
    return 0;
}

int jastrow_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
