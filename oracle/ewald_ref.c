/*
 * ewald_ref.c -- CPU ORACLE (test infrastructure only; see ewald_ref.h for the contract).
 *
 * Written from /root/reference/PAPER.md Eqs. 2-4 (lines 112-120) and the symbol definitions at
 * line 122.  gamma_paper = kappa^2.  Everything is `long double`; trigonometric and error functions
 * are the libm ones (cosl, sincosl, erfcl, expl), evaluated once per (particle, G) or per
 * (pair, image): no recurrences, no symmetry tricks, no blocking.  Shares no code with the CUDA path.
 *
 * Decomposition used by the O-rho form (exact regrouping of Eq. 2, derived in DESIGN.md section 2):
 *   E = E_recip + E_real + E_self + E_bg
 *   3D: E_recip = (2pi/Omega) sum_{G!=0} exp(-G^2/4kappa^2)/G^2 |rho(G)|^2
 *       E_bg    = -pi Q^2 / (2 Omega kappa^2)
 *   2D: E_recip = (pi/A) sum_{G!=0} erfc(G/2kappa)/G |rho(G)|^2            (reading R2)
 *       E_bg    = -sqrt(pi) Q^2 / (A kappa)
 *   both: E_real = sum_{i<j} q_i q_j sum_R erfc(kappa|r_ij-R|)/|r_ij-R|  +  1/2 sum_j q_j^2 xi_R,
 *         xi_R = sum_{R!=0} erfc(kappa R)/R,      E_self = -(kappa/sqrt(pi)) sum_j q_j^2
 *   with rho(G) = sum_i q_i exp(iG.r_i), Q = sum_i q_i, and every real-space term kept iff its
 *   distance is < r_cutoff (reading R3), every G kept iff G^2 <= g_cutoff^2 (1+1e-12) (reading R6).
 */
#define _GNU_SOURCE
#include "ewald_ref.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

#define PI_L 3.14159265358979323846264338327950288L

typedef struct {
    int dim;
    ld a[3][3]; /* lattice vectors as rows; dim = 2 is embedded with a3 = (0,0,1)            */
    ld b[3][3]; /* reciprocal vectors as rows, a_i . b_j = 2 pi delta_ij                     */
    ld vol;     /* |det a| : volume (3D) or area (2D)                                        */
    ld reach;   /* bound on |d| after the fractional-coordinate reduction: (|a1|+|a2|+|a3|)/2 */
} cell_t;

typedef struct {
    int n;      /* number of points                      */
    int (*idx)[3];
    ld (*v)[3];
    ld *w;      /* per-point weight (G lists only)       */
} lattice_list_t;

static ld norm3(const ld *x) { return sqrtl(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]); }

static int cell_init(cell_t *c, int dim, const double *cell)
{
    if ((dim != 2 && dim != 3) || !cell) return 1;
    memset(c, 0, sizeof *c);
    c->dim = dim;
    if (dim == 3) {
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) c->a[i][j] = (ld)cell[3 * i + j];
    } else {
        c->a[0][0] = cell[0]; c->a[0][1] = cell[1];
        c->a[1][0] = cell[3]; c->a[1][1] = cell[4];
        c->a[2][2] = 1.0L;
    }
    const ld(*a)[3] = c->a;
    ld cof[3][3];
    cof[0][0] = a[1][1] * a[2][2] - a[1][2] * a[2][1];
    cof[0][1] = a[1][2] * a[2][0] - a[1][0] * a[2][2];
    cof[0][2] = a[1][0] * a[2][1] - a[1][1] * a[2][0];
    cof[1][0] = a[2][1] * a[0][2] - a[2][2] * a[0][1];
    cof[1][1] = a[2][2] * a[0][0] - a[2][0] * a[0][2];
    cof[1][2] = a[2][0] * a[0][1] - a[2][1] * a[0][0];
    cof[2][0] = a[0][1] * a[1][2] - a[0][2] * a[1][1];
    cof[2][1] = a[0][2] * a[1][0] - a[0][0] * a[1][2];
    cof[2][2] = a[0][0] * a[1][1] - a[0][1] * a[1][0];
    ld det = a[0][0] * cof[0][0] + a[0][1] * cof[0][1] + a[0][2] * cof[0][2];
    if (!(fabsl(det) > 0.0L)) return 2;
    /* b_i = 2 pi (a_j x a_k) / det : rows of 2 pi (A^-1)^T = 2 pi cof / det */
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c->b[i][j] = 2.0L * PI_L * cof[i][j] / det;
    c->vol = fabsl(det);
    c->reach = 0.5L * (norm3(a[0]) + norm3(a[1]) + (dim == 3 ? norm3(a[2]) : 0.0L));
    return 0;
}

/* All integer combinations sum_k m_k basis[k] with squared length <= r2max; m3 = 0 in 2D.
 * `other` is the dual basis (other_k . basis_j = 2 pi delta_kj), used only to bound the integer ranges:
 * |m_k| = |v . other_k| / 2pi <= |v| |other_k| / 2pi.                                              */
static int lattice_points(const cell_t *c, const ld basis[3][3], const ld other[3][3], ld r2max,
                          int skip_zero, lattice_list_t *out)
{
    ld rmax = sqrtl(r2max);
    int lim[3];
    for (int k = 0; k < 3; k++) {
        lim[k] = (int)floorl(rmax * norm3(other[k]) / (2.0L * PI_L) + 1e-9L) + 1;
        if (k >= c->dim) lim[k] = 0;
    }
    size_t cap = (size_t)(2 * lim[0] + 1) * (2 * lim[1] + 1) * (2 * lim[2] + 1);
    out->idx = malloc(cap * sizeof *out->idx);
    out->v = malloc(cap * sizeof *out->v);
    out->w = NULL;
    out->n = 0;
    if (!out->idx || !out->v) return 3;
    for (int m1 = -lim[0]; m1 <= lim[0]; m1++)
        for (int m2 = -lim[1]; m2 <= lim[1]; m2++)
            for (int m3 = -lim[2]; m3 <= lim[2]; m3++) {
                if (skip_zero && m1 == 0 && m2 == 0 && m3 == 0) continue;
                ld v[3];
                for (int x = 0; x < 3; x++)
                    v[x] = m1 * basis[0][x] + m2 * basis[1][x] + m3 * basis[2][x];
                ld v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
                if (v2 > r2max) continue;
                int k = out->n++;
                out->idx[k][0] = m1; out->idx[k][1] = m2; out->idx[k][2] = m3;
                out->v[k][0] = v[0]; out->v[k][1] = v[1]; out->v[k][2] = v[2];
            }
    return 0;
}

static void list_free(lattice_list_t *l)
{
    free(l->idx); free(l->v); free(l->w);
    l->idx = NULL; l->v = NULL; l->w = NULL; l->n = 0;
}

/* Reciprocal-space weight w(G) such that E_recip = sum_{G != 0, full sphere} w(G) |rho(G)|^2.
 * 3D: Eq. 3's (4 pi/Omega) exp(-G^2/4 gamma)/G^2 regrouped over pairs gives the factor 1/2.
 * 2D: (pi/A) erfc(G/2kappa)/G  (reading R2).                                                   */
static ld recip_weight(const cell_t *c, ld kappa, ld g2)
{
    if (c->dim == 3) return 2.0L * PI_L / c->vol * expl(-g2 / (4.0L * kappa * kappa)) / g2;
    ld g = sqrtl(g2);
    return PI_L / c->vol * erfcl(g / (2.0L * kappa)) / g;
}

/* Full-sphere G list (G != 0) with weights; reading R6 for shell membership. */
static int g_list(const cell_t *c, ld kappa, ld gcut, lattice_list_t *out)
{
    int rc = lattice_points(c, c->b, c->a, gcut * gcut * (1.0L + 1e-12L), 1, out);
    if (rc) return rc;
    out->w = malloc((size_t)(out->n > 0 ? out->n : 1) * sizeof *out->w);
    if (!out->w) return 3;
    for (int k = 0; k < out->n; k++) {
        const ld *g = out->v[k];
        out->w[k] = kappa > 0 ? recip_weight(c, kappa, g[0] * g[0] + g[1] * g[1] + g[2] * g[2]) : 0;
    }
    return 0;
}

static int is_plus(const int *n)
{
    if (n[0] != 0) return n[0] > 0;
    if (n[1] != 0) return n[1] > 0;
    return n[2] > 0;
}

/* Half set in lexicographic (n1,n2,n3) order: lattice_points already loops that way. */
static int gplus_list(const cell_t *c, ld kappa, ld gcut, lattice_list_t *out)
{
    lattice_list_t full;
    int rc = g_list(c, kappa, gcut, &full);
    if (rc) return rc;
    int n = 0;
    for (int k = 0; k < full.n; k++)
        if (is_plus(full.idx[k])) {
            memcpy(full.idx[n], full.idx[k], sizeof full.idx[0]);
            memcpy(full.v[n], full.v[k], sizeof full.v[0]);
            full.w[n] = full.w[k];
            n++;
        }
    full.n = n;
    *out = full;
    return 0;
}

/* Lattice vectors R (including 0) that can come within r_cutoff of a displacement of length <= dmax. */
static int image_list(const cell_t *c, ld rcut, ld dmax, lattice_list_t *out)
{
    ld r = rcut + dmax;
    return lattice_points(c, c->a, c->b, r * r * (1.0L + 1e-12L), 0, out);
}

/* d <- d minus the lattice vector that brings its fractional coordinates into [-1/2, 1/2] (reading R10). */
static void reduce_displacement(const cell_t *c, ld *d)
{
    ld f[3];
    for (int k = 0; k < 3; k++) {
        f[k] = (d[0] * c->b[k][0] + d[1] * c->b[k][1] + d[2] * c->b[k][2]) / (2.0L * PI_L);
        f[k] = (k < c->dim) ? nearbyintl(f[k]) : 0.0L;
    }
    for (int x = 0; x < 3; x++)
        d[x] -= f[0] * c->a[0][x] + f[1] * c->a[1][x] + f[2] * c->a[2][x];
}

/* psi(d) = sum_R erfc(kappa |d - R|)/|d - R| over images with |d - R| < rcut; d already reduced. */
static ld psi_images(const lattice_list_t *img, ld kappa, ld rcut, const ld *d)
{
    ld s = 0.0L;
    for (int k = 0; k < img->n; k++) {
        ld x = d[0] - img->v[k][0], y = d[1] - img->v[k][1], z = d[2] - img->v[k][2];
        ld r2 = x * x + y * y + z * z;
        if (r2 < rcut * rcut) {
            ld r = sqrtl(r2);
            s += erfcl(kappa * r) / r;
        }
    }
    return s;
}

/* xi_R = sum_{R != 0, |R| < rcut} erfc(kappa R)/R  (the real-lattice sum of Eq. 4). */
static ld xi_real(const cell_t *c, ld kappa, ld rcut)
{
    lattice_list_t img;
    if (image_list(c, rcut, 0.0L, &img)) return NAN;
    ld s = 0.0L;
    for (int k = 0; k < img.n; k++) {
        const ld *R = img.v[k];
        ld r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
        if (r2 > 0.0L && r2 < rcut * rcut) {
            ld r = sqrtl(r2);
            s += erfcl(kappa * r) / r;
        }
    }
    list_free(&img);
    return s;
}

/* Constant of Eq. 3 / Eq. 4: pi/(Omega gamma) in 3D; 2 sqrt(pi)/(A kappa) in 2D (reading R2). */
static ld background_constant(const cell_t *c, ld kappa)
{
    if (c->dim == 3) return PI_L / (c->vol * kappa * kappa);
    return 2.0L * sqrtl(PI_L) / (c->vol * kappa);
}

static void load_point(int dim, const double *p, ld *out)
{
    out[0] = p[0]; out[1] = p[1]; out[2] = dim == 3 ? p[2] : 0.0L;
}

/* ------------------------------------------------------------------------------------------ */

int ewald_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int ewald_ref_num_g(int dim, const double *cell, double g_cutoff)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(g_cutoff > 0)) return -1;
    lattice_list_t g;
    if (g_list(&c, 0.0L, g_cutoff, &g)) return -1;
    int n = g.n;
    list_free(&g);
    return n;
}

int ewald_ref_gplus(int dim, const double *cell, double g_cutoff, int *n_out)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(g_cutoff > 0) || !n_out) return 1;
    lattice_list_t g;
    int rc = gplus_list(&c, 0.0L, g_cutoff, &g);
    if (rc) return rc;
    for (int k = 0; k < g.n; k++)
        for (int x = 0; x < 3; x++) n_out[3 * k + x] = g.idx[k][x];
    list_free(&g);
    return 0;
}

int ewald_ref_auto_cutoffs(int dim, const double *cell, double kappa, double tol, double *g_cutoff,
                           double *r_cutoff)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(tol > 0 && tol < 1)) return 1;
    /* exp(-G^2/4kappa^2) <= tol and erfc(kappa r) < exp(-kappa^2 r^2) <= tol */
    ld x = sqrtl(-logl((ld)tol));
    if (g_cutoff) *g_cutoff = (double)(2.0L * kappa * x);
    if (r_cutoff) *r_cutoff = (double)(x / kappa);
    return 0;
}

/* Eq. 3 literally: loop every G of the full sphere with cosl, every image with erfcl. */
static ld v_e_literal(const cell_t *c, const lattice_list_t *g, ld kappa, ld rcut, const ld *r)
{
    ld recip = 0.0L;
    for (int k = 0; k < g->n; k++) {
        ld gr = g->v[k][0] * r[0] + g->v[k][1] * r[1] + g->v[k][2] * r[2];
        recip += 2.0L * g->w[k] * cosl(gr); /* 2 w(G) = (4pi/Omega) exp(-G^2/4gamma)/G^2 in 3D */
    }
    lattice_list_t img;
    if (image_list(c, rcut, norm3(r), &img)) return NAN;
    ld real = psi_images(&img, kappa, rcut, r);
    list_free(&img);
    return recip + real - background_constant(c, kappa);
}

/* Eq. 4 literally. */
static ld v_m_literal(const cell_t *c, const lattice_list_t *g, ld kappa, ld rcut)
{
    ld recip = 0.0L;
    for (int k = 0; k < g->n; k++) recip += 2.0L * g->w[k];
    return recip + xi_real(c, kappa, rcut) - 2.0L * kappa / sqrtl(PI_L) - background_constant(c, kappa);
}

int ewald_ref_v_e(int dim, const double *cell, double kappa, double g_cutoff, double r_cutoff,
                  const double *r, double *v_e)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(g_cutoff > 0) || !(r_cutoff > 0) || !r || !v_e)
        return 1;
    lattice_list_t g;
    if (g_list(&c, kappa, g_cutoff, &g)) return 3;
    ld rr[3];
    load_point(dim, r, rr);
    *v_e = (double)v_e_literal(&c, &g, kappa, r_cutoff, rr);
    list_free(&g);
    return 0;
}

int ewald_ref_v_m(int dim, const double *cell, double kappa, double g_cutoff, double r_cutoff,
                  double *v_m)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(g_cutoff > 0) || !(r_cutoff > 0) || !v_m)
        return 1;
    lattice_list_t g;
    if (g_list(&c, kappa, g_cutoff, &g)) return 3;
    *v_m = (double)v_m_literal(&c, &g, kappa, r_cutoff);
    list_free(&g);
    return 0;
}

/* Eq. 2 literally. */
int ewald_ref_energy_pairwise(int dim, const double *cell, double kappa, double g_cutoff,
                              double r_cutoff, int n, const double *pos, const double *q,
                              double *energy)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(g_cutoff > 0) || !(r_cutoff > 0) || n < 1 ||
        !pos || !q || !energy)
        return 1;
    lattice_list_t g;
    if (g_list(&c, kappa, g_cutoff, &g)) return 3;
    ld e = 0.0L;
    for (int i = 0; i < n - 1; i++)
        for (int j = i + 1; j < n; j++) {
            ld ri[3], rj[3], r[3];
            load_point(dim, pos + (size_t)i * dim, ri);
            load_point(dim, pos + (size_t)j * dim, rj);
            for (int x = 0; x < 3; x++) r[x] = ri[x] - rj[x];
            e += (ld)q[i] * (ld)q[j] * v_e_literal(&c, &g, kappa, r_cutoff, r);
        }
    ld vm = v_m_literal(&c, &g, kappa, r_cutoff);
    for (int j = 0; j < n; j++) e += 0.5L * (ld)q[j] * (ld)q[j] * vm;
    *energy = (double)e;
    list_free(&g);
    return 0;
}

/* rho(G) on a G list for one set of charges: direct sincosl of the Cartesian G.r. */
static void rho_direct(const lattice_list_t *g, int n, const ld (*r)[3], const ld *q, ld *re, ld *im)
{
    for (int k = 0; k < g->n; k++) {
        ld sr = 0.0L, si = 0.0L;
        for (int i = 0; i < n; i++) {
            ld s, co;
            sincosl(g->v[k][0] * r[i][0] + g->v[k][1] * r[i][1] + g->v[k][2] * r[i][2], &s, &co);
            sr += q[i] * co;
            si += q[i] * s;
        }
        re[k] = sr;
        im[k] = si;
    }
}

int ewald_ref_rho(int dim, const double *cell, double g_cutoff, int n, const double *pos,
                  const double *q, double *re_im)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(g_cutoff > 0) || n < 1 || !pos || !q || !re_im) return 1;
    lattice_list_t g;
    if (gplus_list(&c, 0.0L, g_cutoff, &g)) return 3;
    ld(*r)[3] = malloc((size_t)n * sizeof *r);
    ld *qq = malloc((size_t)n * sizeof *qq);
    ld *re = malloc((size_t)(g.n + 1) * sizeof *re), *im = malloc((size_t)(g.n + 1) * sizeof *im);
    for (int i = 0; i < n; i++) { load_point(dim, pos + (size_t)i * dim, r[i]); qq[i] = q[i]; }
    rho_direct(&g, n, (const ld(*)[3])r, qq, re, im);
    for (int k = 0; k < g.n; k++) { re_im[2 * k] = (double)re[k]; re_im[2 * k + 1] = (double)im[k]; }
    free(r); free(qq); free(re); free(im);
    list_free(&g);
    return 0;
}

/* Gather mobile particles of one walker plus the fixed ions into one charge set. */
static void gather_charges(int dim, int n, const double *pos, const double *q, int n_ion,
                           const double *ion_pos, const double *ion_q, ld (*r)[3], ld *qq)
{
    for (int i = 0; i < n; i++) { load_point(dim, pos + (size_t)i * dim, r[i]); qq[i] = q[i]; }
    for (int i = 0; i < n_ion; i++) {
        load_point(dim, ion_pos + (size_t)i * dim, r[n + i]);
        qq[n + i] = ion_q[i];
    }
}

int ewald_ref_energy_batch(int dim, const double *cell, double kappa, double g_cutoff,
                           double r_cutoff, int n_walkers, int n, const double *pos,
                           const double *q, int n_ion, const double *ion_pos, const double *ion_q,
                           double *energies, double *components, int n_threads)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(g_cutoff > 0) || !(r_cutoff > 0) ||
        n_walkers < 0 || n < 0 || n_ion < 0 || n + n_ion < 1 || (n > 0 && (!pos || !q)) ||
        (n_ion > 0 && (!ion_pos || !ion_q)) || !energies)
        return 1;
    lattice_list_t g, img;
    if (gplus_list(&c, kappa, g_cutoff, &g)) return 3;
    if (image_list(&c, r_cutoff, c.reach, &img)) return 3;
    const ld xi = xi_real(&c, kappa, r_cutoff);
    const ld bgc = background_constant(&c, kappa);
    const int nt = n + n_ion;
    int err = 0;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int w = 0; w < n_walkers; w++) {
        ld(*r)[3] = malloc((size_t)nt * sizeof *r);
        ld *qq = malloc((size_t)nt * sizeof *qq);
        ld *re = malloc((size_t)(g.n + 1) * sizeof *re), *im = malloc((size_t)(g.n + 1) * sizeof *im);
        if (!r || !qq || !re || !im) { err = 3; free(r); free(qq); free(re); free(im); continue; }
        gather_charges(dim, n, pos + (size_t)w * n * dim, q, n_ion, ion_pos, ion_q, r, qq);

        rho_direct(&g, nt, (const ld(*)[3])r, qq, re, im);
        ld e_recip = 0.0L; /* half set: w(G) = w(-G), |rho(G)| = |rho(-G)| */
        for (int k = 0; k < g.n; k++) e_recip += 2.0L * g.w[k] * (re[k] * re[k] + im[k] * im[k]);

        ld e_real = 0.0L, q2 = 0.0L, qtot = 0.0L;
        for (int i = 0; i < nt; i++) { q2 += qq[i] * qq[i]; qtot += qq[i]; }
        for (int i = 0; i < nt - 1; i++)
            for (int j = i + 1; j < nt; j++) {
                ld d[3] = { r[i][0] - r[j][0], r[i][1] - r[j][1], r[i][2] - r[j][2] };
                reduce_displacement(&c, d);
                e_real += qq[i] * qq[j] * psi_images(&img, kappa, r_cutoff, d);
            }
        e_real += 0.5L * q2 * xi;
        ld e_self = -kappa / sqrtl(PI_L) * q2;
        ld e_bg = -0.5L * bgc * qtot * qtot;

        energies[w] = (double)(e_recip + e_real + e_self + e_bg);
        if (components) {
            components[4 * w + 0] = (double)e_recip;
            components[4 * w + 1] = (double)e_real;
            components[4 * w + 2] = (double)e_self;
            components[4 * w + 3] = (double)e_bg;
        }
        free(r); free(qq); free(re); free(im);
    }
    list_free(&g);
    list_free(&img);
    return err;
}

int ewald_ref_move_chain(int dim, const double *cell, double kappa, double g_cutoff,
                         double r_cutoff, int n_walkers, int n, double *pos, const double *q,
                         int n_ion, const double *ion_pos, const double *ion_q, int n_steps,
                         const int *electron, const double *new_r, double *delta_e,
                         double *rho_out, int n_threads)
{
    cell_t c;
    if (cell_init(&c, dim, cell) || !(kappa > 0) || !(g_cutoff > 0) || !(r_cutoff > 0) ||
        n_walkers < 0 || n < 1 || n_ion < 0 || !pos || !q || (n_ion > 0 && (!ion_pos || !ion_q)) ||
        n_steps < 0 || (n_steps > 0 && (!electron || !new_r || !delta_e)))
        return 1;
    for (long t = 0; t < (long)n_steps * n_walkers; t++)
        if (electron[t] < 0 || electron[t] >= n) return 4;
    lattice_list_t g, img;
    if (gplus_list(&c, kappa, g_cutoff, &g)) return 3;
    if (image_list(&c, r_cutoff, c.reach, &img)) return 3;
    const int nt = n + n_ion;
    int err = 0;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int w = 0; w < n_walkers; w++) {
        ld(*r)[3] = malloc((size_t)nt * sizeof *r);
        ld *qq = malloc((size_t)nt * sizeof *qq);
        ld *re = malloc((size_t)(g.n + 1) * sizeof *re), *im = malloc((size_t)(g.n + 1) * sizeof *im);
        if (!r || !qq || !re || !im) { err = 3; free(r); free(qq); free(re); free(im); continue; }
        double *pw = pos + (size_t)w * n * dim;
        gather_charges(dim, n, pw, q, n_ion, ion_pos, ion_q, r, qq);
        rho_direct(&g, nt, (const ld(*)[3])r, qq, re, im); /* the stored rho(G) of this walker */

        for (int s = 0; s < n_steps; s++) {
            const size_t t = (size_t)s * n_walkers + w;
            const int k = electron[t];
            ld rn[3];
            load_point(dim, new_r + t * dim, rn);
            const ld qk = qq[k];
            /* reciprocal part: delta(G) = exp(iG.r') - exp(iG.r_k);
             * dE = sum_{G+} 2 w(G) [ 2 q_k Re(conj(rho) delta) + q_k^2 |delta|^2 ]; rho += q_k delta */
            ld de_recip = 0.0L;
            for (int m = 0; m < g.n; m++) {
                ld sn, cn, so, co;
                sincosl(g.v[m][0] * rn[0] + g.v[m][1] * rn[1] + g.v[m][2] * rn[2], &sn, &cn);
                sincosl(g.v[m][0] * r[k][0] + g.v[m][1] * r[k][1] + g.v[m][2] * r[k][2], &so, &co);
                ld dr = cn - co, di = sn - so;
                de_recip += 2.0L * g.w[m] *
                            (2.0L * qk * (re[m] * dr + im[m] * di) + qk * qk * (dr * dr + di * di));
                re[m] += qk * dr;
                im[m] += qk * di;
            }
            /* real part: q_k sum_{j != k} q_j [ psi(r' - r_j) - psi(r_k - r_j) ] */
            ld de_real = 0.0L;
            for (int j = 0; j < nt; j++) {
                if (j == k) continue;
                ld dnew[3] = { rn[0] - r[j][0], rn[1] - r[j][1], rn[2] - r[j][2] };
                ld dold[3] = { r[k][0] - r[j][0], r[k][1] - r[j][1], r[k][2] - r[j][2] };
                reduce_displacement(&c, dnew);
                reduce_displacement(&c, dold);
                de_real += qq[j] * (psi_images(&img, kappa, r_cutoff, dnew) -
                                    psi_images(&img, kappa, r_cutoff, dold));
            }
            de_real *= qk;
            delta_e[t] = (double)(de_recip + de_real);
            for (int x = 0; x < 3; x++) r[k][x] = rn[x];
            for (int x = 0; x < dim; x++) pw[(size_t)k * dim + x] = new_r[t * dim + x];
        }
        if (rho_out)
            for (int m = 0; m < g.n; m++) {
                rho_out[((size_t)w * g.n + m) * 2 + 0] = (double)re[m];
                rho_out[((size_t)w * g.n + m) * 2 + 1] = (double)im[m];
            }
        free(r); free(qq); free(re); free(im);
    }
    list_free(&g);
    list_free(&img);
    return err;
}
