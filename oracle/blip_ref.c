/*
 * blip_ref.c -- CPU ORACLE for orbitals in a blip (cubic B-spline) basis.  TEST INFRASTRUCTURE ONLY.
 *
 * /root/reference/PAPER.md section 2.4 (lines 161-165): orbitals re-represented
 * "in a localized blip (B-spline) basis set"; evaluating them at a particle position is "looking up the particle's
 * position in the spline grid followed by the evaluation of a small number of cubic polynomials defining the blip
 * basis functions, followed by multiplication of the blip functions by coefficients for each orbital" -- in CASINO
 * many 64-element ddot / dgemv calls.  The paper prints no formula; the basis is the standard
 * blip function of the cited blip papers (refs. [30, 31]):
 *     Theta(x) = 1 - 3/2 x^2 + 3/4 |x|^3  (|x| <= 1),   1/4 (2 - |x|)^3  (1 <= |x| <= 2),   0 otherwise,
 *     psi_o(r) = sum_{ijk} c_o[i][j][k] Theta(u1 - i) Theta(u2 - j) Theta(u3 - k),   u_k = N_k s_k(r),
 * s = fractional coordinates, the grid N1 x N2 x N3 periodic with the cell (reading R21).
 * This oracle is the definition written out: EVERY grid point is visited for every position (the nearest
 * periodic image of u_k - i), no neighbourhood lookup; gradient and Laplacian by the chain rule with Theta',
 * Theta''.  Long double sums.  Shares nothing with the CUDA path.  Pins: tests/test_blip_pins.py.
 *
 * Layouts (HOST): cell[9] row-major lattice rows; coef [n_orb][N1][N2][N3]; points [n_points][3];
 * psi [n_points][n_orb]; grad [n_points][3][n_orb] (nullable); lap [n_points][n_orb] (nullable).  Return 0 = ok.
 */
#include <math.h>
#include <stddef.h>

typedef long double real;

static void theta(real x, real *f, real *d1, real *d2)
{
    const real ax = fabsl(x), sg = x < 0 ? -1 : 1;
    if (ax <= 1) { *f = 1 - 1.5L * x * x + 0.75L * ax * ax * ax; *d1 = -3 * x + 2.25L * sg * ax * ax; *d2 = -3 + 4.5L * ax; }
    else if (ax < 2) { const real t = 2 - ax; *f = 0.25L * t * t * t; *d1 = -0.75L * sg * t * t; *d2 = 1.5L * t; }
    else { *f = *d1 = *d2 = 0; }
}

int blip_ref_theta(double x, double *f, double *d1, double *d2)
{
    real a, b, c;
    theta(x, &a, &b, &c);
    *f = (double)a; *d1 = (double)b; *d2 = (double)c;
    return 0;
}

int blip_ref_eval(const double *cell, const int *grid, int n_orb, const double *coef, int n_points,
                  const double *points, double *psi, double *grad, double *lap)
{
    real a[3][3], binv[3][3];
    int i, j, k, x, p, o;
    for (i = 0; i < 3; i++) for (j = 0; j < 3; j++) a[i][j] = cell[3 * i + j];
    const real det = a[0][0] * (a[1][1] * a[2][2] - a[1][2] * a[2][1]) - a[0][1] * (a[1][0] * a[2][2] - a[1][2] * a[2][0]) +
                     a[0][2] * (a[1][0] * a[2][1] - a[1][1] * a[2][0]);
    if (det == 0 || grid[0] < 4 || grid[1] < 4 || grid[2] < 4 || n_orb <= 0) return 1;
    for (i = 0; i < 3; i++) { /* binv[k][x]: s_k = sum_x r_x binv[k][x] */
        const int i1 = (i + 1) % 3, i2 = (i + 2) % 3;
        binv[i][0] = (a[i1][1] * a[i2][2] - a[i1][2] * a[i2][1]) / det;
        binv[i][1] = (a[i1][2] * a[i2][0] - a[i1][0] * a[i2][2]) / det;
        binv[i][2] = (a[i1][0] * a[i2][1] - a[i1][1] * a[i2][0]) / det;
    }
    const int N1 = grid[0], N2 = grid[1], N3 = grid[2];
#pragma omp parallel for private(i, j, k, x, o) schedule(dynamic, 1)
    for (p = 0; p < n_points; p++) {
        real u[3], gm[3][3]; /* gm[k][x] = d u_k / d r_x */
        for (k = 0; k < 3; k++) {
            real s = 0;
            for (x = 0; x < 3; x++) { s += (real)points[3 * p + x] * binv[k][x]; gm[k][x] = grid[k] * binv[k][x]; }
            u[k] = grid[k] * (s - floorl(s));
        }
        for (o = 0; o < n_orb; o++) {
            const double *c = coef + (size_t)o * N1 * N2 * N3;
            real v = 0, g[3] = {0, 0, 0}, h[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
            for (i = 0; i < N1; i++) {
                real d0 = u[0] - i; d0 -= N1 * nearbyintl(d0 / N1);
                real f0, f0d, f0dd; theta(d0, &f0, &f0d, &f0dd);
                if (f0 == 0 && f0d == 0 && f0dd == 0) continue;
                for (j = 0; j < N2; j++) {
                    real d1 = u[1] - j; d1 -= N2 * nearbyintl(d1 / N2);
                    real f1, f1d, f1dd; theta(d1, &f1, &f1d, &f1dd);
                    if (f1 == 0 && f1d == 0 && f1dd == 0) continue;
                    for (k = 0; k < N3; k++) {
                        real d2 = u[2] - k; d2 -= N3 * nearbyintl(d2 / N3);
                        real f2, f2d, f2dd; theta(d2, &f2, &f2d, &f2dd);
                        const real cc = c[((size_t)i * N2 + j) * N3 + k];
                        v += cc * f0 * f1 * f2;
                        g[0] += cc * f0d * f1 * f2; g[1] += cc * f0 * f1d * f2; g[2] += cc * f0 * f1 * f2d;
                        h[0][0] += cc * f0dd * f1 * f2; h[1][1] += cc * f0 * f1dd * f2; h[2][2] += cc * f0 * f1 * f2dd;
                        h[0][1] += cc * f0d * f1d * f2; h[0][2] += cc * f0d * f1 * f2d; h[1][2] += cc * f0 * f1d * f2d;
                    }
                }
            }
            h[1][0] = h[0][1]; h[2][0] = h[0][2]; h[2][1] = h[1][2];
            psi[(size_t)p * n_orb + o] = (double)v;
            if (grad)
                for (x = 0; x < 3; x++)
                    grad[((size_t)p * 3 + x) * n_orb + o] = (double)(g[0] * gm[0][x] + g[1] * gm[1][x] + g[2] * gm[2][x]);
            if (lap) {
                real l = 0;
                int kk, ll;
                for (kk = 0; kk < 3; kk++) for (ll = 0; ll < 3; ll++) {
                    real m = 0;
                    for (x = 0; x < 3; x++) m += gm[kk][x] * gm[ll][x];
                    l += m * h[kk][ll];
                }
                lap[(size_t)p * n_orb + o] = (double)l;
            }
        }
    }
    return 0;
}
