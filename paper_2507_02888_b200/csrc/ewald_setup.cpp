/* ewald_setup.cpp -- host-side table construction for the B200 Ewald library.
 *
 * Everything walker-independent in Eqs. 2-4 is evaluated here once, in
 * long double, and handed to the device rounded to FP64 / FP32 (the Ewald lookup
 * tables are "numerically sensitive and are always performed using DP"; "much of the
 * data required can be moved to the GPU once, at the outset").
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>

#include "ewald_internal.h"

namespace ewald {

typedef long double real;
static const real kPi = 3.141592653589793238462643383279502884L;

static real dot3(const real *x, const real *y) { return x[0] * y[0] + x[1] * y[1] + x[2] * y[2]; }
static real len3(const real *x) { return sqrtl(dot3(x, x)); }

/* w(G): E_recip = sum over the full sphere of w(G) |rho(G)|^2.
 * 3D: Eq. 3's (4pi/Omega) exp(-G^2/4gamma)/G^2 summed over ordered pairs -> 2pi/Omega.
 * 2D (reading R2): (pi/A) erfc(G/2kappa)/G. */
static real weight(int dim, real volume, real kappa, real g2)
{
    if (dim == 3) return 2 * kPi / volume * expl(-g2 / (4 * kappa * kappa)) / g2;
    real g = sqrtl(g2);
    return kPi / volume * erfcl(g / (2 * kappa)) / g;
}

/* Pair-function table of the real-space kernels (ewald_realspace.cuh):
 *     F(t) = erfc(sqrt t)/sqrt t,  t = kappa^2 r^2,
 * so that a term of the real-lattice sum of Eq. 3 is kappa q_i q_j F(t) -- no square
 * root on the device.  Bins are cut from the floating-point format of t itself: bin number
 * (e - e_min) 2^K + (top K mantissa bits), e the binary exponent; the same bins serve FP64 (index from
 * the high word) and FP32.  On a bin [t_lo, t_lo + D), D = 2^(e-K), F is replaced by the polynomial
 * through the Chebyshev nodes, expressed in the centred variable u = t - (t_lo + D/2) (t_lo + D/2 is
 * t with its low mantissa bits replaced by 100..0: one logic operation).  Long double throughout
 * ("lookup tables ... always performed using DP arithmetic").  Layout [bin][degree+1]. */
void build_pair_table(int kbits, int degree, int e_min, double t_max, PairTable *out)
{
    out->kbits = kbits; out->degree = degree; out->e_min = e_min;
    out->t_min = std::ldexp(1.0, e_min);
    const int n = degree + 1, per = 1 << kbits;
    int e_top; std::frexp(t_max, &e_top); e_top -= 1;          /* t_max in [2^e_top, 2^(e_top+1)) */
    if (e_top < e_min) e_top = e_min;
    const real frac = (real)t_max / ldexpl(1.0L, e_top) - 1;   /* in [0,1) */
    int last = (int)floorl(frac * per);
    if (last > per - 1) last = per - 1;
    out->n_bins = (e_top - e_min) * per + last + 1;
    out->t_max = (double)(ldexpl(1.0L, e_top) * (1 + (real)(last + 1) / per));
    out->coef.assign((size_t)out->n_bins * n, 0.0);
    std::vector<real> fv(n), cheb(n), mono(n), t0(n), t1(n), t2(n);
    for (int b = 0; b < out->n_bins; b++) {
        const int e = e_min + b / per, m = b % per;
        const real width = ldexpl(1.0L, e - kbits), half = width / 2;
        const real mid = ldexpl(1.0L, e) + m * width + half;
        for (int i = 0; i < n; i++) {
            const real t = mid + half * cosl(kPi * (2 * i + 1) / (2 * n)), z = sqrtl(t);
            fv[i] = erfcl(z) / z;
        }
        for (int k = 0; k < n; k++) {
            real s = 0;
            for (int i = 0; i < n; i++) s += fv[i] * cosl(k * kPi * (2 * i + 1) / (2 * n));
            cheb[k] = (k == 0 ? 1 : 2) * s / n;
        }
        for (int i = 0; i < n; i++) { mono[i] = 0; t0[i] = 0; t1[i] = 0; }
        t0[0] = 1;
        if (n > 1) t1[1] = 1;
        for (int i = 0; i < n; i++) mono[i] += cheb[0] * t0[i];
        if (n > 1) for (int i = 0; i < n; i++) mono[i] += cheb[1] * t1[i];
        for (int k = 2; k < n; k++) {
            for (int i = 0; i < n; i++) t2[i] = (i > 0 ? 2 * t1[i - 1] : 0) - t0[i];
            for (int i = 0; i < n; i++) mono[i] += cheb[k] * t2[i];
            t0 = t1; t1 = t2;
        }
        real scale = 1; /* v = u / half */
        for (int k = 0; k < n; k++) { out->coef[(size_t)b * n + k] = (double)(mono[k] * scale); scale /= half; }
    }
}

/* Far-shell table of the FP64 kernels (ewald_realspace.cuh, FarStack): F(t) for t >= t0 on bins of width
 * 2^-kb, cubic in u = (position inside the bin) - 1/2, FP32 coefficients, `rep` copies interleaved as
 * [bin][copy][4] (each copy is one 16-byte column: conflict-free LDS.128). */
void build_far_table(int t0, int kb, int rep, double t_max, std::vector<float> *tab, int *n_far)
{
    tab->clear();
    *n_far = 0;
    if (!(t_max > t0)) return;
    const int nb = (int)floorl(((real)t_max - t0) * (1 << kb)) + 1;
    const int n = 4;
    tab->assign((size_t)nb * rep * 4, 0.0f);
    for (int b = 0; b < nb; b++) {
        const real width = ldexpl(1.0L, -kb), mid = t0 + (b + 0.5L) * width;
        real fv[4], cheb[4];
        for (int i = 0; i < n; i++) {
            const real t = mid + 0.5L * width * cosl(kPi * (2 * i + 1) / (2 * n)), z = sqrtl(t);
            fv[i] = erfcl(z) / z;
        }
        for (int k = 0; k < n; k++) {
            real s = 0;
            for (int i = 0; i < n; i++) s += fv[i] * cosl(k * kPi * (2 * i + 1) / (2 * n));
            cheb[k] = (k == 0 ? 1 : 2) * s / n;
        }
        /* T0 = 1, T1 = v, T2 = 2v^2 - 1, T3 = 4v^3 - 3v; v = 2u */
        const real m0 = cheb[0] - cheb[2], m1 = cheb[1] - 3 * cheb[3], m2 = 2 * cheb[2], m3 = 4 * cheb[3];
        float c[4] = {(float)m0, (float)(2 * m1), (float)(4 * m2), (float)(8 * m3)};
        /* The same rounded coefficients serve every term that falls in the bin, so the rounding of c0 to float
         * (3e-8 relative) and the mean of the cubic's truncation error are SYSTEMATIC over a walker's ~1e5 far
         * terms.  The u^2 coefficient is re-chosen so that the mean of the float polynomial over the bin,
         * c0 + c2/12, equals the mean of F over the bin (composite Simpson, long double): the error of a term
         * stays <= ~1e-7 F pointwise but averages to zero for terms spread over the bin. */
        {
            const int ns = 64;
            real acc = 0;
            for (int i = 0; i <= ns; i++) {
                const real t = mid + width * ((real)i / ns - 0.5L), z = sqrtl(t);
                acc += (i == 0 || i == ns ? 1 : (i & 1) ? 4 : 2) * erfcl(z) / z;
            }
            const real mean_f = acc / (3 * ns);
            c[2] = (float)(12 * (mean_f - (real)c[0]));
        }
        for (int r = 0; r < rep; r++)
            for (int k = 0; k < 4; k++) (*tab)[((size_t)b * rep + r) * 4 + k] = c[k];
    }
    *n_far = nb;
}

/* Host evaluation of the table exactly as the kernels index it (FP64 format). */
double eval_pair_table(const PairTable &p, double t)
{
    uint64_t bits; std::memcpy(&bits, &t, 8);
    const int hi = (int)(bits >> 32), sh = 20 - p.kbits;
    int idx = (hi >> sh) - ((1023 + p.e_min) << p.kbits);
    if (idx < 0 || idx >= p.n_bins) { const long double z = sqrtl((long double)t); return (double)(erfcl(z) / z); }
    const uint64_t mid_hi = ((uint64_t)(uint32_t)hi & ~((1ull << sh) - 1)) | (1ull << (sh - 1));
    const uint64_t mb = mid_hi << 32;
    double mid; std::memcpy(&mid, &mb, 8);
    const double u = t - mid;
    const double *c = &p.coef[(size_t)idx * (p.degree + 1)];
    double v = c[p.degree];
    for (int k = p.degree - 1; k >= 0; k--) v = std::fma(v, u, c[k]);
    return v;
}

ewald_status build_tables(int dim, const double *cell, double kappa_d, double g_cutoff,
                          double r_cutoff, HostTables *t, std::string *err)
{
    if (dim != 2 && dim != 3) { *err = "dim must be 2 or 3"; return EWALD_EINVAL; }
    if (!cell) { *err = "cell is null"; return EWALD_EINVAL; }
    if (!(kappa_d > 0) || !std::isfinite(kappa_d)) { *err = "gamma (kappa) must be > 0"; return EWALD_ERANGE; }
    if (!(g_cutoff > 0) || !std::isfinite(g_cutoff)) { *err = "g_cutoff must be > 0"; return EWALD_ERANGE; }
    if (r_cutoff < 0 || !std::isfinite(r_cutoff)) { *err = "r_cutoff must be >= 0"; return EWALD_ERANGE; }
    for (int i = 0; i < 9; i++)
        if (!std::isfinite(cell[i])) { *err = "cell has a non-finite entry"; return EWALD_EINVAL; }

    real a[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 1}};
    for (int i = 0; i < dim; i++)
        for (int j = 0; j < dim; j++) a[i][j] = cell[3 * i + j];

    /* reciprocal rows b_k with a_i . b_k = 2pi delta_ik, via cross products */
    real c[3][3];
    for (int k = 0; k < 3; k++) {
        const real *u = a[(k + 1) % 3], *v = a[(k + 2) % 3];
        c[k][0] = u[1] * v[2] - u[2] * v[1];
        c[k][1] = u[2] * v[0] - u[0] * v[2];
        c[k][2] = u[0] * v[1] - u[1] * v[0];
    }
    real det = dot3(a[0], c[0]);
    real scale = len3(a[0]) * len3(a[1]) * len3(a[2]);
    if (!(fabsl(det) > 1e-14L * scale) || !std::isfinite((double)det)) {
        *err = "cell is singular";
        return EWALD_ESINGULAR;
    }
    real b[3][3];
    for (int k = 0; k < 3; k++)
        for (int x = 0; x < 3; x++) b[k][x] = 2 * kPi * c[k][x] / det;

    const real kappa = kappa_d;
    t->dim = dim;
    t->kappa = kappa_d;
    t->g_cutoff = g_cutoff;
    t->volume = (double)fabsl(det);
    if (r_cutoff == 0) r_cutoff = (double)(sqrtl(-logl(1e-17L)) / kappa);
    /* erfc(6.5) = 4e-20: beyond kappa r = 6.5 no term can matter at FP64; bounds the pair table's range */
    if (r_cutoff * kappa_d > 6.5) r_cutoff = 6.5 / kappa_d;
    t->r_cutoff = r_cutoff;
    /* the cull compares high words / FP32 values: cover a little beyond kappa^2 r_c^2 */
    const double t_top = r_cutoff * r_cutoff * kappa_d * kappa_d * (1 + 1e-5);
    build_pair_table(PAIR_K64, PAIR_DEG64, PAIR_EMIN, t_top, &t->pair64);
    build_pair_table(PAIR_K32, PAIR_DEG32, PAIR_EMIN, t_top, &t->pair32);
    build_far_table(FAR_T0, FAR_KB, FAR_REP, t_top, &t->far_tab, &t->n_far);
    bool ortho = true;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            t->a[3 * i + j] = (double)a[i][j];
            t->binv[3 * i + j] = (double)(b[i][j] / (2 * kPi));
            if (i != j && a[i][j] != 0) ortho = false;
        }
    t->orthogonal = ortho;
    t->m_shift = 0;
    for (int k = 0; k < dim; k++) {
        /* image m of axis k is needed iff (|m| - 1/2) L_k < r_c */
        int m = (int)floorl((real)r_cutoff / len3(a[k]) + 0.5L - 1e-12L);
        if (m > t->m_shift) t->m_shift = m;
    }

    /* ---- half set G+ (first non-zero integer component positive), lexicographic ---- */
    const real g2max = (real)g_cutoff * g_cutoff * (1 + 1e-12L); /* reading R6 */
    int lim[3];
    for (int k = 0; k < 3; k++) {
        /* n_k = G . a_k / 2pi  =>  |n_k| <= |G| |a_k| / 2pi */
        lim[k] = k < dim ? (int)floorl(sqrtl(g2max) * len3(a[k]) / (2 * kPi) + 1e-9L) : 0;
        if (lim[k] > 1023) { *err = "G index range exceeds 1023"; return EWALD_ERANGE; }
    }
    t->g_n.clear();
    t->g_w2.clear();
    t->n_max[0] = t->n_max[1] = t->n_max[2] = 0;
    for (int n1 = 0; n1 <= lim[0]; n1++)
        for (int n2 = -lim[1]; n2 <= lim[1]; n2++)
            for (int n3 = -lim[2]; n3 <= lim[2]; n3++) {
                bool plus = n1 > 0 || (n1 == 0 && (n2 > 0 || (n2 == 0 && n3 > 0)));
                if (!plus) continue;
                real g[3];
                for (int x = 0; x < 3; x++) g[x] = n1 * b[0][x] + n2 * b[1][x] + n3 * b[2][x];
                real g2 = dot3(g, g);
                if (g2 > g2max) continue;
                t->g_n.push_back(n1); t->g_n.push_back(n2); t->g_n.push_back(n3);
                t->g_w2.push_back((double)(2 * weight(dim, fabsl(det), kappa, g2)));
                if (n1 > t->n_max[0]) t->n_max[0] = n1;
                if (abs(n2) > t->n_max[1]) t->n_max[1] = abs(n2);
                if (abs(n3) > t->n_max[2]) t->n_max[2] = abs(n3);
            }
    if (t->g_w2.empty()) { *err = "g_cutoff admits no reciprocal vector"; return EWALD_ERANGE; }

    /* ---- lattice images that can come within r_cutoff of a reduced displacement ----
     * A displacement reduced to fractional coordinates |s_k| <= 1/2 lies in the parallelepiped P.
     * Image R = m.a is needed iff dist(R, P) < r_cutoff.  Lower bounds on that distance:
     *   planes: (|m_k| - 1/2) h_k with h_k = 2pi/|b_k| (spacing of the a-planes normal to b_k);
     *   orthogonal cells: root-sum-square of the plane bounds;  any cell: |R| - reach.          */
    const real rc = r_cutoff;
    real reach = 0, h[3];
    for (int k = 0; k < dim; k++) reach += len3(a[k]) / 2;
    for (int k = 0; k < 3; k++) h[k] = 2 * kPi / len3(b[k]);
    int mlim[3];
    for (int k = 0; k < 3; k++) mlim[k] = k < dim ? (int)floorl(rc / h[k] + 0.5L + 1e-9L) : 0;
    t->img.clear();
    t->img_m.clear();
    real xi = 0;
    for (int m1 = -mlim[0]; m1 <= mlim[0]; m1++)
        for (int m2 = -mlim[1]; m2 <= mlim[1]; m2++)
            for (int m3 = -mlim[2]; m3 <= mlim[2]; m3++) {
                int m[3] = {m1, m2, m3};
                real R[3];
                for (int x = 0; x < 3; x++) R[x] = m1 * a[0][x] + m2 * a[1][x] + m3 * a[2][x];
                real rl = len3(R);
                if ((m1 || m2 || m3) && rl < rc) xi += erfcl(kappa * rl) / rl; /* Eq. 4 real sum */
                real lb_max = 0, lb_ss = 0;
                for (int k = 0; k < dim; k++) {
                    real d = (fabsl((real)m[k]) - 0.5L) * h[k];
                    if (d < 0) d = 0;
                    if (d > lb_max) lb_max = d;
                    lb_ss += d * d;
                }
                real lb = ortho ? sqrtl(lb_ss) : lb_max;
                if (rl - reach > lb) lb = rl - reach;
                if (lb >= rc * (1 + 1e-12L)) continue;
                for (int x = 0; x < 3; x++) { t->img.push_back((double)R[x]); t->img_m.push_back(m[x]); }
            }
    t->xi_r = (double)xi;
    t->self_coef = (double)(kappa / sqrtl(kPi));
    real bgc = dim == 3 ? kPi / (fabsl(det) * kappa * kappa) : 2 * sqrtl(kPi) / (fabsl(det) * kappa);
    t->bg_coef = (double)bgc;
    real wsum = 0; /* sum over the full sphere of 2 w(G) = the reciprocal sum of Eq. 4 */
    for (size_t k = 0; k < t->g_w2.size(); k++) wsum += 2 * (real)t->g_w2[k];
    t->v_m = (double)(wsum + xi - 2 * kappa / sqrtl(kPi) - bgc);

    t->n_ion = 0;
    t->ion_pos.clear(); t->ion_q.clear(); t->ion_rho.clear();
    t->ion_q2 = t->ion_qsum = t->ion_real = 0;
    t->ion_uniform = true;
    t->sp_start.assign(1, 0);
    build_oct_plan(t);
    return EWALD_OK;
}

ewald_status build_fixed_charges(HostTables *t, int n_ion, const double *pos, const double *q,
                                 std::string *err)
{
    if (n_ion < 0 || (n_ion > 0 && (!pos || !q))) { *err = "bad fixed-charge arguments"; return EWALD_EINVAL; }
    const int dim = t->dim;
    const size_t ngp = t->g_w2.size();
    /* validate everything before touching the tables: a failed call leaves the previous ions in place */
    for (int i = 0; i < n_ion; i++) {
        if (!std::isfinite(q[i])) { *err = "non-finite ion charge"; return EWALD_EINVAL; }
        for (int x = 0; x < dim; x++)
            if (!std::isfinite(pos[(size_t)i * dim + x])) { *err = "non-finite ion position"; return EWALD_EINVAL; }
    }
    t->n_ion = n_ion;
    t->ion_pos.assign((size_t)3 * n_ion, 0.0);
    t->ion_q.assign((size_t)n_ion, 0.0);
    t->ion_rho.assign(2 * ngp, 0.0);
    /* the fixed charges are kept grouped by charge value ("species"; stable order inside a group): the
     * real-space kernels then treat every species as one segment with a single charge product */
    std::vector<int> order(n_ion);
    for (int i = 0; i < n_ion; i++) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return q[x] < q[y]; });
    t->sp_start.clear();
    for (int k = 0; k < n_ion; k++) {
        const int i = order[k];
        t->ion_q[k] = q[i];
        if (k == 0 || q[i] != q[order[k - 1]]) t->sp_start.push_back(k);
        for (int x = 0; x < dim; x++) t->ion_pos[3 * k + x] = pos[(size_t)i * dim + x];
    }
    t->sp_start.push_back(n_ion);
    q = t->ion_q.data(); /* from here on: the grouped order */
    real q2 = 0, qs = 0;
    for (int i = 0; i < n_ion; i++) { q2 += (real)q[i] * q[i]; qs += q[i]; }
    t->ion_q2 = (double)q2;
    t->ion_qsum = (double)qs;
    /* up to MAX_SPECIES species: the real-space kernels keep bare t on their stacks */
    t->ion_uniform = (int)t->sp_start.size() - 1 <= MAX_SPECIES;

    /* rho_ion(G) = sum_I q_I exp(2 pi i n.s_I) with s = fractional coordinates */
    std::vector<real> s((size_t)3 * n_ion);
    for (int i = 0; i < n_ion; i++)
        for (int k = 0; k < 3; k++) {
            real v = 0;
            for (int x = 0; x < 3; x++) v += (real)t->ion_pos[3 * i + x] * (real)t->binv[3 * k + x];
            s[3 * i + k] = v - nearbyintl(v);
        }
    for (size_t g = 0; g < ngp; g++) {
        real re = 0, im = 0;
        for (int i = 0; i < n_ion; i++) {
            real ph = 0;
            for (int k = 0; k < 3; k++) ph += t->g_n[3 * g + k] * s[3 * i + k];
            ph -= nearbyintl(ph);
            re += q[i] * cosl(2 * kPi * ph);
            im += q[i] * sinl(2 * kPi * ph);
        }
        t->ion_rho[2 * g] = (double)re;
        t->ion_rho[2 * g + 1] = (double)im;
    }

    /* sum_{I<J} q_I q_J psi(r_I - r_J): the real-space part of Eq. 3 between fixed charges */
    const real rc2 = (real)t->r_cutoff * t->r_cutoff, kappa = t->kappa;
    const size_t nimg = t->img.size() / 3;
    real e = 0;
    for (int i = 0; i < n_ion; i++)
        for (int j = i + 1; j < n_ion; j++) {
            real d[3], f[3];
            for (int x = 0; x < 3; x++) d[x] = (real)t->ion_pos[3 * i + x] - (real)t->ion_pos[3 * j + x];
            for (int k = 0; k < 3; k++) {
                f[k] = 0;
                for (int x = 0; x < 3; x++) f[k] += d[x] * (real)t->binv[3 * k + x];
                f[k] = k < dim ? nearbyintl(f[k]) : 0;
            }
            for (int x = 0; x < 3; x++)
                d[x] -= f[0] * t->a[x] + f[1] * t->a[3 + x] + f[2] * t->a[6 + x];
            real psi = 0;
            for (size_t m = 0; m < nimg; m++) {
                real x = d[0] - t->img[3 * m], y = d[1] - t->img[3 * m + 1], z = d[2] - t->img[3 * m + 2];
                real r2 = x * x + y * y + z * z;
                if (r2 < rc2) { real r = sqrtl(r2); psi += erfcl(kappa * r) / r; }
            }
            e += (real)q[i] * q[j] * psi;
        }
    t->ion_real = (double)e;
    fill_oct_ion(t);
    fill_mma_ion(t);
    return EWALD_OK;
}

} // namespace ewald
