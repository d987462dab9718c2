/* jastrow_kernels.cuh -- batched homogeneous two-body Jastrow terms u (Eq. 6) and p (Eq. 7), sm_100a.
 *
 * The paper's offload sums p(r_ij) over pairs with the buffered powers of Eq. 8: O(N^2 N_G)
 * per walker.  Here the pair sum is regrouped exactly, as for the Ewald reciprocal term:
 *     sum_{i<j} cos(G.r_ij) = (|S(G)|^2 - N) / 2,            S(G) = sum_i exp(iG.r_i)
 *     grad_i sum_{j != i} cos(G.r_ij) = -G Im[e_i(G) conj S(G)],   lap_i ... = -G^2 (Re[e_i(G) conj S(G)] - 1)
 * with e_i(G) = exp(iG.r_i) from the per-axis powers of Eq. 8: O(N N_G) per walker for value, gradient and
 * Laplacian.  The u term is a plain minimum-image pair loop (L_u < half the nearest lattice vector).
 *
 *   jastrow_kernel       one CTA per walker: [pass 1] power rows of a chunk of particles in shared memory, one
 *                        thread per (G, particle half) accumulates S(G); [pass 2] one thread per particle: its
 *                        power rows in registers, loop over G (S, a, G read as broadcasts) and over the partners j
 *                        for u; block sums in FP64
 *   jastrow_move_kernel  one CTA per move on the stored S(G) and positions
 */
#pragma once
#include "ewald_kernels_common.cuh"

namespace ewald {

constexpr int JAS_THREADS = 256;
constexpr int JAS_CHUNK = 64;     /* particles per chunk of power rows in pass 1 */
constexpr int JAS_MAXP = 8;       /* largest |n_k| + 1 of a G vector handled with register rows */
constexpr int JAS_MAXU = 16;      /* N_u + 1 */

struct JasTabs {
    int dim, n_g, mmax;           /* mmax = largest |n_k| */
    const short4 *gn;             /* [n_g] (n1, n2, n3, star) */
    const double *ga;             /* [n_g][4] = a_star G_x, a_star G_y, a_star G_z, a_star G^2 */
    const double *acoef;          /* [n_g] a_star */
    int n_u, c_exp;               /* n_u < 0: no u term */
    double alpha[JAS_MAXU];
    double l_u;
    double binv[9];               /* s_k = r . binv[k] */
    double a[9];                  /* lattice rows */
    int ortho;                    /* lattice rows along the Cartesian axes */
};

template <typename T> struct JasArgs {
    const T *pos;                 /* [W][DIM][npad] */
    int n, npad;
    JasTabs t;
    double *value, *grad, *lap;   /* [W], [W][DIM][npad], [W][npad] */
    T *s_out;                     /* [W][2][n_g_pad] stored S(G) or null (jastrow_load_walkers) */
    int n_g_pad;
};

/* exp(2 pi i s)^m, m = 0..mmax, in registers */
template <typename T>
__device__ __forceinline__ void jas_powers(double s, int mmax, typename Num<T>::T2 *row)
{
    typedef typename Num<T>::T2 T2;
    s -= rint(s);
    T sn, cs;
    Num<T>::sincospi_((T)(2 * s), &sn, &cs);
    T2 e; e.x = 1; e.y = 0;
    row[0] = e;
#pragma unroll
    for (int m = 1; m < JAS_MAXP; m++) {
        if (m > mmax) break;
        T2 f;
        f.x = e.x * cs - e.y * sn;
        f.y = e.x * sn + e.y * cs;
        e = f;
        row[m] = e;
    }
}

template <typename T2> __device__ __forceinline__ T2 jas_cmul(T2 a, T2 b)
{
    T2 r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
/* power n (any sign) from a row of non-negative powers */
template <typename T2> __device__ __forceinline__ T2 jas_pick(const T2 *row, int n)
{
    T2 e = row[n < 0 ? -n : n];
    if (n < 0) e.y = -e.y;
    return e;
}

__device__ __forceinline__ double jas_rsqrt(double x) { return rsqrt(x); }
__device__ __forceinline__ float jas_rsqrt(float x) { return rsqrtf(x); }

/* u(r), u'(r)/r and u''(r) of Eq. 6 for r < L_u, Horner in (poly, poly', poly''); inv_r = 1/r from the caller's
 * reciprocal square root (no division, no square root here; 0 where u'/r is not wanted or r = 0) */
template <typename T>
__device__ __forceinline__ void jas_u(const JasTabs &t, T r, T inv_r, T *u, T *du_over_r, T *d2u)
{
    T p = 0, dp = 0, d2p = 0;
    for (int l = t.n_u; l >= 0; l--) {
        d2p = d2p * r + 2 * dp;
        dp = dp * r + p;
        p = p * r + (T)t.alpha[l];
    }
    const T s = r - (T)t.l_u;
    T sc2 = 1;                                  /* (r - L_u)^(C - 2) */
    for (int k = 0; k < t.c_exp - 2; k++) sc2 *= s;
    const T c = (T)t.c_exp;
    const T sc1 = t.c_exp >= 2 ? sc2 * s : (t.c_exp == 1 ? T(1) : T(0));       /* (r - L_u)^(C - 1) */
    const T sc = t.c_exp >= 1 ? sc1 * s : T(1);                                 /* (r - L_u)^C */
    const T d1 = t.c_exp >= 1 ? c * sc1 : T(0), d2 = t.c_exp >= 2 ? c * (c - 1) * sc2 : T(0);
    *u = p * sc;
    const T du = dp * sc + p * d1;
    *du_over_r = du * inv_r;
    *d2u = d2p * sc + 2 * dp * d1 + p * d2;
}

/* minimum image of d (Cartesian) */
template <typename T, int DIM>
__device__ __forceinline__ void jas_min_image(const JasTabs &t, T (&d)[3])
{
    if (t.ortho) { /* diagonal cell: one rounding and one FMA per axis */
#pragma unroll
        for (int x = 0; x < DIM; x++) d[x] -= (T)t.a[4 * x] * Num<T>::rint_(d[x] * (T)t.binv[4 * x]);
        return;
    }
    T f[3] = {0, 0, 0};
#pragma unroll
    for (int k = 0; k < DIM; k++) {
        T s = 0;
#pragma unroll
        for (int x = 0; x < DIM; x++) s += d[x] * (T)t.binv[3 * k + x];
        f[k] = Num<T>::rint_(s);
    }
#pragma unroll
    for (int x = 0; x < DIM; x++)
#pragma unroll
        for (int k = 0; k < DIM; k++) d[x] -= f[k] * (T)t.a[3 * k + x];
    if (!t.ortho) { /* skewed cell: the nearest image may be a neighbour of the fractionally rounded one */
        T best[3] = {d[0], d[1], d[2]}, b2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        for (int m0 = -1; m0 <= 1; m0++)
            for (int m1 = -1; m1 <= 1; m1++)
                for (int m2 = (DIM == 3 ? -1 : 0); m2 <= (DIM == 3 ? 1 : 0); m2++) {
                    T v[3];
#pragma unroll
                    for (int x = 0; x < 3; x++) v[x] = d[x] - m0 * (T)t.a[x] - m1 * (T)t.a[3 + x] - m2 * (T)t.a[6 + x];
                    const T v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
                    if (v2 < b2) { b2 = v2; best[0] = v[0]; best[1] = v[1]; best[2] = v[2]; }
                }
        d[0] = best[0]; d[1] = best[1]; d[2] = best[2];
    }
}

template <typename T, int DIM>
__global__ void __launch_bounds__(JAS_THREADS) jastrow_kernel(JasArgs<T> A)
{
    typedef typename Num<T>::T2 T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const JasTabs &t = A.t;
    const int n = A.n, tid = threadIdx.x, w = blockIdx.x, np = t.mmax + 1;
    /* shared: positions [DIM][n] (T), S(G) [n_g] (T2), chunk rows [JAS_CHUNK][DIM][np] (T2) */
    T *sp = reinterpret_cast<T *>(smem_raw);
    T2 *sS = reinterpret_cast<T2 *>(sp + ((DIM * n + 3) & ~3));
    T2 *rows = sS + t.n_g;
    __shared__ double red[32];
    const T *pw = A.pos + (size_t)w * DIM * A.npad;
    for (int i = tid; i < n; i += JAS_THREADS)
#pragma unroll
        for (int x = 0; x < DIM; x++) sp[x * n + i] = pw[x * A.npad + i];
    __syncthreads();

    double value = 0;
    if (t.n_g > 0) {
        /* [pass 1] S(G): thread (g, half) sums the particles of its half of every chunk */
        const int g = tid % t.n_g, half = tid / t.n_g, halves = JAS_THREADS / t.n_g < 1 ? 1 : JAS_THREADS / t.n_g;
        T2 acc; acc.x = 0; acc.y = 0;
        for (int base = 0; base < n; base += JAS_CHUNK) {
            const int cnt = min(JAS_CHUNK, n - base);
            for (int task = tid; task < cnt * DIM; task += JAS_THREADS) {
                const int p = task / DIM, k = task - p * DIM;
                double s = 0;
#pragma unroll
                for (int x = 0; x < DIM; x++) s += (double)sp[x * n + base + p] * t.binv[3 * k + x];
                T2 row[JAS_MAXP];
                jas_powers<T>(s, t.mmax, row);
                for (int m = 0; m < np; m++) rows[(p * DIM + k) * np + m] = row[m];
            }
            __syncthreads();
            if (half < halves) { /* n_g <= JAS_THREADS (checked at setup): one G per thread */
                const short4 nn = t.gn[g];
                for (int p = half; p < cnt; p += halves) {
                    const T2 *r = rows + p * DIM * np;
                    T2 e = jas_cmul(jas_pick(r, nn.x), jas_pick(r + np, nn.y));
                    if (DIM == 3) e = jas_cmul(e, jas_pick(r + 2 * np, nn.z));
                    acc.x += e.x; acc.y += e.y;
                }
            }
            __syncthreads();
        }
        /* combine the halves in fixed order */
        for (int h = 0; h < halves; h++) {
            if (half == h && tid < halves * t.n_g) {
                if (h == 0) sS[g] = acc;
                else { sS[g].x += acc.x; sS[g].y += acc.y; }
            }
            __syncthreads();
        }
        if (A.s_out)
            for (int gg = tid; gg < t.n_g; gg += JAS_THREADS) {
                A.s_out[(size_t)w * 2 * A.n_g_pad + gg] = sS[gg].x;
                A.s_out[(size_t)w * 2 * A.n_g_pad + A.n_g_pad + gg] = sS[gg].y;
            }
        for (int gg = tid; gg < t.n_g; gg += JAS_THREADS) {
            const double re = sS[gg].x, im = sS[gg].y;
            value += t.acoef[gg] * 0.5 * (re * re + im * im - (double)n);
        }
    }

    /* [pass 2] one thread per particle: gradient and Laplacian of the p term from S(G), the u term over partners */
    for (int i = tid; i < n; i += JAS_THREADS) {
        double gr[3] = {0, 0, 0}, lp = 0, uval = 0;
        T ri[3] = {0, 0, 0};
#pragma unroll
        for (int x = 0; x < DIM; x++) ri[x] = sp[x * n + i];
        if (t.n_g > 0 && (A.grad || A.lap)) {
            T2 row[DIM][JAS_MAXP];
#pragma unroll
            for (int k = 0; k < DIM; k++) {
                double s = 0;
#pragma unroll
                for (int x = 0; x < DIM; x++) s += (double)ri[x] * t.binv[3 * k + x];
                jas_powers<T>(s, t.mmax, row[k]);
            }
            T g0 = 0, g1 = 0, g2 = 0, l0 = 0;
            for (int g = 0; g < t.n_g; g++) {
                const short4 nn = t.gn[g];
                T2 e = jas_cmul(jas_pick(row[0], nn.x), jas_pick(row[1], nn.y));
                if (DIM == 3) e = jas_cmul(e, jas_pick(row[DIM - 1], nn.z));
                const T2 S = sS[g];
                const T re = e.x * S.x + e.y * S.y, im = e.y * S.x - e.x * S.y; /* e conj(S) */
                const double *ga = t.ga + 4 * g;
                g0 -= (T)ga[0] * im; g1 -= (T)ga[1] * im; g2 -= (T)ga[2] * im;
                l0 -= (T)ga[3] * (re - 1);
            }
            gr[0] = g0; gr[1] = g1; gr[2] = g2; lp = l0;
        }
        if (t.n_u >= 0) {
            const T lu2 = (T)(t.l_u * t.l_u);
            T uv = 0, ug[3] = {0, 0, 0}, ul = 0;
            for (int j = 0; j < n; j++) {
                T d[3] = {0, 0, 0};
#pragma unroll
                for (int x = 0; x < DIM; x++) d[x] = ri[x] - sp[x * n + j];
                jas_min_image<T, DIM>(t, d);
                const T r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                if (j != i && r2 < lu2) {
                    /* coincident particles (r = 0): u(0) counts, the gradient term does not (as in the oracle) */
                    const T inv_r = r2 > 0 ? jas_rsqrt(r2) : T(0), r = r2 * inv_r;
                    T u, dur, d2u;
                    jas_u<T>(t, r, inv_r, &u, &dur, &d2u);
                    uv += u;
#pragma unroll
                    for (int x = 0; x < DIM; x++) ug[x] += dur * d[x];
                    ul += d2u + (T)(DIM - 1) * dur;
                }
            }
            uval = 0.5 * (double)uv;
            gr[0] += ug[0]; gr[1] += ug[1]; gr[2] += ug[2]; lp += ul;
        }
        value += uval;
        if (A.grad)
#pragma unroll
            for (int x = 0; x < DIM; x++) A.grad[((size_t)w * DIM + x) * A.npad + i] = gr[x];
        if (A.lap) A.lap[(size_t)w * A.npad + i] = lp;
    }
    value = block_sum(value, red);
    if (tid == 0 && A.value) A.value[w] = value;
}

template <typename T> struct JasMoveArgs {
    T *pos; T *S;                 /* stored [W][DIM][npad], [W][2][n_g_pad] */
    int n, npad, n_walkers, n_g_pad, n_moves;
    JasTabs t;
    const int *walker; const int *electron; const T *new_r;
    int commit;
    double *delta;
};

constexpr int JAS_MOVE_THREADS = 128;

template <typename T, int DIM>
__global__ void __launch_bounds__(JAS_MOVE_THREADS) jastrow_move_kernel(JasMoveArgs<T> A)
{
    typedef typename Num<T>::T2 T2;
    const JasTabs &t = A.t;
    __shared__ double red[32];
    __shared__ T2 rows[2][3][JAS_MAXP];
    const int m = blockIdx.x, tid = threadIdx.x;
    const int w = A.walker[m], k = A.electron[m];
    if (w < 0 || w >= A.n_walkers || k < 0 || k >= A.n) {
        if (tid == 0) A.delta[m] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    T *pw = A.pos + (size_t)w * DIM * A.npad;
    T r_old[3] = {0, 0, 0}, r_new[3] = {0, 0, 0};
#pragma unroll
    for (int x = 0; x < DIM; x++) { r_old[x] = pw[x * A.npad + k]; r_new[x] = A.new_r[(size_t)m * DIM + x]; }
    if (tid < 2 * DIM) {
        const int which = tid / DIM, ax = tid - which * DIM;
        const T *r = which ? r_new : r_old;
        double s = 0;
#pragma unroll
        for (int x = 0; x < DIM; x++) s += (double)r[x] * t.binv[3 * ax + x];
        T2 row[JAS_MAXP];
        jas_powers<T>(s, t.mmax, row);
        for (int q = 0; q <= t.mmax; q++) rows[which][ax][q] = row[q];
    }
    __syncthreads();
    double acc = 0;
    /* p term: sum_{j != k} [cos(G.(r' - r_j)) - cos(G.(r - r_j))] = Re[(e' - e) conj(S - e)]; patch S += e' - e */
    T *Sw = A.S + (size_t)w * 2 * A.n_g_pad;
    for (int g = tid; g < t.n_g; g += JAS_MOVE_THREADS) {
        const short4 nn = t.gn[g];
        T2 e[2];
#pragma unroll
        for (int which = 0; which < 2; which++) {
            T2 v = jas_cmul(jas_pick(rows[which][0], nn.x), jas_pick(rows[which][1], nn.y));
            if (DIM == 3) v = jas_cmul(v, jas_pick(rows[which][DIM - 1], nn.z));
            e[which] = v;
        }
        const T sre = Sw[g], sim = Sw[A.n_g_pad + g];
        const T dr = e[1].x - e[0].x, di = e[1].y - e[0].y;
        acc += t.acoef[g] * (double)(dr * (sre - e[0].x) + di * (sim - e[0].y));
        if (A.commit) { Sw[g] = sre + dr; Sw[A.n_g_pad + g] = sim + di; }
    }
    /* u term over the partners */
    if (t.n_u >= 0) {
        const T lu2 = (T)(t.l_u * t.l_u);
        T part = 0;
        for (int j = tid; j < A.n; j += JAS_MOVE_THREADS) {
            if (j == k) continue;
            T rj[3] = {0, 0, 0};
#pragma unroll
            for (int x = 0; x < DIM; x++) rj[x] = pw[x * A.npad + j];
#pragma unroll
            for (int which = 0; which < 2; which++) {
                T d[3] = {0, 0, 0};
#pragma unroll
                for (int x = 0; x < DIM; x++) d[x] = (which ? r_new[x] : r_old[x]) - rj[x];
                jas_min_image<T, DIM>(t, d);
                const T r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                if (r2 < lu2) {
                    T u, dur, d2u;
                    jas_u<T>(t, sqrt(r2), T(0), &u, &dur, &d2u);
                    part += which ? u : -u;
                }
            }
        }
        acc += (double)part;
    }
    acc = block_sum(acc, red); /* its barriers also order every read of r_old before the commit */
    if (tid == 0) {
        A.delta[m] = acc;
        if (A.commit)
#pragma unroll
            for (int x = 0; x < DIM; x++) pw[x * A.npad + k] = r_new[x];
    }
}

} // namespace ewald
