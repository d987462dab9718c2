/* ewald_realspace.cuh -- the real-lattice sum of Eq. 3,
 *     psi(d) = sum_R erfc(kappa |d - R|) / |d - R|,
 * organised for the B200's FP64 pipe (64 lanes/SM): everything works in kappa-scaled lengths
 * (t = kappa^2 r^2), so a term is kappa * qq * erfc(sqrt t)/sqrt t.
 *
 * Two phases per warp:
 *   A  cull: per pair, the displacement is reduced to the cell and the candidate images are
 *      scanned; the squared distances that pass t < kappa^2 r_c^2 are pushed (ballot-compacted)
 *      into a per-warp shared-memory queue.  Orthorhombic cells build t from per-axis squares
 *      (1 add per candidate); general cells scan the image list.
 *   B  evaluate: 32 queued items at a time, one per lane, no divergence:
 *      y = t^-1/2 (MUFU seed + one cubic Newton step), z = t y, erfc(z) by a piecewise polynomial
 *      (16 bins in z, degree ERFC_DEG, coefficients built in long double at setup -- the "lookup
 *      tables ... always DP" of PAPER.md:359 -- laid out [coef][bin] so a warp's loads hit one
 *      128-byte row without bank conflicts), term = qq y erfc(z).
 */
#pragma once
#include "ewald_kernels_common.cuh"

namespace ewald {

constexpr int ERFC_BINS = 16;
template <typename T> struct ErfcDeg;
template <> struct ErfcDeg<double> { static constexpr int value = 11; };
template <> struct ErfcDeg<float> { static constexpr int value = 6; };
/* table rows: coefficients c_0..c_DEG of erfc on the bin in u in [-1,1], then the row -(2b+1) */
template <typename T> struct ErfcRows { static constexpr int value = ErfcDeg<T>::value + 2; };

/* Geometry in kappa-scaled units. */
template <typename T> struct RealGeom {
    T a[9];      /* lattice rows * kappa                         */
    T binv[9];   /* fractional rows / kappa: s_k = d . binv[k]    */
    T L[3];      /* orthorhombic box lengths * kappa              */
    T invL[3];
    T rc2;       /* kappa^2 r_c^2                                  */
    T inv_h;     /* ERFC_BINS / z_max                              */
    T kappa;
    int m_shift; /* images -m_shift..m_shift scanned per axis (orthorhombic path) */
};

template <typename T> __device__ __forceinline__ T inv_sqrt(T t);
template <> __device__ __forceinline__ float inv_sqrt<float>(float t) { return rsqrtf(t); }
template <> __device__ __forceinline__ double inv_sqrt<double>(double t)
{
    /* FP32 MUFU seed (rel. error ~2^-22), then one third-order step:
     * y <- y (1 + e/2 + 3 e^2/8), e = 1 - t y^2; remaining error ~ (5/16) e^3 < 1e-19 */
    double y = (double)rsqrtf((float)t);
    double e = fma(-(t * y), y, 1.0);
    double p = fma(e, 0.375, 0.5);
    return fma(y * e, p, y);
}

/* qq * erfc(sqrt t)/sqrt t for one queued item; tab = shared [DEG+1][ERFC_BINS]. */
template <typename T>
__device__ __forceinline__ T eval_item(T t, T qq, const T *tab, T inv_h)
{
    constexpr int DEG = ErfcDeg<T>::value;
    const T y = inv_sqrt<T>(t);
    const T z = t * y;
    int b = (int)((float)z * (float)inv_h);
    b = b > ERFC_BINS - 1 ? ERFC_BINS - 1 : b;
    const T u = fma(z, 2 * inv_h, tab[(DEG + 1) * ERFC_BINS + b]); /* bin [b h, (b+1) h] -> [-1, 1] */
    T p = tab[DEG * ERFC_BINS + b];
#pragma unroll
    for (int k = DEG - 1; k >= 0; k--) p = fma(p, u, tab[k * ERFC_BINS + b]);
    return (qq * y) * p;
}

template <typename T> __device__ __forceinline__ bool below(T t, T lim);
template <> __device__ __forceinline__ bool below<float>(float t, float lim) { return t < lim; }
/* positive doubles order like their high words; ties within 2^-20 are accepted (the cut-off is
 * converged: a term at r_c is below 1e-16 of the sum, reading R19) -- keeps the test off the FP64 pipe */
template <> __device__ __forceinline__ bool below<double>(double t, double lim)
{
    return __double2hiint(t) <= __double2hiint(lim);
}

/* Per-warp queue of (t, qq) items in shared memory. */
template <typename T> struct WarpQueue {
    typedef typename Num<T>::T2 T2;
    T2 *buf;
    int cnt; /* warp-uniform */
    int lane;
    __device__ __forceinline__ void push(bool ok, T t, T qq)
    {
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        if (ok) {
            T2 it; it.x = t; it.y = qq;
            buf[cnt + __popc(m & ((1u << lane) - 1u))] = it;
        }
        cnt += __popc(m);
    }
    /* evaluate full groups of 32 */
    __device__ __forceinline__ T drain(const T *tab, T inv_h)
    {
        T acc = 0;
        __syncwarp();
        while (cnt >= 32) {
            cnt -= 32;
            const T2 it = buf[cnt + lane];
            acc += eval_item<T>(it.x, it.y, tab, inv_h);
        }
        __syncwarp();
        return acc;
    }
    /* evaluate what is left (< 32 items) */
    __device__ __forceinline__ T finish(const T *tab, T inv_h)
    {
        T acc = drain(tab, inv_h);
        T2 it; it.x = 1; it.y = 0;
        if (lane < cnt) it = buf[lane];
        acc += eval_item<T>(it.x, it.y, tab, inv_h);
        cnt = 0;
        __syncwarp();
        return acc;
    }
};

constexpr int QUEUE_CAP_ORTHO = 5 * 32 + 32;  /* one x-row of candidates (<= 5) + carry-over */
constexpr int QUEUE_IMG_STEP = 4;             /* general cells: drain every 4 images          */
constexpr int QUEUE_CAP = 192;

/* Phase A for one pair per lane.  d = r_i - r_j (kappa-scaled, not yet reduced).  Returns the sum of
 * the terms evaluated while draining. */
template <typename T, int DIM, bool ORTHO, int M>
__device__ __forceinline__ T scan_pair(const RealGeom<T> &g, T *d, T qq, bool valid, WarpQueue<T> &q,
                                       const T *tab, const T *simg, int nimg)
{
    T acc = 0;
    if (ORTHO) {
#pragma unroll
        for (int k = 0; k < DIM; k++) d[k] = fma(-Num<T>::rint_(d[k] * g.invL[k]), g.L[k], d[k]);
        T sx[2 * M + 1];
#pragma unroll
        for (int m = 0; m <= 2 * M; m++) { T x = fma((T)(M - m), g.L[0], d[0]); sx[m] = x * x; }
        const int mz_hi = DIM == 3 ? M : 0;
        T zz = DIM == 3 ? fma((T)M, g.L[2], d[2]) : T(0);
        for (int mz = -mz_hi; mz <= mz_hi; mz++) {
            const T sz = zz * zz;
            zz -= g.L[2];
            T yy = fma((T)M, g.L[1], d[1]);
            for (int my = -M; my <= M; my++) {
                const T syz = fma(yy, yy, sz);
                yy -= g.L[1];
                if (!__any_sync(0xffffffffu, valid && below<T>(syz, g.rc2))) continue;
#pragma unroll
                for (int m = 0; m <= 2 * M; m++) {
                    const T t = sx[m] + syz;
                    q.push(valid && below<T>(t, g.rc2), t, qq);
                }
                acc += q.drain(tab, g.inv_h);
            }
        }
    } else {
        T f[3];
#pragma unroll
        for (int k = 0; k < DIM; k++) {
            T s = 0;
#pragma unroll
            for (int x = 0; x < DIM; x++) s = fma(d[x], g.binv[3 * k + x], s);
            f[k] = Num<T>::rint_(s);
        }
#pragma unroll
        for (int x = 0; x < DIM; x++) {
#pragma unroll
            for (int k = 0; k < DIM; k++) d[x] = fma(-f[k], g.a[3 * k + x], d[x]);
        }
        for (int m0 = 0; m0 < nimg; m0 += QUEUE_IMG_STEP) {
#pragma unroll
            for (int u = 0; u < QUEUE_IMG_STEP; u++) {
                const int m = m0 + u;
                const bool in = m < nimg;
                const int mm = in ? m : 0;
                T t = 0;
#pragma unroll
                for (int x = 0; x < DIM; x++) { const T v = d[x] - simg[3 * mm + x]; t = fma(v, v, t); }
                q.push(valid && in && below<T>(t, g.rc2), t, qq);
            }
            acc += q.drain(tab, g.inv_h);
        }
    }
    return acc;
}

} // namespace ewald
