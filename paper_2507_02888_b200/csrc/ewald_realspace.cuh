/* ewald_realspace.cuh -- the real-lattice sum of Eq. 3,
 *     psi(d) = sum_R erfc(kappa |d - R|) / |d - R|,
 * organised for the B200's FP64 pipe (64 lanes/SM) and its 128 B/clk of shared-memory bandwidth.
 * Everything works in kappa-scaled squared lengths t = kappa^2 |d - R|^2, and a term is
 *     kappa q_i q_j F(t),   F(t) = erfc(sqrt t)/sqrt t,
 * with F read from a piecewise polynomial IN t (no square root, no exponential on the device):
 * bins are cut from the floating-point bits of t (2^K per binary octave), the local variable is
 * u = t - (bin centre), the coefficients were fitted in long double at setup ("lookup tables ...
 * always DP"; ewald_setup.cpp build_pair_table) and sit in shared memory as
 * [bin][degree+1] (FP64: quintic, 3 LDS.128 per term; FP32: cubic, 1 LDS.128).
 *
 * Two phases per warp:
 *   A  cull: each lane owns one pair, reduces its displacement to the cell, scans the candidate
 *      images and pushes the t that pass t < kappa^2 r_c^2 on its PRIVATE stack in shared memory
 *      (layout [slot][lane]: one predicated store and one predicated add per candidate, no votes);
 *   B  evaluate: whenever every lane holds >= R items the warp pops R per lane and evaluates them with
 *      all 32 lanes busy; a stack that would overflow forces a masked round; the tail is masked.
 * With all charge products equal (the electron gas; electrons against one ion species) the stack holds
 * t alone and the product is applied to the lane's sum; otherwise items are (t, q_i q_j).
 */
#pragma once
#include "ewald_kernels_common.cuh"

namespace ewald {

template <typename T> struct PairFmt;
template <> struct PairFmt<double> { static constexpr int K = 7, DEG = 5, NC = 6, SHIFT = 20 - 7, EBIAS = 1023; };
template <> struct PairFmt<float> { static constexpr int K = 5, DEG = 3, NC = 4, SHIFT = 23 - 5, EBIAS = 127; };

/* Geometry in kappa-scaled units. */
template <typename T> struct RealGeom {
    T a[9];      /* lattice rows * kappa                         */
    T binv[9];   /* fractional rows / kappa: s_k = d . binv[k]    */
    T L[3];      /* orthorhombic box lengths * kappa              */
    T invL[3];
    T kappa;
    int key_rc;  /* order key of kappa^2 r_c^2                    */
    int key_min; /* order key of the table's lower end t_min      */
    int bias;    /* bin index = (key >> SHIFT) - bias             */
    int m_shift; /* images -m_shift..m_shift scanned per axis (orthorhombic path) */
};

/* Positive floating-point numbers order like their leading bits.  FP64 uses the high word: ties within
 * 2^-20 are accepted (the cut-off is converged: a term at r_c is below 1e-16 of the sum, reading R19),
 * which keeps every comparison off the FP64 pipe. */
__device__ __forceinline__ int order_key(double t) { return __double2hiint(t); }
__device__ __forceinline__ int order_key(float t) { return __float_as_int(t); }

/* Centre of the bin of t: the low mantissa bits replaced by 100..0. */
__device__ __forceinline__ double bin_centre(double, int key)
{
    constexpr int S = PairFmt<double>::SHIFT;
    return __hiloint2double((key & ~((1 << S) - 1)) | (1 << (S - 1)), 0);
}
__device__ __forceinline__ float bin_centre(float, int key)
{
    constexpr int S = PairFmt<float>::SHIFT;
    return __int_as_float((key & ~((1 << S) - 1)) | (1 << (S - 1)));
}

/* F(t) from the shared-memory table; requires t_min <= t < t_max. */
__device__ __forceinline__ double pair_f(double t, const double *tab, int bias)
{
    const int key = order_key(t);
    const double u = t - bin_centre(t, key);
    const double2 *c = reinterpret_cast<const double2 *>(tab) + 3 * ((key >> PairFmt<double>::SHIFT) - bias);
    const double2 c01 = c[0], c23 = c[1], c45 = c[2];
    double p = fma(c45.y, u, c45.x);
    p = fma(p, u, c23.y);
    p = fma(p, u, c23.x);
    p = fma(p, u, c01.y);
    return fma(p, u, c01.x);
}
__device__ __forceinline__ float pair_f(float t, const float *tab, int bias)
{
    const int key = order_key(t);
    const float u = t - bin_centre(t, key);
    const float4 c = reinterpret_cast<const float4 *>(tab)[(key >> PairFmt<float>::SHIFT) - bias];
    float p = fmaf(c.w, u, c.z);
    p = fmaf(p, u, c.y);
    return fmaf(p, u, c.x);
}

/* The direct formula, for the rare t below the table (kappa r < 1/8) and for coincident particles
 * (t = 0 gives inf, reading R11). */
__device__ __forceinline__ double pair_f_direct(double t) { const double z = sqrt(t); return erfc(z) / z; }
__device__ __forceinline__ float pair_f_direct(float t) { const float z = sqrtf(t); return erfcf(z) / z; }

/* +-1 with the sign of t; |t| */
__device__ __forceinline__ double sign_unit(double t)
{
    return __hiloint2double((__double2hiint(t) & 0x80000000) | 0x3ff00000, 0);
}
__device__ __forceinline__ float sign_unit(float t) { return __int_as_float((__float_as_int(t) & 0x80000000) | 0x3f800000); }
__device__ __forceinline__ double abs_of(double t) { return fabs(t); }
__device__ __forceinline__ float abs_of(float t) { return fabsf(t); }

/* Item of a lane's stack: t alone when all charge products are equal (UQ), else (t, q_i q_j). */
template <typename T, bool UQ> struct PairItem;
template <typename T> struct PairItem<T, true> {
    T t;
    __device__ __forceinline__ static PairItem make(T t, T) { PairItem i; i.t = t; return i; }
    __device__ __forceinline__ T weight() const { return T(1); }
};
template <typename T> struct __align__(2 * sizeof(T)) PairItem<T, false> {
    T t, w;
    __device__ __forceinline__ static PairItem make(T t, T w) { PairItem i; i.t = t; i.w = w; return i; }
    __device__ __forceinline__ T weight() const { return w; }
};

constexpr int PAIR_R = 4; /* items per lane per evaluation round (independent FMA chains) */

/* Per-lane stack in shared memory, layout [slot][lane] per warp; all control flow that touches it is
 * warp-uniform, the contents are lane-private. */
template <typename T, bool UQ, bool SIGNED = false> struct LaneStack {
    typedef PairItem<T, UQ> Item;
    Item *base;  /* this lane's slot 0 */
    int top;     /* 32 * number of items */
    int cap32;   /* 32 * capacity */
    const T *tab;
    int bias;
    double sum;  /* lane's running sum of weight * F(t) */

    /* t_safe: any t inside the table; slot 0 always holds a valid item so that masked rounds can read it */
    __device__ __forceinline__ void init(void *warp_mem, int lane, int cap, const T *table, int b, T t_safe)
    {
        base = reinterpret_cast<Item *>(warp_mem) + lane;
        top = 0; cap32 = 32 * cap; tab = table; bias = b; sum = 0;
        base[0] = Item::make(t_safe, T(0));
    }
    __device__ __forceinline__ void push(bool ok, T t, T w)
    {
        if (ok) { base[top] = Item::make(t, w); top += 32; }
    }
    /* one round: pop up to R items per lane and add their terms (MASKED: lanes may hold fewer) */
    template <bool MASKED> __device__ __forceinline__ void round()
    {
        T part = 0;
#pragma unroll
        for (int r = 0; r < PAIR_R; r++) {
            const int s = top - 32 * (r + 1);
            const bool have = !MASKED || s >= 0;
            const Item it = base[have ? s : 0];
            /* SIGNED stacks of bare t carry the sign of the term in the sign bit of t */
            const T wt = UQ ? (SIGNED ? sign_unit(it.t) : T(1)) : it.weight();
            const T f = pair_f(UQ && SIGNED ? abs_of(it.t) : it.t, tab, bias);
            if (MASKED) part += have ? f * wt : T(0);
            else part = UQ && !SIGNED ? part + f : fma(f, wt, part);
        }
        top = MASKED ? max(top - 32 * PAIR_R, 0) : top - 32 * PAIR_R;
        sum += (double)part;
    }
    /* Called by the whole warp after each group of at most `limit` pushes per lane. */
    __device__ __forceinline__ void service(int limit)
    {
        int mn = __reduce_min_sync(0xffffffffu, top);
        while (mn >= 32 * PAIR_R) { round<false>(); mn -= 32 * PAIR_R; }
        int mx = __reduce_max_sync(0xffffffffu, top);
        while (mx > cap32 - 32 * limit) { round<true>(); mx -= 32 * PAIR_R; }
    }
    __device__ __forceinline__ void finish()
    {
        int mx = __reduce_max_sync(0xffffffffu, top);
        while (mx > 0) { round<true>(); mx -= 32 * PAIR_R; }
    }
};

/* Images scanned between two services of the stack on the image-list path. */
constexpr int IMG_STEP = 8;

/* Pushes per lane between two services of the stack, and the stack capacity that allows them. */
template <int DIM, bool ORTHO, int M> struct ScanShape {
    static constexpr int ROW = 2 * M + 1;
    static constexpr int ALL = DIM == 3 ? ROW * ROW * ROW : ROW * ROW;
    static constexpr bool WHOLE = ALL <= 27;               /* service once per pair, else once per x-row */
    static constexpr int LIMIT = ORTHO ? (WHOLE ? ALL : ROW) : IMG_STEP;
    static constexpr int MIN_CAP = LIMIT + PAIR_R;
};

/* Phase A for one pair per lane.  d = kappa (r_i - r_j), not yet reduced; w = q_i q_j.  Terms below the
 * table (t < t_min) are evaluated directly into `direct` (weighted by w); the rest go to the stack. */
template <typename T, int DIM, bool ORTHO, int M, bool UQ, bool SIGNED = false, bool NEG = false>
__device__ __forceinline__ void scan_pair(const RealGeom<T> &g, T *d, T w, bool valid,
                                          LaneStack<T, UQ, SIGNED> &st, double &direct, const T *simg, int nimg)
{
    /* NEG (move kernel, old position): the term enters with a minus sign -- in w for (t, w) items (the
     * caller passes -w), in the sign bit of t for bare-t items */
    constexpr bool FLIP = NEG && UQ && SIGNED;
    typedef ScanShape<DIM, ORTHO, M> Shape;
    if (ORTHO) {
        constexpr int ROW = Shape::ROW;
        T sq[DIM][ROW];
#pragma unroll
        for (int k = 0; k < DIM; k++) {
            d[k] = fma(-Num<T>::rint_(d[k] * g.invL[k]), g.L[k], d[k]);
#pragma unroll
            for (int m = 0; m < ROW; m++) { const T x = fma((T)(M - m), g.L[k], d[k]); sq[k][m] = x * x; }
        }
        /* only the un-shifted candidate can fall below the table: |d_k - m L_k| >= L_k/2 otherwise */
        T t0 = sq[0][M] + sq[1][M];
        if (DIM == 3) t0 += sq[2][M];
        const bool tiny = valid && order_key(t0) < g.key_min;
        if (tiny) direct += (double)((FLIP ? -w : w) * pair_f_direct(t0));
        const bool central_ok = valid && !tiny;
#pragma unroll
        for (int mz = 0; mz < (DIM == 3 ? ROW : 1); mz++) {
#pragma unroll
            for (int my = 0; my < ROW; my++) {
                const T syz = DIM == 3 ? sq[1][my] + sq[2][mz] : sq[1][my];
#pragma unroll
                for (int mx = 0; mx < ROW; mx++) {
                    const T t = sq[0][mx] + syz;
                    const bool centre = mx == M && my == M && (DIM == 2 || mz == M);
                    st.push((centre ? central_ok : valid) && order_key(t) <= g.key_rc, FLIP ? -t : t, w);
                }
                if (!Shape::WHOLE) st.service(Shape::LIMIT);
            }
        }
        if (Shape::WHOLE) st.service(Shape::LIMIT);
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
        for (int m0 = 0; m0 < nimg; m0 += IMG_STEP) {
#pragma unroll
            for (int u = 0; u < IMG_STEP; u++) {
                const int m = m0 + u;
                const bool in = valid && m < nimg;
                const int mm = m < nimg ? m : 0;
                T t = 0;
#pragma unroll
                for (int x = 0; x < DIM; x++) { const T v = d[x] - simg[3 * mm + x]; t = fma(v, v, t); }
                const int key = order_key(t);
                const bool tiny = in && key < g.key_min;
                if (tiny) direct += (double)((FLIP ? -w : w) * pair_f_direct(t));
                st.push(in && !tiny && key <= g.key_rc, FLIP ? -t : t, w);
            }
            st.service(Shape::LIMIT);
        }
    }
}

} // namespace ewald
