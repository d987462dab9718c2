/* ewald_realspace.cuh -- the real-lattice sum of Eq. 3,
 *     psi(d) = sum_R erfc(kappa |d - R|) / |d - R|,
 * organised for the B200's FP64 pipe (64 lanes/SM) and its 128 B/clk of shared-memory bandwidth.
 * Everything works in kappa-scaled squared lengths t = kappa^2 |d - R|^2, and a term is
 *     kappa q_i q_j F(t),   F(t) = erfc(sqrt t)/sqrt t,
 * with F read from a piecewise polynomial IN t (no square root, no exponential on the device):
 * bins are cut from the floating-point bits of t (2^K per binary octave), the local variable is
 * u = t - (bin centre), the coefficients were fitted in long double at setup ("lookup tables ...
 * always DP"; ewald_setup.cpp build_pair_table) and sit in shared memory as
 * polynomials per bin (FP64: degree 7, 4 conflict-free LDS.128 per term; FP32: cubic, 1 LDS.128; layouts at PairFmt).
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
/* FP32: cubic on 32 bins per octave, REP = 8 copies interleaved [bin][copy][NC]; lane l reads copy l mod 8, so the
 * 8 lanes of a quarter-warp read 8 different 16-byte columns and the gather has no bank conflicts (6 KB -> 48 KB).
 * FP64: degree 7 on 32 bins per octave (64 bytes per bin; the quintic on 128 bins per octave of round 1 and 2
 * took 48-byte rows from one copy: ~2.6 wavefronts per quarter-warp and LDS.128 instead of 1).  The table is a
 * sequence of 512-byte ROWS [chunk 0..3][slot 0..7][2 doubles], chunk c = coefficients (2c, 2c + 1):
 *   t >= 4 (86 % of the terms below t = 13 of a uniform gas): one bin per row, the 8 slots are 8 copies, lane l
 *           reads slot l mod 8: each of the four LDS.128 of a term is conflict-free (4 wavefronts per warp);
 *   t <  4 (8 octaves, 256 bins): 8 consecutive bins per row, slot = bin mod 8 (one copy: 16 KB instead of 128).
 * Both regions are addressed as row * 512 + slot * 16 + chunk * 128 bytes.  With the far shell from t = 13 the
 * table takes 43 KB (52 + 32 rows); eight copies from t = 1 (72 KB) cost the stacks their depth and were slower. */
template <> struct PairFmt<double> {
    static constexpr int K = 5, DEG = 7, NC = 8, SHIFT = 20 - 5, EBIAS = 1023, REP = 8;
    static constexpr int E_MIN = -6, E_SPLIT = 0;        /* the table starts at 2^E_MIN; copies from 2^E_SPLIT */
    static constexpr int LOW = (E_SPLIT - E_MIN) << K;   /* bins below the split */
    static constexpr int ROW = 64;                       /* doubles per row */
    __host__ __device__ static constexpr int rows(int n_bins) { return n_bins <= LOW ? (n_bins + 7) / 8 : LOW / 8 + (n_bins - LOW); }
    __host__ __device__ static constexpr size_t elems(int n_bins) { return (size_t)rows(n_bins) * ROW; }
};
template <> struct PairFmt<float> {
    static constexpr int K = 5, DEG = 3, NC = 4, SHIFT = 23 - 5, EBIAS = 127, REP = 8;
    __host__ __device__ static constexpr size_t elems(int n_bins) { return (size_t)n_bins * NC * REP; }
};

/* Geometry in kappa-scaled units. */
template <typename T> struct RealGeom {
    T a[9];      /* lattice rows * kappa                         */
    T binv[9];   /* fractional rows / kappa: s_k = d . binv[k]    */
    T L[3];      /* orthorhombic box lengths * kappa              */
    T invL[3];
    T kappa;
    /* FP32 kernels: kappa, kappa L_k and the lattice rows rounded to float are the same for every pair, i.e. a
     * SYSTEMATIC error of up to 6e-8 relative in every t (measured: 1e-7 of E_real with one sign on every walker,
     * more than the 2e-5 of |E| allowed when the components cancel).  A low part added after a rounding is
     * absorbed (it is below half an ulp), so the FP32 orthorhombic scan works in units of the box instead: the box
     * length is exactly 1, every rounding is of a pair-dependent quantity (unbiased), and the only constants,
     * 1/L_k and (kappa L_k)^2, enter through one fma with their low parts: fma(x, c_hi, x c_lo). */
    T kappa_lo, a_lo[9];
    T invLu[3], invLu_lo[3]; /* 1/L_k (unscaled box lengths) */
    T C[3], C_lo[3];         /* (kappa L_k)^2 */
    double kappa_d; /* the unrounded kappa: prefactor of the sums */
    int key_rc;  /* order key of kappa^2 r_c^2                    */
    int key_min; /* order key of the table's lower end t_min      */
    int bias;    /* bin index = (key >> SHIFT) - bias             */
    int m_shift; /* images -m_shift..m_shift scanned per axis (orthorhombic path) */
    int multi_far; /* 3D, m_shift = 1: some L_j^2 + L_k^2 < kappa^2 r_c^2, i.e. two far images can be in range */
    int outer_far; /* every (kappa L_k)^2 >= T0: a candidate with a far image always belongs to the far shell */
    int far_once;  /* outer_far, no multi_far, and the far stack is deep enough for one service per pair */
};

/* kappa * diff; FP32: with the low part of kappa, rounded once. */
template <typename T> __device__ __forceinline__ T scale_kappa(const RealGeom<T> &g, T diff)
{
    if (sizeof(T) == 4) return fma(diff, g.kappa, diff * g.kappa_lo);
    return diff * g.kappa;
}

/* One axis of an orthorhombic cell: from the raw difference to the quantity the image scan shifts.
 * FP64: v = kappa-scaled displacement reduced to (-L/2, L/2], images at v - m L_k, square as is.
 * FP32: v = displacement in units of the box reduced to (-1/2, 1/2], images at v - m (exact), square scaled by
 * (kappa L_k)^2 with its low part. */
template <typename T> __device__ __forceinline__ T axis_reduce(const RealGeom<T> &g, int k, T diff)
{
    if (sizeof(T) == 4) {
        const T s = fma(diff, g.invLu[k], diff * g.invLu_lo[k]);
        return s - Num<T>::rint_(s);
    }
    const T d = diff * g.kappa;
    return fma(-Num<T>::rint_(d * g.invL[k]), g.L[k], d);
}
template <typename T> __device__ __forceinline__ T axis_unit(const RealGeom<T> &g, int k) { return sizeof(T) == 4 ? T(1) : g.L[k]; }
template <typename T> __device__ __forceinline__ T axis_square(const RealGeom<T> &g, int k, T x)
{
    const T x2 = x * x;
    if (sizeof(T) == 4) return fma(x2, g.C[k], x2 * g.C_lo[k]);
    return x2;
}

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

/* F(t) from the shared-memory table; requires t_min <= t < t_max.  slot2 = 2 * (lane mod 8).
 * ESTRIN: 9 operations in a chain of 4 instead of Horner's 7 in a chain of 7: faster in real_kernel (0.662 ->
 * 0.638 ms on config 2), slower in move_kernel, whose 16 warps per SM sit at the 128-register limit (15.2 -> 14.1 M
 * moves/s): each kernel takes its own. */
template <bool ESTRIN>
__device__ __forceinline__ double pair_f(double t, const double *tab, int bias, int slot2)
{
    typedef PairFmt<double> F;
    const int key = order_key(t);
    const double u = t - bin_centre(t, key);
    const int bin = (key >> F::SHIFT) - bias, hb = bin - F::LOW;
    const int off = hb >= 0 ? (hb + F::LOW / 8) * F::ROW + slot2 : (bin >> 3) * F::ROW + 2 * (bin & 7);
    const double2 *c = reinterpret_cast<const double2 *>(tab + off);
    const double2 c01 = c[0], c23 = c[8], c45 = c[16], c67 = c[24];
    if (!ESTRIN) {
        double p = fma(c67.y, u, c67.x);
        p = fma(p, u, c45.y);
        p = fma(p, u, c45.x);
        p = fma(p, u, c23.y);
        p = fma(p, u, c23.x);
        p = fma(p, u, c01.y);
        return fma(p, u, c01.x);
    }
    const double u2 = u * u;
    const double a = fma(c01.y, u, c01.x), b = fma(c23.y, u, c23.x), c4 = fma(c45.y, u, c45.x), d = fma(c67.y, u, c67.x);
    return fma(u2 * u2, fma(d, u2, c4), fma(b, u2, a));
}
template <bool ESTRIN>
__device__ __forceinline__ float pair_f(float t, const float *tab, int bias, int)
{
    const int key = order_key(t);
    const float u = t - bin_centre(t, key);
    const float4 c = reinterpret_cast<const float4 *>(tab)[((key >> PairFmt<float>::SHIFT) - bias) * PairFmt<float>::REP];
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

/* Shared-memory accesses by 32-bit window address: the stacks keep byte addresses, so a push is one store
 * and one add, and a pop is a load at a constant (negative) offset. */
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void st_s(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void st_s(unsigned a, double v, double w) { asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v), "d"(w) : "memory"); }
__device__ __forceinline__ void st_s(unsigned a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void st_s(unsigned a, float v, float w) { asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v), "f"(w) : "memory"); }
__device__ __forceinline__ void st_s(unsigned a, unsigned v) { asm volatile("st.shared.b32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void st_s(unsigned a, unsigned v, float w) { asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(a), "r"(v), "r"(__float_as_uint(w)) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, double &v) { asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, double &v, double &w) { asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v), "=d"(w) : "r"(a) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, float &v) { asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, float &v, float &w) { asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v), "=f"(w) : "r"(a) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, unsigned &v) { asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); }
__device__ __forceinline__ void ld_s(unsigned a, unsigned &v, float &w)
{
    unsigned wb;
    asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(v), "=r"(wb) : "r"(a) : "memory");
    w = __uint_as_float(wb);
}

/* Item of a lane's stack: t alone when all charge products are equal (UQ), else (t, q_i q_j).
 * K = the stored key type (T for the near stack, 32-bit fixed point for the far stack), W = weight type. */
template <typename K, typename W, bool UQ> struct StackItem;
template <typename K, typename W> struct StackItem<K, W, true> {
    static constexpr int BYTES = sizeof(K);
    __device__ __forceinline__ static void store(unsigned a, K t, W) { st_s(a, t); }
    __device__ __forceinline__ static void load(unsigned a, K &t, W &w) { ld_s(a, t); w = W(1); }
};
template <typename K, typename W> struct StackItem<K, W, false> {
    static constexpr int BYTES = sizeof(K) + sizeof(W);
    __device__ __forceinline__ static void store(unsigned a, K t, W w) { st_s(a, t, w); }
    __device__ __forceinline__ static void load(unsigned a, K &t, W &w) { ld_s(a, t, w); }
};

/* Items per lane per evaluation round (independent FMA chains), chosen per kernel (measured in one call, config 2 /
 * 3 / 4 real space in ms with 4, 5, 6 items: 0.626 / 0.490 / 3.40; 0.617 / 0.450 / 3.40; 0.613 / 0.449 / 3.38): the
 * FP64 energy kernel takes 5 (with 6 config 1's stacks do not fit 512 threads), the FP32 energy kernel and the move
 * kernels 4 (FP32 energy 0.366 -> 0.370 ms with 5; moves 15.6 -> 15.4 M / 26.9 -> 22.1 M).  The capacities are sized
 * for the kernel's own value (ScanShape::min_cap, PairTabs::round_items). */
template <typename T, bool SIGNED> struct RoundSize { static constexpr int R = !SIGNED && sizeof(T) == 8 ? 5 : 4; };

/* Per-lane stack in shared memory, layout [slot][lane] per warp, kept as byte addresses; all control flow
 * that touches it is warp-uniform, the contents are lane-private.  Derived classes supply term(). */
template <typename K, typename W, bool UQ, int R, typename Derived> struct StackBase {
    typedef StackItem<K, W, UQ> Item;
    static constexpr int SLOT = 32 * Item::BYTES;  /* bytes between two slots of a lane */
    unsigned base_a;  /* this lane's slot 0 */
    unsigned top_a;   /* this lane's first free slot */
    int cap_b;        /* capacity in bytes of address range (cap * SLOT) */
    double sum;       /* lane's running sum of weight * F(t) */

    __device__ __forceinline__ void init_base(void *warp_mem, int lane, int cap, K safe)
    {
        base_a = smem_addr(warp_mem) + lane * Item::BYTES;
        top_a = base_a; cap_b = cap * SLOT; sum = 0;
        Item::store(base_a, safe, W(0)); /* slot 0 always holds a valid item: masked rounds may read it */
    }
    __device__ __forceinline__ void push(bool ok, K t, W w)
    {
        if (ok) { Item::store(top_a, t, w); top_a += SLOT; }
    }
    /* one round: pop up to R items per lane and add their terms (MASKED: lanes may hold fewer) */
    template <bool MASKED> __device__ __forceinline__ void round()
    {
        typename Derived::Acc part = 0;
#pragma unroll
        for (int r = 0; r < R; r++) {
            const unsigned a = top_a - SLOT * (r + 1);
            const bool have = !MASKED || (int)(a - base_a) >= 0;
            K t; W w;
            Item::load(have ? a : base_a, t, w);
            const typename Derived::Acc f = static_cast<Derived *>(this)->term(t, w);
            part += MASKED ? (have ? f : typename Derived::Acc(0)) : f;
        }
        top_a = MASKED ? base_a + max((int)(top_a - base_a) - SLOT * R, 0) : top_a - SLOT * R;
        sum += (double)part;
    }
    /* Called by the whole warp after each group of at most `limit` pushes per lane. */
    __device__ __forceinline__ void service(int limit)
    {
        int mn = __reduce_min_sync(0xffffffffu, (int)(top_a - base_a));
        while (mn >= SLOT * R) { round<false>(); mn -= SLOT * R; }
        int mx = __reduce_max_sync(0xffffffffu, (int)(top_a - base_a));
        while (mx > cap_b - SLOT * limit) { round<true>(); mx -= SLOT * R; }
    }
    __device__ __forceinline__ void finish()
    {
        int mx = __reduce_max_sync(0xffffffffu, (int)(top_a - base_a));
        while (mx > 0) { round<true>(); mx -= SLOT * R; }
    }
};

/* Near stack: t in the kernel's precision, F from the degree-7 (FP32: cubic) table. */
template <typename T, bool UQ, bool SIGNED = false>
struct LaneStack : StackBase<T, T, UQ, RoundSize<T, SIGNED>::R, LaneStack<T, UQ, SIGNED>> {
    typedef T Acc;
    const T *tab;
    int bias;
    int slot2; /* FP64: 2 * (lane mod 8), the lane's 16-byte column of a table row */
    __device__ __forceinline__ void init(void *warp_mem, int lane, int cap, const T *table, int b, T t_safe)
    {
        /* FP32: this lane's copy; FP64: the table's base (the column is chosen per term, see pair_f) */
        tab = sizeof(T) == 4 ? table + (lane % PairFmt<T>::REP) * PairFmt<T>::NC : table;
        slot2 = 2 * (lane & 7);
        bias = b;
        this->init_base(warp_mem, lane, cap, t_safe);
    }
    __device__ __forceinline__ T term(T t, T w) const
    {
        /* SIGNED stacks of bare t carry the sign of the term in the sign bit of t */
        if (UQ && SIGNED) return pair_f<!SIGNED>(abs_of(t), tab, bias, slot2) * sign_unit(t);
        return UQ ? pair_f<!SIGNED>(t, tab, bias, slot2) : pair_f<!SIGNED>(t, tab, bias, slot2) * w;
    }
};

/* ---- the far shell (FP64 kernels only) ------------------------------------------------------------
 * Terms with t >= T0 = 13 are below F(13) = 9.6e-8 each (a few 1e-4 of a sum of order N^2/2 in all):
 * FP32 arithmetic on them (relative error ~1e-7 per term; the table's u^2 coefficient is chosen at setup so
 * that the error averages to zero over a bin, ewald_setup.cpp build_far_table) changes E by 4e-13 relative on
 * config 2 (measured).  They are kept as
 * 32-bit fixed point x = round(t 2^25) (one FP64 add with 2^27 puts it in the low word; resolution
 * 3e-8 in t, so F keeps 3e-8 relative), evaluated by an FP32 cubic on bins of width 1/8 in t whose index
 * and local variable are bit fields of x, from a table replicated 8 times so that the 8 lanes of a
 * quarter-warp read 8 different 16-byte columns: LDS.128 without bank conflicts. */
struct FarFmt {
    static constexpr int S = 25;            /* x = t 2^S, t < 64; bit 31 = sign of the term       */
    static constexpr int KB = 3;            /* 2^KB bins per unit of t                             */
    static constexpr int MB = S - KB;       /* bits of x inside a bin                              */
    static constexpr int REP = 8;           /* table copies                                        */
#ifndef EWALD_FAR_T0
#define EWALD_FAR_T0 13
#endif
    static constexpr int T0 = EWALD_FAR_T0; /* the far table starts at t = T0 (a kernel may start its far shell later) */
};
__device__ __forceinline__ unsigned far_fixed(double t) { return (unsigned)__double2loint(t + 134217728.0 /* 2^27 */); }

template <bool UQ, bool SIGNED> struct FarStack : StackBase<unsigned, float, UQ, RoundSize<double, SIGNED>::R, FarStack<UQ, SIGNED>> {
    typedef float Acc;
    const float4 *tab; /* [bin][REP] cubic in u = (fraction of the bin) - 1/2; this lane's copy pre-selected */
    /* the staged table starts at bin t0 << KB (t0 = where this kernel's far shell starts): the pointer is biased
     * by that many bins, so that the bin index cut from x addresses it directly */
    __device__ __forceinline__ void init(void *warp_mem, int lane, int cap, const float *table, int t0)
    {
        tab = reinterpret_cast<const float4 *>(table) + (lane & (FarFmt::REP - 1)) - (ptrdiff_t)(t0 << FarFmt::KB) * FarFmt::REP;
        this->init_base(warp_mem, lane, cap, (unsigned)t0 << FarFmt::S);
    }
    __device__ __forceinline__ float term(unsigned x, float w) const
    {
        const int idx = (int)((x & 0x7fffffffu) >> FarFmt::MB);
        /* the MB bits inside the bin become the mantissa of a float in [1, 2) */
        const float u = __uint_as_float(((x << (23 - FarFmt::MB)) & 0x7fffffu) | 0x3f800000u) - 1.5f;
        const float4 c = tab[idx * FarFmt::REP];
        float f = fmaf(fmaf(fmaf(c.w, u, c.z), u, c.y), u, c.x);
        if (UQ && SIGNED) f = __uint_as_float(__float_as_uint(f) ^ (x & 0x80000000u));
        return UQ ? f : f * w;
    }
};

/* The stacks of one lane: near (t in the kernel's precision) and, for FP64 kernels, far. */
template <typename T, bool UQ, bool SIGNED> struct PairStacks;
template <bool UQ, bool SIGNED> struct PairStacks<float, UQ, SIGNED> {
    LaneStack<float, UQ, SIGNED> nr;
    template <bool FLIP> __device__ __forceinline__ void push(bool ok, float t, int, float w) { nr.push(ok, FLIP ? -t : t, w); }
    template <bool FLIP> __device__ __forceinline__ void push_far(bool ok, float t, int key, float w) { push<FLIP>(ok, t, key, w); }
    __device__ __forceinline__ void service(int limit) { nr.service(limit); }
    __device__ __forceinline__ void service_far(int limit) { nr.service(limit); } /* no far stack in FP32 */
    __device__ __forceinline__ void service_near(int limit) { nr.service(limit); }
    __device__ __forceinline__ void finish() { nr.finish(); }
    __device__ __forceinline__ double take() { const double v = nr.sum; nr.sum = 0; return v; }
};
template <bool UQ, bool SIGNED> struct PairStacks<double, UQ, SIGNED> {
    LaneStack<double, UQ, SIGNED> nr;
    FarStack<UQ, SIGNED> fr;
    int key_far; /* order key of T0, or INT_MAX when the far shell is switched off */
    template <bool FLIP> __device__ __forceinline__ void push(bool ok, double t, int key, double w)
    {
        const bool far = key >= key_far;
        nr.push(ok && !far, FLIP ? -t : t, w);
        fr.push(ok && far, far_fixed(t) | (FLIP ? 0x80000000u : 0u), (float)w);
    }
    /* for candidates known to lie in the far shell (t >= T0): no near-stack instructions at all */
    template <bool FLIP> __device__ __forceinline__ void push_far(bool ok, double t, int, double w)
    {
        fr.push(ok, far_fixed(t) | (FLIP ? 0x80000000u : 0u), (float)w);
    }
    /* key_far is uniform over the grid: the far stack is either used by every lane or by none */
    __device__ __forceinline__ bool has_far() const { return key_far != 0x7fffffff; }
    __device__ __forceinline__ void service(int limit) { nr.service(limit); if (has_far()) fr.service(limit); }
    /* after a group that pushed on the far stack only (push_far) */
    __device__ __forceinline__ void service_far(int limit) { fr.service(limit); }
    __device__ __forceinline__ void service_near(int limit) { nr.service(limit); }
    __device__ __forceinline__ void finish() { nr.finish(); if (has_far()) fr.finish(); }
    __device__ __forceinline__ double take() { const double v = nr.sum + fr.sum; nr.sum = 0; fr.sum = 0; return v; }
};

/* Images scanned between two services of the stack on the image-list path. */
constexpr int IMG_STEP = 8;

/* Pushes per lane between two services of the stack, and the stack capacity that allows them. */
template <int DIM, bool ORTHO, int M, bool UQ> struct ScanShape {
    static constexpr int ROW = 2 * M + 1;
    static constexpr int ALL = DIM == 3 ? ROW * ROW * ROW : ROW * ROW;
    /* the stacks are serviced once per pair (few images), after the 8 core and after the 12 one-far candidates
     * (|m| <= 1 in 3D, see scan_pair), else once per x-row: small LIMIT = small stacks = more warps per SM */
    /* (t, qq) items take twice the bytes, i.e. half the capacity: always once per x-row */
    static constexpr bool WHOLE = ALL <= (UQ ? 9 : 3);
    static constexpr bool PLANE = UQ && !WHOLE && DIM == 3 && ROW == 3;
    /* with very few images per pair the energy kernel scans GROUP pairs between two services */
    static constexpr int GROUP = UQ && ORTHO && WHOLE && ALL <= 4 ? 8 / ALL : 1;
    /* image-list path: (t, qq) items have half the capacity, so half the images between two services */
    static constexpr int LIMIT = ORTHO ? (WHOLE ? ALL * GROUP : PLANE ? 12 : ROW) : (UQ ? IMG_STEP : IMG_STEP / 2);
    static constexpr int min_cap(int round_items) { return LIMIT + round_items; }
    static constexpr int FAR_LIMIT = 20; /* PLANE, fast variant: all 20 candidates between two far services */
    /* small batches of small boxes (|m| <= 2 in 3D: 125 candidates per pair): the energy kernel can deal the ROW
     * z-images of a pair to ROW different lanes, so that few walkers still fill the GPU (RealArgs::zsplit) */
    static constexpr bool ZSPLIT = ORTHO && !WHOLE && !PLANE && DIM == 3 && M == 2;
};

/* Phase A for one pair per lane.  d = r_i - r_j (raw, neither scaled nor reduced); w = q_i q_j.  Terms below the
 * table (t < t_min) are evaluated directly into `direct` (weighted by w); the rest go to the stack. */
template <typename T, int DIM, bool ORTHO, int M, bool UQ, bool SIGNED = false, bool NEG = false,
          bool SERVICE = true>
__device__ __forceinline__ void scan_pair(const RealGeom<T> &g, T *d, T w, bool valid,
                                          PairStacks<T, UQ, SIGNED> &st, double &direct, const T *simg, int nimg,
                                          bool list_service = true, int zsel = -1)
{
    /* zsel >= 0 (uniform over the grid; ScanShape::ZSPLIT shapes only): this lane scans the z-image zsel of its
     * pair alone, ROW lanes share the pair */
    /* list_service = false (image-list path, few images): the caller services the stacks after several pairs.
     * NEG (move kernel, old position): the term enters with a minus sign -- in w for (t, w) items (the
     * caller passes -w), in the sign bit of t for bare-t items */
    constexpr bool FLIP = NEG && UQ && SIGNED;
    typedef ScanShape<DIM, ORTHO, M, UQ> Shape;
    if (ORTHO && Shape::PLANE) {
        /* |m| <= 1 in 3D, bare-t items.  Only squared distances matter, so the three images of an axis are
         * taken as {un-shifted, near, far} = {d^2, (L-|d|)^2, (L+|d|)^2}: the 8 core candidates (no far
         * image), the 12 with one far image, and -- only if two box lengths fit inside the cut-off
         * (g.multi_far, uniform over the grid) -- the 7 with two or three. */
        T a[3][3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const T v = axis_reduce(g, k, d[k]), ad = abs_of(v), unit = axis_unit(g, k);
            a[k][0] = axis_square(g, k, v); a[k][1] = axis_square(g, k, unit - ad); a[k][2] = axis_square(g, k, unit + ad);
        }
        const T t0 = a[0][0] + (a[1][0] + a[2][0]);
        const bool tiny = valid && order_key(t0) < g.key_min;
        if (tiny) direct += (double)((FLIP ? -w : w) * pair_f_direct(t0));
        const bool central_ok = valid && !tiny;
        auto cand = [&](int i, int j, int k, bool ok) {
            const T t = a[0][i] + (a[1][j] + a[2][k]);
            const int key = order_key(t);
            st.template push<FLIP>(ok && key <= g.key_rc, t, key, w);
        };
        auto cand_far = [&](int i, int j, int k, bool ok) { /* t >= T0 is known: far stack only */
            const T t = a[0][i] + (a[1][j] + a[2][k]);
            const int key = order_key(t);
            st.template push_far<FLIP>(ok && key <= g.key_rc, t, key, w);
        };
#pragma unroll
        for (int c = 0; c < 8; c++) cand(c & 1, (c >> 1) & 1, c >> 2, c == 0 ? central_ok : valid);
        /* fast = far-image candidates are far-shell terms and there are 12 of them (uniform over the grid):
         * the near stack sees the 8 core candidates only, the far stack (twice the capacity) is serviced once
         * per pair, after all 20 */
        const bool fast = g.far_once != 0;
        if (fast) st.service_near(8); else st.service(Shape::LIMIT);
        if (g.outer_far) {
#pragma unroll
            for (int c = 0; c < 4; c++) { cand_far(2, c & 1, c >> 1, valid); cand_far(c & 1, 2, c >> 1, valid); }
#pragma unroll
            for (int c = 0; c < 4; c++) cand_far(c & 1, c >> 1, 2, valid);
            /* not fast: the next pair's 8 core candidates may push on the far stack before the next service */
            if (fast) st.service_far(Shape::FAR_LIMIT); else st.service_far(Shape::LIMIT);
        } else {
#pragma unroll
            for (int c = 0; c < 4; c++) { cand(2, c & 1, c >> 1, valid); cand(c & 1, 2, c >> 1, valid); }
#pragma unroll
            for (int c = 0; c < 4; c++) cand(c & 1, c >> 1, 2, valid);
        }
        if (g.multi_far) {
            st.service(Shape::LIMIT);
#pragma unroll
            for (int c = 0; c < 2; c++) { cand(2, 2, c, valid); cand(2, c, 2, valid); cand(c, 2, 2, valid); }
            cand(2, 2, 2, valid);
        }
        if (!g.outer_far || g.multi_far) st.service(Shape::LIMIT);
    } else if (ORTHO) {
        constexpr int ROW = Shape::ROW;
        T sq[DIM][ROW];
#pragma unroll
        for (int k = 0; k < DIM; k++) {
            d[k] = axis_reduce(g, k, d[k]);
#pragma unroll
            for (int m = 0; m < ROW; m++) sq[k][m] = axis_square(g, k, fma((T)(M - m), axis_unit(g, k), d[k]));
        }
        /* only the un-shifted candidate can fall below the table: |d_k - m L_k| >= L_k/2 otherwise */
        T t0 = sq[0][M] + sq[1][M];
        if (DIM == 3) t0 += sq[2][M];
        const bool tiny = valid && order_key(t0) < g.key_min;
        if (tiny && (!Shape::ZSPLIT || zsel < 0 || zsel == M)) direct += (double)((FLIP ? -w : w) * pair_f_direct(t0));
        const bool central_ok = valid && !tiny;
        if (Shape::WHOLE) {
#pragma unroll
            for (int mz = 0; mz < (DIM == 3 ? ROW : 1); mz++) {
#pragma unroll
                for (int my = 0; my < ROW; my++) {
                    const T syz = DIM == 3 ? sq[1][my] + sq[2][mz] : sq[1][my];
#pragma unroll
                    for (int mx = 0; mx < ROW; mx++) {
                        const T t = sq[0][mx] + syz;
                        const bool centre = mx == M && my == M && (DIM == 2 || mz == M);
                        const int key = order_key(t);
                        st.template push<FLIP>((centre ? central_ok : valid) && key <= g.key_rc, t, key, w);
                    }
                }
            }
            if (SERVICE) st.service(Shape::LIMIT); /* else the caller does, after Shape::GROUP pairs */
        } else {
            /* rolled loops over the y and z images (the stacks are serviced after every x-row) */
            const bool zs = Shape::ZSPLIT && zsel >= 0;
            const int z_trips = zs ? 1 : (DIM == 3 ? ROW : 1);
#pragma unroll 1
            for (int zi = 0; zi < z_trips; zi++) {
                const int mz = zs ? zsel : zi;
                T sz = 0;
                if (DIM == 3) sz = axis_square(g, 2, fma((T)(M - mz), axis_unit(g, 2), d[2]));
#pragma unroll 1
                for (int my = 0; my < ROW; my++) {
                    const T syz = axis_square(g, 1, fma((T)(M - my), axis_unit(g, 1), d[1])) + sz;
                    const bool crow = my == M && (DIM == 2 || mz == M);
#pragma unroll
                    for (int mx = 0; mx < ROW; mx++) {
                        const T t = sq[0][mx] + syz;
                        const int key = order_key(t);
                        st.template push<FLIP>((mx == M && crow ? central_ok : valid) && key <= g.key_rc, t, key, w);
                    }
                    st.service(Shape::LIMIT);
                }
            }
        }
    } else {
        T f[3];
#pragma unroll
        for (int x = 0; x < DIM; x++) d[x] = scale_kappa(g, d[x]);
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
            for (int k = 0; k < DIM; k++) {
                d[x] = fma(-f[k], g.a[3 * k + x], d[x]);
                if (sizeof(T) == 4) d[x] = fma(-f[k], g.a_lo[3 * k + x], d[x]);
            }
        }
        for (int m0 = 0; m0 < nimg; m0 += Shape::LIMIT) {
            const int m1 = min(m0 + Shape::LIMIT, nimg); /* uniform trip count: no work for images that do not exist */
#pragma unroll 4
            for (int m = m0; m < m1; m++) {
                const bool in = valid;
                T t = 0;
#pragma unroll
                for (int x = 0; x < DIM; x++) {
                    T v = d[x] - simg[3 * m + x];
                    if (sizeof(T) == 4) v -= simg[3 * (nimg + m) + x]; /* low parts follow the nimg high parts */
                    t = fma(v, v, t);
                }
                const int key = order_key(t);
                const bool tiny = in && key < g.key_min;
                if (tiny) direct += (double)((FLIP ? -w : w) * pair_f_direct(t));
                st.template push<FLIP>(in && !tiny && key <= g.key_rc, t, key, w);
            }
            if (list_service) st.service(Shape::LIMIT);
        }
    }
}

} // namespace ewald
