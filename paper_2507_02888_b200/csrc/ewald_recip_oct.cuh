/* ewald_recip_oct.cuh -- [S1-S4] reciprocal-space energy in the octant (real-product) form.
 *
 * In any cell G.r = 2 pi sum_k n_k s_k (s = fractional coordinates) and Eq. 8
 * factorises exp(iG.r) into per-axis powers.  Taking real and imaginary parts per axis,
 * the eight real sums over particles
 *     T_abc(n) = sum_i q_i t^a(2 pi n1 s_i1) t^b(2 pi n2 s_i2) t^c(2 pi n3 s_i3),  t in {cos, sin}, n_k >= 0
 * give rho(+-n1, +-n2, +-n3) for all sign choices, and summing |rho|^2 over the sign choices leaves
 *     E_recip = sum_{n >= 0, n != 0} w(G_n) 2^{nz(n)} sum_abc T_abc(n)^2
 * (nz = number of non-zero n_k; every cross term cancels) when the reciprocal axes are orthogonal; else the
 * four sign classes of an octant point carry their own weights (S4 below, ewald_octplan.cpp).  One real FMA
 * per (particle, G of the full sphere): the algorithmic count 2 N N_G flops per walker, half of the complex half-set form.
 *
 * Work decomposition (host plan, ewald_octplan.cpp):
 *   row    per (walker, particle): the "powers ... computed and buffered" of PAPER.md:157, in shared
 *          memory as (cos, sin) pairs: X1[n = 0..] (times q_i), X2[n = 0..], X3[n = 0..]
 *   item   a block of <= NPB consecutive n1 (plus n1 = 0 in the first block) of either one column
 *          (n2 > 0, n3 > 0) with its four products X2 (x) X3 [FULL], or two half columns ((n2, 0), (0, n3),
 *          (0, 0); in 2D any n2) with their two products each [PAIR]: no product that is identically zero
 *   lane   owns one (walker, item) for the whole kernel: 4 products (unique per lane) times the X1 pairs of
 *          the block (one broadcast LDS.128 per pair) -> 4 x (1 + 2 NP) register accumulators.  The loop is
 *          software-pipelined by hand: the pairs of particle p + 1 are loaded while those of p are multiplied
 *          (a DFMA needs its LDS operand 30 cycles after issue; with one product held in the operand reuse
 *          cache a DFMA reads two register operands and issues every 2 cycles, profiles/r02_recip_summary.md)
 *   warp   32 lanes of one kind and block length: the items of all walkers of the CTA are sorted, so the
 *          spherical cut-off costs no divergent lanes; warps are dealt to the four sub-partitions (warp mod 4)
 *          so that each carries the same number of FP64 operations
 */
#pragma once
#include "ewald_kernels_common.cuh"

namespace ewald {

constexpr int OCT_KIND_FULL = 0, OCT_KIND_PAIR = 1, OCT_KIND_EMPTY = 2; /* = OCT_FULL, ... of ewald_internal.h */

template <typename T> struct OctArgs {
    const T *pos;       /* [W][DIM][npad] */
    const T *q;         /* [n] */
    int n, npad, n_walkers;
    int wc;             /* walkers per CTA */
    int n_slabs;        /* CTAs per walker group: the warp list is dealt to n_slabs CTAs */
    int pc;             /* particles per chunk */
    int rank_stride;    /* most lanes any walker has in one CTA */
    int rowlen;         /* (cos,sin) pairs per (walker, particle) row */
    int wstride;        /* pairs per walker slab (pc * rowlen + bank stagger) */
    int off[3];         /* pair offset of X1, X2, X3 (each n = 0..) within a row */
    int nmax[3];
    const int4 *lane;   /* [n_slabs][blockDim.x] {local walker | rank << 8, item, offA | offB << 16, offX} */
    const int *variant; /* [n_slabs][n_warps] NP | C0 << 8 | kind << 16 */
    const double *wt;   /* [n_items][1 + NPB][4]: class weights per entry (ewald_octplan.cpp) */
    const double *tion; /* [n_items][1 + 2 NPB][4] fixed-charge sums, or null */
    double *e_recip;    /* [W][n_slabs] */
    double binv[9];     /* FP64 also in the FP32 kernels: the reduction of s to one period is done in FP64 */
};

/* Threads per CTA the register file allows: 4 (1 + 2 NPB) accumulators per lane (doubles take two registers
 * each) plus the prefetched pairs of the next particle. */
#ifndef EWALD_OCT_THREADS64
#define EWALD_OCT_THREADS64 384
#endif
#ifndef EWALD_OCT_THREADS32
#define EWALD_OCT_THREADS32 512
#endif
template <typename T, int NPB> struct OctCfg {
    static constexpr int MAX_THREADS = sizeof(T) == 8 ? EWALD_OCT_THREADS64 : EWALD_OCT_THREADS32;
    /* registers per thread when MAX_THREADS are resident: 64 K registers, allocated 8 at a time per thread */
    static constexpr int MAX_REGS = (65536 / MAX_THREADS) / 8 * 8 > 255 ? 255 : (65536 / MAX_THREADS) / 8 * 8;
};

/* (lo, hi) += p * (c.x, c.y).  FP32: one packed FFMA2 (sm_100: two FMAs per issue slot; the FP32 tile is bound by
 * issue slots, measured +30 % over scalar FFMAs), FP64: two DFMAs. */
__device__ __forceinline__ void oct_fma_pair(double p, double2 c, double &lo, double &hi)
{
    lo = fma(p, c.x, lo);
    hi = fma(p, c.y, hi);
}
__device__ __forceinline__ void oct_fma_pair(float p, float2 c, float &lo, float &hi)
{
    const float2 r = __ffma2_rn(make_float2(p, p), c, make_float2(lo, hi));
    lo = r.x;
    hi = r.y;
}

/* Prefetch distance of the pipelined loop in (cos, sin) pairs: the pairs of a particle form a sequence of
 * LEN = NP + C0 entries; a ring of D registers pairs holds the next D of them, D a divisor of LEN so that the
 * ring is in the same state at the start of every particle.  D = 4 pairs = 32 DFMAs ahead of use. */
__host__ __device__ constexpr int oct_ring(int len)
{
    return len <= 5 ? (len < 1 ? 1 : len) : len % 4 == 0 ? 4 : len % 3 == 0 ? 3 : len;
}

/* One chunk of particles for one lane: acc[k][e] += p_k * X1_e, software-pipelined over the particles. */
template <typename T, int NPB, int NP, bool C0, int KIND>
__device__ __forceinline__ void oct_fma(T (&acc)[4][1 + 2 * NPB], const typename Num<T>::T2 *rA,
                                        const typename Num<T>::T2 *rB, const typename Num<T>::T2 *rX,
                                        int cnt, int rowlen)
{
    typedef typename Num<T>::T2 T2;
    constexpr int FIRST = C0 ? 0 : 1, LEN = NP + 1 - FIRST, D = oct_ring(LEN);
    if (LEN == 0) return;
    T2 a = *rA, b = *rB, ring[D];
#pragma unroll
    for (int i = 0; i < D; i++) ring[i] = rX[FIRST + i];
    for (int p = 0; p < cnt; p++) {
        /* the row after the chunk's last one is read but never used: the buffers carry a row of slack */
        T pr[4];
        if (KIND == OCT_KIND_FULL) { pr[0] = a.x * b.x; pr[1] = a.x * b.y; pr[2] = a.y * b.x; pr[3] = a.y * b.y; }
        else { pr[0] = a.x; pr[1] = a.y; pr[2] = b.x; pr[3] = b.y; }
        rA += rowlen; rB += rowlen;
        a = *rA; b = *rB;
#pragma unroll
        for (int i = 0; i < LEN; i++) {
            const int j = FIRST + i;               /* pair index: n1 = block start + j; j = 0 is X1[0] = (q, 0) */
            const T2 c = ring[i % D];
            ring[i % D] = i + D < LEN ? rX[j + D] : rX[rowlen + j + D - LEN];
            if (j == 0) {
#pragma unroll
                for (int k = 0; k < 4; k++) acc[k][0] = fma(pr[k], c.x, acc[k][0]);
            } else {
#pragma unroll
                for (int k = 0; k < 4; k++) oct_fma_pair(pr[k], c, acc[k][2 * j - 1], acc[k][2 * j]);
            }
        }
        rX += rowlen;
    }
}

template <typename T, int NPB, int KIND, int NP>
__device__ __forceinline__ void oct_dispatch_c0(T (&acc)[4][1 + 2 * NPB], bool c0,
                                                const typename Num<T>::T2 *rA, const typename Num<T>::T2 *rB,
                                                const typename Num<T>::T2 *rX, int cnt, int rowlen)
{
    if (c0) oct_fma<T, NPB, NP, true, KIND>(acc, rA, rB, rX, cnt, rowlen);
    else oct_fma<T, NPB, NP, false, KIND>(acc, rA, rB, rX, cnt, rowlen);
}

template <typename T, int NPB, int KIND>
__device__ __forceinline__ void oct_dispatch_np(T (&acc)[4][1 + 2 * NPB], int np, bool c0,
                                                const typename Num<T>::T2 *rA, const typename Num<T>::T2 *rB,
                                                const typename Num<T>::T2 *rX, int cnt, int rowlen)
{
    switch (np) {
#define EWALD_OCT_CASE(NP)                                                                              \
    case NP:                                                                                            \
        if (NP <= NPB) oct_dispatch_c0<T, NPB, KIND, (NP <= NPB ? NP : 0)>(acc, c0, rA, rB, rX, cnt, rowlen); \
        break;
        EWALD_OCT_CASE(0) EWALD_OCT_CASE(1) EWALD_OCT_CASE(2) EWALD_OCT_CASE(3)
        EWALD_OCT_CASE(4) EWALD_OCT_CASE(5) EWALD_OCT_CASE(6) EWALD_OCT_CASE(7)
#undef EWALD_OCT_CASE
    default: break;
    }
}

/* [S1,S2] Phase seeds and power rows of one chunk of particles, for all walkers of the CTA.  A task is one
 * (local walker, particle): the lane builds the rows of all DIM axes together (DIM independent dependency
 * chains: sincospi, then the recurrence).  Tasks are handed out 32 at a time from a shared counter, so warps
 * whose FMA lists are short build most of the next chunk's tables while the long ones still multiply. */
template <typename T, int DIM>
__device__ __forceinline__ void oct_build_rows(const OctArgs<T> &A, typename Num<T>::T2 *tab, int *counter, int w0,
                                               int base_p, int cnt, int lane)
{
    typedef typename Num<T>::T2 T2;
    const int per_walker = (cnt + 31) & ~31;          /* tasks of one walker, padded to whole warps */
    const int n_tasks = A.wc * per_walker;
    int nmax_all = A.nmax[0];
#pragma unroll
    for (int k = 1; k < DIM; k++) nmax_all = max(nmax_all, A.nmax[k]);
    for (;;) {
        int t0 = 0;
        if (lane == 0) t0 = atomicAdd(counter, 32);
        t0 = __shfl_sync(0xffffffffu, t0, 0);
        if (t0 >= n_tasks) break;
        const int wl = t0 / per_walker, p = t0 - wl * per_walker + lane;
        if (p >= cnt || w0 + wl >= A.n_walkers) continue;
        const T *pw = A.pos + (size_t)(w0 + wl) * DIM * A.npad + base_p + p;
        T x[DIM];
#pragma unroll
        for (int k = 0; k < DIM; k++) x[k] = __ldg(pw + k * A.npad);
        const T qp = __ldg(A.q + base_p + p);
        T sn[DIM], cs[DIM];
        T2 e[DIM];
        T2 *row[DIM];
#pragma unroll
        for (int k = 0; k < DIM; k++) {
            double s = 0;
#pragma unroll
            for (int c = 0; c < DIM; c++) s += (double)x[c] * A.binv[3 * k + c];
            s -= rint(s);
            Num<T>::sincospi_((T)(2 * s), &sn[k], &cs[k]);
            row[k] = tab + (size_t)wl * A.wstride + (size_t)p * A.rowlen + A.off[k];
            e[k].x = k == 0 ? qp : T(1); e[k].y = 0; /* the first axis carries q: X1[0] = (q, 0) */
            row[k][0] = e[k];
        }
        for (int n = 1; n <= nmax_all; n++) {
#pragma unroll
            for (int k = 0; k < DIM; k++) {
                T2 f;
                f.x = e[k].x * cs[k] - e[k].y * sn[k];
                f.y = e[k].x * sn[k] + e[k].y * cs[k];
                e[k] = f;
                if (n <= A.nmax[k]) row[k][n] = f;
            }
        }
    }
}

template <typename T, int DIM, int NPB>
__global__ void __maxnreg__((OctCfg<T, NPB>::MAX_REGS)) recip_oct_kernel(OctArgs<T> A)
{
    typedef typename Num<T>::T2 T2;
    constexpr int NE = 1 + 2 * NPB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    /* two table buffers [wc][wstride] plus a row of slack (the pipelined loop reads one row ahead), then the
     * per-lane partial sums */
    const size_t buf_pairs = (size_t)A.wc * A.wstride + A.rowlen;
    T2 *tab0 = reinterpret_cast<T2 *>(smem_raw);
    double *part = reinterpret_cast<double *>(tab0 + 2 * buf_pairs); /* [wc][rank_stride] lane sums by rank */
    __shared__ int counter[2];

    const int tid = threadIdx.x, nthreads = blockDim.x, warp = tid >> 5, lane = tid & 31;
    const int group = blockIdx.x / A.n_slabs, slab = blockIdx.x - group * A.n_slabs;
    const int w0 = group * A.wc;
    int4 L = A.lane[(size_t)slab * nthreads + tid];
    const int rank = (int)((unsigned)L.x >> 8);
    L.x &= 255;
    const int var = A.variant[slab * (nthreads >> 5) + warp];
    const int np = var & 255, kind = var >> 16;
    const bool c0 = ((var >> 8) & 255) != 0;
    if (tid < 2) counter[tid] = 0;

    T acc[4][NE];
#pragma unroll
    for (int k = 0; k < 4; k++)
#pragma unroll
        for (int e = 0; e < NE; e++) acc[k][e] = 0;

    __syncthreads();
    oct_build_rows<T, DIM>(A, tab0, &counter[1], w0, 0, min(A.pc, A.n), lane);
    __syncthreads();
    int it = 0;
    for (int base_p = 0; base_p < A.n; base_p += A.pc, it++) {
        const int cnt = min(A.pc, A.n - base_p);
        const T2 *tab = tab0 + (size_t)(it & 1) * buf_pairs;
        if (tid == 0) counter[(it + 1) & 1] = 0; /* last used before the barrier that ended the previous pass */
        const T2 *lane_base = tab + (size_t)L.x * A.wstride;
        const T2 *baseA = lane_base + (L.z & 0xffff), *baseB = lane_base + (L.z >> 16), *baseX = lane_base + L.w;
        /* [S3] */
        if (DIM == 3 && kind == OCT_KIND_FULL) oct_dispatch_np<T, NPB, OCT_KIND_FULL>(acc, np, c0, baseA, baseB, baseX, cnt, A.rowlen);
        else if (kind == OCT_KIND_PAIR) oct_dispatch_np<T, NPB, OCT_KIND_PAIR>(acc, np, c0, baseA, baseB, baseX, cnt, A.rowlen);
        /* the next chunk's tables go to the other buffer (read last in the previous pass) */
        if (base_p + A.pc < A.n)
            oct_build_rows<T, DIM>(A, tab0 + (size_t)((it + 1) & 1) * buf_pairs, &counter[it & 1], w0, base_p + A.pc,
                                   min(A.pc, A.n - base_p - A.pc), lane);
        __syncthreads();
    }

    /* [S4] E_recip = sum_n sum_classes W(n) |rho(n)|^2 in FP64.  FULL items (products k: 0 = c2 c3, 1 = c2 s3,
     * 2 = s2 c3, 3 = s2 s3; c = cos, s = sin along axes 1, 2, 3), classes (p, q) = signs of n2, n3 relative to n1:
     *   Re rho_pq = T_ccc - p T_ssc - q T_scs - pq T_css,   Im rho_pq = T_scc + p T_csc + q T_ccs - pq T_sss;
     * PAIR items (k = 0,1: cos, sin of half column A; k = 2,3: of B), classes p = sign of the half column's n:
     *   Re rho_p = T_cc - p T_ss,   Im rho_p = T_sc + p T_cs.
     * For orthogonal reciprocal axes the class weights are equal and the sum is W sum_abc T_abc^2.
     * Entries of weight zero are padding (never read as values). */
    double e = 0;
    if (kind != OCT_KIND_EMPTY) {
        const double *wt = A.wt + (size_t)L.y * (NPB + 1) * 4;
        const double *ti = A.tion ? A.tion + (size_t)L.y * NE * 4 : nullptr;
#pragma unroll
        for (int j = 0; j <= NPB; j++) {
            double Tc[4], Ts[4];
#pragma unroll
            for (int k = 0; k < 4; k++) {
                if (j == 0) {
                    Tc[k] = (double)acc[k][0]; Ts[k] = 0;
                    if (ti) Tc[k] += ti[k];
                } else {
                    Tc[k] = (double)acc[k][2 * j - 1]; Ts[k] = (double)acc[k][2 * j];
                    if (ti) { Tc[k] += ti[(2 * j - 1) * 4 + k]; Ts[k] += ti[(2 * j) * 4 + k]; }
                }
            }
#pragma unroll
            for (int cls = 0; cls < 4; cls++) {
                const double wk = wt[4 * j + cls];
                double re, im;
                if (DIM == 3 && kind == OCT_KIND_FULL) {
                    const double p = (cls & 2) ? -1.0 : 1.0, q = (cls & 1) ? -1.0 : 1.0;
                    re = Tc[0] - p * Ts[2] - q * Ts[1] - p * q * Tc[3];
                    im = Ts[0] + p * Tc[2] + q * Tc[1] - p * q * Ts[3];
                } else {
                    const int o = cls & 2;
                    const double p = (cls & 1) ? -1.0 : 1.0;
                    re = Tc[o] - p * Ts[o + 1];
                    im = Ts[o] + p * Tc[o + 1];
                }
                e += wk != 0 ? wk * (re * re + im * im) : 0.0;
            }
        }
    }
    for (int t = tid; t < A.wc * A.rank_stride; t += nthreads) part[t] = 0;
    __syncthreads();
    if (rank != 0xffffff) part[L.x * A.rank_stride + rank] = e;
    __syncthreads();
    /* one warp per walker adds that walker's lane sums in rank order: deterministic, and independent of
     * the walker's place in the batch */
    for (int wl = warp; wl < A.wc; wl += nthreads >> 5) {
        double sum = 0;
        for (int t = lane; t < A.rank_stride; t += 32) sum += part[wl * A.rank_stride + t];
        sum = warp_sum(sum);
        if (lane == 0 && w0 + wl < A.n_walkers) A.e_recip[(size_t)(w0 + wl) * A.n_slabs + slab] = sum;
    }
}

} // namespace ewald
