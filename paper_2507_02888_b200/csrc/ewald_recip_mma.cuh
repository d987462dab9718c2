/* ewald_recip_mma.cuh -- [S1-S4] FP64 reciprocal-space energy, octant form on the FP64 tensor cores.
 *
 * The octant sums of ewald_recip_oct.cuh,
 *     T[d][c] = sum_i X1_d(i) P_c(i),   X1_d = the doubles (q cos, q sin)(2 pi n1 s_i1) of Eq. 8,
 *     P_c = the products t(2 pi n2 s_i2) t(2 pi n3 s_i3) of column c,
 * are a dense contraction over the particles i: M = the n1 entries, N = the products, K = the particles.  The
 * FMA-pipe form of it is bound by shared memory -- a value every lane needs costs one LDS wavefront per 8
 * bytes, 24 to 35 wavefronts per 64 DFMAs (profiles/r02_recip_summary.md) -- so the FP64 path issues it as
 * m8n8k4 DMMAs (same peak as the DFMA pipe on B200, measured 37.0 TFLOP/s for both): every operand is a
 * lane-private register filled by a conflict-free LDS, and one instruction does 256 FMAs.
 *
 *   quad   4 consecutive particles = the K of one DMMA; the table of a chunk of particles is stored
 *          [walker][quad][entry][particle in quad] as (cos, sin) pairs, entries X1[0..] (times q), X2[0..], X3[0..]
 *   A      X1 doubles 8t..8t+7 (M-tile t = n1 in 4t..4t+3; double 1 = q sin 0 = 0 pads tile 0) of the quad:
 *          lane (row = lane / 4, k = lane % 4) loads one double
 *   B      products of 8 columns for the quad: lane (k = lane % 4, column = lane / 4) loads the pairs X2[n2], X3[n3]
 *          of its column and particle (two LDS.128) and forms the four products cc, cs, sc, ss = four B operands
 *          (HALF columns -- n2 = 0 or n3 = 0, all columns in 2D -- have two products: a slot takes two groups)
 *   slot   what a warp accumulates: (8 columns x 4 products) x (2 M-tiles) = 8 accumulator fragments
 *   warp   up to MMA_SMAX slots of ONE walker sharing their M-tiles: per quad 2 + 2 S loads, 4 S DMULs, 8 S DMMAs
 *   CTA    MMA_WARPS warps = nw walkers x wpw warps; a CTA runs its walkers in passes so that the grid is one wave
 */
#pragma once
#include "ewald_kernels_common.cuh"

namespace ewald {

constexpr int MMA_KIND_FULL = 0, MMA_KIND_PAIR = 1, MMA_KIND_EMPTY = 2; /* = OCT_FULL, OCT_PAIR, OCT_EMPTY */
constexpr int MMA_S = 3;        /* = MMA_SMAX of ewald_internal.h */
constexpr int MMA_THREADS = 384;
constexpr int MMA_CTAS_PER_SM = 1;  /* two CTAs of 6 warps per SM were measured slower (config 2: 99 vs 89 us) */
constexpr int MMA_MAX_PASS = 16;

struct MmaPassDev {
    int first, nw, wpw;         /* walkers [first, first + nw) of the CTA's set, wpw warps each */
    const int2 *lane;           /* [wpw][MMA_S][32] operand offsets (pairs within a quad block) */
    const int4 *meta;           /* [wpw][MMA_S] kind, first M-tile of the warp's window, tile mask, slot */
};

struct MmaArgs {
    const double *pos;          /* [W][DIM][npad] */
    const double *q;            /* [n] */
    int n, npad, n_walkers;
    int walkers_per_cta;        /* the CTA's walker set: [blockIdx.x * walkers_per_cta, + walkers_per_cta) */
    int n_pass;
    MmaPassDev pass[MMA_MAX_PASS];
    int pc;                     /* particles per chunk (multiple of 32) */
    int rowlen, qstride, wstride; /* pairs: entries per row, quad block (4 rowlen), walker slab */
    int off[3], nmax[3];
    int n_slots;                /* slots per walker (the plan may split a two-tile slot into two entries) */
    const double *wt;           /* [n_slots][2][4][8][4] */
    const double *tion;         /* [n_slots][2][8][8][4] or null */
    double *e_recip;            /* [W] */
    double binv[9];
};

__device__ __forceinline__ void dmma8x8x4(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

/* [S1,S2] One task = (walker, block of 32 particles, axis): phase seed by sincospi, powers by recurrence, stored
 * quad-interleaved.  Particles beyond n inside the last quad get q = 0 (their X1 row is zero). */
template <int DIM>
__device__ __forceinline__ void mma_build_rows(const MmaArgs &A, double2 *tab, int w0, int nw, int base_p, int cnt,
                                               int warp, int n_warps, int lane)
{
    const int blocks = (cnt + 31) >> 5, n_tasks = nw * blocks * DIM;
    const int cnt4 = (cnt + 3) & ~3;
    for (int t = warp; t < n_tasks; t += n_warps) {
        const int k = t % DIM, r = t / DIM, blk = r % blocks, wl = r / blocks;
        const int p = blk * 32 + lane;
        if (p >= cnt4 || w0 + wl >= A.n_walkers) continue;
        const bool real_p = p < cnt;
        const double *pw = A.pos + (size_t)(w0 + wl) * DIM * A.npad + base_p + p;
        double s = 0;
#pragma unroll
        for (int c = 0; c < DIM; c++) s += (real_p ? __ldg(pw + c * A.npad) : 0.0) * A.binv[3 * k + c];
        s -= rint(s);
        double sn, cs;
        sincospi(2 * s, &sn, &cs);
        double2 e;
        e.x = k == 0 ? (real_p ? __ldg(A.q + base_p + p) : 0.0) : 1.0; /* the first axis carries q */
        e.y = 0;
        double2 *row = tab + (size_t)wl * A.wstride + (size_t)(p >> 2) * A.qstride + (size_t)A.off[k] * 4 + (p & 3);
        row[0] = e;
        const int nm = A.nmax[k];
        for (int n = 1; n <= nm; n++) {
            double2 f;
            f.x = e.x * cs - e.y * sn;
            f.y = e.x * sn + e.y * cs;
            e = f;
            row[n * 4] = f;
        }
    }
}

/* [S3] One chunk of particles for one warp with NS slots: all operand loads of a quad are issued before its
 * first DMMA (no branch inside: a slot that uses one M-tile only has its other DMMAs predicated off). */
template <int DIM, int NS>
__device__ __forceinline__ void mma_chunk(double (&acc)[MMA_S][4][2][2], const double2 *tw, int nq, int qstride,
                                          int oA0, int oA1, const int2 (&lo)[MMA_S], const bool (&full)[MMA_S],
                                          const bool (&use0)[MMA_S], const bool (&use1)[MMA_S])
{
#pragma unroll 2 /* 1: measured 2 % slower */
    for (int q = 0; q < nq; q++) {
        const double2 *qb = tw + (size_t)q * qstride;
        const double *qd = reinterpret_cast<const double *>(qb);
        const double a0 = qd[oA0], a1 = qd[oA1];
        double2 a[NS], b[NS];
#pragma unroll
        for (int s = 0; s < NS; s++) { a[s] = qb[lo[s].x]; b[s] = qb[lo[s].y]; }
#pragma unroll
        for (int s = 0; s < NS; s++) {
            double pr[4];
            if (DIM == 3) { /* FULL: the four products; PAIR: the two pairs as they are */
                pr[0] = full[s] ? a[s].x * b[s].x : a[s].x; pr[1] = full[s] ? a[s].x * b[s].y : a[s].y;
                pr[2] = full[s] ? a[s].y * b[s].x : b[s].x; pr[3] = full[s] ? a[s].y * b[s].y : b[s].y;
            } else { pr[0] = a[s].x; pr[1] = a[s].y; pr[2] = b[s].x; pr[3] = b[s].y; }
            if (use0[s]) {
#pragma unroll
                for (int t = 0; t < 4; t++) dmma8x8x4(acc[s][t][0][0], acc[s][t][0][1], a0, pr[t]);
            }
            if (use1[s]) {
#pragma unroll
                for (int t = 0; t < 4; t++) dmma8x8x4(acc[s][t][1][0], acc[s][t][1][1], a1, pr[t]);
            }
        }
    }
}

template <int DIM>
__device__ __forceinline__ void mma_chunk_ns(int ns, double (&acc)[MMA_S][4][2][2], const double2 *tw, int nq, int qstride,
                                             int oA0, int oA1, const int2 (&lo)[MMA_S], const bool (&full)[MMA_S],
                                             const bool (&use0)[MMA_S], const bool (&use1)[MMA_S])
{
    if (ns == 3) mma_chunk<DIM, 3>(acc, tw, nq, qstride, oA0, oA1, lo, full, use0, use1);
    else if (ns == 2) mma_chunk<DIM, 2>(acc, tw, nq, qstride, oA0, oA1, lo, full, use0, use1);
    else if (ns == 1) mma_chunk<DIM, 1>(acc, tw, nq, qstride, oA0, oA1, lo, full, use0, use1);
}

template <int DIM>
__global__ void __launch_bounds__(MMA_THREADS, MMA_CTAS_PER_SM) recip_mma_kernel(MmaArgs A, int nw_max)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const size_t buf_pairs = (size_t)nw_max * A.wstride;
    double2 *tab0 = reinterpret_cast<double2 *>(smem_raw);
    double *part = reinterpret_cast<double *>(tab0 + 2 * buf_pairs); /* [nw_max][n_slots][2] sums per slot and tile */
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, n_warps = blockDim.x >> 5;
    const int r = lane >> 2, kk = lane & 3;

    for (int pass = 0; pass < A.n_pass; pass++) {
        const MmaPassDev P = A.pass[pass];
        const int w0 = blockIdx.x * A.walkers_per_cta + P.first;
        if (w0 >= A.n_walkers) break; /* uniform over the CTA */
        const int nw = min(P.nw, A.n_walkers - w0);
        const int wl = warp / P.wpw, j = warp - wl * P.wpw;
        const bool active = wl < nw;

        /* slots of this warp: the first ns entries; meta = kind, first M-tile of the WARP's window, tile mask
         * within the window (bit 0: tile t0, bit 1: tile t0 + 1), slot index */
        int kind[MMA_S], slot[MMA_S], st0[MMA_S];
        bool full[MMA_S], use0[MMA_S], use1[MMA_S];
        int2 lo[MMA_S];
        int t0 = 0, ns = 0;
#pragma unroll
        for (int s = 0; s < MMA_S; s++) {
            const int4 m = active ? P.meta[j * MMA_S + s] : make_int4(MMA_KIND_EMPTY, 0, 0, 0);
            kind[s] = m.x; slot[s] = m.w & 0xffff; st0[s] = m.y - (m.w >> 16); /* window tile 0 = tile st0 of the slot's tables */
            full[s] = m.x == MMA_KIND_FULL; use0[s] = (m.z & 1) != 0; use1[s] = (m.z & 2) != 0;
            if (m.x != MMA_KIND_EMPTY) { t0 = m.y; ns = s + 1; }
            lo[s] = P.lane[(j * MMA_S + s) * 32 + lane];
        }
        /* this lane's X1 doubles (A operands) of M-tiles t0 and t0 + 1, as double offsets within a quad block
         * (tile t0 + 1 may lie beyond n1_max: its doubles are then other entries of the row, their weights zero) */
        const int d0 = 8 * t0 + r, d1 = d0 + 8;
        const int oA0 = ((A.off[0] + (d0 >> 1)) * 4 + kk) * 2 + (d0 & 1), oA1 = ((A.off[0] + (d1 >> 1)) * 4 + kk) * 2 + (d1 & 1);

        double acc[MMA_S][4][2][2];
#pragma unroll
        for (int s = 0; s < MMA_S; s++)
#pragma unroll
            for (int t = 0; t < 4; t++) { acc[s][t][0][0] = acc[s][t][0][1] = acc[s][t][1][0] = acc[s][t][1][1] = 0; }

        for (int t = tid; t < nw_max * 2 * A.n_slots; t += blockDim.x) part[t] = 0;
        mma_build_rows<DIM>(A, tab0, w0, nw, 0, min(A.pc, A.n), warp, n_warps, lane);
        __syncthreads();
        int it = 0;
        for (int base_p = 0; base_p < A.n; base_p += A.pc, it++) {
            const int cnt = min(A.pc, A.n - base_p);
            const bool more = base_p + A.pc < A.n;
            double2 *next = tab0 + (size_t)((it + 1) & 1) * buf_pairs;
            /* The table code is latency-bound (global loads, sincospi, a recurrence) and hardly uses the FP64 pipe:
             * of the three warps of a sub-partition one builds its share of the next chunk's tables before its
             * DMMAs, one half-way through and one after them, so that two warps always feed the tensor pipe. */
            const int phase = (warp >> 2) % 3;
            const int next_cnt = more ? min(A.pc, A.n - base_p - A.pc) : 0;
            const double2 *tw = tab0 + (size_t)(it & 1) * buf_pairs + (size_t)wl * A.wstride;
            const int nq = (cnt + 3) >> 2, nq0 = phase == 0 ? 0 : phase == 1 ? nq >> 1 : nq;
            if (active && nq0 > 0) mma_chunk_ns<DIM>(ns, acc, tw, nq0, A.qstride, oA0, oA1, lo, full, use0, use1);
            if (more) mma_build_rows<DIM>(A, next, w0, nw, base_p + A.pc, next_cnt, warp, n_warps, lane);
            if (active && nq0 < nq)
                mma_chunk_ns<DIM>(ns, acc, tw + (size_t)nq0 * A.qstride, nq - nq0, A.qstride, oA0, oA1, lo, full, use0, use1);
            __syncthreads();
        }

        /* [S4] E_recip = sum over octant points and sign classes of W |rho|^2, in FP64.  An accumulator fragment
         * holds, for rows d = lane / 4 (X1 double 8 tile + d: even = cos, odd = sin of n1 = 4 tile + d / 2) and
         * columns 2 (lane % 4) + {0, 1}, the sums T of the four products.  The lanes d and d ^ 1 swap one column
         * each, so that the even lane holds (T_cos, T_sin) of column 2 (lane % 4) and the odd lane of the next.
         * FULL (products k: 0 = c2 c3, 1 = c2 s3, 2 = s2 c3, 3 = s2 s3), classes (p, q) = signs of n2, n3:
         *   Re rho = T_c0 - p T_s2 - q T_s1 - pq T_c3,   Im rho = T_s0 + p T_c2 + q T_c1 - pq T_s3;
         * PAIR (k = 0,1: cos, sin of half column A; k = 2,3: of B), classes = sign of the half column's n:
         *   Re rho = T_c(o) - p T_s(o+1),   Im rho = T_s(o) + p T_c(o+1). */
        if (active) {
            const int odd = r & 1, col = 2 * kk + odd, n1l = r >> 1;
#pragma unroll
            for (int s = 0; s < MMA_S; s++) {
                if (kind[s] == MMA_KIND_EMPTY) continue;
                const double *wt = A.wt + (size_t)slot[s] * 256;
                const double *ti = A.tion ? A.tion + (size_t)slot[s] * 512 : nullptr;
#pragma unroll
                for (int tile = 0; tile < 2; tile++) {
                    if (!(tile ? use1[s] : use0[s])) continue;
                    const int st = st0[s] + tile; /* tile index within the slot's own tables (0 or 1) */
                    double wk[4], t0v[4], t1v[4];
#pragma unroll
                    for (int cls = 0; cls < 4; cls++) wk[cls] = __ldg(wt + ((st * 4 + n1l) * 8 + col) * 4 + cls);
#pragma unroll
                    for (int k = 0; k < 4; k++) {
                        t0v[k] = ti ? __ldg(ti + ((st * 8 + r) * 8 + 2 * kk) * 4 + k) : 0.0;
                        t1v[k] = ti ? __ldg(ti + ((st * 8 + r) * 8 + 2 * kk + 1) * 4 + k) : 0.0;
                    }
                    double e = 0;
                    double Tc[4], Ts[4];
#pragma unroll
                    for (int k = 0; k < 4; k++) {
                        const double own0 = acc[s][k][tile][0] + t0v[k], own1 = acc[s][k][tile][1] + t1v[k];
                        const double recv = __shfl_xor_sync(0xffffffffu, odd ? own0 : own1, 4);
                        Tc[k] = odd ? recv : own0;
                        Ts[k] = odd ? own1 : recv;
                    }
#pragma unroll
                    for (int cls = 0; cls < 4; cls++) {
                        double re, im;
                        if (DIM == 3 && kind[s] == MMA_KIND_FULL) {
                            const double p = (cls & 2) ? -1.0 : 1.0, q = (cls & 1) ? -1.0 : 1.0;
                            re = Tc[0] - p * Ts[2] - q * Ts[1] - p * q * Tc[3];
                            im = Ts[0] + p * Tc[2] + q * Tc[1] - p * q * Ts[3];
                        } else {
                            const int o = cls & 2;
                            const double p = (cls & 1) ? -1.0 : 1.0;
                            re = Tc[o] - p * Ts[o + 1];
                            im = Ts[o] + p * Tc[o + 1];
                        }
                        e += wk[cls] != 0 ? wk[cls] * (re * re + im * im) : 0.0;
                    }
                    /* one sum per (slot, tile): the same lanes in the same order whichever warp holds it */
                    e = warp_sum(e);
                    if (lane == 0) part[wl * 2 * A.n_slots + 2 * slot[s] + st] = e;
                }
            }
        }
        __syncthreads();
        if (tid < nw) { /* the slots in plan order: independent of the walker's place in the batch and of the pass shape */
            double sum = 0;
            for (int si = 0; si < 2 * A.n_slots; si++) sum += part[tid * 2 * A.n_slots + si];
            A.e_recip[w0 + tid] = sum;
        }
        __syncthreads();
    }
}

/* FP64 tensor-core probe: 32 independent m8n8k4 DMMAs per warp and round (the roofline denominator of
 * recip_mma_kernel; on B200 it equals the DFMA-chain peak of fma_probe_kernel). */
__global__ void __launch_bounds__(256) dmma_probe_kernel(int iters, const double *in, double *sink)
{
    double c[8][2], a[4], b[4];
#pragma unroll
    for (int u = 0; u < 8; u++) { c[u][0] = 0; c[u][1] = 0; }
#pragma unroll
    for (int u = 0; u < 4; u++) { a[u] = in[u] + threadIdx.x; b[u] = in[u + 4] + 1; }
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int u = 0; u < 8; u++) dmma8x8x4(c[u][0], c[u][1], a[(u + r) & 3], b[u & 3]);
    }
    double s = 0;
#pragma unroll
    for (int u = 0; u < 8; u++) s += c[u][0] + c[u][1];
    if (s == 123456789.0) sink[0] = s;
}

} // namespace ewald
