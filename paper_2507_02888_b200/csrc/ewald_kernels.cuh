/* ewald_kernels.cuh -- device code of the B200 Ewald library (sm_100a).
 *
 * Kernels (SURVEY.md section 8(a) step names in brackets):
 *   recip_kernel   [S1-S4]  complex half-set form: phase seeds exp(2 pi i s_k) by sincospi, power tables by
 *                           complex recurrence in shared memory (Eq. 8: "powers of these
 *                           exponentials are computed and buffered"), rho(G) on the half set,
 *                           E_recip = sum_{G+} 2 w(G) |rho(G)|^2; stores rho(G) for ewald_load_walkers.
 *                           (The energy path uses recip_oct_kernel, ewald_recip_oct.cuh.)
 *   real_kernel    [S5]     sum_{i<j} q_i q_j sum_R erfc(kappa|r_ij-R|)/|r_ij-R| (real-lattice sum of
 *                           Eq. 3) plus mobile-ion pairs; machinery in ewald_realspace.cuh
 *   [S6] combine            folded into real_kernel: the last CTA of a walker adds the partial sums and the
 *                           constants of Eqs. 3-4; charge_sums_kernel (stored populations) gives
 *                           sum q^2, sum q and the all-equal flag of the mobile charges
 *   move_kernel    [S7a-d]  single-particle moves, one warp per move: Delta E and patch of the stored rho(G)
 *   fma_probe_kernel   measurement helper (roofline denominator); dmma_probe_kernel in ewald_recip_mma.cuh
 * The paper's version-2 loop structure (real-lattice loop || reciprocal-lattice loop, then a
 * combining loop) is kept as three kernels; everything inside them is new.
 */
#pragma once
#include "ewald_kernels_common.cuh"
#include "ewald_realspace.cuh"

namespace ewald {

/* ------------------------------------------------------------------------------------------ */
/* [S1-S4] rho(G) and E_recip.  grid = n_walkers * n_slabs; each thread owns GPT members of G+. */

template <typename T> struct RecipArgs {
    const T *pos;      /* [W][DIM][npad] */
    const T *q;        /* [n] */
    int n, npad;
    const short4 *gn;  /* [ngp] (n1,n2,n3,0) */
    const T *w2;       /* [ngp] */
    const T *ion_rho;  /* [ngp][2] or null */
    int ngp, ngp_pad;
    int nmax[3];
    int off[3], rowlen; /* table row: direction k starts at off[k] */
    T *rho_out;        /* [W][2][ngp_pad] or null */
    double *partial;   /* [W][n_slabs] */
    int n_slabs;
    double binv[9];    /* FP64 in both precisions: s is reduced to one period before it is rounded */
};

constexpr int RECIP_THREADS = 256;
constexpr int RECIP_GPT = 4;
constexpr int RECIP_CHUNK = 32;

template <typename T, int DIM>
__global__ void __launch_bounds__(RECIP_THREADS) recip_kernel(RecipArgs<T> A)
{
    typedef typename Num<T>::T2 T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T2 *tab = reinterpret_cast<T2 *>(smem_raw); /* [RECIP_CHUNK][rowlen] */
    __shared__ double red[32];

    const int w = blockIdx.x / A.n_slabs, slab = blockIdx.x - w * A.n_slabs, tid = threadIdx.x;
    const T *pw = A.pos + (size_t)w * DIM * A.npad;

    int gi[RECIP_GPT];
    int i1[RECIP_GPT], i2[RECIP_GPT], i3[RECIP_GPT];
    T sg2[RECIP_GPT], sg3[RECIP_GPT];
    T2 acc[RECIP_GPT];
#pragma unroll
    for (int u = 0; u < RECIP_GPT; u++) {
        int g = (slab * RECIP_GPT + u) * RECIP_THREADS + tid;
        gi[u] = g < A.ngp ? g : -1;
        short4 nn = A.gn[g < A.ngp ? g : 0];
        i1[u] = A.off[0] + nn.x;
        i2[u] = A.off[1] + (nn.y < 0 ? -nn.y : nn.y);
        i3[u] = DIM == 3 ? A.off[2] + (nn.z < 0 ? -nn.z : nn.z) : 0;
        sg2[u] = nn.y < 0 ? T(-1) : T(1);
        sg3[u] = nn.z < 0 ? T(-1) : T(1);
        acc[u].x = 0; acc[u].y = 0;
    }

    for (int base = 0; base < A.n; base += RECIP_CHUNK) {
        const int cnt = min(RECIP_CHUNK, A.n - base);
        __syncthreads();
        /* [S1,S2] one (particle, direction) per thread */
        for (int t = tid; t < cnt * DIM; t += RECIP_THREADS) {
            const int p = t / DIM, k = t - p * DIM;
            double s = 0;
#pragma unroll
            for (int x = 0; x < DIM; x++) s += (double)pw[x * A.npad + base + p] * A.binv[3 * k + x];
            power_row<T>((T)(s - rint(s)), k == 0 ? A.q[base + p] : T(1), A.nmax[k], tab + p * A.rowlen + A.off[k]);
        }
        __syncthreads();
        /* [S3] rho(G) += q e1^n1 e2^n2 e3^n3 */
        for (int p = 0; p < cnt; p++) {
            const T2 *row = tab + p * A.rowlen;
#pragma unroll
            for (int u = 0; u < RECIP_GPT; u++) {
                T2 e1 = row[i1[u]], e2 = row[i2[u]];
                e2.y *= sg2[u];
                T2 e12;
                e12.x = e1.x * e2.x - e1.y * e2.y;
                e12.y = e1.x * e2.y + e1.y * e2.x;
                if (DIM == 3) {
                    T2 e3 = row[i3[u]];
                    e3.y *= sg3[u];
                    acc[u].x += e12.x * e3.x - e12.y * e3.y;
                    acc[u].y += e12.x * e3.y + e12.y * e3.x;
                } else {
                    acc[u].x += e12.x;
                    acc[u].y += e12.y;
                }
            }
        }
    }

    /* [S4] */
    double e = 0;
#pragma unroll
    for (int u = 0; u < RECIP_GPT; u++) {
        if (gi[u] < 0) continue;
        T re = acc[u].x, im = acc[u].y;
        if (A.ion_rho) { re += A.ion_rho[2 * gi[u]]; im += A.ion_rho[2 * gi[u] + 1]; }
        if (A.rho_out) {
            T *ro = A.rho_out + (size_t)w * 2 * A.ngp_pad;
            ro[gi[u]] = re;
            ro[A.ngp_pad + gi[u]] = im;
        }
        e += (double)(A.w2[gi[u]] * (re * re + im * im));
    }
    e = block_sum(e, red);
    if (tid == 0) A.partial[(size_t)w * A.n_slabs + slab] = e;
}

/* ------------------------------------------------------------------------------------------ */
/* [S5] real-space pair sum.  grid = n_walkers * n_tiles; machinery in ewald_realspace.cuh. */

/* Tables and stack shapes of the real-space machinery, common to the energy and move kernels. */
template <typename T> struct PairTabs {
    const T *pair_tab; int n_bins;   /* PairFmt<T>::elems(n_bins) values in the layout of PairFmt<T>    */
    T t_safe;                        /* some t inside the table                                         */
    const float *far_tab; int n_far; /* FP64 kernels: [n_far][FarFmt::REP][4] far-shell cubics; 0 = none */
    int key_far;                     /* order key of the far shell's start, INT_MAX = none              */
    int far_t0;                      /* t at which this kernel's far shell (and its staged table) starts */
    const double *qinfo;             /* device [4]: sum q^2, sum q, all-equal flag, q_0                  */
    int ion_uniform;                 /* at most 4 distinct fixed charges (species)                      */
    int n_species, sp_start[5];      /* ions [sp_start[s], sp_start[s+1]) carry one charge each         */
    int cap_u, cap_g;                /* near-stack capacity per lane: bare t items / (t, qq) items      */
    int capf_u, capf_g;              /* far-stack capacity per lane                                     */
    int round_items;                 /* host only: RoundSize<T, SIGNED>::R of the kernel these shapes are for */
};

/* [S6] what the combine needs (folded into the last CTA of a walker in real_kernel) */
struct CombineArgs {
    const double *recip_partial; int n_recip;
    const double *real_partial; int n_real;
    double ion_q2, ion_qsum, ion_real;
    double xi_r, self_coef, bg_coef;
    double *energies; double *components; int n_walkers;
};

template <typename T> struct RealArgs {
    const T *pos; const T *q;
    int n, npad;
    const T *img; int nimg;                       /* [nimg][3], kappa-scaled (general cells)   */
    const T *ion_pos; const T *ion_q; int n_ion;  /* [n_ion][3], [n_ion]                        */
    PairTabs<T> P;
    double *partial;                              /* [W][n_tiles] */
    int n_tiles;
    RealGeom<T> g;
    CombineArgs comb;                             /* energies == null: no combine */
    int *done;                                    /* [W] CTAs of the walker that have finished (zero between calls) */
    int zsplit;                                   /* ScanShape::ZSPLIT shapes: one z-image of a pair per lane (small batches) */
};

constexpr int REAL_MAX_THREADS = 512;

/* Shared-memory carve-up common to the real-space and move kernels. */
template <typename T> struct RealSmem {
    T *tab;     /* PairFmt<T>::elems(n_bins) */
    float *far; /* [n_far][REP][4] */
    T *img;     /* [nimg][3]; FP32: followed by the [nimg][3] low parts */
    T *ion;     /* [n_ion][4] = x,y,z,q */
    T *rest;    /* caller's arrays (rest_elems), then the stacks */
    unsigned char *stacks;
    static constexpr int IMG_PARTS = sizeof(T) == 4 ? 2 : 1;
    static __host__ __device__ size_t up4(size_t e) { return (e + 3) & ~(size_t)3; }
    static __host__ __device__ size_t far_bytes(int n_far) { return (size_t)n_far * FarFmt::REP * 16; }
    __device__ __forceinline__ RealSmem(unsigned char *raw, const PairTabs<T> &P, int nimg, int n_ion, size_t rest_elems)
    {
        tab = reinterpret_cast<T *>(raw);
        far = reinterpret_cast<float *>(tab + up4(PairFmt<T>::elems(P.n_bins)));
        img = reinterpret_cast<T *>(reinterpret_cast<unsigned char *>(far) + far_bytes(P.n_far));
        ion = img + up4(3 * IMG_PARTS * (size_t)nimg);
        rest = ion + up4(4 * (size_t)n_ion);
        /* the lane stacks' rows are 128 or 256 bytes: they start on a 128-byte boundary of the window (the kernels
         * keep their static shared memory a multiple of 128 bytes), else every push and pop touches two lines */
        const size_t off = reinterpret_cast<unsigned char *>(rest + up4(rest_elems)) - raw;
        stacks = raw + ((off + 127) & ~(size_t)127);
    }
    /* bytes before the stacks */
    static size_t fixed_bytes(int n_bins, int n_far, int nimg, int n_ion, size_t rest_elems)
    {
        const size_t b = (up4(PairFmt<T>::elems(n_bins)) + up4(3 * IMG_PARTS * (size_t)nimg) + up4(4 * (size_t)n_ion) +
                          up4(rest_elems)) * sizeof(T) + far_bytes(n_far);
        return (b + 127) & ~(size_t)127;
    }
    /* bytes of one warp's stacks (the two item kinds of a stack share the same bytes) */
    static __host__ __device__ size_t warp_stack_bytes(const PairTabs<T> &P)
    {
        return (size_t)P.cap_u * 32 * sizeof(T) + (size_t)P.capf_u * 32 * 4; /* near items, then far items */
    }
    /* bytes of the two tables (multiples of 128) */
    static __host__ __device__ unsigned table_bytes(const PairTabs<T> &P)
    {
        return (unsigned)(PairFmt<T>::elems(P.n_bins) * sizeof(T) + far_bytes(P.n_far));
    }
    /* One thread: the two tables by TMA bulk copies on `bar` (announced by the caller's tma_expect).  A loop of
     * 16-byte loads and stores over the ~100 KB took a CTA 6 us (a dozen dependent global-load latencies per
     * thread): 6 % of a CTA's life on config 2, a third of the kernel on config 1. */
    __device__ __forceinline__ void tma_tables(const PairTabs<T> &P, uint64_t *bar)
    {
        tma_copy_1d(tab, P.pair_tab, (unsigned)(PairFmt<T>::elems(P.n_bins) * sizeof(T)), bar);
        if (P.n_far > 0) tma_copy_1d(far, P.far_tab, (unsigned)far_bytes(P.n_far), bar);
    }
    /* the small arrays: image list and fixed charges */
    __device__ __forceinline__ void fill_small(const T *gimg, int nimg, const T *ion_pos, const T *ion_q, int n_ion,
                                               int tid, int nthreads)
    {
        for (int t = tid; t < 3 * IMG_PARTS * nimg; t += nthreads) img[t] = gimg[t];
        for (int t = tid; t < n_ion; t += nthreads) {
            ion[4 * t + 0] = ion_pos[3 * t + 0];
            ion[4 * t + 1] = ion_pos[3 * t + 1];
            ion[4 * t + 2] = ion_pos[3 * t + 2];
            ion[4 * t + 3] = ion_q[t];
        }
    }
    __device__ __forceinline__ void fill(const PairTabs<T> &P, const T *gimg, int nimg, const T *ion_pos,
                                         const T *ion_q, int n_ion, int tid, int nthreads)
    {
        {   /* a multiple of 16 bytes in both layouts */
            const int n4 = (int)(PairFmt<T>::elems(P.n_bins) * sizeof(T) / 16);
            const int4 *src = reinterpret_cast<const int4 *>(P.pair_tab);
            int4 *dst = reinterpret_cast<int4 *>(tab);
            for (int t = tid; t < n4; t += nthreads) dst[t] = src[t];
        }
        {
            const int n4 = P.n_far * FarFmt::REP;
            const int4 *src = reinterpret_cast<const int4 *>(P.far_tab);
            int4 *dst = reinterpret_cast<int4 *>(far);
            for (int t = tid; t < n4; t += nthreads) dst[t] = src[t];
        }
        for (int t = tid; t < 3 * IMG_PARTS * nimg; t += nthreads) img[t] = gimg[t];
        for (int t = tid; t < n_ion; t += nthreads) {
            ion[4 * t + 0] = ion_pos[3 * t + 0];
            ion[4 * t + 1] = ion_pos[3 * t + 1];
            ion[4 * t + 2] = ion_pos[3 * t + 2];
            ion[4 * t + 3] = ion_q[t];
        }
    }
};

/* Points one lane's stacks at its warp's region of shared memory. */
template <bool UQ, bool SIGNED>
__device__ __forceinline__ void init_stacks(PairStacks<float, UQ, SIGNED> &st, RealSmem<float> &S,
                                            const PairTabs<float> &P, int bias, int warp, int lane)
{
    unsigned char *mem = S.stacks + (size_t)warp * RealSmem<float>::warp_stack_bytes(P);
    st.nr.init(mem, lane, UQ ? P.cap_u : P.cap_g, S.tab, bias, P.t_safe);
}
template <bool UQ, bool SIGNED>
__device__ __forceinline__ void init_stacks(PairStacks<double, UQ, SIGNED> &st, RealSmem<double> &S,
                                            const PairTabs<double> &P, int bias, int warp, int lane)
{
    unsigned char *mem = S.stacks + (size_t)warp * RealSmem<double>::warp_stack_bytes(P);
    st.nr.init(mem, lane, UQ ? P.cap_u : P.cap_g, S.tab, bias, P.t_safe);
    st.key_far = P.key_far;
    if (st.has_far()) st.fr.init(mem + (size_t)P.cap_u * 32 * sizeof(double), lane, UQ ? P.capf_u : P.capf_g, S.far, P.far_t0);
    else { st.fr.base_a = st.fr.top_a = 0; st.fr.cap_b = 0; st.fr.sum = 0; }
}

/* Pairs (i, j = i + k + 1 mod n), rows k = 0..H-1 (H = (n-1)/2) and, for even n, half of row H, dealt
 * round-robin to `team` threads; the cursor advances without divisions. */
struct PairWalk {
    int i, k, di, dk, n;
    __device__ __forceinline__ void init(int gid, int team, int n_)
    {
        n = n_; k = gid / n; i = gid - k * n; dk = team / n; di = team - dk * n;
    }
    __device__ __forceinline__ void next()
    {
        i += di; k += dk;
        if (i >= n) { i -= n; k++; }
    }
};

template <typename T, int DIM, bool ORTHO, int M, bool UQ>
__device__ __forceinline__ double real_body(const RealArgs<T> &A, RealSmem<T> &S, const T *sp, const T *sq,
                                            int tile, T q0)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = A.n;
    PairStacks<T, UQ, false> st;
    init_stacks(st, S, A.P, A.g.bias, warp, lane);
    __syncwarp();
    double total = 0, direct = 0;
    /* work items are pairs, dealt round-robin to the walker's threads; with zsplit an item is (pair, z-image):
     * ROW consecutive threads share a pair */
    typedef ScanShape<DIM, ORTHO, M, UQ> Shape0;
    const bool zs = Shape0::ZSPLIT && A.zsplit != 0;
    const int all_threads = A.n_tiles * blockDim.x, my_thread = tile * blockDim.x + tid;
    const int team = zs ? all_threads / Shape0::ROW : all_threads, gid = zs ? my_thread / Shape0::ROW : my_thread;
    const int zsel = zs ? my_thread - gid * Shape0::ROW : -1;
    const bool active = !zs || gid < team; /* zsplit: the last all_threads mod ROW threads have no item */

    /* mobile-mobile pairs */
    {
        const int H = (n - 1) / 2;
        const bool even = (n & 1) == 0;
        typedef ScanShape<DIM, ORTHO, M, UQ> Shape;
        constexpr int GROUP = Shape::GROUP;
        /* image-list path with few images: LIMIT / nimg pairs between two services */
        const int list_group = !ORTHO && A.nimg > 0 && 2 * A.nimg <= Shape::LIMIT ? Shape::LIMIT / A.nimg : 1;
        const int group = ORTHO ? GROUP : list_group;
        PairWalk pw; pw.init(gid, team, n);
        for (;;) {
            bool valid = active && (pw.k < H || (even && pw.k == H && pw.i < n / 2));
            if (!__any_sync(0xffffffffu, valid)) break;
#pragma unroll
            for (int u = 0; u < (ORTHO ? GROUP : group); u++) {
                if (u > 0) valid = active && (pw.k < H || (even && pw.k == H && pw.i < n / 2));
                T d[3] = {0, 0, 0};
                T w = UQ ? q0 * q0 : T(0);
                if (valid) {
                    const int i = pw.i;
                    int j = i + pw.k + 1;
                    if (j >= n) j -= n;
#pragma unroll
                    for (int x = 0; x < DIM; x++) d[x] = sp[x * A.npad + i] - sp[x * A.npad + j];
                    if (!UQ) w = sq[i] * sq[j];
                }
                scan_pair<T, DIM, ORTHO, M, UQ, false, false, GROUP == 1>(A.g, d, w, valid, st, direct, S.img, A.nimg,
                                                                          group == 1, zsel);
                pw.next();
            }
            if (group > 1) st.service(Shape::LIMIT);
        }
        st.finish();
        total += st.take() * (UQ ? (double)(q0 * q0) : 1.0);
    }
    /* mobile particles against the fixed charges: with bare-t items one segment per species */
    for (int s = 0; s < (UQ ? A.P.n_species : (A.n_ion > 0 ? 1 : 0)); s++) {
        const int k0 = UQ ? A.P.sp_start[s] : 0, k1 = UQ ? A.P.sp_start[s + 1] : A.n_ion;
        const T qion0 = S.ion[4 * k0 + 3];
        PairWalk pw; pw.init(gid, team, n);
        pw.k += k0;
        for (;;) {
            const bool valid = active && pw.k < k1;
            if (!__any_sync(0xffffffffu, valid)) break;
            T d[3] = {0, 0, 0};
            T w = UQ ? q0 * qion0 : T(0);
            if (valid) {
                const int i = pw.i, I = pw.k;
#pragma unroll
                for (int x = 0; x < DIM; x++) d[x] = sp[x * A.npad + i] - S.ion[4 * I + x];
                if (!UQ) w = sq[i] * S.ion[4 * I + 3];
            }
            scan_pair<T, DIM, ORTHO, M, UQ>(A.g, d, w, valid, st, direct, S.img, A.nimg, true, zsel);
            pw.next();
        }
        st.finish();
        total += st.take() * (UQ ? (double)(q0 * qion0) : 1.0);
    }
    return total + direct;
}

template <typename T, int DIM, bool ORTHO, int M>
__global__ void __launch_bounds__(REAL_MAX_THREADS, sizeof(T) == 4 ? 2 : 1) real_kernel(RealArgs<T> A)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RealSmem<T> S(smem_raw, A.P, A.nimg, A.n_ion, (size_t)DIM * A.npad + A.n);
    T *sp = S.rest;                 /* [DIM][npad] positions (unscaled: differences are taken first) */
    T *sq = sp + DIM * A.npad;      /* [n] charges */
    /* static shared memory stays a multiple of 128 bytes: the dynamic part (tables, lane stacks whose rows are
     * 128 / 256 bytes) keeps its 128-byte alignment; red[32] holds the mbarrier of the bulk copy */
    __shared__ __align__(128) double red[48];
    uint64_t *bar = reinterpret_cast<uint64_t *>(&red[32]);
    const int w = blockIdx.x / A.n_tiles, tile = blockIdx.x - w * A.n_tiles, tid = threadIdx.x;
    /* the walker's SoA block [DIM][npad] is contiguous: TMA bulk copies stage it and the two tables while the
     * threads copy the small arrays */
    if (tid == 0) tma_barrier_init(bar);
    __syncthreads();
    if (tid == 0) {
        const unsigned pos_bytes = (unsigned)(DIM * A.npad * sizeof(T));
        tma_expect(bar, pos_bytes + RealSmem<T>::table_bytes(A.P));
        tma_copy_1d(sp, A.pos + (size_t)w * DIM * A.npad, pos_bytes, bar);
        S.tma_tables(A.P, bar);
    }
    for (int t = tid; t < A.n; t += blockDim.x) sq[t] = A.q[t];
    S.fill_small(A.img, A.nimg, A.ion_pos, A.ion_q, A.n_ion, tid, blockDim.x);
    tma_wait(bar, 0);
    __syncthreads();

    /* all mobile charges equal (the electron gas): the stacks then hold bare t (ewald_realspace.cuh) */
    bool eq = true;
    for (int t = tid; t < A.n; t += blockDim.x) eq = eq && sq[t] == sq[0];
    const bool uq = __syncthreads_and(eq) && A.P.ion_uniform;
    const T q0 = sq[0];
    double acc;
    if (uq) acc = real_body<T, DIM, ORTHO, M, true>(A, S, sp, sq, tile, q0);
    else acc = real_body<T, DIM, ORTHO, M, false>(A, S, sp, sq, tile, q0);
    acc = block_sum(acc, red);
    if (tid == 0) A.partial[(size_t)w * A.n_tiles + tile] = acc * A.g.kappa_d;

    /* [S6] The CTA of a walker that finishes last adds the partial sums in fixed order and the constants of
     * Eqs. 3-4: E = E_recip + E_real + E_self + E_bg (the reciprocal kernel ran before this one on the stream). */
    if (A.comb.energies == nullptr) return;
    int *last = reinterpret_cast<int *>(&red[40]); /* inside red[]: static shared memory stays a multiple of 128 bytes */
    if (tid == 0) {
        __threadfence();
        *last = atomicAdd(&A.done[w], 1) == A.n_tiles - 1;
    }
    __syncthreads();
    if (!*last) return;
    double s2 = 0, s1 = 0;
    for (int t = tid; t < A.n; t += blockDim.x) { const double v = (double)sq[t]; s2 += v * v; s1 += v; }
    s2 = block_sum(s2, red);
    s1 = block_sum(s1, red);
    if (tid == 0) {
        __threadfence();
        const CombineArgs &C = A.comb;
        double er = 0, ep = 0;
        for (int k = 0; k < C.n_recip; k++) er += __ldcg(C.recip_partial + (size_t)w * C.n_recip + k);
        for (int k = 0; k < A.n_tiles; k++) ep += __ldcg(A.partial + (size_t)w * A.n_tiles + k);
        const double q2 = s2 + C.ion_q2, qs = s1 + C.ion_qsum;
        const double e_real = ep + C.ion_real + 0.5 * q2 * C.xi_r;
        const double e_self = -C.self_coef * q2;
        const double e_bg = -0.5 * C.bg_coef * qs * qs;
        C.energies[w] = er + e_real + e_self + e_bg;
        if (C.components) {
            C.components[4 * w + 0] = er;
            C.components[4 * w + 1] = e_real;
            C.components[4 * w + 2] = e_self;
            C.components[4 * w + 3] = e_bg;
        }
        A.done[w] = 0;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* [S6] combine as a kernel of its own (large batches: the arrival counter of the folded form costs every CTA of
 * real_kernel a fence and an atomic, ~1.5 % of a many-wave launch).  One thread per walker; every block adds the
 * charges once (the same block size and order for every walker). */
template <typename T>
__global__ void combine_kernel(CombineArgs A, const T *q, int n)
{
    __shared__ double red[32], sums[2];
    double s2 = 0, s1 = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) { const double v = (double)__ldg(q + i); s2 += v * v; s1 += v; }
    s2 = block_sum(s2, red);
    s1 = block_sum(s1, red);
    if (threadIdx.x == 0) { sums[0] = s2; sums[1] = s1; }
    __syncthreads();
    s2 = sums[0]; s1 = sums[1];
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= A.n_walkers) return;
    double er = 0, ep = 0;
    for (int k = 0; k < A.n_recip; k++) er += A.recip_partial[(size_t)w * A.n_recip + k];
    for (int k = 0; k < A.n_real; k++) ep += A.real_partial[(size_t)w * A.n_real + k];
    const double q2 = s2 + A.ion_q2, qs = s1 + A.ion_qsum;
    const double e_real = ep + A.ion_real + 0.5 * q2 * A.xi_r;
    const double e_self = -A.self_coef * q2;
    const double e_bg = -0.5 * A.bg_coef * qs * qs;
    A.energies[w] = er + e_real + e_self + e_bg;
    if (A.components) {
        A.components[4 * w + 0] = er;
        A.components[4 * w + 1] = e_real;
        A.components[4 * w + 2] = e_self;
        A.components[4 * w + 3] = e_bg;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Charge sums of a stored population (ewald_load_walkers): sum q^2, sum q, all-equal flag, q_0. */

template <typename T>
__global__ void charge_sums_kernel(const T *q, int n, double *out)
{
    __shared__ double red[32];
    double s2 = 0, s1 = 0, diff = 0;
    const T q0 = q[0];
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        double v = (double)q[i]; s2 += v * v; s1 += v;
        if (q[i] != q0) diff += 1;
    }
    s2 = block_sum(s2, red);
    s1 = block_sum(s1, red);
    diff = block_sum(diff, red);
    /* out[2]: all charges equal (the real-space kernel then keeps t alone on its stacks); out[3] = q_0 */
    if (threadIdx.x == 0) { out[0] = s2; out[1] = s1; out[2] = diff == 0 ? 1.0 : 0.0; out[3] = (double)q0; }
}

/* ------------------------------------------------------------------------------------------ */
/* [S7] single-particle move.  One WARP per move, persistent CTAs: the tables are staged once per CTA, then
 * warp v of CTA b takes moves (b * warps + v), + gridDim.x * warps, ...  A warp needs no block barrier, its
 * lanes run long loops (N_G+/32 vectors, N/32 partners), and the other warps of the SM hide its latencies. */

template <typename T> struct MoveArgs {
    T *pos;            /* stored [W][DIM][npad] */
    const T *q;        /* stored [n] */
    T *rho;            /* stored [W][2][ngp_pad] */
    int n, npad, n_walkers, n_moves;
    const short4 *gn; const T *w2; int ngp, ngp_pad;
    int nmax[3]; int off[3], rowlen;
    const T *img; int nimg;                       /* kappa-scaled image list (general cells) */
    const T *ion_pos; const T *ion_q; int n_ion;
    PairTabs<T> P;                                /* qinfo: of the stored charges            */
    const int *walker; const int *electron; const T *new_r; /* [n_moves], [n_moves], [n_moves][DIM] */
    int commit;
    double *delta_e;
    double binv[9];                               /* unscaled: s_k = r . binv[k]; FP64 in both precisions */
    RealGeom<T> g;
};

/* [S7c] one warp: sum over the partners j != k of w_j [F-sum(r_new - r_j) - F-sum(r_old - r_j)], w_j = q_j
 * (or 1 with the common charge applied here when UQ). */
template <typename T, int DIM, bool ORTHO, int M, bool UQ>
__device__ __forceinline__ double move_real(const MoveArgs<T> &A, RealSmem<T> &S, const T *pw, int k,
                                            const T *r_old, const T *r_new, T q0)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    PairStacks<T, UQ, true> st;
    init_stacks(st, S, A.P, A.g.bias, warp, lane);
    __syncwarp();
    double total = 0, direct = 0;
    /* segment 0: the mobile partners; then the fixed charges, one segment per species with bare-t items */
    const int n_seg = 1 + (UQ ? A.P.n_species : (A.n_ion > 0 ? 1 : 0));
    for (int seg = 0; seg < n_seg; seg++) {
        const int j0 = seg == 0 || !UQ ? 0 : A.P.sp_start[seg - 1];
        const int cnt = seg == 0 ? A.n : (UQ ? A.P.sp_start[seg] : A.n_ion);
        const T qion0 = seg == 0 ? T(0) : S.ion[4 * j0 + 3];
        /* the partner of the next round is loaded before this round's scan (its latency was 12 % of the kernel) */
        auto fetch = [&](int base, T (&r)[3], T &wt) {
            const int j = base + lane;
            const bool ok = j < cnt && (seg >= 1 || j != k);
            r[0] = r[1] = r[2] = T(0);
            wt = UQ ? T(1) : T(0);
            if (ok) {
                if (seg == 0) {
#pragma unroll
                    for (int x = 0; x < DIM; x++) r[x] = pw[x * A.npad + j];
                    if (!UQ) wt = A.q[j];
                } else {
#pragma unroll
                    for (int x = 0; x < DIM; x++) r[x] = S.ion[4 * j + x];
                    if (!UQ) wt = S.ion[4 * j + 3];
                }
            }
            return ok;
        };
        T rj_next[3], w_next;
        bool valid_next = fetch(j0, rj_next, w_next);
        for (int base = j0; base < cnt; base += 32) {
            const bool valid = valid_next;
            const T rj[3] = {rj_next[0], rj_next[1], rj_next[2]};
            const T w = w_next;
            valid_next = fetch(base + 32, rj_next, w_next);
            T dn[3] = {0, 0, 0}, dold[3] = {0, 0, 0};
#pragma unroll
            for (int x = 0; x < DIM; x++) {
                dn[x] = r_new[x] - rj[x];
                dold[x] = r_old[x] - rj[x];
            }
            scan_pair<T, DIM, ORTHO, M, UQ, true, false>(A.g, dn, w, valid, st, direct, S.img, A.nimg);
            scan_pair<T, DIM, ORTHO, M, UQ, true, true>(A.g, dold, UQ ? w : -w, valid, st, direct, S.img, A.nimg);
        }
        if (cnt > j0) st.finish();
        const double wseg = UQ ? (double)(seg == 0 ? q0 : qion0) : 1.0;
        total += (st.take() + direct) * wseg;
        direct = 0;
    }
    return total;
}

constexpr int MOVE_MAX_THREADS = 512;
/* rho(G) vectors per lane and batch in [S7b] (two batches in flight); more spills registers: FP64 2 / 3 / 4 gave
 * 13.5 / 15.4 / 11.7 M moves/s, FP32 (64 registers) 25.9 / 24.5 / 23.4 */
template <typename T> struct MoveBatch { static constexpr int N = sizeof(T) == 8 ? 3 : 2; };

template <typename T, int DIM, bool ORTHO, int M>
__global__ void __launch_bounds__(MOVE_MAX_THREADS, sizeof(T) == 4 ? 2 : 1) move_kernel(MoveArgs<T> A)
{
    typedef typename Num<T>::T2 T2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n_warps = blockDim.x >> 5;
    RealSmem<T> S(smem_raw, A.P, A.nimg, A.n_ion, 4 * (size_t)A.rowlen * n_warps);
    T2 *tab = reinterpret_cast<T2 *>(S.rest) + (size_t)warp * 2 * A.rowlen; /* this warp's [2][rowlen]: old, new */
    S.fill(A.P, A.img, A.nimg, A.ion_pos, A.ion_q, A.n_ion, tid, blockDim.x);
    __syncthreads();
    const bool uq = A.P.qinfo[2] != 0.0 && A.P.ion_uniform;
    const T q0 = (T)A.P.qinfo[3];

    for (int m = blockIdx.x * n_warps + warp; m < A.n_moves; m += gridDim.x * n_warps) {
        const int w = A.walker[m], k = A.electron[m];
        if (w < 0 || w >= A.n_walkers || k < 0 || k >= A.n) { /* warp-uniform */
            if (lane == 0) A.delta_e[m] = __longlong_as_double(0x7ff8000000000000LL);
            continue;
        }
        T *pw = A.pos + (size_t)w * DIM * A.npad;
        T r_old[3] = {0, 0, 0}, r_new[3] = {0, 0, 0};
#pragma unroll
        for (int x = 0; x < DIM; x++) { r_old[x] = pw[x * A.npad + k]; r_new[x] = A.new_r[(size_t)m * DIM + x]; }
        const T qk = A.q[k];

        /* [S7a] power tables of the two points */
        if (lane < 2 * DIM) {
            const int which = lane / DIM, d = lane - which * DIM;
            const T *r = which ? r_new : r_old;
            double s = 0;
#pragma unroll
            for (int x = 0; x < DIM; x++) s += (double)r[x] * A.binv[3 * d + x];
            power_row<T>((T)(s - rint(s)), T(1), A.nmax[d], tab + which * A.rowlen + A.off[d]);
        }
        __syncwarp();

        /* [S7b] Delta E_recip and the patch of rho(G).  The walker's rho comes from HBM and nothing else of the
         * warp's work can cover that latency, so the loads of MoveBatch<T>::N vectors per lane are issued before the
         * first of them is used (one load in flight per lane ran at 1.1 TB/s over the whole GPU). */
        T *rr = A.rho + (size_t)w * 2 * A.ngp_pad;
        double acc = 0;
        /* (prefetching rho alone and reading the shared G indices and weights when used was slower: 13.3 M) */
        struct GBatch { short4 nn[MoveBatch<T>::N]; T re[MoveBatch<T>::N], im[MoveBatch<T>::N], wg[MoveBatch<T>::N]; };
        auto load = [&](GBatch &b, int g0) {
#pragma unroll
            for (int u = 0; u < MoveBatch<T>::N; u++) {
                const int g = g0 + 32 * u;
                const bool in = g < A.ngp;
                b.nn[u] = in ? __ldg(A.gn + g) : make_short4(0, 0, 0, 0);
                b.re[u] = in ? rr[g] : T(0);
                b.im[u] = in ? rr[A.ngp_pad + g] : T(0);
                b.wg[u] = in ? __ldg(A.w2 + g) : T(0);
            }
        };
        auto patch = [&](const GBatch &b, int g0) {
#pragma unroll
            for (int u = 0; u < MoveBatch<T>::N; u++) {
                const int g = g0 + 32 * u;
                const short4 nn = b.nn[u];
                T2 ph[2];
#pragma unroll
                for (int which = 0; which < 2; which++) {
                    const T2 *row = tab + which * A.rowlen;
                    T2 e1 = row[A.off[0] + nn.x];
                    T2 e2 = row[A.off[1] + (nn.y < 0 ? -nn.y : nn.y)];
                    if (nn.y < 0) e2.y = -e2.y;
                    T2 e;
                    e.x = e1.x * e2.x - e1.y * e2.y;
                    e.y = e1.x * e2.y + e1.y * e2.x;
                    if (DIM == 3) {
                        T2 e3 = row[A.off[2] + (nn.z < 0 ? -nn.z : nn.z)];
                        if (nn.z < 0) e3.y = -e3.y;
                        T2 f;
                        f.x = e.x * e3.x - e.y * e3.y;
                        f.y = e.x * e3.y + e.y * e3.x;
                        e = f;
                    }
                    ph[which] = e;
                }
                const T dr = ph[1].x - ph[0].x, di = ph[1].y - ph[0].y;
                acc += (double)(b.wg[u] * (2 * qk * (b.re[u] * dr + b.im[u] * di) + qk * qk * (dr * dr + di * di)));
                if (A.commit && g < A.ngp) { rr[g] = b.re[u] + qk * dr; rr[A.ngp_pad + g] = b.im[u] + qk * di; }
            }
        };
        {   /* two batches in flight: the loads of the next one are issued before the current one is used */
            constexpr int STEP = 32 * MoveBatch<T>::N;
            GBatch b0, b1;
            int g0 = lane;
            load(b0, g0);
            while (g0 < A.ngp) {
                load(b1, g0 + STEP);
                patch(b0, g0);
                g0 += STEP;
                if (g0 >= A.ngp) break;
                load(b0, g0 + STEP);
                patch(b1, g0);
                g0 += STEP;
            }
        }

        /* [S7c] Delta E_real = q_k sum_{j != k} q_j [psi(r'-r_j) - psi(r-r_j)] */
        double accr;
        if (uq) accr = move_real<T, DIM, ORTHO, M, true>(A, S, pw, k, r_old, r_new, q0);
        else accr = move_real<T, DIM, ORTHO, M, false>(A, S, pw, k, r_old, r_new, q0);
        acc += (double)qk * accr * A.g.kappa_d;
        acc = warp_sum(acc); /* its shuffles also order every lane's read of r_old before the commit */
        if (lane == 0) {
            A.delta_e[m] = acc;
            if (A.commit) {
#pragma unroll
                for (int x = 0; x < DIM; x++) pw[x * A.npad + k] = r_new[x];
            }
        }
        __syncwarp(); /* the power tables are reused by this warp's next move */
    }
}

/* ------------------------------------------------------------------------------------------ */
/* FMA-pipe probe: 8 independent dependent chains per thread. */
template <typename T>
__global__ void __launch_bounds__(256) fma_probe_kernel(int iters, T a, T b, T *sink)
{
    T x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
            x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
        }
    }
    T s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == T(123456789)) sink[0] = s;
}

} // namespace ewald
