/* blip_api.cu -- include/blip.h: batched blip-orbital evaluation, one kernel for all positions and orbitals.
 *
 * blip_kernel: one warp per position.  The lanes share the position, so the 12 one-dimensional blip values and
 * derivatives (4 per axis) and the five weights of each of the 64 neighbouring grid points -- value, Cartesian
 * gradient, Laplacian through the metric of the cell -- are warp-uniform; a lane owns orbitals lane, lane + 32, ...
 * and reads c[point][orbital] (orbital fastest: a warp reads 256 contiguous bytes per grid point) with 5 FMAs per
 * coefficient.  The coefficient table (tens of MB) lives in L2; the kernel is bound by L2 gather bandwidth
 * (64 x n_orb coefficients per position, 10 flops per coefficient).  No CPU fallback. */
#include <cmath>
#include <new>
#include <string>
#include <vector>

#include "blip.h"
#include "ewald_kernels_common.cuh"

using namespace ewald;

constexpr int BLIP_THREADS = 256;
constexpr int BLIP_OPL = 4; /* orbitals per lane and pass: 128 orbitals per pass */

template <typename T> struct BlipArgs {
    const T *points;  /* [3][n_pad] */
    int n_points, n_pad;
    const T *coef;    /* [N1][N2][N3][no_pad] */
    int grid[3], n_orb, no_pad;
    double binv[9];   /* s_k = r . binv[k] */
    double gm[9];     /* gm[k][x] = N_k binv[k][x] = d u_k / d r_x */
    double metric[6]; /* (gm gm^T): 00, 11, 22, 01, 02, 12 */
    double *psi, *grad, *lap;
};

/* Theta, Theta', Theta'' at the four neighbours of a point with fractional offset t in [0, 1): x = t+1, t, t-1, t-2 */
template <typename T> __device__ __forceinline__ void blip_1d(T t, T (&f)[4], T (&d1)[4], T (&d2)[4])
{
    const T x0 = t + 1, x3 = 2 - t;          /* |x| in [1, 2]: 1/4 (2 - |x|)^3 */
    const T a0 = 2 - x0, a3 = 2 - x3;
    f[0] = T(0.25) * a0 * a0 * a0; d1[0] = T(-0.75) * a0 * a0; d2[0] = T(1.5) * a0;
    f[3] = T(0.25) * a3 * a3 * a3; d1[3] = T(0.75) * a3 * a3; d2[3] = T(1.5) * a3;   /* x = t - 2 < 0: sign flips */
    const T x1 = t, x2 = 1 - t;              /* |x| <= 1: 1 - 3/2 x^2 + 3/4 |x|^3 */
    f[1] = 1 + x1 * x1 * (T(0.75) * x1 - T(1.5)); d1[1] = x1 * (T(2.25) * x1 - 3); d2[1] = T(4.5) * x1 - 3;
    f[2] = 1 + x2 * x2 * (T(0.75) * x2 - T(1.5)); d1[2] = -x2 * (T(2.25) * x2 - 3); d2[2] = T(4.5) * x2 - 3;
}

template <typename T>
__global__ void __launch_bounds__(BLIP_THREADS) blip_kernel(BlipArgs<T> A)
{
    const int lane = threadIdx.x & 31, warps = (gridDim.x * blockDim.x) >> 5;
    /* The 36 one-dimensional blip values of a position (Theta, Theta', Theta'' x 3 axes x 4 neighbours) are the same
     * for the whole warp and are indexed by the loop counters below: as per-thread arrays they sat in LOCAL memory
     * (288 bytes per thread, more than L1 holds for 2048 threads), whose traffic competed in L2 with the
     * coefficient gather (FP64: 2.5 to 5.7 ms per launch depending on how ptxas scheduled the reloads).  Lane k < 3
     * computes axis k; the warp reads them from shared memory (one broadcast wavefront per read). */
    __shared__ T s1d[BLIP_THREADS / 32][3][3][4]; /* [warp][f, d1, d2][axis][neighbour] */
    T (*f)[4] = s1d[threadIdx.x >> 5][0], (*d1)[4] = s1d[threadIdx.x >> 5][1], (*d2)[4] = s1d[threadIdx.x >> 5][2];
    for (int p = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; p < A.n_points; p += warps) {
        int i0[3];
        {
            const int k = lane < 3 ? lane : 0;
            double s = 0;
#pragma unroll
            for (int x = 0; x < 3; x++) s += (double)A.points[x * A.n_pad + p] * A.binv[3 * k + x];
            s -= floor(s);
            const double u = s * A.grid[k];
            int i = (int)floor(u);
            if (i >= A.grid[k]) i = A.grid[k] - 1; /* s rounded up to 1 */
            T tf[4], td1[4], td2[4];
            blip_1d<T>((T)(u - i), tf, td1, td2);
            __syncwarp(); /* the previous position's reads are done */
            if (lane < 3) {
#pragma unroll
                for (int a = 0; a < 4; a++) { f[k][a] = tf[a]; d1[k][a] = td1[a]; d2[k][a] = td2[a]; }
            }
#pragma unroll
            for (int kk = 0; kk < 3; kk++) i0[kk] = __shfl_sync(0xffffffffu, i, kk);
            __syncwarp();
        }
        /* FP32: the values of axis 2 (indexed by the unrolled innermost loop) and those of the current a and b are
         * kept in registers (1.74 -> 1.35 ms); FP64 reads all of them from shared memory where they are used (in
         * registers the kernel needs 178 of them: 1.90 -> 3.34 ms, or 2.53 ms bounded to 128 with spills) */
        constexpr bool HOIST = sizeof(T) == 4;
        T f2[4], d12[4], d22[4];
#pragma unroll
        for (int c = 0; c < 4; c++) { f2[c] = HOIST ? f[2][c] : T(0); d12[c] = HOIST ? d1[2][c] : T(0); d22[c] = HOIST ? d2[2][c] : T(0); }
#define F2(c) (HOIST ? f2[c] : f[2][c])
#define D12(c) (HOIST ? d12[c] : d1[2][c])
#define D22(c) (HOIST ? d22[c] : d2[2][c])
        for (int ob = 0; ob < A.n_orb; ob += 32 * BLIP_OPL) {
            T v[BLIP_OPL], gx[BLIP_OPL], gy[BLIP_OPL], gz[BLIP_OPL], lp[BLIP_OPL];
#pragma unroll
            for (int q = 0; q < BLIP_OPL; q++) v[q] = gx[q] = gy[q] = gz[q] = lp[q] = 0;
            for (int a = 0; a < 4; a++) {
                int ia = i0[0] + a - 1; ia += ia < 0 ? A.grid[0] : 0; ia -= ia >= A.grid[0] ? A.grid[0] : 0;
                const T f0a = HOIST ? f[0][a] : T(0), d10a = HOIST ? d1[0][a] : T(0), d20a = HOIST ? d2[0][a] : T(0);
                for (int b = 0; b < 4; b++) {
                    int ib = i0[1] + b - 1; ib += ib < 0 ? A.grid[1] : 0; ib -= ib >= A.grid[1] ? A.grid[1] : 0;
                    T f01, g0, g1, h00, h11, h01;
                    if (HOIST) {
                        const T f1b = f[1][b], d11b = d1[1][b], d21b = d2[1][b];
                        f01 = f0a * f1b; g0 = d10a * f1b; g1 = f0a * d11b;
                        h00 = d20a * f1b; h11 = f0a * d21b; h01 = d10a * d11b;
                    } else {
                        f01 = f[0][a] * f[1][b]; g0 = d1[0][a] * f[1][b]; g1 = f[0][a] * d1[1][b];
                        h00 = d2[0][a] * f[1][b]; h11 = f[0][a] * d2[1][b]; h01 = d1[0][a] * d1[1][b];
                    }
#pragma unroll
                    for (int c = 0; c < 4; c++) {
                        int ic = i0[2] + c - 1; ic += ic < 0 ? A.grid[2] : 0; ic -= ic >= A.grid[2] ? A.grid[2] : 0;
                        const T w = f01 * F2(c);
                        const T u0 = g0 * F2(c), u1 = g1 * F2(c), u2 = f01 * D12(c); /* fractional gradient */
                        const T wx = u0 * (T)A.gm[0] + u1 * (T)A.gm[3] + u2 * (T)A.gm[6];
                        const T wy = u0 * (T)A.gm[1] + u1 * (T)A.gm[4] + u2 * (T)A.gm[7];
                        const T wz = u0 * (T)A.gm[2] + u1 * (T)A.gm[5] + u2 * (T)A.gm[8];
                        const T wl = (T)A.metric[0] * h00 * F2(c) + (T)A.metric[1] * h11 * F2(c) + (T)A.metric[2] * f01 * D22(c) +
                                     2 * ((T)A.metric[3] * h01 * F2(c) + (T)A.metric[4] * g0 * D12(c) + (T)A.metric[5] * g1 * D12(c));
                        const T *cp = A.coef + ((size_t)(ia * A.grid[1] + ib) * A.grid[2] + ic) * A.no_pad + ob + lane;
#pragma unroll
                        for (int q = 0; q < BLIP_OPL; q++) {
                            if (ob + 32 * q < A.no_pad) { /* uniform */
                                const T cc = __ldg(cp + 32 * q);
                                v[q] += cc * w; gx[q] += cc * wx; gy[q] += cc * wy; gz[q] += cc * wz; lp[q] += cc * wl;
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < BLIP_OPL; q++) {
                const int o = ob + 32 * q + lane;
                if (o < A.n_orb) {
                    /* streaming stores: the 1.3 GB of outputs of a launch must not push the coefficient table
                     * (14 MB, re-read 64 times per position) out of L2 */
                    __stcs(A.psi + (size_t)p * A.n_orb + o, (double)v[q]);
                    if (A.grad) {
                        __stcs(A.grad + ((size_t)p * 3 + 0) * A.n_orb + o, (double)gx[q]);
                        __stcs(A.grad + ((size_t)p * 3 + 1) * A.n_orb + o, (double)gy[q]);
                        __stcs(A.grad + ((size_t)p * 3 + 2) * A.n_orb + o, (double)gz[q]);
                    }
                    if (A.lap) __stcs(A.lap + (size_t)p * A.n_orb + o, (double)lp[q]);
                }
            }
        }
    }
}

#undef F2
#undef D12
#undef D22

struct blip_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int grid[3] = {0, 0, 0}, n_orb = 0, no_pad = 0, sm_count = 148;
    double binv[9], gm[9], metric[6];
    double *d_coef = nullptr;
    float *d_coeff = nullptr;
    bool prof = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> recs;
};

#define BCU(ctx, expr)                                                                           \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                     \
            return e_ == cudaErrorMemoryAllocation ? EWALD_ENOMEM : EWALD_ECUDA;                 \
        }                                                                                        \
    } while (0)

struct BDev {
    int prev = -1; bool ok = false;
    explicit BDev(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;
    }
    ~BDev() { if (prev >= 0) cudaSetDevice(prev); }
};

extern "C" const char *blip_last_error(const blip_ctx *c) { return c ? c->err.c_str() : ""; }

extern "C" void blip_destroy(blip_ctx *c)
{
    if (!c) return;
    BDev g(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_coef); cudaFree(c->d_coeff);
    for (auto &r : c->recs) { cudaEventDestroy(r.first); cudaEventDestroy(r.second); }
    delete c;
}

extern "C" ewald_status blip_setup(blip_ctx **out, const double *cell, const int *grid, int n_orb, const double *coef,
                                   int device, void *stream)
{
    if (!out) return EWALD_EINVAL;
    *out = nullptr;
    if (!cell || !grid || !coef || n_orb <= 0 || grid[0] < 4 || grid[1] < 4 || grid[2] < 4) return EWALD_EINVAL;
    long double A[3][3], B[3][3];
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) A[i][j] = cell[3 * i + j];
    const long double det = A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0]) +
                            A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
    if (!(fabsl(det) > 0)) return EWALD_ESINGULAR;
    blip_ctx *c = new (std::nothrow) blip_ctx;
    if (!c) return EWALD_ENOMEM;
    c->device = device; c->stream = (cudaStream_t)stream; c->n_orb = n_orb; c->no_pad = (n_orb + 31) & ~31;
    for (int i = 0; i < 3; i++) {
        const int i1 = (i + 1) % 3, i2 = (i + 2) % 3;
        B[i][0] = (A[i1][1] * A[i2][2] - A[i1][2] * A[i2][1]) / det;
        B[i][1] = (A[i1][2] * A[i2][0] - A[i1][0] * A[i2][2]) / det;
        B[i][2] = (A[i1][0] * A[i2][1] - A[i1][1] * A[i2][0]) / det;
        c->grid[i] = grid[i];
    }
    long double G[3][3];
    for (int k = 0; k < 3; k++) for (int x = 0; x < 3; x++) { c->binv[3 * k + x] = (double)B[k][x]; G[k][x] = grid[k] * B[k][x]; c->gm[3 * k + x] = (double)G[k][x]; }
    auto dot = [&](int k, int l) { long double s = 0; for (int x = 0; x < 3; x++) s += G[k][x] * G[l][x]; return (double)s; };
    c->metric[0] = dot(0, 0); c->metric[1] = dot(1, 1); c->metric[2] = dot(2, 2);
    c->metric[3] = dot(0, 1); c->metric[4] = dot(0, 2); c->metric[5] = dot(1, 2);
    BDev guard(device);
    if (!guard.ok) { delete c; return EWALD_ECUDA; }
    const size_t npts = (size_t)grid[0] * grid[1] * grid[2];
    std::vector<double> t64(npts * c->no_pad, 0.0);
    std::vector<float> t32(npts * c->no_pad, 0.0f);
    for (int o = 0; o < n_orb; o++)
        for (size_t pt = 0; pt < npts; pt++) {
            const double v = coef[(size_t)o * npts + pt];
            t64[pt * c->no_pad + o] = v; t32[pt * c->no_pad + o] = (float)v;
        }
    auto up = [&](void **dst, const void *src, size_t bytes) -> ewald_status {
        BCU(c, cudaMalloc(dst, bytes));
        BCU(c, cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
        return EWALD_OK;
    };
    ewald_status st = up((void **)&c->d_coef, t64.data(), t64.size() * sizeof(double));
    if (st == EWALD_OK) st = up((void **)&c->d_coeff, t32.data(), t32.size() * sizeof(float));
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && v > 0) c->sm_count = v;
    if (st != EWALD_OK) { blip_destroy(c); return st; }
    *out = c;
    return EWALD_OK;
}

template <typename T>
static ewald_status blip_launch(blip_ctx *c, int n_points, int n_pad, const T *points, const T *coef, double *psi, double *grad, double *lap)
{
    BlipArgs<T> A;
    A.points = points; A.n_points = n_points; A.n_pad = n_pad; A.coef = coef;
    for (int k = 0; k < 3; k++) A.grid[k] = c->grid[k];
    A.n_orb = c->n_orb; A.no_pad = c->no_pad;
    for (int i = 0; i < 9; i++) { A.binv[i] = c->binv[i]; A.gm[i] = c->gm[i]; }
    for (int i = 0; i < 6; i++) A.metric[i] = c->metric[i];
    A.psi = psi; A.grad = grad; A.lap = lap;
    const int warps_per_cta = BLIP_THREADS / 32;
    int blocks = (n_points + warps_per_cta - 1) / warps_per_cta;
    const int cap = c->sm_count * 8; /* persistent-style: every warp loops over positions */
    if (blocks > cap) blocks = cap;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (c->prof) { BCU(c, cudaEventCreate(&e0)); BCU(c, cudaEventCreate(&e1)); BCU(c, cudaEventRecord(e0, c->stream)); }
    blip_kernel<T><<<blocks, BLIP_THREADS, 0, c->stream>>>(A);
    if (c->prof) { BCU(c, cudaEventRecord(e1, c->stream)); c->recs.push_back({e0, e1}); }
    BCU(c, cudaGetLastError());
    return EWALD_OK;
}

extern "C" ewald_status blip_eval_batch(blip_ctx *c, int n_points, int n_pad, ewald_prec prec, const void *points,
                                        double *psi, double *grad, double *lap)
{
    if (!c) return EWALD_EINVAL;
    if (n_points < 0 || n_pad < n_points || (prec != EWALD_F64 && prec != EWALD_F32)) { c->err = "bad argument"; return EWALD_EINVAL; }
    if (n_points == 0) return EWALD_OK;
    if (!points || !psi) { c->err = "null points or psi"; return EWALD_EINVAL; }
    BDev g(c->device);
    if (!g.ok) { c->err = "cudaSetDevice failed"; return EWALD_ECUDA; }
    if (prec == EWALD_F64) return blip_launch<double>(c, n_points, n_pad, (const double *)points, c->d_coef, psi, grad, lap);
    return blip_launch<float>(c, n_points, n_pad, (const float *)points, c->d_coeff, psi, grad, lap);
}

extern "C" ewald_status blip_profile_enable(blip_ctx *c, int on)
{
    if (!c) return EWALD_EINVAL;
    c->prof = on != 0;
    return EWALD_OK;
}

extern "C" ewald_status blip_profile_read(blip_ctx *c, double *ms, int *launches)
{
    if (!c || !ms || !launches) return EWALD_EINVAL;
    BDev g(c->device);
    BCU(c, cudaStreamSynchronize(c->stream));
    double total = 0;
    for (auto &r : c->recs) {
        float t = 0;
        if (cudaEventElapsedTime(&t, r.first, r.second) == cudaSuccess) total += t;
        cudaEventDestroy(r.first); cudaEventDestroy(r.second);
    }
    *ms = total; *launches = (int)c->recs.size();
    c->recs.clear();
    return EWALD_OK;
}
