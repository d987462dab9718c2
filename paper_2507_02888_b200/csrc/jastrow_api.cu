/* jastrow_api.cu -- the C ABI of include/jastrow.h: context, device tables, launches.  No CPU fallback. */
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "jastrow.h"
#include "jastrow_kernels.cuh"

using namespace ewald;

struct jastrow_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    JasTabs t;
    short4 *d_gn = nullptr;
    double *d_ga = nullptr, *d_acoef = nullptr;
    int n_g_pad = 0;
    /* stored population */
    void *st_pos = nullptr, *st_S = nullptr;
    int st_w = 0, st_n = 0, st_npad = 0;
    ewald_prec st_prec = EWALD_F64;
    bool loaded = false;
    /* profile */
    bool prof = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> recs;
};

#define JCU(ctx, expr)                                                                           \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                     \
            return e_ == cudaErrorMemoryAllocation ? EWALD_ENOMEM : EWALD_ECUDA;                 \
        }                                                                                        \
    } while (0)

struct JDev {
    int prev = -1; bool ok = false;
    explicit JDev(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;
    }
    ~JDev() { if (prev >= 0) cudaSetDevice(prev); }
};

static ewald_status jfail(jastrow_ctx *c, ewald_status s, const char *m) { if (c) c->err = m; return s; }

extern "C" const char *jastrow_last_error(const jastrow_ctx *c) { return c ? c->err.c_str() : ""; }

extern "C" void jastrow_destroy(jastrow_ctx *c)
{
    if (!c) return;
    JDev g(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_gn); cudaFree(c->d_ga); cudaFree(c->d_acoef); cudaFree(c->st_pos); cudaFree(c->st_S);
    for (auto &r : c->recs) { cudaEventDestroy(r.first); cudaEventDestroy(r.second); }
    delete c;
}

extern "C" ewald_status jastrow_setup(jastrow_ctx **out, int dim, const double *cell, int n_u, const double *alpha,
                                      double l_u, int c_exp, int n_g, const int *g_n, const int *star, int n_stars,
                                      const double *a, int device, void *stream)
{
    if (!out) return EWALD_EINVAL;
    *out = nullptr;
    if ((dim != 2 && dim != 3) || !cell || n_g < 0 || n_u >= JAS_MAXU || c_exp < 0) return EWALD_EINVAL;
    if (n_u >= 0 && (!alpha || !(l_u > 0))) return EWALD_EINVAL;
    if (n_g > 0 && (!g_n || !star || !a || n_stars <= 0)) return EWALD_EINVAL;
    if (n_g > JAS_THREADS) return EWALD_ERANGE;
    jastrow_ctx *c = new (std::nothrow) jastrow_ctx;
    if (!c) return EWALD_ENOMEM;
    c->device = device; c->stream = (cudaStream_t)stream;
    JasTabs &t = c->t;
    std::memset(&t, 0, sizeof t);
    /* lattice rows (dim = 2 embedded with a3 = (0, 0, 1)), reciprocal rows / 2 pi, in long double */
    long double A[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}}, B[3][3];
    if (dim == 3) for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) A[i][j] = cell[3 * i + j];
    else { A[0][0] = cell[0]; A[0][1] = cell[1]; A[1][0] = cell[3]; A[1][1] = cell[4]; }
    const long double det = A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0]) +
                            A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
    if (!(fabsl(det) > 0)) { delete c; return EWALD_ESINGULAR; }
    for (int i = 0; i < 3; i++) {
        const int i1 = (i + 1) % 3, i2 = (i + 2) % 3;
        B[i][0] = (A[i1][1] * A[i2][2] - A[i1][2] * A[i2][1]) / det;
        B[i][1] = (A[i1][2] * A[i2][0] - A[i1][0] * A[i2][2]) / det;
        B[i][2] = (A[i1][0] * A[i2][1] - A[i1][1] * A[i2][0]) / det;
    }
    t.ortho = 1;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            t.a[3 * i + j] = (double)A[i][j]; t.binv[3 * i + j] = (double)B[i][j];
            if (i != j && A[i][j] != 0) t.ortho = 0;
        }
    t.dim = dim; t.n_g = n_g; t.n_u = n_u; t.c_exp = c_exp; t.l_u = n_u >= 0 ? l_u : 0.0;
    for (int l = 0; l <= n_u; l++) t.alpha[l] = alpha[l];
    if (n_u >= 0) { /* L_u below half the distance to the nearest lattice point */
        long double shortest = 1e300L;
        for (int m0 = -2; m0 <= 2; m0++) for (int m1 = -2; m1 <= 2; m1++) for (int m2 = (dim == 3 ? -2 : 0); m2 <= (dim == 3 ? 2 : 0); m2++) {
            if (!m0 && !m1 && !m2) continue;
            long double v2 = 0;
            for (int x = 0; x < 3; x++) { const long double v = m0 * A[0][x] + m1 * A[1][x] + m2 * A[2][x]; v2 += v * v; }
            if (sqrtl(v2) < shortest) shortest = sqrtl(v2);
        }
        if (!(l_u < 0.5L * shortest)) { delete c; return EWALD_ERANGE; }
    }
    std::vector<short4> gn(n_g);
    std::vector<double> ga((size_t)4 * n_g), ac(n_g);
    const long double two_pi = 6.283185307179586476925286766559L;
    for (int g = 0; g < n_g; g++) {
        int mx = 0;
        for (int k = 0; k < 3; k++) mx = std::max(mx, std::abs(g_n[3 * g + k]));
        if (mx >= JAS_MAXP || star[g] < 0 || star[g] >= n_stars) { delete c; return EWALD_ERANGE; }
        t.mmax = std::max(t.mmax, mx);
        gn[g] = make_short4((short)g_n[3 * g], (short)g_n[3 * g + 1], (short)(dim == 3 ? g_n[3 * g + 2] : 0), (short)star[g]);
        long double G[3] = {0, 0, 0}, g2 = 0;
        for (int k = 0; k < dim; k++) for (int x = 0; x < 3; x++) G[x] += two_pi * g_n[3 * g + k] * B[k][x];
        for (int x = 0; x < 3; x++) g2 += G[x] * G[x];
        ac[g] = a[star[g]];
        for (int x = 0; x < 3; x++) ga[4 * g + x] = (double)(a[star[g]] * G[x]);
        ga[4 * g + 3] = (double)(a[star[g]] * g2);
    }
    c->n_g_pad = (n_g + 31) & ~31;
    JDev guard(device);
    if (!guard.ok) { delete c; return EWALD_ECUDA; }
    ewald_status st = EWALD_OK;
    auto up = [&](void **dst, const void *src, size_t bytes) -> ewald_status {
        if (!bytes) return EWALD_OK;
        JCU(c, cudaMalloc(dst, bytes));
        JCU(c, cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
        return EWALD_OK;
    };
    st = up((void **)&c->d_gn, gn.data(), gn.size() * sizeof(short4));
    if (st == EWALD_OK) st = up((void **)&c->d_ga, ga.data(), ga.size() * sizeof(double));
    if (st == EWALD_OK) st = up((void **)&c->d_acoef, ac.data(), ac.size() * sizeof(double));
    if (st != EWALD_OK) { jastrow_destroy(c); return st; }
    t.gn = c->d_gn; t.ga = c->d_ga; t.acoef = c->d_acoef;
    *out = c;
    return EWALD_OK;
}

template <typename T>
static ewald_status jas_launch(jastrow_ctx *c, int W, int n, const T *pos, double *value, double *grad, double *lap, T *s_out)
{
    typedef typename Num<T>::T2 T2;
    JasArgs<T> A;
    A.pos = pos; A.n = n; A.npad = ewald_padded_n(n); A.t = c->t;
    A.value = value; A.grad = grad; A.lap = lap; A.s_out = s_out; A.n_g_pad = c->n_g_pad;
    const int dim = c->t.dim, np = c->t.mmax + 1;
    const size_t smem = (size_t)((dim * n + 3) & ~3) * sizeof(T) + ((size_t)c->t.n_g + (size_t)JAS_CHUNK * dim * np) * sizeof(T2);
    if (smem > 200 * 1024) return jfail(c, EWALD_ERANGE, "too many particles for shared memory");
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (c->prof) { JCU(c, cudaEventCreate(&e0)); JCU(c, cudaEventCreate(&e1)); JCU(c, cudaEventRecord(e0, c->stream)); }
    if (dim == 3) {
        if (smem > 48 * 1024) JCU(c, cudaFuncSetAttribute(jastrow_kernel<T, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        jastrow_kernel<T, 3><<<W, JAS_THREADS, smem, c->stream>>>(A);
    } else {
        if (smem > 48 * 1024) JCU(c, cudaFuncSetAttribute(jastrow_kernel<T, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        jastrow_kernel<T, 2><<<W, JAS_THREADS, smem, c->stream>>>(A);
    }
    if (c->prof) { JCU(c, cudaEventRecord(e1, c->stream)); c->recs.push_back({e0, e1}); }
    JCU(c, cudaGetLastError());
    return EWALD_OK;
}

extern "C" ewald_status jastrow_batch(jastrow_ctx *c, int W, int n, ewald_prec prec, const void *pos,
                                      double *value, double *grad, double *lap)
{
    if (!c) return EWALD_EINVAL;
    if (W < 0 || n <= 0 || (prec != EWALD_F64 && prec != EWALD_F32)) return jfail(c, EWALD_EINVAL, "bad argument");
    if (W == 0) return EWALD_OK;
    if (!pos || !value) return jfail(c, EWALD_EINVAL, "null positions or value");
    JDev g(c->device);
    if (!g.ok) return jfail(c, EWALD_ECUDA, "cudaSetDevice failed");
    if (prec == EWALD_F64) return jas_launch<double>(c, W, n, (const double *)pos, value, grad, lap, nullptr);
    return jas_launch<float>(c, W, n, (const float *)pos, value, grad, lap, nullptr);
}

extern "C" ewald_status jastrow_load_walkers(jastrow_ctx *c, int W, int n, ewald_prec prec, const void *pos)
{
    if (!c) return EWALD_EINVAL;
    if (W <= 0 || n <= 0 || !pos || (prec != EWALD_F64 && prec != EWALD_F32)) return jfail(c, EWALD_EINVAL, "bad argument");
    JDev g(c->device);
    if (!g.ok) return jfail(c, EWALD_ECUDA, "cudaSetDevice failed");
    const size_t es = prec == EWALD_F64 ? 8 : 4;
    const int npad = ewald_padded_n(n);
    JCU(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->st_pos); cudaFree(c->st_S); c->st_pos = c->st_S = nullptr; c->loaded = false;
    const size_t pb = (size_t)W * c->t.dim * npad * es, sb = (size_t)W * 2 * (c->n_g_pad ? c->n_g_pad : 32) * es;
    JCU(c, cudaMalloc(&c->st_pos, pb));
    JCU(c, cudaMalloc(&c->st_S, sb));
    JCU(c, cudaMemcpyAsync(c->st_pos, pos, pb, cudaMemcpyDeviceToDevice, c->stream));
    JCU(c, cudaMemsetAsync(c->st_S, 0, sb, c->stream));
    c->st_w = W; c->st_n = n; c->st_npad = npad; c->st_prec = prec;
    /* S(G) by the batch kernel (value into a scratch slot of the S buffer is avoided: a one-double scratch) */
    double *scratch = nullptr;
    JCU(c, cudaMalloc((void **)&scratch, (size_t)W * sizeof(double)));
    const bool prof = c->prof; c->prof = false;
    ewald_status st = prec == EWALD_F64 ? jas_launch<double>(c, W, n, (const double *)c->st_pos, scratch, nullptr, nullptr, (double *)c->st_S)
                                        : jas_launch<float>(c, W, n, (const float *)c->st_pos, scratch, nullptr, nullptr, (float *)c->st_S);
    c->prof = prof;
    cudaStreamSynchronize(c->stream);
    cudaFree(scratch);
    if (st != EWALD_OK) return st;
    c->loaded = true;
    return EWALD_OK;
}

template <typename T>
static ewald_status jas_move(jastrow_ctx *c, int n_moves, const int *walker, const int *electron, const T *new_r, int commit, double *delta)
{
    JasMoveArgs<T> A;
    A.pos = (T *)c->st_pos; A.S = (T *)c->st_S; A.n = c->st_n; A.npad = c->st_npad; A.n_walkers = c->st_w;
    A.n_g_pad = c->n_g_pad ? c->n_g_pad : 32; A.n_moves = n_moves; A.t = c->t;
    A.walker = walker; A.electron = electron; A.new_r = new_r; A.commit = commit; A.delta = delta;
    if (c->t.dim == 3) jastrow_move_kernel<T, 3><<<n_moves, JAS_MOVE_THREADS, 0, c->stream>>>(A);
    else jastrow_move_kernel<T, 2><<<n_moves, JAS_MOVE_THREADS, 0, c->stream>>>(A);
    JCU(c, cudaGetLastError());
    return EWALD_OK;
}

extern "C" ewald_status jastrow_move_delta_batch(jastrow_ctx *c, int n_moves, const int *walker, const int *electron,
                                                 const void *new_r, int commit, double *delta)
{
    if (!c) return EWALD_EINVAL;
    if (!c->loaded) return jfail(c, EWALD_ESTATE, "no walkers loaded");
    if (n_moves < 0) return jfail(c, EWALD_EINVAL, "n_moves < 0");
    if (n_moves == 0) return EWALD_OK;
    if (!walker || !electron || !new_r || !delta) return jfail(c, EWALD_EINVAL, "null argument");
    JDev g(c->device);
    if (!g.ok) return jfail(c, EWALD_ECUDA, "cudaSetDevice failed");
    if (c->st_prec == EWALD_F64) return jas_move<double>(c, n_moves, walker, electron, (const double *)new_r, commit, delta);
    return jas_move<float>(c, n_moves, walker, electron, (const float *)new_r, commit, delta);
}

extern "C" ewald_status jastrow_profile_enable(jastrow_ctx *c, int on)
{
    if (!c) return EWALD_EINVAL;
    c->prof = on != 0;
    return EWALD_OK;
}

extern "C" ewald_status jastrow_profile_read(jastrow_ctx *c, double *ms, int *launches)
{
    if (!c || !ms || !launches) return EWALD_EINVAL;
    JDev g(c->device);
    JCU(c, cudaStreamSynchronize(c->stream));
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
