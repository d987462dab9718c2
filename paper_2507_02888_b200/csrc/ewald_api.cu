/* ewald_api.cu -- the C ABI of include/ewald.h: context, device tables, launches.
 * No torch types; plain pointers and sizes.  No CPU fallback: every compute entry point launches
 * the sm_100a kernels of ewald_kernels.cuh or fails with EWALD_ECUDA. */
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "ewald.h"
#include "ewald_internal.h"
#include "ewald_kernels.cuh"
#include "ewald_recip_oct.cuh"
#include "ewald_recip_mma.cuh"
#include <map>

using namespace ewald;

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
};

struct ProfRec {
    int kind;
    cudaEvent_t a, b;
};

/* Device copy of one OctLaunch and the launch shape chosen for it. */
struct OctDev {
    OctLaunch L;
    int4 *d_lane = nullptr;
    int *d_variant = nullptr;
    int pc = 0, wstride = 0;
    size_t smem = 0;
};

/* Device copy of one MmaLaunch. */
struct MmaDev {
    MmaLaunch L;
    int2 *d_lane = nullptr;
    int4 *d_meta = nullptr;
};

struct ewald_ctx {
    bool prof = false;
    int recip_variant = 0;                 /* 0 auto, 1 complex half-set kernel, 2 octant FMA-pipe kernel, 3 octant DMMA kernel */
    double *d_oct_wt = nullptr, *d_oct_tion = nullptr;
    double *d_mma_wt = nullptr, *d_mma_tion = nullptr;
    std::map<int, MmaDev> mma_dev;         /* key: warps per walker */
    std::map<long long, OctDev> oct_dev;   /* key: wc | prec << 16 */
    std::map<long long, int> oct_choice;   /* key: W | prec << 40 | n << 41 ... -> wc */
    std::vector<ProfRec> recs;
    std::vector<void *> retired;           /* outgrown scratch buffers, freed at destroy */
    long long launches = 0; /* kernels launched since setup */
    int shape[2][8] = {{0}};               /* ewald_launch_shape: last real-space [0] and move [1] launch */
    HostTables t;
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int ngp = 0, ngp_pad = 0, nimg = 0;
    int off[3] = {0, 0, 0}, rowlen = 0;

    /* tables, FP64 and FP32 copies */
    short4 *d_gn = nullptr;
    double *d_w2 = nullptr; float *d_w2f = nullptr;
    double *d_img = nullptr; float *d_imgf = nullptr;
    double *d_ion_rho = nullptr; float *d_ion_rhof = nullptr;
    double *d_ion_pos = nullptr; float *d_ion_posf = nullptr;
    double *d_ion_q = nullptr; float *d_ion_qf = nullptr;
    double *d_pair = nullptr; float *d_pairf = nullptr;   /* pair-function table F(t) */
    float *d_far = nullptr;                               /* far-shell cubics (FP64 kernels) */
    int real_variant = 0;                                 /* 0: far shell t >= 16 in FP32; 1: every term in FP64 */
    int sm_count = 148; size_t smem_optin = 227 * 1024;

    /* scratch */
    DevBuf partial_recip, partial_real, qsums, done;
    DevBuf stage_pos, stage_q, stage_e, stage_comp;           /* *_host entry points */
    DevBuf mv_walker, mv_electron, mv_newr, mv_de;

    /* ewald_recip_energy_static: device address of the file-scope scratch array on this context's device (null:
     * the address could not be taken at set-up, static_err says why) */
    double *static_scratch = nullptr;
    std::string static_err;

    /* stored walker population */
    int st_walkers = 0, st_n = 0, st_npad = 0;
    ewald_prec st_prec = EWALD_F64;
    DevBuf st_pos, st_q, st_rho, st_qinfo;
    bool loaded = false;
};

static const char *kVersion = "ewald-b200 0.1 (sm_100a)";

#define CU_TRY(ctx, expr)                                                                        \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                     \
            return e_ == cudaErrorMemoryAllocation ? EWALD_ENOMEM : EWALD_ECUDA;                 \
        }                                                                                        \
    } while (0)

/* Brackets one kernel launch with events when profiling is on. */
struct ProfScope {
    ewald_ctx *c;
    ProfRec r;
    bool on;
    ProfScope(ewald_ctx *ctx, int kind) : c(ctx), on(ctx->prof)
    {
        c->launches++;
        if (!on) return;
        r.kind = kind;
        on = cudaEventCreate(&r.a) == cudaSuccess && cudaEventCreate(&r.b) == cudaSuccess &&
             cudaEventRecord(r.a, c->stream) == cudaSuccess;
    }
    ~ProfScope()
    {
        if (on && cudaEventRecord(r.b, c->stream) == cudaSuccess) c->recs.push_back(r);
    }
};

/* Makes the context's device current for one entry point and restores the caller's on exit. */
struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define EWALD_DEVICE(c)                                                                          \
    DeviceGuard guard_((c)->device);                                                             \
    if (!guard_.ok) { (c)->err = "cudaSetDevice failed"; return EWALD_ECUDA; }

static ewald_status fail(ewald_ctx *c, ewald_status s, const char *msg)
{
    if (c) c->err = msg;
    return s;
}

/* Grows a scratch buffer without synchronising the stream: kernels already enqueued may still use the old
 * allocation, so it is retired (freed by ewald_destroy or the next synchronising call), not freed here. */
static ewald_status ensure(ewald_ctx *c, DevBuf *b, size_t bytes)
{
    if (bytes <= b->cap) return EWALD_OK;
    if (b->p) { c->retired.push_back(b->p); b->p = nullptr; b->cap = 0; }
    size_t want = bytes + bytes / 4 + 256;
    CU_TRY(c, cudaMalloc(&b->p, want));
    b->cap = want;
    return EWALD_OK;
}

static void release(DevBuf *b)
{
    if (b->p) cudaFree(b->p);
    b->p = nullptr;
    b->cap = 0;
}

template <typename T>
static ewald_status upload(ewald_ctx *c, T **dst, const std::vector<T> &src)
{
    if (*dst) { CU_TRY(c, cudaFree(*dst)); *dst = nullptr; }
    if (src.empty()) return EWALD_OK;
    CU_TRY(c, cudaMalloc((void **)dst, src.size() * sizeof(T)));
    CU_TRY(c, cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return EWALD_OK;
}

static std::vector<float> to_f32(const std::vector<double> &v)
{
    std::vector<float> f(v.size());
    for (size_t i = 0; i < v.size(); i++) f[i] = (float)v[i];
    return f;
}

static int host_key(double t) { uint64_t b; std::memcpy(&b, &t, 8); return (int)(b >> 32); }
static int host_key(float t) { int b; std::memcpy(&b, &t, 4); return b; }
template <typename T> static const PairTable &pair_of(const HostTables &t);
template <> const PairTable &pair_of<double>(const HostTables &t) { return t.pair64; }
template <> const PairTable &pair_of<float>(const HostTables &t) { return t.pair32; }

/* Real-space geometry in kappa-scaled lengths (ewald_realspace.cuh). */
template <typename T> static void fill_geom(const HostTables &t, RealGeom<T> *g)
{
    for (int i = 0; i < 9; i++) {
        g->a[i] = (T)(t.a[i] * t.kappa); g->binv[i] = (T)(t.binv[i] / t.kappa);
        g->a_lo[i] = (T)(t.a[i] * t.kappa - (double)g->a[i]);
    }
    for (int k = 0; k < 3; k++) {
        const double l = t.a[4 * k], c2 = l * t.kappa * l * t.kappa;
        g->L[k] = (T)(l * t.kappa); g->invL[k] = (T)(1.0 / (l * t.kappa));
        g->invLu[k] = (T)(1.0 / l); g->invLu_lo[k] = (T)(1.0 / l - (double)g->invLu[k]);
        g->C[k] = (T)c2; g->C_lo[k] = (T)(c2 - (double)g->C[k]);
    }
    g->kappa = (T)t.kappa;
    g->kappa_lo = (T)(t.kappa - (double)g->kappa); /* zero in FP64 */
    g->kappa_d = t.kappa;
    g->m_shift = t.m_shift;
    g->multi_far = 0;
    g->outer_far = 0; g->far_once = 0; /* set by set_outer_far once the far shell and the capacities are known */
    {
        const double rc2 = t.r_cutoff * t.r_cutoff * (1 + 1e-5);
        for (int j = 0; j < 3; j++)
            for (int k = j + 1; k < 3; k++)
                if (t.a[4 * j] * t.a[4 * j] + t.a[4 * k] * t.a[4 * k] < rc2) g->multi_far = 1;
    }
    g->key_rc = host_key((T)(t.r_cutoff * t.r_cutoff * t.kappa * t.kappa));
    g->key_min = host_key((T)pair_of<T>(t).t_min);
    g->bias = (PairFmt<T>::EBIAS + pair_of<T>(t).e_min) << PairFmt<T>::K;
}

static std::vector<double> scaled(const std::vector<double> &v, double f)
{
    std::vector<double> o(v);
    for (double &x : o) x *= f;
    return o;
}

extern "C" int ewald_padded_n(int n) { return n <= 0 ? 0 : (n + 3) & ~3; }
extern "C" const char *ewald_version(void) { return kVersion; }
extern "C" const char *ewald_last_error(const ewald_ctx *c) { return c ? c->err.c_str() : ""; }

/* ---- scratch of the allocation-free entry point (ewald_recip_energy_static, end of this file) ----
 * One file-scope device array per GPU that loads the library, held until the process exits.  In HOST code the name
 * `g_static_scratch` is only a stand-in for the symbol, not a device address: the address is taken once per device,
 * at set-up, with that device current, by cudaGetSymbolAddress, and it is that pointer the kernels receive. */
static_assert(EWALD_STATIC_SCRATCH_BYTES % 256 == 0, "scratch size");
constexpr size_t STATIC_SCRATCH_DOUBLES = EWALD_STATIC_SCRATCH_BYTES / sizeof(double);
static __device__ __align__(256) double g_static_scratch[STATIC_SCRATCH_DOUBLES];

constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_static_mutex;
static bool g_static_tried[STATIC_MAX_DEVICES];
static double *g_static_addr[STATIC_MAX_DEVICES];
static cudaError_t g_static_status[STATIC_MAX_DEVICES];

/* Call with c->device current.  A failure does not fail the set-up: only the static entry point needs the address
 * and it reports the recorded error. */
static void resolve_static_scratch(ewald_ctx *c)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    const int d = c->device;
    double *ptr = nullptr;
    cudaError_t e;
    if (d >= 0 && d < STATIC_MAX_DEVICES && g_static_tried[d]) {
        ptr = g_static_addr[d]; e = g_static_status[d];
    } else {
        e = cudaGetSymbolAddress((void **)&ptr, g_static_scratch);
        if (e != cudaSuccess) { ptr = nullptr; (void)cudaGetLastError(); }
        if (d >= 0 && d < STATIC_MAX_DEVICES) { g_static_tried[d] = true; g_static_addr[d] = ptr; g_static_status[d] = e; }
    }
    c->static_scratch = ptr;
    if (e != cudaSuccess) c->static_err = std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e);
}

extern "C" ewald_status ewald_setup(ewald_ctx **out, int dim, const double *cell, double gamma,
                                    double g_cutoff, const ewald_opts *opts)
{
    if (!out) return EWALD_EINVAL;
    *out = nullptr;
    ewald_ctx *c = new (std::nothrow) ewald_ctx;
    if (!c) return EWALD_ENOMEM;
    std::string err;
    ewald_status st = build_tables(dim, cell, gamma, g_cutoff, opts ? opts->r_cutoff : 0.0, &c->t, &err);
    if (st != EWALD_OK) { delete c; return st; }
    c->device = opts ? opts->device : 0;
    c->stream = opts ? (cudaStream_t)opts->stream : nullptr;
    DeviceGuard guard_(c->device);
    if (!guard_.ok) { delete c; return EWALD_ECUDA; }
    resolve_static_scratch(c);

    const HostTables &t = c->t;
    c->ngp = (int)t.g_w2.size();
    c->ngp_pad = (c->ngp + 31) & ~31;
    c->nimg = (int)(t.img.size() / 3);
    int o = 0;
    for (int k = 0; k < 3; k++) { c->off[k] = o; if (k < dim) o += t.n_max[k] + 1; }
    c->rowlen = o;

    std::vector<short4> gn(c->ngp);
    for (int g = 0; g < c->ngp; g++)
        gn[g] = make_short4((short)t.g_n[3 * g], (short)t.g_n[3 * g + 1], (short)t.g_n[3 * g + 2], 0);
    st = upload(c, &c->d_gn, gn);
    if (st == EWALD_OK) st = upload(c, &c->d_w2, t.g_w2);
    if (st == EWALD_OK) st = upload(c, &c->d_w2f, to_f32(t.g_w2));
    if (st == EWALD_OK) st = upload(c, &c->d_img, scaled(t.img, t.kappa));
    {   /* FP32 image list: high parts, then the low parts (ewald_realspace.cuh, RealGeom) */
        const std::vector<double> im = scaled(t.img, t.kappa);
        std::vector<float> hl(2 * im.size());
        for (size_t i = 0; i < im.size(); i++) { hl[i] = (float)im[i]; hl[im.size() + i] = (float)(im[i] - (double)hl[i]); }
        if (st == EWALD_OK) st = upload(c, &c->d_imgf, hl);
    }
    {   /* FP64 table in 512-byte rows [chunk][slot][2] (PairFmt<double>): 8 bins per row below t = 2^E_SPLIT, one bin in
         * 8 copies per row above */
        typedef PairFmt<double> F;
        static_assert(F::K == PAIR_K64 && F::DEG == PAIR_DEG64 && F::NC == PAIR_DEG64 + 1 && F::E_MIN == PAIR_EMIN,
                      "device and host formats of the FP64 pair table differ");
        const PairTable &pt = t.pair64;
        std::vector<double> rows(F::elems(pt.n_bins), 0.0);
        for (int b = 0; b < pt.n_bins; b++)
            for (int ch = 0; ch < 4; ch++) {
                const double c0 = pt.coef[(size_t)b * F::NC + 2 * ch], c1 = pt.coef[(size_t)b * F::NC + 2 * ch + 1];
                const size_t row = b < F::LOW ? b >> 3 : F::LOW / 8 + (b - F::LOW);
                for (int s = b < F::LOW ? (b & 7) : 0; s < (b < F::LOW ? (b & 7) + 1 : 8); s++) {
                    rows[row * F::ROW + (size_t)ch * 16 + 2 * s] = c0;
                    rows[row * F::ROW + (size_t)ch * 16 + 2 * s + 1] = c1;
                }
            }
        if (st == EWALD_OK) st = upload(c, &c->d_pair, rows);
    }
    {   /* FP32 table: PairFmt<float>::REP interleaved copies */
        const std::vector<float> one = to_f32(t.pair32.coef);
        constexpr int R = PairFmt<float>::REP, NCF = PairFmt<float>::NC;
        std::vector<float> rep(one.size() * R);
        for (size_t b = 0; b < one.size() / NCF; b++)
            for (int r = 0; r < R; r++)
                for (int k = 0; k < NCF; k++) rep[(b * R + r) * NCF + k] = one[b * NCF + k];
        if (st == EWALD_OK) st = upload(c, &c->d_pairf, rep);
    }
    if (st == EWALD_OK) st = upload(c, &c->d_far, t.far_tab);
    if (st == EWALD_OK) st = ensure(c, &c->qsums, 4 * sizeof(double));
    if (st == EWALD_OK) st = ensure(c, &c->st_qinfo, 4 * sizeof(double));
    {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && v > 0) c->sm_count = v;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device) == cudaSuccess && v > 0)
            c->smem_optin = (size_t)v;
    }
    if (st == EWALD_OK && t.oct.valid) {
        std::vector<double> wt(t.oct.wt);
        wt.resize(wt.size() + (size_t)(t.oct.npb + 1) * 4, 0.0); /* the zero-weight dummy item */
        st = upload(c, &c->d_oct_wt, wt);
    }
    if (st == EWALD_OK && t.mma.valid) st = upload(c, &c->d_mma_wt, t.mma.wt);
    if (st != EWALD_OK) { ewald_destroy(c); return st; }
    *out = c;
    return EWALD_OK;
}

extern "C" ewald_status ewald_setup_summary(int dim, const double *cell, double gamma, double g_cutoff,
                                            double r_cutoff, int *num_g, int *num_images, int *n_max,
                                            double *xi_r, double *v_m)
{
    HostTables t;
    std::string err;
    ewald_status st = build_tables(dim, cell, gamma, g_cutoff, r_cutoff, &t, &err);
    if (st != EWALD_OK) return st;
    if (num_g) *num_g = 2 * (int)t.g_w2.size();
    if (num_images) *num_images = (int)(t.img.size() / 3);
    if (n_max) for (int k = 0; k < 3; k++) n_max[k] = t.n_max[k];
    if (xi_r) *xi_r = t.xi_r;
    if (v_m) *v_m = t.v_m;
    return EWALD_OK;
}

extern "C" ewald_status ewald_oct_plan_summary(int dim, const double *cell, double gamma, double g_cutoff,
                                               int n_walkers_per_cta, int *n_items, int *npb, int *n_warps,
                                               double *weight_sum, double *fma_per_particle)
{
    HostTables t;
    std::string err;
    ewald_status st = build_tables(dim, cell, gamma, g_cutoff, 0.0, &t, &err);
    if (st != EWALD_OK) return st;
    if (!t.oct.valid) return EWALD_ESTATE;
    if (n_walkers_per_cta < 1) return EWALD_EINVAL;
    const OctPlan &P = t.oct;
    long double ws = 0;
    for (int it = 0; it < P.n_items; it++)
        for (int j = 0; j <= P.npb; j++)
            for (int cls = 0; cls < 4; cls++) ws += P.wt[((size_t)it * (P.npb + 1) + j) * 4 + cls];
    OctLaunch L;
    make_oct_launch(P, n_walkers_per_cta, 1 << 20, &L);
    if (n_items) *n_items = P.n_items;
    if (npb) *npb = P.npb;
    if (n_warps) *n_warps = L.n_warps;
    if (weight_sum) *weight_sum = (double)ws;
    if (fma_per_particle) *fma_per_particle = L.fma_ops / n_walkers_per_cta;
    return EWALD_OK;
}

extern "C" ewald_status ewald_mma_plan_summary(int dim, const double *cell, double gamma, double g_cutoff,
                                               int *n_slots, int *walkers_per_pass, double *weight_sum,
                                               double *dmma_per_quad)
{
    HostTables t;
    std::string err;
    ewald_status st = build_tables(dim, cell, gamma, g_cutoff, 0.0, &t, &err);
    if (st != EWALD_OK) return st;
    if (!t.mma.valid) return EWALD_ESTATE;
    long double ws = 0;
    for (double v : t.mma.wt) ws += v;
    int cap = 0;
    for (int nw = MMA_WARPS; nw >= 1 && !cap; nw--) {
        MmaLaunch L;
        make_mma_launch(t.mma, MMA_WARPS / nw, &L);
        if (L.valid) cap = nw;
    }
    if (n_slots) *n_slots = (int)t.mma.slots.size();
    if (walkers_per_pass) *walkers_per_pass = cap;
    if (weight_sum) *weight_sum = (double)ws;
    if (dmma_per_quad) *dmma_per_quad = t.mma.dmma_per_quad;
    return EWALD_OK;
}

extern "C" ewald_status ewald_pair_table_eval(ewald_prec prec, double t_max, int n, const double *t, double *value)
{
    if (!(t_max > 0) || n < 0 || (n > 0 && (!t || !value))) return EWALD_EINVAL;
    if (prec != EWALD_F64 && prec != EWALD_F32) return EWALD_EINVAL;
    PairTable p;
    if (prec == EWALD_F64) build_pair_table(PAIR_K64, PAIR_DEG64, PAIR_EMIN, t_max, &p);
    else build_pair_table(PAIR_K32, PAIR_DEG32, PAIR_EMIN, t_max, &p);
    for (int i = 0; i < n; i++) value[i] = eval_pair_table(p, t[i]);
    return EWALD_OK;
}

extern "C" void ewald_destroy(ewald_ctx *c)
{
    if (!c) return;
    DeviceGuard guard_(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_gn); cudaFree(c->d_w2); cudaFree(c->d_w2f); cudaFree(c->d_img); cudaFree(c->d_imgf);
    cudaFree(c->d_ion_rho); cudaFree(c->d_ion_rhof); cudaFree(c->d_ion_pos); cudaFree(c->d_ion_posf);
    cudaFree(c->d_ion_q); cudaFree(c->d_ion_qf); cudaFree(c->d_pair); cudaFree(c->d_pairf); cudaFree(c->d_far);
    cudaFree(c->d_oct_wt); cudaFree(c->d_oct_tion); cudaFree(c->d_mma_wt); cudaFree(c->d_mma_tion);
    for (auto &kv : c->mma_dev) { cudaFree(kv.second.d_lane); cudaFree(kv.second.d_meta); }
    for (auto &kv : c->oct_dev) { cudaFree(kv.second.d_lane); cudaFree(kv.second.d_variant); }
    DevBuf *bufs[] = {&c->partial_recip, &c->partial_real, &c->qsums, &c->done, &c->stage_pos, &c->stage_q,
                      &c->stage_e, &c->stage_comp, &c->mv_walker, &c->mv_electron, &c->mv_newr,
                      &c->mv_de, &c->st_pos, &c->st_q, &c->st_rho, &c->st_qinfo};
    for (DevBuf *b : bufs) release(b);
    for (ProfRec &r : c->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (void *p : c->retired) cudaFree(p);
    delete c;
}

extern "C" ewald_status ewald_set_recip_variant(ewald_ctx *c, int variant)
{
    if (!c || variant < 0 || variant > 3) return EWALD_EINVAL;
    c->recip_variant = variant;
    return EWALD_OK;
}

extern "C" ewald_status ewald_set_real_variant(ewald_ctx *c, int variant)
{
    if (!c || variant < 0 || variant > 1) return EWALD_EINVAL;
    c->real_variant = variant;
    return EWALD_OK;
}

extern "C" ewald_status ewald_set_stream(ewald_ctx *c, void *stream)
{
    if (!c) return EWALD_EINVAL;
    c->stream = (cudaStream_t)stream;
    return EWALD_OK;
}

extern "C" ewald_status ewald_set_fixed_charges(ewald_ctx *c, int n_ion, const double *pos, const double *q)
{
    if (!c) return EWALD_EINVAL;
    EWALD_DEVICE(c);
    std::string err;
    ewald_status st = build_fixed_charges(&c->t, n_ion, pos, q, &err);
    if (st != EWALD_OK) return fail(c, st, err.c_str());
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    const HostTables &t = c->t;
    st = upload(c, &c->d_ion_rho, n_ion ? t.ion_rho : std::vector<double>());
    if (st == EWALD_OK) st = upload(c, &c->d_ion_rhof, n_ion ? to_f32(t.ion_rho) : std::vector<float>());
    if (st == EWALD_OK) st = upload(c, &c->d_ion_pos, t.ion_pos);
    if (st == EWALD_OK) st = upload(c, &c->d_ion_posf, to_f32(t.ion_pos));
    if (st == EWALD_OK) st = upload(c, &c->d_ion_q, t.ion_q);
    if (st == EWALD_OK) st = upload(c, &c->d_ion_qf, to_f32(t.ion_q));
    if (st == EWALD_OK) {
        std::vector<double> ti(t.oct.tion);
        if (!ti.empty()) ti.resize(ti.size() + (size_t)(1 + 2 * t.oct.npb) * 4, 0.0);
        st = upload(c, &c->d_oct_tion, ti);
    }
    if (st == EWALD_OK) st = upload(c, &c->d_mma_tion, t.mma.tion);
    c->loaded = false; /* a stored rho(G) would no longer match */
    return st;
}

/* ---- launches ---------------------------------------------------------------------------- */

template <typename T> struct Tabs;
template <> struct Tabs<double> {
    static const double *w2(const ewald_ctx *c) { return c->d_w2; }
    static const double *img(const ewald_ctx *c) { return c->d_img; }
    static const double *ion_rho(const ewald_ctx *c) { return c->d_ion_rho; }
    static const double *ion_pos(const ewald_ctx *c) { return c->d_ion_pos; }
    static const double *ion_q(const ewald_ctx *c) { return c->d_ion_q; }
    static const double *pair(const ewald_ctx *c) { return c->d_pair; }
};
template <> struct Tabs<float> {
    static const float *w2(const ewald_ctx *c) { return c->d_w2f; }
    static const float *img(const ewald_ctx *c) { return c->d_imgf; }
    static const float *ion_rho(const ewald_ctx *c) { return c->d_ion_rhof; }
    static const float *ion_pos(const ewald_ctx *c) { return c->d_ion_posf; }
    static const float *ion_q(const ewald_ctx *c) { return c->d_ion_qf; }
    static const float *pair(const ewald_ctx *c) { return c->d_pairf; }
};

template <typename K> static ewald_status allow_smem(ewald_ctx *c, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024) {
        if (bytes > c->smem_optin) return fail(c, EWALD_ERANGE, "problem too large for shared memory");
        CU_TRY(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    }
    return EWALD_OK;
}

template <typename T>
static ewald_status launch_recip(ewald_ctx *c, int W, int n, const T *pos, const T *q, T *rho_out,
                                 int *n_slabs_out)
{
    typedef typename Num<T>::T2 T2;
    const int per = RECIP_THREADS * RECIP_GPT;
    const int n_slabs = (c->ngp + per - 1) / per;
    ewald_status st = ensure(c, &c->partial_recip, (size_t)W * n_slabs * sizeof(double));
    if (st != EWALD_OK) return st;
    RecipArgs<T> A;
    A.pos = pos; A.q = q; A.n = n; A.npad = ewald_padded_n(n);
    A.gn = c->d_gn; A.w2 = Tabs<T>::w2(c); A.ion_rho = c->t.n_ion ? Tabs<T>::ion_rho(c) : nullptr;
    A.ngp = c->ngp; A.ngp_pad = c->ngp_pad;
    for (int k = 0; k < 3; k++) { A.nmax[k] = c->t.n_max[k]; A.off[k] = c->off[k]; }
    A.rowlen = c->rowlen;
    A.rho_out = rho_out;
    A.partial = (double *)c->partial_recip.p;
    A.n_slabs = n_slabs;
    for (int i = 0; i < 9; i++) A.binv[i] = c->t.binv[i];
    const size_t smem = (size_t)RECIP_CHUNK * c->rowlen * sizeof(T2);
    const long long grid = (long long)W * n_slabs;
    if (grid > 0x7fffffffLL) return fail(c, EWALD_ERANGE, "grid too large");
    if (c->t.dim == 3) {
        st = allow_smem(c, recip_kernel<T, 3>, smem);
        if (st != EWALD_OK) return st;
        ProfScope ps(c, 0);
        recip_kernel<T, 3><<<(unsigned)grid, RECIP_THREADS, smem, c->stream>>>(A);
    } else {
        st = allow_smem(c, recip_kernel<T, 2>, smem);
        if (st != EWALD_OK) return st;
        ProfScope ps(c, 0);
        recip_kernel<T, 2><<<(unsigned)grid, RECIP_THREADS, smem, c->stream>>>(A);
    }
    CU_TRY(c, cudaGetLastError());
    *n_slabs_out = n_slabs;
    return EWALD_OK;
}

/* ---- octant-form reciprocal kernel: launch shape and launch -------------------------------- */

template <typename T, int DIM, int NPB>
static ewald_status oct_launch_inst(ewald_ctx *c, const OctArgs<T> &A, int grid, int threads, size_t smem,
                                    int *ctas_per_sm /* nullable: query only */)
{
    ewald_status st = allow_smem(c, recip_oct_kernel<T, DIM, NPB>, smem);
    if (st != EWALD_OK) return st;
    if (ctas_per_sm) {
        CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, recip_oct_kernel<T, DIM, NPB>,
                                                                threads, smem));
        return EWALD_OK;
    }
    ProfScope ps(c, 0);
    recip_oct_kernel<T, DIM, NPB><<<grid, threads, smem, c->stream>>>(A);
    return EWALD_OK;
}

template <typename T>
static ewald_status oct_launch_any(ewald_ctx *c, const OctArgs<T> &A, int grid, int threads, size_t smem,
                                   int *ctas_per_sm)
{
    const int dim = c->t.dim, npb = c->t.oct.npb;
#define EWALD_OCT_INST(D, N) if (dim == D && npb == N) return oct_launch_inst<T, D, N>(c, A, grid, threads, smem, ctas_per_sm);
    EWALD_OCT_INST(3, 4) EWALD_OCT_INST(3, 5) EWALD_OCT_INST(3, 6) EWALD_OCT_INST(3, 7)
    EWALD_OCT_INST(2, 4) EWALD_OCT_INST(2, 5) EWALD_OCT_INST(2, 6) EWALD_OCT_INST(2, 7)
#undef EWALD_OCT_INST
    return fail(c, EWALD_ERANGE, "no octant kernel for this block length");
}

template <typename T> static int oct_max_threads(int npb)
{
    (void)npb;
    return OctCfg<T, 7>::MAX_THREADS;
}

/* Shared-memory shape of a CTA of wc walkers: particles per chunk, slab stride, bytes. */
static bool oct_shape(const OctPlan &P, int wc, int /*n_warps*/, int n, size_t es2, int *pc, int *wstride, size_t *smem)
{
    int p = n < 32 ? n : 32;
    for (; p >= 1; p--) {
        const int ws = p * P.rowlen + 1; /* +1 pair: staggers the walkers' slabs over the banks */
        /* two table buffers (the next chunk is built while this one is multiplied), partial sums, walker tags */
        const size_t b = 2 * ((size_t)wc * ws + P.rowlen) * es2 + (size_t)wc * (P.n_items + 1) * sizeof(double);
        if (b <= 200 * 1024) { *pc = p; *wstride = ws; *smem = b; return true; }
    }
    return false;
}

template <typename T>
static ewald_status get_oct_dev(ewald_ctx *c, int wc, OctDev **out)
{
    const int max_warps = oct_max_threads<T>(c->t.oct.npb) / 32;
    const long long key = wc | ((long long)max_warps << 16);
    auto it = c->oct_dev.find(key);
    if (it == c->oct_dev.end()) {
        OctDev d;
        make_oct_launch(c->t.oct, wc, max_warps, &d.L);
        CU_TRY(c, cudaMalloc((void **)&d.d_lane, d.L.lane.size() * sizeof(int)));
        CU_TRY(c, cudaMemcpy(d.d_lane, d.L.lane.data(), d.L.lane.size() * sizeof(int), cudaMemcpyHostToDevice));
        CU_TRY(c, cudaMalloc((void **)&d.d_variant, d.L.variant.size() * sizeof(int)));
        CU_TRY(c, cudaMemcpy(d.d_variant, d.L.variant.data(), d.L.variant.size() * sizeof(int), cudaMemcpyHostToDevice));
        it = c->oct_dev.emplace(key, d).first;
    }
    *out = &it->second;
    return EWALD_OK;
}

template <typename T>
static void oct_fill_args(ewald_ctx *c, OctArgs<T> *A, int W, int n, const T *pos, const T *q,
                          const OctDev &d, int pc, int wstride, double *e_recip)
{
    const OctPlan &P = c->t.oct;
    A->pos = pos; A->q = q; A->n = n; A->npad = ewald_padded_n(n); A->n_walkers = W;
    A->wc = d.L.wc; A->n_slabs = d.L.n_slabs; A->rank_stride = d.L.rank_stride; A->pc = pc; A->rowlen = P.rowlen; A->wstride = wstride;
    for (int k = 0; k < 3; k++) { A->off[k] = P.off[k]; A->nmax[k] = c->t.n_max[k]; }
    A->lane = d.d_lane; A->variant = d.d_variant;
    A->wt = c->d_oct_wt; A->tion = c->t.n_ion ? c->d_oct_tion : nullptr;
    A->e_recip = e_recip;
    for (int i = 0; i < 9; i++) A->binv[i] = c->t.binv[i];
}

/* Picks the walkers-per-CTA that minimises (waves x work per wave) on this device. */
template <typename T>
static ewald_status oct_choose(ewald_ctx *c, int W, int n, int *wc_out)
{
    const long long key = (long long)W | ((long long)n << 24) | ((long long)(sizeof(T) == 4) << 60);
    auto it = c->oct_choice.find(key);
    if (it != c->oct_choice.end()) { *wc_out = it->second; return EWALD_OK; }
    const OctPlan &P = c->t.oct;
    cudaDeviceProp prop;
    CU_TRY(c, cudaGetDeviceProperties(&prop, c->device));
    const int sms = prop.multiProcessorCount;
    double best = 1e300;
    int best_wc = 0;
    for (int wc = 1; wc <= 16 && wc <= W; wc++) {
        OctDev *d;
        ewald_status st = get_oct_dev<T>(c, wc, &d);
        if (st != EWALD_OK) return st;
        int pc, ws; size_t smem;
        if (!oct_shape(P, wc, d->L.n_warps, n, 2 * sizeof(T), &pc, &ws, &smem)) continue;
        OctArgs<T> A;
        int per_sm = 0;
        st = oct_launch_any<T>(c, A, 0, 32 * d->L.n_warps, smem, &per_sm);
        if (st != EWALD_OK) return st;
        if (per_sm < 1) continue;
        const long long ctas = (long long)((W + wc - 1) / wc) * d->L.n_slabs;
        const long long waves = (ctas + (long long)sms * per_sm - 1) / ((long long)sms * per_sm);
        /* work of one CTA per particle: FMA phase + table rows (~90 operations per (walker, axis)) */
        const double cta_work = d->L.cost / d->L.n_slabs + 90.0 * P.dim * wc;
        if (d->L.n_slabs > 1 && wc > 1) break; /* several slabs: one walker per group is enough */
        const double t = (double)waves * per_sm * cta_work;
        if (t < best * (1 - 1e-9)) { best = t; best_wc = wc; }
    }
    if (!best_wc) return fail(c, EWALD_ERANGE, "octant kernel: no launch shape fits");
    c->oct_choice[key] = best_wc;
    *wc_out = best_wc;
    return EWALD_OK;
}

template <typename T>
static ewald_status launch_recip_oct(ewald_ctx *c, int W, int n, const T *pos, const T *q, int *n_slabs_out)
{
    int wc = 0;
    ewald_status st = oct_choose<T>(c, W, n, &wc);
    if (st != EWALD_OK) return st;
    OctDev *d;
    if ((st = get_oct_dev<T>(c, wc, &d)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->partial_recip, (size_t)W * d->L.n_slabs * sizeof(double))) != EWALD_OK) return st;
    int pc, ws; size_t smem;
    if (!oct_shape(c->t.oct, wc, d->L.n_warps, n, 2 * sizeof(T), &pc, &ws, &smem))
        return fail(c, EWALD_ERANGE, "octant kernel: shared memory");
    OctArgs<T> A;
    oct_fill_args<T>(c, &A, W, n, pos, q, *d, pc, ws, (double *)c->partial_recip.p);
    const long long grid = (long long)((W + wc - 1) / wc) * d->L.n_slabs;
    if (grid > 0x7fffffffLL) return fail(c, EWALD_ERANGE, "grid too large");
    st = oct_launch_any<T>(c, A, (int)grid, 32 * d->L.n_warps, smem, nullptr);
    if (st != EWALD_OK) return st;
    CU_TRY(c, cudaGetLastError());
    *n_slabs_out = d->L.n_slabs;
    return EWALD_OK;
}

/* ---- octant kernel on the FP64 tensor cores (ewald_recip_mma.cuh): launch shape and launch ------------ */

static ewald_status get_mma_dev(ewald_ctx *c, int wpw, MmaDev **out)
{
    auto it = c->mma_dev.find(wpw);
    if (it == c->mma_dev.end()) {
        MmaDev d;
        make_mma_launch(c->t.mma, wpw, &d.L);
        if (d.L.valid) {
            CU_TRY(c, cudaMalloc((void **)&d.d_lane, d.L.lane.size() * sizeof(int)));
            CU_TRY(c, cudaMemcpy(d.d_lane, d.L.lane.data(), d.L.lane.size() * sizeof(int), cudaMemcpyHostToDevice));
            CU_TRY(c, cudaMalloc((void **)&d.d_meta, d.L.meta.size() * sizeof(int)));
            CU_TRY(c, cudaMemcpy(d.d_meta, d.L.meta.data(), d.L.meta.size() * sizeof(int), cudaMemcpyHostToDevice));
        }
        it = c->mma_dev.emplace(wpw, d).first;
    }
    *out = &it->second;
    return EWALD_OK;
}

/* true when the tensor-core kernel can take this problem (a plan exists and some split of the warps fits) */
static ewald_status mma_max_walkers(ewald_ctx *c, int *nw_cap)
{
    *nw_cap = 0;
    if (!c->t.mma.valid) return EWALD_OK;
    for (int nw = MMA_WARPS; nw >= 1; nw--) {
        MmaDev *d;
        ewald_status st = get_mma_dev(c, MMA_WARPS / nw, &d);
        if (st != EWALD_OK) return st;
        if (d->L.valid) { *nw_cap = nw; return EWALD_OK; }
    }
    return EWALD_OK;
}

static ewald_status launch_recip_mma(ewald_ctx *c, int W, int n, const double *pos, const double *q, int *n_slabs_out)
{
    const MmaPlan &M = c->t.mma;
    int nw_cap = 0;
    ewald_status st = mma_max_walkers(c, &nw_cap);
    if (st != EWALD_OK) return st;
    if (nw_cap < 1) return fail(c, EWALD_ESTATE, "tensor-core octant kernel: the plan does not fit");
    if ((st = ensure(c, &c->partial_recip, (size_t)W * sizeof(double))) != EWALD_OK) return st;
    /* walkers per CTA so that the grid is one wave; shared memory bounds the walkers of a pass */
    const int pc = 32, qstride = 4 * M.rowlen, wstride = (pc / 4) * qstride; /* 64-particle chunks: -1 to -3 % only, twice the shared memory */
    const size_t slab_bytes = (size_t)wstride * sizeof(double2);
    const size_t part_bytes = (size_t)MMA_WARPS * 2 * M.slots.size() * sizeof(double);
    const size_t avail = c->smem_optin / MMA_CTAS_PER_SM - 2048 - part_bytes;
    int nw_pass = (int)(avail / (2 * slab_bytes));
    if (nw_pass > nw_cap) nw_pass = nw_cap;
    if (nw_pass < 1) return fail(c, EWALD_ERANGE, "tensor-core octant kernel: shared memory");
    const int slots = c->sm_count * MMA_CTAS_PER_SM;
    int wpc = (W + slots - 1) / slots;                      /* walkers per CTA */
    if (wpc > MMA_MAX_PASS * nw_pass) wpc = MMA_MAX_PASS * nw_pass;
    const int n_pass = (wpc + nw_pass - 1) / nw_pass;
    MmaArgs A;
    A.pos = pos; A.q = q; A.n = n; A.npad = ewald_padded_n(n); A.n_walkers = W;
    A.walkers_per_cta = wpc; A.n_pass = n_pass;
    int nw_max = 0, first = 0;
    for (int p = 0; p < n_pass; p++) { /* passes as equal as possible: 7 walkers = 4 + 3 */
        const int nw = (wpc - first + (n_pass - p) - 1) / (n_pass - p);
        MmaDev *d;
        if ((st = get_mma_dev(c, MMA_WARPS / nw, &d)) != EWALD_OK) return st;
        if (!d->L.valid) return fail(c, EWALD_ESTATE, "tensor-core octant kernel: pass shape");
        A.pass[p].first = first; A.pass[p].nw = nw; A.pass[p].wpw = MMA_WARPS / nw;
        A.pass[p].lane = d->d_lane; A.pass[p].meta = d->d_meta;
        first += nw;
        if (nw > nw_max) nw_max = nw;
    }
    A.pc = pc; A.rowlen = M.rowlen; A.qstride = qstride; A.wstride = wstride;
    for (int k = 0; k < 3; k++) { A.off[k] = M.off[k]; A.nmax[k] = c->t.n_max[k]; }
    A.n_slots = (int)M.slots.size();
    A.wt = c->d_mma_wt; A.tion = c->t.n_ion ? c->d_mma_tion : nullptr;
    A.e_recip = (double *)c->partial_recip.p;
    for (int i = 0; i < 9; i++) A.binv[i] = c->t.binv[i];
    const size_t smem = 2 * (size_t)nw_max * slab_bytes + (size_t)nw_max * 2 * M.slots.size() * sizeof(double);
    const int grid = (W + wpc - 1) / wpc;
    if (c->t.dim == 3) {
        if ((st = allow_smem(c, recip_mma_kernel<3>, smem)) != EWALD_OK) return st;
        ProfScope ps(c, 0);
        recip_mma_kernel<3><<<grid, MMA_THREADS, smem, c->stream>>>(A, nw_max);
    } else {
        if ((st = allow_smem(c, recip_mma_kernel<2>, smem)) != EWALD_OK) return st;
        ProfScope ps(c, 0);
        recip_mma_kernel<2><<<grid, MMA_THREADS, smem, c->stream>>>(A, nw_max);
    }
    CU_TRY(c, cudaGetLastError());
    *n_slabs_out = 1;
    return EWALD_OK;
}

/* With the far shell on and every (kappa L_k)^2 >= FAR_T0, a candidate that has a far image on some axis lies in
 * the far shell whatever the other components are: the scan then touches the far stack only for those. */
template <typename T> static void set_outer_far(const ewald_ctx *c, const PairTabs<T> &P, RealGeom<T> *g)
{
    g->outer_far = 0;
    g->far_once = 0;
    if (P.n_far <= 0) return;
    for (int k = 0; k < c->t.dim; k++) {
        const double l = c->t.a[4 * k] * c->t.kappa;
        if (l * l < P.far_t0 * (1 + 1e-9)) return;
    }
    g->outer_far = 1;
    /* ... and if the far stack holds all 20 candidates of a pair plus a round, it is serviced once per pair
     * (call after real_shape has fixed the capacities) */
    g->far_once = !g->multi_far && P.capf_u >= 20 + P.round_items;
}

/* The orthorhombic image scan needs boxes that reach the cut-off within +-2 images and that are wide enough
 * for only the un-shifted image to fall below the pair table (kappa L_k / 2 > sqrt(t_min)). */
static bool real_ortho(const ewald_ctx *c)
{
    if (!c->t.orthogonal || c->t.m_shift > 2) return false;
    for (int k = 0; k < c->t.dim; k++)
        if (c->t.a[4 * k] * c->t.kappa < 0.5) return false;
    return true;
}

template <typename T> static void fill_species(const ewald_ctx *c, PairTabs<T> *P)
{
    P->ion_uniform = c->t.ion_uniform ? 1 : 0;
    P->n_species = c->t.ion_uniform ? (int)c->t.sp_start.size() - 1 : 0;
    for (int s = 0; s < 5; s++)
        P->sp_start[s] = s < (int)c->t.sp_start.size() && c->t.ion_uniform ? c->t.sp_start[s] : c->t.n_ion;
}

/* Fills the table part of PairTabs and returns the bytes of shared memory the tables take. */
template <typename T> static void fill_pair_tabs(const ewald_ctx *c, const double *qinfo, PairTabs<T> *P);
template <> void fill_pair_tabs<float>(const ewald_ctx *c, const double *qinfo, PairTabs<float> *P)
{
    const PairTable &pt = c->t.pair32;
    P->pair_tab = c->d_pairf; P->n_bins = pt.n_bins; P->t_safe = (float)pt.t_min;
    P->far_tab = nullptr; P->n_far = 0; P->key_far = 0x7fffffff; P->far_t0 = 0;
    P->qinfo = qinfo;
    fill_species(c, P);
    P->capf_u = P->capf_g = 0;
}
template <> void fill_pair_tabs<double>(const ewald_ctx *c, const double *qinfo, PairTabs<double> *P)
{
    const PairTable &pt = c->t.pair64;
    bool far = c->real_variant == 0 && c->t.n_far > 0;
    P->pair_tab = c->d_pair; P->t_safe = pt.t_min;
    /* the far table starts at FAR_T0; a kernel may start its far shell later (P->far_t0 set by the caller: the
     * move kernel keeps 16, where the longer table would cost its stacks a slot) */
    if (P->far_t0 < FAR_T0) P->far_t0 = FAR_T0;
    if (P->far_t0 > 16) P->far_t0 = 16;
    const int skip = (P->far_t0 - FAR_T0) << FAR_KB;
    if (c->t.n_far - skip <= 0) far = false;
    /* with the far shell on, the near table is needed below far_t0 only: the bins that start below it */
    int e_far;
    const double m_far = std::frexp((double)P->far_t0, &e_far); /* far_t0 = m 2^e, m in [1/2, 1) */
    const int near_bins = ((e_far - 1 - pt.e_min) << pt.kbits) + (int)std::ceil((2 * m_far - 1) * (1 << pt.kbits));
    P->n_bins = far && near_bins < pt.n_bins ? near_bins : pt.n_bins;
    P->far_tab = far ? c->d_far + (size_t)skip * FAR_REP * 4 : nullptr; P->n_far = far ? c->t.n_far - skip : 0;
    P->key_far = far ? host_key((double)P->far_t0) : 0x7fffffff;
    P->qinfo = qinfo;
    fill_species(c, P);
    P->capf_u = P->capf_g = 0;
}

/* CTA size and per-lane stack capacities that fit the shared memory left after `fixed` bytes of tables.
 * The two item kinds of a stack (bare t / (t, qq)) share the same bytes, so the (t, qq) capacity is half.
 * min_cap = ScanShape::min_cap(P->round_items) of the kernel variant. */
template <typename T>
static bool real_shape(const ewald_ctx *c, size_t fixed, int min_cap_u, int min_cap_g, int max_threads,
                       PairTabs<T> *P, int *threads, size_t *smem, bool allow_two = true)
{
    const size_t full = c->smem_optin > 2048 ? c->smem_optin - 2048 : 0; /* static arrays of the kernels */
    /* first choice: two CTAs of max_threads per SM (228 KB per SM, 1 KB reserved per CTA), if the tables are
     * small enough for that (the FP32 kernels); then one CTA, with fewer threads if need be */
    const size_t half = (228 * 1024 - 2 * 1024) / 2 - 2048;
    const bool far = P->n_far > 0;
    for (int pass = allow_two && 2 * max_threads <= 2048 ? 0 : 1; pass < 2; pass++) {
        const size_t budget = pass == 0 ? (half < full ? half : full) : full;
        for (int th = max_threads; th >= 32; th /= 2) {
            if (fixed >= budget) break;
            /* bytes per lane for the stacks of the CTA's th / 32 warps */
            const long long lane_bytes = (long long)((budget - fixed) / ((size_t)(th / 32) * 32));
            const long long want = 2 * (min_cap_u > min_cap_g ? min_cap_u : min_cap_g) + 8;
            const long long need = min_cap_u > 2 * min_cap_g ? min_cap_u : 2 * min_cap_g;
            long long cu = 0, cf = 0;
            if (!far) {
                cu = lane_bytes / (long long)sizeof(T);
                if (cu > want) cu = want;
                cu &= ~1LL;
            } else {
                /* the far stack receives twice the terms: first choice twice the near capacity (the same bytes);
                 * if that does not fit, the near stack at its minimum and the rest to the far stack, which at
                 * 20 + round_items items is serviced once per pair (set_outer_far); else equal capacities */
                cu = lane_bytes / (long long)(sizeof(T) + 8);
                if (cu > want) cu = want;
                cu &= ~1LL;
                cf = 2 * cu;
                if (cu < need) {
                    cu = need + (need & 1);
                    cf = ((lane_bytes - cu * (long long)sizeof(T)) / 4) & ~1LL;
                    if (cf > 2 * cu) cf = 2 * cu;
                    if (cf < 20 + P->round_items) {
                        cu = (lane_bytes / (long long)(sizeof(T) + 4)) & ~1LL;
                        if (cu > want) cu = want;
                        cf = cu;
                    }
                }
            }
            if (cu >= need && (!far || cf >= need)) {
                *threads = th;
                P->cap_u = (int)cu; P->cap_g = (int)(cu / 2);
                P->capf_u = far ? (int)cf : 0; P->capf_g = far ? (int)(cf / 2) : 0;
                *smem = fixed + (size_t)(th / 32) * 32 * ((size_t)cu * sizeof(T) + (far ? (size_t)cf * 4 : 0));
                return true;
            }
            if (pass == 0) break; /* two CTAs per SM only at full size */
        }
    }
    return false;
}

template <int DIM, bool ORTHO, int M> static int scan_min_cap(bool uq, int r)
{
    return uq ? ScanShape<DIM, ORTHO, M, true>::min_cap(r) : ScanShape<DIM, ORTHO, M, false>::min_cap(r);
}
static int real_min_cap(const ewald_ctx *c, bool ortho, bool uq, int r)
{
    const int m = c->t.m_shift;
    if (c->t.dim == 3) return !ortho ? scan_min_cap<3, false, 0>(uq, r) : m == 0 ? scan_min_cap<3, true, 0>(uq, r)
                            : m == 1 ? scan_min_cap<3, true, 1>(uq, r) : scan_min_cap<3, true, 2>(uq, r);
    return !ortho ? scan_min_cap<2, false, 0>(uq, r) : m == 0 ? scan_min_cap<2, true, 0>(uq, r)
         : m == 1 ? scan_min_cap<2, true, 1>(uq, r) : scan_min_cap<2, true, 2>(uq, r);
}

template <typename T>
static ewald_status launch_real(ewald_ctx *c, int W, int n, const T *pos, const T *q, int n_slabs, double *energies,
                                double *components)
{
    RealArgs<T> A;
    A.pos = pos; A.q = q; A.n = n; A.npad = ewald_padded_n(n);
    A.img = Tabs<T>::img(c); A.nimg = c->nimg;
    A.ion_pos = Tabs<T>::ion_pos(c); A.ion_q = Tabs<T>::ion_q(c); A.n_ion = c->t.n_ion;
    A.P.far_t0 = FAR_T0;
    A.P.round_items = RoundSize<T, false>::R;
    fill_pair_tabs<T>(c, nullptr, &A.P); /* the kernel finds the all-equal flag of the charges itself */
    fill_geom(c->t, &A.g);
    const bool ortho = real_ortho(c);
    if (ortho) A.nimg = 0; /* the orthorhombic path does not read the image list */
    const size_t fixed = RealSmem<T>::fixed_bytes(A.P.n_bins, A.P.n_far, A.nimg, A.n_ion, (size_t)c->t.dim * ewald_padded_n(n) + n);
    int threads = 0; size_t smem = 0;
    if (!real_shape<T>(c, fixed, real_min_cap(c, ortho, true, A.P.round_items), real_min_cap(c, ortho, false, A.P.round_items), REAL_MAX_THREADS, &A.P,
                       &threads, &smem))
        return fail(c, EWALD_ERANGE, "real-space kernel: problem too large for shared memory");
    set_outer_far(c, A.P, &A.g);

    const long long H = (n - 1) / 2;
    const long long total = (long long)n * H + ((n & 1) ? 0 : n / 2) + (long long)n * c->t.n_ion;
    long long n_tiles = (4LL * c->sm_count + W - 1) / W;
    long long max_tiles = (total + threads - 1) / threads;
    /* Small batches of small boxes (|m| <= 2 in 3D, 125 candidates per pair; config 1): with one pair per thread the
     * grid is a fraction of the GPU (8 walkers x 3 tiles), so the five z-images of a pair go to five lanes
     * (ScanShape::ZSPLIT): five times the items, each a fifth of the work plus the pair's set-up again -- only when
     * the pairs alone cannot fill the SMs */
    A.zsplit = ortho && c->t.dim == 3 && c->t.m_shift == 2 && (long long)W * max_tiles < c->sm_count ? 1 : 0;
    if (A.zsplit) max_tiles = (5 * total + threads - 1) / threads;
    if (n_tiles > max_tiles) n_tiles = max_tiles;
    if (n_tiles < 1) n_tiles = 1;
    ewald_status st = ensure(c, &c->partial_real, (size_t)W * n_tiles * sizeof(double));
    if (st != EWALD_OK) return st;
    A.partial = (double *)c->partial_real.p;
    A.n_tiles = (int)n_tiles;
    /* [S6] folded into the kernel: per-walker arrival counters (zero between calls: the last CTA resets its own) */
    if ((size_t)W * sizeof(int) > c->done.cap) {
        if ((st = ensure(c, &c->done, (size_t)W * sizeof(int))) != EWALD_OK) return st;
        CU_TRY(c, cudaMemsetAsync(c->done.p, 0, c->done.cap, c->stream));
    }
    A.done = (int *)c->done.p;
    A.comb.recip_partial = (const double *)c->partial_recip.p; A.comb.n_recip = n_slabs;
    A.comb.real_partial = A.partial; A.comb.n_real = (int)n_tiles;
    A.comb.ion_q2 = c->t.ion_q2; A.comb.ion_qsum = c->t.ion_qsum; A.comb.ion_real = c->t.ion_real;
    A.comb.xi_r = c->t.xi_r; A.comb.self_coef = c->t.self_coef; A.comb.bg_coef = c->t.bg_coef;
    A.comb.energies = energies; A.comb.components = components; A.comb.n_walkers = W;
    const long long grid = (long long)W * n_tiles;
    /* small batches (at most two waves of CTAs): [S6] inside the kernel, one launch less; large ones: combine_kernel */
    const bool fold = grid <= 2LL * c->sm_count;
    const CombineArgs comb = A.comb;
    if (!fold) A.comb.energies = nullptr;
    if (grid > 0x7fffffffLL) return fail(c, EWALD_ERANGE, "grid too large");
    {
        const int sh[8] = {threads, (int)smem, A.P.cap_u, A.P.capf_u, A.P.n_bins, A.P.n_far, (int)grid, A.g.far_once};
        std::memcpy(c->shape[0], sh, sizeof sh);
    }
#define EWALD_LAUNCH_REAL(DIM, ORTHO, M)                                                          \
    do {                                                                                          \
        st = allow_smem(c, real_kernel<T, DIM, ORTHO, M>, smem);                                  \
        if (st != EWALD_OK) return st;                                                            \
        ProfScope ps(c, 1);                                                                       \
        real_kernel<T, DIM, ORTHO, M><<<(unsigned)grid, threads, smem, c->stream>>>(A);           \
    } while (0)
    const int m = c->t.m_shift;
    if (c->t.dim == 3) {
        if (!ortho) EWALD_LAUNCH_REAL(3, false, 0);
        else if (m == 0) EWALD_LAUNCH_REAL(3, true, 0);
        else if (m == 1) EWALD_LAUNCH_REAL(3, true, 1);
        else EWALD_LAUNCH_REAL(3, true, 2);
    } else {
        if (!ortho) EWALD_LAUNCH_REAL(2, false, 0);
        else if (m == 0) EWALD_LAUNCH_REAL(2, true, 0);
        else if (m == 1) EWALD_LAUNCH_REAL(2, true, 1);
        else EWALD_LAUNCH_REAL(2, true, 2);
    }
#undef EWALD_LAUNCH_REAL
    CU_TRY(c, cudaGetLastError());
    if (!fold) {
        ProfScope ps(c, 2);
        combine_kernel<T><<<(W + 127) / 128, 128, 0, c->stream>>>(comb, q, n);
        CU_TRY(c, cudaGetLastError());
    }
    return EWALD_OK;
}

/* FP64: the tensor-core form of the octant kernel (variant 0 or 3) when its plan fits; FP32 and variant 2: the
 * FMA-pipe form; variant 1 or no octant plan: the complex half-set kernel. */
template <typename T>
static ewald_status launch_recip_any(ewald_ctx *c, bool oct, int W, int n, const T *pos, const T *q, int *n_slabs);
template <>
ewald_status launch_recip_any<double>(ewald_ctx *c, bool oct, int W, int n, const double *pos, const double *q, int *n_slabs)
{
    if (!oct) return launch_recip<double>(c, W, n, pos, q, nullptr, n_slabs);
    if (c->recip_variant != 2) {
        int nw_cap = 0;
        ewald_status st = mma_max_walkers(c, &nw_cap);
        if (st != EWALD_OK) return st;
        if (nw_cap >= 1) return launch_recip_mma(c, W, n, pos, q, n_slabs);
        if (c->recip_variant == 3) return fail(c, EWALD_ESTATE, "tensor-core octant kernel: the plan does not fit");
    }
    return launch_recip_oct<double>(c, W, n, pos, q, n_slabs);
}
template <>
ewald_status launch_recip_any<float>(ewald_ctx *c, bool oct, int W, int n, const float *pos, const float *q, int *n_slabs)
{
    if (!oct) return launch_recip<float>(c, W, n, pos, q, nullptr, n_slabs);
    return launch_recip_oct<float>(c, W, n, pos, q, n_slabs);
}

template <typename T>
static ewald_status energy_batch_t(ewald_ctx *c, int W, int n, const T *pos, const T *q,
                                   double *energies, double *components)
{
    /* two launches: [S1-S4] reciprocal, then [S5] real space with [S6] folded into the last CTA of every walker */
    int n_slabs = 0;
    const bool oct = c->recip_variant != 1 && c->t.oct.valid;
    if (c->recip_variant >= 2 && !oct) return fail(c, EWALD_ESTATE, "octant kernel: no plan for this G set");
    ewald_status st = launch_recip_any<T>(c, oct, W, n, pos, q, &n_slabs);
    if (st != EWALD_OK) return st;
    return launch_real<T>(c, W, n, pos, q, n_slabs, energies, components);
}

static ewald_status check_batch(ewald_ctx *c, int W, int n, ewald_prec prec, const void *pos, const void *q)
{
    if (!c) return EWALD_EINVAL;
    if (W < 0 || n <= 0) return fail(c, EWALD_EINVAL, "n_walkers < 0 or n_particles <= 0");
    if (prec != EWALD_F64 && prec != EWALD_F32) return fail(c, EWALD_EINVAL, "bad precision");
    if (W > 0 && (!pos || !q)) return fail(c, EWALD_EINVAL, "null positions or charges");
    return EWALD_OK;
}

extern "C" ewald_status ewald_energy_batch(ewald_ctx *c, int W, int n, ewald_prec prec, const void *pos,
                                           const void *q, double *energies, double *components)
{
    ewald_status st = check_batch(c, W, n, prec, pos, q);
    if (st != EWALD_OK) return st;
    if (W == 0) return EWALD_OK;
    if (!energies) return fail(c, EWALD_EINVAL, "null energies");
    EWALD_DEVICE(c);
    if (prec == EWALD_F64)
        return energy_batch_t<double>(c, W, n, (const double *)pos, (const double *)q, energies, components);
    return energy_batch_t<float>(c, W, n, (const float *)pos, (const float *)q, energies, components);
}

extern "C" ewald_status ewald_energy_batch_host(ewald_ctx *c, int W, int n, ewald_prec prec,
                                                const void *pos, const void *q, double *energies,
                                                double *components)
{
    ewald_status st = check_batch(c, W, n, prec, pos, q);
    if (st != EWALD_OK) return st;
    if (W == 0) return EWALD_OK;
    if (!energies) return fail(c, EWALD_EINVAL, "null energies");
    EWALD_DEVICE(c);
    const size_t es = prec == EWALD_F64 ? 8 : 4;
    const size_t pbytes = (size_t)W * c->t.dim * ewald_padded_n(n) * es, qbytes = (size_t)n * es;
    if ((st = ensure(c, &c->stage_pos, pbytes)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->stage_q, qbytes)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->stage_e, (size_t)W * 8)) != EWALD_OK) return st;
    if (components && (st = ensure(c, &c->stage_comp, (size_t)W * 32)) != EWALD_OK) return st;
    CU_TRY(c, cudaMemcpyAsync(c->stage_pos.p, pos, pbytes, cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->stage_q.p, q, qbytes, cudaMemcpyHostToDevice, c->stream));
    st = ewald_energy_batch(c, W, n, prec, c->stage_pos.p, c->stage_q.p, (double *)c->stage_e.p,
                            components ? (double *)c->stage_comp.p : nullptr);
    if (st != EWALD_OK) return st;
    CU_TRY(c, cudaMemcpyAsync(energies, c->stage_e.p, (size_t)W * 8, cudaMemcpyDeviceToHost, c->stream));
    if (components)
        CU_TRY(c, cudaMemcpyAsync(components, c->stage_comp.p, (size_t)W * 32, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return EWALD_OK;
}

extern "C" ewald_status ewald_load_walkers(ewald_ctx *c, int W, int n, ewald_prec prec, const void *pos,
                                           const void *q)
{
    ewald_status st = check_batch(c, W, n, prec, pos, q);
    if (st != EWALD_OK) return st;
    if (W == 0) return fail(c, EWALD_EINVAL, "n_walkers must be > 0");
    EWALD_DEVICE(c);
    const size_t es = prec == EWALD_F64 ? 8 : 4;
    const int npad = ewald_padded_n(n);
    const size_t pbytes = (size_t)W * c->t.dim * npad * es;
    c->loaded = false;
    if ((st = ensure(c, &c->st_pos, pbytes)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->st_q, (size_t)n * es)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->st_rho, (size_t)W * 2 * c->ngp_pad * es)) != EWALD_OK) return st;
    CU_TRY(c, cudaMemcpyAsync(c->st_pos.p, pos, pbytes, cudaMemcpyDeviceToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->st_q.p, q, (size_t)n * es, cudaMemcpyDeviceToDevice, c->stream));
    CU_TRY(c, cudaMemsetAsync(c->st_rho.p, 0, (size_t)W * 2 * c->ngp_pad * es, c->stream));
    int n_slabs = 0;
    if (prec == EWALD_F64)
        st = launch_recip<double>(c, W, n, (const double *)c->st_pos.p, (const double *)c->st_q.p,
                                  (double *)c->st_rho.p, &n_slabs);
    else
        st = launch_recip<float>(c, W, n, (const float *)c->st_pos.p, (const float *)c->st_q.p,
                                 (float *)c->st_rho.p, &n_slabs);
    if (st != EWALD_OK) return st;
    {
        ProfScope ps(c, 2);
        if (prec == EWALD_F64) charge_sums_kernel<double><<<1, 256, 0, c->stream>>>((const double *)c->st_q.p, n, (double *)c->st_qinfo.p);
        else charge_sums_kernel<float><<<1, 256, 0, c->stream>>>((const float *)c->st_q.p, n, (double *)c->st_qinfo.p);
    }
    CU_TRY(c, cudaGetLastError());
    c->st_walkers = W; c->st_n = n; c->st_npad = npad; c->st_prec = prec;
    c->loaded = true;
    return EWALD_OK;
}

template <typename T>
static ewald_status move_batch_t(ewald_ctx *c, int n_moves, const int *walker, const int *electron,
                                 const T *new_r, int commit, double *delta_e)
{
    typedef typename Num<T>::T2 T2;
    MoveArgs<T> A;
    A.pos = (T *)c->st_pos.p; A.q = (const T *)c->st_q.p; A.rho = (T *)c->st_rho.p;
    A.n = c->st_n; A.npad = c->st_npad; A.n_walkers = c->st_walkers;
    A.gn = c->d_gn; A.w2 = Tabs<T>::w2(c); A.ngp = c->ngp; A.ngp_pad = c->ngp_pad;
    for (int k = 0; k < 3; k++) { A.nmax[k] = c->t.n_max[k]; A.off[k] = c->off[k]; }
    A.rowlen = c->rowlen;
    A.img = Tabs<T>::img(c); A.nimg = c->nimg;
    A.ion_pos = Tabs<T>::ion_pos(c); A.ion_q = Tabs<T>::ion_q(c); A.n_ion = c->t.n_ion;
    A.P.round_items = RoundSize<T, true>::R;
    A.P.far_t0 = 16; /* the move kernel's far shell starts later than the energy kernels' */
    fill_pair_tabs<T>(c, (const double *)c->st_qinfo.p, &A.P);
    A.n_moves = n_moves;
    A.walker = walker; A.electron = electron; A.new_r = new_r; A.commit = commit; A.delta_e = delta_e;
    for (int i = 0; i < 9; i++) A.binv[i] = c->t.binv[i];
    fill_geom(c->t, &A.g);
    const bool ortho = real_ortho(c);
    if (ortho) A.nimg = 0;
    /* one warp per move; the CTA size follows from the shared memory the stacks need */
    int threads = 0; size_t smem = 0;
    bool fits = false;
    for (int th = MOVE_MAX_THREADS; th >= 32 && !fits; th /= 2) {
        const size_t fixed = RealSmem<T>::fixed_bytes(A.P.n_bins, A.P.n_far, A.nimg, A.n_ion,
                                                      4 * (size_t)c->rowlen * (th / 32));
        fits = real_shape<T>(c, fixed, real_min_cap(c, ortho, true, A.P.round_items), real_min_cap(c, ortho, false, A.P.round_items), th, &A.P, &threads,
                             &smem) && threads == th;
    }
    if (!fits) return fail(c, EWALD_ERANGE, "move kernel: tables too large for shared memory");
    set_outer_far(c, A.P, &A.g);
    const int warps = threads / 32;
    const int want_grid = (n_moves + warps - 1) / warps;
    ewald_status st;
    /* persistent CTAs (the tables are staged once per CTA): as many as the SMs hold at once */
#define EWALD_LAUNCH_MOVE(DIM, ORTHO, M)                                                          \
    do {                                                                                          \
        if ((st = allow_smem(c, move_kernel<T, DIM, ORTHO, M>, smem)) != EWALD_OK) return st;     \
        int per_sm = 1;                                                                           \
        CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, move_kernel<T, DIM, ORTHO, M>, threads, \
                                                                smem));                           \
        if (per_sm < 1) per_sm = 1;                                                               \
        const int grid = want_grid < c->sm_count * per_sm ? want_grid : c->sm_count * per_sm;     \
        const int sh[8] = {threads, (int)smem, A.P.cap_u, A.P.capf_u, A.P.n_bins, A.P.n_far, grid, A.g.far_once}; \
        std::memcpy(c->shape[1], sh, sizeof sh);                                                  \
        ProfScope ps(c, 3);                                                                       \
        move_kernel<T, DIM, ORTHO, M><<<grid, threads, smem, c->stream>>>(A);                     \
    } while (0)
    const int m = c->t.m_shift;
    if (c->t.dim == 3) {
        if (!ortho) EWALD_LAUNCH_MOVE(3, false, 0);
        else if (m == 0) EWALD_LAUNCH_MOVE(3, true, 0);
        else if (m == 1) EWALD_LAUNCH_MOVE(3, true, 1);
        else EWALD_LAUNCH_MOVE(3, true, 2);
    } else {
        if (!ortho) EWALD_LAUNCH_MOVE(2, false, 0);
        else if (m == 0) EWALD_LAUNCH_MOVE(2, true, 0);
        else if (m == 1) EWALD_LAUNCH_MOVE(2, true, 1);
        else EWALD_LAUNCH_MOVE(2, true, 2);
    }
#undef EWALD_LAUNCH_MOVE
    CU_TRY(c, cudaGetLastError());
    return EWALD_OK;
}

extern "C" ewald_status ewald_move_delta_batch(ewald_ctx *c, int n_moves, const int *walker,
                                               const int *electron, const void *new_r, int commit,
                                               double *delta_e)
{
    if (!c) return EWALD_EINVAL;
    if (!c->loaded) return fail(c, EWALD_ESTATE, "no walkers loaded (call ewald_load_walkers first)");
    if (n_moves < 0) return fail(c, EWALD_EINVAL, "n_moves < 0");
    if (n_moves == 0) return EWALD_OK;
    if (!walker || !electron || !new_r || !delta_e) return fail(c, EWALD_EINVAL, "null move argument");
    EWALD_DEVICE(c);
    if (c->st_prec == EWALD_F64)
        return move_batch_t<double>(c, n_moves, walker, electron, (const double *)new_r, commit, delta_e);
    return move_batch_t<float>(c, n_moves, walker, electron, (const float *)new_r, commit, delta_e);
}

extern "C" ewald_status ewald_move_delta_batch_host(ewald_ctx *c, int n_moves, const int *walker,
                                                    const int *electron, const void *new_r, int commit,
                                                    double *delta_e)
{
    if (!c) return EWALD_EINVAL;
    if (!c->loaded) return fail(c, EWALD_ESTATE, "no walkers loaded (call ewald_load_walkers first)");
    if (n_moves < 0) return fail(c, EWALD_EINVAL, "n_moves < 0");
    if (n_moves == 0) return EWALD_OK;
    if (!walker || !electron || !new_r || !delta_e) return fail(c, EWALD_EINVAL, "null move argument");
    EWALD_DEVICE(c);
    const size_t es = c->st_prec == EWALD_F64 ? 8 : 4;
    const size_t rbytes = (size_t)n_moves * c->t.dim * es;
    ewald_status st;
    if ((st = ensure(c, &c->mv_walker, (size_t)n_moves * 4)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->mv_electron, (size_t)n_moves * 4)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->mv_newr, rbytes)) != EWALD_OK) return st;
    if ((st = ensure(c, &c->mv_de, (size_t)n_moves * 8)) != EWALD_OK) return st;
    CU_TRY(c, cudaMemcpyAsync(c->mv_walker.p, walker, (size_t)n_moves * 4, cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->mv_electron.p, electron, (size_t)n_moves * 4, cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->mv_newr.p, new_r, rbytes, cudaMemcpyHostToDevice, c->stream));
    st = ewald_move_delta_batch(c, n_moves, (const int *)c->mv_walker.p, (const int *)c->mv_electron.p,
                                c->mv_newr.p, commit, (double *)c->mv_de.p);
    if (st != EWALD_OK) return st;
    CU_TRY(c, cudaMemcpyAsync(delta_e, c->mv_de.p, (size_t)n_moves * 8, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return EWALD_OK;
}

extern "C" ewald_status ewald_move_delta(ewald_ctx *c, int walker, int electron, const double *new_r,
                                         int commit, double *delta_e)
{
    if (!c) return EWALD_EINVAL;
    if (!c->loaded) return fail(c, EWALD_ESTATE, "no walkers loaded (call ewald_load_walkers first)");
    if (!new_r || !delta_e) return fail(c, EWALD_EINVAL, "null move argument");
    if (walker < 0 || walker >= c->st_walkers) return fail(c, EWALD_ESTATE, "walker index out of range");
    if (electron < 0 || electron >= c->st_n) return fail(c, EWALD_ESTATE, "electron index out of range");
    float rf[3];
    for (int x = 0; x < c->t.dim; x++) rf[x] = (float)new_r[x];
    const void *r = c->st_prec == EWALD_F64 ? (const void *)new_r : (const void *)rf;
    return ewald_move_delta_batch_host(c, 1, &walker, &electron, r, commit, delta_e);
}

/* ---- per-kernel timers -------------------------------------------------------------------- */

extern "C" ewald_status ewald_launch_shape(const ewald_ctx *c, int which, int *out)
{
    if (!c || !out || which < 0 || which > 1) return EWALD_EINVAL;
    std::memcpy(out, c->shape[which], sizeof c->shape[which]);
    return EWALD_OK;
}

extern "C" ewald_status ewald_profile_enable(ewald_ctx *c, int on)
{
    if (!c) return EWALD_EINVAL;
    c->prof = on != 0;
    return EWALD_OK;
}

extern "C" ewald_status ewald_profile_read(ewald_ctx *c, double *ms, int *launches)
{
    if (!c || !ms || !launches) return EWALD_EINVAL;
    EWALD_DEVICE(c);
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < 4; k++) { ms[k] = 0; launches[k] = 0; }
    for (ProfRec &r : c->recs) {
        float t = 0;
        if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess && r.kind >= 0 && r.kind < 4) {
            ms[r.kind] += t;
            launches[r.kind]++;
        }
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    c->recs.clear();
    return EWALD_OK;
}

extern "C" long long ewald_launch_count(const ewald_ctx *c) { return c ? c->launches : -1; }

/* ---- introspection ------------------------------------------------------------------------ */

extern "C" int ewald_num_g(const ewald_ctx *c) { return c ? 2 * c->ngp : -1; }
extern "C" int ewald_num_images(const ewald_ctx *c) { return c ? c->nimg : -1; }
extern "C" double ewald_r_cutoff(const ewald_ctx *c) { return c ? c->t.r_cutoff : NAN; }

extern "C" ewald_status ewald_get_g(const ewald_ctx *c, int *n_out)
{
    if (!c || !n_out) return EWALD_EINVAL;
    memcpy(n_out, c->t.g_n.data(), c->t.g_n.size() * sizeof(int));
    return EWALD_OK;
}

extern "C" ewald_status ewald_get_constants(const ewald_ctx *c, double *xi_r, double *v_m, double *e_fixed)
{
    if (!c) return EWALD_EINVAL;
    if (xi_r) *xi_r = c->t.xi_r;
    if (v_m) *v_m = c->t.v_m;
    if (e_fixed) {
        /* Eq. 2 restricted to the fixed charges: recip + real + self + background */
        long double er = 0;
        for (int g = 0; g < c->ngp && c->t.n_ion; g++)
            er += (long double)c->t.g_w2[g] * ((long double)c->t.ion_rho[2 * g] * c->t.ion_rho[2 * g] +
                                               (long double)c->t.ion_rho[2 * g + 1] * c->t.ion_rho[2 * g + 1]);
        *e_fixed = (double)(er + c->t.ion_real + 0.5L * c->t.ion_q2 * c->t.xi_r -
                            (long double)c->t.self_coef * c->t.ion_q2 -
                            0.5L * c->t.bg_coef * c->t.ion_qsum * c->t.ion_qsum);
    }
    return EWALD_OK;
}

extern "C" ewald_status ewald_get_rho(ewald_ctx *c, int walker, double *re_im)
{
    if (!c || !re_im) return EWALD_EINVAL;
    if (!c->loaded) return fail(c, EWALD_ESTATE, "no walkers loaded");
    if (walker < 0 || walker >= c->st_walkers) return fail(c, EWALD_ESTATE, "walker index out of range");
    EWALD_DEVICE(c);
    const size_t es = c->st_prec == EWALD_F64 ? 8 : 4;
    std::vector<unsigned char> h((size_t)2 * c->ngp_pad * es);
    CU_TRY(c, cudaMemcpyAsync(h.data(), (const char *)c->st_rho.p + (size_t)walker * h.size(), h.size(),
                              cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    for (int g = 0; g < c->ngp; g++) {
        if (es == 8) {
            const double *d = (const double *)h.data();
            re_im[2 * g] = d[g]; re_im[2 * g + 1] = d[c->ngp_pad + g];
        } else {
            const float *f = (const float *)h.data();
            re_im[2 * g] = f[g]; re_im[2 * g + 1] = f[c->ngp_pad + g];
        }
    }
    return EWALD_OK;
}

extern "C" ewald_status ewald_get_positions(ewald_ctx *c, int walker, double *pos)
{
    if (!c || !pos) return EWALD_EINVAL;
    if (!c->loaded) return fail(c, EWALD_ESTATE, "no walkers loaded");
    if (walker < 0 || walker >= c->st_walkers) return fail(c, EWALD_ESTATE, "walker index out of range");
    EWALD_DEVICE(c);
    const size_t es = c->st_prec == EWALD_F64 ? 8 : 4;
    const int dim = c->t.dim, npad = c->st_npad, n = c->st_n;
    std::vector<unsigned char> h((size_t)dim * npad * es);
    CU_TRY(c, cudaMemcpyAsync(h.data(), (const char *)c->st_pos.p + (size_t)walker * h.size(), h.size(),
                              cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < n; i++)
        for (int x = 0; x < dim; x++)
            pos[(size_t)i * dim + x] = es == 8 ? ((const double *)h.data())[x * npad + i]
                                               : (double)((const float *)h.data())[x * npad + i];
    return EWALD_OK;
}

extern "C" ewald_status ewald_probe_dmma(ewald_ctx *c, int iters, double *flops)
{
    if (!c || !flops || iters <= 0) return EWALD_EINVAL;
    EWALD_DEVICE(c);
    ewald_status st = ensure(c, &c->stage_e, 64);
    if (st != EWALD_OK) return st;
    CU_TRY(c, cudaMemsetAsync(c->stage_e.p, 0, 64, c->stream));
    const int blocks = c->sm_count, threads = 256;
    cudaEvent_t e0, e1;
    CU_TRY(c, cudaEventCreate(&e0));
    CU_TRY(c, cudaEventCreate(&e1));
    for (int rep = 0; rep < 2; rep++) { /* first pass warms up */
        CU_TRY(c, cudaEventRecord(e0, c->stream));
        dmma_probe_kernel<<<blocks, threads, 0, c->stream>>>(iters, (const double *)c->stage_e.p, (double *)c->stage_e.p);
        CU_TRY(c, cudaEventRecord(e1, c->stream));
        CU_TRY(c, cudaEventSynchronize(e1));
    }
    float ms = 0;
    CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *flops = 2.0 * 256.0 * 32.0 * iters * (double)blocks * (threads / 32) / (ms * 1e-3);
    return EWALD_OK;
}

extern "C" ewald_status ewald_probe_fma(ewald_ctx *c, ewald_prec prec, int iters, double *flops)
{
    if (!c || !flops || iters <= 0) return EWALD_EINVAL;
    EWALD_DEVICE(c);
    cudaDeviceProp prop;
    CU_TRY(c, cudaGetDeviceProperties(&prop, c->device));
    ewald_status st = ensure(c, &c->stage_e, 64);
    if (st != EWALD_OK) return st;
    const int blocks = prop.multiProcessorCount * 8, threads = 256;
    cudaEvent_t e0, e1;
    CU_TRY(c, cudaEventCreate(&e0));
    CU_TRY(c, cudaEventCreate(&e1));
    for (int rep = 0; rep < 2; rep++) { /* first pass warms up */
        CU_TRY(c, cudaEventRecord(e0, c->stream));
        if (prec == EWALD_F64)
            fma_probe_kernel<double><<<blocks, threads, 0, c->stream>>>(iters, 1.0000001, 1e-9, (double *)c->stage_e.p);
        else
            fma_probe_kernel<float><<<blocks, threads, 0, c->stream>>>(iters, 1.0001f, 1e-6f, (float *)c->stage_e.p);
        CU_TRY(c, cudaEventRecord(e1, c->stream));
        CU_TRY(c, cudaEventSynchronize(e1));
    }
    float ms = 0;
    CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *flops = 2.0 * 64.0 * iters * (double)blocks * threads / (ms * 1e-3);
    return EWALD_OK;
}

/* ---- allocation-free entry point ------------------------------------------------------------------------
 * ewald_recip_energy_static: E_recip per walker (S1-S4, the reciprocal sum of Eq. 3) by the
 * complex half-set kernel recip_kernel -- the kernel whose per-(walker, slab) partial sums are its scratch --
 * with that scratch in g_static_scratch instead of the context's growing buffer.  No cudaMalloc, no cudaFree, no
 * event creation, no synchronisation: two kernel launches on the context's stream. */

/* out[w] = sum over the slabs, in slab order (the order combine_kernel uses). */
__global__ void static_slab_sum_kernel(const double *partial, int n_slabs, int n_walkers, double *out)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_walkers) return;
    double e = 0;
    for (int k = 0; k < n_slabs; k++) e += partial[(size_t)w * n_slabs + k];
    out[w] = e;
}

template <typename T>
static ewald_status recip_energy_static_t(ewald_ctx *c, int W, int n, const T *pos, const T *q, int n_slabs,
                                          double *e_recip)
{
    typedef typename Num<T>::T2 T2;
    RecipArgs<T> A;
    A.pos = pos; A.q = q; A.n = n; A.npad = ewald_padded_n(n);
    A.gn = c->d_gn; A.w2 = Tabs<T>::w2(c); A.ion_rho = c->t.n_ion ? Tabs<T>::ion_rho(c) : nullptr;
    A.ngp = c->ngp; A.ngp_pad = c->ngp_pad;
    for (int k = 0; k < 3; k++) { A.nmax[k] = c->t.n_max[k]; A.off[k] = c->off[k]; }
    A.rowlen = c->rowlen;
    A.rho_out = nullptr;
    A.partial = c->static_scratch; /* the device address from cudaGetSymbolAddress, never the symbol's name */
    A.n_slabs = n_slabs;
    for (int i = 0; i < 9; i++) A.binv[i] = c->t.binv[i];
    const size_t smem = (size_t)RECIP_CHUNK * c->rowlen * sizeof(T2);
    const long long grid = (long long)W * n_slabs;
    ewald_status st;
    if (c->t.dim == 3) {
        if ((st = allow_smem(c, recip_kernel<T, 3>, smem)) != EWALD_OK) return st;
        recip_kernel<T, 3><<<(unsigned)grid, RECIP_THREADS, smem, c->stream>>>(A);
    } else {
        if ((st = allow_smem(c, recip_kernel<T, 2>, smem)) != EWALD_OK) return st;
        recip_kernel<T, 2><<<(unsigned)grid, RECIP_THREADS, smem, c->stream>>>(A);
    }
    CU_TRY(c, cudaGetLastError());
    static_slab_sum_kernel<<<(W + 127) / 128, 128, 0, c->stream>>>(c->static_scratch, n_slabs, W, e_recip);
    CU_TRY(c, cudaGetLastError());
    c->launches += 2;
    return EWALD_OK;
}

extern "C" ewald_status ewald_recip_energy_static(ewald_ctx *c, int W, int n, ewald_prec prec, const void *pos,
                                                  const void *q, double *e_recip)
{
    ewald_status st = check_batch(c, W, n, prec, pos, q);
    if (st != EWALD_OK) return st;
    if (W == 0) return EWALD_OK;
    if (!e_recip) return fail(c, EWALD_EINVAL, "null e_recip");
    EWALD_DEVICE(c);
    if (!c->static_scratch) {
        c->err = "static scratch unavailable: " + c->static_err;
        return EWALD_ECUDA;
    }
    const int per = RECIP_THREADS * RECIP_GPT;
    const int n_slabs = (c->ngp + per - 1) / per;
    const unsigned long long need = (unsigned long long)W * (unsigned long long)n_slabs;
    if (need > STATIC_SCRATCH_DOUBLES) {
        char msg[256];
        std::snprintf(msg, sizeof msg,
                      "ewald_recip_energy_static: n_walkers (%d) x slabs (%d) = %llu partial sums exceed the static "
                      "scratch of %llu doubles (EWALD_STATIC_SCRATCH_BYTES = %d); at most %llu walkers per call here",
                      W, n_slabs, need, (unsigned long long)STATIC_SCRATCH_DOUBLES, (int)EWALD_STATIC_SCRATCH_BYTES,
                      (unsigned long long)(STATIC_SCRATCH_DOUBLES / n_slabs));
        return fail(c, EWALD_ERANGE, msg);
    }
    if (prec == EWALD_F64)
        return recip_energy_static_t<double>(c, W, n, (const double *)pos, (const double *)q, n_slabs, e_recip);
    return recip_energy_static_t<float>(c, W, n, (const float *)pos, (const float *)q, n_slabs, e_recip);
}
