/*
 * ewald.h -- C ABI of the B200 (sm_100a) batched Ewald library.
 *
 * What it computes (arxiv 2507.02888, text in /root/reference/PAPER.md; "PAPER.md:<line>"):
 *   Eq. 2  V_Ew = sum_{i<j} q_i q_j v_E(r_i - r_j) + 1/2 sum_j q_j^2 v_M
 *   Eq. 3  v_E(r) = 4pi/Omega sum_{G!=0} exp(-G^2/4gamma + iG.r)/G^2
 *                                 + sum_R erfc(sqrt(gamma)|r-R|)/|r-R| - pi/(Omega gamma)
 *   Eq. 4  v_M    = the r -> 0 limit without the R = 0 term, minus 2 sqrt(gamma/pi)
 *   PAPER.md:122          2D analogue ("similar expressions ... in two dimensions", not printed;
 *                         DESIGN.md reading R2 gives the form used)
 *   PAPER.md:94           single-particle moves and "(changes in) the potential energy"
 *   Eq. 8  exp(iG.r) = prod_k (exp(i b_k.r))^{n_k}: the phase-power factorisation
 * for many walkers (independent particle configurations) at once.  Eq. 2 is
 * regrouped exactly through the structure factor rho(G) = sum_i q_i exp(iG.r_i):
 *   E = E_recip + E_real + E_self + E_bg
 *
 * Conventions
 *   - `gamma` arguments are kappa, an INVERSE LENGTH: exp(-G^2/4kappa^2), erfc(kappa r).  The paper's
 *     gamma equals kappa^2 (reading R1).  Hartree atomic units: bohr in, Hartree out.
 *   - Pointers are tagged HOST or DEVICE.  DEVICE pointers must live on the context's device.
 *     The caller owns every buffer it passes; the context owns its tables, the stored rho(G) and the
 *     stored positions.
 *   - Batch calls taking DEVICE pointers are asynchronous on the context's stream and never
 *     synchronise; they return launch errors only.  Calls taking HOST data pointers
 *     (`*_host`, ewald_move_delta, ewald_get_rho, ewald_get_positions) copy inside the call and
 *     synchronise the stream before returning.
 *   - A context is not thread-safe.  Coincident particles give inf/nan in that walker's output,
 *     not an error (reading R11).
 *   - Every function returning ewald_status returns EWALD_OK (0) on success; on failure the
 *     context (when there is one) keeps a message readable with ewald_last_error().
 *   - There is no CPU fallback: without a usable CUDA device ewald_setup fails with EWALD_ECUDA.
 *
 * Position layout ("SoA"): [n_walkers][dim][n_pad] with n_pad = ewald_padded_n(n_particles)
 * (n_particles rounded up to a multiple of 4; pad entries are never read as particles).
 */
#ifndef EWALD_B200_H
#define EWALD_B200_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ewald_ctx ewald_ctx; /* opaque */

typedef enum {
    EWALD_OK = 0,
    EWALD_EINVAL = 1,    /* null pointer, n <= 0, dim not 2/3, bad precision enum, ...            */
    EWALD_ESINGULAR = 2, /* |det(cell)| is zero / not finite                                     */
    EWALD_ERANGE = 3,    /* kappa <= 0, g_cutoff <= 0, r_cutoff < 0, G index range beyond tables  */
    EWALD_ESTATE = 4,    /* move before load, walker / electron index out of range, n mismatch    */
    EWALD_ECUDA = 5,     /* CUDA runtime error (message in ewald_last_error)                      */
    EWALD_ENOMEM = 6
} ewald_status;

typedef enum { EWALD_F64 = 0, EWALD_F32 = 1 } ewald_prec;

typedef struct {
    double r_cutoff; /* real-space spherical cut-off (bohr): terms with |r_ij - R| < r_cutoff are
                        kept (reading R3).  0 => automatic: sqrt(-ln 1e-17)/kappa                  */
    int device;      /* CUDA ordinal                                                              */
    void *stream;    /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default */
} ewald_opts;

/* n rounded up to a multiple of 4: the leading dimension of the SoA position layout. */
int ewald_padded_n(int n_particles);

/* Setup (PAPER.md:122 symbols; "moved to the GPU once"; PAPER.md:359 tables in DP):
 * reciprocal basis, the G list 0 < |G|, G^2 <= g_cutoff^2 (1+1e-12) (reading R6), weights, lattice
 * images, Madelung constants -- computed on the host in long double, stored on the device in FP64
 * and as an FP32 rounded copy.
 *   cell : HOST, row-major lattice vectors a1,a2,a3 (bohr); dim = 2 uses entries [0,1,3,4].        */
ewald_status ewald_setup(ewald_ctx **out, int dim, const double cell[9], double gamma,
                         double g_cutoff, const ewald_opts *opts /* nullable */);

void ewald_destroy(ewald_ctx *ctx);

/* Host-only dry run of the same table construction (no CUDA call, usable without a GPU): counts and
 * the walker-independent constants of Eq. 4.  Any output pointer may be null.
 *   num_g: full-sphere G count; num_images: lattice images scanned per pair; n_max[3]: largest
 *   |n_k| in the G list; xi_r = sum_{R!=0} erfc(kappa R)/R; v_m = Eq. 4.                          */
ewald_status ewald_setup_summary(int dim, const double cell[9], double gamma, double g_cutoff,
                                 double r_cutoff, int *num_g, int *num_images, int n_max[3],
                                 double *xi_r, double *v_m);

/* Host-only summary of the work plan of the octant-form reciprocal kernel (any cell): items per walker,
 * n1 pairs per block, warps of a CTA of n_walkers_per_cta walkers, the sum of all class weights of the
 * octant points (must equal the full-sphere sum of w(G): the plan covers every G exactly once) and the FMA + product operations the kernel executes per particle and walker
 * (to compare with the algorithmic N_G + 1).  Any output pointer may be null. */
ewald_status ewald_oct_plan_summary(int dim, const double cell[9], double gamma, double g_cutoff,
                                    int n_walkers_per_cta, int *n_items, int *npb, int *n_warps,
                                    double *weight_sum, double *fma_per_particle);

/* Host-only summary of the plan of the tensor-core (FP64 DMMA) form of the octant kernel: the structure-factor
 * sums of Eq. 8 as a contraction over the particles, cut into slots of 8 columns x 2 M-tiles
 * of 4 n1 values.  n_slots per walker; walkers_per_pass = the most walkers one CTA pass can hold (0: the plan does
 * not fit 12 warps x 3 slots, the FMA-pipe form is used); weight_sum as above (covers every G exactly once);
 * dmma_per_quad = m8n8k4 instructions per four particles and walker.  Any output pointer may be null. */
ewald_status ewald_mma_plan_summary(int dim, const double cell[9], double gamma, double g_cutoff,
                                    int *n_slots, int *walkers_per_pass, double *weight_sum,
                                    double *dmma_per_quad);

/* Host-only evaluation of the pair-function table the real-space kernels read,
 *     F(t) = erfc(sqrt t)/sqrt t,  t = kappa^2 |r_ij - R|^2   (a term of the real-lattice sum of Eq. 3,
 * PAPER.md:117, is kappa q_i q_j F(t)): a piecewise polynomial in t on bins cut from the binary format of
 * t (FP64 kernels: 128 bins per octave, quintic; FP32 kernels: 32 bins per octave, cubic), built in long
 * double at setup to cover 2^-6 <= t < t_max; outside that range the direct formula is
 * returned, as in the kernels.  t, value: HOST [n].  For tests of the table builder.               */
ewald_status ewald_pair_table_eval(ewald_prec prec, double t_max, int n, const double *t, double *value);

/* Change the stream later calls are issued on (cudaStream_t; NULL = default stream). */
ewald_status ewald_set_stream(ewald_ctx *ctx, void *stream);

/* Which reciprocal-space kernel ewald_energy_batch uses (both compute the same E_recip; for tests
 * and measurements): 0 = automatic (FP64: the octant form on the FP64 tensor cores when its plan fits, else
 * and in FP32 the octant form on the FMA pipe), 1 = complex half-set form, 3 = tensor-core octant form (FP64;
 * EWALD_ESTATE at the next energy call when its plan does not fit),
 * 2 = octant form (EWALD_ESTATE at the next energy call if no plan could be built: G indices beyond
 * 16 bits). */
ewald_status ewald_set_recip_variant(ewald_ctx *ctx, int variant);

/* How the FP64 real-space kernels treat the far shell of the real-lattice sum of Eq. 3:
 * 0 = default: terms with kappa^2 |r_ij - R|^2 >= 16 (each below erfc(4)/4 = 3.9e-9 in units of
 *     kappa q_i q_j) are evaluated in FP32 arithmetic from a fixed-point copy of t; this changes the sum
 *     by less than 1e-7 of the far shell's own total, i.e. < 1e-14 of E_real;
 * 1 = every term in FP64.  FP32 contexts ignore the setting.  For tests and measurements. */
ewald_status ewald_set_real_variant(ewald_ctx *ctx, int variant);

/* Fixed charges (ions) that belong to every walker and never move (config 4; reading R13).  They
 * enter rho(G), the real-space sum, E_self and E_bg exactly like mobile particles (Eq. 2 over all
 * charges); their mutual terms are evaluated once here.  n_ion = 0 removes them.
 *   pos : HOST [n_ion][dim],  q : HOST [n_ion].  Must be called before ewald_load_walkers.        */
ewald_status ewald_set_fixed_charges(ewald_ctx *ctx, int n_ion, const double *pos, const double *q);

/* Full Ewald energy of every walker (Eq. 2 with Eqs. 3-4).
 *   positions : DEVICE SoA [n_walkers][dim][n_pad], double (EWALD_F64) or float (EWALD_F32)
 *   charges   : DEVICE [n_particles], same type; shared by all walkers (reading R20)
 *   energies  : DEVICE [n_walkers] double, Hartree (always FP64, reading R16)
 *   components: DEVICE [n_walkers][4] double = E_recip, E_real, E_self, E_bg; nullable
 * n_walkers = 0 is a no-op.  EWALD_F32: all hot-loop arithmetic in FP32, block partial sums and the
 * final combination in FP64 (reading R16).                                                         */
ewald_status ewald_energy_batch(ewald_ctx *ctx, int n_walkers, int n_particles, ewald_prec prec,
                                const void *positions, const void *charges, double *energies,
                                double *components);

/* Same through HOST buffers: copies positions and charges to the device, runs, copies the
 * energies (and components, if non-null) back, synchronises.  Layouts as above.                   */
ewald_status ewald_energy_batch_host(ewald_ctx *ctx, int n_walkers, int n_particles,
                                     ewald_prec prec, const void *positions, const void *charges,
                                     double *energies, double *components);

/* Allocation-free entry point, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops,
 * harnesses that forbid it): the reciprocal-space energy E_recip of every walker (steps S1-S4: the reciprocal sum
 * of Eq. 3; the same value as components[...][0] of ewald_energy_batch), computed by the complex
 * half-set kernel (the one ewald_set_recip_variant(ctx, 1) selects) with its scratch -- one partial sum per walker
 * and slab of 1024 G-vectors of the half set -- in a file-scope device array of EWALD_STATIC_SCRATCH_BYTES that
 * every GPU holding the library keeps until the process exits.  Its device address is taken at ewald_setup.
 *   positions, charges : DEVICE, layouts and types as for ewald_energy_batch
 *   e_recip            : DEVICE [n_walkers] double, Hartree
 * Limit: n_walkers * ceil(N_G+ / 1024) <= EWALD_STATIC_SCRATCH_BYTES / 8 = 131072 (N_G+ = ewald_num_g / 2; e.g.
 * 131072 walkers per call on configs 1-5, whose half sets fit one slab); beyond it EWALD_ERANGE, nothing launched,
 * ewald_last_error says by how much.  EWALD_ECUDA if the array's address could not be taken at set-up.
 * The call enqueues two kernels on the context's stream and returns; it calls no cudaMalloc, cudaFree, event or
 * stream creation and does not synchronise.  Nothing in the array has to start at zero: every element a call reads
 * it has written itself, so leftovers of earlier calls are harmless.  EVERY call on a device, from any context,
 * shares the one array: calls that can overlap on the GPU (different streams, different contexts or host threads
 * without ordering between them) race on it; order them on one stream or with events.  n_walkers = 0 is a
 * no-op.  The fixed charges of ewald_set_fixed_charges enter as in ewald_energy_batch. */
#define EWALD_STATIC_SCRATCH_BYTES (1 << 20)
ewald_status ewald_recip_energy_static(ewald_ctx *ctx, int n_walkers, int n_particles, ewald_prec prec,
                                       const void *positions, const void *charges, double *e_recip);

/* Store a walker population in the context for single-particle moves: copies the positions and
 * charges and computes and stores rho(G) (of mobile particles plus fixed charges) per walker, in
 * the precision given.  Replaces any earlier population.  DEVICE pointers, layouts as above.       */
ewald_status ewald_load_walkers(ewald_ctx *ctx, int n_walkers, int n_particles, ewald_prec prec,
                                const void *positions, const void *charges);

/* Single-particle moves.  Move m takes particle electron[m] of walker walker[m] from its
 * stored position r to new_r[m]:
 *   delta_e[m] = E(after) - E(before)
 *     = sum_{G+} 2 w(G) [ 2 q Re(conj(rho(G)) d(G)) + q^2 |d(G)|^2 ],  d(G) = e^{iG.r'} - e^{iG.r}
 *     + q sum_{j != k} q_j [ psi(r' - r_j) - psi(r - r_j) ],  psi(d) = sum_R erfc(kappa|d-R|)/|d-R|
 * (the self, background and Madelung terms of Eqs. 2-4 do not change).  commit = 1 also patches
 * rho(G) += q d(G) and the stored position; commit = 0 leaves the state untouched.
 *   walker, electron : DEVICE [n_moves] int; walker indices distinct within one call
 *   new_r            : DEVICE [n_moves][dim], type of the loaded precision
 *   delta_e          : DEVICE [n_moves] double
 * Out-of-range indices make that move's delta_e NaN and leave the state untouched.               */
ewald_status ewald_move_delta_batch(ewald_ctx *ctx, int n_moves, const int *walker,
                                    const int *electron, const void *new_r, int commit,
                                    double *delta_e);

/* Same through HOST buffers (copies in, runs, copies delta_e back, synchronises). */
ewald_status ewald_move_delta_batch_host(ewald_ctx *ctx, int n_moves, const int *walker,
                                         const int *electron, const void *new_r, int commit,
                                         double *delta_e);

/* Scalar form: one move, HOST new_r (double[dim] whatever the loaded precision), HOST delta_e.
 * Validates the indices (EWALD_ESTATE) and synchronises.                                          */
ewald_status ewald_move_delta(ewald_ctx *ctx, int walker, int electron, const double *new_r,
                              int commit, double *delta_e);

/* Introspection.  Canonical half set G+: integer triples (n1,n2,n3), G = n1 b1 + n2 b2 + n3 b3,
 * first non-zero component positive, sorted lexicographically by (n1,n2,n3); n3 = 0 in 2D.       */
int ewald_num_g(const ewald_ctx *ctx);      /* full-sphere count, G = 0 excluded (= 2 |G+|)   */
int ewald_num_images(const ewald_ctx *ctx); /* lattice images scanned per pair                */
double ewald_r_cutoff(const ewald_ctx *ctx);
ewald_status ewald_get_g(const ewald_ctx *ctx, int *n_out /* HOST [num_g/2][3] */);
/* Stored rho(G) of one walker on G+, canonical order, as (re, im) doubles. */
ewald_status ewald_get_rho(ewald_ctx *ctx, int walker, double *re_im /* HOST [num_g/2][2] */);
/* Stored positions of one walker as points, doubles. */
ewald_status ewald_get_positions(ewald_ctx *ctx, int walker, double *pos /* HOST [n][dim] */);
/* Walker-independent constants: xi_R = sum_{R!=0} erfc(kappa R)/R, v_M of Eq. 4, and the
 * energy of the fixed charges among themselves (0 without ions).  Any pointer may be null.      */
ewald_status ewald_get_constants(const ewald_ctx *ctx, double *xi_r, double *v_m, double *e_fixed);

/* Arithmetic-pipe probe used by bench.py for the roofline denominator: every thread runs `iters`
 * rounds of 8 independent dependent-chain FMAs (FP64 or FP32); returns the achieved FLOP/s in
 * *flops (2 per FMA), timed with CUDA events on the context's stream.  Synchronises.            */
ewald_status ewald_probe_fma(ewald_ctx *ctx, ewald_prec prec, int iters, double *flops);

/* FP64 tensor-core probe (the roofline denominator of the tensor-core form of the reciprocal kernel): every warp
 * of one 256-thread CTA per SM issues `iters` rounds of 32 independent m8n8k4 DMMAs; *flops = FLOP/s (512 per
 * DMMA).  On B200 it measures the same 37 TFLOP/s as the FP64 FMA chain.  Synchronises. */
ewald_status ewald_probe_dmma(ewald_ctx *ctx, int iters, double *flops);

/* Per-kernel device timers: when enabled, every kernel launch is bracketed by CUDA events on the
 * context's stream.  ewald_profile_read synchronises, returns and resets the accumulated device
 * milliseconds and launch counts per kernel class:
 *   [0] reciprocal (S1-S4)  [1] real-space (S5)  [2] combine + charge sums (S6)  [3] move (S7).   */
ewald_status ewald_profile_enable(ewald_ctx *ctx, int on);
ewald_status ewald_profile_read(ewald_ctx *ctx, double ms[4], int launches[4]);

/* Shape of the context's last real-space launch (which = 0: real_kernel) or move launch (which = 1: move_kernel),
 * zeros before the first: out HOST [8] = threads per CTA, dynamic shared memory in bytes, near-stack and far-stack
 * capacity per lane in bare-t items, bins of the near table staged, bins of the far table staged (0 = far shell
 * off), CTAs launched, 1 if the far stack is serviced once per pair.  No device work. */
ewald_status ewald_launch_shape(const ewald_ctx *ctx, int which, int out[8]);

/* Number of kernels this context has launched since ewald_setup. */
long long ewald_launch_count(const ewald_ctx *ctx);

const char *ewald_last_error(const ewald_ctx *ctx); /* never null; "" if none */
const char *ewald_version(void);

#ifdef __cplusplus
}
#endif
#endif
