/* jastrow.h -- C ABI of the batched homogeneous two-body Jastrow terms.
 *
 * /root/reference/PAPER.md section 2.3: "the cost of evaluating the Jastrow factor is usually dominated by the
 * evaluation of the homogeneous two-body terms.  We therefore focus on offloading the evaluation of the values
 * and derivatives of the two-body terms u(r) and p(r)", with
 *   Eq. 6  u(r) = sum_{l=0}^{N_u} alpha_l r^l (r - L_u)^C Theta(L_u - r),
 *   Eq. 7  p(r) = sum_{m=1}^{N_p} a_m sum_{G in star_m^+} cos(G.r),
 *   Eq. 8  cos(G.r) from powers of three complex exponentials, "computed and buffered".
 * For every walker of a batch the library returns J = sum_{i<j} [u(r_ij) + p(r_ij)] and, per particle i,
 * grad_i J and lap_i J; and, on a stored population, Delta J of single-particle moves.
 * L_u must be below half the distance to the nearest lattice point: only the minimum image of a
 * pair can lie inside the cut-off.  Same conventions as ewald.h: plain HOST / DEVICE pointers, opaque context,
 * ewald_status codes, asynchronous on the context's stream unless stated, no CPU fallback.
 */
#ifndef JASTROW_H
#define JASTROW_H
#include "ewald.h"
#ifdef __cplusplus
extern "C" {
#endif

typedef struct jastrow_ctx jastrow_ctx;

/* n_u < 0: no u term; n_g = 0: no p term.  alpha: HOST [n_u + 1]; g_n: HOST [n_g][3] integer coefficients of
 * G = n1 b1 + n2 b2 + n3 b3 (n3 = 0 in 2D), one G of each +-G pair; star: HOST [n_g], index into a: HOST [n_stars].
 * EWALD_EINVAL: bad argument; EWALD_ERANGE: l_u not below half the shortest lattice vector, or |n_k| > 31. */
ewald_status jastrow_setup(jastrow_ctx **out, int dim, const double cell[9], int n_u, const double *alpha,
                           double l_u, int c_exp, int n_g, const int *g_n, const int *star, int n_stars,
                           const double *a, int device, void *stream);

/* positions: DEVICE SoA [n_walkers][dim][n_pad] (n_pad = ewald_padded_n(n)), double or float per prec.
 * value: DEVICE [n_walkers]; grad: DEVICE [n_walkers][dim][n_pad] or null; lap: DEVICE [n_walkers][n_pad] or
 * null -- always double.  The FP32 path computes in float with FP64 block sums. */
ewald_status jastrow_batch(jastrow_ctx *ctx, int n_walkers, int n_particles, ewald_prec prec, const void *positions,
                           double *value, double *grad, double *lap);

/* Stores a population (positions and the structure factors S(G) = sum_i exp(iG.r_i) of the p term). */
ewald_status jastrow_load_walkers(jastrow_ctx *ctx, int n_walkers, int n_particles, ewald_prec prec,
                                  const void *positions);
/* Delta J of moving `electron` of `walker` to new_r (DEVICE [n_moves][dim], the loaded precision); commit = 1
 * patches the stored S(G) and position.  Walkers of one call must be distinct.  delta: DEVICE [n_moves] double;
 * an out-of-range walker or electron gives NaN and changes nothing. */
ewald_status jastrow_move_delta_batch(jastrow_ctx *ctx, int n_moves, const int *walker, const int *electron,
                                      const void *new_r, int commit, double *delta);

/* Device milliseconds and launches of jastrow_batch since the last read (CUDA events on the stream when enabled). */
ewald_status jastrow_profile_enable(jastrow_ctx *ctx, int on);
ewald_status jastrow_profile_read(jastrow_ctx *ctx, double *ms, int *launches);
const char *jastrow_last_error(const jastrow_ctx *ctx);
void jastrow_destroy(jastrow_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
