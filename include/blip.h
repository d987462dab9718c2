/* blip.h -- C ABI of the batched evaluation of orbitals in a blip (cubic B-spline) basis.
 *
 * /root/reference/PAPER.md section 2.4 (lines 161-165): an orbital at a particle position = "looking up the
 * particle's position in the spline grid followed by the evaluation of a small number of cubic polynomials defining
 * the blip basis functions, followed by multiplication of the blip functions by coefficients for each orbital".
 * CASINO does this with many 64-element ddot / dgemv calls, which the paper could not make pay through cuBLAS
 * ("batching ... left for future investigation"); here ONE kernel evaluates every orbital at
 * every position of a batch, value, gradient and Laplacian:
 *     psi_o(r) = sum_{abc in 4x4x4} c_o[i1+a][i2+b][i3+c] Theta(u1-i1-a) Theta(u2-i2-b) Theta(u3-i3-c),  u_k = N_k s_k(r),
 *     Theta(x) = 1 - 3/2 x^2 + 3/4 |x|^3 (|x| <= 1), 1/4 (2 - |x|)^3 (1 <= |x| <= 2), 0 otherwise (reading R21).
 * Same conventions as ewald.h (status codes, HOST / DEVICE pointers, stream, no CPU fallback).  3D cells only.
 */
#ifndef BLIP_H
#define BLIP_H
#include "ewald.h"
#ifdef __cplusplus
extern "C" {
#endif

typedef struct blip_ctx blip_ctx;

/* coef: HOST [n_orb][N1][N2][N3] doubles (copied, stored on the device point-major [N1][N2][N3][n_orb padded to 32]
 * in FP64 and FP32); grid = (N1, N2, N3), each >= 4, periodic with the cell. */
ewald_status blip_setup(blip_ctx **out, const double cell[9], const int grid[3], int n_orb, const double *coef,
                        int device, void *stream);
/* points: DEVICE SoA [3][n_pad] (double or float per prec), n_points <= n_pad.
 * psi: DEVICE [n_points][n_orb]; grad: DEVICE [n_points][3][n_orb] or null; lap: DEVICE [n_points][n_orb] or
 * null -- always double; the FP32 path reads the FP32 coefficients and accumulates in float. */
ewald_status blip_eval_batch(blip_ctx *ctx, int n_points, int n_pad, ewald_prec prec, const void *points,
                             double *psi, double *grad, double *lap);
ewald_status blip_profile_enable(blip_ctx *ctx, int on);
ewald_status blip_profile_read(blip_ctx *ctx, double *ms, int *launches);
const char *blip_last_error(const blip_ctx *ctx);
void blip_destroy(blip_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
