/*
 * ewald_ref.h -- CPU ORACLE for periodic Coulomb (Ewald) energies.  TEST INFRASTRUCTURE ONLY.
 *
 * This is the plain, slow, obviously-correct restatement of what the hot path computes, written
 * from the paper text (arxiv 2507.02888, /root/reference/PAPER.md):
 *   Eq. 2  V_Ew = sum_{i<j} q_i q_j v_E(r_i - r_j) + 1/2 sum_j q_j^2 v_M
 *   Eq. 3  v_E(r) = 4pi/Omega sum_{G!=0} exp(-G^2/4gamma + iG.r)/G^2
 *                                 + sum_R erfc(sqrt(gamma)|r-R|)/|r-R| - pi/(Omega gamma)
 *   Eq. 4  v_M    = same at r -> 0 without the R = 0 term, minus 2 sqrt(gamma/pi)
 *   PAPER.md:122          symbols; "similar expressions ... in two dimensions" (formula not printed)
 *   PAPER.md:84           Hartree atomic units (energies in Ha, lengths in bohr)
 *   PAPER.md:94           single-particle moves and "(changes in) the potential energy"
 *
 * Convention: every `kappa` below is an inverse length; the paper's gamma = kappa^2
 * (reading R1).  All sums are accumulated in `long double`; results are returned rounded
 * to double.  Nothing here is shared with, imported by, or imports the CUDA path: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Parity pins (tests/test_oracle_pins.py): Madelung constants (NaCl, CsCl, zincblende), Wigner-crystal
 * energies (sc, bcc, fcc; 2D square and triangular), kappa-invariance, brute-force direct lattice
 * sums, O-pair vs O-rho agreement, rho(G) closed forms, scaling/translation/supercell invariances.
 * Configs 1-5 at scale are pinned only through those (no external value exists): see DESIGN.md.
 *
 * Layouts (all HOST memory, caller-owned):
 *   cell[9]   row-major lattice vectors a1,a2,a3 (bohr); dim = 2 uses entries [0,1,3,4]
 *   pos       [n_walkers][n][dim] doubles (array of points)
 *   q         [n] doubles, shared by all walkers
 *   ion_pos   [n_ion][dim], ion_q [n_ion]   (fixed charges, same for all walkers; n_ion may be 0)
 * Return value of every int function: 0 = ok, nonzero = bad argument.
 */
#ifndef EWALD_REF_H
#define EWALD_REF_H
#ifdef __cplusplus
extern "C" {
#endif

/* Number of reciprocal-lattice points with 0 < |G| and G^2 <= g_cutoff^2 (1 + 1e-12)  (full sphere). */
int ewald_ref_num_g(int dim, const double *cell, double g_cutoff);

/* Half set G+ (first non-zero integer component positive), lexicographic order in (n1,n2,n3).
 * n_out: [num_g/2][3] integer coefficients of G = n1 b1 + n2 b2 + n3 b3 (n3 = 0 in 2D).          */
int ewald_ref_gplus(int dim, const double *cell, double g_cutoff, int *n_out);

/* Cut-offs giving truncation below `tol` (relative to the leading term) for a given kappa.          */
int ewald_ref_auto_cutoffs(int dim, const double *cell, double kappa, double tol,
                           double *g_cutoff, double *r_cutoff);

/* O-pair: the paper's Eqs. 2-4 evaluated literally, pair by pair (3D), or their 2D analogue
 * (reading R2).  O(n^2 (N_G + N_img)); meant for n <= ~16.                              */
int ewald_ref_energy_pairwise(int dim, const double *cell, double kappa, double g_cutoff,
                              double r_cutoff, int n, const double *pos, const double *q,
                              double *energy);

/* Pair potential v_E(r) (Eq. 3) and self-image constant v_M (Eq. 4); 2D analogues for dim = 2.     */
int ewald_ref_v_e(int dim, const double *cell, double kappa, double g_cutoff, double r_cutoff,
                  const double *r, double *v_e);
int ewald_ref_v_m(int dim, const double *cell, double kappa, double g_cutoff, double r_cutoff,
                  double *v_m);

/* O-rho: E = E_recip + E_real + E_self + E_bg with rho(G) by direct sincosl per (particle, G).
 * energies [n_walkers]; components [n_walkers][4] = recip, real, self, background (nullable).
 * Mobile particles and fixed ions are simply one set of charges.  n_threads <= 0: OpenMP default. */
int ewald_ref_energy_batch(int dim, const double *cell, double kappa, double g_cutoff,
                           double r_cutoff, int n_walkers, int n, const double *pos,
                           const double *q, int n_ion, const double *ion_pos, const double *ion_q,
                           double *energies, double *components, int n_threads);

/* rho(G) = sum_i q_i exp(i G.r_i) of one configuration on the half set, order of ewald_ref_gplus.
 * re_im: [num_g/2][2].                                                                              */
int ewald_ref_rho(int dim, const double *cell, double g_cutoff, int n, const double *pos,
                  const double *q, double *re_im);

/* Incremental single-particle-move oracle with its own long-double stored rho(G) per walker.
 * For step s = 0..n_steps-1 and walker w: particle electron[s*n_walkers+w] of walker w moves to
 * new_r[(s*n_walkers+w)*dim ..]; delta_e[s*n_walkers+w] = E(after) - E(before); every move is
 * committed (positions in `pos` are updated in place; rho patched).  Fixed ions take part in the
 * real-space and reciprocal sums but never move.  rho_out (nullable): final stored rho of every walker,
 * [n_walkers][num_g/2][2].                                                                          */
int ewald_ref_move_chain(int dim, const double *cell, double kappa, double g_cutoff,
                         double r_cutoff, int n_walkers, int n, double *pos, const double *q,
                         int n_ion, const double *ion_pos, const double *ion_q, int n_steps,
                         const int *electron, const double *new_r, double *delta_e,
                         double *rho_out, int n_threads);

/* Number of OpenMP threads a batch call with n_threads <= 0 will use. */
int ewald_ref_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
