/* ewald_internal.h -- shared between the host setup (ewald_setup.cpp) and the CUDA side
 * (ewald_kernels.cu, ewald_api.cu).  Not part of the public boundary (include/ewald.h). */
#ifndef EWALD_INTERNAL_H
#define EWALD_INTERNAL_H

#include <string>
#include <vector>

#include "ewald.h"

namespace ewald {

/* Host plan of the octant-form reciprocal kernel (ewald_recip_oct.cuh; any cell).
 * A table row of one (walker, particle) holds the (cos, sin) pairs X1[0..nmax1] (times q), X2[0..nmax2],
 * X3[0..nmax3].  An item is a block of <= npb consecutive n1 >= 1 (block 0 also carries n1 = 0) of
 *   OCT_FULL  one column (n2 > 0, n3 > 0): four products X2[n2] (x) X3[n3] per particle, or
 *   OCT_PAIR  two half columns -- (n2, 0), (0, n3) or (0, 0); in 2D any two n2 -- with two products each.
 * Offsets are in pair units within a row. */
constexpr int OCT_FULL = 0, OCT_PAIR = 1, OCT_EMPTY = 2;
struct OctPlan {
    bool valid = false;
    int dim = 3, npb = 0;
    int rowlen = 0, off[3] = {0, 0, 0};
    int n_items = 0;
    std::vector<int> kind, offA, offB, offX, np, c0; /* [n_items] */
    std::vector<int> col;                      /* [n_items][5] = axis and n of half A, of half B (axis -1: none), first n1 of the block - 1 */
    std::vector<double> wt;                    /* [n_items][1 + npb][4] class weights (FULL: ++, +-, -+, --; PAIR: A+, A-, B+, B-) */
    std::vector<double> tion;                  /* [n_items][1 + 2 npb][4]; empty without fixed charges */
};

/* Lane assignment of the CTAs of one group of `wc` walkers (make_oct_launch). */
struct OctLaunch {
    int wc = 0, n_warps = 0, n_slabs = 1; /* warps per CTA; CTAs per walker group */
    int rank_stride = 1;        /* most lanes any walker has in one CTA */
    double cost = 0;            /* FP64 operations per particle the group is charged: 128 n_slabs x its busiest sub-partition */
    double fma_ops = 0;         /* FMA + product operations per particle actually executed, whole group */
    std::vector<int> lane;      /* [n_slabs][32 n_warps][4] = local walker | rank << 8, item, offA | offB << 16, offX */
    std::vector<int> variant;   /* [n_slabs][n_warps] np | c0 << 8 | kind << 16 */
};

/* Host plan of the FP64 tensor-core form of the octant kernel (ewald_recip_mma.cuh): the structure-factor sums
 * T[entry][product] = sum_i X1_entry(i) P_product(i) are a contraction over the particles, done by m8n8k4 DMMAs.
 * A group is 8 columns of one kind (FULL: (n2 > 0, n3 > 0), four products; HALF: one phase, two products);
 * a slot is what one warp accumulates in one set of registers: a FULL group or two HALF groups, times the M-tiles
 * t0, t0 + 1 (M-tile t = the X1 doubles 8t..8t+7 = cos/sin of n1 = 4t..4t+3). */
constexpr int MMA_SMAX = 3;     /* slots per warp */
constexpr int MMA_WARPS = 12;   /* warps per CTA */
struct MmaSlot {
    int kind = OCT_FULL;        /* OCT_FULL or OCT_PAIR (two HALF groups) */
    int t0 = 0, nt = 1;         /* first M-tile, number of M-tiles (1 or 2) */
    int ax[2][8], n[2][8];      /* FULL: [0] = (axis 1, n2), [1] = (axis 2, n3) of column c; PAIR: half column c of group A / B; axis -1: none */
};
struct MmaPlan {
    bool valid = false;
    int dim = 3, rowlen = 0, off[3] = {0, 0, 0};
    std::vector<MmaSlot> slots;
    std::vector<double> wt;     /* [n_slots][2 tiles][4 n1][8 columns][4 classes] */
    std::vector<double> tion;   /* [n_slots][2 tiles][8 doubles][8 columns][4 products]; empty without fixed charges */
    double dmma_per_quad = 0;   /* DMMAs per four particles and walker */
};
/* Slots of one walker dealt to `wpw` warps (all slots of a warp share t0, at most MMA_SMAX each). */
struct MmaLaunch {
    int wpw = 0;
    bool valid = false;
    double max_dmma = 0;        /* DMMAs per quad of the busiest warp */
    std::vector<int> lane;      /* [wpw][MMA_SMAX][32][2]: offsets (in pairs, within a quad block) of the lane's two operands */
    std::vector<int> meta;      /* [wpw][MMA_SMAX][4]: kind (OCT_EMPTY: none), t0, nt, slot index */
};

/* Pair-function table F(t) = erfc(sqrt t)/sqrt t on bins cut from the bits of t (ewald_setup.cpp). */
struct PairTable {
    int kbits = 0, degree = 0, e_min = 0; /* 2^kbits bins per binary octave, from 2^e_min upwards   */
    int n_bins = 0;
    double t_min = 0, t_max = 0;          /* the table covers [t_min, t_max)                         */
    std::vector<double> coef;             /* [n_bins][degree + 1], variable u = t - bin centre       */
};
constexpr int PAIR_K64 = 5, PAIR_DEG64 = 7;  /* FP64:  32 bins per octave, degree 7: rel. error < 2e-14 */
constexpr int PAIR_K32 = 5, PAIR_DEG32 = 3;  /* FP32:  32 bins per octave, cubic:   rel. error < 3e-9  */
#ifndef EWALD_FAR_T0
#define EWALD_FAR_T0 13
#endif
constexpr int FAR_T0 = EWALD_FAR_T0, FAR_KB = 3, FAR_REP = 8; /* far shell of the FP64 kernels (FarFmt) */
constexpr int MAX_SPECIES = 4;               /* distinct fixed charges the bare-t real-space path handles  */
constexpr int PAIR_EMIN = -6;                /* t < 2^-6 (kappa r < 1/8) takes the direct formula      */

/* Everything ewald_setup computes on the host, in long double, before rounding (PAPER.md:359:
 * "lookup tables for Ewald interactions ... always performed using DP arithmetic"). */
struct HostTables {
    int dim = 3;
    double kappa = 0, g_cutoff = 0, r_cutoff = 0;
    double a[9];     /* lattice vectors as rows (dim = 2 embedded with a3 = (0,0,1))            */
    double binv[9];  /* rows b_k / 2pi : fractional coordinate s_k = r . binv[k]                 */
    double volume = 0;
    bool orthogonal = false; /* a_k along Cartesian axis k                                       */
    int n_max[3] = {0, 0, 0};
    /* canonical half set G+, lexicographic in (n1,n2,n3) */
    std::vector<int> g_n;      /* [ngp][3]                                                      */
    std::vector<double> g_w2;  /* [ngp]  2 w(G): E_recip = sum_{G+} g_w2 |rho|^2                */
    /* lattice images scanned per (reduced) pair displacement */
    std::vector<double> img;   /* [nimg][3] Cartesian R                                         */
    std::vector<int> img_m;    /* [nimg][3] integer coefficients                                */
    double xi_r = 0;       /* sum_{R != 0, R < rc} erfc(kappa R)/R                               */
    double self_coef = 0;  /* E_self = -self_coef * sum q^2,  self_coef = kappa/sqrt(pi)          */
    double bg_coef = 0;    /* E_bg = -bg_coef/2 * Q^2 ; pi/(Omega kappa^2) (3D), 2 sqrt(pi)/(A kappa) (2D) */
    double v_m = 0;        /* Eq. 4 */
    /* real-space evaluation tables (ewald_realspace.cuh) */
    int m_shift = 0;              /* orthorhombic cells: images -m..m per axis reach r_cutoff      */
    PairTable pair64, pair32;
    std::vector<float> far_tab;   /* [n_far][FAR_REP][4] */
    int n_far = 0;
    /* fixed charges */
    int n_ion = 0;
    std::vector<double> ion_pos; /* [n_ion][3] */
    std::vector<double> ion_q;
    std::vector<double> ion_rho; /* [ngp][2], sum_I q_I exp(iG.r_I)                              */
    bool ion_uniform = true;     /* at most MAX_SPECIES distinct fixed charges */
    std::vector<int> sp_start;   /* [n_species + 1] first ion of each species (ions are kept grouped by charge) */
    double ion_q2 = 0, ion_qsum = 0, ion_real = 0; /* sum q^2, sum q, sum_{I<J} q_I q_J psi(r_IJ) */
    OctPlan oct;
    MmaPlan mma;
};

struct HostTables;
void build_oct_plan(HostTables *t);
void fill_oct_ion(HostTables *t);
void make_oct_launch(const OctPlan &p, int wc, int max_warps, OctLaunch *out);
void fill_mma_ion(HostTables *t);
void make_mma_launch(const MmaPlan &p, int wpw, MmaLaunch *out);


/* Returns EWALD_OK or an error status with a message. */
ewald_status build_tables(int dim, const double *cell, double kappa, double g_cutoff,
                          double r_cutoff, HostTables *out, std::string *err);
void build_pair_table(int kbits, int degree, int e_min, double t_max, PairTable *out);
double eval_pair_table(const PairTable &p, double t);
void build_far_table(int t0, int kb, int rep, double t_max, std::vector<float> *tab, int *n_far);
ewald_status build_fixed_charges(HostTables *t, int n_ion, const double *pos, const double *q,
                                 std::string *err);

} // namespace ewald
#endif
