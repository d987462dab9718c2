"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module holds NO Ewald arithmetic: only cell sizes, cut-off parameters and random draws.  The same
arrays are handed to the CPU oracle and to the CUDA path (neither imports the other).  The inputs stand in
for the paper's CASINO VMC workloads (3D HEG N = 100-1630; 2D HEG; bulk
solids), whose input decks are not available: uniform-random positions replace
Metropolis-sampled ones (same shapes, sizes and costs).

Every array is float64; the FP32 path receives these arrays rounded to float32 by the caller.
Positions are arrays of points [n_walkers, n, dim]; the library's SoA layout is produced by the binding.
"""
import math
from dataclasses import dataclass, field

import numpy as np

SEED0 = 250702888  # arxiv id; seed of config c is SEED0 + c


@dataclass
class Workload:
    name: str
    index: int            # 1..5, position in BASELINE.json "configs" (1-based)
    dim: int
    n: int                # mobile particles per walker
    n_walkers: int
    L: float              # cell side (bohr); all five cells are cubic / square
    kappa: float          # splitting parameter, inverse bohr (paper's gamma = kappa^2)
    n2_max: int           # keep integer G with n1^2+n2^2+n3^2 <= n2_max
    r_cutoff: float       # real-space spherical cut-off (bohr)
    precisions: tuple
    n_steps: int = 0      # config 5: sequential single-electron moves per walker
    step_sigma: float = 0.0
    cell: np.ndarray = field(default=None, repr=False)
    charges: np.ndarray = field(default=None, repr=False)
    ion_pos: np.ndarray = field(default=None, repr=False)
    ion_q: np.ndarray = field(default=None, repr=False)
    g_cut: float = 0.0    # non-cubic cells: explicit |G| cut-off (inverse bohr); 0 = from n2_max
    sigma: float = 1.0    # electrons around ions: Gaussian width (bohr)

    @property
    def g_cutoff(self):
        if self.g_cut > 0:
            return self.g_cut
        # shell membership is decided by the integer n^2 <= n2_max; the next shell is >= 0.5 % away
        return 2.0 * math.pi / self.L * math.sqrt(self.n2_max) * (1.0 + 1e-9)

    @property
    def n_max(self):
        return int(math.isqrt(self.n2_max))

    @property
    def seed(self):
        return SEED0 + self.index

    def positions(self, n_walkers=None):
        """[n_walkers, n, dim] float64; the first k walkers of a larger draw equal a draw of k walkers."""
        nw = self.n_walkers if n_walkers is None else n_walkers
        rng = np.random.Generator(np.random.PCG64(self.seed))
        if self.ion_pos is None:
            return rng.random((nw, self.n, self.dim)) * self.L
        # config 4: electron 4I+m sits at ion I plus N(0,1) per component (reading R13)
        per_ion = self.n // len(self.ion_pos)
        base = np.repeat(self.ion_pos, per_ion, axis=0)
        return base[None, :, :] + self.sigma * rng.standard_normal((nw, self.n, self.dim))

    def moves(self, n_walkers=None, n_steps=None):
        """Config 5 move stream (reading R14): electron [S, W] int32, displacement [S, W, dim] float64."""
        nw = self.n_walkers if n_walkers is None else n_walkers
        ns = self.n_steps if n_steps is None else n_steps
        rng_e = np.random.Generator(np.random.PCG64(self.seed + 1000))
        rng_d = np.random.Generator(np.random.PCG64(self.seed + 2000))
        # drawn walker-major so that a walker subset / a step prefix is a prefix of the full stream
        electron = rng_e.integers(0, self.n, size=(nw, self.n_steps or ns), dtype=np.int32)[:, :ns]
        disp = rng_d.standard_normal((nw, self.n_steps or ns, self.dim))[:, :ns] * self.step_sigma
        return np.ascontiguousarray(electron.T), np.ascontiguousarray(disp.transpose(1, 0, 2))


def _cubic(L, dim):
    return np.eye(dim) * L


def _diamond_ions(a, reps):
    """Conventional diamond cell (8 sites), reps^3 cells; order: cell loops (i,j,k) outer, basis inner."""
    fcc = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])
    basis = np.concatenate([fcc, fcc + 0.25])
    pts = []
    for i in range(reps):
        for j in range(reps):
            for k in range(reps):
                pts.append((basis + np.array([i, j, k])) * a)
    return np.concatenate(pts)


def config(index):
    """Workload for BASELINE.json configs[index-1]; parameters of SURVEY.md section 8(d)."""
    if index == 1:
        n, rs = 54, 2.0
        L = rs * (4.0 * math.pi * n / 3.0) ** (1.0 / 3.0)
        return Workload("heg3d_n54", 1, 3, n, 8, L, 2.8 / L, 36, 2.2 * L, ("f64",),
                        cell=_cubic(L, 3), charges=-np.ones(n))
    if index == 2:
        n, rs = 250, 1.0
        L = rs * (4.0 * math.pi * n / 3.0) ** (1.0 / 3.0)
        return Workload("heg3d_n250", 2, 3, n, 1024, L, 4.4 / L, 61, 1.3 * L, ("f64", "f32"),
                        cell=_cubic(L, 3), charges=-np.ones(n))
    if index == 3:
        n, rs = 450, 5.0
        L = rs * math.sqrt(math.pi * n)
        return Workload("heg2d_n450", 3, 2, n, 1024, L, 12.0 / L, 484, 0.5 * L, ("f64", "f32"),
                        cell=_cubic(L, 2), charges=-np.ones(n))
    if index == 4:
        a = 10.26
        L = 2 * a
        ions = _diamond_ions(a, 2)
        return Workload("diamond_2x2x2", 4, 3, 256, 4096, L, 4.8 / L, 81, 1.2 * L, ("f64",),
                        cell=_cubic(L, 3), charges=-np.ones(256), ion_pos=ions,
                        ion_q=4.0 * np.ones(len(ions)))
    if index == 5:
        n, rs = 1000, 1.0
        L = rs * (4.0 * math.pi * n / 3.0) ** (1.0 / 3.0)
        return Workload("heg3d_n1000_moves", 5, 3, n, 4096, L, 5.4 / L, 97, 1.1 * L, ("f64", "f32"),
                        n_steps=100, step_sigma=0.3 * rs, cell=_cubic(L, 3), charges=-np.ones(n))
    if index == 6:
        return hbn_hexagonal()
    raise ValueError("config index must be 1..6")


def hbn_hexagonal():
    """a slab-like workload in a NON-orthogonal cell, shaped like the paper's
    9 x 9 hexagonal boron-nitride supercell (synthetic positions, the paper's input deck is
    not available).  Hexagonal cell a1 = (A, 0, 0), a2 = (-A/2, A sqrt(3)/2, 0), a3 = (0, 0, c) with
    A = 9 x 4.75 bohr and c = 20 bohr; 81 B (q = +3) and 81 N (q = +5) ions in the plane z = c/2; 648 electrons,
    4 per ion at the ion plus N(0, 1) per component (neutral cell); kappa = 0.32 / bohr with cut-offs for a
    truncation of 1e-14 (~25 000 G-vectors).  Exercises the general-cell paths: complex half-set reciprocal
    kernel, image-list real-space scan, two ion species (so (t, qq) stack items)."""
    a, reps, c = 4.75, 9, 20.0
    A = a * reps
    cell = np.array([[A, 0.0, 0.0], [-0.5 * A, 0.5 * math.sqrt(3.0) * A, 0.0], [0.0, 0.0, c]])
    prim = np.array([[a, 0.0, 0.0], [-0.5 * a, 0.5 * math.sqrt(3.0) * a, 0.0]])
    ions, q = [], []
    for i in range(reps):
        for j in range(reps):
            for (f1, f2, qq) in ((1.0 / 3.0, 2.0 / 3.0, 3.0), (2.0 / 3.0, 1.0 / 3.0, 5.0)):
                xy = (i + f1) * prim[0] + (j + f2) * prim[1]
                ions.append([xy[0], xy[1], 0.5 * c])
                q.append(qq)
    ions, q = np.array(ions), np.array(q)
    kappa = 0.32
    x = math.sqrt(-math.log(1e-14))
    n = 4 * len(ions)
    return Workload("hbn_9x9_hexagonal", 6, 3, n, 256, A, kappa, 0, x / kappa, ("f64", "f32"),
                    cell=cell, charges=-np.ones(n), ion_pos=ions, ion_q=q, g_cut=2.0 * kappa * x)


class JastrowWorkload:
    """the homogeneous two-body Jastrow terms u (Eq. 6) and p
    (Eq. 7) on the electron gas of a BASELINE energy config.  Inputs only: the integer G vectors of
    the first n_stars stars of the cubic (square) cell -- a star = the G related by permutations and sign changes of
    (n1, n2, n3), one G of each +-G pair kept -- seeded coefficients a_m decaying like 1/|n|^2, and a seeded
    polynomial u with N_u = 8, C = 3 and L_u = 0.49 L (below half the distance to the nearest lattice point,
    PAPER.md:151).  They stand in for CASINO's optimised Jastrow parameters, which are not available."""

    def __init__(self, base_index=2, n_stars=15, n_u=8, C=3, seed=250702888 + 70):
        w = config(base_index)
        self.base, self.dim, self.cell, self.L, self.n, self.n_walkers = w, w.dim, w.cell, w.L, w.n, w.n_walkers
        rng = np.random.Generator(np.random.PCG64(seed))
        m = 6
        rngs = [range(-m, m + 1)] * w.dim + [range(0, 1)] * (3 - w.dim)
        stars = {}
        for n1 in rngs[0]:
            for n2 in rngs[1]:
                for n3 in rngs[2]:
                    v = (n1, n2, n3)
                    if v == (0, 0, 0) or next(c for c in v if c != 0) < 0:   # keep one G of each +-G pair
                        continue
                    key = (n1 * n1 + n2 * n2 + n3 * n3, tuple(sorted(abs(c) for c in v)))
                    stars.setdefault(key, []).append(v)
        keys = sorted(stars)[:n_stars]
        self.g_n = np.array([v for k in keys for v in stars[k]], dtype=np.int32)
        self.star = np.array([i for i, k in enumerate(keys) for _ in stars[k]], dtype=np.int32)
        self.a = np.array([0.05 * rng.uniform(0.5, 1.5) / k[0] for k in keys])
        self.n_stars = len(keys)
        self.C, self.L_u = C, 0.49 * w.L
        # u(r) = (r - L_u)^C sum alpha_l r^l: coefficients so that every term is O(0.1) at r ~ L_u / 2
        self.alpha = np.array([0.1 * rng.uniform(-1, 1) / (0.5 * self.L_u) ** (l + C) for l in range(n_u + 1)])

    def positions(self, n_walkers=None):
        return self.base.positions(n_walkers)


class BlipWorkload:
    """orbitals in a blip basis on the electron gas of BASELINE configs[1] (N = 250,
    so 125 doubly occupied orbitals), a 24^3 blip grid, seeded N(0, 1) coefficients smoothed over neighbouring grid
    points (they stand in for the plane-wave orbitals CASINO re-represents, which are not available).
    A batch = the positions of all electrons of n_walkers walkers."""

    def __init__(self, base_index=2, n_orb=125, grid=(24, 24, 24), seed=250702888 + 90):
        w = config(base_index)
        self.base, self.cell, self.n, self.n_walkers, self.n_orb, self.grid = w, w.cell, w.n, w.n_walkers, n_orb, grid
        rng = np.random.Generator(np.random.PCG64(seed))
        c = rng.standard_normal((n_orb,) + tuple(grid))
        for ax in (1, 2, 3):
            c = 0.5 * c + 0.25 * (np.roll(c, 1, axis=ax) + np.roll(c, -1, axis=ax))
        self.coef = c

    def points(self, n_walkers=None):
        """All electron positions of the first n_walkers walkers as [P, 3]."""
        return self.base.positions(n_walkers).reshape(-1, 3)


def all_configs():
    return [config(i) for i in range(1, 6)]   # the five BASELINE.json configs; config(6) is the NEXT-1 workload
