"""Pins for the CPU oracle against things the paper and the mathematics fix (no GPU, no CUDA code).

Each test is chosen so that a plausible mistake in oracle/ewald_ref.c (dropped term, wrong sign or
prefactor, transposed lattice, wrong half-set weight, wrong 2D form) fails at least one of them.
Formulas under test: PAPER.md Eqs. 2-4 (lines 112-120), 2D analogue (reading R2).
"""
import math

import mpmath
import numpy as np
import pytest

from oracle import ewald_ref as ora

SQ3 = math.sqrt(3.0)


def energy(dim, cell, kappa, pos, q, tol=1e-17, **kw):
    g, r = ora.auto_cutoffs(dim, cell, kappa, tol)
    e, comp = ora.energy_batch(dim, cell, kappa, g, r, np.asarray(pos, float)[None], q, **kw)
    return e[0]


def wigner_E_rs(dim, cell, basis_frac, kappa):
    cell = np.asarray(cell, float)
    pos = np.asarray(basis_frac, float) @ cell
    n = len(pos)
    vol = abs(np.linalg.det(cell))
    rs = (3 * vol / (4 * math.pi * n)) ** (1 / 3) if dim == 3 else math.sqrt(vol / (math.pi * n))
    return energy(dim, cell, kappa, pos, -np.ones(n)) / n * rs


FCC = [[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]]


# ------------------------------------------------------------------ closed forms, 3D
def test_vm_simple_cubic(golden):
    # Eq. 4 alone: all four pieces (G sum, R sum, -2 sqrt(gamma/pi), -pi/(Omega gamma)) must be right
    for L, kappa in [(1.0, 2.3), (3.7, 0.9)]:
        cell = np.eye(3) * L
        g, r = ora.auto_cutoffs(3, cell, kappa)
        assert ora.v_m(3, cell, kappa, g, r) * L == pytest.approx(golden["vm_L_sc_3d"], rel=2e-15)


def test_wigner_crystals_3d(golden):
    assert wigner_E_rs(3, np.eye(3), [[0, 0, 0]], 2.5) == pytest.approx(golden["wigner_sc_E_rs"], rel=1e-14)
    assert wigner_E_rs(3, np.eye(3), [[0, 0, 0], [.5, .5, .5]], 3.0) == pytest.approx(
        golden["wigner_bcc_E_rs"], rel=1e-14)
    assert wigner_E_rs(3, np.eye(3), FCC, 3.5) == pytest.approx(golden["wigner_fcc_E_rs"], rel=1e-14)
    dia = FCC + [[x + .25, y + .25, z + .25] for x, y, z in FCC]
    assert wigner_E_rs(3, np.eye(3), dia, 4.0) == pytest.approx(golden["wigner_diamond_E_rs"], rel=1e-14)
    # primitive (non-orthogonal) cells of the same crystals: exercises the general-cell path
    bcc_prim = 0.5 * np.array([[-1, 1, 1], [1, -1, 1], [1, 1, -1.]])
    fcc_prim = 0.5 * np.array([[0, 1, 1], [1, 0, 1], [1, 1, 0.]])
    assert wigner_E_rs(3, bcc_prim, [[0, 0, 0]], 3.0) == pytest.approx(golden["wigner_bcc_E_rs"], rel=1e-14)
    assert wigner_E_rs(3, fcc_prim, [[0, 0, 0]], 3.0) == pytest.approx(golden["wigner_fcc_E_rs"], rel=1e-14)


def nacl_cell(a=1.0):
    pos, q = [], []
    for i in range(2):
        for j in range(2):
            for k in range(2):
                pos.append([i * a / 2, j * a / 2, k * a / 2])
                q.append((-1.0) ** (i + j + k))
    return np.eye(3) * a, np.array(pos), np.array(q)


def test_madelung_nacl_benson_series(golden):
    # Benson's formula (independent of Ewald): M = 12 pi sum_{m,n odd >= 1} sech^2(pi/2 sqrt(m^2+n^2))
    s = mpmath.mpf(0)
    for m in range(1, 40, 2):
        for n in range(1, 40, 2):
            s += mpmath.sech(mpmath.pi / 2 * mpmath.sqrt(m * m + n * n)) ** 2
    M = float(12 * mpmath.pi * s)
    assert M == pytest.approx(golden["madelung_nacl"], rel=1e-15)
    a = 1.7
    cell, pos, q = nacl_cell(a)
    assert energy(3, cell, 2.0, pos, q) == pytest.approx(-8 * M / a, rel=1e-14)
    # 2-ion fcc primitive cell (non-orthogonal): E = -M/(a/2)
    prim = 0.5 * a * np.array([[0, 1, 1], [1, 0, 1], [1, 1, 0.]])
    e2 = energy(3, prim, 2.2, [[0, 0, 0], [a / 2, 0, 0]], [1.0, -1.0])
    assert e2 == pytest.approx(-M / (a / 2), rel=1e-14)


def test_madelung_cscl_zincblende(golden):
    a = 1.3
    e = energy(3, np.eye(3) * a, 2.4, [[0, 0, 0], [a / 2, a / 2, a / 2]], [1.0, -1.0])
    assert e == pytest.approx(-golden["madelung_cscl"] / (SQ3 * a / 2), rel=1e-14)
    pos = np.array(FCC + [[x + .25, y + .25, z + .25] for x, y, z in FCC]) * a
    q = np.array([1.0] * 4 + [-1.0] * 4)
    e = energy(3, np.eye(3) * a, 3.0, pos, q)
    assert e == pytest.approx(-4 * golden["madelung_zincblende"] / (SQ3 * a / 4), rel=1e-14)


# ------------------------------------------------------------------ closed forms, 2D
def dirichlet_beta(s):
    return (mpmath.zeta(s, mpmath.mpf(1) / 4) - mpmath.zeta(s, mpmath.mpf(3) / 4)) / mpmath.mpf(4) ** s


def test_vm_square_2d_closed_form(golden):
    mpmath.mp.dps = 30
    closed = float(4 * mpmath.zeta(0.5) * dirichlet_beta(mpmath.mpf(1) / 2))
    assert closed == pytest.approx(golden["vm_L_square_2d"], rel=1e-15)
    for L, kappa in [(1.0, 2.0), (2.5, 1.1)]:
        cell = np.eye(2) * L
        g, r = ora.auto_cutoffs(2, cell, kappa)
        assert ora.v_m(2, cell, kappa, g, r) * L == pytest.approx(closed, rel=3e-15)


def test_wigner_crystals_2d(golden):
    assert wigner_E_rs(2, np.eye(2), [[0, 0]], 2.5) == pytest.approx(golden["wigner_square_E_rs"], rel=1e-14)
    hexc = np.array([[1.0, 0.0], [0.5, SQ3 / 2]])
    assert wigner_E_rs(2, hexc, [[0, 0]], 2.5) == pytest.approx(golden["wigner_triangular_E_rs"], rel=1e-14)
    rect = np.array([[1.0, 0.0], [0.0, SQ3]])
    assert wigner_E_rs(2, rect, [[0, 0], [.5, .5]], 2.2) == pytest.approx(
        golden["wigner_triangular_E_rs"], rel=1e-14)


def test_madelung_checkerboard_2d(golden):
    mpmath.mp.dps = 30
    M = float(4 * (mpmath.sqrt(2) - 1) * abs(mpmath.zeta(0.5)) * dirichlet_beta(mpmath.mpf(1) / 2))
    assert M == pytest.approx(golden["madelung_checkerboard"], rel=1e-15)
    # 2x2 cell, nearest-neighbour distance 1, 2 ion pairs: E = -2M
    pos = [[0, 0], [1, 0], [0, 1], [1, 1]]
    q = [1.0, -1.0, -1.0, 1.0]
    assert energy(2, np.eye(2) * 2, 1.4, pos, q) == pytest.approx(-2 * M, rel=1e-14)


# ------------------------------------------------------------------ "Ewald = periodic Coulomb": brute force
def direct_sum(cell, pos, q, ncell):
    """1/2 sum_{R in sphere} sum_{ij}' q_i q_j / |r_i - r_j - R| with whole cells inside a sphere."""
    cell = np.asarray(cell, float)
    dim = cell.shape[0]
    rng = np.arange(-ncell, ncell + 1)
    m = np.stack(np.meshgrid(*([rng] * dim), indexing="ij"), -1).reshape(-1, dim)
    R = m @ cell
    rad = ncell * min(np.linalg.norm(cell, axis=1)) * 0.999
    R = R[np.einsum("ij,ij->i", R, R) <= rad * rad]
    e = 0.0
    n = len(q)
    for i in range(n):
        for j in range(n):
            d = pos[i] - pos[j] - R
            r = np.sqrt(np.einsum("ij,ij->i", d, d))
            if i == j:
                r = r[r > 0]
            e += 0.5 * q[i] * q[j] * np.sum(1.0 / r)
    return e


def test_direct_sum_zero_dipole_3d():
    # quadrupole-like 4-charge cell: no dipole -> the plain spherical sum converges to Eqs. 2-4
    cell = np.diag([1.0, 1.1, 0.9])
    pos = np.array([[0.1, 0.1, 0.1], [0.6, 0.1, 0.1], [0.1, 0.65, 0.5], [0.6, 0.65, 0.5]])
    q = np.array([1.0, -1.0, -1.0, 1.0])
    dip = q @ pos
    assert np.allclose(dip, 0)
    ew = energy(3, cell, 2.5, pos, q)
    e1, e2 = direct_sum(cell, pos, q, 20), direct_sum(cell, pos, q, 40)
    assert abs(e2 - ew) < 2e-5 * abs(ew)
    assert abs(e2 - ew) < abs(e1 - ew) + 1e-9  # and it is converging towards it


def test_direct_sum_with_dipole_3d():
    # spherical summation order adds 2 pi |M|^2 / (3 Omega) to the tin-foil (Ewald) energy
    cell = np.eye(3)
    pos = np.array([[0.2, 0.3, 0.25], [0.55, 0.45, 0.6]])
    q = np.array([1.0, -1.0])
    M = q @ pos
    ew = energy(3, cell, 2.5, pos, q)
    e = direct_sum(cell, pos, q, 40)
    assert e == pytest.approx(ew + 2 * math.pi * (M @ M) / 3.0, abs=2e-5)


def test_direct_sum_2d():
    cell = np.array([[1.0, 0.0], [0.2, 1.1]])
    pos = np.array([[0.1, 0.1], [0.6, 0.2], [0.3, 0.7]])
    q = np.array([1.0, 1.0, -2.0])
    ew = energy(2, cell, 2.5, pos, q)
    # neutral 2D cell: dipole lattice sums converge absolutely (1/R^3 in the plane), no shape term
    e1, e2 = direct_sum(cell, pos, q, 200), direct_sum(cell, pos, q, 400)
    rich = e2 + (e2 - e1)  # error ~ 1/R
    assert rich == pytest.approx(ew, abs=5e-5)


# ------------------------------------------------------------------ splitting-parameter invariance
@pytest.mark.parametrize("dim,neutral", [(3, True), (3, False), (2, True), (2, False)])
def test_kappa_invariance(dim, neutral):
    rng = np.random.default_rng(7 + dim + neutral)
    cell = np.eye(dim) * 2.0 + 0.3 * rng.standard_normal((dim, dim))
    n = 7
    pos = rng.random((n, dim)) @ cell
    q = rng.choice([-1.0, 1.0, 2.0], size=n)
    if neutral:
        q[-1] -= q.sum()
    k0 = 2.2 / abs(np.linalg.det(cell)) ** (1 / dim)
    es = [energy(dim, cell, k0 * f, pos, q) for f in (0.7, 1.0, 1.3, 1.6)]
    assert np.ptp(es) < 1e-12 * abs(es[1])


# ------------------------------------------------------------------ O-pair (Eqs. 2-4 literal) vs O-rho
@pytest.mark.parametrize("dim", [2, 3])
def test_pairwise_vs_rho(dim):
    rng = np.random.default_rng(11 + dim)
    cell = np.eye(dim) * 1.5 + 0.2 * rng.standard_normal((dim, dim))
    n = 9
    pos = (rng.random((n, dim)) * 3 - 1) @ cell  # also outside the cell (reading R9)
    q = rng.standard_normal(n)
    kappa = 2.0
    g, r = 9.0, 2.6  # deliberately truncated cut-offs: the two forms must still agree term by term
    e_rho, comp = ora.energy_batch(dim, cell, kappa, g, r, pos[None], q)
    e_pair = ora.energy_pairwise(dim, cell, kappa, g, r, pos, q)
    assert e_pair == pytest.approx(e_rho[0], rel=1e-14, abs=1e-14)
    assert comp[0].sum() == pytest.approx(e_rho[0], rel=1e-15)


def test_v_e_periodic_and_even():
    cell = np.array([[1.0, 0.1, 0.0], [0.0, 1.2, 0.2], [0.1, 0.0, 0.9]])
    kappa = 2.5
    g, r = ora.auto_cutoffs(3, cell, kappa)
    x = np.array([0.3, -0.2, 0.45])
    v = ora.v_e(3, cell, kappa, g, r, x)
    assert ora.v_e(3, cell, kappa, g, r, -x) == pytest.approx(v, rel=1e-14)
    assert ora.v_e(3, cell, kappa, g, r, x + cell[0] - 2 * cell[2]) == pytest.approx(v, rel=1e-13)


# ------------------------------------------------------------------ rho(G)
def test_rho_closed_forms():
    L = 2.0
    cell = np.eye(3) * L
    gc = 2 * math.pi / L * 4.01
    nvec = ora.gplus(3, cell, gc)
    assert len(nvec) * 2 == ora.num_g(3, cell, gc)
    # first non-zero component positive, lexicographic order, all inside the sphere
    assert all((v[v != 0][0] > 0) for v in nvec)
    assert [tuple(v) for v in nvec] == sorted(tuple(v) for v in nvec)
    assert (np.sum(nvec.astype(int) ** 2, 1) <= 16).all()
    # one charge at the origin: rho(G) = q for every G
    rho = ora.rho(3, cell, gc, [[0, 0, 0]], [-1.5])
    assert np.allclose(rho, -1.5, atol=1e-15)
    # m^3 charges on the L/m sub-lattice: rho = N q if all n_k = 0 (mod m), else 0
    m = 2
    pts = np.array([[i, j, k] for i in range(m) for j in range(m) for k in range(m)]) * L / m
    rho = ora.rho(3, cell, gc, pts, np.full(len(pts), 0.5))
    on = np.all(nvec % m == 0, axis=1)
    assert np.allclose(rho[on], 0.5 * m ** 3, atol=1e-14)
    assert np.allclose(rho[~on], 0, atol=1e-14)


def test_rho_general_cell_against_numpy():
    rng = np.random.default_rng(5)
    cell = np.eye(3) + 0.2 * rng.standard_normal((3, 3))
    gc = 14.0
    nvec = ora.gplus(3, cell, gc)
    B = 2 * math.pi * np.linalg.inv(cell).T
    G = nvec @ B
    assert (np.einsum("ij,ij->i", G, G) <= gc * gc * (1 + 1e-12)).all()
    # count equals a brute-force count over a big box
    r = np.arange(-12, 13)
    allm = np.stack(np.meshgrid(r, r, r, indexing="ij"), -1).reshape(-1, 3)
    g2 = np.einsum("ij,ij->i", allm @ B, allm @ B)
    assert ((g2 <= gc * gc) & (g2 > 0)).sum() == 2 * len(nvec)
    pos = rng.random((6, 3)) @ cell
    q = rng.standard_normal(6)
    rho = ora.rho(3, cell, gc, pos, q)
    assert np.allclose(rho, (q * np.exp(1j * G @ pos.T)).sum(1), atol=1e-13)


# ------------------------------------------------------------------ invariances
def test_invariances_3d_and_2d():
    for dim in (2, 3):
        rng = np.random.default_rng(3 + dim)
        cell = np.eye(dim) * 1.8 + 0.25 * rng.standard_normal((dim, dim))
        n = 6
        pos = rng.random((n, dim)) @ cell
        q = rng.choice([-1.0, 2.0], size=n)
        kappa = 1.6
        e0 = energy(dim, cell, kappa, pos, q)
        # rigid translation, permutation
        assert energy(dim, cell, kappa, pos + rng.random(dim), q) == pytest.approx(e0, rel=1e-13)
        p = rng.permutation(n)
        assert energy(dim, cell, kappa, pos[p], q[p]) == pytest.approx(e0, rel=1e-14)
        # shifting one particle by a lattice vector
        pos2 = pos.copy()
        pos2[2] += 2 * cell[0] - cell[dim - 1]
        assert energy(dim, cell, kappa, pos2, q) == pytest.approx(e0, rel=1e-13)
        # E(lambda q) = lambda^2 E ; E(lambda r, lambda cell, kappa/lambda) = E/lambda
        assert energy(dim, cell, kappa, pos, 1.5 * q) == pytest.approx(2.25 * e0, rel=1e-14)
        assert energy(dim, 2.5 * cell, kappa / 2.5, 2.5 * pos, q) == pytest.approx(e0 / 2.5, rel=1e-13)
        # doubled cell holding 2^dim replicas has 2^dim times the energy
        shifts = np.array(np.meshgrid(*([[0, 1]] * dim), indexing="ij")).reshape(dim, -1).T @ cell
        big = np.concatenate([pos + s for s in shifts])
        e_big = energy(dim, 2 * cell, kappa, big, np.tile(q, 2 ** dim))
        assert e_big == pytest.approx(2 ** dim * e0, rel=1e-13)


def test_fixed_ions_are_just_charges():
    rng = np.random.default_rng(17)
    cell = np.eye(3) * 2.0
    pos = rng.random((2, 5, 3)) * 2
    q = -np.ones(5)
    ion_pos = rng.random((3, 3)) * 2
    ion_q = np.array([2.0, 2.0, 1.0])
    g, r = ora.auto_cutoffs(3, cell, 2.0, 1e-16)
    e_a, _ = ora.energy_batch(3, cell, 2.0, g, r, pos, q, ion_pos, ion_q)
    allpos = np.concatenate([pos, np.broadcast_to(ion_pos, (2, 3, 3))], axis=1)
    e_b, _ = ora.energy_batch(3, cell, 2.0, g, r, allpos, np.concatenate([q, ion_q]))
    assert np.allclose(e_a, e_b, rtol=1e-15)


# ------------------------------------------------------------------ single-particle moves
@pytest.mark.parametrize("dim", [2, 3])
def test_move_delta_vs_full_energies(dim):
    rng = np.random.default_rng(23 + dim)
    cell = np.eye(dim) * 2.0 + 0.1 * rng.standard_normal((dim, dim))
    nw, n, ns = 3, 8, 6
    pos = rng.random((nw, n, dim)) @ cell
    q = rng.choice([-1.0, 1.0], size=n)
    ion_pos = rng.random((2, dim)) @ cell
    ion_q = np.array([2.0, -1.0])
    kappa = 1.9
    g, r = ora.auto_cutoffs(dim, cell, kappa, 1e-16)
    electron = rng.integers(0, n, size=(ns, nw))
    cur = pos.copy()
    new_r = np.zeros((ns, nw, dim))
    e_prev, _ = ora.energy_batch(dim, cell, kappa, g, r, cur, q, ion_pos, ion_q)
    de_def = np.zeros((ns, nw))
    for s in range(ns):
        for w in range(nw):
            new_r[s, w] = cur[w, electron[s, w]] + 0.4 * rng.standard_normal(dim)
            cur[w, electron[s, w]] = new_r[s, w]
        e_now, _ = ora.energy_batch(dim, cell, kappa, g, r, cur, q, ion_pos, ion_q)
        de_def[s] = e_now - e_prev
        e_prev = e_now
    de, final, rho = ora.move_chain(dim, cell, kappa, g, r, pos, q, electron, new_r, ion_pos, ion_q,
                                    want_rho=True)
    scale = np.abs(e_prev).max()
    assert np.abs(de - de_def).max() < 1e-13 * scale
    assert np.array_equal(final, cur)
    # stored rho after the chain equals a fresh rho of the final configuration (ions included)
    for w in range(nw):
        fresh = ora.rho(dim, cell, g, np.concatenate([cur[w], ion_pos]), np.concatenate([q, ion_q]))
        assert np.allclose(rho[w], fresh, atol=1e-13)


def test_move_and_return_sums_to_zero():
    rng = np.random.default_rng(31)
    cell = np.eye(3) * 3.0
    pos = rng.random((2, 10, 3)) * 3
    q = -np.ones(10)
    kappa = 1.2
    g, r = ora.auto_cutoffs(3, cell, kappa, 1e-16)
    electron = np.array([[4, 7], [4, 7]])
    new_r = np.stack([pos[[0, 1], [4, 7]] + 0.5, pos[[0, 1], [4, 7]]])
    de, final, rho = ora.move_chain(3, cell, kappa, g, r, pos, q, electron, new_r, want_rho=True)
    assert np.abs(de.sum(0)).max() < 1e-14
    assert np.abs(de[0]).min() > 1e-4  # the move did change the energy
    assert np.allclose(rho[0], ora.rho(3, cell, g, pos[0], q), atol=1e-14)
