"""Pins of the Jastrow oracle (oracle/jastrow_ref.c; Eqs. 6-7) against closed forms,
an independent numpy evaluation, finite differences and invariances.  No GPU."""
import math

import numpy as np

from oracle import jastrow_ref as jr
from paper_2507_02888_b200 import workloads

L = 7.3
CUBE = np.eye(3) * L


def test_u_closed_forms():
    # N_u = 0, alpha_0 = 1, C = 2: u = (r - L_u)^2
    for r in (0.3, 1.7, 2.9):
        u, du, d2u = jr.u([1.0], 3.0, 2, r)
        assert abs(u - (r - 3.0) ** 2) < 1e-15 and abs(du - 2 * (r - 3.0)) < 1e-15 and abs(d2u - 2.0) < 1e-15
    # alpha = (0, 1), C = 3: u = r (r - L)^3, u' = (r - L)^3 + 3 r (r - L)^2, u'' = 6 (r - L)^2 + 6 r (r - L)
    Lu = 2.5
    for r in (0.2, 1.1, 2.4):
        s = r - Lu
        u, du, d2u = jr.u([0.0, 1.0], Lu, 3, r)
        assert abs(u - r * s ** 3) < 1e-14 and abs(du - (s ** 3 + 3 * r * s * s)) < 1e-14
        assert abs(d2u - (6 * s * s + 6 * r * s)) < 1e-14
    # Theta(L_u - r): zero at and beyond the cut-off, and C - 1 continuous derivatives there
    assert jr.u([1.0, 0.5], Lu, 3, Lu) == (0.0, 0.0, 0.0) and jr.u([1.0, 0.5], Lu, 3, Lu + 0.1) == (0.0, 0.0, 0.0)
    u, du, d2u = jr.u([1.0, 0.5], Lu, 3, Lu - 1e-6)
    assert abs(u) < 1e-17 and abs(du) < 1e-11 and abs(d2u) < 2e-5      # (r - L_u)^3, 3 (r - L_u)^2, 6 (r - L_u) times 2.25


def test_p_one_star_two_particles_closed_form():
    # star of (1,0,0) in a cubic cell: p(r) = a [cos(2 pi x/L) + cos(2 pi y/L) + cos(2 pi z/L)]
    g_n = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1]])
    a = np.array([0.37])
    pos = np.array([[[0.4, 1.1, -0.3], [2.0, 0.2, 5.5]]])
    d = pos[0, 0] - pos[0, 1]
    k = 2 * math.pi / L
    val, grad, lap = jr.batch(3, CUBE, pos, g_n=g_n, star=[0, 0, 0], a=a)
    assert abs(val[0] - a[0] * np.cos(k * d).sum()) < 1e-15
    assert np.abs(grad[0, 0] + a[0] * k * np.sin(k * d)).max() < 1e-15       # grad_0 p(r_0 - r_1)
    assert np.abs(grad[0, 0] + grad[0, 1]).max() < 1e-15
    assert abs(lap[0, 0] + a[0] * k * k * np.cos(k * d).sum()) < 1e-15 and abs(lap[0, 1] - lap[0, 0]) < 1e-15


def _numpy_p_value(cell, pos, g_n, star, a):
    """sum_{i<j} cos(G.r_ij) = (|S(G)|^2 - N)/2 with S = sum_i exp(iG.r_i): an evaluation that shares nothing
    with the oracle's pair loop."""
    b = 2 * math.pi * np.linalg.inv(cell).T
    G = np.asarray(g_n, dtype=float)[:, :cell.shape[0]] @ b
    out = []
    for p in pos:
        S = np.exp(1j * (p @ G.T)).sum(axis=0)
        out.append((np.asarray(a)[star] * 0.5 * (np.abs(S) ** 2 - len(p))).sum())
    return np.array(out)


def test_p_value_matches_structure_factor_identity():
    j = workloads.JastrowWorkload(base_index=1, n_stars=15)
    assert j.n_stars == 15 and len(j.g_n) == 128
    pos = j.positions(3)
    val, _, _ = jr.batch(3, j.cell, pos, g_n=j.g_n, star=j.star, a=j.a)
    want = _numpy_p_value(j.cell, pos, j.g_n, j.star, j.a)
    assert np.abs(val - want).max() <= 1e-12 * np.abs(want).max()
    # 2D, non-orthogonal cell
    cell = np.array([[5.0, 0.0], [-2.0, 4.5]])
    rng = np.random.default_rng(3)
    pos = rng.random((2, 9, 2)) @ cell
    g_n = np.array([[1, 0, 0], [0, 1, 0], [1, 1, 0], [1, -1, 0], [2, 1, 0]])
    star, a = np.array([0, 0, 1, 2, 3]), np.array([0.3, -0.2, 0.1, 0.05])
    val, _, _ = jr.batch(2, cell, pos, g_n=g_n, star=star, a=a)
    assert np.abs(val - _numpy_p_value(cell, pos, g_n, star, a)).max() <= 1e-13


def test_gradient_and_laplacian_against_finite_differences():
    rng = np.random.default_rng(11)
    for dim, cell in ((3, CUBE), (2, np.array([[6.0, 0.0], [1.5, 5.0]]))):
        j = workloads.JastrowWorkload(base_index=1 if dim == 3 else 3, n_stars=6)
        g_n, star, a = j.g_n, j.star, j.a * 3
        alpha, Lu, C = np.array([0.3, -0.2, 0.05, 0.01]), 2.4, 3
        n = 7
        pos = (rng.random((1, n, dim)) @ cell) * 0.6     # crowded: several pairs inside L_u
        kw = dict(alpha=alpha, L_u=Lu, C=C, g_n=g_n, star=star, a=a)
        val, grad, lap = jr.batch(dim, cell, pos, **kw)
        assert np.abs(grad[0].sum(axis=0)).max() < 1e-13       # translation invariance
        h = 1e-4
        for i in (0, 3):
            second = 0.0
            for x in range(dim):
                pp, pm = pos.copy(), pos.copy()
                pp[0, i, x] += h
                pm[0, i, x] -= h
                vp, vm = jr.batch(dim, cell, pp, **kw)[0][0], jr.batch(dim, cell, pm, **kw)[0][0]
                assert abs((vp - vm) / (2 * h) - grad[0, i, x]) < 1e-6 * max(1.0, abs(grad[0, i, x]))
                second += (vp - 2 * val[0] + vm) / (h * h)
            assert abs(second - lap[0, i]) < 1e-5 * max(1.0, abs(lap[0, i]))


def test_periodicity_and_point_group():
    j = workloads.JastrowWorkload(base_index=1, n_stars=8)
    pos = j.positions(2)[:, :12]
    kw = dict(alpha=j.alpha, L_u=j.L_u, C=j.C, g_n=j.g_n, star=j.star, a=j.a)
    val, grad, lap = jr.batch(3, j.cell, pos, **kw)
    moved = pos.copy()
    moved[:, 5] += np.array([2, -1, 3]) @ j.cell               # a lattice vector: nothing changes
    v2, g2, l2 = jr.batch(3, j.cell, moved, **kw)
    assert np.abs(v2 - val).max() < 1e-12 * np.abs(val).max() and np.abs(g2 - grad).max() < 1e-12
    assert np.abs(l2 - lap).max() < 1e-11
    # full stars of a cubic cell are invariant under permutations and reflections of the axes
    perm = pos[:, :, [2, 0, 1]] * np.array([1.0, -1.0, 1.0])
    v3, _, _ = jr.batch(3, j.cell, perm, **kw)
    assert np.abs(v3 - val).max() < 1e-12 * np.abs(val).max()
    # p is even: J is unchanged by inversion of every position
    v4, g4, _ = jr.batch(3, j.cell, -pos, **kw)
    assert np.abs(v4 - val).max() < 1e-12 * np.abs(val).max() and np.abs(g4 + grad).max() < 1e-12


def test_u_minimum_image_in_a_skewed_cell():
    cell = np.array([[4.0, 0.0], [3.0, 3.5]])      # the fractionally rounded image is not always the nearest
    alpha, Lu, C = np.array([1.0, 0.3]), 1.7, 2
    rng = np.random.default_rng(5)
    pos = rng.random((1, 6, 2)) @ cell
    val, _, _ = jr.batch(2, cell, pos, alpha=alpha, L_u=Lu, C=C)
    want = 0.0
    for i in range(6):
        for k in range(i + 1, 6):
            d = pos[0, i] - pos[0, k]
            r = min(np.linalg.norm(d - m0 * cell[0] - m1 * cell[1]) for m0 in range(-3, 4) for m1 in range(-3, 4))
            if r < Lu:
                want += (alpha[0] + alpha[1] * r) * (r - Lu) ** C
    assert abs(val[0] - want) < 1e-13


def test_move_chain_equals_difference_of_values():
    j = workloads.JastrowWorkload(base_index=1, n_stars=5)
    rng = np.random.default_rng(8)
    pos = j.positions(3)[:, :20]
    kw = dict(alpha=j.alpha, L_u=j.L_u, C=j.C, g_n=j.g_n, star=j.star, a=j.a)
    S = 4
    electron = rng.integers(0, 20, (S, 3)).astype(np.int32)
    new_r = rng.random((S, 3, 3)) * j.L
    delta, final = jr.move_chain(3, j.cell, pos, electron, new_r, **kw)
    cur = pos.copy()
    for s in range(S):
        before = jr.batch(3, j.cell, cur, **kw)[0]
        cur[np.arange(3), electron[s]] = new_r[s]
        after = jr.batch(3, j.cell, cur, **kw)[0]
        assert np.abs(delta[s] - (after - before)).max() < 1e-11 * np.abs(after).max()
    assert np.array_equal(final, cur)
