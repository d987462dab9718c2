"""Pins of the blip-orbital oracle (oracle/blip_ref.c, reading R21) against the closed forms of
the cubic B-spline, polynomial reproduction, an independent numpy evaluation and finite differences.  No GPU."""
import numpy as np

from oracle import blip_ref as br


def test_theta_values_and_continuity():
    assert br.theta(0.0) == (1.0, 0.0, -3.0)
    f, d1, d2 = br.theta(1.0)
    assert abs(f - 0.25) < 1e-16 and abs(d1 + 0.75) < 1e-16 and abs(d2 - 1.5) < 1e-16
    assert br.theta(2.0) == (0.0, 0.0, 0.0) and br.theta(-2.5) == (0.0, 0.0, 0.0)
    for x in (0.3, 0.999999, 1.000001, 1.7):       # even, C2 across |x| = 1
        assert br.theta(-x)[0] == br.theta(x)[0] and br.theta(-x)[1] == -br.theta(x)[1]
    a, b = br.theta(1 - 1e-9), br.theta(1 + 1e-9)
    assert all(abs(p - q) < 1e-8 for p, q in zip(a, b))
    # Theta = 3/2 x the cardinal cubic B-spline (Theta(0) = 1): sum_i Theta(x - i) = 3/2, sum_i i Theta = 3/2 x,
    # sum_i i^2 Theta = 3/2 (x^2 + 1/3)
    for x in (0.0, 0.37, 0.5, 0.91):
        i = np.arange(-3, 5)
        th = np.array([br.theta(x - k)[0] for k in i])
        assert abs(th.sum() - 1.5) < 1e-15 and abs((i * th).sum() - 1.5 * x) < 1e-15
        assert abs((i * i * th).sum() - 1.5 * (x * x + 1.0 / 3.0)) < 1e-14


def test_constant_and_linear_coefficients():
    cell = np.array([[6.0, 0, 0], [1.0, 5.0, 0], [0.5, -0.3, 7.0]])
    N = (8, 6, 10)
    rng = np.random.default_rng(1)
    pts = (rng.random((5, 3)) * 2 - 0.5) @ cell
    coef = np.ones((1,) + N)
    psi, grad, lap = br.evaluate(cell, coef, pts)
    assert np.abs(psi - 3.375).max() < 1e-14 and np.abs(grad).max() < 1e-13 and np.abs(lap).max() < 1e-12   # (3/2)^3
    # c = grid index along axis 1 -> psi = (3/2)^3 u1, u1 = N1 s1, away from the periodic seam: gradient =
    # (3/2)^3 N1 times column 1 of the inverse cell, Laplacian 0
    coef = np.broadcast_to(np.arange(N[0], dtype=float)[:, None, None], N)[None].copy()
    frac = np.column_stack([rng.uniform(0.3, 0.7, 4), rng.random(4), rng.random(4)])
    pts = frac @ cell
    psi, grad, lap = br.evaluate(cell, coef, pts)
    binv = np.linalg.inv(cell)            # s = r @ inv(cell): d s_1 / d r_x = inv(cell)[x, 0]
    assert np.abs(psi[:, 0] - 3.375 * N[0] * frac[:, 0]).max() < 1e-13
    assert np.abs(grad[:, :, 0] - 3.375 * N[0] * binv[:, 0]).max() < 1e-13 and np.abs(lap).max() < 1e-11


def _numpy_eval(cell, coef, pts):
    """The 4 x 4 x 4 neighbourhood form in numpy with the textbook piecewise cubic -- a different route from the
    oracle's loop over every grid point."""
    def th(x):
        ax = np.abs(x)
        return np.where(ax <= 1, 1 - 1.5 * ax ** 2 + 0.75 * ax ** 3, np.where(ax < 2, 0.25 * (2 - ax) ** 3, 0.0))
    n_orb, N = coef.shape[0], np.array(coef.shape[1:])
    s = pts @ np.linalg.inv(cell)
    u = (s - np.floor(s)) * N
    out = np.zeros((len(pts), n_orb))
    for p in range(len(pts)):
        i0 = np.floor(u[p]).astype(int)
        for a in range(-1, 3):
            for b in range(-1, 3):
                for c in range(-1, 3):
                    w = th(u[p, 0] - (i0[0] + a)) * th(u[p, 1] - (i0[1] + b)) * th(u[p, 2] - (i0[2] + c))
                    out[p] += w * coef[:, (i0[0] + a) % N[0], (i0[1] + b) % N[1], (i0[2] + c) % N[2]]
    return out


def test_random_coefficients_numpy_and_finite_differences():
    rng = np.random.default_rng(2)
    cell = np.array([[5.0, 0.4, 0], [0, 6.0, 0.2], [0.3, 0, 4.5]])
    coef = rng.standard_normal((3, 7, 5, 6))
    pts = (rng.random((6, 3)) * 3 - 1) @ cell
    psi, grad, lap = br.evaluate(cell, coef, pts)
    assert np.abs(psi - _numpy_eval(cell, coef, pts)).max() < 1e-13
    moved = pts + np.array([2, -1, 1]) @ cell      # periodic with the cell
    assert np.abs(br.evaluate(cell, coef, moved)[0] - psi).max() < 1e-12
    h = 1e-4
    second = np.zeros_like(lap)
    for x in range(3):
        e = np.zeros(3); e[x] = h
        pp, pm = br.evaluate(cell, coef, pts + e)[0], br.evaluate(cell, coef, pts - e)[0]
        assert np.abs((pp - pm) / (2 * h) - grad[:, x, :]).max() < 1e-6
        second += (pp - 2 * psi + pm) / (h * h)
    assert np.abs(second - lap).max() < 2e-4       # Theta''' jumps at the knots: second differences are O(h) there
