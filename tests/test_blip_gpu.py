"""GPU parity of the batched blip-orbital evaluation against the oracle
(oracle/blip_ref.c) through the C ABI of include/blip.h.  Tolerances: FP64 1e-11, FP32 2e-5, relative to the
largest |psi| (|grad|, |lap|) over the orbitals of a position (a single orbital can vanish at a point)."""
import numpy as np
import pytest

from oracle import blip_ref as br
from paper_2507_02888_b200 import blip as B
from paper_2507_02888_b200 import workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-11, "f32": 2e-5}


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _gpu_eval(torch, ctx, pts, dtype, derivs=True):
    npdt = np.float64 if dtype == "f64" else np.float32
    P = len(pts)
    npad = (P + 3) & ~3
    soa = np.zeros((3, npad), dtype=npdt)
    soa[:, :P] = pts.T
    d_pts = torch.from_numpy(soa).cuda()
    psi = torch.full((P, ctx.n_orb), float("nan"), dtype=torch.float64, device="cuda")
    grad = torch.zeros((P, 3, ctx.n_orb), dtype=torch.float64, device="cuda") if derivs else None
    lap = torch.zeros((P, ctx.n_orb), dtype=torch.float64, device="cuda") if derivs else None
    B.blip_eval_batch(ctx, P, d_pts, psi, grad, lap)
    torch.cuda.synchronize()
    return psi.cpu().numpy(), (grad.cpu().numpy() if derivs else None), (lap.cpu().numpy() if derivs else None)


def _assert(got, want, tol):
    for g, w in zip(got, want):
        assert np.all(np.isfinite(g))
        scale = np.abs(w).reshape(len(w), -1).max(axis=1)
        assert (np.abs(g - w).reshape(len(w), -1).max(axis=1) / scale).max() <= tol


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_blip_workload_matches_oracle(torch_cuda, dtype):
    """125 orbitals on a 24^3 grid at the 250 electron positions of 2 walkers of BASELINE configs[1]."""
    wl = workloads.BlipWorkload()
    pts = wl.points(2)
    if dtype == "f32":
        pts = pts.astype(np.float32).astype(np.float64)
    ctx = B.blip_setup(wl.cell, wl.coef)
    got = _gpu_eval(torch_cuda, ctx, pts, dtype)
    coef = wl.coef if dtype == "f64" else wl.coef.astype(np.float32).astype(np.float64)
    _assert(got, br.evaluate(wl.cell, coef, pts), TOL[dtype])


def test_blip_general_cell_ragged_orbitals_and_points(torch_cuda):
    """Triclinic cell, unequal grid, orbital counts that are not multiples of 32 (1, 33, 130: a second pass), points
    outside the cell and exactly on grid planes, value-only call."""
    rng = np.random.default_rng(4)
    cell = np.array([[5.0, 0.4, 0], [0.7, 6.0, 0.2], [0.3, -0.5, 4.5]])
    for n_orb, grid in ((1, (4, 5, 6)), (33, (7, 5, 9)), (130, (6, 6, 5))):
        coef = rng.standard_normal((n_orb,) + grid)
        pts = (rng.random((37, 3)) * 3 - 1) @ cell
        pts[:4] = (np.array([[0, 0, 0], [1, 2, 3], [2, 0, 4], [6, 4, 8]]) / np.array(grid)) @ cell   # on the knots
        ctx = B.blip_setup(cell, coef)
        want = br.evaluate(cell, coef, pts)
        got = _gpu_eval(torch_cuda, ctx, pts, "f64")
        assert np.abs(got[0] - want[0]).max() <= 1e-11 * np.abs(want[0]).max()
        assert np.abs(got[1] - want[1]).max() <= 1e-11 * np.abs(want[1]).max()
        # on a knot the third derivative jumps but the second does not: the Laplacian is well defined
        assert np.abs(got[2] - want[2]).max() <= 1e-11 * np.abs(want[2]).max()
        v_only = _gpu_eval(torch_cuda, ctx, pts, "f64", derivs=False)[0]
        assert np.array_equal(v_only, got[0])


def test_blip_full_batch_sampled(torch_cuda):
    """All 256 000 positions of the 1024 walkers in one launch (the shape bench.py times): 64 sampled positions."""
    wl = workloads.BlipWorkload()
    pts = wl.points()
    ctx = B.blip_setup(wl.cell, wl.coef)
    psi, grad, lap = _gpu_eval(torch_cuda, ctx, pts, "f64")
    sample = np.random.default_rng(9).choice(len(pts), 64, replace=False)
    want = br.evaluate(wl.cell, wl.coef, pts[sample])
    _assert((psi[sample], grad[sample], lap[sample]), want, TOL["f64"])
