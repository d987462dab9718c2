"""GPU parity of the batched Jastrow u and p terms against the oracle
(oracle/jastrow_ref.c), element by element through the C ABI of include/jastrow.h.  Tolerances: FP64 1e-11,
FP32 2e-5, relative to the walker's J for the value and to the largest |grad_i| (|lap_i|) of the walker for the
per-particle derivatives (a single component can vanish); Delta J per reading R12."""
import numpy as np
import pytest

from oracle import jastrow_ref as jr
from paper_2507_02888_b200 import ewald as E
from paper_2507_02888_b200 import jastrow as J
from paper_2507_02888_b200 import workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-11, "f32": 2e-5}


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _gpu_batch(torch, ctx, pos, dtype, derivs=True):
    npdt = np.float64 if dtype == "f64" else np.float32
    W, n, dim = pos.shape
    npad = E.ewald_padded_n(n)
    d_pos = torch.from_numpy(E.to_soa(pos, npdt)).cuda()
    val = torch.full((W,), float("nan"), dtype=torch.float64, device="cuda")
    grad = torch.zeros((W, dim, npad), dtype=torch.float64, device="cuda") if derivs else None
    lap = torch.zeros((W, npad), dtype=torch.float64, device="cuda") if derivs else None
    J.jastrow_batch(ctx, n, d_pos, val, grad, lap)
    torch.cuda.synchronize()
    if not derivs:
        return val.cpu().numpy(), None, None
    return val.cpu().numpy(), grad.cpu().numpy()[:, :, :n].transpose(0, 2, 1), lap.cpu().numpy()[:, :n]


def _assert_batch(got, want, tol):
    v, g, l = got
    vr, gr, lr = want
    assert np.all(np.isfinite(v))
    assert (np.abs(v - vr) / np.abs(vr)).max() <= tol
    assert (np.abs(g - gr).max(axis=(1, 2)) / np.abs(gr).max(axis=(1, 2))).max() <= tol
    assert (np.abs(l - lr).max(axis=1) / np.abs(lr).max(axis=1)).max() <= tol


def _r(a, dtype):
    return a if dtype == "f64" else a.astype(np.float32).astype(np.float64)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("terms", ["p", "u", "up"])
def test_jastrow_heg_n250_matches_oracle(torch_cuda, dtype, terms):
    """3D HEG N = 250 (BASELINE configs[1]'s cell), N_p = 15 stars (128 G vectors), N_u = 8, C = 3: value, gradient
    and Laplacian of 4 walkers."""
    j = workloads.JastrowWorkload(base_index=2, n_stars=15)
    kw = {}
    if "p" in terms:
        kw.update(g_n=j.g_n, star=j.star, a=j.a)
    if "u" in terms:
        kw.update(alpha=j.alpha, C=j.C)
    pos = _r(j.positions(4), dtype)
    want = jr.batch(3, j.cell, pos, L_u=j.L_u if "u" in terms else 0.0, **kw)
    if "C" in kw:
        kw["c_exp"] = kw.pop("C")
    ctx = J.jastrow_setup(3, j.cell, l_u=j.L_u if "u" in terms else 0.0, **kw)
    _assert_batch(_gpu_batch(torch_cuda, ctx, pos, dtype), want, TOL[dtype])


def test_jastrow_full_batch_sampled_and_value_only(torch_cuda):
    """All 1024 walkers of the workload in one launch (the shape bench.py times); the oracle checks 6 of them;
    value-only call gives the same values."""
    j = workloads.JastrowWorkload(base_index=2, n_stars=15)
    pos = j.positions()
    ctx = J.jastrow_setup(3, j.cell, alpha=j.alpha, l_u=j.L_u, c_exp=j.C, g_n=j.g_n, star=j.star, a=j.a)
    v, g, l = _gpu_batch(torch_cuda, ctx, pos, "f64")
    sample = np.array([0, 1, 377, 512, 1000, 1023])
    want = jr.batch(3, j.cell, pos[sample], j.alpha, j.L_u, j.C, j.g_n, j.star, j.a)
    _assert_batch((v[sample], g[sample], l[sample]), want, TOL["f64"])
    v2, _, _ = _gpu_batch(torch_cuda, ctx, pos, "f64", derivs=False)
    assert np.array_equal(v, v2)


@pytest.mark.parametrize("dim", [2, 3])
def test_jastrow_general_cells_and_ragged_sizes(torch_cuda, dim):
    """Non-orthogonal cells (minimum image of u among the neighbours of the rounded image), N = 1, 2, 5, 33, 70
    (fewer particles than a chunk, a ragged last chunk), positions outside the cell."""
    rng = np.random.default_rng(60 + dim)
    cell = np.array([[5.0, 0, 0], [1.5, 4.0, 0], [0.3, 0.2, 6.0]]) if dim == 3 else np.array([[5.0, 0.0], [-2.0, 4.5]])
    g_n = np.array([[1, 0, 0], [0, 1, 0], [1, 1, 0], [1, -1, 0], [2, -1, 0], [0, 0, 1], [1, 0, -2], [3, 1, 1]])
    if dim == 2:
        g_n = g_n[:5]
    star = np.arange(len(g_n)) % 3
    a = np.array([0.2, -0.1, 0.05])
    alpha, Lu, C = np.array([0.5, -0.3, 0.1, 0.02]), 1.9, 2
    ctx = J.jastrow_setup(dim, cell, alpha=alpha, l_u=Lu, c_exp=C, g_n=g_n, star=star, a=a)
    for n in (1, 2, 5, 33, 70):
        pos = (rng.random((3, n, dim)) * 1.6 - 0.3) @ cell
        want = jr.batch(dim, cell, pos, alpha, Lu, C, g_n, star, a)
        v, g, l = _gpu_batch(torch_cuda, ctx, pos, "f64")
        scale = max(np.abs(want[0]).max(), 1e-3)
        assert np.abs(v - want[0]).max() <= 1e-11 * scale
        assert np.abs(g - want[1]).max() <= 1e-11 * max(np.abs(want[1]).max(), 1.0)
        assert np.abs(l - want[2]).max() <= 1e-11 * max(np.abs(want[2]).max(), 1.0)
    with pytest.raises(E.EwaldError):       # L_u must stay below half the shortest lattice vector
        J.jastrow_setup(dim, cell, alpha=alpha, l_u=2.6, c_exp=C)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_jastrow_move_chain_matches_oracle(torch_cuda, dtype):
    """Stored S(G) and positions: 12 committed single-particle moves on 6 walkers, then an uncommitted proposal;
    Delta J per reading R12; the stored state equals a fresh evaluation of the final configuration."""
    torch = torch_cuda
    j = workloads.JastrowWorkload(base_index=2, n_stars=15)
    rng = np.random.default_rng(21)
    W, S, n = 6, 12, j.n
    npdt, tdt = (np.float64, torch.float64) if dtype == "f64" else (np.float32, torch.float32)
    pos = _r(j.positions(W), dtype)
    electron = rng.integers(0, n, (S, W)).astype(np.int32)
    cur = pos.copy()
    new_r = np.zeros((S, W, 3))
    for s in range(S):
        new_r[s] = _r(cur[np.arange(W), electron[s]] + 0.3 * rng.standard_normal((W, 3)), dtype)
        cur[np.arange(W), electron[s]] = new_r[s]
    d_ref, final = jr.move_chain(3, j.cell, pos, electron, new_r, j.alpha, j.L_u, j.C, j.g_n, j.star, j.a)
    ctx = J.jastrow_setup(3, j.cell, alpha=j.alpha, l_u=j.L_u, c_exp=j.C, g_n=j.g_n, star=j.star, a=j.a)
    J.jastrow_load_walkers(ctx, n, torch.from_numpy(E.to_soa(pos, npdt)).cuda())
    d_w = torch.arange(W, dtype=torch.int32, device="cuda")
    got = np.zeros((S, W))
    for s in range(S):
        d_de = torch.zeros(W, dtype=torch.float64, device="cuda")
        d_r = torch.from_numpy(new_r[s].astype(npdt)).cuda()
        if s == 3:   # a rejected proposal first: no change of the stored state
            trial = torch.zeros(W, dtype=torch.float64, device="cuda")
            J.jastrow_move_delta_batch(ctx, d_w, torch.from_numpy(electron[s]).cuda(), d_r, 0, trial)
        J.jastrow_move_delta_batch(ctx, d_w, torch.from_numpy(electron[s]).cuda(), d_r, 1, d_de)
        if s == 3:
            assert torch.equal(trial, d_de)
        got[s] = d_de.cpu().numpy()
    rms = np.sqrt((d_ref ** 2).mean(axis=1, keepdims=True))
    assert (np.abs(got - d_ref) / np.maximum(np.abs(d_ref), rms)).max() <= TOL[dtype]
    # one more move of every walker from the stored state must agree with the oracle continuing from `final`
    el = rng.integers(0, n, (1, W)).astype(np.int32)
    nr = _r(final[np.arange(W), el[0]] + 0.2 * rng.standard_normal((W, 3)), dtype)[None]
    d2, _ = jr.move_chain(3, j.cell, final, el, nr, j.alpha, j.L_u, j.C, j.g_n, j.star, j.a)
    d_de = torch.zeros(W, dtype=torch.float64, device="cuda")
    J.jastrow_move_delta_batch(ctx, d_w, torch.from_numpy(el[0]).cuda(), torch.from_numpy(nr[0].astype(npdt)).cuda(), 0, d_de)
    rms2 = np.sqrt((d2 ** 2).mean())
    assert (np.abs(d_de.cpu().numpy() - d2[0]) / np.maximum(np.abs(d2[0]), rms2)).max() <= 4 * TOL[dtype]
    bad = torch.zeros(2, dtype=torch.float64, device="cuda")
    J.jastrow_move_delta_batch(ctx, torch.tensor([0, 99], dtype=torch.int32, device="cuda"),
                               torch.tensor([1, 1], dtype=torch.int32, device="cuda"),
                               torch.zeros((2, 3), dtype=tdt, device="cuda"), 0, bad)
    out = bad.cpu().numpy()
    assert np.isfinite(out[0]) and np.isnan(out[1])
