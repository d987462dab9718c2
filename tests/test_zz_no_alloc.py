"""ewald_recip_energy_static (include/ewald.h): the allocation-free entry point.  Its kernel's scratch lives in a
file-scope device array of the library (EWALD_STATIC_SCRATCH_BYTES) instead of a buffer the context allocates, so
callers that cannot call cudaMalloc can use it.  Checked here against the existing path (components[:, 0] of
ewald_energy_batch) on two calls in a row, within the tolerances of tests/test_gpu_parity.py (1e-11 relative FP64,
2e-5 FP32), and bit for bit against the same kernel reached through ewald_set_recip_variant(ctx, 1).

The file name sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide other tests.
Nothing here depends on what ran before: every context is set up inside the test."""
import numpy as np
import pytest

from oracle import ewald_ref as ref
from paper_2507_02888_b200 import ewald as E
from paper_2507_02888_b200 import workloads

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-11, 2e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _ctx(w):
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)
    if w.ion_pos is not None:
        E.ewald_set_fixed_charges(ctx, w.ion_pos, w.ion_q)
    return ctx


def _device_inputs(torch, w, pos, dtype):
    npdt = np.float64 if dtype == "f64" else np.float32
    d_pos = torch.from_numpy(E.to_soa(pos, npdt)).cuda()
    d_q = torch.from_numpy(np.asarray(w.charges, dtype=npdt)).cuda()
    return d_pos, d_q


def _existing_recip(torch, ctx, w, d_pos, d_q):
    W = d_pos.shape[0]
    d_e = torch.full((W,), float("nan"), dtype=torch.float64, device="cuda")
    d_c = torch.full((W, 4), float("nan"), dtype=torch.float64, device="cuda")
    E.ewald_energy_batch(ctx, w.n, d_pos, d_q, d_e, d_c)
    torch.cuda.synchronize()
    return d_c.cpu().numpy()[:, 0]


def _static_recip(torch, ctx, w, d_pos, d_q):
    d_out = torch.full((d_pos.shape[0],), float("nan"), dtype=torch.float64, device="cuda")
    E.ewald_recip_energy_static(ctx, w.n, d_pos, d_q, d_out)
    torch.cuda.synchronize()
    return d_out.cpu().numpy()


@pytest.mark.parametrize("index,n_walkers,dtype", [(2, 96, "f64"), (2, 96, "f32"), (3, 40, "f64"), (4, 48, "f64"),
                                                    (6, 6, "f64")])
def test_static_entry_point_matches_existing_path_twice(torch_cuda, index, n_walkers, dtype):
    """Two calls in a row on DIFFERENT batches (the second smaller, so that leftovers of the first call sit in the
    shared array beyond and inside the part the second uses), each against the existing path.  Config 6 has 13
    slabs of G-vectors per walker and two ion species, config 4 fixed charges, config 3 is 2D."""
    torch = torch_cuda
    w = workloads.config(index)
    tol = TOL64 if dtype == "f64" else TOL32
    pos = w.positions(n_walkers)
    batches = [pos, pos[::-1][: max(1, n_walkers // 3)].copy()]
    ctx = _ctx(w)
    got, inputs = [], []
    for p in batches:                      # the two static calls back to back, nothing in between
        d_pos, d_q = _device_inputs(torch, w, p, dtype)
        inputs.append((d_pos, d_q))
        got.append(_static_recip(torch, ctx, w, d_pos, d_q))
    for g, (d_pos, d_q) in zip(got, inputs):
        want = _existing_recip(torch, ctx, w, d_pos, d_q)
        assert np.isfinite(g).all() and np.isfinite(want).all()
        assert np.max(np.abs(g - want) / np.abs(want)) <= tol
    # the same kernel through the existing path: bit for bit
    E.ewald_set_recip_variant(ctx, 1)
    for g, (d_pos, d_q) in zip(got, inputs):
        assert np.array_equal(g, _existing_recip(torch, ctx, w, d_pos, d_q))
    # a second context on the same device shares the array and gives the same values
    ctx2 = _ctx(w)
    assert np.array_equal(got[0], _static_recip(torch, ctx2, w, *inputs[0]))


def test_static_entry_point_matches_oracle(torch_cuda):
    torch = torch_cuda
    w = workloads.config(1)
    pos = w.positions()
    ctx = _ctx(w)
    d_pos, d_q = _device_inputs(torch, w, pos, "f64")
    got = _static_recip(torch, ctx, w, d_pos, d_q)
    _, c_ref = ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges, w.ion_pos, w.ion_q)
    assert np.max(np.abs(got - c_ref[:, 0]) / np.abs(c_ref[:, 0])) <= TOL64


def test_static_entry_point_rejects_sizes_beyond_the_array(torch_cuda):
    """One partial sum per walker and slab: config 1 has one slab, so 131072 walkers fit and 131073 do not.  The
    refused call launches nothing (the output keeps its NaNs) and says why."""
    torch = torch_cuda
    w = workloads.config(1)
    ctx = _ctx(w)
    limit = E.EWALD_STATIC_SCRATCH_BYTES // 8
    n_pad = E.ewald_padded_n(w.n)
    d_q = torch.from_numpy(np.asarray(w.charges, dtype=np.float32)).cuda()
    d_pos = torch.rand((limit + 1, w.dim, n_pad), dtype=torch.float32, device="cuda") * float(w.L)
    d_out = torch.full((limit + 1,), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(E.EwaldError) as err:
        E.ewald_recip_energy_static(ctx, w.n, d_pos, d_q, d_out)
    torch.cuda.synchronize()
    assert "EWALD_ERANGE" in str(err.value) and "static scratch" in str(err.value)
    assert torch.isnan(d_out).all()
    # exactly at the limit it runs, and agrees with the existing path on a sample of walkers
    d_out2 = torch.full((limit,), float("nan"), dtype=torch.float64, device="cuda")
    E.ewald_recip_energy_static(ctx, w.n, d_pos[:limit], d_q, d_out2)
    torch.cuda.synchronize()
    assert torch.isfinite(d_out2).all()
    pick = torch.tensor([0, 1, limit // 2, limit - 1], device="cuda")
    sample = d_pos[pick].contiguous()
    want = _existing_recip(torch, ctx, w, sample, d_q)
    got = d_out2[pick].cpu().numpy()
    assert np.max(np.abs(got - want) / np.abs(want)) <= TOL32
