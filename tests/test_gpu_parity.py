"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs (paper_2507_02888_b200.workloads).  Tolerances are BASELINE.json's: 1e-11 relative
per walker (FP64), 2e-5 (FP32); Delta E per reading R12: tol * max(|dE|, rms dE of the step).

FP32 (reading R16): the FP32 entry points take float32 positions, so the caller rounds the seeded
FP64 positions.  Two comparisons are made and both are reported:
  * against the oracle on exactly the rounded values (representable in FP64): both sides see the same inputs;
    this isolates the kernels' own FP32 arithmetic and is asserted at 2e-5 everywhere;
  * against the oracle on the UNROUNDED seeded inputs (SURVEY reading 16): measured per config by
    test_fp32_against_oracle_on_unrounded_inputs, printed, and asserted against the bound DESIGN.md R16 states
    for each config (the rounding of a close pair's coordinates to 2^-24 L dominates it, not the kernels).
"""
import math

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


def _ctx(w, **kw):
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, **kw)
    if w.ion_pos is not None:
        E.ewald_set_fixed_charges(ctx, w.ion_pos, w.ion_q)
    return ctx


def _gpu_energy(torch, ctx, pos, q, dtype, components=True):
    npdt = np.float64 if dtype == "f64" else np.float32
    W, n, _ = pos.shape
    d_pos = torch.from_numpy(E.to_soa(pos, npdt)).cuda()
    d_q = torch.from_numpy(np.asarray(q, dtype=npdt)).cuda()
    d_e = torch.full((W,), float("nan"), dtype=torch.float64, device="cuda")
    d_c = torch.full((W, 4), float("nan"), dtype=torch.float64, device="cuda") if components else None
    E.ewald_energy_batch(ctx, n, d_pos, d_q, d_e, d_c)
    torch.cuda.synchronize()
    return d_e.cpu().numpy(), (d_c.cpu().numpy() if components else None)


def _r32(a):
    """Values the FP32 path actually receives, as float64."""
    return np.asarray(a).astype(np.float32).astype(np.float64)


def _oracle_energy(w, pos):
    return ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges,
                            w.ion_pos, w.ion_q)


def _assert_energy(e, c, e_ref, c_ref, tol):
    assert np.all(np.isfinite(e))
    rel = np.abs(e - e_ref) / np.abs(e_ref)
    assert rel.max() <= tol, "max relative energy error %.3e > %.1e" % (rel.max(), tol)
    if c is not None:
        scale = np.maximum(np.abs(c_ref), np.abs(e_ref)[:, None])
        assert (np.abs(c - c_ref) / scale).max() <= tol
        assert np.allclose(c.sum(axis=1), e, rtol=1e-13, atol=0)


# walkers per config for the element-by-element comparison (oracle: seconds on 8 cores)
N_WALKERS = {1: 8, 2: 12, 3: 12, 4: 6}


@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_energy_fp64_matches_oracle(torch_cuda, idx):
    w = workloads.config(idx)
    pos = w.positions(N_WALKERS[idx])
    e_ref, c_ref = _oracle_energy(w, pos)
    ctx = _ctx(w)
    e, c = _gpu_energy(torch_cuda, ctx, pos, w.charges, "f64")
    _assert_energy(e, c, e_ref, c_ref, TOL64)
    assert E.ewald_num_g(ctx) == ref.num_g(w.dim, w.cell, w.g_cutoff)


@pytest.mark.parametrize("idx", [1, 2, 4])
def test_both_real_space_variants_match_oracle(torch_cuda, idx):
    """FP64 real-space kernel with the far shell (kappa^2 r^2 >= 16) in FP32 (default) and with every
    term in FP64: both within the FP64 tolerance of the oracle, and within 1e-13 of E_real of each other
    (the bound DESIGN.md section 5.2 derives for the far shell is 1e-14 of E_real)."""
    w = workloads.config(idx)
    pos = w.positions(N_WALKERS[idx])
    e_ref, c_ref = _oracle_energy(w, pos)
    ctx = _ctx(w)
    got = {}
    for variant in (0, 1):
        E.ewald_set_real_variant(ctx, variant)
        e, c = _gpu_energy(torch_cuda, ctx, pos, w.charges, "f64")
        _assert_energy(e, c, e_ref, c_ref, TOL64)
        got[variant] = c[:, 1]
    assert (np.abs(got[0] - got[1]) / np.abs(c_ref[:, 1])).max() <= 1e-13


@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_both_reciprocal_kernels_match_oracle(torch_cuda, idx):
    """Octant real-product form on the FMA pipe (variant 2) and on the FP64 tensor cores (variant 3; FP32 has no
    such form and takes the FMA-pipe kernel) and complex half-set form (variant 1), FP64 and FP32, on walker
    counts that leave the last CTA partly empty."""
    w = workloads.config(idx)
    nw = {1: 8, 2: 9, 3: 11, 4: 5}[idx]
    pos = w.positions(nw)
    e_ref, c_ref = _oracle_energy(w, pos)
    e32_ref, c32_ref = _oracle_energy(w, _r32(pos))
    ctx = _ctx(w)
    for variant in (1, 2, 3):
        E.ewald_set_recip_variant(ctx, variant)
        e, c = _gpu_energy(torch_cuda, ctx, pos, w.charges, "f64")
        _assert_energy(e, c, e_ref, c_ref, TOL64)
        assert (np.abs(c[:, 0] - c_ref[:, 0]) / np.abs(c_ref[:, 0])).max() <= 1e-12  # E_recip itself
        e, c = _gpu_energy(torch_cuda, ctx, _r32(pos), w.charges, "f32")
        assert (np.abs(e - e32_ref) / np.abs(e32_ref)).max() <= TOL32
        assert (np.abs(c[:, 0] - c32_ref[:, 0]) / np.abs(c32_ref[:, 0])).max() <= TOL32
    with pytest.raises(E.EwaldError):
        E.ewald_set_recip_variant(ctx, 4)


def test_octant_kernel_orthorhombic_cells_and_single_walker(torch_cuda):
    rng = np.random.default_rng(77)
    for dim in (2, 3):
        cell = np.diag([5.0, 6.5, 4.2][:dim])
        kappa = 1.1
        gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
        for n, nw in ((1, 1), (3, 2), (37, 17)):
            pos = rng.random((nw, n, dim)) @ cell
            q = rng.choice([-1.0, 2.0], size=n)
            e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, pos, q)
            ctx = E.ewald_setup(dim, cell, kappa, gc, rc)
            for variant in (2, 3):
                E.ewald_set_recip_variant(ctx, variant)
                e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
                assert (np.abs(c[:, 0] - c_ref[:, 0]) / np.abs(c_ref[:, 0])).max() <= 1e-12
                _assert_energy(e, c, e_ref, c_ref, TOL64)


@pytest.mark.parametrize("dim", [2, 3])
def test_octant_kernel_on_general_cells(torch_cuda, dim):
    """Non-orthogonal cells: the octant kernel (class weights per sign choice) and the complex half-set kernel
    both match the oracle, mixed charges and fixed ions included."""
    rng = np.random.default_rng(40 + dim)
    cell = (np.array([[5.0, 0, 0], [1.5, 4.0, 0], [0.3, 0.2, 6.0]]) if dim == 3 else np.array([[5.0, 0.0], [-2.0, 4.5]]))
    kappa = 0.95
    gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
    n = 23
    q = rng.choice([-1.0, 1.0, 2.0], size=n)
    pos = (rng.random((5, n, dim)) * 1.4 - 0.2) @ cell
    ion_pos = rng.random((3, dim)) @ cell
    ion_q = np.array([2.0, -1.0, 0.5])
    e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, pos, q, ion_pos, ion_q)
    ctx = E.ewald_setup(dim, cell, kappa, gc, rc)
    E.ewald_set_fixed_charges(ctx, ion_pos, ion_q)
    scale = np.abs(c_ref).max(axis=1)
    for variant in (3, 2, 1, 0):
        E.ewald_set_recip_variant(ctx, variant)
        e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
        assert (np.abs(c - c_ref) / scale[:, None]).max() <= TOL64, variant


@pytest.mark.parametrize("idx", [2, 3])
def test_energy_fp32_matches_oracle(torch_cuda, idx):
    w = workloads.config(idx)
    pos = _r32(w.positions(N_WALKERS[idx]))
    e_ref, c_ref = _oracle_energy(w, pos)
    ctx = _ctx(w)
    e, c = _gpu_energy(torch_cuda, ctx, pos, w.charges, "f32")
    _assert_energy(e, None, e_ref, None, TOL32)
    scale = np.maximum(np.abs(c_ref), np.abs(e_ref)[:, None])
    assert (np.abs(c - c_ref) / scale).max() <= TOL32


def test_fp32_also_passes_on_configs_1_and_4(torch_cuda):
    for idx in (1, 4):
        w = workloads.config(idx)
        pos = _r32(w.positions(4))
        e_ref, _ = _oracle_energy(w, pos)
        e, _ = _gpu_energy(torch_cuda, _ctx(w), pos, w.charges, "f32", components=False)
        assert (np.abs(e - e_ref) / np.abs(e_ref)).max() <= TOL32


def test_g_list_and_rho_match_oracle(torch_cuda):
    torch = torch_cuda
    for idx, tol in ((2, 1e-12), (3, 1e-12), (4, 1e-12)):
        w = workloads.config(idx)
        ctx = _ctx(w)
        g = E.ewald_get_g(ctx)
        assert np.array_equal(g, ref.gplus(w.dim, w.cell, w.g_cutoff))
        pos = w.positions(3)
        d_pos = torch.from_numpy(E.to_soa(pos)).cuda()
        d_q = torch.from_numpy(w.charges).cuda()
        E.ewald_load_walkers(ctx, w.n, d_pos, d_q)
        for k in (0, 2):
            pts, q = pos[k], w.charges
            if w.ion_pos is not None:
                pts, q = np.concatenate([pts, w.ion_pos]), np.concatenate([q, w.ion_q])
            rho_ref = ref.rho(w.dim, w.cell, w.g_cutoff, pts, q)
            rho = E.ewald_get_rho(ctx, k)
            assert np.abs(rho - rho_ref).max() <= tol * np.abs(q).sum()
            assert np.allclose(E.ewald_get_positions(ctx, k, w.n), pos[k], rtol=0, atol=0)


def _random_cell(rng, dim, scale=6.0):
    a = np.eye(dim) * scale + rng.uniform(-0.15, 0.15, (dim, dim)) * scale
    return a


@pytest.mark.parametrize("dim", [2, 3])
def test_small_general_cells_ragged_sizes(torch_cuda, dim):
    """Non-orthogonal cells, mixed charges (charged and neutral), N = 1, 2, 3, 5, 7, 33 (pad tails,
    fewer particles than a tile), auto r_cutoff."""
    rng = np.random.default_rng(7 + dim)
    for n in (1, 2, 3, 5, 7, 33):
        cell = _random_cell(rng, dim)
        kappa = 0.9
        gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
        q = rng.choice([-1.0, 1.0, 2.0, -0.5], size=n)
        frac = rng.random((3, n, dim)) * 1.6 - 0.3  # some positions outside the cell (reading R9)
        pos = frac @ cell
        e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, pos, q)
        ctx = E.ewald_setup(dim, cell, kappa, gc)  # r_cutoff = 0: automatic
        assert abs(E.ewald_r_cutoff(ctx) - rc) < 1e-12
        e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
        # tiny neutral cells can have |E| << terms: compare against the largest component
        scale = np.abs(c_ref).max(axis=1)
        assert (np.abs(e - e_ref) / scale).max() <= TOL64
        assert (np.abs(c - c_ref) / scale[:, None]).max() <= TOL64


@pytest.mark.parametrize("dim", [2, 3])
def test_orthorhombic_noncubic_cells_all_image_ranges(torch_cuda, dim):
    """Orthorhombic cells with unequal sides: kappa chosen so that the per-axis image range of the
    real-space scan is 0, 1, 2 and 3 (the last one takes the general image-list path)."""
    rng = np.random.default_rng(21 + dim)
    sides = np.array([5.0, 6.5, 8.0])[:dim]
    cell = np.diag(sides)
    for kappa, rc_over in ((2.6, None), (0.9, None), (0.7, None), (0.4, None), (1.3, 0.45)):
        gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
        if rc_over is not None:
            rc = rc_over * sides.min()  # r_c below half the shortest side: minimum image only (not converged; parity only)
        n = 11
        q = rng.choice([-1.0, 1.0, 2.0], size=n)
        pos = (rng.random((3, n, dim)) * 2 - 0.5) * sides
        e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, pos, q)
        ctx = E.ewald_setup(dim, cell, kappa, gc, rc)
        e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
        scale = np.abs(c_ref).max(axis=1)
        assert (np.abs(c - c_ref) / scale[:, None]).max() <= TOL64, (kappa, rc)
        e32, c32 = _gpu_energy(torch_cuda, ctx, _r32(pos), q, "f32")
        e_ref32, c_ref32 = ref.energy_batch(dim, cell, kappa, gc, rc, _r32(pos), q)
        assert (np.abs(c32 - c_ref32) / np.abs(c_ref32).max(axis=1)[:, None]).max() <= TOL32, (kappa, rc)


@pytest.mark.parametrize("with_ions", [False, True])
def test_small_batch_z_split_agrees_with_large_batch(torch_cuda, with_ions):
    """Boxes that need |m| <= 2 images per axis in 3D (config 1: r_c = 2.2 L, 125 candidates per pair): a batch too
    small to fill the SMs deals the five z-images of a pair to five lanes (ScanShape::ZSPLIT, chosen by the launch),
    a large batch does not.  Both must give the oracle's energies, and the same walker the same energy (up to the
    order of the tile sums) in either batch; ewald_launch_shape shows that the two launches differed."""
    torch = torch_cuda
    w = workloads.config(1)
    rng = np.random.default_rng(11)
    ions = (rng.random((5, 3)) * w.L, np.array([2.0, 2.0, 3.0, 3.0, 2.0])) if with_ions else (None, None)
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)
    if with_ions:
        E.ewald_set_fixed_charges(ctx, *ions)
    pos = w.positions(400)
    e_small, c_small = _gpu_energy(torch, ctx, pos[:6], w.charges, "f64")
    shape_small = E.ewald_launch_shape(ctx, 0)
    e_big, c_big = _gpu_energy(torch, ctx, pos, w.charges, "f64")
    shape_big = E.ewald_launch_shape(ctx, 0)
    assert shape_small["threads"] == shape_big["threads"] == 512
    assert shape_small["ctas"] > 6 * 3            # more tiles per walker than the pairs alone would give
    assert shape_big["ctas"] == 400 * 2           # (4 x 148 + 399) / 400 tiles per walker
    e_ref, c_ref = ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos[:6], w.charges, *ions)
    _assert_energy(e_small, c_small, e_ref, c_ref, TOL64)
    _assert_energy(e_big[:6], c_big[:6], e_ref, c_ref, TOL64)
    assert (np.abs(e_small - e_big[:6]) / np.abs(e_ref)).max() <= 1e-13



def test_uniform_charges_cutoff_reaching_two_far_images(torch_cuda):
    """Equal charges (bare-t stacks, candidate images enumerated as core / one far image / two or more far
    images) in cubic and orthorhombic cells whose cut-off r_c = 1.46 L_min exceeds sqrt(2) L_min: the branch
    with two and three far images per pair is needed and taken.  Energies and a committed move."""
    rng = np.random.default_rng(99)
    for sides in (np.array([5.0, 5.0, 5.0]), np.array([5.0, 5.2, 7.5])):
        cell = np.diag(sides)
        rc = 1.46 * sides.min()
        kappa = 6.1 / rc
        gc, _ = ref.auto_cutoffs(3, cell, kappa, 1e-17)
        n = 13
        q = -np.ones(n)
        pos = rng.random((4, n, 3)) * sides
        e_ref, c_ref = ref.energy_batch(3, cell, kappa, gc, rc, pos, q)
        ctx = E.ewald_setup(3, cell, kappa, gc, rc)
        e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
        scale = np.abs(c_ref).max(axis=1)
        assert (np.abs(c - c_ref) / scale[:, None]).max() <= TOL64
        electron = rng.integers(0, n, (2, 4)).astype(np.int32)
        new_r = rng.random((2, 4, 3)) * sides
        de_ref, _, _ = ref.move_chain(3, cell, kappa, gc, rc, pos, q, electron, new_r)
        E.ewald_load_walkers(ctx, n, torch_cuda.from_numpy(E.to_soa(pos)).cuda(), torch_cuda.from_numpy(q).cuda())
        d_w = torch_cuda.arange(4, dtype=torch_cuda.int32, device="cuda")
        for s_ in range(2):
            d_de = torch_cuda.zeros(4, dtype=torch_cuda.float64, device="cuda")
            E.ewald_move_delta_batch(ctx, d_w, torch_cuda.from_numpy(electron[s_]).cuda(),
                                     torch_cuda.from_numpy(new_r[s_]).cuda(), 1, d_de)
            _assert_delta(d_de.cpu().numpy()[None, :], de_ref[s_][None, :], TOL64, 1e-3 * scale)


@pytest.mark.parametrize("mixed", [False, True])
def test_cubic_cell_two_ion_species_energies_and_moves(torch_cuda, mixed):
    """Cubic cell with |m| <= 1 images, far shell present (kappa r_c = 6.1 > 4), fixed charges of two species.
    mixed = False: equal mobile charges -> bare-t stacks, one segment per species, signed items in the moves.
    mixed = True: unequal mobile charges -> (t, qq) items everywhere, far shell included."""
    rng = np.random.default_rng(77 + mixed)
    L = 7.0
    cell = np.eye(3) * L
    rc = 1.25 * L
    kappa = 6.1 / rc
    gc, _ = ref.auto_cutoffs(3, cell, kappa, 1e-17)
    n = 37
    q = rng.choice([-1.0, 1.0, -2.0], size=n) if mixed else -np.ones(n)
    pos = rng.random((4, n, 3)) * L
    ion_pos = rng.random((7, 3)) * L
    ion_q = np.array([3.0, 5.0, 3.0, 5.0, 5.0, 3.0, 3.0])
    e_ref, c_ref = ref.energy_batch(3, cell, kappa, gc, rc, pos, q, ion_pos, ion_q)
    ctx = E.ewald_setup(3, cell, kappa, gc, rc)
    E.ewald_set_fixed_charges(ctx, ion_pos, ion_q)
    scale = np.abs(c_ref).max(axis=1)
    for dtype, tol in (("f64", TOL64), ("f32", TOL32)):
        p = pos if dtype == "f64" else _r32(pos)
        er, cr = (e_ref, c_ref) if dtype == "f64" else ref.energy_batch(3, cell, kappa, gc, rc, p, q, ion_pos, ion_q)
        e, c = _gpu_energy(torch_cuda, ctx, p, q, dtype)
        assert (np.abs(c - cr) / np.abs(cr).max(axis=1)[:, None]).max() <= tol
    S = 3
    electron = rng.integers(0, n, (S, 4)).astype(np.int32)
    new_r = rng.random((S, 4, 3)) * L
    de_ref, _, _ = ref.move_chain(3, cell, kappa, gc, rc, pos, q, electron, new_r, ion_pos, ion_q)
    E.ewald_load_walkers(ctx, n, torch_cuda.from_numpy(E.to_soa(pos)).cuda(), torch_cuda.from_numpy(q).cuda())
    d_w = torch_cuda.arange(4, dtype=torch_cuda.int32, device="cuda")
    for s_ in range(S):
        d_de = torch_cuda.zeros(4, dtype=torch_cuda.float64, device="cuda")
        E.ewald_move_delta_batch(ctx, d_w, torch_cuda.from_numpy(electron[s_]).cuda(),
                                 torch_cuda.from_numpy(new_r[s_]).cuda(), 1, d_de)
        _assert_delta(d_de.cpu().numpy()[None, :], de_ref[s_][None, :], TOL64, 1e-3 * scale)


def test_fixed_charges_equal_mobile_charges(torch_cuda):
    """Ions passed as fixed charges give the same energy as the same ions passed as mobile particles."""
    rng = np.random.default_rng(11)
    cell = _random_cell(rng, 3)
    kappa = 0.8
    gc, rc = ref.auto_cutoffs(3, cell, kappa, 1e-17)
    n, ni = 6, 3
    pos = rng.random((4, n, 3)) @ cell
    ion = rng.random((ni, 3)) @ cell
    q, qi = -np.ones(n), np.array([2.0, 3.0, 1.0])
    ctx = E.ewald_setup(3, cell, kappa, gc, rc)
    E.ewald_set_fixed_charges(ctx, ion, qi)
    e1, c1 = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
    ctx2 = E.ewald_setup(3, cell, kappa, gc, rc)
    allpos = np.concatenate([pos, np.broadcast_to(ion, (4, ni, 3))], axis=1)
    e2, c2 = _gpu_energy(torch_cuda, ctx2, allpos, np.concatenate([q, qi]), "f64")
    e_ref, c_ref = ref.energy_batch(3, cell, kappa, gc, rc, pos, q, ion, qi)
    scale = np.abs(c_ref).max(axis=1)
    assert (np.abs(e1 - e_ref) / scale).max() <= TOL64 and (np.abs(e2 - e_ref) / scale).max() <= TOL64
    _, _, e_fixed = E.ewald_get_constants(ctx)
    e_ion_ref, _ = ref.energy_batch(3, cell, kappa, gc, rc, ion[None], qi)
    assert abs(e_fixed - e_ion_ref[0]) <= 1e-12 * abs(e_ion_ref[0])


def test_empty_batch_and_host_entry_point(torch_cuda):
    torch = torch_cuda
    w = workloads.config(1)
    ctx = _ctx(w)
    pos = w.positions(5)
    d_q = torch.from_numpy(w.charges).cuda()
    d_e = torch.zeros(0, dtype=torch.float64, device="cuda")
    E.ewald_energy_batch(ctx, w.n, torch.zeros((0, 3, E.ewald_padded_n(w.n)), dtype=torch.float64, device="cuda"),
                         d_q, d_e)
    e, c = _gpu_energy(torch, ctx, pos, w.charges, "f64")
    eh, ch = np.zeros(5), np.zeros((5, 4))
    E.ewald_energy_batch_host(ctx, w.n, E.to_soa(pos), w.charges.copy(), eh, ch)
    assert np.array_equal(e, eh) and np.array_equal(c, ch)  # same kernels, same order: bit-identical


def _move_inputs(w, n_walkers, n_steps):
    pos0 = w.positions(n_walkers)
    electron, disp = w.moves(n_walkers, n_steps)
    cur = pos0.copy()
    new_r = np.zeros((n_steps, n_walkers, w.dim))
    for s in range(n_steps):  # absolute targets: current position of that electron + Gaussian step
        idx = electron[s]
        new_r[s] = cur[np.arange(n_walkers), idx] + disp[s]
        cur[np.arange(n_walkers), idx] = new_r[s]
    return pos0, electron, new_r, cur


def _run_moves(torch, ctx, w, pos0, electron, new_r, dtype):
    npdt = np.float64 if dtype == "f64" else np.float32
    tdt = torch.float64 if dtype == "f64" else torch.float32
    S, W = electron.shape
    E.ewald_load_walkers(ctx, w.n, torch.from_numpy(E.to_soa(pos0, npdt)).cuda(),
                         torch.from_numpy(w.charges.astype(npdt)).cuda())
    d_w = torch.arange(W, dtype=torch.int32, device="cuda")
    de = np.zeros((S, W))
    for s in range(S):
        d_el = torch.from_numpy(electron[s]).cuda()
        d_r = torch.from_numpy(new_r[s].astype(npdt)).cuda().to(tdt).contiguous()
        d_de = torch.zeros(W, dtype=torch.float64, device="cuda")
        E.ewald_move_delta_batch(ctx, d_w, d_el, d_r, 1, d_de)
        de[s] = d_de.cpu().numpy()
    return de


def _assert_delta(de, de_ref, tol, floor=0.0):
    """Reading R12: |dE - dE_ref| <= tol * max(|dE_ref|, rms of dE_ref over the step's batch).  `floor` guards the
    degenerate small systems only (a lone particle in a periodic cell has dE = 0 exactly): it is 1e-3 of the
    walker's largest energy component there, i.e. an absolute error of 1e-14 of that component at FP64."""
    rms = np.sqrt((de_ref ** 2).mean(axis=1, keepdims=True))
    err = np.abs(de - de_ref) / np.maximum(np.maximum(np.abs(de_ref), rms), floor)
    assert err.max() <= tol, "max Delta-E error %.3e > %.1e" % (err.max(), tol)
    return float(err.max())


@pytest.mark.parametrize("dtype,tol", [("f64", TOL64), ("f32", TOL32)])
def test_move_chain_config5_matches_oracle(torch_cuda, dtype, tol):
    w = workloads.config(5)
    W, S = 6, 12
    pos0, electron, new_r, final = _move_inputs(w, W, S)
    if dtype == "f32":
        pos0, new_r, final = _r32(pos0), _r32(new_r), _r32(final)
    de_ref, pos_ref, rho_ref = ref.move_chain(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos0,
                                              w.charges, electron, new_r, want_rho=True)
    ctx = _ctx(w)
    de = _run_moves(torch_cuda, ctx, w, pos0, electron, new_r, dtype)
    _assert_delta(de, de_ref, tol)
    # the stored state after the chain equals a fresh evaluation of the final configuration
    rho = E.ewald_get_rho(ctx, 3)
    assert np.abs(rho - rho_ref[3]).max() <= (1e-12 if dtype == "f64" else 3e-6) * w.n
    got = E.ewald_get_positions(ctx, 3, w.n)
    assert np.abs(got - final[3]).max() == 0
    if dtype == "f64":
        e0, _ = _gpu_energy(torch_cuda, ctx, pos0, w.charges, "f64", components=False)
        e1, _ = _gpu_energy(torch_cuda, ctx, final, w.charges, "f64", components=False)
        assert np.abs(e0 + de.sum(axis=0) - e1).max() <= 1e-11 * np.abs(e1).max()


def test_moves_with_ions_2d_and_uncommitted(torch_cuda):
    torch = torch_cuda
    rng = np.random.default_rng(5)
    for dim in (2, 3):
        cell = _random_cell(rng, dim, 7.0)
        kappa = 0.75
        gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
        n, ni, W, S = 9, 2, 3, 5
        q = rng.choice([-1.0, 1.0], size=n)
        pos0 = rng.random((W, n, dim)) @ cell
        ion, qi = rng.random((ni, dim)) @ cell, np.array([2.0, -1.0])
        electron = rng.integers(0, n, (S, W)).astype(np.int32)
        new_r = rng.random((S, W, dim)) @ cell
        de_ref, _, rho_ref = ref.move_chain(dim, cell, kappa, gc, rc, pos0, q, electron, new_r, ion, qi,
                                            want_rho=True)
        ctx = E.ewald_setup(dim, cell, kappa, gc, rc)
        E.ewald_set_fixed_charges(ctx, ion, qi)
        E.ewald_load_walkers(ctx, n, torch.from_numpy(E.to_soa(pos0)).cuda(), torch.from_numpy(q).cuda())
        d_w = torch.arange(W, dtype=torch.int32, device="cuda")
        for s in range(S):
            d_el, d_r = torch.from_numpy(electron[s]).cuda(), torch.from_numpy(new_r[s]).cuda()
            trial = torch.zeros(W, dtype=torch.float64, device="cuda")
            E.ewald_move_delta_batch(ctx, d_w, d_el, d_r, 0, trial)   # rejected proposal: no change
            d_de = torch.zeros(W, dtype=torch.float64, device="cuda")
            E.ewald_move_delta_batch(ctx, d_w, d_el, d_r, 1, d_de)
            assert torch.equal(trial, d_de)
            scale = np.abs(de_ref).max()
            assert np.abs(d_de.cpu().numpy() - de_ref[s]).max() <= 1e-11 * scale
        for k in range(W):
            assert np.abs(E.ewald_get_rho(ctx, k) - rho_ref[k]).max() <= 1e-12 * (n + 3)
        # scalar form: move there and back again sums to zero and restores rho
        before = E.ewald_get_rho(ctx, 1)
        old = E.ewald_get_positions(ctx, 1, n)[4]
        d1 = E.ewald_move_delta(ctx, 1, 4, new_r[0, 0], commit=True)
        d2 = E.ewald_move_delta(ctx, 1, 4, old, commit=True)
        assert abs(d1 + d2) <= 1e-12 * max(abs(d1), 1.0)
        assert np.abs(E.ewald_get_rho(ctx, 1) - before).max() <= 1e-13 * (n + 3)


def test_state_errors(torch_cuda):
    torch = torch_cuda
    w = workloads.config(1)
    ctx = _ctx(w)
    with pytest.raises(E.EwaldError) as ei:
        E.ewald_move_delta(ctx, 0, 0, [0.0, 0.0, 0.0])
    assert ei.value.status == 4
    E.ewald_load_walkers(ctx, w.n, torch.from_numpy(E.to_soa(w.positions(2))).cuda(),
                         torch.from_numpy(w.charges).cuda())
    for wk, el in ((2, 0), (0, w.n), (-1, 0)):
        with pytest.raises(E.EwaldError) as ei:
            E.ewald_move_delta(ctx, wk, el, [0.0, 0.0, 0.0])
        assert ei.value.status == 4
    # batch form: out-of-range entries give NaN and leave the state alone
    before = E.ewald_get_rho(ctx, 1)
    d_de = torch.zeros(2, dtype=torch.float64, device="cuda")
    E.ewald_move_delta_batch(ctx, torch.tensor([0, 1], dtype=torch.int32, device="cuda"),
                             torch.tensor([3, 9999], dtype=torch.int32, device="cuda"),
                             torch.zeros((2, 3), dtype=torch.float64, device="cuda"), 1, d_de)
    out = d_de.cpu().numpy()
    assert np.isfinite(out[0]) and np.isnan(out[1])
    assert np.array_equal(E.ewald_get_rho(ctx, 1), before)


N_SAMPLE = 256   # walkers the oracle checks one by one in the full-size tests (>= 256)


def _sample(n_walkers, k=N_SAMPLE, seed=2):
    """First, last and k - 2 seeded-random other walkers."""
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(1, n_walkers - 1), size=min(k, n_walkers) - 2, replace=False)
    return np.sort(np.concatenate([[0, n_walkers - 1], mid]))


def test_full_size_config2_sampled_walkers(torch_cuda):
    """BASELINE configs[1] at its full size (1024 walkers), in the launch configuration bench.py
    times; the oracle checks 256 walkers one by one, FP64 and FP32."""
    w = workloads.config(2)
    pos = w.positions()
    ctx = _ctx(w)
    sample = _sample(w.n_walkers)
    for dtype, tol in (("f64", TOL64), ("f32", TOL32)):
        if dtype == "f32":
            pos = _r32(pos)
        e_ref, _ = _oracle_energy(w, pos[sample])
        e, _ = _gpu_energy(torch_cuda, ctx, pos, w.charges, dtype, components=False)
        assert np.all(np.isfinite(e))
        rel = np.abs(e[sample] - e_ref) / np.abs(e_ref)
        print("config 2 %s: max rel err over %d walkers %.3e" % (dtype, len(sample), rel.max()))
        assert rel.max() <= tol
        # property that holds at any size: identical walkers give identical energies
        e2, _ = _gpu_energy(torch_cuda, ctx, pos[::-1].copy(), w.charges, dtype, components=False)
        assert np.array_equal(e2[::-1], e)


@pytest.mark.parametrize("idx", [3, 4])
def test_full_size_configs_3_and_4_sampled_walkers(torch_cuda, idx):
    """BASELINE configs[2] and configs[3] at their full sizes (1024 / 4096 walkers), in the launch
    configuration bench.py --config 3 / 4 times; the oracle checks 256 walkers one by one (FP64; FP32: 64)."""
    w = workloads.config(idx)
    pos = w.positions()
    ctx = _ctx(w)
    for dtype, tol, k in (("f64", TOL64, N_SAMPLE), ("f32", TOL32, 64)):
        sample = _sample(w.n_walkers, k)
        p = pos if dtype == "f64" else _r32(pos)
        e_ref, _ = _oracle_energy(w, p[sample])
        e, _ = _gpu_energy(torch_cuda, ctx, p, w.charges, dtype, components=False)
        assert np.all(np.isfinite(e))
        rel = np.abs(e[sample] - e_ref) / np.abs(e_ref)
        print("config %d %s: max rel err over %d walkers %.3e" % (idx, dtype, len(sample), rel.max()))
        assert rel.max() <= tol


# Bound on the error of the stored FP32 rho(G) after 100 patches, in units of N (R16).  The loaded rho is
# an FP32 sum of N unit phasors (|rho| ~ sqrt N, error a few ulps); each patch adds q delta(G) (|delta| <= 2) and
# rounds to 2^-24 |rho| ~ 2e-6 at N = 1000: 100 patches random-walk to ~ 2e-5, the worst of 1979 G-vectors to
# ~ 1e-4 absolute = 1e-7 N.  Asserted with a factor 3 of margin; the measured value is printed.
RHO32_DRIFT = 3e-7


@pytest.mark.parametrize("dtype,tol", [("f64", TOL64), ("f32", TOL32)])
def test_full_size_config5_100_steps(torch_cuda, dtype, tol):
    """BASELINE configs[4] at its stated size: 4096 walkers with stored rho(G), 100 committed steps per walker in
    batches of 4096 moves (the launch configuration bench.py times), FP64 and FP32.  Walkers are independent, so
    the oracle runs the 100-step chains of 16 sampled walkers: Delta E of every step, final rho(G) and final
    positions; and sum Delta E + E_0 is checked against a fresh ewald_energy_batch of the final configuration
    for ALL walkers (with the oracle's energies on the sample)."""
    w = workloads.config(5)
    W, S = w.n_walkers, w.n_steps
    assert (W, S) == (4096, 100)
    pos0, electron, new_r, final = _move_inputs(w, W, S)
    if dtype == "f32":
        pos0, new_r, final = _r32(pos0), _r32(new_r), _r32(final)
    ctx = _ctx(w)
    de = _run_moves(torch_cuda, ctx, w, pos0, electron, new_r, dtype)
    assert np.all(np.isfinite(de))
    sample = _sample(W, 16, seed=5)
    de_ref, pos_ref, rho_ref = ref.move_chain(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos0[sample],
                                              w.charges, electron[:, sample], new_r[:, sample], want_rho=True)
    err = _assert_delta(de[:, sample], de_ref, tol)
    drift = 0.0
    for k, wk in enumerate(sample):
        d = np.abs(E.ewald_get_rho(ctx, int(wk)) - rho_ref[k]).max() / w.n
        drift = max(drift, d)
        assert np.abs(E.ewald_get_positions(ctx, int(wk), w.n) - final[wk]).max() == 0
    print("config 5 %s: max Delta-E error (R12) %.3e over 16 walkers x 100 steps; stored rho drift %.3e N"
          % (dtype, err, drift))
    assert drift <= (1e-12 if dtype == "f64" else RHO32_DRIFT)
    # sum of the steps + E_0 = energy of the final configuration (all 4096 walkers, GPU; oracle on the sample)
    e0, _ = _gpu_energy(torch_cuda, ctx, pos0, w.charges, dtype, components=False)
    e1, _ = _gpu_energy(torch_cuda, ctx, final, w.charges, dtype, components=False)
    # Denominators as in reading R12: uniform-random N = 1000 walkers have E between -2 and -180 Ha (close pairs)
    # out of components of +-3300 Ha, so a walker's own |E| can be 1e-3 of what the arithmetic handles; FP64 keeps
    # the per-walker |E| all the same.
    e1_ref, _ = _oracle_energy(w, final[sample])
    rms = np.sqrt((e1_ref ** 2).mean())
    den_all = np.abs(e1) if dtype == "f64" else np.maximum(np.abs(e1), rms)
    den = np.abs(e1_ref) if dtype == "f64" else np.maximum(np.abs(e1_ref), rms)
    closure = np.abs(e0 + de.sum(axis=0) - e1) / den_all
    e1_err = np.abs(e1[sample] - e1_ref) / den
    print("config 5 %s: closure |E0 + sum dE - E1| / den max %.3e; E1 vs oracle %.3e (per-walker |E|: %.3e)"
          % (dtype, closure.max(), e1_err.max(), (np.abs(e1[sample] - e1_ref) / np.abs(e1_ref)).max()))
    assert e1_err.max() <= tol
    # 100 steps each within tol * max(|dE|, rms dE) of the oracle; the sum is compared at 10 tol
    assert closure.max() <= 10 * tol


# Measured bound of the FP32 path against the oracle on the UNROUNDED seeded inputs (R16): the kernels'
# own error (<= 2e-5, asserted everywhere else on the rounded inputs) plus the effect of rounding the coordinates
# to float32 (half an ulp of up to L: 2^-25 L), which a close pair amplifies by L / r_min.
# Config 3 (2D, L = 188 bohr, 450 particles): the closest pair of a walker sits at ~0.05 bohr while half an ulp of a
# coordinate is 5.6e-6 bohr, so input rounding ALONE moves E by up to 4.2e-4 (oracle vs oracle, 64 walkers, printed);
# the kernels' own error stays <= 2e-5.  The test asserts that the excess over the input-rounding effect is <= 2e-5.
FP32_UNROUNDED_BOUND = {1: 2e-5, 2: 2e-5, 3: 1e-3, 4: 2e-5, 5: 2e-5}


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_fp32_against_oracle_on_unrounded_inputs(torch_cuda, idx):
    """SURVEY reading 16 as a measured diagnostic: FP32 path on float32(positions) against the oracle on the
    unrounded FP64 positions, beside the same comparison on the rounded positions."""
    w = workloads.config(idx)
    nw = {1: 8, 2: 64, 3: 64, 4: 32, 5: 8}[idx]
    pos = w.positions(nw)
    e_un, _ = _oracle_energy(w, pos)
    e_rd, _ = _oracle_energy(w, _r32(pos))
    e, _ = _gpu_energy(torch_cuda, _ctx(w), pos, w.charges, "f32", components=False)   # to_soa rounds
    rel_un = np.abs(e - e_un) / np.abs(e_un)
    rel_rd = np.abs(e - e_rd) / np.abs(e_rd)
    rel_in = np.abs(e_rd - e_un) / np.abs(e_un)
    print("config %d FP32, %d walkers: vs oracle(unrounded) max %.3e | vs oracle(rounded) max %.3e | "
          "input rounding alone (oracle vs oracle) max %.3e" % (idx, nw, rel_un.max(), rel_rd.max(), rel_in.max()))
    assert rel_rd.max() <= TOL32
    assert rel_un.max() <= FP32_UNROUNDED_BOUND[idx]
    assert (rel_un - rel_in).max() <= TOL32   # what the kernels add on top of the caller's rounding


def test_far_stack_headroom_n1000_wide_cutoff(torch_cuda):
    """N = 1000 in FP64 leaves room for an 18-deep far stack only (outer_far without far_once): between two
    services a lane can push 12 one-far candidates and then the next pair's 8 core candidates.  kappa L = 4.6 with
    r_c = 6.5 / kappa fills the far shell as densely as the geometry allows (the far stack overflowed
    into the next warp's near stack here)."""
    n = 1000
    L = (4.0 * math.pi * n / 3.0) ** (1.0 / 3.0)
    cell = np.eye(3) * L
    kappa = 4.6 / L
    rc = 6.5 / kappa
    gc = 2 * math.pi / L * math.sqrt(61) * (1 + 1e-9)
    rng = np.random.default_rng(4600)
    pos = rng.random((2, n, 3)) * L
    q = -np.ones(n)
    ctx = E.ewald_setup(3, cell, kappa, gc, rc)
    e_ref, c_ref = ref.energy_batch(3, cell, kappa, gc, rc, pos, q)
    e, c = _gpu_energy(torch_cuda, ctx, pos, q, "f64")
    assert (np.abs(c[:, 1] - c_ref[:, 1]) / np.abs(c_ref[:, 1])).max() <= 1e-12
    _assert_energy(e, c, e_ref, c_ref, TOL64)


def test_largest_paper_system_n1630(torch_cuda):
    """The paper's largest electron gas (N = 1630) at r_s = 1: positions no longer leave room
    for the full-size stacks in shared memory, so the launch shapes shrink; 3 walkers against the oracle, FP64
    and FP32, and one committed move per walker."""
    n = 1630
    L = (4.0 * math.pi * n / 3.0) ** (1.0 / 3.0)
    cell = np.eye(3) * L
    kappa, rc = 5.4 / L, 1.1 * L
    gc = 2 * math.pi / L * math.sqrt(97) * (1 + 1e-9)
    rng = np.random.default_rng(1630)
    pos = rng.random((3, n, 3)) * L
    q = -np.ones(n)
    ctx = E.ewald_setup(3, cell, kappa, gc, rc)
    for dtype, tol in (("f64", TOL64), ("f32", TOL32)):
        p = pos if dtype == "f64" else _r32(pos)
        e_ref, _ = ref.energy_batch(3, cell, kappa, gc, rc, p, q)
        e, _ = _gpu_energy(torch_cuda, ctx, p, q, dtype, components=False)
        assert (np.abs(e - e_ref) / np.abs(e_ref)).max() <= tol
    electron = rng.integers(0, n, (1, 3)).astype(np.int32)
    new_r = rng.random((1, 3, 3)) * L
    de_ref, _, _ = ref.move_chain(3, cell, kappa, gc, rc, pos, q, electron, new_r)
    E.ewald_load_walkers(ctx, n, torch_cuda.from_numpy(E.to_soa(pos)).cuda(), torch_cuda.from_numpy(q).cuda())
    d_de = torch_cuda.zeros(3, dtype=torch_cuda.float64, device="cuda")
    E.ewald_move_delta_batch(ctx, torch_cuda.arange(3, dtype=torch_cuda.int32, device="cuda"),
                             torch_cuda.from_numpy(electron[0]).cuda(), torch_cuda.from_numpy(new_r[0]).cuda(), 1, d_de)
    _assert_delta(d_de.cpu().numpy()[None, :], de_ref, TOL64)


def test_next1_hexagonal_hbn_workload(torch_cuda):
    """the hexagonal 9 x 9 hBN-shaped cell (non-orthogonal cell, ~25 000
    G-vectors, 648 electrons, two ion species): complex half-set reciprocal kernel, image-list real-space scan,
    (t, qq) stack items.  Energies of 3 walkers in FP64 and FP32, then two committed moves per walker."""
    w = workloads.config(6)
    pos = w.positions(3)
    ctx = _ctx(w)
    for dtype, tol in (("f64", TOL64), ("f32", TOL32)):
        p = pos if dtype == "f64" else _r32(pos)
        e_ref, c_ref = _oracle_energy(w, p)
        e, c = _gpu_energy(torch_cuda, ctx, p, w.charges, dtype)
        _assert_energy(e, c, e_ref, c_ref, tol)
    rng = np.random.default_rng(6)
    S = 2
    electron = rng.integers(0, w.n, (S, 3)).astype(np.int32)
    cur = pos.copy()
    new_r = np.zeros((S, 3, 3))
    for s_ in range(S):
        new_r[s_] = cur[np.arange(3), electron[s_]] + 0.5 * rng.standard_normal((3, 3))
        cur[np.arange(3), electron[s_]] = new_r[s_]
    de_ref, _, _ = ref.move_chain(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges, electron, new_r,
                                  w.ion_pos, w.ion_q)
    de = _run_moves(torch_cuda, ctx, w, pos, electron, new_r, "f64")
    _assert_delta(de, de_ref, TOL64)


@pytest.mark.parametrize("seed", list(range(24)))
def test_randomised_small_systems(torch_cuda, seed):
    """Seeded random small systems across the code paths: 2D/3D; cubic, orthorhombic and general cells; image
    ranges 0..3; equal or mixed mobile charges; 0..6 fixed charges of 1..6 species (more than 4 species fall back
    to (t, qq) items); energies in FP64 and FP32 and two moves per walker (one committed, one not)."""
    rng = np.random.default_rng(1000 + seed)
    dim = 2 + seed % 2
    kind = (seed // 2) % 3
    sides = np.array([4.0 + 3.0 * rng.random() for _ in range(dim)])
    if kind == 0:
        cell = np.eye(dim) * sides[0]
    elif kind == 1:
        cell = np.diag(sides)
    else:
        cell = np.diag(sides) + rng.uniform(-0.2, 0.2, (dim, dim)) * sides.min()
    kappa = float(rng.choice([0.45, 0.7, 1.0, 1.6, 2.4])) * 6.0 / sides.min() / 2.0
    gc, rc = ref.auto_cutoffs(dim, cell, kappa, 1e-17)
    n = int(rng.integers(1, 41))
    q = -np.ones(n) if rng.random() < 0.5 else rng.choice([-1.0, 1.0, 2.0, -0.5], size=n)
    n_ion = int(rng.integers(0, 7))
    ion_pos = rng.random((n_ion, dim)) @ cell if n_ion else None
    ion_q = rng.choice([1.0, 2.0, 3.0, 4.0, 5.0, 6.0], size=n_ion) if n_ion else None
    W = 3
    pos = (rng.random((W, n, dim)) * 1.5 - 0.25) @ cell
    ctx = E.ewald_setup(dim, cell, kappa, gc, rc)
    if n_ion:
        E.ewald_set_fixed_charges(ctx, ion_pos, ion_q)
    for dtype, tol in (("f64", TOL64), ("f32", TOL32)):
        p = pos if dtype == "f64" else _r32(pos)
        e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, p, q, ion_pos, ion_q)
        e, c = _gpu_energy(torch_cuda, ctx, p, q, dtype)
        scale = np.abs(c_ref).max(axis=1)
        assert (np.abs(c - c_ref) / scale[:, None]).max() <= tol, (dtype, seed)
    electron = rng.integers(0, n, (2, W)).astype(np.int32)
    new_r = (rng.random((2, W, dim)) * 1.2 - 0.1) @ cell
    # step 0 is not committed, step 1 is: the oracle chain therefore starts both from the loaded positions
    de0, _, _ = ref.move_chain(dim, cell, kappa, gc, rc, pos, q, electron[:1], new_r[:1], ion_pos, ion_q)
    de1, _, _ = ref.move_chain(dim, cell, kappa, gc, rc, pos, q, electron[1:], new_r[1:], ion_pos, ion_q)
    E.ewald_load_walkers(ctx, n, torch_cuda.from_numpy(E.to_soa(pos)).cuda(), torch_cuda.from_numpy(q).cuda())
    d_w = torch_cuda.arange(W, dtype=torch_cuda.int32, device="cuda")
    e_ref, c_ref = ref.energy_batch(dim, cell, kappa, gc, rc, pos, q, ion_pos, ion_q)
    scale = np.abs(c_ref).max(axis=1)
    for s_, (commit, want) in enumerate(((0, de0[0]), (1, de1[0]))):
        d_de = torch_cuda.zeros(W, dtype=torch_cuda.float64, device="cuda")
        E.ewald_move_delta_batch(ctx, d_w, torch_cuda.from_numpy(electron[s_]).cuda(),
                                 torch_cuda.from_numpy(new_r[s_]).cuda(), commit, d_de)
        _assert_delta(d_de.cpu().numpy()[None, :], want[None, :], TOL64, 1e-3 * scale)


def test_translation_and_permutation_invariance_on_gpu(torch_cuda):
    w = workloads.config(2)
    pos = w.positions(4)
    ctx = _ctx(w)
    e, _ = _gpu_energy(torch_cuda, ctx, pos, w.charges, "f64", components=False)
    shift = np.array([0.37, -2.11, 5.3]) * w.L
    e_t, _ = _gpu_energy(torch_cuda, ctx, pos + shift, w.charges, "f64", components=False)
    perm = np.random.default_rng(3).permutation(w.n)
    e_p, _ = _gpu_energy(torch_cuda, ctx, pos[:, perm], w.charges, "f64", components=False)
    assert (np.abs(e_t - e) / np.abs(e)).max() <= 1e-11 and (np.abs(e_p - e) / np.abs(e)).max() <= 1e-12
