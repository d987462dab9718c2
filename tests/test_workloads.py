"""Seeded input generators and the five configurations; CPU only."""
import numpy as np
import pytest

from oracle import ewald_ref as ora
from paper_2507_02888_b200 import workloads

EXPECTED_NG = {1: 924, 2: 2006, 3: 1516, 4: 3070, 5: 3958}


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_g_counts_and_shapes(idx):
    w = workloads.config(idx)
    assert ora.num_g(w.dim, w.cell, w.g_cutoff) == EXPECTED_NG[idx]
    pos = w.positions(3)
    assert pos.shape == (3, w.n, w.dim) and pos.dtype == np.float64
    assert np.array_equal(pos, w.positions(5)[:3])          # walker-prefix property
    assert np.array_equal(pos, workloads.config(idx).positions(3))  # seeded
    assert len(w.charges) == w.n


def test_config4_geometry():
    w = workloads.config(4)
    assert w.ion_pos.shape == (64, 3) and np.all(w.ion_q == 4.0)
    assert w.ion_q.sum() + w.charges.sum() == 0
    # nearest-neighbour distance of diamond = sqrt(3) a / 4
    d = np.linalg.norm(w.ion_pos[:, None] - w.ion_pos[None], axis=-1)
    d[d == 0] = 1e9
    assert d.min() == pytest.approx(np.sqrt(3) * 10.26 / 4)
    pos = w.positions(2)
    disp = pos - np.repeat(w.ion_pos, 4, axis=0)[None]
    assert abs(disp.std() - 1.0) < 0.05


def test_config5_moves():
    w = workloads.config(5)
    el, disp = w.moves(4, 10)
    assert el.shape == (10, 4) and disp.shape == (10, 4, 3)
    assert el.min() >= 0 and el.max() < w.n
    el2, disp2 = w.moves(8, 100)
    assert np.array_equal(el2[:10, :4], el) and np.array_equal(disp2[:10, :4], disp)


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_config_cutoffs_are_converged(idx):
    """The configs' (kappa, G_cut, r_cut) reproduce a fully converged evaluation at kappa' = 1.3 kappa."""
    w = workloads.config(idx)
    pos = w.positions(1)
    e, comp = ora.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges,
                               w.ion_pos, w.ion_q)
    k2 = 1.3 * w.kappa
    g2, r2 = ora.auto_cutoffs(w.dim, w.cell, k2, 1e-17)
    e2, _ = ora.energy_batch(w.dim, w.cell, k2, g2, r2, pos, w.charges, w.ion_pos, w.ion_q)
    assert e[0] == pytest.approx(e2[0], rel=1e-12)


def test_config6_hexagonal_geometry():
    """NEXT-1 workload: neutral hexagonal cell, B-N nearest-neighbour distance a / sqrt(3), ~25 000 G-vectors."""
    w = workloads.config(6)
    assert w.ion_pos.shape == (162, 3) and w.n == 648
    assert w.ion_q.sum() + w.charges.sum() == 0
    frac = w.ion_pos @ np.linalg.inv(w.cell)
    assert frac.min() >= 0 and frac.max() < 1
    d = w.ion_pos[:, None] - w.ion_pos[None]
    f = d @ np.linalg.inv(w.cell)
    d = (f - np.rint(f)) @ w.cell
    r = np.linalg.norm(d, axis=-1)
    r[r == 0] = 1e9
    assert r.min() == pytest.approx(4.75 / np.sqrt(3))
    ng = ora.num_g(w.dim, w.cell, w.g_cutoff)
    assert 20000 < ng < 30000
    # the cut-offs reproduce a converged evaluation at another splitting (one walker)
    pos = w.positions(1)
    e, _ = ora.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges, w.ion_pos, w.ion_q)
    k2 = 0.8 * w.kappa
    g2, r2 = ora.auto_cutoffs(w.dim, w.cell, k2, 1e-17)
    e2, _ = ora.energy_batch(w.dim, w.cell, k2, g2, r2, pos, w.charges, w.ion_pos, w.ion_q)
    assert e[0] == pytest.approx(e2[0], rel=1e-11)
