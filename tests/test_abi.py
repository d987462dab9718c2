"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/ewald.h declares; the host-only setup tables reproduce the closed forms of Eq. 4
(PAPER.md:120); argument validation.  No compute call is made (there is no GPU here)."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from paper_2507_02888_b200 import ewald as E
from paper_2507_02888_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "ewald.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ewald_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported():
    lib = ctypes.CDLL(E.load_library()._name)
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), "library does not export %s" % name
    assert sorted(E.SYMBOLS) == declared, "binding's symbol list differs from the header"


def test_jastrow_header_symbols_exported_and_bound():
    """include/jastrow.h: every declared call is exported by the library and has a
    binding of the same name."""
    from paper_2507_02888_b200 import jastrow as J
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "jastrow.h")).read(), flags=re.S)
    declared = sorted(set(re.findall(r"\b(jastrow_[a-z0-9_]+)\s*\(", text)))
    lib = ctypes.CDLL(E.load_library()._name)
    assert len(declared) == 8 and declared == sorted(J.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), "library does not export %s" % name
        if name != "jastrow_last_error":
            assert hasattr(J, name), "python binding lacks %s" % name


def test_blip_header_symbols_exported_and_bound():
    """include/blip.h."""
    from paper_2507_02888_b200 import blip as B
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "blip.h")).read(), flags=re.S)
    declared = sorted(set(re.findall(r"\b(blip_[a-z0-9_]+)\s*\(", text)))
    lib = ctypes.CDLL(E.load_library()._name)
    assert len(declared) == 6 and declared == sorted(B.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), "library does not export %s" % name
        if name != "blip_last_error":
            assert hasattr(B, name), "python binding lacks %s" % name


def test_binding_has_same_names():
    for name in _declared_symbols():
        if name in ("ewald_last_error", "ewald_destroy"):
            continue
        assert hasattr(E, name), "python binding lacks %s" % name


def test_version_and_padding():
    assert "sm_100a" in E.ewald_version()
    assert [E.ewald_padded_n(n) for n in (0, 1, 4, 5, 250, 1000)] == [0, 4, 4, 8, 252, 1000]


def test_setup_summary_counts_match_config_table():
    # SURVEY.md 8(d) / DESIGN.md: full-sphere G counts of the five configs (reading R5)
    want = {1: (924, [6, 6, 6]), 2: (2006, [7, 7, 7]), 3: (1516, [22, 22, 0]), 4: (3070, [9, 9, 9]),
            5: (3958, [9, 9, 9])}
    for idx, (ng, nmax) in want.items():
        w = workloads.config(idx)
        s = E.ewald_setup_summary(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)
        assert s["num_g"] == ng and s["n_max"] == nmax
        assert 1 <= s["num_images"] <= 125


def test_setup_madelung_constant_closed_forms(golden):
    # v_M L of a cubic / square cell is a pure number: -2.837297... (3D), 4 zeta(1/2) beta(1/2) (2D)
    for idx in (1, 2, 4, 5):
        w = workloads.config(idx)
        s = E.ewald_setup_summary(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)
        assert abs(s["v_m"] * w.L - golden["vm_L_sc_3d"]) < 2e-13
    w = workloads.config(3)
    s = E.ewald_setup_summary(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)
    assert abs(s["v_m"] * w.L - golden["vm_L_square_2d"]) < 2e-13


def test_setup_v_m_independent_of_kappa_noncubic():
    cell = np.array([[5.0, 0.3, 0.1], [0.4, 6.0, -0.2], [0.2, 0.5, 7.0]])
    vals = []
    for kappa in (0.5, 0.65, 0.8):
        x = math.sqrt(-math.log(1e-17))
        s = E.ewald_setup_summary(3, cell, kappa, 2 * kappa * x, x / kappa)
        vals.append(s["v_m"])
    assert max(vals) - min(vals) < 1e-13 * abs(vals[0])


def test_setup_argument_errors():
    cell = np.eye(3) * 4.0
    for args, status in (((4, cell, 1.0, 3.0), 1), ((3, cell, -1.0, 3.0), 3), ((3, cell, 1.0, 0.0), 3),
                         ((3, np.zeros((3, 3)), 1.0, 3.0), 2), ((3, cell, 1.0, 1e-3), 3)):
        with pytest.raises(E.EwaldError) as ei:
            E.ewald_setup_summary(*args)
        assert ei.value.status == status


def test_setup_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(E.EwaldError) as ei:
        E.ewald_setup(3, np.eye(3) * 4.0, 1.0, 3.0)
    assert ei.value.status == 5  # EWALD_ECUDA: no fallback path


def test_to_soa_layout():
    pos = np.arange(2 * 5 * 3, dtype=np.float64).reshape(2, 5, 3)
    soa = E.to_soa(pos)
    assert soa.shape == (2, 3, 8)
    assert np.array_equal(soa[1, 2, :5], pos[1, :, 2]) and np.all(soa[:, :, 5:] == 0)


def test_pair_table_matches_erfc():
    """The real-space kernels' table of F(t) = erfc(sqrt t)/sqrt t (built in long double at setup,
    PAPER.md:359) against mpmath.  Bound: |error| <= eps_rel F(t) + eps_abs, so a real-space sum of n
    terms is off by at most eps_rel * sum + n * eps_abs (FP64: 1e-15 and 3e-17 -- the bins widen with t,
    where F ~ exp(-t) is tiny).  Samples include both ends of every bin (bits of t next to the bin
    boundaries) and values below the table, where the direct formula answers."""
    import mpmath as mp
    mp.mp.dps = 30
    rng = np.random.default_rng(0)
    for t_max in (5.72 ** 2, 6.16 ** 2, 42.25):
        edges = []
        for e in range(-6, 6):
            for m in range(0, 128, 5):
                lo = 2.0 ** e * (1 + m / 128)
                edges += [lo, np.nextafter(lo, 0), np.nextafter(lo, 100)]
        t = np.concatenate([np.exp(rng.uniform(np.log(2.0 ** -9), np.log(t_max), 1500)), np.array(edges)])
        t = t[(t > 0) & (t < t_max)]
        want = np.array([float(mp.erfc(mp.sqrt(mp.mpf(float(v)))) / mp.sqrt(mp.mpf(float(v)))) for v in t])
        got64 = E.ewald_pair_table_eval(E.EWALD_F64, t_max, t)
        got32 = E.ewald_pair_table_eval(E.EWALD_F32, t_max, t)
        assert (np.abs(got64 - want) <= 1e-15 * want + 3e-17).all()
        assert (np.abs(got32 - want) <= 6e-8 * want + 1e-9).all()


def _full_sphere_weight_sum(dim, L, kappa, n2_max):
    """sum over 0 < n^2 <= n2_max of w(G), G = 2 pi n / L, with w of DESIGN.md section 2 (cubic / square)."""
    nm = math.isqrt(n2_max)
    rng = range(-nm, nm + 1)
    tot = 0.0
    for n1 in rng:
        for n2 in rng:
            for n3 in (rng if dim == 3 else (0,)):
                m = n1 * n1 + n2 * n2 + n3 * n3
                if m == 0 or m > n2_max:
                    continue
                g = 2 * math.pi / L * math.sqrt(m)
                if dim == 3:
                    tot += 2 * math.pi / L ** 3 * math.exp(-g * g / (4 * kappa * kappa)) / (g * g)
                else:
                    tot += math.pi / L ** 2 * math.erfc(g / (2 * kappa)) / g
    return tot


def test_octant_plan_covers_every_g_once():
    # sum over the octant of w(G_n) 2^nz must equal the full-sphere sum of w(G)
    for idx in range(1, 6):
        w = workloads.config(idx)
        ng = E.ewald_setup_summary(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff)["num_g"]
        for wc in (1, 3, 7):
            o = E.ewald_oct_plan_summary(w.dim, w.cell, w.kappa, w.g_cutoff, wc)
            want = _full_sphere_weight_sum(w.dim, w.L, w.kappa, w.n2_max)
            assert abs(o["weight_sum"] - want) <= 1e-13 * want
            # warps never mix item kinds and are dealt to the four sub-partitions
            assert 4 <= o["npb"] <= 7 and o["n_warps"] >= max(4, -(-wc * o["n_items"] // 32))
            # executed FMA + products per particle can never be below the algorithmic N_G + 1
            assert o["fma_per_particle"] >= ng + 1
        # the tensor-core plan covers the same set: weights, and 64 FMAs per DMMA and particle >= N_G + 1
        m = E.ewald_mma_plan_summary(w.dim, w.cell, w.kappa, w.g_cutoff)
        assert abs(m["weight_sum"] - want) <= 1e-13 * want and m["walkers_per_pass"] >= 1
        assert ng + 1 <= 64 * m["dmma_per_quad"] <= 2.0 * (ng + 1)   # config 1 (n_max = 6): 1.94; config 2: 1.53
        assert (ng + 1) / o["fma_per_particle"] > 0.7    # wc = 7: products + padding cost < 43 % of the algorithmic FMAs (config 1; 22 % on config 2)


def test_octant_plan_any_cell():
    """The octant plan exists for every cell (fractional coordinates); for a triclinic cell the class weights
    still add up to the full-sphere weight sum, computed here from the plain definition over all G."""
    cell = np.array([[4.0, 0, 0], [0, 5.0, 0], [0, 0, 6.5]])
    o = E.ewald_oct_plan_summary(3, cell, 0.9, 5.0, 2)
    assert o["n_items"] > 0
    tri = np.array([[4.0, 0, 0], [1.0, 5.0, 0], [0.3, -0.4, 6.5]])
    kappa, gc = 0.9, 5.0
    o = E.ewald_oct_plan_summary(3, tri, kappa, gc, 2)
    b = 2 * math.pi * np.linalg.inv(tri).T      # rows: reciprocal basis
    vol = abs(np.linalg.det(tri))
    nm = 8
    tot = 0.0
    for n1 in range(-nm, nm + 1):
        for n2 in range(-nm, nm + 1):
            for n3 in range(-nm, nm + 1):
                g = n1 * b[0] + n2 * b[1] + n3 * b[2]
                g2 = float(g @ g)
                if 0 < g2 <= gc * gc * (1 + 1e-12):
                    tot += 2 * math.pi / vol * math.exp(-g2 / (4 * kappa * kappa)) / g2
    assert abs(o["weight_sum"] - tot) <= 1e-13 * tot
