#!/usr/bin/env python
"""bench.py -- whole-hot-path throughput on B200 (contract in the task statement).

A "step" is one pass of the hot path over one batch: ewald_energy_batch on all walkers of the workload
(BASELINE.json configs[1]: 3D HEG, N = 250, 1024 walkers, ~2000 G-vectors), i.e. S1-S6 of DESIGN.md.
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle instead (rank 0 only).

  python bench.py --gpus 1 --steps 500 --warmup 3
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
      --master-port P bench.py --gpus N --steps K --warmup W
"""
import argparse
import json
import math
import os
import statistics
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2507_02888_b200 import shard, workloads  # noqa: E402

METRIC = "ewald_walker_energies_per_s"
UNIT = "walker-energies/s"
SM_COUNT, FP64_LANES, FP32_LANES = 148, 64, 128   # B200: lanes per SM per clock


def parse():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=500)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--config", type=int, default=2,
                   help="BASELINE.json config index (1-based): 1..4 energies, 5 moves; 6 = NEXT-1 hexagonal cell")
    p.add_argument("--prec", default="f64", choices=["f64", "f32"])
    p.add_argument("--no-extras", action="store_true", help="skip FP32 / move / cpu_baseline legs")
    return p.parse_args()


def recorded_traffic(key, kernel):
    """DRAM bytes per launch from the committed ncu --set full capture (profiles/), or None."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "r02_traffic.json")))[key][kernel]
    except Exception:
        return None


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML from a thread DURING the timed region
    (the recipe's clocks line in B200_PROFILING.md; same counters as its nvidia-smi query)."""

    def __init__(self, torch, cuda_index, period_s=0.01):
        import threading
        self.samples, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            p = torch.cuda.get_device_properties(cuda_index)
            bus = "%08x:%02x:%02x.0" % (p.pci_domain_id, p.pci_bus_id, p.pci_device_id)
            h = pynvml.nvmlDeviceGetHandleByPciBusId(bus.encode())
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            names = {"hw_slowdown": getattr(pynvml, "nvmlClocksEventReasonHwSlowdown", 0x8),
                     "hw_thermal_slowdown": getattr(pynvml, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                     "sw_thermal_slowdown": getattr(pynvml, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                     "sw_power_cap": getattr(pynvml, "nvmlClocksEventReasonSwPowerCap", 0x4)}
            get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons

            def loop():
                while not self._stop.is_set():
                    try:
                        self.samples.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        self.power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
                        r = get_reasons(h)
                        for k, bit in names.items():
                            if r & bit:
                                self.reasons.add(k)
                    except Exception:
                        pass
                    self._stop.wait(period_s)

            self._thread = threading.Thread(target=loop, daemon=True)
            self._thread.start()
        except Exception as ex:  # no NVML: the line says so instead of inventing clocks
            self.error = str(ex)

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        if self._thread is None:
            out["error"] = getattr(self, "error", "NVML unavailable")
            return out
        self._stop.set()
        self._thread.join(timeout=2)
        if self.samples:
            out.update(sm_mhz=statistics.median(self.samples), samples=len(self.samples),
                       power_w_max=max(self.power) if self.power else None, reasons=sorted(self.reasons))
        return out


def run_reference(args, rank):
    """The CPU oracle as it stands, on this arm's config/metric; each step is a bounded sample."""
    if rank != 0:
        return
    from oracle import ewald_ref as ref
    w = workloads.config(args.config)
    cores = ref.max_threads()
    per_step = max(cores, 8)
    pos = w.positions(per_step)

    def step():
        ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos, w.charges, w.ion_pos, w.ion_q)

    for _ in range(min(args.warmup, 1)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = per_step * args.steps / dt
    sample = "%d walkers of %s per step (of %d), all %d host threads" % (per_step, w.name, w.n_walkers, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64(long double sums)",
        "data": "synthetic", "config": workload_config(w, per_step, "n/a (CPU)"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


FAR_T0 = 13.0  # start of the FP32 far shell of the FP64 energy kernel


def count_pair_terms(w, pos):
    """Pairs and pair-image terms (|r_ij - R| < r_c) per walker of an orthorhombic workload, counted with
    numpy on a few walkers: the unit count of the real-space kernel's roofline.
    Returns pairs, terms, terms of the far shell (kappa^2 r^2 >= 13, evaluated in FP32 by the FP64 energy kernel),
    images per axis."""
    sides = np.diag(w.cell)[:w.dim]
    m = int(math.floor(w.r_cutoff / sides.min() + 0.5 - 1e-12))
    shifts = np.array(np.meshgrid(*[np.arange(-m, m + 1)] * w.dim, indexing="ij")).reshape(w.dim, -1).T * sides
    terms, far = [], []
    for p in pos:
        others = [p] if w.ion_pos is None else [p, w.ion_pos]
        cnt = cnt_far = 0
        for k, o in enumerate(others):
            d = p[:, None, :] - o[None, :, :]
            d -= np.rint(d / sides) * sides
            r2 = ((d[:, :, None, :] - shifts[None, None, :, :]) ** 2).sum(-1)
            inside = r2 < w.r_cutoff ** 2
            outer = inside & (r2 * w.kappa ** 2 >= FAR_T0)
            if k == 0:
                iu = np.triu_indices(len(p), 1)
                cnt += int(inside[iu].sum()); cnt_far += int(outer[iu].sum())
            else:
                cnt += int(inside.sum()); cnt_far += int(outer.sum())
        terms.append(cnt); far.append(cnt_far)
    n_ion = 0 if w.ion_pos is None else len(w.ion_pos)
    pairs = w.n * (w.n - 1) // 2 + w.n * n_ion
    return pairs, float(np.mean(terms)), float(np.mean(far)), m


def real_space_work(w, pos, n_images):
    """Algorithmic work of the real-space kernel per walker: pairs, pair-image terms, and a
    flop count in FP64 equivalents -- per pair 12 (displacement and reduction to the cell) + 5 per axis image
    square + 2 per enumerated candidate (20 in 3D with one image per side, else (2M+1)^dim); per near term
    (kappa^2 r^2 < 13) 12 FP64 flops (u, degree-7 polynomial, accumulate); per far term 8 FP32 flops = 4 FP64
    equivalents (the FP64 kernel evaluates the far shell by an FP32 cubic; FP32 peak = 2 x FP64 peak)."""
    n_ion = 0 if w.ion_q is None else len(w.ion_q)
    if np.count_nonzero(w.cell - np.diag(np.diag(w.cell))) == 0:
        pairs, terms, far, m_img = count_pair_terms(w, pos[:4])
        row = 2 * m_img + 1
        n_cand = 20 if (w.dim == 3 and m_img == 1) else row ** w.dim
        per_pair = 12 + 5 * w.dim * row + 2 * n_cand
        flops = per_pair * pairs + 12.0 * (terms - far) + 4.0 * far
        return {"pairs_per_walker": pairs, "pair_image_terms_per_walker": terms, "far_shell_terms_per_walker": far,
                "candidates_per_pair": n_cand, "alg_flops_per_walker_fp64_equiv": flops}
    pairs = w.n * (w.n - 1) // 2 + w.n * n_ion   # general cell: the image list is scanned, terms not counted here
    return {"pairs_per_walker": pairs, "pair_image_terms_per_walker": None, "images_scanned_per_pair": n_images,
            "alg_flops_per_walker_fp64_equiv": (21 + 6 * n_images) * pairs}


def kernel_report(E, ctx, w, pos, prec, W, prof, n_prof, peak_tf):
    """Per-kernel device times (CUDA events inside the library, on its launch stream) and what SURVEY 8(d) asks
    for each kernel: reciprocal = algorithmic 2 N N_G flops per walker over the measured FMA-chain peak;
    real space = pair-image terms/s and FP64-equivalent flops over the same peak."""
    kernels = {}
    for name, (ms, cnt) in prof.items():
        if cnt:
            kernels[name] = {"ms_per_launch": ms / cnt, "launches_per_step": cnt / n_prof}
    step_ms = sum(k["ms_per_launch"] * k["launches_per_step"] for k in kernels.values())
    for k in kernels.values():
        k["share_of_step"] = k["ms_per_launch"] * k["launches_per_step"] / step_ms
    n_g = E.ewald_num_g(ctx)
    recip_flops = 2.0 * w.n * n_g * W
    t_rec = kernels["recip"]["ms_per_launch"] * 1e-3
    kernels["recip"].update(alg_flops_per_launch=recip_flops, achieved_tflops=recip_flops / t_rec / 1e12,
                            frac_of_peak=recip_flops / t_rec / 1e12 / peak_tf)
    work = real_space_work(w, pos, E.ewald_num_images(ctx))
    t_real = kernels["real"]["ms_per_launch"] * 1e-3
    real_flops = work["alg_flops_per_walker_fp64_equiv"] * W * (1.0 if prec == "f64" else 0.5)
    kernels["real"].update(work)
    if work["pair_image_terms_per_walker"] is not None:
        kernels["real"]["pair_image_terms_per_s"] = work["pair_image_terms_per_walker"] * W / t_real
    kernels["real"].update(alg_flops_per_launch=real_flops, achieved_tflops=real_flops / t_real / 1e12,
                           frac_of_peak=real_flops / t_real / 1e12 / peak_tf)
    return kernels


def energy_leg(torch, E, device, stream, idx, prec, steps, flush, peak_tf, n_oracle):
    """One energy workload, device-resident: walker-energies/s (CUDA events per step, L2 flushed in between),
    per-kernel times, and parity of the first n_oracle walkers against the oracle (same inputs as the GPU got)."""
    w = workloads.config(idx)
    W = w.n_walkers
    npdt = np.float64 if prec == "f64" else np.float32
    pos = w.positions(W)
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, device=device, stream=stream)
    if w.ion_pos is not None:
        E.ewald_set_fixed_charges(ctx, w.ion_pos, w.ion_q)
    soa = E.to_soa(pos, npdt)
    d_pos = torch.from_numpy(soa).cuda()
    d_q = torch.from_numpy(w.charges.astype(npdt)).cuda()
    d_e = torch.zeros(W, dtype=torch.float64, device="cuda")
    for _ in range(3):
        E.ewald_energy_batch(ctx, w.n, d_pos, d_q, d_e)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush.zero_()
        a.record()
        E.ewald_energy_batch(ctx, w.n, d_pos, d_q, d_e)
        b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / steps
    n_prof = min(steps, 20)
    E.ewald_profile_enable(ctx, True)
    for _ in range(n_prof):
        flush.zero_()
        E.ewald_energy_batch(ctx, w.n, d_pos, d_q, d_e)
    prof = E.ewald_profile_read(ctx)
    E.ewald_profile_enable(ctx, False)
    kernels = kernel_report(E, ctx, w, pos, prec, W, prof, n_prof, peak_tf)
    out = {"workload": workload_config(w, W, "flushed")["workload"], "dtype": prec, "walkers": W, "value": W / (ms * 1e-3),
           "unit": UNIT, "ms_per_step": ms, "steps": steps,
           "kernels": {k: {kk: v[kk] for kk in ("ms_per_launch", "share_of_step", "frac_of_peak", "achieved_tflops",
                                                "pair_image_terms_per_s") if kk in v} for k, v in kernels.items()}}
    if n_oracle:
        from oracle import ewald_ref as ref
        sample = pos[:n_oracle] if prec == "f64" else pos[:n_oracle].astype(np.float32).astype(np.float64)
        e_ref, _ = ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, sample, w.charges, w.ion_pos, w.ion_q)
        got = d_e.cpu().numpy()[:n_oracle]
        out["parity_max_rel_err_vs_oracle"] = float((np.abs(got - e_ref) / np.abs(e_ref)).max())
        out["parity_walkers"] = int(n_oracle)
    E.ewald_destroy(ctx)
    return out


def jastrow_leg(torch, device, stream, flush, chain_tf, steps=20):
    """u + p Jastrow terms (value, gradient, Laplacian) of all 1024 walkers of
    BASELINE configs[1] per launch; algorithmic flops per walker: p term 14 N N_G (structure
    factor) + 24 N N_G (per-particle derivatives), u term 20 per ordered pair + 80 per pair inside L_u."""
    from oracle import jastrow_ref as jr
    from paper_2507_02888_b200 import ewald as E, jastrow as J
    j = workloads.JastrowWorkload(base_index=2, n_stars=15)
    out = []
    pos = j.positions()
    W, n = pos.shape[0], j.n
    npad = E.ewald_padded_n(n)
    inside = (4.0 / 3.0) * math.pi * j.L_u ** 3 / j.L ** 3
    flops = 38.0 * n * len(j.g_n) + n * (n - 1) * (20.0 + 80.0 * inside)
    k = 4
    t0 = time.perf_counter()
    want = jr.batch(3, j.cell, pos[:k], j.alpha, j.L_u, j.C, j.g_n, j.star, j.a)
    t_or = time.perf_counter() - t0
    for prec in ("f64", "f32"):
        npdt = np.float64 if prec == "f64" else np.float32
        ctx = J.jastrow_setup(3, j.cell, alpha=j.alpha, l_u=j.L_u, c_exp=j.C, g_n=j.g_n, star=j.star, a=j.a,
                              device=device, stream=stream)
        d_pos = torch.from_numpy(E.to_soa(pos, npdt)).cuda()
        val = torch.zeros(W, dtype=torch.float64, device="cuda")
        grad = torch.zeros((W, 3, npad), dtype=torch.float64, device="cuda")
        lap = torch.zeros((W, npad), dtype=torch.float64, device="cuda")
        for _ in range(3):
            J.jastrow_batch(ctx, n, d_pos, val, grad, lap)
        J.jastrow_profile_enable(ctx, True)
        for _ in range(steps):
            flush.zero_()
            J.jastrow_batch(ctx, n, d_pos, val, grad, lap)
        ms, cnt = J.jastrow_profile_read(ctx)
        t = ms / cnt * 1e-3
        g = grad.cpu().numpy()[:k, :, :n].transpose(0, 2, 1)
        err = max(float((np.abs(val.cpu().numpy()[:k] - want[0]) / np.abs(want[0])).max()),
                  float((np.abs(g - want[1]).max(axis=(1, 2)) / np.abs(want[1]).max(axis=(1, 2))).max()),
                  float((np.abs(lap.cpu().numpy()[:k, :n] - want[2]).max(axis=1) / np.abs(want[2]).max(axis=1)).max()))
        peak = chain_tf[prec]
        out.append({"workload": "u + p Jastrow terms on BASELINE configs[1] (N = 250, 1024 walkers, %d stars / %d G, N_u = %d)"
                                % (j.n_stars, len(j.g_n), len(j.alpha) - 1), "dtype": prec,
                    "walker_evaluations_per_s": W / t, "ms_per_launch": t * 1e3,
                    "roofline": {"kernel": "jastrow", "bound": "alu", "unit": "TFLOP/s", "achieved": flops * W / t / 1e12,
                                 "peak": peak, "frac": flops * W / t / 1e12 / peak, "alg_flops_per_walker": flops,
                                 "traffic": None},
                    "parity_max_rel_err_vs_oracle": err, "parity_walkers": k, "parity_inputs": "oracle on the FP64 positions",
                    "cpu_baseline": {"value": k / t_or, "unit": "walker-evaluations/s", "kind": "oracle (pair by pair, O(N^2 N_G))",
                                     "cores": jr._load().jastrow_ref_max_threads(), "sample": "%d walkers, %.1f s" % (k, t_or)}})
        J.jastrow_destroy(ctx)
    return out


def blip_leg(torch, device, stream, flush, hbm_gbs, steps=10):
    """125 blip orbitals (24^3 grid) at the 256 000 electron positions of the 1024 walkers of
    BASELINE configs[1] per launch: value, gradient, Laplacian.  Algorithmic bytes per position: the gather of
    64 x n_orb coefficients (served by L2: the table is 14 MB in FP64) + the 5 n_orb doubles written to HBM."""
    from oracle import blip_ref as br
    from paper_2507_02888_b200 import blip as B
    wl = workloads.BlipWorkload()
    pts = wl.points()
    P = len(pts)
    npad = (P + 3) & ~3
    k = 32
    t0 = time.perf_counter()
    want = br.evaluate(wl.cell, wl.coef, pts[:k])
    t_or = time.perf_counter() - t0
    out = []
    for prec in ("f64", "f32"):
        npdt, es = (np.float64, 8) if prec == "f64" else (np.float32, 4)
        ctx = B.blip_setup(wl.cell, wl.coef, device=device, stream=stream)
        soa = np.zeros((3, npad), dtype=npdt)
        soa[:, :P] = pts.T
        d_pts = torch.from_numpy(soa).cuda()
        psi = torch.zeros((P, wl.n_orb), dtype=torch.float64, device="cuda")
        grad = torch.zeros((P, 3, wl.n_orb), dtype=torch.float64, device="cuda")
        lap = torch.zeros((P, wl.n_orb), dtype=torch.float64, device="cuda")
        for _ in range(2):
            B.blip_eval_batch(ctx, P, d_pts, psi, grad, lap)
        B.blip_profile_enable(ctx, True)
        for _ in range(steps):
            flush.zero_()
            B.blip_eval_batch(ctx, P, d_pts, psi, grad, lap)
        ms, cnt = B.blip_profile_read(ctx)
        t = ms / cnt * 1e-3
        got = (psi[:k].cpu().numpy(), grad[:k].cpu().numpy(), lap[:k].cpu().numpy())
        err = max(float((np.abs(g - w_).reshape(k, -1).max(axis=1) / np.abs(w_).reshape(k, -1).max(axis=1)).max())
                  for g, w_ in zip(got, want))
        gather = 64.0 * wl.n_orb * es * P
        written = 5.0 * wl.n_orb * 8 * P
        out.append({"workload": "%d blip orbitals on a %dx%dx%d grid at %d positions (1024 walkers x 250 electrons)"
                                % ((wl.n_orb,) + tuple(wl.grid) + (P,)), "dtype": prec,
                    "orbital_evaluations_per_s": P * wl.n_orb / t, "ms_per_launch": t * 1e3,
                    "roofline": {"kernel": "blip", "bound": "hbm", "unit": "GB/s", "achieved": written / t / 1e9,
                                 "peak": hbm_gbs, "frac": written / t / 1e9 / hbm_gbs,
                                 "alg_bytes_written_per_launch": written, "l2_gather_bytes_per_launch": gather,
                                 "l2_gather_gbs": gather / t / 1e9, "traffic": None,
                                 "note": "HBM: the outputs (5 doubles per position and orbital); the coefficient gather is "
                                         "served by L2"},
                    "achieved_tflops": 10.0 * 64 * wl.n_orb * P / t / 1e12,
                    "parity_max_rel_err_vs_oracle": err, "parity_positions": k,
                    "cpu_baseline": {"value": k * wl.n_orb / t_or, "unit": "orbital-evaluations/s", "kind": "oracle (every grid point)",
                                     "cores": "OpenMP", "sample": "%d positions, %.1f s" % (k, t_or)}})
        B.blip_destroy(ctx)
    return out


def move_leg(torch, E, device, stream, prec, n_steps, flush, hbm_peak_gbs):
    """BASELINE configs[4]: 3D HEG N = 1000, 4096 walkers with stored rho(G); each step moves one seeded-random
    electron per walker by a Gaussian step (reading R14), always committed.  Returns moves/s (device-resident,
    CUDA events around each batch of 4096 moves, L2 flushed in between) and the HBM roofline of the move kernel:
    algorithmic bytes per move = read + write of rho(G+) (2 x N_G+ complex) + one read of the walker's
    positions."""
    w = workloads.config(5)
    npdt, tdt = (np.float64, torch.float64) if prec == "f64" else (np.float32, torch.float32)
    es = 8 if prec == "f64" else 4
    W, S = w.n_walkers, min(n_steps, w.n_steps)
    pos0 = w.positions(W)
    electron, disp = w.moves(W, S)
    cur = pos0.copy()
    new_r = np.zeros((S, W, w.dim))
    ar = np.arange(W)
    for s_ in range(S):
        new_r[s_] = cur[ar, electron[s_]] + disp[s_]
        cur[ar, electron[s_]] = new_r[s_]
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, device=device, stream=stream)
    E.ewald_load_walkers(ctx, w.n, torch.from_numpy(E.to_soa(pos0, npdt)).cuda(),
                         torch.from_numpy(w.charges.astype(npdt)).cuda())
    d_w = torch.arange(W, dtype=torch.int32, device="cuda")
    d_el = torch.from_numpy(electron).cuda()
    d_r = torch.from_numpy(new_r.astype(npdt)).cuda()
    d_de = torch.zeros((S, W), dtype=torch.float64, device="cuda")
    warm = min(3, S // 2)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(S)]
    for s_ in range(S):
        flush.zero_()
        ev[s_][0].record()
        E.ewald_move_delta_batch(ctx, d_w, d_el[s_], d_r[s_], 1, d_de[s_])
        ev[s_][1].record()
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in ev][warm:]
    t = sum(ms) * 1e-3 / len(ms)
    ngp = E.ewald_num_g(ctx) // 2
    bytes_per_move = 2 * ngp * 2 * es + w.dim * w.n * es
    gbs = bytes_per_move * W / t / 1e9
    E.ewald_destroy(ctx)
    # parity of the timed moves themselves: the chains of the first 4 walkers against the oracle (reading R12)
    from oracle import ewald_ref as ref
    k = 4
    r32 = (lambda a: a) if prec == "f64" else (lambda a: a.astype(np.float32).astype(np.float64))
    de_ref, _, _ = ref.move_chain(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, r32(pos0[:k]), w.charges,
                                  electron[:, :k], r32(new_r[:, :k]))
    de = d_de.cpu().numpy()[:, :k]
    rms = np.sqrt((de_ref ** 2).mean(axis=1, keepdims=True))
    parity = float((np.abs(de - de_ref) / np.maximum(np.abs(de_ref), rms)).max())
    return {"workload": "BASELINE configs[4]: %s" % w.name, "dtype": prec, "moves_per_s": W / t,
            "ms_per_batch_of_%d_moves" % W: t * 1e3, "timed_batches": len(ms), "warmup_batches": warm,
            "roofline": {"kernel": "move", "bound": "hbm", "unit": "GB/s", "achieved": gbs, "peak": hbm_peak_gbs,
                         "frac": gbs / hbm_peak_gbs, "alg_bytes_per_move": bytes_per_move,
                         "alg_bytes_per_launch": bytes_per_move * W,
                         "traffic": recorded_traffic("cfg5_%s" % prec, "move")},
            "delta_e_finite": bool(torch.isfinite(d_de).all().item()),
            "parity_max_err_vs_oracle_R12": parity, "parity_walkers": k, "parity_steps": S}


def workload_config(w, walkers_per_gpu, l2_note):
    label = "BASELINE configs[%d]" % (w.index - 1) if w.index <= 5 else "SURVEY 8(f) NEXT-1"
    return {"workload": "%s: %s" % (label, w.name), "dim": w.dim, "n_particles": w.n,
            "n_fixed": 0 if w.ion_q is None else len(w.ion_q), "walkers_per_gpu": walkers_per_gpu,
            "kappa_L": round(w.kappa * w.L, 6), "n2_max": w.n2_max, "r_cutoff_over_L": round(w.r_cutoff / w.L, 6),
            "l2": l2_note, "parallelism": "walkers sharded across GPUs, no data-path collective"}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2507_02888_b200 import ewald as E

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    if args.config == 5:   # the single-move metric alone (used for profiling; the default run reports it in extras)
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
        r = move_leg(torch, E, local, torch.cuda.current_stream().cuda_stream, args.prec, args.steps, flush,
                     float(measured_peaks().get("hbm_gbs", 6542.1)))
        if rank == 0:
            print(json.dumps({"metric": "single_move_delta_e_per_s", "value": r["moves_per_s"] * world,
                              "unit": "moves/s", "n_gpus": world, "steps": r["timed_batches"],
                              "warmup": r["warmup_batches"], "ms_per_step": r["ms_per_batch_of_4096_moves"],
                              "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.prec,
                              "data": "synthetic", "config": {"workload": r["workload"]}, "roofline": r["roofline"]}))
        if world > 1:
            dist.destroy_process_group()
        return

    w = workloads.config(args.config)
    W = w.n_walkers
    npdt, tdt = (np.float64, torch.float64) if args.prec == "f64" else (np.float32, torch.float32)
    lo, hi = shard.walker_range(W * world, rank, world)       # every rank its own W walkers (weak scaling)
    pos = w.positions(W * world)[lo:hi]
    stream = torch.cuda.current_stream().cuda_stream
    ctx = E.ewald_setup(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, device=local, stream=stream)
    if w.ion_pos is not None:
        E.ewald_set_fixed_charges(ctx, w.ion_pos, w.ion_q)
    soa = E.to_soa(pos, npdt)
    q_np = w.charges.astype(npdt)
    d_pos, d_q = torch.from_numpy(soa).cuda(), torch.from_numpy(q_np).cuda()
    d_e = torch.zeros(W, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def step():
        E.ewald_energy_batch(ctx, w.n, d_pos, d_q, d_e)

    # ---- device-resident throughput -------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(torch, local) if rank == 0 else None
    lc0 = E.ewald_launch_count(ctx)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()            # L2 flush between timed iterations (outside the event pair)
        a.record()
        step()
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = E.ewald_launch_count(ctx) - lc0
    ms_total = max_over_ranks(sum(a.elapsed_time(b) for a, b in ev))
    clocks = sampler.stop() if sampler else None
    value = W * world * args.steps / (ms_total * 1e-3)

    # ---- end to end through the host-buffer entry point ------------------------------------
    h_pos = torch.from_numpy(soa).pin_memory()
    h_q = torch.from_numpy(q_np).pin_memory()
    h_e = torch.zeros(W, dtype=torch.float64).pin_memory()
    for _ in range(2):
        E.ewald_energy_batch_host(ctx, w.n, h_pos.numpy(), h_q.numpy(), h_e.numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        E.ewald_energy_batch_host(ctx, w.n, h_pos.numpy(), h_q.numpy(), h_e.numpy())
    barrier()
    t_e2e = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": W * world * args.steps / t_e2e, "unit": UNIT,
           "h2d_bytes_per_step": int(h_pos.numel() * h_pos.element_size() + h_q.numel() * h_q.element_size()),
           "d2h_bytes_per_step": int(h_e.numel() * 8)}
    assert np.array_equal(h_e.numpy(), d_e.cpu().numpy())

    # ---- roofline denominators measured in this run: FMA-chain (and DMMA) probes of the library ----------
    peaks = measured_peaks()
    chain = {"f64": E.ewald_probe_fma(ctx, E.EWALD_F64, 2048) / 1e12, "f32": E.ewald_probe_fma(ctx, E.EWALD_F32, 4096) / 1e12}
    dmma_tf = E.ewald_probe_dmma(ctx, 2048) / 1e12
    peak_tf = chain[args.prec]

    # ---- per-kernel device times (CUDA events inside the library, on its launch stream) -----
    n_prof = min(args.steps, 50)
    E.ewald_profile_enable(ctx, True)
    for _ in range(n_prof):
        flush.zero_()
        step()
    prof = E.ewald_profile_read(ctx)
    E.ewald_profile_enable(ctx, False)
    kernels = kernel_report(E, ctx, w, pos, args.prec, W, prof, n_prof, peak_tf)
    dominant = max(("recip", "real"), key=lambda k: kernels[k]["share_of_step"])
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    lanes = FP64_LANES if args.prec == "f64" else FP32_LANES
    roofline = {"kernel": dominant, "bound": "alu", "unit": "TFLOP/s", "peak": peak_tf,
                "peak_source": "measured in this run: %s FMA-chain probe of the library (ewald_probe_fma); derived "
                               "%d SMs x %d lanes x 2 x %.0f MHz = %.2f; FP64 tensor (DMMA) probe %.2f"
                               % (args.prec, SM_COUNT, lanes, sm_max_mhz, SM_COUNT * lanes * 2 * sm_max_mhz * 1e-6, dmma_tf),
                "achieved": kernels[dominant]["achieved_tflops"], "frac": kernels[dominant]["frac_of_peak"],
                "traffic": recorded_traffic("cfg%d_%s" % (args.config, args.prec), dominant),
                "traffic_note": "DRAM bytes per launch (ncu --set full, profiles/r02_traffic.json); algorithmic: the "
                                "positions once = %d bytes" % (soa.nbytes),
                "note": "real-space kernel: FP64-equivalent algorithmic flops (DESIGN.md section 6: enumerated candidates, "
                        "near terms FP64, far-shell terms FP32 at half weight); it is limited by shared-memory "
                        "wavefronts, see profiles/ and kernels.real.pair_image_terms_per_s"}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
           "config": workload_config(w, W, "flushed between timed steps (256 MiB write); inputs 6 MB"),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
           "kernels": kernels, "wall_s_timed_region": t_wall}

    if rank == 0 and not args.no_extras:
        extras = {"fma_chain_tflops": chain, "dmma_tflops": dmma_tf}
        # the other precision of the same workload (BASELINE configs[1] is quoted in FP64 and FP32)
        other = "f32" if args.prec == "f64" else "f64"
        o_np, o_t = (np.float32, torch.float32) if other == "f32" else (np.float64, torch.float64)
        o_pos = torch.from_numpy(E.to_soa(pos, o_np)).cuda()
        o_q = torch.from_numpy(w.charges.astype(o_np)).cuda()
        o_e = torch.zeros(W, dtype=torch.float64, device="cuda")
        for _ in range(3):
            E.ewald_energy_batch(ctx, w.n, o_pos, o_q, o_e)
        oev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
        for a, b in oev:
            flush.zero_()
            a.record()
            E.ewald_energy_batch(ctx, w.n, o_pos, o_q, o_e)
            b.record()
        torch.cuda.synchronize()
        o_ms = sum(a.elapsed_time(b) for a, b in oev) / len(oev)
        extras["energy_other_precision"] = {"dtype": other, "value": W / (o_ms * 1e-3), "unit": UNIT,
                                            "ms_per_step": o_ms}
        # single-move Delta-E/s (BASELINE.json's second metric), both precisions
        hbm = float(peaks.get("hbm_gbs", 6542.1))
        extras["single_move"] = [move_leg(torch, E, local, stream, p, 100, flush, hbm) for p in ("f64", "f32")]
        # the other workloads of BASELINE.json (configs 1, 3, 4) and SURVEY 8(f) NEXT-1 (config 6), short runs
        extras["per_config"] = [energy_leg(torch, E, local, stream, idx, p, 30, flush, chain[p], n_or)
                                for idx, p, n_or in ((1, "f64", 8), (3, "f64", 16), (3, "f32", 16), (4, "f64", 16),
                                                     (6, "f64", 2))]
        # SURVEY 8(f) NEXT-2/3 (Jastrow u and p terms) and NEXT-4 (blip orbitals), each with parity and its roofline
        extras["next"] = {"jastrow": jastrow_leg(torch, local, stream, flush, chain),
                          "blip": blip_leg(torch, local, stream, flush, hbm)}
        out["extras"] = extras
    if rank == 0 and world == 1 and not args.no_extras:
        from oracle import ewald_ref as ref
        cores = ref.max_threads()
        t0 = time.perf_counter()   # size the sample for about 12 s of oracle time
        ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos[:cores], w.charges, w.ion_pos, w.ion_q)
        dt0 = time.perf_counter() - t0
        want = cores * max(1, round(12.0 / max(dt0, 1e-3)))     # walkers worth 12 s
        nsamp = int(min(W, want))
        passes, dt = 0, 0.0                                       # a small workload is evaluated several times
        while passes < 8 and dt < 10.0:
            t0 = time.perf_counter()
            e_ref, _ = ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos[:nsamp], w.charges,
                                        w.ion_pos, w.ion_q)
            dt += time.perf_counter() - t0
            passes += 1
        out["cpu_baseline"] = {"value": nsamp * passes / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": "first %d of %d walkers of %s, %d pass(es), %d OpenMP threads, %.1f s" %
                                         (nsamp, W, w.name, passes, cores, dt)}
        got = d_e.cpu().numpy()[:nsamp]
        out["parity_max_rel_err_vs_oracle"] = float((np.abs(got - e_ref) / np.abs(e_ref)).max())
        out["parity_sample_min_abs_energy"] = float(np.abs(e_ref).min())  # a walker with E ~ 0 inflates the line above
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
