#!/usr/bin/env python
"""bench.py -- whole-hot-path throughput on B200 (contract in the task statement).

A "step" is one pass of the hot path over one batch: ewald_energy_batch on all walkers of the workload
(BASELINE.json configs[1]: 3D HEG, N = 250, 1024 walkers, ~2000 G-vectors), i.e. S1-S6 of DESIGN.md.
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle instead (rank 0 only).

  python bench.py --gpus 1 --steps 20 --warmup 3
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
      --master-port P bench.py --gpus N --steps K --warmup W
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2507_02888_b200 import workloads  # noqa: E402

METRIC = "ewald_walker_energies_per_s"
UNIT = "walker-energies/s"
SM_COUNT, FP64_LANES, FP32_LANES = 148, 64, 128   # B200: lanes per SM per clock


def parse():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=20)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--config", type=int, default=2, help="BASELINE.json config index (1-based), 1..4")
    p.add_argument("--prec", default="f64", choices=["f64", "f32"])
    p.add_argument("--no-extras", action="store_true", help="skip FP32 / move / cpu_baseline legs")
    return p.parse_args()


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, reasons, power = [], [], set(), []
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                               c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(smax), samples=len(sm),
                       power_w_max=max(power), reasons=sorted(reasons))
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


def workload_config(w, walkers_per_gpu, l2_note):
    return {"workload": "BASELINE configs[%d]: %s" % (w.index - 1, w.name), "dim": w.dim, "n_particles": w.n,
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

    w = workloads.config(args.config)
    W = w.n_walkers
    npdt, tdt = (np.float64, torch.float64) if args.prec == "f64" else (np.float32, torch.float32)
    pos = w.positions(W * world)[rank * W:(rank + 1) * W]     # every rank its own walkers (weak scaling)
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
    sampler = ClockSampler(local) if rank == 0 else None
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

    # ---- per-kernel device times (CUDA events inside the library, on its launch stream) -----
    E.ewald_profile_enable(ctx, True)
    for _ in range(args.steps):
        flush.zero_()
        step()
    prof = E.ewald_profile_read(ctx)
    E.ewald_profile_enable(ctx, False)
    peaks = measured_peaks()
    sm_max_hz = 1e6 * float(peaks.get("sm_max_mhz", 1965.0))
    lanes = FP64_LANES if args.prec == "f64" else FP32_LANES
    peak_flops = SM_COUNT * lanes * 2 * sm_max_hz      # derived ALU peak
    n_g = E.ewald_num_g(ctx)
    kernels = {}
    for name, (ms, cnt) in prof.items():
        if cnt:
            kernels[name] = {"ms_per_launch": ms / cnt, "launches_per_step": cnt / args.steps}
    step_ms = sum(k["ms_per_launch"] * k["launches_per_step"] for k in kernels.values())
    for k in kernels.values():
        k["share_of_step"] = k["ms_per_launch"] * k["launches_per_step"] / step_ms
    # reciprocal kernel: algorithmic flops = 2 N N_G per walker (1 FMA per particle and G of the full sphere)
    recip_flops = 2.0 * w.n * n_g * W
    kernels["recip"].update(alg_flops_per_launch=recip_flops,
                            achieved_tflops=recip_flops / (kernels["recip"]["ms_per_launch"] * 1e-3) / 1e12,
                            frac_of_peak=recip_flops / (kernels["recip"]["ms_per_launch"] * 1e-3) / peak_flops)
    dominant = max(("recip", "real"), key=lambda k: kernels[k]["share_of_step"])
    roofline = {"kernel": dominant, "bound": "alu", "unit": "TFLOP/s", "peak": peak_flops / 1e12,
                "peak_source": "derived: %d SMs x %d %s lanes x 2 x %.0f MHz (sm_max_mhz)" %
                               (SM_COUNT, lanes, args.prec, sm_max_hz / 1e6),
                "traffic": None}
    if dominant == "recip":
        roofline.update(achieved=kernels["recip"]["achieved_tflops"], frac=kernels["recip"]["frac_of_peak"])
    else:
        roofline.update(achieved=None, frac=None,
                        note="real-space kernel: no algorithmic flop count defined yet for erfc(kappa r)/r")

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
           "config": workload_config(w, W, "flushed between timed steps (256 MiB write); inputs 6 MB"),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
           "kernels": kernels, "wall_s_timed_region": t_wall}

    if rank == 0 and not args.no_extras:
        extras = {}
        try:
            extras["fma_chain_tflops"] = {"f64": E.ewald_probe_fma(ctx, E.EWALD_F64, 2048) / 1e12,
                                          "f32": E.ewald_probe_fma(ctx, E.EWALD_F32, 4096) / 1e12}
        except Exception as ex:  # the probe is informative only
            extras["fma_chain_tflops"] = str(ex)
        out["extras"] = extras
    if rank == 0 and world == 1 and not args.no_extras:
        from oracle import ewald_ref as ref
        cores = ref.max_threads()
        nsamp = min(W, 96)
        t0 = time.perf_counter()
        e_ref, _ = ref.energy_batch(w.dim, w.cell, w.kappa, w.g_cutoff, w.r_cutoff, pos[:nsamp], w.charges,
                                    w.ion_pos, w.ion_q)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": nsamp / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": "first %d of %d walkers of %s, %d OpenMP threads, %.1f s" %
                                         (nsamp, W, w.name, cores, dt)}
        got = d_e.cpu().numpy()[:nsamp]
        out["parity_max_rel_err_vs_oracle"] = float((np.abs(got - e_ref) / np.abs(e_ref)).max())
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
