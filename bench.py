#!/usr/bin/env python
"""bench.py -- orbit-library construction throughput (BASELINE.json metric) on N B200s of one node.

    python bench.py --gpus N --steps K --warmup W            # the CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on a bounded sample

A "step" is one full pass of the hot path (integrate + project + bin + flush the dense matrix) over the
workload: by default BASELINE.json configs[1] (20,000 orbits x 10,000 steps, fp64).  With N > 1 every rank
builds its own library from its own seed (weak scaling, no data-path collective: orbits are independent).
Prints ONE JSON line on rank 0.  See DESIGN.md "Measurement" for every field.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "orbit-steps/sec incl. projection+binning"
UNIT = "orbit-steps/s"
# fp64/fp32 arithmetic instructions executed per orbit-step by the integrator for the config-1 potential
# (DFMA/DMUL/DADD resp. FFMA/FMUL/FADD from the ncu capture under profiles/; FMA = 2 flops).  DESIGN.md.
FLOPS_PER_ORBIT_STEP = {"f64": 2 * 330.0, "f32": 2 * 420.0}
FMA_PEAK_DERIVED = {"f64": 148 * 64 * 2 * 1.965e9, "f32": 148 * 128 * 2 * 1.965e9}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default 1)")
    ap.add_argument("--precision", default=None, choices=["f64", "f32"])
    ap.add_argument("--n-orb", type=int, default=None, help="override (profiling only; marks the line reduced)")
    ap.add_argument("--n-steps", type=int, default=None, help="override (profiling only; marks the line reduced)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 5]
        os.unlink(self.f.name)
        if not rows:
            return out
        sm = [float(r[0]) for r in rows if r[0].strip().replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any("Active" in r[2 + i] and "Not" not in r[2 + i] for r in rows)]
        out.update(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=float(rows[0][1]), reasons=reasons, samples=len(rows))
        return out


def workload(args):
    from paper_2607_00117_b200 import inputs
    cfg = dict(inputs.CONFIGS[args.config])
    reduced = False
    if args.n_orb:
        cfg["n_orb"] = args.n_orb; reduced = True
    if args.n_steps:
        cfg["n_steps"] = args.n_steps; reduced = True
    prec = args.precision or ("f32" if cfg["precision"] == "f32" else "f64")
    return cfg, prec, reduced


def oracle_sample(cfg, ics, n_orbits):
    """Time the oracle, as it stands, on the first n_orbits of the workload (all steps). -> (orbit-steps/s, cores, seconds)."""
    from oracle import smo
    t0 = time.perf_counter()
    smo.build_library(cfg["potential"], ics[:n_orbits], cfg["dt"], cfg["n_steps"], cfg["stride"], cfg["projections"], cfg["grids"])
    dt = time.perf_counter() - t0
    return n_orbits * cfg["n_steps"] / dt, smo.num_threads(), dt


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded sample of the same workload, one sample per 'step'."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import smo
    from paper_2607_00117_b200 import inputs
    cfg, prec, reduced = workload(args)
    n_sample = 8 if cfg["ics"] == "disc" else 256
    ics = inputs.make_ics(cfg, lambda p, x: smo.eval_force(p, x, 0.0, want_phi=False), n_orb=max(n_sample, 8))
    for _ in range(args.warmup):
        oracle_sample(cfg, ics, min(2, n_sample))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample(cfg, ics, n_sample)
    el = time.perf_counter() - t0
    val = n_sample * cfg["n_steps"] * args.steps / el
    sample = f"first {n_sample} orbits x {cfg['n_steps']} steps of {cfg['name']} per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg["name"], "sample": sample, "reduced": reduced},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": smo.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import torch.distributed as dist
    from paper_2607_00117_b200 import binding, inputs
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg, prec, reduced = workload(args)
    cfg["seed"] = cfg["seed"] + 1000 * rank  # every rank builds its own library (weak scaling)
    pot = binding.sm_make_potential(cfg["potential"])
    ics_host = inputs.make_ics(cfg, lambda p, x: binding.sm_eval_force(pot, x, 0.0, want_phi=False).cpu().numpy())
    n_orb, n_steps, g = len(ics_host), cfg["n_steps"], cfg["grids"]
    n_proj, nlos, nden = len(cfg["projections"]), g["nx"] * g["ny"] * g["nv"], g["dx"] * g["dy"] * g["dz"]
    out_bytes = 4 * n_orb * (n_proj * nlos + nden)
    free_b, _ = torch.cuda.mem_get_info()
    if out_bytes > 0.8 * free_b:
        raise SystemExit(f"config {args.config} needs a {out_bytes / 1e9:.1f} GB matrix: stream it in orbit chunks (see DESIGN.md); "
                         "choose --config 1 or 2 for the single-call bench")
    ics = torch.as_tensor(ics_host).cuda()
    losvd = torch.empty((n_proj, n_orb, nlos), dtype=torch.float32, device="cuda")
    dens = torch.empty((n_orb, nden), dtype=torch.float32, device="cuda")
    nout = torch.empty((n_proj + 1, n_orb), dtype=torch.int32, device="cuda")

    def step():
        binding.sm_build_library(pot, ics, cfg["dt"], n_steps, cfg["stride"], cfg["projections"], g, precision=prec,
                                 losvd=losvd, dens=dens, nout=nout)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fma_peak = binding.sm_measure_fma_peak(prec)  # also warms the clocks
    binding.sm_set_debug_flags(4)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = binding.sm_launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    kt = {"phase_ms": 0.0, "integrate_ms": 0.0, "rowbuild_ms": 0.0}
    ev[0].record()
    for _ in range(args.steps):
        step()
        for k, v in binding.sm_last_kernel_times().items():  # syncs on the call's own events only
            kt[k] += v
    ev[1].record()
    barrier()
    launches = binding.sm_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = ev[0].elapsed_time(ev[1])
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = t.item()
    value = world * n_orb * n_steps * args.steps / (ms * 1e-3)
    binding.sm_set_debug_flags(0)
    rows_ok = bool(((losvd[0].sum(1) + nout[0]) == n_steps // cfg["stride"]).all().item())

    # binning overhead A/B: integrator alone (recording compiled out) against the full path
    binding.sm_set_debug_flags(1)
    step(); torch.cuda.synchronize()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    e[0].record(); step(); e[1].record(); torch.cuda.synchronize()
    ms_norec = e[0].elapsed_time(e[1])
    binding.sm_set_debug_flags(0)

    # e2e: host buffers in, host buffers out, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        k2 = min(args.steps, 3)
        h_ics = torch.as_tensor(ics_host).pin_memory()
        h_losvd = torch.empty(losvd.shape, dtype=torch.float32).pin_memory()
        h_dens = torch.empty(dens.shape, dtype=torch.float32).pin_memory()
        h_nout = torch.empty(nout.shape, dtype=torch.int32).pin_memory()

        def e2e_step():
            ics.copy_(h_ics, non_blocking=True)
            step()
            h_losvd.copy_(losvd, non_blocking=True); h_dens.copy_(dens, non_blocking=True); h_nout.copy_(nout, non_blocking=True)
        e2e_step(); barrier()
        e[0].record()
        for _ in range(k2):
            e2e_step()
        e[1].record(); barrier()
        t2 = torch.tensor([e[0].elapsed_time(e[1])], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t2, op=dist.ReduceOp.MAX)
        e2e = {"value": world * n_orb * n_steps * k2 / (t2.item() * 1e-3), "unit": UNIT, "steps": k2,
               "h2d_bytes_per_step": int(h_ics.numel() * 8), "d2h_bytes_per_step": int(out_bytes + h_nout.numel() * 4)}
        del h_losvd, h_dens

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    int_ms = kt["integrate_ms"] / args.steps
    flops = FLOPS_PER_ORBIT_STEP[prec] * n_orb * n_steps
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        peaks = {}
    hbm = peaks.get("hbm_gbs", 6650.0)
    row_ms = kt["rowbuild_ms"] / args.steps
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "library_build_ms": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": cfg["name"], "baseline_config_index": args.config, "n_orb_per_gpu": n_orb, "n_steps": n_steps,
                   "stride": cfg["stride"], "n_proj": n_proj, "losvd_bins": nlos, "density_bins": nden, "matrix_bytes": out_bytes,
                   "reduced": reduced, "parallelism": f"orbit-sharded x{world}, no collective",
                   "l2": "each step rewrites the %.2f GB matrix, far larger than the 126 MB L2" % (out_bytes / 1e9)},
        "roofline": {"bound": "alu", "kernel": "integrate_kernel", "achieved": flops / (int_ms * 1e-3) / 1e12, "peak": fma_peak / 1e12,
                     "unit": "TFLOP/s", "frac": flops / (int_ms * 1e-3) / fma_peak, "traffic": None,
                     "peak_kind": f"measured live by sm_measure_fma_peak ({prec} FMA, all SMs)",
                     "peak_derived_tflops": FMA_PEAK_DERIVED[prec] / 1e12, "flops_per_orbit_step": FLOPS_PER_ORBIT_STEP[prec],
                     "kernel_ms": int_ms},
        "flush": {"bound": "hbm", "kernel": "rowbuild_kernel", "achieved": out_bytes / (row_ms * 1e-3) / 1e9 if row_ms else None,
                  "peak": hbm, "unit": "GB/s", "frac": out_bytes / (row_ms * 1e-3) / 1e9 / hbm if row_ms else None,
                  "kernel_ms": row_ms, "peak_kind": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650"},
        "binning_overhead_frac": 1.0 - ms_norec / (ms / args.steps), "integrator_only_ms": ms_norec,
        "row_sums_ok": rows_ok, "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
        "paper_context": "full model construction ~1 s on an A100 (PAPER.md:15), another machine and a different pipeline",
    }
    if not args.no_cpu_baseline:
        # ~10-30 s of oracle work: 64 full-length barred orbits (~1e-4 s per force evaluation per core), or all of config 0
        n_s = min(64 if cfg["ics"] == "disc" else 1000, n_orb)
        v, cores, secs = oracle_sample(cfg, ics_host, n_s)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
                                "sample": f"first {n_s} orbits x {n_steps} steps of {cfg['name']}"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
