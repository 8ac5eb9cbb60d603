#!/usr/bin/env python
"""bench.py -- orbit-library construction throughput (BASELINE.json metric) on N B200s of one node.

    python bench.py --gpus N --steps K --warmup W            # the CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on a bounded sample

A "step" is one full pass of the hot path (integrate + project + bin + flush the dense matrix) over the
workload: by default BASELINE.json configs[2] (100,000 orbits x 20,000 steps, fp64, 70.7 GB matrix: "timed as the full
library build", the largest configuration that fits one GPU); the default run adds compact sub-records of the other four
configs and of config 2 in fp32.  Workloads whose matrix exceeds HBM (configs 3, 4) are streamed through a ring of dense
chunk buffers: every row is still written.
With N > 1 every rank builds its own library from its own seed (weak scaling, no data-path collective:
orbits are independent).  Prints ONE JSON line on rank 0.  See DESIGN.md "Measurement" for every field.
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
# Executed floating-point operations per orbit-step and thread of the integrator kernels, and their DRAM bytes per launch, come
# from the committed ncu captures of the CURRENT kernels: profiles/kernel_counts.json, written by
# `python -m paper_2607_00117_b200.ncu_summary` from the .ncu-rep (smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd,ffma,fmul,fadd}_pred_on).
# tests/test_library_host.py fails when the kernel sources have changed since the capture.  Only the operations of the kernel's
# own arithmetic type count against that type's FMA peak (the fp64 kernel's fp32 lambda iteration does not).


def kernel_counts(key):
    """-> (flop per orbit-step, dram bytes per launch, orbit-steps of the profiled launch, source csv) or (None, ...) if not captured."""
    try:
        c = json.load(open(os.path.join(ROOT, "profiles", "kernel_counts.json")))[key]
    except (OSError, KeyError, ValueError):
        return None, None, None, None
    o = c["per_orbit_step"]
    flop = 2 * o["dfma"] + o["dmul"] + o["dadd"] if key.endswith("f64") else 2 * o["ffma"] + o["fmul"] + o["fadd"]
    return flop, c["dram_bytes_per_launch"], c["orbit_steps_per_launch"], c["source"]


FMA_PEAK_DERIVED = {"f64": 148 * 64 * 2 * 1.965e9, "f32": 148 * 128 * 2 * 1.965e9}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2: the library-scale build, the largest configuration whose matrix fits one GPU)")
    ap.add_argument("--precision", default=None, choices=["f64", "f32"])
    ap.add_argument("--n-orb", type=int, default=None, help="override (profiling only; marks the line reduced)")
    ap.add_argument("--n-steps", type=int, default=None, help="override (profiling only; marks the line reduced)")
    ap.add_argument("--n-trials", type=int, default=None, help="override for config 3 (marks the line reduced)")
    ap.add_argument("--chunk-gb", type=float, default=40.0, help="largest dense chunk buffer (GB)")
    ap.add_argument("--bundle", type=int, default=1, help="co-add this many consecutive orbits per row (sm_build_bundled_library)")
    ap.add_argument("--fourfold", action="store_true", help="fourfold symmetrisation of PAPER.md Table 1 (sm_build_bundled_library)")
    ap.add_argument("--apertures", type=int, default=0, help="regroup image pixels into this many synthetic apertures (sm_build_observable_library)")
    ap.add_argument("--gh", action="store_true", help="Gauss-Hermite sums per aperture instead of the v_los histogram (needs --apertures; sm_build_gh_library)")
    ap.add_argument("--bar", default="ferrers", choices=["ferrers", "dehnen"], help="dehnen: the paper's own stellar model in place of configs[1]'s Ferrers bar: "
                    "Miyamoto-Nagai disc + Dehnen & Aly T_3 long bar + V_4 bulge + NFW (PAPER.md:196-237, inputs.paper_bar_potential); single-potential configs")
    ap.add_argument("--cylindrical", action="store_true", help="the paper's 600 density cells uniform in (R, phi, z), R < 10, |z| < 3 kpc (PAPER.md:106,260)")
    ap.add_argument("--weights", action="store_true", help="time the weight solve (sm_solve_weights, PAPER.md:118-136) on a paper-sized "
                    "synthetic system instead of the library build: --n-orb rows (default 7500 = 30 000 ICs in bundles of 4), 600 "
                    "density cells, --apertures (default 600), --w-rhs bootstrap realisations, --w-iter ADMM iterations")
    ap.add_argument("--model", action="store_true", help="time one model chi^2 evaluation of the paper's shape end to end (PAPER.md:262): "
                    "Gauss-Hermite library of 30 000 ICs x 5 000 steps in symmetrised bundles of 4, 600 apertures, 600 cylindrical "
                    "density cells -> sm_solve_weights on that library in place (--w-rhs realisations, --w-iter iterations) -> Eq. 5-6")
    ap.add_argument("--rk32", action="store_true", help="time the library build with the paper's own integrator (sm_build_library_rk32: adaptive "
                    "Bogacki-Shampine RK3(2) in the rotating frame, rtol 1e-4, delta-t-weighted rows; PAPER.md:75,104) on the chosen config's "
                    "orbits, grids and potential; --n-steps = step attempts per orbit (default 5000, the paper's)")
    ap.add_argument("--w-rhs", type=int, default=100)
    ap.add_argument("--w-iter", type=int, default=500)
    ap.add_argument("--w-dens", type=int, default=600)
    ap.add_argument("--debug-flags", type=lambda v: int(v, 0), default=0, help="A/B only: OR these sm_set_debug_flags bits (include/schwarmax.h) into "
                    "every call the run makes, e.g. 32768 = zero fill by the paced store loop instead of the bulk-copy engine")
    ap.add_argument("--zero-fill", type=float, default=0.0, metavar="GB", help="A/B only: time sm_zero_async alone on a buffer of this many GB and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sub", action="store_true", help="skip the compact sub-records of the other configs (default run only)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
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
    if args.n_trials and "n_trials" in cfg:
        cfg["n_trials"] = args.n_trials; reduced = True
    prec = args.precision or ("f32" if cfg["precision"] == "f32" else "f64")
    if args.bar == "dehnen":
        if cfg["ics"] != "disc" or "n_trials" in cfg:
            raise SystemExit("--bar dehnen needs a single-potential disc config (1, 2 or 4)")
        cfg["potential"] = inputs.paper_bar_potential()
        cfg["name"] += "_paperbar"
    if args.cylindrical:
        cfg["grids"] = dict(cfg["grids"], dx=10, dy=12, dz=5, bx0=0.0, bx1=10.0, by0=0.0, by1=2 * np.pi, bz0=-3.0, bz1=3.0)
    return cfg, prec, reduced


def oracle_sample(cfg, ics, n_orbits, bundle=1, fourfold=False, ap=None, dens_mode=0, gh=None):
    """Time the oracle, as it stands, on the first n_orbits of the workload (all steps). -> (orbit-steps/s, cores, seconds)."""
    from oracle import smo
    t0 = time.perf_counter()
    if gh is not None:
        smo.build_gh_library(cfg["potential"], ics[:n_orbits], cfg["dt"], cfg["n_steps"], cfg["stride"], cfg["projections"],
                             cfg["grids"], ap[0], ap[1], gh[0], gh[1], n_bundle=bundle, fourfold=fourfold, density_mode=dens_mode)
    elif ap is not None or dens_mode:
        ap = ap or (None, 0)
        smo.build_observable_library(cfg["potential"], ics[:n_orbits], cfg["dt"], cfg["n_steps"], cfg["stride"], cfg["projections"],
                                     cfg["grids"], ap[0], ap[1], n_bundle=bundle, fourfold=fourfold, density_mode=dens_mode)
    elif bundle > 1 or fourfold:
        smo.build_bundled_library(cfg["potential"], ics[:n_orbits], cfg["dt"], cfg["n_steps"], cfg["stride"], cfg["projections"],
                                  cfg["grids"], n_bundle=bundle, fourfold=fourfold)
    else:
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
    # one orbit per host thread at least (OpenMP over orbits), so that no core idles: ~1e-4 s per force evaluation per core keeps
    # K+W samples of that many full-length barred orbits (or 256 Plummer orbits) within minutes
    n_sample = max(8, smo.num_threads()) if cfg["ics"] == "disc" else 256
    n_sample -= n_sample % args.bundle
    ics = inputs.make_ics(cfg, lambda p, x: smo.eval_force(p, x, 0.0, want_phi=False), n_orb=max(n_sample, 8))
    for _ in range(args.warmup):
        oracle_sample(cfg, ics, args.bundle * max(1, 2 // args.bundle), args.bundle, args.fourfold)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample(cfg, ics, n_sample, args.bundle, args.fourfold)
    el = time.perf_counter() - t0
    val = n_sample * cfg["n_steps"] * args.steps / el
    sample = f"first {n_sample} orbits x {cfg['n_steps']} steps of {cfg['name']} per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg["name"], "sample": sample, "reduced": reduced},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": smo.num_threads(), "kind": "oracle", "sample": sample,
                         "note": "the parity oracle as it stands: every force in software __float128, OpenMP over orbits"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


class Runner:
    """One rank's workload: potential(s), resident ICs, a ring of dense chunk buffers, and the pass over all chunks."""

    def __init__(self, args, cfg, prec, rank):
        import torch
        from paper_2607_00117_b200 import binding, inputs, shard
        self.torch, self.binding, self.cfg, self.prec = torch, binding, cfg, prec
        cfg["seed"] = shard.rank_seed(cfg["seed"], rank)  # every rank builds its own library (weak scaling)
        g = cfg["grids"]
        self.n_proj = len(cfg["projections"])
        self.nlos, self.nden = g["nx"] * g["ny"] * g["nv"], g["dx"] * g["dy"] * g["dz"]
        self.n_orb, self.n_steps = cfg["n_orb"], cfg["n_steps"]
        self.batch = "n_trials" in cfg
        self.n_trials = cfg.get("n_trials", 1)
        self.bundle, self.fourfold = args.bundle, args.fourfold
        self.bundled = args.bundle > 1 or args.fourfold or args.apertures > 0 or args.cylindrical
        self.dens_mode = 1 if args.cylindrical else 0
        self.n_ap, self.ap_map = args.apertures, None
        if self.n_ap:
            self.ap_host = inputs.aperture_map(g, self.n_ap, cfg["seed"])
            self.ap_map = torch.as_tensor(self.ap_host).cuda()
            self.nlos = self.n_ap * g["nv"]
        self.gh = args.gh
        if self.gh:
            if not self.n_ap:
                raise SystemExit("--gh needs --apertures")
            rng = np.random.default_rng(cfg["seed"] + 7)   # stand-ins for the observed mean and dispersion of each aperture
            self.gh_v0_host, self.gh_s_host = rng.normal(0.0, 60.0, self.n_ap), rng.uniform(70.0, 160.0, self.n_ap)
            self.gh_v0, self.gh_s = torch.as_tensor(self.gh_v0_host).cuda(), torch.as_tensor(self.gh_s_host).cuda()
            self.nlos = self.n_ap * 6
        if self.bundled and self.n_orb % self.bundle:
            raise SystemExit("--bundle/--fourfold need n_orb divisible by the bundle size")
        dev_force = lambda pot: (lambda p, x: binding.sm_eval_force(pot, x, 0.0, want_phi=False).cpu().numpy())
        if self.batch:
            draws = inputs.trial_draws(self.n_trials, cfg["seed"])
            self.pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
            self.projs = [[d["projection"]] for d in draws]
            ics = []
            for t, d in enumerate(draws):  # common random numbers, each trial's own v_c (R11)
                ff = lambda p, x, t=t: binding.sm_eval_force(self.pot, x, 0.0, trial=t, want_phi=False).cpu().numpy()
                ics.append(inputs.make_ics(cfg, ff, potential=d["potential"]))
            self.ics_host = np.stack(ics)
        else:
            self.pot = binding.sm_make_potential(cfg["potential"])
            self.ics_host = inputs.make_ics(cfg, dev_force(self.pot))
        self.row_bytes = 4 * (self.n_proj * self.nlos + self.nden)
        self.unit_bytes = self.row_bytes * (self.n_orb // self.bundle if self.batch else 1)   # bytes per chunkable unit (trial / row)
        self.n_units = self.n_trials if self.batch else self.n_orb // self.bundle   # rows = bundles
        self.matrix_bytes = self.unit_bytes * self.n_units
        self.ics = torch.as_tensor(self.ics_host).cuda()
        free_b, _ = torch.cuda.mem_get_info()
        if self.matrix_bytes <= 0.75 * free_b:
            self.set_chunk(self.n_units, 1)
        else:
            per = max(1, int(min(args.chunk_gb * 1e9, 0.35 * free_b) // self.unit_bytes))
            if not self.batch and per >= 512:
                per = per // 512 * 512
            if self.bundled:
                raise SystemExit("--bundle/--fourfold: the matrix must fit one buffer")
            per = min(per, self.n_units)
            # three ring buffers where they fit beside the two staging buffers (<= ~6 GB each): one more window zeroed ahead of its scatter
            self.set_chunk(per, 3 if 3 * per * self.unit_bytes + 14e9 < 0.85 * free_b else 2)

    def set_chunk(self, per, ring):
        torch = self.torch
        self.per, self.ring = per, ring
        self.batches = None
        self.stage_bufs = None
        self.chunks = [(a, min(a + per, self.n_units)) for a in range(0, self.n_units, per)]
        self.bufs = None
        torch.cuda.empty_cache()
        lead = (per,) if self.batch else ()
        n_o = self.n_orb // self.bundle if self.batch else per
        self.bufs = [dict(losvd=torch.empty(lead + (self.n_proj, n_o, self.nlos), dtype=torch.float32, device="cuda"),
                          dens=torch.empty(lead + (n_o, self.nden), dtype=torch.float32, device="cuda"),
                          nout=torch.empty(lead + (self.n_proj + 1, n_o), dtype=torch.int32, device="cuda")) for _ in range(ring)]

    def build(self, c, buf, ics=None):
        a, b = self.chunks[c]
        cfg, bd = self.cfg, self.binding
        n = b - a
        if self.batch and self.bundled:   # the paper's row forms for a range of trials in one launch
            out = dict(dens=buf["dens"][:n], nout=buf["nout"][:n])
            out["gh" if self.gh else "losvd"] = buf["losvd"][:n].view(n, self.n_proj, -1, self.n_ap, 6) if self.gh else buf["losvd"][:n]
            bd.sm_build_observable_library_batch(self.pot, (self.ics if ics is None else ics)[a:b], cfg["dt"], self.n_steps, cfg["stride"],
                                                 self.projs[a:b], cfg["grids"], self.ap_map, self.n_ap, n_bundle=self.bundle,
                                                 fourfold=self.fourfold, precision=self.prec, density_mode=self.dens_mode,
                                                 gh=(self.gh_v0, self.gh_s) if self.gh else None, trial0=a, n_trials=n, out=out)
        elif self.batch:
            bd.sm_build_library_batch(self.pot, (self.ics if ics is None else ics)[a:b], cfg["dt"], self.n_steps, cfg["stride"],
                                      self.projs[a:b], cfg["grids"], precision=self.prec, trial0=a, n_trials=n,
                                      losvd=buf["losvd"][:n], dens=buf["dens"][:n], nout=buf["nout"][:n])
        else:
            v = {k: (buf[k][:, :n] if k != "dens" else buf[k][:n]) for k in buf}
            if n != self.per:  # ragged last chunk: contiguous views of the right shape
                v = dict(losvd=buf["losvd"].view(-1)[:self.n_proj * n * self.nlos].view(self.n_proj, n, self.nlos),
                         dens=buf["dens"][:n], nout=buf["nout"].view(-1)[:(self.n_proj + 1) * n].view(self.n_proj + 1, n))
            src = self.ics if ics is None else ics
            if self.bundled:
                if self.gh:
                    bd.sm_build_gh_library(self.pot, src[a * self.bundle:b * self.bundle], cfg["dt"], self.n_steps, cfg["stride"],
                                           cfg["projections"], cfg["grids"], self.ap_map, self.n_ap, self.gh_v0, self.gh_s,
                                           n_bundle=self.bundle, fourfold=self.fourfold, precision=self.prec, density_mode=self.dens_mode,
                                           gh=v["losvd"].view(self.n_proj, n, self.n_ap, 6), dens=v["dens"], nout=v["nout"])
                elif self.n_ap or self.dens_mode:
                    bd.sm_build_observable_library(self.pot, src[a * self.bundle:b * self.bundle], cfg["dt"], self.n_steps, cfg["stride"],
                                                   cfg["projections"], cfg["grids"], self.ap_map, self.n_ap, n_bundle=self.bundle,
                                                   fourfold=self.fourfold, precision=self.prec, density_mode=self.dens_mode,
                                                   losvd=v["losvd"], dens=v["dens"], nout=v["nout"])
                else:
                    bd.sm_build_bundled_library(self.pot, src[a * self.bundle:b * self.bundle], cfg["dt"], self.n_steps, cfg["stride"],
                                                cfg["projections"], cfg["grids"], n_bundle=self.bundle, fourfold=self.fourfold,
                                                precision=self.prec, losvd=v["losvd"], dens=v["dens"], nout=v["nout"])
            else:
                bd.sm_build_library(self.pot, src[a:b], cfg["dt"], self.n_steps, cfg["stride"],
                                    cfg["projections"], cfg["grids"], precision=self.prec, losvd=v["losvd"], dens=v["dens"], nout=v["nout"])
            return v
        return {k: buf[k][:n] for k in buf}

    # ---- staged route (matrix larger than HBM): integrate batches that fill the GPU into the compact staged library
    # (sm_stage_library_batch) and flush row windows through the ring (sm_zero_async + sm_scatter_rows) on a second stream while the
    # next batch is integrated: the windows are zeroed AHEAD (as soon as their ring buffer is free, beside the ALU-bound integrator),
    # the latency-bound scatter follows when the batch is staged.  Fill and scatter never run beside each other (profiles/r2l.md).
    def call_name(self):
        if self.bundled:
            base = "sm_build_gh_library" if self.gh else ("sm_build_observable_library" if (self.n_ap or self.dens_mode) else "sm_build_bundled_library")
            if self.batch:
                return "sm_build_gh_library_batch" if self.gh else "sm_build_observable_library_batch"
            return base
        return "sm_build_library_batch" if self.batch else "sm_build_library"

    def staged(self):
        return len(self.chunks) > 1 and not self.bundled   # the paper's row forms go through their own calls, chunk by chunk

    def make_batches(self):
        torch = self.torch
        n_rec = self.n_steps // self.cfg["stride"]
        orbs_per_unit = self.n_orb if self.batch else 1
        want = max(1, -(-131072 // orbs_per_unit))                 # units that give >= 128k orbits per launch
        per_batch = self.per * max(1, -(-want // self.per))        # a whole number of flush chunks
        self.batches = [(a, min(a + per_batch, self.n_units)) for a in range(0, self.n_units, per_batch)]
        n_hist = self.n_proj + 1
        self.stage_elems = (per_batch if self.batch else 1) * n_hist * (self.n_orb if self.batch else per_batch) * n_rec
        self.stage_bufs = [torch.empty(self.stage_elems, dtype=torch.int32, device="cuda") for _ in range(min(2, len(self.batches)))]
        self.flush_stream = torch.cuda.Stream()
        self.ev = {n: [torch.cuda.Event() for _ in range(2)] for n in ("staged", "flushed")}

    def stage_batch(self, k, ics=None):
        a, b = self.batches[k]
        cfg, bd = self.cfg, self.binding
        n, n_hist, n_rec = b - a, self.n_proj + 1, self.n_steps // cfg["stride"]
        buf = self.stage_bufs[k % len(self.stage_bufs)]
        src = self.ics if ics is None else ics
        if self.batch:
            st = buf[:n * n_hist * self.n_orb * n_rec].view(n, n_hist, self.n_orb, n_rec)
            bd.sm_stage_library_batch(self.pot, src[a:b], cfg["dt"], self.n_steps, cfg["stride"], self.projs[a:b], cfg["grids"],
                                      precision=self.prec, trial0=a, n_trials=n, stage=st)
        else:
            st = buf[:n_hist * n * n_rec].view(1, n_hist, n, n_rec)
            bd.sm_stage_library_batch(self.pot, src[a:b], cfg["dt"], self.n_steps, cfg["stride"], [cfg["projections"]], cfg["grids"],
                                      precision=self.prec, stage=st)
        return st

    def chunk_views(self, c, buf):
        """The views of ring buffer buf that hold chunk c: (arguments of the calls, what the caller reads)."""
        a, b = self.chunks[c]
        n = b - a
        if self.batch:   # chunk = trial range, all orbits
            v = {k2: buf[k2][:n] for k2 in buf}
            return v, v
        v = dict(losvd=buf["losvd"].view(-1)[:self.n_proj * n * self.nlos].view(1, self.n_proj, n, self.nlos),
                 dens=buf["dens"].view(-1)[:n * self.nden].view(1, n, self.nden),
                 nout=buf["nout"].view(-1)[:(self.n_proj + 1) * n].view(1, self.n_proj + 1, n))
        return v, {k2: v[k2][0] for k2 in v}

    def zero_chunk(self, c, buf):
        # the window is zeroed by the library's small fill kernel (sm_zero_async): one CTA per SM that fits beside a running integrator
        v, _ = self.chunk_views(c, buf)
        self.binding.sm_zero_async(v["losvd"]); self.binding.sm_zero_async(v["dens"])

    def scatter_chunk(self, st, k, c, buf):
        """Only the non-zero cells of chunk c (inside batch k) from the staged batch st into the zeroed ring buffer buf."""
        a, b = self.chunks[c]
        a0 = self.batches[k][0]
        v, out = self.chunk_views(c, buf)
        if self.batch:
            self.binding.sm_scatter_rows(st[a - a0:b - a0], 0, self.n_orb, self.cfg["grids"], losvd=v["losvd"], dens=v["dens"], nout=v["nout"])
        else:
            self.binding.sm_scatter_rows(st, a - a0, b - a, self.cfg["grids"], losvd=v["losvd"], dens=v["dens"], nout=v["nout"])
        return out

    def flush_chunk(self, st, k, c, buf):
        """Dense rows of chunk c (inside batch k) from the staged batch st into ring buffer buf, on the current stream."""
        self.zero_chunk(c, buf)
        return self.scatter_chunk(st, k, c, buf)

    def chunks_of(self, k):
        a, b = self.batches[k]
        return [c for c, (x, y) in enumerate(self.chunks) if a <= x < b]

    def run_pass_staged(self, overlap=True, after_stage=None, after_flush=None, h_ics=None, after_chunk=None):
        torch = self.torch
        if getattr(self, "batches", None) is None:
            self.make_batches()
        s_int = torch.cuda.current_stream()
        s_fl = self.flush_stream if overlap else s_int
        last = None
        for k in range(len(self.batches)):
            i = k % len(self.stage_bufs)
            s_int.wait_event(self.ev["flushed"][i])                  # this staging buffer has been flushed
            if h_ics is not None:
                a, b = self.batches[k]
                self.ics[a:b].copy_(h_ics[a:b], non_blocking=True)
            st = self.stage_batch(k)
            if after_stage:
                after_stage()
            self.ev["staged"][i].record(s_int)
            cs = self.chunks_of(k)
            # zero ahead: a window needs no staged data to be zeroed, only its ring buffer back -- the first `ring` windows of the batch are
            # zeroed in front of the wait for the integrator (beside it), every later one right after the scatter that frees its buffer
            ahead = overlap and after_chunk is None
            if ahead:
                with torch.cuda.stream(s_fl):
                    for c in cs[:self.ring]:
                        self.zero_chunk(c, self.bufs[c % self.ring])
            s_fl.wait_event(self.ev["staged"][i])
            with torch.cuda.stream(s_fl):
                for n, c in enumerate(cs):
                    if after_chunk:
                        last = after_chunk(c, lambda buf, c=c, st=st, k=k: self.flush_chunk(st, k, c, buf))
                    elif ahead:
                        last = self.scatter_chunk(st, k, c, self.bufs[c % self.ring])
                        if n + self.ring < len(cs):
                            self.zero_chunk(cs[n + self.ring], self.bufs[c % self.ring])
                    else:
                        last = self.flush_chunk(st, k, c, self.bufs[c % self.ring])
                    if after_flush:
                        after_flush()
                self.ev["flushed"][i].record(s_fl)
        s_int.wait_stream(s_fl)
        return last

    def run_pass(self):
        """Inputs resident in HBM; every chunk's dense rows are written to the ring."""
        if self.staged():
            return self.run_pass_staged()
        last = None
        for c in range(len(self.chunks)):
            last = self.build(c, self.bufs[c % self.ring])
        return last

    def rows_ok(self, out):
        n_rec = (self.n_steps // self.cfg["stride"]) * self.bundle * (4 if self.fourfold else 1)
        if self.gh and self.batch:
            cnt = out["losvd"].view(out["losvd"].shape[0], self.n_proj, -1, self.n_ap, 6)[:, 0, :, :, 0].sum(-1)
            return bool(((cnt + out["nout"][:, 0]) == n_rec).all().item() and ((out["dens"].sum(-1) + out["nout"][:, -1]) == n_rec).all().item())
        if self.gh:   # sample counts per aperture (slot 0 of every aperture) + nout
            cnt = out["losvd"].view(self.n_proj, -1, self.n_ap, 6)[0, :, :, 0].sum(-1)
            return bool(((cnt + out["nout"][0]) == n_rec).all().item() and ((out["dens"].sum(-1) + out["nout"][-1]) == n_rec).all().item())
        if self.batch:
            return bool(((out["losvd"][:, 0].sum(-1) + out["nout"][:, 0]) == n_rec).all().item()
                        and ((out["dens"].sum(-1) + out["nout"][:, -1]) == n_rec).all().item())
        return bool(((out["losvd"][0].sum(-1) + out["nout"][0]) == n_rec).all().item()
                    and ((out["dens"].sum(-1) + out["nout"][-1]) == n_rec).all().item())


def e2e_pass(R, pinned, streams, events):
    """One pass with HOST buffers: ICs host->device, build, every row device->host on a copy stream (double-buffered)."""
    torch = R.torch
    comp, copy = streams

    def ship(i, out):   # rows of ring buffer i -> pinned host buffer i, on the copy stream
        cur = torch.cuda.current_stream()
        events["built"][i].record(cur)
        copy.wait_event(events["built"][i])
        with torch.cuda.stream(copy):
            for k in ("losvd", "dens", "nout"):
                dst = pinned[k][i].view(-1)[:out[k].numel()].view(out[k].shape)
                dst.copy_(out[k], non_blocking=True)
            events["copied"][i].record(copy)

    if R.staged():
        def chunk_hook(c, do_flush):
            i = c % len(R.bufs)
            torch.cuda.current_stream().wait_event(events["copied"][i])   # the ring buffer has been shipped
            out = do_flush(R.bufs[i])
            ship(i, out)
            return out
        R.run_pass_staged(h_ics=pinned["ics"], after_chunk=chunk_hook)
    else:
        for c in range(len(R.chunks)):
            a, b = R.chunks[c]
            i = c % len(R.bufs)
            comp.wait_event(events["copied"][i])          # the device buffer is free again
            R.ics[a * R.bundle:b * R.bundle].copy_(pinned["ics"][a * R.bundle:b * R.bundle], non_blocking=True)
            out = R.build(c, R.bufs[i])
            ship(i, out)
    comp.wait_stream(copy)


class CompactE2E:
    """The end-to-end pass a HOST consumer of the library would run: ICs from pinned host memory, sm_stage_library_batch, then the
    rows in COMPACT form (sm_flush_rows_compact: the non-zero cells as (cell, count) pairs, 1-2 % of the dense matrix) copied to
    pinned host memory window by window on a copy stream while the next window is built.  The host ends up with every number of
    the matrix; the dense form through PCIe is timed too (`e2e_dense`)."""

    def __init__(self, R, n_win=4):
        torch = R.torch
        self.R, self.n_win = R, n_win
        cfg = R.cfg
        self.n_rec = R.n_steps // cfg["stride"]
        self.n_hist = R.n_proj + 1
        self.stage = torch.empty((1, self.n_hist, R.n_orb, self.n_rec), dtype=torch.int32, device="cuda")
        self.win = [(a, min(a + -(-R.n_orb // n_win), R.n_orb)) for a in range(0, R.n_orb, -(-R.n_orb // n_win))]
        n_w = max(b - a for a, b in self.win)
        cap = self.n_hist * n_w * min(self.n_rec, 1024)            # ~500 distinct cells per row; total > capacity is checked
        mk = lambda shape, dt, pin: torch.empty(shape, dtype=dt).pin_memory() if pin else torch.empty(shape, dtype=dt, device="cuda")
        self.dev, self.host = [], []
        self.n_buf = n_buf = len(self.win)   # a device and a pinned host buffer per window: no flush waits for a copy of the same pass
        for _ in range(n_buf):
            for store, pin in ((self.dev, False), (self.host, True)):
                store.append(dict(cell=mk(cap, torch.int32, pin), count=mk(cap, torch.float32, pin),
                                  row_start=mk((1, self.n_hist, n_w), torch.int64, pin), row_nnz=mk((1, self.n_hist, n_w), torch.int32, pin),
                                  nout=mk((1, self.n_hist, n_w), torch.int32, pin), total=mk(1, torch.int64, pin)))
        self.h_ics = torch.as_tensor(R.ics_host).pin_memory()
        self.copy, self.small = torch.cuda.Stream(), torch.cuda.Stream()   # bulk copies; the entry counts (not queued behind the bulk)
        # timing-enabled on purpose: with plain events here the next pass's integrator started ~11 ms late on this driver (580.159), as if the
        # stream's work behind the record were held back until the copy stream had drained (A/B: 55.3 against 47.0 ms per pass; cause not isolated)
        self.ev_built = [torch.cuda.Event(enable_timing=True) for _ in range(n_buf)]
        self.ev_total = [torch.cuda.Event() for _ in range(n_buf)]
        self.ev_copied = [torch.cuda.Event() for _ in range(n_buf)]
        self.d2h_bytes = 0
        self.entries = 0

    def ship(self, i, n):
        """entries of device buffer i -> host buffer i (the entry count comes back first)."""
        torch = self.R.torch
        self.ev_total[i].synchronize()
        total = int(self.host[i]["total"].item())
        if total > self.dev[i]["cell"].numel():
            raise SystemExit("compact e2e: capacity too small (%d > %d)" % (total, self.dev[i]["cell"].numel()))
        with torch.cuda.stream(self.copy):
            self.host[i]["cell"][:total].copy_(self.dev[i]["cell"][:total], non_blocking=True)
            self.host[i]["count"][:total].copy_(self.dev[i]["count"][:total], non_blocking=True)
            for k in ("row_start", "row_nnz", "nout"):
                self.host[i][k].view(-1)[:self.n_hist * n].copy_(self.dev[i][k].view(-1)[:self.n_hist * n], non_blocking=True)
            self.ev_copied[i].record(self.copy)
        self.d2h_bytes += 8 + 8 * total + 16 * self.n_hist * n
        self.entries += total

    def run(self):
        R, torch, bd = self.R, self.R.torch, self.R.binding
        cfg = R.cfg
        self.d2h_bytes = self.entries = 0
        cur = torch.cuda.current_stream()
        R.ics.copy_(self.h_ics, non_blocking=True)
        bd.sm_stage_library_batch(R.pot, R.ics, cfg["dt"], R.n_steps, cfg["stride"], [cfg["projections"]], cfg["grids"],
                                  precision=R.prec, stage=self.stage)
        # all windows are built first and their entry counts read back (tiny copies: a count queued behind a bulk copy on the same
        # copy engine would hold the host, and with it the next pass, until that copy is over); then the bulk copies are enqueued
        for w, (a, b) in enumerate(self.win):
            i = w % self.n_buf
            cur.wait_event(self.ev_copied[i])                      # device buffer i has been shipped (by the previous pass)
            d = self.dev[i]
            v = {k: (d[k].view(-1)[:self.n_hist * (b - a)].view(1, self.n_hist, b - a) if k in ("row_start", "row_nnz", "nout") else d[k]) for k in d}
            bd.sm_flush_rows_compact(self.stage, a, b - a, cfg["grids"], out=v)
            self.ev_built[i].record(cur)
            self.copy.wait_event(self.ev_built[i])
            self.small.wait_event(self.ev_built[i])
            with torch.cuda.stream(self.small):
                self.host[i]["total"].copy_(d["total"], non_blocking=True)
                self.ev_total[i].record(self.small)
        for w, (a, b) in enumerate(self.win):
            self.ship(w % self.n_buf, b - a)
        # no wait for the copy stream here: the next pass integrates while the rows of this one are still crossing PCIe (finish())

    def finish(self):
        """Every row of every pass so far is in host memory once the current stream gets past this."""
        self.R.torch.cuda.current_stream().wait_stream(self.copy)


# dram__bytes_read.sum + dram__bytes_write.sum of one x-update launch at the default --weights size (profiles/r1d_weights.md)
W_DRAM_TRAFFIC = 460.3e6 + 18.8e6
W_METRIC, W_UNIT = "ADMM iterations x bootstrap realisations per second incl. Gram matrix and inverse", "rhs-iterations/s"


def weights_oracle_sample(p, lam, rho, n_rhs, n_iter):
    """The oracle's weight solve on the same system with fewer realisations / iterations. -> (rhs-iterations/s, seconds)."""
    from oracle import nnls as onnls
    n_orb = p["dens"].shape[0]
    t0 = time.perf_counter()
    blocks, tg, sg, o = [], [], [], 0
    for name, c0, st, nc in p["blocks"]:
        blocks.append(p[name].reshape(n_orb, -1)[:, c0::st][:, :nc])
        tg.append(p["target"][o:o + nc]); sg.append(p["sigma"][o:o + nc]); o += nc
    U, y, _ = onnls.stack_system(blocks, tg, sg, keep=p["keep"].astype(bool))
    onnls.admm_nnls(U, onnls.bootstrap(y, p["xi"][:n_rhs]), lam, rho, n_iter)
    dt = time.perf_counter() - t0
    return n_rhs * n_iter / dt, dt


def weights_problem(args, rank=0):
    from paper_2607_00117_b200 import inputs
    n_orb, n_ap = args.n_orb or 7500, args.apertures or 600
    p = inputs.weight_problem(n_orb, args.w_dens, n_ap, args.w_rhs, seed=rank)
    # rho = 0.1 x the mean squared column norm of U, lambda such that d_i = 2e-3 rho
    sq = 0.0
    o = 0
    for name, c0, st, nc in p["blocks"]:
        b = p[name].reshape(n_orb, -1)[:, c0::st][:, :nc].astype(np.float64) / p["sigma"][o:o + nc]
        sq += float(np.sum(b * b)); o += nc
    rho = 0.1 * sq / n_orb
    return p, 1e-3 * rho * n_orb, rho


def run_weights_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    p, lam, rho = weights_problem(args)
    n_rhs, n_iter = min(args.w_rhs, 10), min(args.w_iter, 20)
    for _ in range(min(args.warmup, 1)):
        weights_oracle_sample(p, lam, rho, 1, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        weights_oracle_sample(p, lam, rho, n_rhs, n_iter)
    el = time.perf_counter() - t0
    val = n_rhs * n_iter * args.steps / el
    sample = f"the same {p['n_con']} x {p['dens'].shape[0]} system, {n_rhs} realisations x {n_iter} iterations per step (stacking, Gram matrix and Cholesky included)"
    print(json.dumps({
        "impl": "reference", "metric": W_METRIC, "value": val, "unit": W_UNIT, "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": "weight_solve", "sample": sample},
        "cpu_baseline": {"value": val, "unit": W_UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": W_UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def run_weights(args):
    """--weights: one step = one sm_solve_weights call (assemble, Gram matrix, inverse, n_iter ADMM iterations on all
    realisations, chi^2 per block) + sm_marginal_chi2 (Eq. 5-6).  Under torchrun every rank solves its own set of realisations (weak scaling, no collective)."""
    import torch
    import torch.distributed as dist
    from paper_2607_00117_b200 import binding, shard
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    p, lam, rho = weights_problem(args, rank)
    n_orb, n_con, n_rhs, n_iter = p["dens"].shape[0], p["n_con"], args.w_rhs, args.w_iter
    host = {k: torch.as_tensor(p[k]).pin_memory() for k in ("dens", "gh", "target", "sigma", "xi", "keep")}
    dev = {k: v.cuda() for k, v in host.items()}
    warmup = max(args.warmup, 3)

    def solve(d):
        blocks = [(d[name], c0, st, nc) for name, c0, st, nc in p["blocks"]]
        out = binding.sm_solve_weights(blocks, d["target"], d["sigma"], lam, rho, n_iter, xi=d["xi"], keep=d["keep"], want_chi2=True)
        out["chi2_model"] = binding.sm_marginal_chi2(out["chi2"], (1 << len(blocks)) - 2)   # Eq. 5-6, without the 3-D density block
        return out

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fma_peak = binding.sm_measure_fma_peak("f64")
    for _ in range(warmup):
        out = solve(dev)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = binding.sm_launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev[0].record()
    for _ in range(args.steps):
        out = solve(dev)
    ev[1].record()
    barrier()
    launches = binding.sm_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = shard.max_over_ranks(ev[0].elapsed_time(ev[1]), "cuda")
    value = world * n_rhs * n_iter * args.steps / (ms * 1e-3)
    w = out["w"]
    ok = bool(torch.isfinite(w).all() and (w >= 0).all() and torch.isfinite(out["chi2_model"]).all())
    # per-phase device times from events inside the library, separate pass
    binding.sm_set_debug_flags(4)
    solve(dev)
    kt = binding.sm_last_solve_times()
    binding.sm_set_debug_flags(0)
    x_ms = kt["xupdate_sampled_ms"] / ((n_iter + 15) // 16)
    x_flops = 2.0 * n_orb * n_orb * n_rhs
    # e2e: matrices, targets and draws from pinned host memory, weights back to the host, every step
    e2e = None
    if not args.no_e2e:
        w_host = torch.empty((n_rhs, n_orb), dtype=torch.float64).pin_memory()

        def e2e_step():
            d = {k: v.cuda(non_blocking=True) for k, v in host.items()}
            w_host.copy_(solve(d)["w"], non_blocking=True)
        e2e_step(); barrier()
        k2 = min(args.steps, 3)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        e[0].record()
        for _ in range(k2):
            e2e_step()
        e[1].record(); barrier()
        ms2 = shard.max_over_ranks(e[0].elapsed_time(e[1]), "cuda")
        e2e = {"value": world * n_rhs * n_iter * k2 / (ms2 * 1e-3), "unit": W_UNIT, "steps": k2, "ms_per_step": ms2 / k2,
               "h2d_bytes_per_step": int(sum(v.numel() * v.element_size() for v in host.values())),
               "d2h_bytes_per_step": int(w_host.numel() * 8)}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = {
        "metric": W_METRIC, "value": value, "unit": W_UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "weight_solve", "n_orb": n_orb, "n_con": n_con, "density_cells": args.w_dens, "apertures": args.apertures or 600,
                   "n_rhs_per_gpu": n_rhs, "n_iter": n_iter, "lambda": lam, "rho": rho,
                   "parallelism": f"bootstrap realisations sharded x{world}, no collective",
                   "l2": "the %.0f MB inverse is re-read every iteration, larger than the 126 MB L2" % (8e-6 * n_orb * n_orb)},
        "roofline": {"bound": "alu", "kernel": "gemm_f64_mma_kernel (x-update)", "achieved": x_flops / (x_ms * 1e-3) / 1e12,
                     "peak": fma_peak / 1e12, "unit": "TFLOP/s", "frac": x_flops / (x_ms * 1e-3) / fma_peak,
                     "traffic": W_DRAM_TRAFFIC if (n_orb, n_rhs) == (7500, 100) else None,
                     "peak_kind": "measured live by sm_measure_fma_peak (f64 FMA, all SMs; the m8n8k4 matrix instruction runs on the same unit: 37.0 in a microbenchmark)", "kernel_ms": x_ms,
                     "flops_per_launch": x_flops},
        "phases_ms": kt, "weights_ok": ok, "chi2_model": float(out["chi2_model"][0]), "chi2_min": float(out["chi2_model"][1]), "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
    }
    if not args.no_cpu_baseline:
        n_r, n_i = min(n_rhs, 10), min(n_iter, 20)
        v, secs = weights_oracle_sample(p, lam, rho, n_r, n_i)
        line["cpu_baseline"] = {"value": v, "unit": W_UNIT, "cores": os.cpu_count(), "kind": "oracle", "seconds": secs,
                                "sample": f"the same system, {n_r} realisations x {n_i} iterations (stacking, Gram matrix and Cholesky included)"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


M_METRIC, M_UNIT = "model chi^2 evaluations per second (orbit library + weight solve + likelihood)", "evaluations/s"


def model_args(args):
    """The paper's model shape on BASELINE.json configs[1]'s potential and IC recipe."""
    args.config, args.bundle, args.fourfold, args.gh, args.cylindrical = 1, 4, True, True, True
    args.apertures = args.apertures or 600
    args.n_orb, args.n_steps = args.n_orb or 30000, args.n_steps or 5000
    return args


def model_targets(torch, gh0, dens, n_rhs, seed):
    """Input recipe for the mock data of --model: the model of hidden non-negative weights (half of the bundles
    unused) on the library just built, perturbed by the tolerances; 1 % tolerances on the two density blocks, 2 % of the
    aperture's surface density on h_1..h_4; unit-normal bootstrap draws, zero on the 3-D density rows and in realisation 0."""
    gen = torch.Generator(device="cuda").manual_seed(1000 + seed)
    n_rows, n_ap = gh0.shape[0], gh0.shape[1]
    w_h = torch.rand(n_rows, generator=gen, device="cuda", dtype=torch.float64) * \
        (torch.rand(n_rows, generator=gen, device="cuda") < 0.5) / n_rows
    t_dens = w_h @ dens.double()
    t_gh = torch.einsum("i,iac->ca", w_h, gh0.double())
    s_sig = 0.01 * torch.clamp(t_gh[0], min=1e-3 * float(t_gh[0].max()))
    sigma = torch.cat([0.01 * torch.clamp(t_dens, min=1e-3 * float(t_dens.max())), s_sig] + [2.0 * s_sig] * 4)
    target = torch.cat([t_dens, t_gh[0]] + [t_gh[1 + m] for m in range(1, 5)])
    noise = torch.randn(target.numel(), generator=gen, device="cuda", dtype=torch.float64)
    noise[:t_dens.numel()] = 0.0
    target = target + sigma * noise
    xi = torch.randn((n_rhs, target.numel()), generator=gen, device="cuda", dtype=torch.float64)
    xi[:, :t_dens.numel()] = 0.0
    xi[0] = 0.0
    return target, sigma, xi


def run_model(args):
    """--model: one step = one model chi^2 evaluation: library build (R.run_pass), sm_solve_weights on the library matrices in
    place, sm_marginal_chi2.  Under torchrun every rank evaluates its own model (weak scaling: trial models are independent)."""
    import torch
    import torch.distributed as dist
    from paper_2607_00117_b200 import binding, shard
    args = model_args(args)
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg, prec, _ = workload(args)
    R = Runner(args, cfg, prec, rank)
    n_rows, n_ap, n_rhs, n_iter = R.n_units, R.n_ap, args.w_rhs, args.w_iter
    rk = args.rk32   # the pipeline the paper runs: adaptive RK3(2), delta-t-weighted rows, orbits above the Jacobi-drift cut dropped
    if rk:
        rk_out = dict(gh=R.bufs[0]["losvd"].view(R.n_proj, n_rows, n_ap, 6), dens=R.bufs[0]["dens"],
                      wout=torch.empty((R.n_proj + 1, n_rows), dtype=torch.float32, device="cuda"),
                      t_end=torch.empty(R.n_orb, dtype=torch.float64, device="cuda"),
                      diag=torch.empty((R.n_orb, 2), dtype=torch.float64, device="cuda"))
        keep = torch.empty(n_rows, dtype=torch.uint8, device="cuda")

        def build_rk(ics=None):
            binding.sm_build_observable_library_rk32(R.pot, R.ics if ics is None else ics, R.n_steps, cfg["projections"], cfg["grids"],
                                                     R.ap_map, n_ap, n_bundle=R.bundle, fourfold=True, density_mode=R.dens_mode,
                                                     gh=(R.gh_v0, R.gh_s), want_diag=True, out=rk_out)
            d = rk_out["diag"].view(n_rows, R.bundle, 2)   # a bundle is kept when every member passes the 1e-1 cut of PAPER.md:86
            torch.logical_and((d[:, :, 0] <= 0.1).all(1), (d[:, :, 1] == 0).all(1), out=keep.view(torch.bool))
        build_rk()
    else:
        R.run_pass()
    gh0 = R.bufs[0]["losvd"][0].view(n_rows, n_ap, 6)
    dens = R.bufs[0]["dens"]
    blocks = [(dens,), (gh0, 0, 6, n_ap)] + [(gh0, 1 + m, 6, n_ap) for m in range(1, 5)]
    target, sigma, xi = model_targets(torch, gh0, dens, n_rhs, cfg["seed"])
    sq = (dens.double() / sigma[:R.nden]).pow(2).sum()
    for k, col in enumerate([0, 2, 3, 4, 5]):
        sq = sq + (gh0[:, :, col].double() / sigma[R.nden + k * n_ap:R.nden + (k + 1) * n_ap]).pow(2).sum()
    rho = 0.1 * float(sq) / n_rows
    lam = 1e-3 * rho * n_rows
    warmup = max(args.warmup, 3)

    def step(ics=None):
        if rk:
            build_rk(ics)
        else:
            for c in range(len(R.chunks)):
                R.build(c, R.bufs[0], ics=ics)
        out = binding.sm_solve_weights(blocks, target, sigma, lam, rho, n_iter, xi=xi, keep=keep if rk else None, want_chi2=True, want_resid=False)
        out["chi2_model"] = binding.sm_marginal_chi2(out["chi2"], 0b111110)
        return out

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fma_peak = binding.sm_measure_fma_peak("f64")
    for _ in range(warmup):
        out = step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = binding.sm_launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev[0].record()
    for _ in range(args.steps):
        out = step()
    ev[1].record()
    barrier()
    launches = binding.sm_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = shard.max_over_ranks(ev[0].elapsed_time(ev[1]), "cuda")
    if rk:   # weighted rows: sample weights per aperture + the weight outside = 1 per member orbit and copy of Table 1
        rows_ok = bool(((gh0[:, :, 0].sum(1) + rk_out["wout"][0] - 4 * R.bundle).abs() < 1e-3 * 4 * R.bundle).all().item())
    else:
        rows_ok = R.rows_ok(R.bufs[0])
    ok = bool(torch.isfinite(out["w"]).all() and (out["w"] >= 0).all() and torch.isfinite(out["chi2_model"]).all() and rows_ok)
    # phases: library kernels, then the solve's phases, from events inside the library (separate passes)
    binding.sm_set_debug_flags(4)
    if rk:
        build_rk()
    else:
        R.build(0, R.bufs[0])
    lib_t = binding.sm_last_kernel_times()
    binding.sm_solve_weights(blocks, target, sigma, lam, rho, n_iter, xi=xi, keep=keep if rk else None, want_chi2=True, want_resid=False)
    kt = binding.sm_last_solve_times()
    binding.sm_set_debug_flags(0)
    x_ms = kt["xupdate_sampled_ms"] / ((n_iter + 15) // 16)
    x_flops = 2.0 * n_rows * n_rows * n_rhs
    e2e = None
    if not args.no_e2e:
        h_ics = torch.as_tensor(R.ics_host).pin_memory()
        h_out = torch.empty(2, dtype=torch.float64).pin_memory()

        def e2e_step():
            h_out.copy_(step(h_ics.cuda(non_blocking=True))["chi2_model"], non_blocking=True)
        e2e_step(); barrier()
        k2 = min(args.steps, 3)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        e[0].record()
        for _ in range(k2):
            e2e_step()
        e[1].record(); barrier()
        ms2 = shard.max_over_ranks(e[0].elapsed_time(e[1]), "cuda")
        e2e = {"value": world * k2 / (ms2 * 1e-3), "unit": M_UNIT, "steps": k2, "ms_per_step": ms2 / k2,
               "h2d_bytes_per_step": int(h_ics.numel() * 8), "d2h_bytes_per_step": 16,
               "note": "initial conditions from pinned host memory, chi2_model back to the host; the mock data stay resident"}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = {
        "metric": M_METRIC, "value": world * args.steps / (ms * 1e-3), "unit": M_UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "model_evaluation_rk32" if rk else "model_evaluation", "integrator": "adaptive RK3(2), rtol 1e-4, fixed count of step attempts, delta-t weights, "
                   "bundles with a member above the 1e-1 Jacobi-drift cut dropped (PAPER.md:75,86,104)" if rk else "fixed-step kick-drift-kick",
                   "kept_bundles": int(keep.sum().item()) if rk else n_rows,
                   "potential": cfg["name"], "n_ics": R.n_orb, "n_steps": R.n_steps, "n_bundle": R.bundle,
                   "fourfold": True, "rows": n_rows, "apertures": n_ap, "density_cells": R.nden, "gauss_hermite": 4,
                   "n_con": int(target.numel()), "n_rhs_per_gpu": n_rhs, "n_iter": n_iter, "lambda": lam, "rho": rho,
                   "parallelism": f"one model per GPU x{world}, no collective",
                   "l2": "the %.0f MB inverse is re-read every iteration, larger than the 126 MB L2" % (8e-6 * n_rows * n_rows)},
        "roofline": {"bound": "alu", "kernel": "gemm_f64_mma_kernel (x-update)", "achieved": x_flops / (x_ms * 1e-3) / 1e12,
                     "peak": fma_peak / 1e12, "unit": "TFLOP/s", "frac": x_flops / (x_ms * 1e-3) / fma_peak,
                     "traffic": W_DRAM_TRAFFIC if (n_rows, n_rhs) == (7500, 100) else None,
                     "peak_kind": "measured live by sm_measure_fma_peak (f64 FMA, all SMs)", "kernel_ms": x_ms, "flops_per_launch": x_flops},
        "phases_ms": dict(lib_t, **kt), "model_ok": ok, "chi2_model": float(out["chi2_model"][0]), "chi2_min": float(out["chi2_model"][1]),
        "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
        "paper_context": "one model chi^2 evaluation ~1.3 s on an A100 (PAPER.md:262): adaptive RK3 instead of KDK, ADMM iteration count not printed",
    }
    if not args.no_cpu_baseline:
        # the oracle chain on bounded samples of the two stages, extrapolated to one evaluation (labelled)
        n_s = 64 - 64 % R.bundle
        v_lib, cores, s1 = oracle_sample(cfg, R.ics_host, n_s, R.bundle, True, (R.ap_host, R.n_ap), 1, (R.gh_v0_host, R.gh_s_host))
        import copy
        wa = copy.copy(args)
        wa.n_orb, wa.w_dens = n_rows, R.nden
        p, lam_o, rho_o = weights_problem(wa)            # the seeded stand-in system of --weights at the same size
        n_r, n_i = min(n_rhs, 10), min(n_iter, 20)
        _, s2 = weights_oracle_sample(p, lam_o, rho_o, n_r, n_i)
        t_full = R.n_orb * R.n_steps / v_lib + s2 * (n_rhs * n_iter) / (n_r * n_i)
        line["cpu_baseline"] = {"value": 1.0 / t_full, "unit": M_UNIT, "cores": cores, "kind": "oracle", "seconds": s1 + s2,
                                "sample": f"EXTRAPOLATED from two timed samples: library oracle on the first {n_s} ICs x {R.n_steps} steps "
                                          f"({v_lib:.3g} orbit-steps/s) and the ADMM oracle on the stand-in system of --weights at the same size, {n_r} realisations x {n_i} iterations "
                                          f"({s2:.1f} s incl. Gram matrix and Cholesky), scaled linearly to {R.n_orb} ICs and {n_rhs} x {n_iter}"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_rk32_batch(args, cfg, reduced):
    """--rk32 --config 3: the MCMC batch on the paper's own pipeline -- all trial potentials of BASELINE.json configs[3] in one
    sm_build_gh_library_rk32_batch call per step (adaptive RK3(2), 5 000 step attempts, delta-t-weighted Gauss-Hermite rows over 600
    apertures + density rows; plain pixel histograms of 64 trials would be 246 GB).  Also timed: the same trials one call each."""
    import torch
    from paper_2607_00117_b200 import binding, inputs
    torch.cuda.set_device(0)
    n_steps, n_trials, n_orb, n_ap = args.n_steps or 5000, cfg["n_trials"], cfg["n_orb"], args.apertures or 600
    draws = inputs.trial_draws(n_trials, cfg["seed"])
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    ics = np.stack([inputs.make_ics(cfg, lambda p_, x, t=t: binding.sm_eval_force(pot, x, 0.0, trial=t, want_phi=False).cpu().numpy(),
                                    potential=d["potential"]) for t, d in enumerate(draws)])
    d_ics, pinned = torch.as_tensor(ics).cuda(), torch.as_tensor(ics).pin_memory()
    projs, g = [[d["projection"]] for d in draws], cfg["grids"]
    ap = torch.as_tensor(inputs.aperture_map(g, n_ap, cfg["seed"])).cuda()
    rng = np.random.default_rng(cfg["seed"] + 7)
    gh = (torch.as_tensor(rng.normal(0.0, 60.0, n_ap)).cuda(), torch.as_tensor(rng.uniform(70.0, 160.0, n_ap)).cuda())
    kw = dict(ap_map=ap, n_ap=n_ap, gh=gh, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3)
    fma_peak = binding.sm_measure_fma_peak("f64")
    warmup, out = max(args.warmup, 3), None
    for _ in range(warmup):
        out = binding.sm_build_observable_library_rk32_batch(pot, d_ics, n_steps, projs, g, out=out, **kw)
    torch.cuda.synchronize()
    sampler, l0 = ClockSampler(0), binding.sm_launch_count()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    e[0].record()
    for _ in range(args.steps):
        out = binding.sm_build_observable_library_rk32_batch(pot, d_ics, n_steps, projs, g, out=out, **kw)
    e[1].record(); torch.cuda.synchronize()
    ms, launches, clocks = e[0].elapsed_time(e[1]) / args.steps, binding.sm_launch_count() - l0, sampler.stop()
    prev = binding.sm_set_debug_flags(4)
    try:
        out = binding.sm_build_observable_library_rk32_batch(pot, d_ics, n_steps, projs, g, out=out, **kw)
        kt = binding.sm_last_kernel_times()
    finally:
        binding.sm_set_debug_flags(prev)
    rows_ok = bool(((out["gh"][:, 0, :, :, 0].sum(-1) + out["wout"][:, 0] - 1).abs() < 1e-3).all().item())
    # the same trials one call each (what a caller without the batched entry point would do), on the first four trials
    singles, o1 = [binding.sm_make_potential(d["potential"]) for d in draws[:4]], None
    for rep in range(2):
        if rep == 1:
            torch.cuda.synchronize(); e[0].record()
        for t, p1 in enumerate(singles):
            o1 = binding.sm_build_observable_library_rk32(p1, d_ics[t], n_steps, projs[t], g, out=o1, **kw)
    e[1].record(); torch.cuda.synchronize()
    ms_single = e[0].elapsed_time(e[1]) / len(singles)
    e[0].record()
    o2 = binding.sm_build_observable_library_rk32_batch(pot, pinned.cuda(non_blocking=True), n_steps, projs, g, out=out, **kw)
    back = (o2["wout"].cpu(), o2["t_end"].cpu())
    e[1].record(); torch.cuda.synchronize()
    ms2 = e[0].elapsed_time(e[1])
    work = n_trials * n_orb * n_steps
    fl_att, _, _, rk_src = kernel_counts("rk32_kernel/barred/f64")
    flops = (fl_att or 0.0) * work
    print(json.dumps({
        "metric": METRIC, "value": work / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"] + "_rk32", "n_trials": n_trials, "n_orb": n_orb, "step_attempts": n_steps, "apertures": n_ap,
                   "gauss_hermite": True, "force_evaluations_per_attempt": 3, "rtol": 1e-4, "reduced": reduced,
                   "matrix_bytes": int(out["gh"].numel() * 4 + out["dens"].numel() * 4),
                   "l2": "every pass re-stages %.0f GB of samples in orbit chunks and rewrites the matrix, far larger than the 126 MB L2" % (16e-9 * work)},
        "roofline": {"bound": "alu", "kernel": "rk32_kernel", "achieved": flops / (kt["integrate_ms"] * 1e-3) / 1e12 if flops else None,
                     "peak": fma_peak / 1e12, "unit": "TFLOP/s", "frac": flops / (kt["integrate_ms"] * 1e-3) / fma_peak if flops else None, "traffic": None,
                     "peak_kind": "measured live by sm_measure_fma_peak (f64 FMA, all SMs)", "kernel_ms": kt["integrate_ms"],
                     "flops_per_step_attempt": fl_att, "counts_from": ("profiles/" + rk_src) if rk_src else None,
                     "note": "executed-flop count of the plain-row instantiation; the row-form instantiation stages more per attempt"},
        "rows_ms": kt["rowbuild_ms"], "rows_sum_to_one": rows_ok, "gpu_launches": int(launches // args.steps), "clocks": clocks,
        "one_trial_per_call": {"ms_per_trial": ms_single, "value": n_orb * n_steps / (ms_single * 1e-3), "unit": UNIT,
                               "note": "sm_build_gh_library_rk32 on the first four trials, one call each: one warp per scheduler"},
        "e2e": {"value": work / (ms2 * 1e-3), "unit": UNIT, "steps": 1, "ms_per_step": ms2, "h2d_bytes_per_step": int(pinned.numel() * 8),
                "d2h_bytes_per_step": int(sum(b.numel() * b.element_size() for b in back)),
                "note": "ICs of all trials from pinned host memory, outside weights and integration times back; the matrices stay resident"}}))


def run_rk32(args):
    """--rk32: one step = one sm_build_library_rk32 call (adaptive RK3(2) integration, projection, binning, delta-t-weighted dense
    rows) on the config's orbits.  An orbit-step is one step ATTEMPT (three force evaluations; the paper's fixed count).
    --impl reference: the oracle (smo.build_library_rk32) on the first 64 orbits per step.  Single GPU (rank 0 runs alone)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2607_00117_b200 import inputs
    from oracle import smo
    cfg, prec, reduced = workload(args)
    if "n_trials" in cfg and args.impl != "reference":
        return run_rk32_batch(args, cfg, reduced)
    if "n_trials" in cfg or cfg["ics"] != "disc":
        raise SystemExit("--rk32 needs a disc config (1, 2 or 4; 3 = the batched potentials)")
    n_steps = args.n_steps or 5000
    n_orb = cfg["n_orb"]
    ics = inputs.make_ics(cfg, lambda pot, pts: smo.eval_force(pot, pts, 0.0, want_phi=False)) if args.impl == "reference" else None
    tol = dict(rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3)
    name = cfg["name"] + "_rk32"
    if args.impl == "reference":
        n_s = 64
        for _ in range(args.warmup):
            smo.build_library_rk32(cfg["potential"], ics[:8], n_steps, cfg["projections"], cfg["grids"], **tol)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            smo.build_library_rk32(cfg["potential"], ics[:n_s], n_steps, cfg["projections"], cfg["grids"], **tol)
        dt = time.perf_counter() - t0
        v = n_s * n_steps * args.steps / dt
        sample = f"first {n_s} orbits x {n_steps} step attempts of {name} per step"
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                          "data": "synthetic", "config": {"workload": name, "sample": sample},
                          "cpu_baseline": {"value": v, "unit": UNIT, "cores": smo.num_threads(), "kind": "oracle", "sample": sample},
                          "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))
        return
    import torch
    from paper_2607_00117_b200 import binding
    torch.cuda.set_device(0)
    pot = binding.sm_make_potential(cfg["potential"])
    ics = inputs.make_ics(cfg, lambda p_, pts: binding.sm_eval_force(binding.sm_make_potential(p_), pts, 0.0, want_phi=False).cpu().numpy())
    d_ics = torch.as_tensor(ics).cuda()
    pinned = torch.as_tensor(ics).pin_memory()
    fma_peak = binding.sm_measure_fma_peak("f64")
    warmup = max(args.warmup, 3)
    out = None                                   # one set of caller-owned output buffers, rewritten by every pass
    for _ in range(warmup):
        out = binding.sm_build_library_rk32(pot, d_ics, n_steps, cfg["projections"], cfg["grids"], out=out, **tol)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    l0 = binding.sm_launch_count()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    e[0].record()
    for _ in range(args.steps):
        out = binding.sm_build_library_rk32(pot, d_ics, n_steps, cfg["projections"], cfg["grids"], out=out, **tol)
    e[1].record(); torch.cuda.synchronize()
    ms = e[0].elapsed_time(e[1])
    launches = binding.sm_launch_count() - l0
    clocks = sampler.stop()
    # kernel times of one more pass, outside the timed region (CUDA events inside the library around each launch)
    prev = binding.sm_set_debug_flags(4)
    try:
        out = binding.sm_build_library_rk32(pot, d_ics, n_steps, cfg["projections"], cfg["grids"], out=out, **tol)
        kt = binding.sm_last_kernel_times()
    finally:
        binding.sm_set_debug_flags(prev)
    rows_ok = bool(((out["losvd"][0].sum(1) + out["wout"][0] - 1).abs() < 1e-4).all().item())
    matrix_bytes = sum(out[k].numel() * 4 for k in ("losvd", "dens"))
    # e2e: ICs from pinned host memory, the per-orbit outside weights and integration times back (the matrix stays on the device)
    k2 = min(args.steps, 2)
    e[0].record()
    for _ in range(k2):
        o2 = binding.sm_build_library_rk32(pot, pinned.cuda(non_blocking=True), n_steps, cfg["projections"], cfg["grids"], out=out, **tol)
        back = (o2["wout"].cpu(), o2["t_end"].cpu())
    e[1].record(); torch.cuda.synchronize()
    ms2 = e[0].elapsed_time(e[1])
    work = n_orb * n_steps
    fl_att, rk_dram, rk_work, rk_src = kernel_counts("rk32_kernel/%s/f64" % ("paperbar" if args.bar == "dehnen" else "barred"))
    flops = (fl_att or 0.0) * work
    line = {"metric": METRIC, "value": work * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "n_orb": n_orb, "step_attempts": n_steps, "force_evaluations_per_attempt": 3, "rtol": 1e-4,
                       "n_proj": len(cfg["projections"]), "matrix_bytes": matrix_bytes, "reduced": reduced,
                       "l2": "every pass rewrites the %.2f GB matrix and its %.2f GB of staged samples, far larger than the 126 MB L2"
                             % (matrix_bytes / 1e9, 4 * (len(cfg["projections"]) + 2) * work / 1e9)},
            "roofline": {"bound": "alu", "kernel": "rk32_kernel", "achieved": flops / (kt["integrate_ms"] * 1e-3) / 1e12 if flops else None,
                         "peak": fma_peak / 1e12, "unit": "TFLOP/s", "frac": flops / (kt["integrate_ms"] * 1e-3) / fma_peak if flops else None,
                         "traffic": rk_dram if (flops and rk_work == work) else None,
                         "peak_kind": "measured live by sm_measure_fma_peak (f64 FMA, all SMs)", "kernel_ms": kt["integrate_ms"],
                         "flops_per_step_attempt": fl_att, "counts_from": ("profiles/" + rk_src) if rk_src else None},
            "flush": {"bound": "hbm", "kernel": "rk32_rows_kernel", "achieved": matrix_bytes / (kt["rowbuild_ms"] * 1e-3) / 1e9, "unit": "GB/s",
                      "kernel_ms": kt["rowbuild_ms"]},
            "median_t_end": float(out["t_end"].median().item()), "rows_sum_to_one": rows_ok, "gpu_launches": int(launches), "clocks": clocks,
            "e2e": {"value": work * k2 / (ms2 * 1e-3), "unit": UNIT, "steps": k2, "ms_per_step": ms2 / k2, "h2d_bytes_per_step": int(pinned.numel() * 8),
                    "d2h_bytes_per_step": int(sum(t.numel() * t.element_size() for t in back)),
                    "note": "ICs from pinned host memory, outside weights and integration times back; the matrix stays resident"}}
    if not args.no_cpu_baseline:
        t0 = time.perf_counter()
        smo.build_library_rk32(cfg["potential"], ics[:256], n_steps, cfg["projections"], cfg["grids"], **tol)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": 256 * n_steps / dt, "unit": UNIT, "cores": smo.num_threads(), "kind": "oracle", "seconds": dt,
                                "sample": f"first 256 orbits x {n_steps} step attempts of {name}"}
    print(json.dumps(line))


def measure(R, binding, torch, shard, world, steps, warmup, barrier, clock_index=None):
    """Warm-up, the timed region (K passes, device-resident inputs, CUDA events on the launching stream, no host sync inside,
    max over ranks), then two separate passes for the per-kernel device times (events recorded inside the library around its
    launches) and for the integrator with recording compiled out (binning-overhead A/B)."""
    out = None
    for _ in range(warmup):
        out = R.run_pass()
    barrier()
    sampler = ClockSampler(clock_index) if clock_index is not None else None
    l0 = binding.sm_launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev[0].record()
    for _ in range(steps):
        out = R.run_pass()
    ev[1].record()
    barrier()
    launches = binding.sm_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = shard.max_over_ranks(ev[0].elapsed_time(ev[1]), "cuda")
    rows_ok = R.rows_ok(out)
    binding.sm_set_debug_flags(4)
    kt = {"phase_ms": 0.0, "integrate_ms": 0.0, "rowbuild_ms": 0.0, "zero_fill_ms": 0.0}

    def add_times():
        for k, v in binding.sm_last_kernel_times().items():
            kt[k] += v
    staged = R.staged()
    if staged:
        R.run_pass_staged(overlap=False, after_stage=add_times, after_flush=add_times)
    else:
        for c in range(len(R.chunks)):
            R.build(c, R.bufs[c % R.ring]); add_times()
    binding.sm_set_debug_flags(4 | 1)
    norec = [0.0]

    def add_norec():
        norec[0] += binding.sm_last_kernel_times()["integrate_ms"]
    if staged:
        for k in range(len(R.batches)):
            R.stage_batch(k); add_norec()
    else:
        for c in range(len(R.chunks)):
            R.build(c, R.bufs[c % R.ring]); add_norec()
    binding.sm_set_debug_flags(0)
    torch.cuda.synchronize()
    return {"ms": ms, "launches": int(launches), "clocks": clocks, "rows_ok": rows_ok, "kt": kt, "norec_ms": norec[0]}


def roofline_record(kind, prec, peak_prec, work, int_ms, fma_peak, one_launch):
    """Roofline of integrate_kernel: executed flop of the kernel's arithmetic type (profiles/kernel_counts.json) x orbit-steps /
    its CUDA-event time, against the FMA rate measured live on the same GPU."""
    flop, dram, prof_work, src = kernel_counts("integrate_kernel/%s/%s" % (kind, prec))
    rec = {"bound": "alu", "kernel": "integrate_kernel", "achieved": None, "peak": fma_peak / 1e12, "unit": "TFLOP/s", "frac": None,
           "traffic": None, "kernel_ms": int_ms, "kernel_orbit_steps_per_s": work / (int_ms * 1e-3),
           "peak_kind": f"measured live by sm_measure_fma_peak ({peak_prec} FMA, all SMs); derived 148 SM x lanes x 2 x 1.965 GHz = "
                        f"{FMA_PEAK_DERIVED[peak_prec] / 1e12:.1f}"}
    if flop is None:
        rec["note"] = "no ncu capture of this kernel in profiles/kernel_counts.json: executed-flop count unknown"
        return rec
    ach = flop * work / (int_ms * 1e-3)
    rec.update(achieved=ach / 1e12, frac=ach / fma_peak, flops_per_orbit_step=flop, counts_from="profiles/" + src,
               traffic=dram if (one_launch and prof_work == work) else None)
    return rec


def flush_record(matrix_bytes, kt, hbm, staged, peak_kind):
    """Row a-7.  Where the outputs were zeroed by the copy engines under the integrator (zero_fill_ms > 0, or the staged route,
    whose windows bench.py zeroes with sm_zero_async on the flush stream), the HBM-bound part is that fill and the kernel after
    the integrator only scatters the non-zero cells; otherwise the row build writes the dense matrix itself."""
    row_ms, z_ms = kt["rowbuild_ms"], kt["zero_fill_ms"]
    if z_ms > 0 or staged:
        rec = {"bound": "hbm", "kernel": "zero_fill_kernel beside the integrator (hidden) + rowbuild_sparse_kernel (scatter of the non-zero cells)",
               "achieved": matrix_bytes / (z_ms * 1e-3) / 1e9 if z_ms else None, "peak": hbm, "unit": "GB/s",
               "frac": matrix_bytes / (z_ms * 1e-3) / 1e9 / hbm if z_ms else None, "zero_fill_ms": z_ms if z_ms else None,
               "scatter_kernel_ms": row_ms, "kernel_ms": row_ms, "peak_kind": peak_kind}
        if staged:
            rec["note"] = "staged route: every ring window is zeroed with sm_zero_async on the flush stream (not timed separately)"
        return rec
    return {"bound": "hbm", "kernel": "rowbuild_kernel", "achieved": matrix_bytes / (row_ms * 1e-3) / 1e9 if row_ms else None,
            "peak": hbm, "unit": "GB/s", "frac": matrix_bytes / (row_ms * 1e-3) / 1e9 / hbm if row_ms else None,
            "kernel_ms": row_ms, "peak_kind": peak_kind}


def sub_record(args, cid, prec, rank, world, mods, peaks, barrier, **row_form):
    """Compact record of another config (2 warm-up + 2 timed passes, same route and checks as the headline); row_form overrides
    the row-form arguments (gh, apertures, bundle, fourfold, cylindrical)."""
    import copy
    torch, binding, shard = mods
    a2 = copy.copy(args)
    a2.config, a2.precision, a2.n_orb, a2.n_steps, a2.n_trials = cid, prec, None, None, None
    for k, v in row_form.items():
        setattr(a2, k, v)
    cfg, prec, _ = workload(a2)
    R = Runner(a2, cfg, prec, rank)
    work = R.n_trials * R.n_orb * R.n_steps
    m = measure(R, binding, torch, shard, world, 2, 2, barrier)
    kind = "plummer" if cfg["ics"] == "plummer" else "barred"
    roof = roofline_record(kind, prec, prec, work, m["kt"]["integrate_ms"], peaks[prec], not R.staged() and len(R.chunks) == 1)
    row_ms = m["kt"]["rowbuild_ms"]
    rec = {"workload": cfg["name"], "dtype": prec, "value": world * work * 2 / (m["ms"] * 1e-3), "ms_per_step": m["ms"] / 2,
           "orbit_steps_per_pass": work, "matrix_bytes": R.matrix_bytes, "chunks": len(R.chunks),
           "integrate_ms": m["kt"]["integrate_ms"], "rowbuild_ms": row_ms, "zero_fill_ms": m["kt"]["zero_fill_ms"], "roofline_frac": roof["frac"],
           "roofline_achieved_tflops": roof["achieved"], "flush_gbs": R.matrix_bytes / (row_ms * 1e-3) / 1e9 if row_ms else None,
           "binning_overhead_frac": 1.0 - m["norec_ms"] / (m["ms"] / 2), "row_sums_ok": m["rows_ok"],
           "gpu_launches": m["launches"], "steps": 2, "warmup": 2}
    if row_form:
        rec["row_form"] = {k: v for k, v in row_form.items()}
    R.bufs = R.stage_bufs = None
    del R
    torch.cuda.empty_cache()
    return rec


def run_zero_fill(args):
    """sm_zero_async alone on the GPU (no integrator beside it): the fill kernels' own HBM write rate."""
    import torch
    from paper_2607_00117_b200 import binding
    buf = torch.empty(int(args.zero_fill * 1e9) // 4, dtype=torch.float32, device="cuda")
    cfg = workload(args)[0]   # one tiny integrator launch first: the fill takes the shared-memory carve-out of the device's integrator launches
    binding.sm_build_library(binding.sm_make_potential(cfg["potential"]), np.ones((32, 6)), 1e-3, 4, 1, cfg["projections"], cfg["grids"])
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    for i in range(max(args.warmup, 1) + args.steps):
        if i == max(args.warmup, 1):
            ev[0].record()
        binding.sm_zero_async(buf)
    ev[1].record()
    torch.cuda.synchronize()
    ms = ev[0].elapsed_time(ev[1]) / args.steps
    print(json.dumps({"metric": "zero fill alone", "value": buf.numel() * 4 / ms / 1e6, "unit": "GB/s", "ms": ms, "bytes": buf.numel() * 4,
                      "debug_flags": args.debug_flags, "zeroed": bool(buf[-1000003:].abs().max().item() == 0.0)}))


def main():
    args = parse()
    if args.debug_flags:
        from paper_2607_00117_b200 import binding as _b
        _set = _b.sm_set_debug_flags
        _b.sm_set_debug_flags = lambda f: _set(int(f) | args.debug_flags)
        _set(args.debug_flags)
    if args.zero_fill:
        return run_zero_fill(args)
    if args.model:
        if args.impl == "reference":
            print(json.dumps({"impl": "reference", "unavailable": "--model has no reference arm; see --weights and the default library arm"}))
            return
        return run_model(args)
    if args.weights:
        return run_weights_reference(args) if args.impl == "reference" else run_weights(args)
    if args.rk32:
        return run_rk32(args)
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import torch.distributed as dist
    from paper_2607_00117_b200 import binding, shard
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg, prec, reduced = workload(args)
    R = Runner(args, cfg, prec, rank)
    work = R.n_trials * R.n_orb * R.n_steps  # orbit-steps per pass per rank
    warmup = max(args.warmup, 3)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # the needle integrals of --bar dehnen are fp64 in both precisions: their roofline is the FP64 one
    peak_prec = "f64" if args.bar == "dehnen" else prec
    peaks = {p_: binding.sm_measure_fma_peak(p_) for p_ in ("f64", "f32")}  # also warms the clocks
    fma_peak = peaks[peak_prec]
    m = measure(R, binding, torch, shard, world, args.steps, warmup, barrier, clock_index=local if rank == 0 else None)
    ms, kt, norec_ms = m["ms"], m["kt"], m["norec_ms"]
    value = world * work * args.steps / (ms * 1e-3)
    staged = R.staged()
    n_batches = len(R.batches) if staged else 0

    # ---- e2e: the same pass through the C-ABI binding with pinned HOST buffers, copies inside the timed region
    e2e = e2e_dense = None
    if not args.no_e2e:
        k2 = min(args.steps, 3 if R.matrix_bytes < 20e9 else 1)
        full_chunking = (R.per, R.ring)
        per = max(1, int(4e9 // R.unit_bytes))     # <= 4 GB chunks so that the pinned ring stays small
        if not R.batch and per >= 512:
            per = per // 512 * 512
        R.set_chunk(min(per, R.n_units), 2)
        pinned = {"ics": torch.as_tensor(R.ics_host).pin_memory()}
        for k in ("losvd", "dens", "nout"):
            pinned[k] = [torch.empty(R.bufs[0][k].shape, dtype=R.bufs[0][k].dtype).pin_memory() for _ in range(2)]
        comp, copy = torch.cuda.current_stream(), torch.cuda.Stream()
        events = {n: [torch.cuda.Event() for _ in range(2)] for n in ("built", "copied")}
        e2e_pass(R, pinned, (comp, copy), events); barrier()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        e[0].record()
        for _ in range(k2):
            e2e_pass(R, pinned, (comp, copy), events)
        e[1].record(); barrier()
        ms2 = shard.max_over_ranks(e[0].elapsed_time(e[1]), "cuda")
        e2e = {"value": world * work * k2 / (ms2 * 1e-3), "unit": UNIT, "steps": k2, "ms_per_step": ms2 / k2,
               "h2d_bytes_per_step": int(R.ics_host.nbytes),
               "d2h_bytes_per_step": int(R.matrix_bytes + 4 * R.n_trials * (R.n_orb // R.bundle) * (R.n_proj + 1)),
               "chunks": len(R.chunks), "rows": "dense", "api": R.call_name() + " per <= 4 GB chunk",
               "note": "pinned host ring, D2H of chunk c overlaps the build of chunk c+1; every dense row crosses PCIe"}
        del pinned
        R.set_chunk(*full_chunking)
        # the route a host consumer should take: the same library in compact form (every non-zero cell of every row)
        if not R.batch and not R.bundled:
            e2e_dense = e2e
            R.bufs = None
            torch.cuda.empty_cache()
            ce = CompactE2E(R)
            ce.run(); ce.finish(); barrier()
            k3 = min(args.steps, 8)   # the last pass's rows cross PCIe after its integrator (no later pass to hide them): K passes amortise that tail
            e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            e[0].record()
            for _ in range(k3):
                ce.run()
            ce.finish()                                            # the rows of the last pass too
            e[1].record(); barrier()
            ms3 = shard.max_over_ranks(e[0].elapsed_time(e[1]), "cuda")
            e2e = {"value": world * work * k3 / (ms3 * 1e-3), "unit": UNIT, "steps": k3, "ms_per_step": ms3 / k3,
                   "h2d_bytes_per_step": int(R.ics_host.nbytes), "d2h_bytes_per_step": int(ce.d2h_bytes), "rows": "compact",
                   "entries_per_step": int(ce.entries), "api": "sm_stage_library_batch + sm_flush_rows_compact per window of rows",
                   "note": "ICs from pinned host memory; every non-zero cell of every row (cell, count), row offsets and out-of-grid "
                           "counters back to pinned host memory on a copy stream, window by window, while the next window is built and the next pass "
                           "integrates (the timed region ends when the rows of the last pass are in host memory); the dense form is e2e_dense"}
            del ce
            torch.cuda.empty_cache()
            R.set_chunk(*full_chunking)
        else:
            e2e_dense = None

    kind = "plummer" if cfg["ics"] == "plummer" else ("paperbar" if args.bar == "dehnen" else "barred")
    int_ms = kt["integrate_ms"]
    try:
        hw = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        hw = {}
    hbm = hw.get("hbm_gbs", 6650.0)
    row_ms = kt["rowbuild_ms"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": ms / args.steps, "library_build_ms": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": cfg["name"], "baseline_config_index": args.config, "n_trials": R.n_trials, "n_orb_per_gpu": R.n_orb,
                   "n_steps": R.n_steps, "stride": cfg["stride"], "n_proj": R.n_proj, "losvd_bins": R.nlos, "density_bins": R.nden,
                   "rows": R.n_units * (1 if not R.batch else R.n_orb), "n_bundle": R.bundle, "fourfold": R.fourfold, "apertures": R.n_ap, "gauss_hermite": R.gh, "cylindrical_density": bool(R.dens_mode),
                   "matrix_bytes": R.matrix_bytes, "chunks": len(R.chunks), "ring_buffers": R.ring, "reduced": reduced,
                   "route": ("sm_stage_library_batch per batch of >=128k orbits (%d batches) + sm_flush_rows per chunk on a second stream" % n_batches) if staged else R.call_name() + " per chunk",
                   "parallelism": f"orbit-sharded x{world}, no collective",
                   "l2": "every pass rewrites the %.2f GB matrix, far larger than the 126 MB L2" % (R.matrix_bytes / 1e9)},
        "roofline": roofline_record(kind, prec, peak_prec, work, int_ms, fma_peak, not staged and len(R.chunks) == 1 and not reduced),
        "flush": flush_record(R.matrix_bytes, kt, hbm, staged, "MEASURED_PEAKS.json hbm_gbs" if hw else "fallback 6650"),
        "binning_overhead_frac": 1.0 - norec_ms / (ms / args.steps), "integrator_norec_ms": norec_ms,
        "row_sums_ok": m["rows_ok"], "gpu_launches": m["launches"], "clocks": m["clocks"], "e2e": e2e, "e2e_dense": e2e_dense,
        "paper_context": "full model construction ~1 s on an A100 (PAPER.md:15), another machine and a different pipeline",
    }
    ics_host, batch, n_orb, n_steps, bundle, R_bundled = R.ics_host, R.batch, R.n_orb, R.n_steps, R.bundle, R.bundled
    oracle_args = (R.fourfold, (R.ap_host, R.n_ap) if R.n_ap else None, R.dens_mode, (R.gh_v0_host, R.gh_s_host) if R.gh else None)
    # ---- the other configs as compact sub-records of the same line (default workload, one GPU only)
    default_run = args.config == 2 and not reduced and prec == "f64" and args.bar == "ferrers" and not R.bundled
    if default_run and world == 1 and not args.no_sub:
        R.bufs = R.stage_bufs = None
        del R
        torch.cuda.empty_cache()
        subs = []
        for cid, p2 in ((0, "f64"), (1, "f64"), (2, "f32"), (3, "f32"), (4, "f64")):
            try:
                subs.append(sub_record(args, cid, p2, rank, world, (torch, binding, shard), peaks, barrier))
            except Exception as ex:  # a sub-record must never take the headline down with it
                subs.append({"workload": "config %d %s" % (cid, p2), "error": repr(ex)[:300]})
        try:   # the MCMC batch in the paper's row form: Gauss-Hermite sums over 600 apertures for all 64 trials
            subs.append(sub_record(args, 3, "f32", rank, world, (torch, binding, shard), peaks, barrier, gh=True, apertures=600))
        except Exception as ex:
            subs.append({"workload": "config 3 f32 gh", "error": repr(ex)[:300]})
        line["other_configs"] = subs
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    if not args.no_cpu_baseline:
        # ~10-30 s of oracle work: 512 full-length config-1 orbits (~6e-5 s per force evaluation on 16 cores), or all of config 0
        c1 = dict(cfg)
        ics1 = ics_host[0] if batch else ics_host
        if batch:
            from paper_2607_00117_b200 import inputs
            d0 = inputs.trial_draws(1, cfg["seed"])[0]
            c1["potential"], c1["projections"] = d0["potential"], [d0["projection"]]
        n_s = min(512 if cfg["ics"] == "disc" else 1000, n_orb)
        if cfg["ics"] == "disc" and n_steps > 10000:
            n_s = max(64, int(512 * 10000 / n_steps))
        n_s -= n_s % bundle
        v, cores, secs = oracle_sample(c1, ics1, n_s, bundle, *oracle_args)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
                                "sample": f"first {n_s} orbits x {n_steps} steps of {cfg['name']}" + (" (trial 0)" if batch else ""),
                                "note": "the parity oracle as it stands: every force in software __float128, OpenMP over orbits; "
                                        "a reported baseline, not a tuned CPU code -- no GPU/CPU ratio is quoted from it"}
        if not R_bundled:
            # the same oracle with its force expressions compiled for plain double (oracle state_prec = 2): what a plain CPU code costs
            # without software quad arithmetic.  Still plain loops, one force per step, OpenMP over orbits; not tuned, not the parity oracle.
            from oracle import smo
            n_d = min(n_orb, 8 * n_s)
            t0 = time.perf_counter()
            smo.build_library(c1["potential"], ics1[:n_d], c1["dt"], c1["n_steps"], c1["stride"], c1["projections"], c1["grids"], state_prec=2)
            sd = time.perf_counter() - t0
            line["cpu_baseline_double"] = {"value": n_d * n_steps / sd, "unit": UNIT, "cores": cores, "kind": "oracle, forces compiled for plain double",
                                           "seconds": sd, "sample": f"first {n_d} orbits x {n_steps} steps of {cfg['name']}" + (" (trial 0)" if batch else "")}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
