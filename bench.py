#!/usr/bin/env python
"""bench.py -- zone-cycles/s of the fp64 HARM step on B200 (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one full predictor-corrector update (kh_step: every row of SURVEY.md section 8(a)) of one
mesh block of synthetic input.  Default workload = BASELINE.json configs[2], the 192x128x128 FMKS
Fishbone-Moncrief torus (Kerr a = 0.9375, WENO5) that the metric's target is quoted on.

Printed: ONE JSON line (rank 0) with
  value     zone-cycles/s, all ranks, state resident in HBM, CUDA-graph replay, device-resident dt
  e2e       the same through the C ABI with HOST buffers: kh_set_prims(host) + kh_step + kh_get_prims(host)
            every step (pinned memory), copies inside the timed region
  roofline  the dominant kernel against the roof that binds it
  kernels   device ms per step of every kernel kind, from CUDA events around each launch on the grid's
            stream (an extra instrumented pass of the same K steps: kh_set_profile)
  cpu_baseline  the CPU oracle, as it stands, on this box's host cores on a bounded sample

--impl reference times the oracle (there is no reference implementation to install: /root/reference
holds only the paper's text).  N > 1: independent replicas, one per GPU (replicas
only, no data-path collective); torch.distributed is used for the barrier and the max-over-ranks time.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

WORKLOADS = {
    # name: (config number of BASELINE.json (1-based), resolution or None = the config's own, recon or None)
    "torus_sane_192x128x128_weno5": (3, None, None),
    "torus_mad_288x128x128_mc": (4, None, None),
    "torus_sane_192x128x128_mc": (3, None, 0),
    "torus_sane_192x128x128_weno5_kastaun": (3, None, None),      # same block, kh_params.inverter = KH_INV_KASTAUN
    "torus_sane_192x128x128_weno5_fofc": (3, None, None),         # same block, kh_params.fofc = 1
    "torus_sane_192x128x128_weno5_drift": (3, None, None),        # same block, kh_params.floor_frame = KH_FRAME_DRIFT
    "torus_sane_192x128x128_weno5_facect": (3, None, None),       # same block, kh_params.transport = KH_B_FACE_CT
    "torus_sane_192x128x128_weno5_facect_upwind": (3, None, None),  # ... and kh_params.emf = KH_EMF_UPWIND
    # the same block cut in x3 into two linked blocks of 192 x 128 x 64 with halo exchange (kh_step_blocks)
    "torus_sane_192x128x128_weno5_2blocks": (3, None, None),
    # two of the paper's weak-scaling units (128^3 per GPU) as linked blocks on one GPU: a 128 x 128 x 256 periodic box
    "minkowski_2x128cubed_weno5_2blocks": (5, (128, 128, 256), 1),
    "minkowski_128_mc": (5, 128, 0), "minkowski_128_weno5": (5, 128, 1),
    "minkowski_256_mc": (5, 256, 0), "minkowski_256_weno5": (5, 256, 1),
    "minkowski_64_mc": (5, 64, 0), "minkowski_192_mc": (5, 192, 0), "minkowski_320_mc": (5, 320, 0),
    "minkowski_64_weno5": (5, 64, 1), "minkowski_192_weno5": (5, 192, 1), "minkowski_320_weno5": (5, 320, 1),
}
DEFAULT_WORKLOAD = "torus_sane_192x128x128_weno5"

# Algorithmic HBM bytes per interior zone and LAUNCH of each kernel kind (from
# SURVEY.md 8(d)): doubles read + written, x 8 B; geometry tables are 2-D and L2 resident (counted 0).
ALG_DOUBLES = {
    "flux": 8 + 7 + 1,            # P_s in; 7 flux components + ctop out
    "emf": 6 + 3,                 # 6 B-flux components in; 3 edge EMFs out
    "update_pred": 15 + 3 + 8 + 8,        # hydro fluxes, EMFs, P_i in; P_f out
    "update_corr": 15 + 3 + 8 + 8 + 3 + 8,  # + P_s and ctop in
}
ALG_BYTES_PER_ZONE_STEP = 8 * 193     # whole step, both sub-steps
# Algorithmic fp64 flops per zone and launch (FMA = 2, div/sqrt = 1): DESIGN.md "Rooflines"; ncu instruction
# counts (profiles/) are the check.  Keyed (kind, recon, flat).
ALG_FLOPS = {
    ("flux", 0, False): 460 + 120, ("flux", 1, False): 460 + 713,
    ("flux", 0, True): 250 + 120, ("flux", 1, True): 250 + 713,
    ("emf", 0, False): 24, ("emf", 1, False): 24, ("emf", 0, True): 24, ("emf", 1, True): 24,
    ("update", 0, False): 1076, ("update", 1, False): 1076, ("update", 0, True): 600, ("update", 1, True): 600,
}


# DRAM traffic per launch (bytes) of the default workload's kernels: dram__bytes_read.sum + dram__bytes_write.sum of one
# `ncu --set full` capture (update = mean of the predictor and the corrector launch).  Source file in profiles/.
NCU_DRAM_SOURCE = "profiles/r02_ncu_full.md"
NCU_DRAM_BYTES_PER_LAUNCH = {"flux1": 215.7e6 + 165.4e6, "flux2": 229.0e6 + 166.9e6, "flux3": 227.5e6 + 165.8e6, "emf": 159.6e6 + 53.5e6,
                             "update": 0.5 * (1068.7e6 + 192.4e6 + 728.5e6 + 190.5e6)}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)", {}


def workload_params(name):
    import kharm_inputs as ki
    cfg, n, recon = WORKLOADS[name]
    p = ki.config_params(cfg, n=n, recon=recon)
    if name.endswith("_kastaun"):
        p["inverter"] = ki.params.INV_KASTAUN
    if name.endswith("_fofc"):
        p["fofc"] = 1
    if name.endswith("_drift"):
        p["floor_frame"] = ki.params.FRAME_DRIFT
    if name.endswith("_facect") or name.endswith("_facect_upwind"):
        p["transport"] = ki.params.B_FACE_CT
    if name.endswith("_upwind"):
        p["emf"] = ki.params.EMF_UPWIND
    return cfg, p


def workload_state(name, p, seed):
    from kharm_inputs import modes, torus
    cfg = WORKLOADS[name][0]
    if cfg in (3, 4):
        return torus.torus_state(p, mad=(cfg == 4), seed=seed)
    return modes.config5(p, seed=seed, amp=1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="kh_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        with open(self.path) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
                except ValueError:
                    continue
                for nm, val in zip(names, c[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
        os.unlink(self.path)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


def oracle_sample_params(p):
    """Bounded sample of a workload for the CPU oracle: the same block cut to 32 zones in x3 with the same
    zone size (a quarter wedge for the torus) -- zone-cycles/s is a per-zone rate."""
    q = dict(p)
    if p["n3"] > 32:
        q["n3"] = 32
        q["xmax"] = list(p["xmax"])
        q["xmax"][2] = p["xmin"][2] + (p["xmax"][2] - p["xmin"][2]) * 32.0 / p["n3"]
    return q


def time_oracle(name, steps, warmup, seed=1, omp=True, full=False, budget_s=None):
    """Zone-cycles/s of the oracle as it stands: omp=True the OpenMP build of the same source (bit-identical to the
    single-thread one; tested), omp=False the single-thread library.  full=False cuts the block to 32 zones in x3.
    budget_s: stop after the first step that ends beyond this many seconds (at least one step is timed)."""
    from oracle import kho
    _, p = workload_params(name)
    q = dict(p) if full else oracle_sample_params(p)
    cfg = WORKLOADS[name][0]
    from kharm_inputs import modes, torus
    P0 = torus.torus_state(q, mad=(cfg == 4), seed=seed) if cfg in (3, 4) else modes.config5(q, seed=seed, amp=1e-3)
    g = kho.Grid(q, omp=omp)
    g.set_prims(P0)
    dt = g.estimate_dt()
    for _ in range(warmup):
        dt = g.step(dt)
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        dt = g.step(dt)
        done += 1
        if budget_s is not None and time.perf_counter() - t0 > budget_s:
            break
    el = time.perf_counter() - t0
    zones = q["n1"] * q["n2"] * q["n3"]
    if omp:
        cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    else:
        cores = 1
    what = "%s at %dx%dx%d%s" % (name, q["n1"], q["n2"], q["n3"], "" if full or q["n3"] == p["n3"] else " (cut in x3, same zone size)")
    return dict(value=zones * done / el, unit="zone-cycles/s", cores=cores, kind="oracle",
                sample="%s, %d steps after %d warm-up, oracle/%s" % (what, done, warmup, "libkho_omp.so" if omp else "libkho.so")), el / done * 1e3


def single_thread_leg(name, steps, budget_s):
    """SURVEY 8(d) 'Timing the oracle beside it': the single-threaded oracle pinned with `taskset -c 0` in a child
    process; returns its cpu_baseline dict with '1 of N cores' stated."""
    cmd = ["taskset", "-c", "0", sys.executable, os.path.abspath(__file__), "--oracle-leg", name, "--steps", str(steps),
           "--leg-budget", str(budget_s)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=max(600.0, 20 * budget_s))
        d = json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as e:       # taskset missing, oracle not built, ...: report, do not fail the GPU line
        return {"error": "%s: %s" % (type(e).__name__, str(e)[:200])}
    d["pinning"] = "taskset -c 0, 1 of %d cores" % (os.cpu_count() or 1)
    return d


def run_oracle_leg(args):
    cb, _ = time_oracle(args.oracle_leg, steps=args.steps, warmup=0, omp=False, full=True, budget_s=args.leg_budget)
    print(json.dumps(cb))
    return 0


def cpu_baseline_legs(workload, full_protocol):
    """The oracle timed on this box's host cores (a reported baseline, not the target).  `value` is the OpenMP build on
    all cores on the default bounded sample; `single_thread` holds the SURVEY 8(d) single-thread legs: config 5 at 64^3
    (MC and WENO5) and the full config-3 block.  full_protocol: 20 steps / 2 steps as 8(d) states (minutes of CPU work);
    otherwise each leg stops after the first step that ends beyond ~10 s, so the default run stays within a few minutes."""
    cb, _ = time_oracle(workload, steps=8, warmup=1)
    cb["label"] = "OpenMP build of the oracle, %d threads" % cb["cores"]
    budget = 1e9 if full_protocol else 10.0
    legs = {}
    for leg, steps in (("minkowski_64_mc", 20), ("minkowski_64_weno5", 20), ("torus_sane_192x128x128_weno5", 2)):
        legs[leg] = single_thread_leg(leg, steps, budget)
    cb["single_thread"] = legs
    cb["protocol"] = "SURVEY 8(d): 64^3 x 20 steps, config 3 x 2 steps" if full_protocol else \
        "bounded: each single-thread leg stops after the first step ending beyond 10 s (--cpu-full runs 20 / 2 steps)"
    return cb


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cb, ms = time_oracle(args.workload, args.steps, args.warmup)
    _, p = workload_params(args.workload)
    line = {"impl": "reference", "metric": "zone-cycles/sec (fp64 HARM step)", "value": cb["value"], "unit": "zone-cycles/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "n1": p["n1"], "n2": p["n2"], "n3": p["n3"],
                       "note": "CPU oracle on host cores; each step is a bounded sample of the workload"},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": "zone-cycles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def kernel_table(prof, steps, zones, recon, flat, hbm_peak, fp64_peak_tf):
    """Per kernel kind: ms per step, launches per step, achieved GB/s and TFLOP/s of the algorithmic work and
    the fraction of each roof; `bound` = the roof that takes longer for that kernel's algorithmic work."""
    rows = {}
    # The three flux directions of a sub-step run CONCURRENTLY (x2 and x3 on side streams): the library
    # then brackets the group as one entry under "flux1" and reports nothing for flux2 / flux3.  It is listed as "flux" here:
    # one launch group = the three kernels of one sub-step.
    grouped = prof.get("flux1", (0, 0))[1] > 0 and prof.get("flux2", (0, 0))[1] == 0 and prof.get("flux3", (0, 0))[1] == 0
    for kind, (ms, cnt) in prof.items():
        if cnt == 0:
            continue
        per_step, lps = ms / steps, cnt / steps
        if grouped and kind == "flux1":
            kind = "flux"
        row = {"ms_per_step": per_step, "launch_groups_per_step": lps}
        base = "flux" if kind.startswith("flux") else kind
        if base in ("flux", "emf", "update"):
            ndir = 3 if kind == "flux" else 1              # kernels per launch group
            if base == "update":   # one predictor + one corrector launch per step
                dbl = ALG_DOUBLES["update_pred"] + ALG_DOUBLES["update_corr"]
                nl = 2
            else:
                dbl, nl = ALG_DOUBLES[base] * 2 * ndir, 2 * ndir
            byts = 8.0 * dbl * zones                       # per step (nl launches)
            flops = ALG_FLOPS[(base, recon, flat)] * nl * zones
            t = per_step * 1e-3
            gbs, tfs = byts / t / 1e9, flops / t / 1e12
            t_hbm, t_alu = byts / (hbm_peak * 1e9), flops / (fp64_peak_tf * 1e12)
            row.update(alg_bytes_per_launch=byts / nl, alg_flops_per_launch=flops / nl, ms_per_launch=per_step / nl,
                       alg_bytes_per_step=byts, alg_flops_per_step=flops, kernel_launches_per_step=nl,
                       gbs=gbs, tflops=tfs, frac_hbm=gbs / hbm_peak, frac_alu=tfs / fp64_peak_tf,
                       bound="hbm" if t_hbm >= t_alu else "alu")
        rows[kind] = row
    return rows


class Ranks:
    """Replica plumbing of `--gpus N` (independent replicas, no data-path collective):
    RANK / LOCAL_RANK / WORLD_SIZE from the launcher's environment, a barrier and the max-over-ranks of a scalar.
    backend "nccl" on the GPU box; tests drive the same code with "gloo" on CPU (tests/test_bench_ranks.py)."""

    def __init__(self, backend="nccl"):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = backend
        self.dist = None
        if self.world > 1:
            import torch
            import torch.distributed as dist
            if backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            else:
                dist.init_process_group(backend)
            self.dist = dist

    def _device(self):
        return "cuda" if self.backend == "nccl" else "cpu"

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        if self.backend == "nccl":
            import torch
            torch.cuda.synchronize()

    def max(self, x):
        if self.dist is None:
            return float(x)
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self._device())
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_rate(self, units_per_rank, seconds_local):
        """Units all ranks processed / the slowest rank's time (every rank holds the same number of units)."""
        return self.world * units_per_rank / self.max(seconds_local)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
            self.dist = None


def run_blocks(args, kh, p, P0, stream, R, cfg):
    """`..._2blocks` workloads: the block cut in x3 into two linked blocks stepped by kh_step_blocks (halo exchange after
    U -> P and after the fix-up, dt_next = minimum over the blocks).  Device-resident timing only (direct launches)."""
    import torch
    K, W = args.steps, max(args.warmup, 3)
    n3 = p["n3"] // 2
    dx3 = (p["xmax"][2] - p["xmin"][2]) / p["n3"]
    parts = []
    for m in range(2):
        q = dict(p, n3=n3, xmin=list(p["xmin"]), xmax=list(p["xmax"]), bc=list(p["bc"]))
        q["xmin"][2] = p["xmin"][2] + m * n3 * dx3
        q["xmax"][2] = p["xmin"][2] + (m + 1) * n3 * dx3
        q["bc"][4] = q["bc"][5] = kh.BC_BLOCK             # x3 is periodic in every bench workload: both sides are linked
        parts.append(q)
    with torch.cuda.stream(stream):
        blocks = [kh.Grid(q, stream=stream.cuda_stream) for q in parts]
        kh.link_blocks(blocks[0], blocks[1], 3)
        kh.link_blocks(blocks[1], blocks[0], 3)
        for m, g in enumerate(blocks):
            g.set_prims(np.ascontiguousarray(P0[:, m * n3:(m + 1) * n3]))
        kh.exchange_halos(blocks)
        dt0 = min(g.estimate_dt() for g in blocks)
        clocks = ClockSampler(R.local)
        clocks.start()
        kh.step_blocks(blocks, dt0, sync=False)
        for _ in range(W - 1):
            kh.step_blocks(blocks, -1.0, sync=False)
        R.barrier()
        l0 = sum(g.launch_count() for g in blocks)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            kh.step_blocks(blocks, -1.0, sync=False)
        e1.record(stream)
        R.barrier()
        ms_total = R.max(e0.elapsed_time(e1))
        launches = sum(g.launch_count() for g in blocks) - l0
        clk = clocks.stop()
        assert all(np.isfinite(g.get_prims()).all() for g in blocks)
        divb = max(g.divB() for g in blocks)
    if R.rank != 0:
        R.close()
        return 0
    zones = p["n1"] * p["n2"] * p["n3"]
    hbm_peak, hbm_src, _ = load_peaks()
    ms_step = ms_total / K
    halo = 2 * 2 * 2 * 9 * 8 * 3 * (p["n1"] + 6) * (p["n2"] + 6)        # 2 sub-steps x 2 exchanges x 2 sides x (8 + flag) doubles x 3 layers
    line = {"metric": "zone-cycles/sec (fp64 HARM step)", "value": R.world * zones * K / (ms_total * 1e-3), "unit": "zone-cycles/s",
            "n_gpus": R.world, "steps": K, "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "baseline_config": cfg, "n1": p["n1"], "n2": p["n2"], "n3": p["n3"],
                       "blocks": "2 linked blocks of %dx%dx%d on one GPU, cut in x3 (periodic: both sides exchange)" % (p["n1"], p["n2"], n3),
                       "halo_bytes_per_block_step": halo, "launch": "direct launches (kh_step_blocks), device-resident dt"},
            "clocks": clk, "gpu_launches": int(launches), "e2e": None,
            "roofline_step": {"alg_bytes_per_zone_cycle": ALG_BYTES_PER_ZONE_STEP, "hbm_peak_gbs": hbm_peak,
                              "frac_hbm": ALG_BYTES_PER_ZONE_STEP * zones / (ms_step * 1e-3) / 1e9 / hbm_peak},
            "state": {"divB_max": divb}}
    print(json.dumps(line))
    R.close()
    return 0


def run_ours(args):
    import torch
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    R = Ranks("nccl")              # world 1: no process group
    rank, world, local = R.rank, R.world, R.local
    import paper_2408_01361_b200 as kh

    cfg, p = workload_params(args.workload)
    zones = p["n1"] * p["n2"] * p["n3"]
    flat = p["coords"] == 0
    P0 = workload_state(args.workload, p, seed=1 + rank)          # every replica its own seeded block
    stream = torch.cuda.Stream()
    K, W = args.steps, max(args.warmup, 3)
    barrier, max_over_ranks = R.barrier, R.max

    if args.workload.endswith("_2blocks"):
        return run_blocks(args, kh, p, P0, stream, R, cfg)
    with torch.cuda.stream(stream):
        g = kh.Grid(p, stream=stream.cuda_stream)
        g.set_prims(P0)
        if p.get("transport", 0) == 1:       # face-centred CT: a divergence-free poloidal loop on the faces (Stokes)
            from kharm_inputs import facefield
            g.set_face_B(*facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.5)))
        dt0 = g.estimate_dt()
        # ---- device-resident timing: W warm-up steps, then exactly K steps between two events on the grid's stream
        clocks = ClockSampler(local)      # samples the warm-up and the timed steps (both under load)
        clocks.start()
        g.step(dt0, sync=False)
        for _ in range(W - 1):
            g.step(-1.0, sync=False)
        barrier()
        l0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            g.step(-1.0, sync=False)
        e1.record(stream)
        barrier()
        ms_total = max_over_ranks(e0.elapsed_time(e1))
        launches = g.launch_count() - l0
        clk = clocks.stop()
        npf, nff = g.count_flags()
        divb = g.divB()
        assert np.isfinite(g.get_prims()).all(), "non-finite primitives after the timed steps"

        # ---- instrumented pass: events around every launch (no graph), same K steps
        g.set_profile(True)
        for _ in range(K):
            g.step(-1.0, sync=False)
        prof = g.get_profile()
        g.set_profile(False)

        # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
        hin = torch.from_numpy(P0).pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        a_in, a_out = hin.numpy(), hout.numpy()
        g.set_prims(a_in)
        dt = g.estimate_dt()
        Ke = max(3, min(K, 10))
        for _ in range(2):
            g.set_prims(a_in); dt = g.step(dt); g.get_prims(out=a_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            g.set_prims(a_in)
            dt = g.step(dt)
            g.get_prims(out=a_out)
            a_in, a_out = a_out, a_in
        torch.cuda.synchronize()
        e2e_s = max_over_ranks(time.perf_counter() - t0)
        state_bytes = 8 * 8 * zones
    if rank != 0:
        R.close()
        return 0

    hbm_peak, hbm_src, peaks = load_peaks()
    fp64_tf, fp64_mhz = kh.measure_fp64_peak()
    ms_step = ms_total / K
    value = world * zones * K / (ms_total * 1e-3)
    kern = kernel_table(prof, K, zones, p["recon"], flat, hbm_peak, fp64_tf)
    timed = {k: v for k, v in kern.items() if "bound" in v}
    # The three flux directions are ONE kernel template (flux_x1_kernel / flux_march_kernel<2|3> share the reconstruction
    # and the face flux): aggregate them before picking the dominant kernel of the step.
    fl = [kern[k] for k in ("flux", "flux1", "flux2", "flux3") if k in kern]
    groups = {k: v["ms_per_step"] for k, v in kern.items() if not k.startswith("flux")}
    if fl:
        groups["flux"] = sum(v["ms_per_step"] for v in fl)
    dom = max(groups, key=groups.get)
    if dom == "flux":
        nl = 6.0                                                   # kernel launches of the template per step (3 directions x 2 sub-steps)
        byts = sum(v["alg_bytes_per_step"] for v in fl)
        flops = sum(v["alg_flops_per_step"] for v in fl)
        t = groups["flux"] * 1e-3
        d = {"ms_per_launch": groups["flux"] / nl, "gbs": byts / t / 1e9, "tflops": flops / t / 1e12}
        d["frac_hbm"], d["frac_alu"] = d["gbs"] / hbm_peak, d["tflops"] / fp64_tf
        d["bound"] = "hbm" if byts / (hbm_peak * 1e9) >= flops / (fp64_tf * 1e12) else "alu"
        traffic = float(np.mean([NCU_DRAM_BYTES_PER_LAUNCH[k] for k in ("flux1", "flux2", "flux3")]))
    else:
        d = kern[dom]
        traffic = NCU_DRAM_BYTES_PER_LAUNCH.get(dom)
    roof = {"kernel": dom, "bound": d.get("bound"), "share_of_step": groups[dom] / sum(groups.values())}
    if d.get("bound") == "alu":
        roof.update(achieved=d["tflops"], peak=fp64_tf, unit="TFLOP/s", frac=d["frac_alu"],
                    peak_source="measured here: kh_measure_fp64_peak (DFMA chains)")
    else:
        roof.update(achieved=d.get("gbs"), peak=hbm_peak, unit="GB/s", frac=d.get("frac_hbm"), peak_source=hbm_src)
    roof["frac_hbm"], roof["frac_alu"] = d.get("frac_hbm"), d.get("frac_alu")
    # dram__bytes_read.sum + dram__bytes_write.sum per launch of that kernel from the committed ncu --set full capture
    # (not measurable in-process); only the default workload has one
    roof["traffic"] = traffic if args.workload == DEFAULT_WORKLOAD else None
    roof["traffic_source"] = NCU_DRAM_SOURCE if roof["traffic"] else None
    roof["ms_per_launch"] = d.get("ms_per_launch")
    prof_ms_step = sum(v["ms_per_step"] for v in kern.values())
    step_gbs = ALG_BYTES_PER_ZONE_STEP * zones / (ms_step * 1e-3) / 1e9
    step_flops = sum(v["alg_flops_per_step"] for v in timed.values())
    step_tf = step_flops / (ms_step * 1e-3) / 1e12
    t_hbm, t_alu = ALG_BYTES_PER_ZONE_STEP * zones / (hbm_peak * 1e9), step_flops / (fp64_tf * 1e12)

    cb = cpu_baseline_legs(args.workload, args.cpu_full) if not args.no_cpu else None
    line = {
        "metric": "zone-cycles/sec (fp64 HARM step)", "value": value, "unit": "zone-cycles/s", "n_gpus": world,
        "steps": K, "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "baseline_config": cfg, "n1": p["n1"], "n2": p["n2"], "n3": p["n3"],
                   "recon": "weno5" if p["recon"] else "mc", "coords": ("minkowski", "ks", "fmks")[p["coords"]],
                   "parallelism": "replicas x%d (no collective on the data path)" % world,
                   "l2": "working set %.2f GB per step >> 126 MB L2 (inputs larger than L2, no flush needed)"
                         % (54 * 8 * (p["n1"] + 6) * (p["n2"] + 6) * (p["n3"] + 6) / 1e9),
                   "launch": "CUDA-graph replay, device-resident dt"},
        "clocks": clk,
        "e2e": {"value": world * zones * Ke / e2e_s, "unit": "zone-cycles/s", "h2d_bytes_per_step": state_bytes,
                "d2h_bytes_per_step": state_bytes + 8, "steps": Ke,
                "how": "kh_set_prims(host pinned) + kh_step(dt)->dt_next + kh_get_prims(host pinned) every step"},
        "gpu_launches": int(launches),
        "roofline": roof,
        "roofline_step": {"alg_bytes_per_zone_cycle": ALG_BYTES_PER_ZONE_STEP, "alg_flops_per_zone_cycle": step_flops / zones,
                          "gbs": step_gbs, "frac_hbm": step_gbs / hbm_peak, "hbm_peak_gbs": hbm_peak, "hbm_peak_source": hbm_src,
                          "frac_hbm_nominal_8TBs": step_gbs / 8000.0,
                          "tflops": step_tf, "frac_alu": step_tf / fp64_tf, "fp64_peak_tflops": fp64_tf,
                          "fp64_peak_implied_sm_mhz": fp64_mhz, "bound": "hbm" if t_hbm >= t_alu else "alu",
                          "frac_of_binding_roof": max(t_hbm, t_alu) / (ms_step * 1e-3)},
        "kernels": kern,
        "instrumented_ms_per_step": prof_ms_step,
        "state": {"pflag_zones_last_substep": npf, "fflag_zones_last_substep": nff, "divB_max": divb},
        "cpu_baseline": cb,
        "paper_context": "KHARMA: ~21 M ZCPS/V100, ~35 M ZCPS/A100, ~25 M ZCPS/MI250X card (PAPER.md lines 429-433)",
    }
    print(json.dumps(line))
    R.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--cpu-full", action="store_true", help="single-thread oracle legs with SURVEY 8(d)'s full step counts")
    ap.add_argument("--oracle-leg", default=None, choices=sorted(WORKLOADS), help=argparse.SUPPRESS)   # child of single_thread_leg
    ap.add_argument("--leg-budget", type=float, default=10.0, help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_leg:
        return run_oracle_leg(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
