#!/usr/bin/env python
"""bench.py -- the headline measurement of the staggered mixed-precision CG hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config NAME]

One STEP = one full mixed-precision CG solve (mode 3: fp32 iteration on 12-real compressed
links -- the paper's single-precision kernel also reads compressed links, P:L113 -- with the
corrected restart + reliable + group-wise updates of section 3.2 done in fp64 on the full
18-real links, tol 1e-10) of A x = b on the
28^3 x 96 lattice of BASELINE.json configs[3] (the lattice the paper's numbers are quoted on,
P:L62): every row S1-S7 of the hot path runs.  `value` is the paper's own figure of merit,
"GFLOPS derived from the entire CG sequence" (Table 1 caption), with the flop
convention of DESIGN.md section 8: 1224 flop per even site per iteration (two 576-flop hops,
P:L62, plus 72 for the vector algebra).  Inputs are seeded synthetic fields (no MILC
configurations here); links, b and x are resident in HBM for `value`; `e2e` runs the same
solve through stag_cg_solve_host with b and x in pinned HOST memory (copies inside the timed
region; the gauge field stays resident, as it does across the many solves of one
configuration).  The dominant kernel (fp32 Dslash) is timed alone for the roofline.

--impl reference times the CPU oracle (oracle/) as it stands on the host cores on a bounded
sample (a fixed number of CG iterations of the same workload).
With N > 1 (torchrun) the path does not shard on this single-GPU design: N independent
replicas, weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE_HOP = 576
FLOP_PER_SITE_ITER = 2 * 576 + 72
METRIC = "mixed_cg_gflops"
UNIT = "GFLOPS"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f:
            c = [v.strip() for v in line.split(",")]
            if len(c) < 8:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            load = [v for v in sm if v >= 0.5 * max(sm)] or sm
            out["sm_mhz"] = statistics.median(load)
            out["sm_max_mhz"] = max(mx)
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def host_threads():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_sample(cfg, W, b, target_seconds: float):
    """Time the oracle's CG (as it stands) for a bounded number of iterations of the workload."""
    import oracle
    t0 = time.perf_counter()
    oracle.apply_A(b, W, cfg.dims, cfg.mass)
    t_a = time.perf_counter() - t0
    iters = int(max(3, min(1000, target_seconds / max(t_a * 1.15, 1e-6))))
    t0 = time.perf_counter()
    _, it, _, _, _ = oracle.cg(b, W, cfg.dims, cfg.mass, 1e-30, iters)
    dt = time.perf_counter() - t0
    return {"iters": it, "seconds": dt, "gflops": it * FLOP_PER_SITE_ITER * cfg.vh / dt * 1e-9}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same metric / config."""
    import fieldgen
    from paper_1111_0125_b200 import replicas
    rank, _, world = replicas.env_world()
    if rank != 0:
        return 0
    cfg = fieldgen.CONFIGS[args.config]
    W, b = cfg.links(), cfg.source()
    per_step = 6.0
    for _ in range(args.warmup):
        oracle_sample(cfg, W, b, 1.0)
    t_tot, it_tot = 0.0, 0
    for _ in range(args.steps):
        r = oracle_sample(cfg, W, b, per_step)
        t_tot += r["seconds"]; it_tot += r["iters"]
    value = it_tot * FLOP_PER_SITE_ITER * cfg.vh / t_tot * 1e-9
    cores = host_threads()
    sample = "%d oracle CG iterations (Fig. 1, fp64) per step on %s, plus the initial and final residual" % (it_tot // max(1, args.steps), cfg.name)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_tot / max(1, args.steps) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args.gpus, sample=sample),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(cfg, n_gpus, **extra):
    c = {"workload": "%s staggered mixed-precision CG solve (mode 3, fp32 iteration on 12-real links, fp64 updates on 18-real links), random SU(3) links with eta and antiperiodic-t folded in, Gaussian even-site source, m=%g, tol=%g" % (cfg.name, cfg.mass, cfg.tol),
         "dims": list(cfg.dims), "even_sites": cfg.vh, "mass": cfg.mass, "tol": cfg.tol,
         "maxiter": cfg.maxiter, "parallelism": "replicas x%d (no collective)" % n_gpus,
         "flop_convention": "1224 flop / even site / iteration = 2 x 576 (P:L62) + 72",
         "l2": "inputs exceed L2 (fp32 12-real links 405 MB per hop, 809 MB per iteration, fp64 links 1214 MB per update hop; 126 MB L2); the stand-alone Dslash timing rotates six input/output spinors"}
    c.update(extra)
    return c


def time_dslash(stag, torch, fieldgen, cfg, L, prec, launches=60, nrot=6):
    """Average device time of one Dslash hop launched alone, CUDA events on the launch stream.
    nrot input/output spinors rotate so neither they nor the links can live in L2."""
    ins = [stag.spinor_pack(fieldgen.spinor_gaussian(cfg.dims, 0, seed=100 + i), cfg.dims, prec) for i in range(nrot)]
    outs = [stag.empty_spinor(cfg.dims, prec) for _ in range(nrot)]
    for i in range(5):
        stag.dslash(ins[i % nrot], L, 1, prec, out=outs[i % nrot])
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(launches):
        stag.dslash(ins[i % nrot], L, 1, prec, out=outs[i % nrot])
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / launches
    f32 = prec in (stag.PREC_F32, stag.PREC_F32_R12, stag.PREC_F32_R8)
    reals = {stag.PREC_F64: 18, stag.PREC_F32: 18, stag.PREC_F64_R12: 12, stag.PREC_F32_R12: 12,
             stag.PREC_F64_R8: 8, stag.PREC_F32_R8: 8}[prec]
    bytes_site = (8 * reals + 6 + 6) * (4 if f32 else 8)        # 8 links + 1 vector in + 1 out
    paper_bytes = (8 * 18 + 8 * 6 + 6) * (4 if f32 else 8)      # P:L62 convention, no reuse
    return {"us": sec * 1e6, "algorithmic_bytes_per_site": bytes_site,
            "gbs": bytes_site * cfg.vh / sec * 1e-9, "gflops": FLOP_PER_SITE_HOP * cfg.vh / sec * 1e-9,
            "paper_convention_gbs": paper_bytes * cfg.vh / sec * 1e-9}


def time_dslash_mrhs(stag, torch, fieldgen, cfg, L, prec, nrhs, launches=30, nrot=3, layout=0):
    """The same for a batch of nrhs spinors through stag_dslash_batch (links read once per chunk of
    4 fp32 / 2 fp64 right-hand sides); layout 0 = blocked (stag_dslash_mrhs), 1 = paired."""
    srcs = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=300 + k) for k in range(nrhs)]
    ins = [stag.batch_convert(stag.spinor_pack_mrhs(srcs, cfg.dims, prec), cfg.dims, prec, layout) for _ in range(nrot)]
    outs = [torch.empty_like(ins[0]) for _ in range(nrot)]
    for i in range(3):
        stag.dslash_mrhs(ins[i % nrot], L, 1, prec, out=outs[i % nrot], layout=layout)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(launches):
        stag.dslash_mrhs(ins[i % nrot], L, 1, prec, out=outs[i % nrot], layout=layout)
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / launches
    f32 = prec in (stag.PREC_F32, stag.PREC_F32_R12)
    rows = 2 if prec in (stag.PREC_F64_R12, stag.PREC_F32_R12) else 3
    sz = 4 if f32 else 8
    chunks = -(-nrhs // (4 if f32 else 2))
    bytes_site = (chunks * 8 * 6 * rows + nrhs * 12) * sz       # links once per chunk + in/out per rhs
    return {"nrhs": nrhs, "us": sec * 1e6, "us_per_rhs": sec * 1e6 / nrhs,
            "algorithmic_bytes_per_site": bytes_site, "gbs": bytes_site * cfg.vh / sec * 1e-9,
            "gflops": FLOP_PER_SITE_HOP * nrhs * cfg.vh / sec * 1e-9}


def run_ours(args):
    import numpy as np
    import torch
    import fieldgen
    import paper_1111_0125_b200 as stag
    from paper_1111_0125_b200 import replicas

    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the hot path has no CPU fallback", file=sys.stderr)
        return 2
    rank, local, world = replicas.init("nccl")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    stag.lib()                                   # fail loudly here if libstag.so is missing
    cfg = fieldgen.CONFIGS[args.config]
    peak, peak_src = measured_peaks()

    # ---- setup (S0), timed separately ---------------------------------------------------------
    W = cfg.links()
    seed = replicas.replica_seed(fieldgen.SOURCE_SEED + cfg.index, rank)
    b_np = fieldgen.spinor_gaussian(cfg.dims, 0, seed)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    L = stag.Links(cfg.dims, W)
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    b_dev = stag.spinor_pack(b_np, cfg.dims, stag.PREC_F64)
    b_host = torch.from_numpy(b_np.view(np.float64).reshape(-1).copy()).pin_memory()
    x_host = torch.zeros_like(b_host).pin_memory()

    def solve_device():
        return stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)

    def solve_host():
        x_host.zero_()
        return stag.cg_solve_host(b_host, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, x_host=x_host, recon12=True)

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize(); replicas.barrier(); torch.cuda.synchronize()
        stag.reset_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        last = None
        for _ in range(steps):
            _, last = fn()
        e1.record()
        torch.cuda.synchronize(); replicas.barrier(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, last, stag.launch_count()

    sampler = ClockSampler(local) if rank == 0 else None
    sec, st, launches = timed(solve_device, args.steps, args.warmup)
    clocks = sampler.stop() if sampler else None
    flops_rank = args.steps * st["iters"] * FLOP_PER_SITE_ITER * cfg.vh
    agg = replicas.aggregate_throughput(flops_rank, sec, dev)

    sec_e2e, st_e2e, _ = timed(solve_host, args.steps, 1)
    agg_e2e = replicas.aggregate_throughput(args.steps * st_e2e["iters"] * FLOP_PER_SITE_ITER * cfg.vh, sec_e2e, dev)

    if rank != 0:
        replicas.finalize()
        return 0

    # ---- rank 0, N = any: the per-kernel numbers and the CPU baseline ---------------------------
    dsl = {stag.PREC_NAMES[p]: time_dslash(stag, torch, fieldgen, cfg, L, p) for p in range(4)}
    for p in (stag.PREC_F64_R8, stag.PREC_F32_R8):      # refused on fields with nearly-unit links
        try:
            dsl[stag.PREC_NAMES[p]] = time_dslash(stag, torch, fieldgen, cfg, L, p)
            dsl[stag.PREC_NAMES[p]]["rebuilt_entry_error"] = L.recon8_error(p)
        except stag.StagError as e:
            dsl[stag.PREC_NAMES[p]] = {"refused": str(e)}
    dom = dsl["fp32/12"]
    roofline = {"bound": "hbm", "kernel": "dslash_kernel<float,2,*> (fp32, 12-real links: the hop of the timed solve)",
                "achieved": dom["gbs"], "peak": peak, "unit": "GB/s", "frac": dom["gbs"] / peak,
                "peak_source": peak_src, "traffic": args.traffic if cfg.name == "c4_28^3x96" else None,
                "traffic_source": "profiles/r1e_dslash_fp32r12_ncu_full.md (dram__bytes_read.sum + dram__bytes_write.sum, one launch)",
                "algorithmic_bytes_per_launch": dom["algorithmic_bytes_per_site"] * cfg.vh,
                "us_per_launch": dom["us"], "frac_of_nominal_8TBs": dom["gbs"] / 8000.0}
    x64, st64 = stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_F64)
    x18, st18 = stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
    x64c, st64c = stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_F64, recon12=True)

    # several right-hand sides sharing each pass over the links: three
    # Gaussian sources in lockstep, and the batch hop alone
    b3 = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(cfg.dims, 0, seed + 1000 + k) for k in range(3)],
                               cfg.dims, stag.PREC_F64)
    x3, st3 = stag.cg_solve_mrhs(b3, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
    mrhs = {"nrhs": 3, "iters": [t["iters"] for t in st3], "true_resid": [t["true_resid"] for t in st3],
            "time_to_solution_s": st3[0]["seconds"],
            "gflops": sum(t["iters"] for t in st3) * FLOP_PER_SITE_ITER * cfg.vh / st3[0]["seconds"] * 1e-9,
            "us_per_iteration_per_rhs": st3[0]["seconds"] / max(1, max(t["iters"] for t in st3)) / 3 * 1e6,
            "dslash": {"%s x%d" % (stag.PREC_NAMES[p], n): time_dslash_mrhs(stag, torch, fieldgen, cfg, L, p, n, layout=stag.BATCH_PAIRED if p in (stag.PREC_F32, stag.PREC_F32_R12) else 0)
                       for p, n in ((stag.PREC_F32_R12, 2), (stag.PREC_F32_R12, 3), (stag.PREC_F32_R12, 4), (stag.PREC_F32, 4), (stag.PREC_F64, 2))},
            "dslash_blocked_layout": {"%s x%d" % (stag.PREC_NAMES[p], n): time_dslash_mrhs(stag, torch, fieldgen, cfg, L, p, n)
                                      for p, n in ((stag.PREC_F32_R12, 3), (stag.PREC_F32_R12, 4), (stag.PREC_F32, 4))},
            "layout": "fp32 batches paired (include/stag.h batch layouts), fp64 blocked"}
    del b3, x3

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample(cfg, W, b_np, 15.0)
        cpu = {"value": r["gflops"], "unit": UNIT, "cores": host_threads(), "kind": "oracle",
               "sample": "%d oracle CG iterations (Fig. 1, fp64) on %s, %.1f s" % (r["iters"], cfg.name, r["seconds"])}

    line = {
        "metric": METRIC, "value": agg["throughput"] * 1e-9, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": agg["seconds"] / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 iteration + f64 reliable updates", "data": "synthetic",
        "config": workload_config(cfg, world),
        "e2e": {"value": agg_e2e["throughput"] * 1e-9, "unit": UNIT,
                "h2d_bytes_per_step": 2 * cfg.vh * 48, "d2h_bytes_per_step": cfg.vh * 48,
                "ms_per_step": agg_e2e["seconds"] / args.steps * 1e3,
                "entry": "stag_cg_solve_host (b, x0 in pinned host memory -> x in host memory; links resident)"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "cg": {"iters": st["iters"], "n_updates": st["n_updates"], "applies_f64": st["applies_f64"],
               "fp32_share_of_A_applications": st["iters"] / (st["iters"] + st["applies_f64"]),
               "true_resid": st["true_resid"], "time_to_solution_s": st["seconds"],
               "ms_per_iteration": st["seconds"] / max(1, st["iters"]) * 1e3,
               "fp64_cg": {"iters": st64["iters"], "time_to_solution_s": st64["seconds"], "true_resid": st64["true_resid"]},
               "fp64_cg_12real_links": {"iters": st64c["iters"], "time_to_solution_s": st64c["seconds"], "true_resid": st64c["true_resid"]},
               "mixed_18real_links": {"iters": st18["iters"], "time_to_solution_s": st18["seconds"], "true_resid": st18["true_resid"],
                                      "ms_per_iteration": st18["seconds"] / max(1, st18["iters"]) * 1e3},
               "speedup_mixed_vs_fp64": st64["seconds"] / st["seconds"]},
        "dslash": dsl,
        "mrhs": mrhs,
        "setup_s0_seconds": setup_s,
        "paper_context": "GTX480: 145 GFLOPS SP / 55 DP per GPU pure-GPU CG (P:L131), 1.04 / 2.77 ms per Dirac op on a quarter lattice (Table 1)",
    }
    print(json.dumps(line), flush=True)
    replicas.finalize()
    return 0


def run_slabs(args):
    """--decomp slabs: ONE lattice split along time over the N ranks (strong scaling): the T-slab
    hop with peer-to-peer halo exchange and the slab CG with its global sums through peer memory
    (DESIGN.md section 14).  One process per GPU; torch.distributed only carries the IPC handles,
    the barrier around the timed region and the max over ranks of the time."""
    import numpy as np
    import torch
    import fieldgen
    import paper_1111_0125_b200 as stag
    from paper_1111_0125_b200 import replicas, slab

    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the hot path has no CPU fallback", file=sys.stderr)
        return 2
    rank, local, world = replicas.init("nccl")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    stag.lib()
    cfg = fieldgen.CONFIGS[args.config]
    peak, peak_src = measured_peaks()
    W = cfg.links()
    b_np = cfg.source()
    S = slab.SlabLinks(cfg.dims, W, rank, world)
    del W
    S.connect_distributed()
    b_loc = np.ascontiguousarray(slab.scatter_spinor(b_np, cfg.dims, rank, world))
    b_dev = stag.spinor_pack(b_loc, S.dims, stag.PREC_F64)
    b_host = torch.from_numpy(b_loc.view(np.float64).reshape(-1).copy()).pin_memory()
    x_host = torch.zeros_like(b_host).pin_memory()

    def solve_device():
        return S.cg_solve(b_dev, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)

    def solve_host():
        bd = stag.spinor_pack(b_host.to(dev, non_blocking=True), S.dims, stag.PREC_F64)
        x, st = S.cg_solve(bd, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
        x_host.copy_(stag.spinor_unpack(x, S.dims, stag.PREC_F64, to_numpy=False))
        return x, st

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize(); replicas.barrier(); torch.cuda.synchronize()
        stag.reset_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        last = None
        for _ in range(steps):
            _, last = fn()
        e1.record()
        torch.cuda.synchronize(); replicas.barrier(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, last, stag.launch_count()

    sampler = ClockSampler(local) if rank == 0 else None
    sec, st, launches = timed(solve_device, args.steps, args.warmup)
    clocks = sampler.stop() if sampler else None
    tmax = replicas.max_over_ranks(sec, dev)
    flops = args.steps * st["iters"] * FLOP_PER_SITE_ITER * cfg.vh          # the whole lattice
    sec_e2e, st_e2e, _ = timed(solve_host, args.steps, 1)
    tmax_e2e = replicas.max_over_ranks(sec_e2e, dev)

    # the slab hop alone (push + hop), this rank's share of the lattice
    vh_loc = cfg.vh // world
    prec = stag.PREC_F32_R12
    vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(fieldgen.spinor_gaussian(cfg.dims, 0, seed=100 + i), cfg.dims, rank, world)), S.dims, prec) for i in range(4)]
    outs = [stag.empty_spinor(S.dims, prec) for _ in range(4)]
    for i in range(4):
        S.dslash(vs[i], 1, prec, out=outs[i])
    torch.cuda.synchronize(); replicas.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(40):
        S.dslash(vs[i % 4], 1, prec, out=outs[i % 4])
    e1.record()
    torch.cuda.synchronize(); replicas.barrier()
    hop_us = replicas.max_over_ranks(e0.elapsed_time(e1) / 40 * 1e3, dev)
    if rank != 0:
        replicas.finalize()
        return 0
    hop_bytes = 432 * vh_loc
    line = {
        "metric": METRIC, "value": flops / tmax * 1e-9, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tmax / args.steps * 1e3, "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "f32 iteration + f64 reliable updates",
        "data": "synthetic",
        "config": workload_config(cfg, world, parallelism="T-slabs x%d: peer-to-peer halo exchange per hop, two global sums per iteration through peer memory" % world),
        "e2e": {"value": args.steps * st_e2e["iters"] * FLOP_PER_SITE_ITER * cfg.vh / tmax_e2e * 1e-9, "unit": UNIT,
                "h2d_bytes_per_step": cfg.vh * 48, "d2h_bytes_per_step": cfg.vh * 48,
                "ms_per_step": tmax_e2e / args.steps * 1e3,
                "entry": "slab.SlabLinks.cg_solve with each rank's b in pinned host memory and x copied back"},
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "face_push_kernel + dslash_kernel<float,2,PLAIN,1,HALO> on one slab",
                     "achieved": hop_bytes / hop_us * 1e-3, "peak": peak, "unit": "GB/s",
                     "frac": hop_bytes / hop_us * 1e-3 / peak, "peak_source": peak_src, "traffic": None,
                     "algorithmic_bytes_per_launch": hop_bytes, "us_per_launch": hop_us},
        "cpu_baseline": None,
        "cg": {"iters": st["iters"], "n_updates": st["n_updates"], "true_resid": st["true_resid"],
               "time_to_solution_s": st["seconds"], "ms_per_iteration": st["seconds"] / max(1, st["iters"]) * 1e3},
    }
    print(json.dumps(line), flush=True)
    replicas.finalize()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", default="c4_28^3x96")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--decomp", choices=["replicas", "slabs"], default="replicas",
                    help="N > 1: independent replicas (weak scaling, default) or one lattice in T-slabs (strong)")
    ap.add_argument("--traffic", type=float, default=436.2e6,
                    help="dram bytes (read + write) per launch of the dominant kernel from the ncu --set full "
                         "capture profiles/r1e_dslash_fp32r12_ncu_full.md (28^3x96, fp32/12 plain hop)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.decomp == "slabs":
        return run_slabs(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
