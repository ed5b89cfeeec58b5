#!/usr/bin/env python
"""bench.py -- the headline measurement of the staggered mixed-precision CG hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config NAME]
                    [--only all|hops|mrhs|solve] [--persistent auto|on|off] [--cpu-full] [--no-cpu-baseline] [--decomp replicas|slabs]

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

--only hops skips the solves and times the stand-alone hops alone (what the ncu captures under
profiles/ run); --cpu-full also runs the oracle's complete fp64 solve on the bench config (minutes).

--impl reference times the CPU oracle (oracle/) as it stands on the host cores on a bounded
sample (a fixed number of CG iterations of the same workload).
With N > 1 (torchrun) the path does not shard on this single-GPU design: N independent
replicas, weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import re
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


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def kernel_source_sha():
    """Identifies the build of the hop: sha256 over the device headers the hop is made of."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1111_0125_b200", "csrc")
    for name in ("stag_common.cuh", "stag_mem.cuh", "stag_dslash.cuh"):
        h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def traffic_from_profiles(kernel_tag: str, config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    newest profiles/*_ncu_full.md whose header lines
        traffic_kernel = <tag> / traffic_config = <config> / traffic_source_sha = <kernel_source_sha()>
        traffic_bytes_per_launch = <bytes>
    match this build; None (and why) otherwise -- never a number typed in from an older kernel."""
    pdir = os.path.join(ROOT, "profiles")
    sha = kernel_source_sha()
    best = None
    try:
        names = sorted(n for n in os.listdir(pdir) if n.endswith("_ncu_full.md"))
    except OSError:
        names = []
    for n in names:
        kv = dict(re.findall(r"^(traffic_\w+)\s*=\s*(.+?)\s*$", open(os.path.join(pdir, n)).read(), flags=re.M))
        if kv.get("traffic_kernel") == kernel_tag and kv.get("traffic_config") == config and kv.get("traffic_source_sha") == sha:
            try:
                best = (float(kv["traffic_bytes_per_launch"]), "profiles/" + n)
            except (KeyError, ValueError):
                pass
    if best:
        return best[0], best[1] + " (dram__bytes_read.sum + dram__bytes_write.sum, one launch, same kernel sources)"
    return None, "no ncu --set full capture under profiles/ matches this build of the hop (source sha %s)" % sha


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


def oracle_hop(cfg, W, b):
    """One oracle Dslash hop, best of 5 after one warm-up."""
    import oracle
    oracle.dslash(b, W, cfg.dims, 1)
    best = float("inf")
    for _ in range(5):
        t0 = time.perf_counter()
        oracle.dslash(b, W, cfg.dims, 1)
        best = min(best, time.perf_counter() - t0)
    return {"seconds": best, "gflops": FLOP_PER_SITE_HOP * cfg.vh / best * 1e-9,
            "paper_convention_gbs": 1584 * cfg.vh / best * 1e-9}


def oracle_solve(cfg, W, b):
    """The oracle's complete fp64 solve (Fig. 1) to the config's tolerance."""
    import oracle
    t0 = time.perf_counter()
    _, it, rho, restarts, rc = oracle.cg(b, W, cfg.dims, cfg.mass, cfg.tol, cfg.maxiter)
    dt = time.perf_counter() - t0
    return {"seconds": dt, "iters": it, "true_resid": rho, "restarts": restarts, "status": rc, "kind": "measured",
            "gflops": it * FLOP_PER_SITE_ITER * cfg.vh / dt * 1e-9}


def cpu_baseline_block(cfg, W, b, full: bool, iters_fp64=None):
    """cpu_baseline of the JSON line: the oracle as it stands (same source; built -O3 -march=native
    on this host for the timing) on a bounded CG sample of the bench
    workload, plus one hop (best of 5) and the complete fp64 solve -- measured on the configs the
    oracle finishes in seconds and with --cpu-full, otherwise extrapolated from the sample and
    labelled so."""
    import fieldgen
    import oracle
    flags = oracle.use_native_build()
    threads = oracle.max_threads()
    r = oracle_sample(cfg, W, b, 15.0)
    cpu = {"value": r["gflops"], "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": "%d oracle CG iterations (Fig. 1, fp64) on %s, %.1f s" % (r["iters"], cfg.name, r["seconds"]),
           "threads": threads, "nproc": os.cpu_count(), "affinity": host_threads(), "cpu_model": cpu_model(),
           "compile_flags": " ".join(flags), "hop": oracle_hop(cfg, W, b)}
    if full:
        cpu["solve"] = oracle_solve(cfg, W, b)
    elif iters_fp64:
        per_it = r["seconds"] / max(1, r["iters"])
        cpu["solve"] = {"seconds": per_it * iters_fp64, "iters": iters_fp64, "kind": "extrapolated: sample seconds per iteration x the %d iterations the GPU's fp64 CG needed (run with --cpu-full to measure)" % iters_fp64}
    others = {}
    for name in ("c1_4^4", "c2_8^4", "c3_16^3x32"):
        if name == cfg.name:
            continue
        c = fieldgen.CONFIGS[name]
        Wc, bc = c.links(), c.source()
        others[name] = {"hop": oracle_hop(c, Wc, bc), "solve": oracle_solve(c, Wc, bc)}
    return cpu, others


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same metric / config."""
    import fieldgen
    from paper_1111_0125_b200 import replicas
    rank, _, world = replicas.env_world()
    if rank != 0:
        return 0
    import oracle
    cfg = fieldgen.CONFIGS[args.config]
    W, b = cfg.links(), cfg.source()
    flags = oracle.use_native_build()
    per_step = 6.0
    for _ in range(args.warmup):
        oracle_sample(cfg, W, b, 1.0)
    t_tot, it_tot = 0.0, 0
    for _ in range(args.steps):
        r = oracle_sample(cfg, W, b, per_step)
        t_tot += r["seconds"]; it_tot += r["iters"]
    value = it_tot * FLOP_PER_SITE_ITER * cfg.vh / t_tot * 1e-9
    cores = oracle.max_threads()
    sample = "%d oracle CG iterations (Fig. 1, fp64) per step on %s, plus the initial and final residual" % (it_tot // max(1, args.steps), cfg.name)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_tot / max(1, args.steps) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args.gpus),      # the repo arm's dict exactly; the sample is in cpu_baseline
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "threads": cores, "nproc": os.cpu_count(), "affinity": host_threads(),
                         "cpu_model": cpu_model(), "compile_flags": " ".join(flags)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def link_kind(cfg):
    """The config's gauge field in words (fieldgen.CONFIGS; BASELINE.json configs)."""
    if cfg.kind == "smooth":
        return "smooth SU(3) links U = exp(i eps H), eps = %g" % cfg.eps
    return {"random": "random SU(3) links", "unit": "unit links (free field)"}.get(cfg.kind, cfg.kind + " links")


def workload_config(cfg, n_gpus, **extra):
    c = {"workload": "%s staggered mixed-precision CG solve (mode 3, fp32 iteration on 12-real links, fp64 updates on 18-real links), %s with eta and antiperiodic-t folded in, Gaussian even-site source, m=%g, tol=%g" % (cfg.name, link_kind(cfg), cfg.mass, cfg.tol),
         "dims": list(cfg.dims), "even_sites": cfg.vh, "mass": cfg.mass, "tol": cfg.tol,
         "maxiter": cfg.maxiter, "parallelism": "replicas x%d (no collective)" % n_gpus,
         "flop_convention": "1224 flop / even site / iteration = 2 x 576 (P:L62) + 72",
         "l2": "inputs exceed L2 (fp32 12-real links 405 MB per hop, 809 MB per iteration, fp64 links 1214 MB per update hop; 126 MB L2); the stand-alone Dslash timing rotates six input/output spinors"}
    c.update(extra)
    return c


def _time_batches(torch, launch, warmups=10, batches=12, per_batch=10):
    """10 warm-up launches, then >= 100 timed ones; CUDA events on the
    launch stream around batches of 10 back-to-back launches (an event pair per launch would add
    its own ~2 us to a 70 us kernel); returns (median, mean) seconds per launch over the batches."""
    for i in range(warmups):
        launch(i)
    torch.cuda.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(batches + 1)]
    k = warmups
    evs[0].record()
    for bi in range(batches):
        for _ in range(per_batch):
            launch(k)
            k += 1
        evs[bi + 1].record()
    torch.cuda.synchronize()
    per = [evs[i].elapsed_time(evs[i + 1]) * 1e-3 / per_batch for i in range(batches)]
    return statistics.median(per), sum(per) / len(per)


def time_dslash(stag, torch, fieldgen, cfg, L, prec, nrot=6):
    """Device time of one Dslash hop launched alone.  nrot input/output spinors rotate so neither
    they nor the links can live in L2."""
    ins = [stag.spinor_pack(fieldgen.spinor_gaussian(cfg.dims, 0, seed=100 + i), cfg.dims, prec) for i in range(nrot)]
    outs = [stag.empty_spinor(cfg.dims, prec) for _ in range(nrot)]
    sec, mean = _time_batches(torch, lambda i: stag.dslash(ins[i % nrot], L, 1, prec, out=outs[i % nrot]))
    f32 = prec in (stag.PREC_F32, stag.PREC_F32_R12, stag.PREC_F32_R8)
    reals = {stag.PREC_F64: 18, stag.PREC_F32: 18, stag.PREC_F64_R12: 12, stag.PREC_F32_R12: 12,
             stag.PREC_F64_R8: 8, stag.PREC_F32_R8: 8}[prec]
    bytes_site = (8 * reals + 6 + 6) * (4 if f32 else 8)        # 8 links + 1 vector in + 1 out
    paper_bytes = (8 * 18 + 8 * 6 + 6) * (4 if f32 else 8)      # P:L62 convention, no reuse
    return {"us": sec * 1e6, "us_mean": mean * 1e6, "timing": "median of 12 batches of 10 launches after 10 warm-ups",
            "algorithmic_bytes_per_site": bytes_site,
            "gbs": bytes_site * cfg.vh / sec * 1e-9, "gflops": FLOP_PER_SITE_HOP * cfg.vh / sec * 1e-9,
            "paper_convention_gbs": paper_bytes * cfg.vh / sec * 1e-9}


def time_dslash_mrhs(stag, torch, fieldgen, cfg, L, prec, nrhs, launches=30, nrot=3, layout=0):
    """The same for a batch of nrhs spinors through stag_dslash_batch (links read once per chunk of
    4 fp32 / 2 fp64 right-hand sides); layout 0 = blocked (stag_dslash_mrhs), 1 = paired."""
    srcs = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=300 + k) for k in range(nrhs)]
    ins = [stag.batch_convert(stag.spinor_pack_mrhs(srcs, cfg.dims, prec), cfg.dims, prec, layout) for _ in range(nrot)]
    outs = [torch.empty_like(ins[0]) for _ in range(nrot)]
    sec, mean = _time_batches(torch, lambda i: stag.dslash_mrhs(ins[i % nrot], L, 1, prec, out=outs[i % nrot], layout=layout))
    f32 = prec in (stag.PREC_F32, stag.PREC_F32_R12)
    rows = 2 if prec in (stag.PREC_F64_R12, stag.PREC_F32_R12) else 3
    sz = 4 if f32 else 8
    chunks = -(-nrhs // (4 if f32 else 2))
    bytes_site = (chunks * 8 * 6 * rows + nrhs * 12) * sz       # links once per chunk + in/out per rhs
    return {"nrhs": nrhs, "us": sec * 1e6, "us_mean": mean * 1e6, "us_per_rhs": sec * 1e6 / nrhs,
            "algorithmic_bytes_per_site": bytes_site, "gbs": bytes_site * cfg.vh / sec * 1e-9,
            "gflops": FLOP_PER_SITE_HOP * nrhs * cfg.vh / sec * 1e-9}


def hop_timings(stag, torch, fieldgen, cfg, L, select=None):
    """Stand-alone hops: the six single forms and the batch hops.  select: names to run (--hops),
    e.g. {"fp32/12", "fp32/12 x4"}; None = all."""
    want = (lambda name: True) if not select else (lambda name: name in select)
    dsl = {stag.PREC_NAMES[p]: time_dslash(stag, torch, fieldgen, cfg, L, p) for p in range(4) if want(stag.PREC_NAMES[p])}
    for p in (stag.PREC_F64_R8, stag.PREC_F32_R8):      # refused on fields with nearly-unit links
        if not want(stag.PREC_NAMES[p]):
            continue
        try:
            dsl[stag.PREC_NAMES[p]] = time_dslash(stag, torch, fieldgen, cfg, L, p)
            dsl[stag.PREC_NAMES[p]]["rebuilt_entry_error"] = L.recon8_error(p)
        except stag.StagError as e:
            dsl[stag.PREC_NAMES[p]] = {"refused": str(e)}
    f32 = (stag.PREC_F32, stag.PREC_F32_R12)
    batch = {"%s x%d" % (stag.PREC_NAMES[p], n): time_dslash_mrhs(stag, torch, fieldgen, cfg, L, p, n, layout=stag.BATCH_PAIRED if p in f32 else 0)
             for p, n in ((stag.PREC_F32_R12, 2), (stag.PREC_F32_R12, 3), (stag.PREC_F32_R12, 4), (stag.PREC_F32, 4), (stag.PREC_F64, 2))
             if want("%s x%d" % (stag.PREC_NAMES[p], n))}
    blocked = {"%s x%d" % (stag.PREC_NAMES[p], n): time_dslash_mrhs(stag, torch, fieldgen, cfg, L, p, n)
               for p, n in ((stag.PREC_F32_R12, 3), (stag.PREC_F32_R12, 4), (stag.PREC_F32, 4))
               if want("%s x%d blocked" % (stag.PREC_NAMES[p], n))}
    return dsl, batch, blocked


def propagator_timings(stag, torch, cfg, L, peak):
    """The production call (eq. 2.2): stag_solve_M, the
    staggered propagator (D + m) psi = h, for the three colour point sources of one site (nrhs = 3)
    and of four sites (nrhs = 12: three chunks of four, the links re-read once per chunk).  The whole
    call is timed (CUDA events on the stream the library launches on): b_e = m h_e - D_eo h_o, the
    lockstep mixed-precision solve, psi_o = (h_o - D_oe psi_e) / m.  byte floor per source and pass:
    2 hops x 384 B of 12-real links shared by the chunk + 14 vector passes x 24 B."""
    n = stag.spinor_bytes(cfg.dims, stag.PREC_F64) // 8          # reals per device spinor
    vh_pad = n // 6
    out = {}
    for nsites in (1, 4):
        nrhs = 3 * nsites
        he = torch.zeros((nrhs, n), dtype=torch.float64, device="cuda")
        ho = torch.zeros_like(he)
        for j in range(nsites):
            cb = (12345 + 77777 * j) % cfg.vh                    # odd-parity checkerboard index of the source site
            for c in range(3):
                ho[3 * j + c, (c * vh_pad + cb) * 2] = 1.0       # Re of colour c at that site (device layout v[c][cb])
        stag.solve_M(he, ho, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)      # warm-up: graphs, workspace
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        pe, po, sts = stag.solve_M(he, ho, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
        e1.record()
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3
        iters = [t["iters"] for t in sts]
        chunk = min(nrhs, 4)
        floor_bytes = (2 * 384.0 / chunk + 14 * 24.0) * cfg.vh
        us = sec / max(1, max(iters)) / nrhs * 1e6
        out["nrhs_%d" % nrhs] = {
            "sources": "%d site(s) x 3 colours, point sources on odd sites" % nsites,
            "status": [t["status"] for t in sts], "iters": iters, "true_resid_max": max(t["true_resid"] for t in sts),
            "time_to_solution_s": sec, "cg_seconds": sts[0]["seconds"],
            "gflops": sum(iters) * FLOP_PER_SITE_ITER * cfg.vh / sec * 1e-9,
            "us_per_iteration_per_source": us,
            "byte_floor_us_per_iteration_per_source": floor_bytes / peak * 1e-3,
            "frac_of_byte_floor": floor_bytes / peak * 1e-3 / us,
            "links_passes_per_hop": (nrhs + 3) // 4}
        del he, ho, pe, po
    return out


def roofline_block(dsl, cfg, peak, peak_src):
    dom = dsl["fp32/12"]
    traffic, traffic_src = traffic_from_profiles("dslash_kernel<float,2,HOP_PLAIN,1>", cfg.name)
    return {"bound": "hbm", "kernel": "dslash_kernel<float,2,*> (fp32, 12-real links: the hop of the timed solve)",
            "achieved": dom["gbs"], "peak": peak, "unit": "GB/s", "frac": dom["gbs"] / peak,
            "peak_source": peak_src, "traffic": traffic, "traffic_source": traffic_src,
            "algorithmic_bytes_per_launch": dom["algorithmic_bytes_per_site"] * cfg.vh,
            "us_per_launch": dom["us"], "us_per_launch_mean": dom["us_mean"], "timing": dom["timing"],
            "frac_of_nominal_8TBs": dom["gbs"] / 8000.0}


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

    if args.only == "hops":                      # what the ncu captures under profiles/ run
        if rank == 0:
            select = set(v.strip() for v in args.hops.split(",")) if args.hops else None
            dsl, batch, blocked = hop_timings(stag, torch, fieldgen, cfg, L, select)
            out = {"only": "hops", "config": {"workload": cfg.name}, "dslash": dsl,
                   "mrhs_dslash": batch, "mrhs_dslash_blocked_layout": blocked}
            if "fp32/12" in dsl:
                out["roofline"] = roofline_block(dsl, cfg, peak, peak_src)
            print(json.dumps(out), flush=True)
        replicas.finalize()
        return 0

    if args.only == "mrhs":
        if rank == 0:
            b3 = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(cfg.dims, 0, seed + 1000 + k) for k in range(3)],
                                       cfg.dims, stag.PREC_F64)
            x3, st3 = stag.cg_solve_mrhs(b3, L, cfg.mass, cfg.tol, args.maxiter or cfg.maxiter, stag.CG_RELIABLE, recon12=True)
            print(json.dumps({"only": "mrhs", "config": {"workload": cfg.name}, "nrhs": 3,
                              "iters": [t["iters"] for t in st3], "time_to_solution_s": st3[0]["seconds"],
                              "us_per_iteration_per_rhs": st3[0]["seconds"] / max(1, max(t["iters"] for t in st3)) / 3 * 1e6}), flush=True)
        replicas.finalize()
        return 0

    if args.only == "solve":                     # the timed solve alone: what the in-place ncu captures run
        if rank == 0:
            b_dev = stag.spinor_pack(b_np, cfg.dims, stag.PREC_F64)
            kw = {} if args.persistent == "auto" else {"persistent": args.persistent == "on"}
            for _ in range(max(1, args.steps)):
                _, st = stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, args.maxiter or cfg.maxiter, stag.CG_RELIABLE, recon12=True, **kw)
            print(json.dumps({"only": "solve", "config": {"workload": cfg.name}, "persistent": args.persistent,
                              "iters": st["iters"], "time_to_solution_s": st["seconds"],
                              "us_per_iteration": st["seconds"] / max(1, st["iters"]) * 1e6}), flush=True)
        replicas.finalize()
        return 0

    b_dev = stag.spinor_pack(b_np, cfg.dims, stag.PREC_F64)
    b_host = torch.from_numpy(b_np.view(np.float64).reshape(-1).copy()).pin_memory()
    x_host = torch.zeros_like(b_host).pin_memory()
    # the caller owns the workspace (include/stag.h): one allocation for all the solves below
    ws = torch.empty(max(stag.cg_workspace_bytes(cfg.dims, m, 3) for m in (stag.CG_F64, stag.CG_RELIABLE)),
                     dtype=torch.uint8, device="cuda")
    stag.set_workspace(ws)

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
    dsl, batch, blocked = hop_timings(stag, torch, fieldgen, cfg, L)
    roofline = roofline_block(dsl, cfg, peak, peak_src)

    def brief(t, **extra):
        d = {"iters": t["iters"], "n_updates": t["n_updates"], "applies_f64": t["applies_f64"],
             "time_to_solution_s": t["seconds"], "true_resid": t["true_resid"],
             "ms_per_iteration": t["seconds"] / max(1, t["iters"]) * 1e3}
        d.update(extra)
        return d

    def solve(mode, **kw):
        stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, mode, **kw)      # warm: graph instantiated, links derived
        return stag.cg_solve(b_dev, L, cfg.mass, cfg.tol, cfg.maxiter, mode, **kw)[1]

    # the iteration as one persistent kernel per <= 1024 passes against the kernel-per-step CUDA graph
    # (DESIGN.md section 17); the timed solve above let the library choose by volume
    st_pk = solve(stag.CG_RELIABLE, recon12=True, persistent=True)
    st_ks = solve(stag.CG_RELIABLE, recon12=True, persistent=False)
    st64 = solve(stag.CG_F64)
    st18 = solve(stag.CG_RELIABLE)
    st64c = solve(stag.CG_F64, recon12=True)
    # Fig. 2 (defect correction: a fresh inner CG per outer step) against section 3.2
    # (direction kept across restarts + reliable / group-wise updates): same links, same
    # source, same tolerance.  P:L84 "preserving the total number of CG iterations"
    # "significantly faster convergence" of the corrected scheme.
    st_dc = solve(stag.CG_DEFECT, recon12=True)
    eps_sweep = {}
    for eps in (0.1, 0.2, 0.3, 0.5):             # eps_in is never given a value
        eps_sweep["%.1f" % eps] = brief(solve(stag.CG_RELIABLE, recon12=True, eps_in=eps))
    dc_sweep = {}
    for eps in (1e-1, 1e-2, 1e-3):
        dc_sweep["%g" % eps] = brief(solve(stag.CG_DEFECT, recon12=True, eps_in=eps))

    # several right-hand sides sharing each pass over the links: three
    # Gaussian sources in lockstep
    b3 = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(cfg.dims, 0, seed + 1000 + k) for k in range(3)],
                               cfg.dims, stag.PREC_F64)
    stag.cg_solve_mrhs(b3, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
    x3, st3 = stag.cg_solve_mrhs(b3, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
    mrhs = {"nrhs": 3, "iters": [t["iters"] for t in st3], "true_resid": [t["true_resid"] for t in st3],
            "time_to_solution_s": st3[0]["seconds"],
            "gflops": sum(t["iters"] for t in st3) * FLOP_PER_SITE_ITER * cfg.vh / st3[0]["seconds"] * 1e-9,
            "us_per_iteration_per_rhs": st3[0]["seconds"] / max(1, max(t["iters"] for t in st3)) / 3 * 1e6,
            "dslash": batch, "dslash_blocked_layout": blocked,
            "layout": "fp32 batches paired (include/stag.h batch layouts), fp64 blocked"}
    del b3, x3
    stag.set_workspace(None)
    propagator = propagator_timings(stag, torch, cfg, L, peak)

    cpu, cpu_others = None, None
    if world == 1 and not args.no_cpu_baseline:
        cpu, cpu_others = cpu_baseline_block(cfg, W, b_np, args.cpu_full, iters_fp64=st64["iters"])

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
        "cpu_baseline_other_configs": cpu_others,
        "cg": {"iters": st["iters"], "n_updates": st["n_updates"], "applies_f64": st["applies_f64"],
               "fp32_share_of_A_applications": st["iters"] / (st["iters"] + st["applies_f64"]),
               "true_resid": st["true_resid"], "time_to_solution_s": st["seconds"],
               "ms_per_iteration": st["seconds"] / max(1, st["iters"]) * 1e3,
               "iteration_path": "chosen by volume (params.persistent = 0): %s" % (
                   "persistent kernel" if cfg.vh <= 300000 else "kernel per step, CUDA graph of 32 passes"),
               "persistent_kernel": brief(st_pk),
               "kernel_per_step": brief(st_ks),
               "fp64_cg": brief(st64),
               "fp64_cg_12real_links": brief(st64c),
               "mixed_18real_links": brief(st18),
               "defect_correction": brief(st_dc, outer_steps=st_dc["n_updates"], eps_in=1e-2,
                                          iters_vs_reliable=st_dc["iters"] / max(1, st["iters"]),
                                          time_vs_reliable=st_dc["seconds"] / st["seconds"]),
               "defect_correction_eps_in_sweep": dc_sweep,
               "reliable_eps_in_sweep": eps_sweep,
               "speedup_mixed_vs_fp64": st64["seconds"] / st["seconds"]},
        "dslash": dsl,
        "mrhs": mrhs,
        "propagator": propagator,
        "setup_s0_seconds": setup_s,
        "workspace": "caller-owned (stag_set_workspace), %d bytes" % ws.numel(),
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
    # each rank generates and hands over only its own time slices of the links plus the t-links of
    # the slice before them (stag_slab_create_local): no rank ever holds the whole gauge field
    t0, t1 = slab.slab_range(cfg.dims, rank, world)
    W_loc = cfg.links_slices(t0, t1 - t0)
    W_back = np.ascontiguousarray(cfg.links_slices(t0 - 1, 1)[3])
    b_np = cfg.source()
    S = slab.SlabLinks(cfg.dims, W_loc, rank, world, W_back=W_back)
    del W_loc, W_back
    S.connect_distributed()
    replicas.barrier()          # rank skew counts against the slab watchdog: start the first exchange together
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
    # the same solve on the kernel-per-step slab path (six launches per pass, a CUDA graph per 32 passes)
    S.cg_solve(b_dev, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True, persistent=False)
    replicas.barrier()
    _, st_step = S.cg_solve(b_dev, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True, persistent=False)
    step_path = {"iters": st_step["iters"], "time_to_solution_s": replicas.max_over_ranks(st_step["seconds"], dev),
                 "ms_per_iteration": replicas.max_over_ranks(st_step["seconds"], dev) / max(1, st_step["iters"]) * 1e3}
    S.cg_solve(b_dev, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True, persistent=True)
    replicas.barrier()
    _, st_pers = S.cg_solve(b_dev, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True, persistent=True)
    pers_path = {"iters": st_pers["iters"], "time_to_solution_s": replicas.max_over_ranks(st_pers["seconds"], dev),
                 "ms_per_iteration": replicas.max_over_ranks(st_pers["seconds"], dev) / max(1, st_pers["iters"]) * 1e3}
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
               "time_to_solution_s": st["seconds"], "ms_per_iteration": st["seconds"] / max(1, st["iters"]) * 1e3,
               "iteration_path": "chosen by volume (params.persistent = 0): %s" % (
                   "persistent kernel, one cooperative launch per <= 1024 passes" if world == 1 and cfg.vh <= 800000
                   else "kernel per step, CUDA graph of 32 passes"),
               "persistent_kernel": pers_path, "kernel_per_step": step_path},
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
    ap.add_argument("--only", choices=["all", "hops", "mrhs", "solve"], default="all",
                    help="hops: time the stand-alone hops only; mrhs: only the three-source lockstep solve; "
                         "solve: only the mixed solve (the commands the ncu captures under profiles/ run)")
    ap.add_argument("--persistent", choices=["auto", "on", "off"], default="auto",
                    help="with --only solve: force the persistent-kernel iteration on or off")
    ap.add_argument("--maxiter", type=int, default=0, help="with --only mrhs: cap the iterations (0 = the config's)")
    ap.add_argument("--hops", default="",
                    help='with --only hops: comma-separated names to run, e.g. "fp32/12,fp32/12 x4,fp32/12 x4 blocked"')
    ap.add_argument("--cpu-full", action="store_true",
                    help="also run the oracle's complete fp64 solve on the bench config (minutes of CPU)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.decomp == "slabs":
        return run_slabs(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
