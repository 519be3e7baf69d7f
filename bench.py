#!/usr/bin/env python
"""Benchmark of the diffuse-radiation ray sweep (BASELINE.json metric: ray-segment updates/sec on
one B200 and % of the HBM/L2 roofline; oracle host time beside it).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A step = one rt_sweep over all directions ("one iteration") of the synthetic workload.
Prints ONE JSON line (rank 0).  The headline (`value`, `e2e`, `roofline`) is config C4 (256^3 x 3072 directions,
the config BASELINE.json's metric is quoted on); the default run also times the other four configs (3 steps
each) and adds them under "configs" ("report for every config").
For N > 1 (torchrun) every rank sweeps a full replica ("replicas only": north_star fixes one GPU; DESIGN.md
"Multi-GPU"), or, with --shard directions, its share of the directions followed by one all-reduce.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ray_segment_updates_per_sec"
UNIT = "updates/s"
ALGO_BYTES_PER_CELL_DIR_BIN = 16.0     # read kappa,S (8 B) + read-modify-write J accumulator (8 B), SURVEY 8(d)
# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per cell-direction-bin of the hot kernel, from committed
# ncu captures; valid only for the kernel sources whose git blob hashes the table names (see traffic_table()).
TRAFFIC_TABLE = os.path.join(ROOT, "profiles", "dram_traffic.json")
KERNEL_SOURCES = ["paper_1410_0763_b200/csrc/rt_sweep.cuh", "paper_1410_0763_b200/csrc/rt_api.cu",
                  "paper_1410_0763_b200/csrc/rt_internal.h"]
# memory level the 16-byte model is held against, per config: the level that holds the fields
BOUND = {"C1": "l2", "C2": "l2", "C3": "l2", "C4": "hbm", "C5": "hbm"}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def git_blob_sha(path):
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def traffic_table():
    """The ncu-measured DRAM bytes per cell-direction-bin, if the table was taken with exactly these kernel sources."""
    try:
        t = json.load(open(TRAFFIC_TABLE))
    except Exception:
        return {}, "no table"
    for rel, sha in t.get("kernel_sources", {}).items():
        if git_blob_sha(os.path.join(ROOT, rel)) != sha:
            return {}, "stale: %s changed since the ncu capture" % rel
    return t.get("entries", {}), "ok"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, reasons = [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1]))
                out["sm_max_mhz"] = float(r[2])
                for n, v in zip(names, r[5:9]):
                    if v.strip().lower() == "active":
                        reasons.add(n)
            except Exception:
                continue
        if sm:
            out["sm_mhz"] = float(np.median(sm))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def host_cores():
    try:
        return max(1, min(len(os.sched_getaffinity(0)), 32))
    except AttributeError:
        return max(1, min(os.cpu_count() or 1, 32))


def oracle_rate(oracle, kap, S, dirs, nd, cores, nbins):
    """The oracle as it stands on `nd` directions spread over the set, `cores` OpenMP threads."""
    stride = max(1, dirs.shape[0] // nd)
    sub = dirs[::stride][:nd]
    t0 = time.perf_counter()
    r = oracle.sweep(kap, S, sub, nthreads=cores, want_counts=False)
    dt = time.perf_counter() - t0
    return r["seg_total"] * nbins / dt, dt, len(sub), stride


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on all host cores; each step is a bounded sample (a subset
    of the directions, full mesh) of the same workload, sized so that the whole run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle
    from rt_inputs import make_fields, CONFIGS
    spec = CONFIGS[args.config]
    kap, S = make_fields(args.config)
    dirs = oracle.healpix_dirs(spec.nside)
    cores = host_cores()
    if args.ref_dirs:
        nd = args.ref_dirs
    else:
        # the same sample as the cpu_baseline leg of the GPU arm (--cpu-dirs, 96 directions: about 12 s per step at C4),
        # whatever --steps is, so that the two legs quote one rate: with fewer directions per step each thread's
        # start-up cost (its private accumulators are allocated and first touched per call) weighs more and the rate
        # drops (round 2's driver record: 1.34e8 with 32 per step against 2.02e8 with 96).  Only a run of more than
        # 24 steps is thinned, to stay within a few minutes.
        nd = args.cpu_dirs if args.steps <= 24 else max(cores, (args.cpu_dirs * 24 // args.steps) // cores * cores)
    nd = max(1, min(spec.ndirs, nd))
    stride = max(1, spec.ndirs // nd)
    sub = dirs[::stride][:nd]
    for _ in range(1 if args.warmup > 0 else 0):
        oracle.sweep(kap, S, sub[:cores], nthreads=cores, want_counts=False)
    t0 = time.perf_counter()
    upd = 0
    for _ in range(args.steps):
        r = oracle.sweep(kap, S, sub, nthreads=cores, want_counts=False)
        upd += r["seg_total"] * spec.nbins
    dt = time.perf_counter() - t0
    val = upd / dt
    sample = "%d of %d directions per step (every %dth), full mesh, %d threads" % (len(sub), spec.ndirs, stride, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(spec), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(), "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_point(args):
    """--workload point: one JSON line of its own."""
    print(json.dumps(point_line(args, cpu=not args.no_cpu_baseline)))


def point_line(args, cpu=True):
    """rt_point_sources on the config's mesh and kappa with seeded sources (one at a box corner, one at the centre,
    the rest uniform in the box, positions in 1/256 cell): the record --workload point prints, also carried by the
    default line under "point" so that the driver's record holds the paper's second workload."""
    import torch
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields, CONFIGS
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    spec = CONFIGS[args.config]
    kap, S = make_fields(args.config)
    nx, ny, nz = spec.dims
    rng = np.random.default_rng(100 + spec.seed)
    src = np.stack([rng.integers(0, 256 * nx + 1, args.sources), rng.integers(0, 256 * ny + 1, args.sources),
                    rng.integers(0, 256 * nz + 1, args.sources)], 1).astype(np.int32)
    src[0] = 0
    if args.sources > 1:
        src[1] = [128 * nx, 128 * ny, 128 * nz]
    lum = rng.uniform(0.5, 2.0, (args.sources, spec.nbins))
    tr = rt.RayTracer(spec.dims, spec.nbins, rt.healpix_dirs(1))
    tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
    _, _, steps = tr.point_sources(src, lum, want_steps=True)
    for _ in range(max(args.warmup, 3)):
        tr.point_sources(src, lum)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        Q, _, _ = tr.point_sources(src, lum)
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / args.steps
    tr.close()
    want_cpu, cpu = cpu, None
    if want_cpu:
        from oracle import oracle
        ns = min(args.sources, 2)
        t0 = time.perf_counter()
        r = oracle.point_sources(kap, src[:ns], lum[:ns], want_diag=False)
        dt = time.perf_counter() - t0
        cpu = {"value": r["steps"] * spec.nbins / dt, "unit": "ray steps/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "%d of %d sources, full mesh, %.1f s" % (ns, args.sources, dt)}
    # issue-slot ceiling: the kernel is bound by instruction issue, not by memory.  Executed
    # thread-instructions per ray step come from the committed ncu capture, valid for the kernel source it names.
    roof, note = None, "no committed instruction count for this kernel source"
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "point_sources.json")))
        if git_blob_sha(os.path.join(ROOT, t["kernel_source"])) == t["kernel_source_sha"]:
            props = torch.cuda.get_device_properties(0)
            clk = 1e6 * float(clocks.get("sm_max_mhz") or 1965.0)
            peak = props.multi_processor_count * 4 * 32 * clk          # 4 schedulers x 1 warp-instruction per clock x 32 lanes
            ach = float(t["thread_instructions_per_ray_step"]) * steps * spec.nbins / (ms * 1e-3)
            roof = {"bound": "alu", "achieved": ach, "peak": peak, "unit": "thread-instructions/s", "frac": ach / peak,
                    "traffic": None, "thread_instructions_per_ray_step": t["thread_instructions_per_ray_step"],
                    "peak_kind": "SMs x 4 schedulers x 32 lanes x max SM clock (issue slots)", "source": t["source"]}
            note = "issue-bound gather along long characteristics; DRAM traffic is negligible (kappa is L2-resident)"
        else:
            note = "stale: %s changed since the ncu capture" % t["kernel_source"]
    except Exception:
        pass
    return {
        "metric": "point_source_ray_steps_per_sec", "value": steps * spec.nbins / (ms * 1e-3), "unit": "ray steps/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 path sums over f32 kappa", "data": "synthetic",
        "config": {"workload": "point sources on " + workload_name(spec), "sources": args.sources,
                   "ray_steps_per_step": steps * spec.nbins, "rays_per_step": args.sources * spec.ncell * spec.nbins},
        "clocks": clocks, "gpu_launches": args.steps,
        "roofline": roof, "note": note,
        "cpu_baseline": cpu}


def run_probe(args):
    """--probe: the streaming bandwidth probe of the library (rt_probe_bandwidth) over L2- and HBM-sized buffers."""
    import torch
    import paper_1410_0763_b200 as rt
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    l2 = torch.cuda.get_device_properties(0).L2_cache_size
    out = {"probe": "rt_probe_bandwidth: 8 CTAs/SM x 512 threads, float4 ld.cg / st.cg, best of 10", "l2_bytes": l2, "unit": "GB/s"}
    for label, nbytes in (("l2_24MB", 24 << 20), ("l2_48MB", 48 << 20), ("l2_96MB", 96 << 20), ("hbm_2GB", 2 << 30)):
        out[label] = {"read": rt.rt_probe_bandwidth(nbytes, 0, 10), "rmw": rt.rt_probe_bandwidth(nbytes, 1, 10)}
    print(json.dumps(out))


def workload_name(spec):
    return "%s: %dx%dx%d mesh, Nside=%d (%d directions), %d bin(s), seed %d" % (
        spec.name, spec.dims[0], spec.dims[1], spec.dims[2], spec.nside, spec.ndirs, spec.nbins, spec.seed)


def sweep_entries(rec):
    """Work entries of one owned sweep: a direction and its mirror image along the memory-contiguous transverse axis
    (same dominant axis, march sense, |slopes|) are carried by one warp and share every accumulator read-modify-write;
    directions without a partner (zero slope along that axis) run alone.  From rt_direction_records (host data)."""
    from collections import Counter
    pos, neg, n = Counter(), Counter(), len(rec)
    for a, refl, Mb, Mc, _, _ in rec:
        if Mb == 0:
            continue
        b, c = (1 if a == 0 else 0), (1 if a == 2 else 2)
        key = (int(a), (int(refl) >> int(a)) & 1, (int(refl) >> c) & 1, int(Mb), int(Mc))
        (neg if (int(refl) >> b) & 1 else pos)[key] += 1
    pairs = sum(min(v, neg.get(k, 0)) for k, v in pos.items())
    return pairs + (n - 2 * pairs)


class Runner:
    """One config on this rank's GPU: device-resident timing, end-to-end timing, roofline figures."""

    def __init__(self, name, args, rt, torch, dist, world, rank):
        from rt_inputs import make_fields, CONFIGS
        self.name, self.args, self.rt, self.torch, self.dist, self.world, self.rank = name, args, rt, torch, dist, world, rank
        self.spec = spec = CONFIGS[name]
        self.kap, self.S = make_fields(name)
        dirs = rt.healpix_dirs(spec.nside)
        self.sharded = world > 1 and args.shard == "directions"
        self.ndirs_total = dirs.shape[0]
        if self.sharded:
            dirs = dirs[rt.shard_directions(dirs, world, rank)]
        self.dirs = dirs
        self.tr = rt.RayTracer(spec.dims, spec.nbins, dirs, flags=args.flags, slots=args.slots, rows=args.rows, stages=args.stages,
                               pair=args.pair, tune=dict((kv.split('=')[0], int(kv.split('=')[1])) for kv in args.tune))
        self.stream = torch.cuda.current_stream()
        self.kap_h = torch.from_numpy(self.kap).pin_memory()
        self.S_h = torch.from_numpy(self.S).pin_memory()
        self.kd = self.kap_h.cuda(non_blocking=True)
        self.sd = self.S_h.cuda(non_blocking=True)
        self.J = torch.empty(self.tr.shape(), dtype=torch.float32, device="cuda")
        self.J_h = torch.empty(self.tr.shape(), dtype=torch.float32).pin_memory()
        self.tr.set_fields(self.kd, self.sd)
        self.updates = self.tr.total_segments() * spec.nbins          # exact integer traversal count x bins
        self.cell_dir_bins = spec.ncell * dirs.shape[0] * spec.nbins
        self.entries = sweep_entries(self.tr.direction_records()[0]) if (args.flags == 0 and args.pair in (None, 1)) else dirs.shape[0]
        if self.sharded:                                               # whole-job updates: sum over the shares
            t = torch.tensor([self.updates], device="cuda", dtype=torch.int64)
            dist.all_reduce(t)
            self.updates = int(t.item())
        self.l2_bytes = torch.cuda.get_device_properties(torch.cuda.current_device()).L2_cache_size
        self.working_set = self.tr.working_set_bytes()
        # timing rule: inputs larger than L2, else L2 flushed between timed steps (a write pass over 2 x L2)
        self.flush = self.working_set <= 2 * self.l2_bytes
        self.flush_buf = torch.empty(2 * self.l2_bytes // 4, dtype=torch.float32, device="cuda") if self.flush else None
        self.default_tuning = (args.flags == 0 and args.slots is None and args.rows is None and args.stages is None
                               and args.pair is None and not args.tune and not self.sharded)

    def step(self):
        if self.sharded:
            self.rt.sweep_sharded(self.tr, self.ndirs_total, what=self.rt.RT_J_IN, out=self.J)
        else:
            self.tr.sweep(out=self.J)

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, ms):
        if self.dist is not None:
            t = self.torch.tensor([ms], device="cuda", dtype=self.torch.float64)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    def timed(self, fn, steps):
        """Device time of `steps` calls of fn on the current stream (CUDA events), in ms, flushing L2 between the
        calls when the working set would otherwise stay resident (the flush is outside the timed intervals)."""
        torch = self.torch
        if not self.flush:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            for _ in range(steps):
                fn()
            e1.record(self.stream)
            self.barrier()
            return e0.elapsed_time(e1)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            self.flush_buf.zero_()
            a.record(self.stream)
            fn()
            b.record(self.stream)
        self.barrier()
        return sum(a.elapsed_time(b) for a, b in ev)

    def run(self, steps, warmup, sample_clocks):
        torch, tr = self.torch, self.tr
        for _ in range(max(warmup, 3)):
            self.step()
        self.barrier()
        sampler = ClockSampler(torch.cuda.current_device()) if (sample_clocks and self.rank == 0) else None
        if sampler:
            sampler.start()
        self.barrier()
        ms = self.timed(self.step, steps)
        clocks = sampler.stop() if sampler else None
        kernel_ms = tr.last_sweep_kernel_ms()          # traversal launches of the last timed sweep (library-side CUDA events)
        launches = tr.last_launch_count()
        graph = tr.last_sweep_was_graph()              # one CUDA-graph replay: kernel_ms then spans the normalisation kernel too
        ms = self.max_over_ranks(ms)
        jobs = 1 if self.sharded else self.world       # replicas: every rank sweeps the whole set
        value = jobs * self.updates * steps / (ms * 1e-3)

        # ---- end to end through the C ABI with HOST buffers: H2D of kappa,S + repack + sweep + D2H of J per step
        self.barrier()
        ph = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(steps)]

        def e2e_step(i=[0]):
            p = ph[i[0]]
            i[0] += 1
            p[0].record(self.stream)
            self.kd.copy_(self.kap_h, non_blocking=True)
            self.sd.copy_(self.S_h, non_blocking=True)
            p[1].record(self.stream)
            tr.set_fields(self.kd, self.sd)
            p[2].record(self.stream)
            self.step()
            p[3].record(self.stream)
            self.J_h.copy_(self.J, non_blocking=True)
            p[4].record(self.stream)
        ms_e2e = self.max_over_ranks(self.timed(e2e_step, steps))
        phase = [sum(p[k].elapsed_time(p[k + 1]) for p in ph) / steps for k in range(4)]
        e2e = {"value": jobs * self.updates * steps / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e / steps,
               "h2d_bytes_per_step": int(self.kap_h.numel() * 4 + self.S_h.numel() * 4), "d2h_bytes_per_step": int(self.J_h.numel() * 4),
               "h2d_ms": phase[0], "pack_ms": phase[1], "sweep_ms": phase[2], "d2h_ms": phase[3],
               "kernel_ms": tr.last_sweep_kernel_ms()}

        # ---- roofline of the dominant kernel (k_sweep_tma): SURVEY.md 8(d)'s 16 B per cell-direction-bin
        n_sweep_launches = max(1, launches - 1)                             # minus the normalise kernel
        # (a graph replay is timed as a whole: the normalisation kernel's time is then charged to the traversal launches,
        # which under-states `achieved`; roofline.timed_interval says which interval it was)
        avg_launch_ms = kernel_ms / n_sweep_launches
        bytes_per_launch = ALGO_BYTES_PER_CELL_DIR_BIN * self.cell_dir_bins / n_sweep_launches
        achieved = bytes_per_launch / (avg_launch_ms * 1e-3) / 1e9
        return {"ms": ms, "steps": steps, "value": value, "e2e": e2e, "clocks": clocks, "launches": launches,
                "floor_bytes": 8.0 * self.spec.ncell * self.spec.nbins * self.entries, "entries": self.entries,
                "kernel_ms": kernel_ms, "graph_replay": graph, "n_sweep_launches": n_sweep_launches, "avg_launch_ms": avg_launch_ms,
                "bytes_per_launch": bytes_per_launch, "achieved": achieved}

    def close(self):
        self.tr.close()
        self.flush_buf = None
        self.kd = self.sd = self.J = None
        self.torch.cuda.empty_cache()


def roofline_of(r, name, run, peaks, default_tuning):
    """`roofline` object of one config: algorithmic-byte model against the level that holds the fields, plus the
    ncu-measured DRAM traffic of the same launches when the committed table still matches the kernel sources."""
    bound = BOUND.get(name, "hbm")
    hbm_peak, hbm_kind = peaks["hbm"]
    peak, kind = (hbm_peak, hbm_kind) if bound == "hbm" else (peaks["l2_read"], "measured in this run (rt_probe_bandwidth, 48 MB read)")
    out = {"bound": bound, "achieved": run["achieved"], "peak": peak, "unit": "GB/s", "frac": run["achieved"] / peak,
           "traffic": None, "peak_kind": kind, "kernel": "k_sweep_tma",
           # the 16-byte model is SURVEY.md 8(d)'s figure, not a bound on this schedule (see note): the fraction that is
           # held against a ceiling is dram_frac_from_traffic (measured DRAM bytes over the HBM copy peak)
           "frac_is_ceiling": False,
           "model": "16 B per cell-direction-bin (read kappa,S 8 B + accumulator read-modify-write 8 B) x cell-direction-bins per launch",
           "launches_per_step": run["n_sweep_launches"], "avg_launch_ms": run["avg_launch_ms"],
           "algorithmic_bytes_per_launch": run["bytes_per_launch"],
           "kernel_share_of_step": run["kernel_ms"] / (run["ms"] / run["steps"]),
           "timed_interval": "whole sweep replayed as one CUDA graph (traversal + normalisation kernels)" if run.get("graph_replay")
                             else "traversal launches only (library-side CUDA events around them)",
           "frac_of_hbm_peak": run["achieved"] / hbm_peak,
           "note": "a mirror pair of directions shares every field load and accumulator read-modify-write, and the entries "
                   "of a launch find the fields in L2, so the 16-byte model is no upper bound on this schedule and frac "
                   "may exceed 1 (SURVEY.md 8(d)); dram_frac_from_traffic is the fraction of the HBM peak the kernel really draws"}
    # what THIS schedule must move through HBM at the least: one 4-byte read + one 4-byte write of a private slot
    # accumulator per cell, bin and work entry (a mirror pair of directions is one entry); <= 1 by construction
    floor_gbs = run["floor_bytes"] / (run["kernel_ms"] * 1e-3) / 1e9
    out["schedule_floor"] = {"what": "accumulator read-modify-write, 8 B per cell, bin and work entry", "entries": run["entries"],
                             "bytes_per_step": run["floor_bytes"], "gbs": floor_gbs, "frac_of_hbm_peak": floor_gbs / hbm_peak}
    if bound == "l2" and r.working_set > r.l2_bytes:
        # the packed fields stay in L2, the slot accumulators do not: a mixed bound, so the model against the L2 peak is
        # an upper estimate of nothing; the two measured fractions below are what each level really carries
        out["bound_detail"] = ("mixed: packed fields L2-resident, working set %.0f MB (fields + slot accumulators) streams through "
                               "HBM (L2 %.0f MB); read dram_frac_from_traffic and l2_frac_from_traffic, not frac") % (
                                   r.working_set / 1e6, r.l2_bytes / 1e6)
    table, state = traffic_table()
    out["traffic_table"] = state
    if default_tuning and name in table:
        per = float(table[name]["bytes_per_cell_dir_bin"])
        traffic = per * r.cell_dir_bins / run["n_sweep_launches"]
        out["traffic"] = traffic
        out["traffic_source"] = table[name].get("source")
        out["dram_gbs_from_traffic"] = traffic / (run["avg_launch_ms"] * 1e-3) / 1e9
        out["dram_frac_from_traffic"] = out["dram_gbs_from_traffic"] / hbm_peak
        if "l2_sm_bytes_per_cell_dir_bin" in table[name]:
            # bytes the SMs request from L2 in the same launches, against what the streaming probe reaches for this
            # read / write mix: 1 / ((1 - w) / read + w / write), with write from the read-modify-write probe
            # (2 / rmw = 1 / read + 1 / write)
            w = float(table[name].get("l2_sm_write_share", 0.25))
            l2t = float(table[name]["l2_sm_bytes_per_cell_dir_bin"]) * r.cell_dir_bins / run["n_sweep_launches"]
            rd, rmw = peaks["l2_read"], peaks["l2_rmw"]
            wr = 1.0 / max(2.0 / rmw - 1.0 / rd, 1e-9)
            ceiling = 1.0 / ((1.0 - w) / rd + w / wr)
            out["l2_gbs_from_traffic"] = l2t / (run["avg_launch_ms"] * 1e-3) / 1e9
            out["l2_mix_ceiling_gbs"] = ceiling
            out["l2_frac_from_traffic"] = out["l2_gbs_from_traffic"] / ceiling
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-dirs", type=int, default=0, help="directions per step of the reference arm (0: by --steps)")
    ap.add_argument("--cpu-dirs", type=int, default=96, help="directions of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="time --config only (skip the other four configs)")
    ap.add_argument("--slots", type=int, default=None)
    ap.add_argument("--rows", type=int, default=None)
    ap.add_argument("--stages", type=int, default=None)
    ap.add_argument("--pair", type=int, default=None, help="0: switch the mirror-pair schedule off (ablation)")
    ap.add_argument("--tune", action="append", default=[], help="key=value passed to rt_tune (experiments)")
    ap.add_argument("--flags", type=int, default=0, help="0 owned, 1 atomic ablation, 2 paper's four groups")
    ap.add_argument("--workload", default="diffuse", choices=["diffuse", "point"],
                    help="diffuse: the ray sweep (BASELINE.json's metric, default); point: rt_point_sources, the paper's "
                         "second workload (PAPER.md:64-82), SURVEY.md 8(f).4")
    ap.add_argument("--sources", type=int, default=8, help="--workload point: number of seeded point sources")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "directions"],
                    help="N > 1: independent replicas (default; north_star fixes one GPU) or the paper's direction "
                         "sharding with one all-reduce (PAPER.md:228-230)")
    ap.add_argument("--probe", action="store_true", help="print the L2 / HBM streaming-probe bandwidths and exit")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.probe:
        return run_probe(args)
    if args.workload == "point":
        return run_point(args)

    import torch
    import paper_1410_0763_b200 as rt
    from rt_inputs import CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        # leave NCCL's communicator lines in the log (ranks, transports) so that a scaling run can be checked
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---------------- headline config ----------------
    r = Runner(args.config, args, rt, torch, dist, world, rank)
    head = r.run(args.steps, args.warmup, sample_clocks=True)
    spec = r.spec
    kap, S = r.kap, r.S
    sharded, default_tuning = r.sharded, r.default_tuning
    working_set, l2_bytes, flushed = r.working_set, r.l2_bytes, r.flush
    cell_dir_bins = r.cell_dir_bins

    peaks = {"hbm": measured_peaks()}
    if rank == 0:
        peaks["l2_read"] = rt.rt_probe_bandwidth(48 << 20, 0, 10)
        peaks["l2_rmw"] = rt.rt_probe_bandwidth(48 << 20, 1, 10)
    roofline = roofline_of(r, args.config, head, peaks, default_tuning) if rank == 0 else None
    r.close()

    # ---------------- the other configs (device-resident + end to end, 3 steps each) ----------------
    configs = {}
    if not args.no_all_configs and world == 1 and default_tuning:
        for name in ("C1", "C2", "C3", "C4", "C5"):
            if name == args.config:
                run, rr = head, None
                ws, fl, cdb, upd, sp = working_set, flushed, cell_dir_bins, r.updates, spec
            else:
                rr = Runner(name, args, rt, torch, dist, world, rank)
                run = rr.run({"C1": 20, "C2": 10, "C3": 5}.get(name, 3), 3, sample_clocks=False)   # short sweeps: more of them
                ws, fl, cdb, upd, sp = rr.working_set, rr.flush, rr.cell_dir_bins, rr.updates, rr.spec
            rf = roofline_of(rr or r, name, run, peaks, True)
            configs[name] = {
                "workload": workload_name(sp), "ms_per_step": run["ms"] / run["steps"], "steps": run["steps"], "value": run["value"],
                "unit": UNIT, "updates_per_step": upd, "gpu_launches_per_step": run["launches"],
                "e2e": {k: run["e2e"][k] for k in ("value", "ms_per_step", "h2d_ms", "pack_ms", "sweep_ms", "d2h_ms")},
                "bound": rf["bound"], "bound_detail": rf.get("bound_detail"), "peak": rf["peak"], "model_frac": rf["frac"], "model_frac_of_hbm_peak": rf["frac_of_hbm_peak"],
                "dram_frac_from_traffic": rf.get("dram_frac_from_traffic"), "l2_frac_from_traffic": rf.get("l2_frac_from_traffic"),
                "schedule_floor_frac": rf["schedule_floor"]["frac_of_hbm_peak"],
                "kernel_share_of_step": rf["kernel_share_of_step"],
                # what a step spends outside the traversal launches: seam-accumulator clears + the normalisation kernel
                # (not separable when the sweep is one graph replay)
                "clear_and_normalise_ms": None if run.get("graph_replay") else max(0.0, run["ms"] / run["steps"] - run["kernel_ms"]),
                "graph_replay": bool(run.get("graph_replay")),
                "working_set_bytes": ws, "l2": "L2 flushed between timed steps" if fl else "working set larger than L2",
            }
            if rr is not None:
                rr.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------- CPU baseline: the oracle, as it stands, on a bounded sample ----------------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import oracle
        cores = host_cores()
        dirs_all = oracle.healpix_dirs(spec.nside)
        val, dt, nd, stride = oracle_rate(oracle, kap, S, dirs_all, max(1, min(spec.ndirs, args.cpu_dirs)), cores, spec.nbins)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
               "sample": "%d of %d directions (every %dth), full mesh, %.1f s" % (nd, spec.ndirs, stride, dt)}
        n1 = max(1, min(spec.ndirs, args.cpu_dirs // 12))
        v1, dt1, nd1, st1 = oracle_rate(oracle, kap, S, dirs_all, n1, 1, spec.nbins)
        cpu["single_thread"] = {"value": v1, "unit": UNIT, "cores": 1,
                                "sample": "%d of %d directions (every %dth), full mesh, %.1f s" % (nd1, spec.ndirs, st1, dt1)}

    l2_note = ("L2 flushed between timed steps (working set %.0f MB, L2 %.0f MB)" if flushed else
               "working set (packed fields + slot accumulators, %.0f MB) larger than L2 (%.0f MB)") % (working_set / 1e6, l2_bytes / 1e6)
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": head["ms"] / args.steps, "higher_is_better": True,
        "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(spec), "updates_per_step": r.updates,
                   "parallelism": ("directions sharded, 1 all-reduce" if sharded else "replicas only") if world > 1 else "1 gpu",
                   "l2": l2_note, "variant": ["owned", "atomic_ablation", "paper_groups"][args.flags]},
        "clocks": head["clocks"], "gpu_launches": head["launches"] * args.steps,
        "e2e": head["e2e"], "roofline": roofline, "cpu_baseline": cpu,
        "peaks": {"hbm_gbs": peaks["hbm"][0], "hbm_kind": peaks["hbm"][1], "l2_read_gbs": peaks.get("l2_read"),
                  "l2_rmw_gbs": peaks.get("l2_rmw"), "l2_probe": "rt_probe_bandwidth over 48 MB, best of 10", "l2_bytes": l2_bytes},
    }
    if configs:
        line["configs"] = configs
        # the paper's second workload (RT from point sources) on the same mesh, outside the timed region
        # of the headline: its own metric, time and issue-slot roofline (bench.py --workload point prints the same record)
        p = point_line(args, cpu=False)
        line["point"] = {k: p[k] for k in ("metric", "value", "unit", "ms_per_step", "config", "roofline", "note")}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
