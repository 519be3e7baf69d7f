#!/usr/bin/env python
"""Benchmark of the diffuse-radiation ray sweep (BASELINE.json metric: ray-segment updates/sec on
one B200 and % of the HBM roofline; oracle host time beside it).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A step = one rt_sweep over all directions ("one iteration") of the synthetic workload.
Prints ONE JSON line (rank 0).  For N > 1 (torchrun) every rank sweeps a full replica ("replicas
only": the path does not shard in this build).
"""
from __future__ import annotations

import argparse
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
# dram__bytes_read.sum + dram__bytes_write.sum per cell-direction-bin of the hot kernel, from the ncu --set full
# capture named beside it (profiles/); multiplied by the cell-direction-bins of one launch to give `traffic`.
NCU_DRAM_BYTES_PER_CELL_DIR_BIN = {"C4": (5.426, "profiles/r1e_sweep_tma_full_c4.md")}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


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


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores; each step is a bounded
    sample (a subset of directions) of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle
    from rt_inputs import make_fields, CONFIGS
    spec = CONFIGS[args.config]
    kap, S = make_fields(args.config)
    dirs = oracle.healpix_dirs(spec.nside)
    nd = max(1, min(spec.ndirs, args.ref_dirs))
    sub = dirs[:: max(1, spec.ndirs // nd)][:nd]
    cores = min(os.cpu_count() or 1, 32, len(sub))
    for _ in range(args.warmup if args.warmup < 1 else 1):
        oracle.sweep(kap, S, sub[:cores], nthreads=cores, want_counts=False)
    t0 = time.perf_counter()
    upd = 0
    for _ in range(args.steps):
        r = oracle.sweep(kap, S, sub, nthreads=cores, want_counts=False)
        upd += r["seg_total"] * spec.nbins
    dt = time.perf_counter() - t0
    val = upd / dt
    sample = "%d of %d directions per step (every %dth), full mesh" % (len(sub), spec.ndirs, max(1, spec.ndirs // nd))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(spec), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_point(args):
    """--workload point: rt_point_sources on the config's mesh and kappa with seeded sources (one at a box corner,
    one at the centre, the rest uniform in the box, positions in 1/256 cell).  One JSON line of its own."""
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
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import oracle
        ns = min(args.sources, 2)
        t0 = time.perf_counter()
        r = oracle.point_sources(kap, src[:ns], lum[:ns], want_diag=False)
        dt = time.perf_counter() - t0
        cpu = {"value": r["steps"] * spec.nbins / dt, "unit": "ray steps/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "%d of %d sources, full mesh, %.1f s" % (ns, args.sources, dt)}
    print(json.dumps({
        "metric": "point_source_ray_steps_per_sec", "value": steps * spec.nbins / (ms * 1e-3), "unit": "ray steps/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 path sums over f32 kappa", "data": "synthetic",
        "config": {"workload": "point sources on " + workload_name(spec), "sources": args.sources,
                   "ray_steps_per_step": steps * spec.nbins, "rays_per_step": args.sources * spec.ncell * spec.nbins},
        "clocks": clocks, "gpu_launches": args.steps,
        "roofline": None, "note": "gather along long characteristics: latency / integer-ALU bound, no roofline claimed",
        "cpu_baseline": cpu}))


def workload_name(spec):
    return "%s: %dx%dx%d mesh, Nside=%d (%d directions), %d bin(s), seed %d" % (
        spec.name, spec.dims[0], spec.dims[1], spec.dims[2], spec.nside, spec.ndirs, spec.nbins, spec.seed)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-dirs", type=int, default=8, help="directions per step of the reference arm")
    ap.add_argument("--cpu-dirs", type=int, default=96, help="directions of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "point":
        return run_point(args)

    import torch
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields, CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    spec = CONFIGS[args.config]
    kap, S = make_fields(args.config)
    dirs = rt.healpix_dirs(spec.nside)
    sharded = world > 1 and args.shard == "directions"
    ndirs_total = dirs.shape[0]
    if sharded:
        dirs = dirs[rt.shard_directions(dirs, world, rank)]
    tr = rt.RayTracer(spec.dims, spec.nbins, dirs, flags=args.flags, slots=args.slots, rows=args.rows, stages=args.stages, pair=args.pair,
                      tune=dict((kv.split('=')[0], int(kv.split('=')[1])) for kv in args.tune))
    stream = torch.cuda.current_stream()
    kap_h = torch.from_numpy(kap).pin_memory()
    S_h = torch.from_numpy(S).pin_memory()
    kd = kap_h.cuda(non_blocking=True)
    sd = S_h.cuda(non_blocking=True)
    J = torch.empty(tr.shape(), dtype=torch.float32, device="cuda")
    J_h = torch.empty(tr.shape(), dtype=torch.float32).pin_memory()
    tr.set_fields(kd, sd)
    updates_per_sweep = tr.total_segments() * spec.nbins        # exact integer traversal count x bins
    cell_dir_bins = spec.ncell * dirs.shape[0] * spec.nbins
    if sharded:                                                  # whole-job updates: sum over the shares
        t = torch.tensor([updates_per_sweep], device="cuda", dtype=torch.int64)
        dist.all_reduce(t)
        updates_per_sweep = int(t.item())

    def step():
        if sharded:
            rt.sweep_sharded(tr, ndirs_total, what=rt.RT_J_IN, out=J)
        else:
            tr.sweep(out=J)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing (value) ----------------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms = []
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    # traversal-kernel time of the last timed sweep (cudaEvents on the launching stream, inside the library)
    kernel_ms.append(tr.last_sweep_kernel_ms())
    launches_per_sweep = tr.last_launch_count()
    if dist is not None:
        t = torch.tensor([ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    jobs = 1 if sharded else world                               # replicas: every rank sweeps the whole set
    value = jobs * updates_per_sweep * args.steps / (ms * 1e-3)

    # ---------------- end-to-end through the C ABI with host buffers ----------------
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(args.steps):
        kd.copy_(kap_h, non_blocking=True)
        sd.copy_(S_h, non_blocking=True)
        tr.set_fields(kd, sd)
        step()
        J_h.copy_(J, non_blocking=True)
    f1.record(stream)
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    if dist is not None:
        t = torch.tensor([ms_e2e], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_e2e = float(t.item())
    e2e_value = jobs * updates_per_sweep * args.steps / (ms_e2e * 1e-3)
    tr.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------- roofline of the dominant kernel (k_sweep_owned) ----------------
    peak, peak_kind = measured_peaks()
    n_sweep_launches = max(1, launches_per_sweep - 1)                   # minus the normalise kernel
    avg_launch_ms = kernel_ms[0] / n_sweep_launches
    bytes_per_launch = ALGO_BYTES_PER_CELL_DIR_BIN * cell_dir_bins / n_sweep_launches
    achieved = bytes_per_launch / (avg_launch_ms * 1e-3) / 1e9
    traffic, traffic_src = None, None
    if args.config in NCU_DRAM_BYTES_PER_CELL_DIR_BIN and args.flags == 0:
        per, traffic_src = NCU_DRAM_BYTES_PER_CELL_DIR_BIN[args.config]
        traffic = per * cell_dir_bins / n_sweep_launches
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src, "peak_kind": peak_kind, "kernel": "k_sweep_tma",
                # the same launches against the DRAM bytes ncu measured (mirror pairs share loads, so the
                # algorithmic-byte fraction above exceeds 1; this one is the bandwidth the kernel really draws)
                "dram_gbs_from_traffic": (traffic / (avg_launch_ms * 1e-3) / 1e9) if traffic else None,
                "dram_frac_from_traffic": (traffic / (avg_launch_ms * 1e-3) / 1e9 / peak) if traffic else None,
                "launches_per_step": n_sweep_launches, "avg_launch_ms": avg_launch_ms,
                "algorithmic_bytes_per_launch": bytes_per_launch,
                "kernel_share_of_step": kernel_ms[0] / (ms / args.steps)}

    # ---------------- CPU baseline: the oracle on a bounded sample ----------------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import oracle
        nd = max(1, min(spec.ndirs, args.cpu_dirs))
        stride = max(1, spec.ndirs // nd)
        sub = oracle.healpix_dirs(spec.nside)[::stride][:nd]
        cores = min(os.cpu_count() or 1, 32, len(sub))
        t0 = time.perf_counter()
        r = oracle.sweep(kap, S, sub, nthreads=cores, want_counts=False)
        dt = time.perf_counter() - t0
        cpu = {"value": r["seg_total"] * spec.nbins / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%d of %d directions (every %dth), full mesh, %.1f s" % (len(sub), spec.ndirs, stride, dt)}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(spec), "updates_per_step": updates_per_sweep,
                   "parallelism": ("directions sharded, 1 all-reduce" if sharded else "replicas only") if world > 1 else "1 gpu",
                   "l2": "working set (packed fields + slot accumulators) larger than L2",
                   "variant": ["owned", "atomic_ablation", "paper_groups"][args.flags]},
        "clocks": clocks, "gpu_launches": launches_per_sweep * args.steps,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                "h2d_bytes_per_step": int(kap_h.numel() * 4 + S_h.numel() * 4), "d2h_bytes_per_step": int(J_h.numel() * 4)},
        "roofline": roofline, "cpu_baseline": cpu,
    }))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
