"""bench.py's reference arm runs on the host (the oracle on a bounded sample) and prints one JSON line with
the contract's keys; the GPU arm refuses to run without a CUDA device (no CPU fallback)."""
import json

import numpy as np
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                          "--steps", "1", "--warmup", "0", "--ref-dirs", "4"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["metric"] == "ray_segment_updates_per_sec" and d["unit"] == "updates/s"
    assert d["higher_is_better"] is True and d["value"] > 0 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert "workload" in d["config"]


def test_gpu_arm_fails_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a GPU is present")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--config", "C1"],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


def _run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


import pytest  # noqa: E402


@pytest.mark.gpu
def test_gpu_arm_prints_the_contract_line():
    """The line the driver parses: metric, whole-job value, e2e with host copies, roofline, cpu_baseline, clocks,
    launch count (small config so that it runs in seconds)."""
    d = _run_bench("--config", "C2", "--steps", "3", "--warmup", "3", "--cpu-dirs", "24", "--no-all-configs")
    assert d["metric"] == "ray_segment_updates_per_sec" and d["unit"] == "updates/s" and d["n_gpus"] == 1
    assert d["steps"] == 3 and d["warmup"] >= 3 and d["higher_is_better"] is True and d["dtype"] == "f32"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert d["gpu_launches"] > 0 and "workload" in d["config"] and "configs" not in d
    assert "flushed" in d["config"]["l2"] or "larger than L2" in d["config"]["l2"]      # the bench says how it timed it
    e = d["e2e"]
    assert 0 < e["value"] <= d["value"] * 1.05 and e["h2d_bytes_per_step"] == 2 * 4 * 64 ** 3 and e["d2h_bytes_per_step"] == 4 * 64 ** 3
    assert e["h2d_ms"] > 0 and e["pack_ms"] > 0 and e["sweep_ms"] > 0 and e["d2h_ms"] > 0 and e["kernel_ms"] > 0
    assert abs(e["h2d_ms"] + e["pack_ms"] + e["sweep_ms"] + e["d2h_ms"] - e["ms_per_step"]) < 0.05 * e["ms_per_step"]
    r = d["roofline"]
    assert r["bound"] == "l2" and r["unit"] == "GB/s" and r["peak"] > 5000 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert 0.5 < r["kernel_share_of_step"] < 1.2
    assert d["peaks"]["l2_read_gbs"] > d["peaks"]["hbm_gbs"] > 1000
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    assert c["single_thread"]["cores"] == 1 and c["single_thread"]["value"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


@pytest.mark.gpu
def test_default_line_carries_all_five_configs():
    """The driver's own command (default config C4) with fewer steps: one JSON line with the headline on C4 and a
    `configs` record for C1 ... C5 (report for every config)."""
    d = _run_bench("--steps", "3", "--warmup", "3", "--cpu-dirs", "16")
    assert d["config"]["workload"].startswith("C4") and d["roofline"]["bound"] == "hbm" and "larger than L2" in d["config"]["l2"]
    assert sorted(d["configs"]) == ["C1", "C2", "C3", "C4", "C5"]
    for name, c in d["configs"].items():
        assert c["value"] > 0 and c["ms_per_step"] > 0 and c["e2e"]["value"] > 0 and c["model_frac"] > 0
        assert c["bound"] == ("hbm" if name in ("C4", "C5") else "l2")
    assert d["configs"]["C4"]["ms_per_step"] == d["ms_per_step"]
    assert d["roofline"]["frac_is_ceiling"] is False and d["configs"]["C1"]["graph_replay"] is True
    assert d["configs"]["C3"]["bound_detail"].startswith("mixed") and d["configs"]["C4"]["bound_detail"] is None
    p = d["point"]                                                     # the second workload rides on the default line
    assert p["metric"] == "point_source_ray_steps_per_sec" and p["value"] > 0 and p["ms_per_step"] > 0 and p["config"]["sources"] == 8
    t = d["roofline"]
    assert t["traffic_table"] == "ok" or t["traffic"] is None        # never a stale ncu figure


def test_traffic_table_names_the_kernel_sources():
    """profiles/dram_traffic.json ties the ncu-measured DRAM bytes to the git blob hashes of the kernel sources;
    bench.py drops `traffic` when a source has changed since the capture."""
    sys.path.insert(0, ROOT)
    import bench
    t = json.load(open(bench.TRAFFIC_TABLE))
    assert set(t["kernel_sources"]) == set(bench.KERNEL_SOURCES)
    for name, e in t["entries"].items():
        assert name in ("C1", "C2", "C3", "C4", "C5") and e["bytes_per_cell_dir_bin"] > 0 and os.path.exists(os.path.join(ROOT, e["source"]))
    entries, state = bench.traffic_table()
    assert state == "ok" or (state.startswith("stale") and entries == {})


@pytest.mark.gpu
def test_point_workload_line():
    d = _run_bench("--workload", "point", "--config", "C2", "--steps", "2", "--sources", "3")
    assert d["metric"] == "point_source_ray_steps_per_sec" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"


def test_point_source_instruction_count_names_its_kernel_source():
    """profiles/point_sources.json ties the ncu-measured thread-instructions per ray step to the git blob hash of the
    kernel source; bench.py --workload point drops its issue-slot roofline when the source has changed."""
    t = json.load(open(os.path.join(ROOT, "profiles", "point_sources.json")))
    assert os.path.exists(os.path.join(ROOT, t["kernel_source"])) and os.path.exists(os.path.join(ROOT, t["source"]))
    assert len(t["kernel_source_sha"]) == 40 and 10 < t["thread_instructions_per_ray_step"] < 200


def test_sweep_entries_counts_mirror_pairs():
    """bench.sweep_entries (host logic of the schedule floor): a direction and its mirror image along the
    memory-contiguous transverse axis are one work entry; directions with a zero slope along that axis run alone."""
    sys.path.insert(0, ROOT)
    import bench
    # records: (dominant axis a, reflection bits x|y<<1|z<<2, Mb, Mc, generic flag, rays); b = y for a = 0, else x
    rec = np.array([
        [2, 0b000, 100, 50, 0, 1], [2, 0b001, 100, 50, 0, 1],      # z-dominant, mirrored in x: one pair
        [2, 0b100, 100, 50, 0, 1],                                  # other march sense: no partner
        [2, 0b000, 0, 70, 0, 1], [2, 0b001, 0, 70, 0, 1],           # zero slope along b: two singles
        [0, 0b000, 30, 20, 0, 1], [0, 0b010, 30, 20, 0, 1],         # x-dominant, mirrored in y: one pair
        [1, 0b000, 30, 20, 0, 1], [1, 0b100, 30, 20, 0, 1],         # y-dominant, c = z reflected: different rows, no pair
    ], dtype=np.int64)
    assert bench.sweep_entries(rec) == 1 + 1 + 2 + 1 + 2
    from oracle import oracle
    oracle.build()
    dirs = oracle.healpix_dirs(16)
    # HEALPix: every direction with a non-zero b-slope has its mirror image in the set (128 of 3072 have none)
    recs = np.array([[int(np.argmax(np.abs(d))), (d[0] < 0) | ((d[1] < 0) << 1) | ((d[2] < 0) << 2), 0, 0, 0, 1] for d in dirs], dtype=np.int64)
    for i, d in enumerate(dirs):
        a = recs[i, 0]
        b, c = (1 if a == 0 else 0), (1 if a == 2 else 2)
        recs[i, 2] = round(abs(d[b] / d[a]) * 2 ** 20)
        recs[i, 3] = round(abs(d[c] / d[a]) * 2 ** 20)
    assert bench.sweep_entries(recs) == 1594
