"""Parity gates at BASELINE.json's full sizes (SURVEY.md 8(d) "Parity gates per config", the
paper's own mesh sizes), in the launch configuration bench.py times.  All tests need a GPU; the oracle side runs
on the box's host cores (full C3 sweep ~ 30 s on 16 threads; sampled cells of C4 / C5 ~ 1-2 min each).

  C3 (128^3 x 3072):  EVERY cell: J_in and J within tolerance, direction-summed counts identical, per-direction
                      count arrays for 16 sampled directions, total segments == oracle == tests/golden, sum ds of
                      all 3072 directions vs the oracle and vs N_m L; two further seeds of the recipe (J only).
  C4 (256^3 x 3072):  EVERY cell once: J_in against the whole oracle sweep (4-8 min of host time on 16 threads).
  C4, C5:             >= 4096 (C5: >= 16384) sampled cells through orc_sweep_cells (random + three full axis lines
                      through the most opaque cell + the eight corners), counts at those cells, total segments == the
                      oracle's exact totals in tests/golden/segment_totals.txt, SHA-256 of the per-cell counts summed
                      over the directions == the oracle's (same file: every cell, bit-exact), sum ds of a 128-direction
                      subset vs oracle.
  128^3 x 12288:      N_side = 32 on the C3 mesh, 1024 sampled cells (four times the directions in the fp32 sums).

Every test appends its maxima to gpurun_out/parity_report.txt (scratch) so that a run leaves the numbers behind.
"""
import hashlib
import json
import os
import time

import numpy as np
import pytest

from tests.test_gpu_parity import DS_TOL, J_TOL, _torch, rel_err, sample_dirs

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
# the accuracy margin bought in round 2: the full-size maxima must stay below half the tolerance
J_MARGIN = 0.5 * J_TOL


def golden_totals():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "segment_totals.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            out[k] = int(v)
    return out


def golden_count_hashes():
    """SHA-256 of the oracle's per-cell segment counts summed over the directions (uint32 little-endian, [nz][ny][nx]),
    written by tests/golden/make_segment_totals.py from oracle/ alone."""
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "segment_totals.txt")):
        w = line.split()
        if w and not line.startswith("#"):
            assert len(w) >= 5 and len(w[4]) == 64, "segment_totals.txt has no count hash for %s" % w[0]
            out[w[0]] = w[4]
    return out


def count_hash(cnt):
    return hashlib.sha256(np.ascontiguousarray(cnt, dtype="<u4").tobytes()).hexdigest()


def report(**kw):
    d = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_report.txt"), "a") as f:
            f.write(json.dumps(kw) + "\n")
    except OSError:
        pass


def sample_cells(dims, n, seed, kap):
    """n random cells + the eight corners + three full axis lines through the most opaque cell (bin 0) + the most
    transparent cell."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    cells = [np.stack([rng.integers(0, nx, n), rng.integers(0, ny, n), rng.integers(0, nz, n)], 1)]
    cells.append(np.array([[x, y, z] for x in (0, nx - 1) for y in (0, ny - 1) for z in (0, nz - 1)]))
    zm, ym, xm = np.unravel_index(np.argmax(kap[0]), kap[0].shape)
    cells.append(np.stack([np.arange(nx), np.full(nx, ym), np.full(nx, zm)], 1))
    cells.append(np.stack([np.full(ny, xm), np.arange(ny), np.full(ny, zm)], 1))
    cells.append(np.stack([np.full(nz, xm), np.full(nz, ym), np.arange(nz)], 1))
    zt, yt, xt = np.unravel_index(np.argmin(kap[0]), kap[0].shape)
    cells.append(np.array([[xt, yt, zt]]))
    return np.unique(np.concatenate(cells), axis=0).astype(np.int32)


def stats(e):
    return float(e.max()), float(np.quantile(e, 0.999)), float(np.median(e))


# ---------------------------------------------------------------------------------------------
def test_c3_every_cell(orc):
    """Config 3 in full: the whole oracle sweep against the whole GPU sweep."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS["C3"]
    kap, S = make_fields("C3")
    dirs = orc.healpix_dirs(spec.nside)
    cd = sample_dirs(orc, dirs, 16)
    tr = rt.RayTracer(spec.dims, 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        J = tr.sweep(what=rt.RT_J_TOTAL).cpu().numpy()
        cnt = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
        cnt_d = np.stack([tr.segment_counts(int(i)).cpu().numpy().astype(np.uint32) for i in cd])
        seg_total = tr.total_segments()
        sum_ds, mn, mx = tr.sum_ds()
        rec, L = tr.direction_records()
    finally:
        tr.close()
    t0 = time.time()
    ref = orc.sweep(kap, S, dirs, count_dirs=cd)
    dt = time.time() - t0
    # integer traversal data: bit-exact
    assert np.array_equal(cnt, ref["cnt_sum"])
    assert np.array_equal(cnt_d, ref["cnt_dirs"])
    assert seg_total == ref["seg_total"] == golden_totals()["C3"]
    assert count_hash(cnt) == count_hash(ref["cnt_sum"]) == golden_count_hashes()["C3"]
    # sum ds of every direction: vs the oracle and vs the closed form N_m L (pin P3)
    assert np.abs(sum_ds / ref["sum_ds"] - 1).max() <= DS_TOL
    assert np.abs(sum_ds / (spec.ncell * L) - 1).max() <= DS_TOL
    assert np.abs(mn / L - 1).max() <= 2e-6 and np.abs(mx / L - 1).max() <= 2e-6
    e_in, e_J = rel_err(Jin, ref["Jin"]), rel_err(J, ref["J"])
    m_in, m_J = stats(e_in), stats(e_J)
    report(test="c3_every_cell", seed=spec.seed, J_in_max=m_in[0], J_in_p999=m_in[1], J_in_median=m_in[2], J_max=m_J[0],
           cells=int(e_in.size), seg_total=seg_total, oracle_s=dt, oracle_threads=orc.num_threads(),
           oracle_updates_per_s=ref["seg_total"] / dt)
    assert m_in[0] <= J_MARGIN, "C3 J_in max rel err %.3e (p99.9 %.3e, median %.3e)" % m_in
    assert m_J[0] <= J_MARGIN, "C3 J max rel err %.3e (p99.9 %.3e, median %.3e)" % m_J


@pytest.mark.parametrize("seed", [11, 12])
def test_c3_further_seeds_every_cell(orc, seed):
    """Two further realisations of C3's recipe: the accuracy margin must not hang on one seed."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS["C3"]
    kap, S = make_fields("C3", seed=seed)
    dirs = orc.healpix_dirs(spec.nside)
    tr = rt.RayTracer(spec.dims, 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
    finally:
        tr.close()
    ref = orc.sweep(kap, S, dirs, want_counts=False)
    m = stats(rel_err(Jin, ref["Jin"]))
    report(test="c3_every_cell", seed=seed, J_in_max=m[0], J_in_p999=m[1], J_in_median=m[2])
    assert m[0] <= J_MARGIN, "C3 seed %d J_in max rel err %.3e (p99.9 %.3e, median %.3e)" % ((seed,) + m)


def test_c4_every_cell(orc):
    """Config 4 (the benchmark's headline workload) in full, once: J_in of the whole GPU sweep against the whole oracle
    sweep, every one of the 16.8 M cells (the sampled gate below cannot see an error in a cell it did not draw)."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS["C4"]
    kap, S = make_fields("C4")
    dirs = orc.healpix_dirs(spec.nside)
    tr = rt.RayTracer(spec.dims, 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        rec, _ = tr.direction_records()
    finally:
        tr.close()
    assert np.all(rec[:, 4] == 0)
    t0 = time.time()
    ref = orc.sweep(kap, S, dirs, want_counts=False)
    dt = time.time() - t0
    assert ref["seg_total"] == golden_totals()["C4"]
    e = rel_err(Jin, ref["Jin"])
    m = stats(e)
    report(test="c4_every_cell", cells=int(e.size), J_in_max=m[0], J_in_p999=m[1], J_in_median=m[2], oracle_s=dt,
           oracle_threads=orc.num_threads(), oracle_updates_per_s=ref["seg_total"] / dt)
    # The bar is north_star's tolerance.  The half-tolerance margin that the sampled gates keep (J_MARGIN) is held here by
    # the 99.9th percentile; the maximum over all 16.8 M cells, first measured in round 3, is 5.2e-6 (the 4871-cell
    # sample had shown 3.7e-6: a sample under-states the tail).
    assert m[0] <= J_TOL, "C4 J_in max rel err %.3e (p99.9 %.3e, median %.3e) over %d cells" % (m + (e.size,))
    assert m[1] <= J_MARGIN, "C4 J_in p99.9 rel err %.3e (max %.3e)" % (m[1], m[0])


@pytest.mark.parametrize("name", ["C4", "C5"])
def test_full_size_4096_cells(orc, name):
    """Configs 4 and 5 at full size: >= 4096 sampled cells computed by the oracle ray by ray, exact totals, sum ds."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS[name]
    kap, S = make_fields(name)
    nb = kap.shape[0]
    dirs = orc.healpix_dirs(spec.nside)
    nsample = 4096 if name == "C4" else 16384          # C4 is also compared on every cell (test_c4_every_cell)
    cells = sample_cells(spec.dims, nsample, 7, kap)
    assert len(cells) >= nsample
    sub = np.arange(0, spec.ndirs, 24)                 # 128 of the 3072 directions for the sum-of-ds gate
    tr = rt.RayTracer(spec.dims, nb, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN)
        J = tr.sweep(what=rt.RT_J_TOTAL)
        cnt = tr.segment_counts(-1)
        seg_total = tr.total_segments()
        rec, L = tr.direction_records()
        assert np.all(rec[:, 4] == 0)
        ix = torch.from_numpy(cells.astype(np.int64)).cuda()
        got_in = Jin[:, ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy()
        got_J = J[:, ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy()
        got_cnt = cnt[ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy().astype(np.uint32)
        assert bool(torch.isfinite(Jin).all()) and float(Jin.min()) >= 0.0
        cnt_total = int(cnt.to(torch.int64).sum().item())
        cnt_sha = count_hash(cnt.cpu().numpy())
    finally:
        tr.close()
    got_packed = None
    if nb % 3 == 0:                                    # C5: the multi-bin packed kernel (three bins per row) at full size
        tr = rt.RayTracer(spec.dims, nb, dirs, tune={"binpack": 1})
        try:
            tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
            Jp = tr.sweep(what=rt.RT_J_IN)
            got_packed = Jp[:, ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy()
            assert bool(torch.isfinite(Jp).all()) and float(Jp.min()) >= 0.0
            del Jp
        finally:
            tr.close()
    tr = rt.RayTracer(spec.dims, 1, dirs[sub])
    try:
        sum_ds, mn, mx = tr.sum_ds()
        _, Ls = tr.direction_records()
    finally:
        tr.close()
    # integer data: the oracle's exact totals (tests/golden/segment_totals.txt, written from oracle/ alone)
    assert seg_total == cnt_total == golden_totals()[name]
    # ... and on every cell: the hash of the whole direction-summed count array is the oracle's
    assert cnt_sha == golden_count_hashes()[name], "%s: per-cell segment counts differ from the oracle's somewhere in the mesh" % name
    t0 = time.time()
    ref = orc.sweep_cells(kap, S, dirs, cells)
    dt = time.time() - t0
    assert np.array_equal(got_cnt, ref["cnt"])
    # sum ds of the subset: vs the oracle (one bin, unit medium: ds does not depend on the fields) and vs N_m L
    nx, ny, nz = spec.dims
    ref_ds = orc.sweep(np.ones((1, nz, ny, nx), np.float32), np.zeros((1, nz, ny, nx), np.float32), dirs[sub],
                       want_counts=False)["sum_ds"]
    assert np.abs(sum_ds / ref_ds - 1).max() <= DS_TOL
    assert np.abs(sum_ds / (spec.ncell * Ls) - 1).max() <= DS_TOL
    assert np.abs(mn / Ls - 1).max() <= 2e-6 and np.abs(mx / Ls - 1).max() <= 2e-6
    m_in, m_J = stats(rel_err(got_in, ref["Jin"])), stats(rel_err(got_J, ref["J"]))
    report(test="full_size_4096_cells", config=name, cells=int(len(cells)), J_in_max=m_in[0], J_in_p999=m_in[1],
           J_in_median=m_in[2], J_max=m_J[0], seg_total=seg_total, oracle_cells_s=dt)
    assert m_in[0] <= J_MARGIN, "%s J_in max rel err %.3e (p99.9 %.3e, median %.3e)" % ((name,) + m_in)
    assert m_J[0] <= J_MARGIN, "%s J max rel err %.3e (p99.9 %.3e, median %.3e)" % ((name,) + m_J)
    if got_packed is not None:
        m_p = stats(rel_err(got_packed, ref["Jin"]))
        report(test="full_size_packed_bins", config=name, cells=int(len(cells)), J_in_max=m_p[0], J_in_p999=m_p[1], J_in_median=m_p[2])
        assert m_p[0] <= J_MARGIN, "%s binpack J_in max rel err %.3e (p99.9 %.3e, median %.3e)" % ((name,) + m_p)


def test_c3_mesh_nside32_sampled(orc):
    """128^3 with N_side = 32 (12288 directions): four times the terms in every fp32 sum of C3."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS["C3"]
    kap, S = make_fields("C3")
    dirs = orc.healpix_dirs(32)
    cells = sample_cells(spec.dims, 640, 9, kap)
    tr = rt.RayTracer(spec.dims, 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN)
        cnt = tr.segment_counts(-1)
        ix = torch.from_numpy(cells.astype(np.int64)).cuda()
        got_in = Jin[:, ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy()
        got_cnt = cnt[ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy().astype(np.uint32)
    finally:
        tr.close()
    ref = orc.sweep_cells(kap, S, dirs, cells)
    assert np.array_equal(got_cnt, ref["cnt"])
    m = stats(rel_err(got_in, ref["Jin"]))
    report(test="c3_mesh_nside32", cells=int(len(cells)), J_in_max=m[0], J_in_p999=m[1], J_in_median=m[2])
    assert m[0] <= J_MARGIN, "128^3 x 12288 J_in max rel err %.3e (p99.9 %.3e, median %.3e)" % m


# ---------------------------------------------------------------------------------------------
# the no-atomics claim: one writer per cell, accumulator array and launch (SURVEY.md 7 hard part 4)
@pytest.mark.parametrize("case", [
    dict(cfg="C2"),                                                  # the benchmark's own launch configuration
    dict(cfg="C3", dims=(128, 128, 64), nside=8),                    # 128-cell rows, four ray rows per warp
    dict(cfg="C4", dims=(256, 256, 16), nside=4),                    # 256-cell rows, two ray rows per warp
    dict(cfg="C4", dims=(200, 130, 24), nside=4),                    # padded rows (256-wide pitch both layouts)
    dict(cfg="C2", dims=(64, 32, 48), nside=4, rays=2),              # r = 2: four sub-lattices per direction
    dict(cfg="C3", dims=(128, 64, 40), nside=4, tune={"handoff": 1}, rows=2),   # seam handoff inside the CTA
    dict(cfg="C5", dims=(64, 32, 96), nside=4),                      # three bins
    dict(cfg="C2", dims=(64, 64, 30), nside=4, rows=1, slots=3),     # few slots: launches of whole entries
    dict(cfg="C1", pair=0),                                          # single directions, both march senses
    dict(cfg="C2", tune={"overlap": 0}),                             # one launch after the other (the schedule of large meshes)
    dict(cfg="C3", dims=(128, 128, 64), nside=8, tune={"overlap": 1, "wave_div": 3}),   # overlapped classes, third-wave launches
])
def test_one_writer_per_cell_and_launch(case):
    """rt_debug_writer_counts: the launches of rt_sweep with every accumulator store turned into an atomic increment.
    No element of a slot accumulator or seam accumulator may be stored to twice within a launch, and over a sweep
    every element of an entry's accumulator volume is stored to exactly once."""
    from rt_inputs import CONFIGS
    import paper_1410_0763_b200 as rt
    _torch()
    spec = CONFIGS[case["cfg"]]
    dims = case.get("dims", spec.dims)
    dirs = rt.healpix_dirs(case.get("nside", spec.nside))
    tr = rt.RayTracer(dims, spec.nbins, dirs, rays_per_cell=case.get("rays", 1), tune=case.get("tune"), rows=case.get("rows"),
                      slots=case.get("slots"), pair=case.get("pair"))
    try:
        w = tr.debug_writer_counts()
    finally:
        tr.close()
    report(test="one_writer", case={k: (list(v) if isinstance(v, tuple) else v) for k, v in case.items()}, **w)
    assert w["launches"] >= 1 and w["entries"] >= 1
    assert w["max_writers"] == 1, w
    assert w["max_seam_writers"] <= 1, w
    assert w["stores"] == w["expected_stores"], w
    # (C2's launches are whole entries when its wave of resident CTAs happens to be a multiple of its 16 tiles per entry)
    if case["cfg"] == "C3" and "slots" not in case and "handoff" not in (case.get("tune") or {}):
        assert w["partial_launches"] >= 1, "this case is meant to cover launches that start or end inside an entry: %r" % (w,)


# ---------------------------------------------------------------------------------------------
def test_long_dominant_axis(orc):
    """A dominant axis longer than 16384 slabs (slab programs for every slab) and rows wider than 512 cells (generic
    kernel for that layout): rt_create used to accept it and sweep uninitialised programs."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    dims = (20000, 8, 8)
    rng = np.random.default_rng(3)
    kap = rng.uniform(0.01, 0.2, (1, 8, 8, 20000)).astype(np.float32)
    S = rng.uniform(0.0, 1.0, (1, 8, 8, 20000)).astype(np.float32)
    dirs = np.concatenate([orc.healpix_dirs(1), np.array([[1, 1e-4, 2e-4], [-1, 3e-4, 0]], dtype=np.float64)])
    ref = orc.sweep(kap, S, dirs)
    tr = rt.RayTracer(dims, 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        cnt = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
        nseg = tr.total_segments()
    finally:
        tr.close()
    assert np.array_equal(cnt, ref["cnt_sum"]) and nseg == ref["seg_total"]
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL


def test_create_limits():
    import paper_1410_0763_b200 as rt
    _torch()
    d = rt.healpix_dirs(1)
    for kw in [dict(nx=(1 << 20) + 1, ny=1, nz=1), dict(nx=8, ny=8, nz=8, rays=16, dirs=rt.healpix_dirs(64))]:
        with pytest.raises(rt.RtError) as ei:
            rt.rt_create(kw["nx"], kw["ny"], kw["nz"], 1, kw.get("dirs", d), kw.get("rays", 1))
        assert ei.value.code == -1


@pytest.mark.parametrize("case", [
    dict(cfg="C2", n=60), dict(cfg="C3", n=12), dict(cfg="C4", dims=(200, 130, 96), nside=8, n=40),
    dict(cfg="C4", dims=(200, 130, 96), nside=8, n=40, tune={"handoff": 1}), dict(cfg="C5", dims=(512, 40, 24), nside=8, n=40),
    dict(cfg="C4", dims=(96, 64, 64), nside=8, n=40, rays=2),
])
def test_determinism_soak(case):
    """No atomics on the data path: repeated sweeps of one context are bitwise identical (the first sweep of a
    context runs with fresh slot accumulators, the later ones reuse them)."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS[case["cfg"]]
    dims = case.get("dims", spec.dims)
    kap, S = make_fields(case["cfg"], dims=dims)
    tr = rt.RayTracer(dims, spec.nbins, rt.healpix_dirs(case.get("nside", spec.nside)), rays_per_cell=case.get("rays", 1),
                      tune=case.get("tune"))
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        first = tr.sweep().clone()
        bad = 0
        for _ in range(case["n"]):
            bad += int(not torch.equal(tr.sweep(), first))
    finally:
        tr.close()
    assert bad == 0, "%d of %d repeated sweeps differ bitwise" % (bad, case["n"])
