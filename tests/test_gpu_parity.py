"""Parity of the CUDA path (through the C ABI) against the CPU oracle.  All tests need a GPU.

Bars (BASELINE.json north_star): integer traversal data bit-exact; summed ds within 1e-6 relative;
J within 1e-5 max relative error (reading A14 for the floor).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

J_TOL = 1e-5
DS_TOL = 1e-6


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def rel_err(got, ref):
    """A14: |got - ref| / max(|ref|, 1e-30 * max|ref|)."""
    ref = np.asarray(ref, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    floor = max(1e-30 * np.abs(ref).max(), 1e-300)
    return np.abs(got - ref) / np.maximum(np.abs(ref), floor)


def gpu_run(kap, S, dirs, Ibc=None, cell_width=1.0, flags=0, count_dirs=(), want_ds=True, slots=None, rows=None,
            stages=None, pair=None):
    import paper_1410_0763_b200 as rt
    torch = _torch()
    nb, nz, ny, nx = kap.shape
    tr = rt.RayTracer((nx, ny, nz), nb, dirs, cell_width=cell_width, flags=flags, slots=slots, rows=rows, stages=stages, pair=pair)
    out = {}
    try:
        if Ibc is not None:
            tr.set_inflow(Ibc)
        kd = torch.from_numpy(kap).cuda()
        sd = torch.from_numpy(S).cuda()
        tr.set_fields(kd, sd)
        out["Jin"] = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        out["J"] = tr.sweep(what=rt.RT_J_TOTAL).cpu().numpy()
        out["cnt_sum"] = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
        out["cnt_dirs"] = np.stack([tr.segment_counts(int(i)).cpu().numpy().astype(np.uint32) for i in count_dirs]) \
            if len(count_dirs) else None
        out["seg_total"] = tr.total_segments()
        if want_ds:
            out["sum_ds"], out["min_ds"], out["max_ds"] = tr.sum_ds()
        out["rec"], out["L"] = tr.direction_records()
        torch.cuda.synchronize()
    finally:
        tr.close()
    return out


def sample_dirs(orc, dirs, n=16, seed=0):
    """Seeded sample of directions that includes every degenerate class (zero slope, unit slope)."""
    recs = [orc.dir_record(d) for d in dirs]
    zero = [i for i, r in enumerate(recs) if r["Mb"] == 0 or r["Mc"] == 0]
    unit = [i for i, r in enumerate(recs) if r["Mb"] == 2 ** 20 or r["Mc"] == 2 ** 20]
    rng = np.random.default_rng(seed)
    pick = set(zero[:3] + unit[:3])
    for a in range(3):
        cand = [i for i, r in enumerate(recs) if r["a"] == a]
        pick.update(rng.choice(cand, size=min(3, len(cand)), replace=False).tolist())
    while len(pick) < min(n, len(dirs)):
        pick.add(int(rng.integers(0, len(dirs))))
    return sorted(pick)


def check_records(orc, dirs, out):
    for i, d in enumerate(dirs):
        r = orc.dir_record(d)
        assert out["rec"][i, 0] == r["a"]
        assert out["rec"][i, 1] == r["refl"][0] | (r["refl"][1] << 1) | (r["refl"][2] << 2)
        assert out["rec"][i, 2] == r["Mb"] and out["rec"][i, 3] == r["Mc"]
        assert abs(out["L"][i] - r["L"]) <= 1e-15 * r["L"]


def check_full(orc, kap, S, dirs, out, ref, cell_width=1.0):
    ncell = kap.shape[1] * kap.shape[2] * kap.shape[3]
    # integer traversal data: bit-exact
    assert np.array_equal(out["cnt_sum"], ref["cnt_sum"])
    assert out["seg_total"] == ref["seg_total"]
    if ref.get("cnt_dirs") is not None and out["cnt_dirs"] is not None:
        assert np.array_equal(out["cnt_dirs"], ref["cnt_dirs"])
    # summed ds: vs oracle and vs the closed form N_m * L (pin P3)
    if "sum_ds" in out:
        assert np.abs(out["sum_ds"] / ref["sum_ds"] - 1).max() <= DS_TOL
        closed = ncell * out["L"] * cell_width
        assert np.abs(out["sum_ds"] / closed - 1).max() <= DS_TOL
        assert np.abs(out["min_ds"] / (out["L"] * cell_width) - 1).max() <= 2e-6
        assert np.abs(out["max_ds"] / (out["L"] * cell_width) - 1).max() <= 2e-6
    # J_in (strict) and J
    e_in = rel_err(out["Jin"], ref["Jin"])
    e_tot = rel_err(out["J"], ref["J"])
    assert e_in.max() <= J_TOL, "J_in max rel err %.3e" % e_in.max()
    assert e_tot.max() <= J_TOL, "J max rel err %.3e" % e_tot.max()
    return e_in.max()


# ---------------------------------------------------------------------------------------------
def test_healpix_library_matches_oracle(orc):
    import paper_1410_0763_b200 as rt
    for nside in (1, 2, 3, 8, 16):
        assert np.abs(rt.healpix_dirs(nside) - orc.healpix_dirs(nside)).max() <= 1e-15


def test_c1_full(orc):
    """Config 1: 32^3, Nside 2 (48 directions), uniform random fields: everything compared in full."""
    from rt_inputs import make_fields, CONFIGS
    kap, S = make_fields("C1")
    dirs = orc.healpix_dirs(CONFIGS["C1"].nside)
    out = gpu_run(kap, S, dirs, count_dirs=range(48))
    ref = orc.sweep(kap, S, dirs, count_dirs=range(48))
    check_records(orc, dirs, out)
    assert np.all(out["rec"][:, 4] == 0), "C1 must run on the owned (atomic-free) fast path"
    check_full(orc, kap, S, dirs, out, ref)


def test_c2_full(orc):
    """Config 2: 64^3, Nside 8 (768 directions), lognormal density."""
    from rt_inputs import make_fields, CONFIGS
    kap, S = make_fields("C2")
    dirs = orc.healpix_dirs(CONFIGS["C2"].nside)
    cd = sample_dirs(orc, dirs, 16)
    out = gpu_run(kap, S, dirs, count_dirs=cd)
    ref = orc.sweep(kap, S, dirs, count_dirs=cd)
    check_records(orc, dirs, out)
    assert np.all(out["rec"][:, 4] == 0)
    check_full(orc, kap, S, dirs, out, ref)


@pytest.mark.parametrize("name,dims,nside", [
    ("C3", (64, 32, 128), 4),      # bubbles generator, anisotropic dims: three different Nb/Nc/Na per axis
    ("C5", (32, 64, 128), 4),      # 3 bins, anisotropic
    ("C4", (128, 256, 32), 2),     # wide rows (G = 2 and 4 chunks per thread)
    ("C2", (256, 32, 64), 2),
])
def test_reduced_configs_full(orc, name, dims, nside):
    """The C3/C4/C5 generators at reduced, anisotropic sizes: full comparison on every cell."""
    from rt_inputs import make_fields
    kap, S = make_fields(name, dims=dims)
    dirs = orc.healpix_dirs(nside)
    cd = sample_dirs(orc, dirs, 12)
    out = gpu_run(kap, S, dirs, count_dirs=cd)
    ref = orc.sweep(kap, S, dirs, count_dirs=cd)
    check_records(orc, dirs, out)
    assert np.all(out["rec"][:, 4] == 0)
    check_full(orc, kap, S, dirs, out, ref)


def _sample_cells(dims, n, seed, kap):
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    cells = np.stack([rng.integers(0, nx, n), rng.integers(0, ny, n), rng.integers(0, nz, n)], 1)
    corners = [[0, 0, 0], [nx - 1, ny - 1, nz - 1], [nx - 1, 0, nz - 1], [0, ny - 1, 0], [nx // 2, ny // 2, nz // 2]]
    # most and least opaque cells (bin 0)
    zmax, ymax, xmax = np.unravel_index(np.argmax(kap[0]), kap[0].shape)
    zmin, ymin, xmin = np.unravel_index(np.argmin(kap[0]), kap[0].shape)
    extra = corners + [[xmax, ymax, zmax], [xmin, ymin, zmin]]
    return np.unique(np.concatenate([cells, np.array(extra)]), axis=0).astype(np.int32)


@pytest.mark.parametrize("name,ncells", [("C3", 40), ("C4", 40), ("C5", 32)])
def test_full_size_sampled(orc, name, ncells):
    """Configs 3-5 at BASELINE.json's full sizes, in the launch configuration bench.py times:
    sampled cells the oracle computes one by one (J_in, J, counts), plus properties that hold at
    any size (total segments from the per-direction closed count, sum ds = N_m L)."""
    from rt_inputs import make_fields, CONFIGS
    import paper_1410_0763_b200 as rt
    torch = _torch()
    spec = CONFIGS[name]
    kap, S = make_fields(name)
    nb, nz, ny, nx = kap.shape
    dirs = orc.healpix_dirs(spec.nside)
    cells = _sample_cells(spec.dims, ncells, 7, kap)
    ref = orc.sweep_cells(kap, S, dirs, cells)
    tr = rt.RayTracer(spec.dims, nb, dirs)
    try:
        kd, sd = torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda()
        tr.set_fields(kd, sd)
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
    finally:
        tr.close()
    assert np.array_equal(got_cnt, ref["cnt"])                       # integer data: bit-exact
    assert seg_total == cnt_total
    e_in, e_J = rel_err(got_in, ref["Jin"]), rel_err(got_J, ref["J"])
    assert e_in.max() <= J_TOL, "%s J_in max rel err %.3e" % (name, e_in.max())
    assert e_J.max() <= J_TOL, "%s J max rel err %.3e" % (name, e_J.max())
    # segments per direction: N_m (1 + m_b + m_c) within the degenerate-slope deficit (pin P4 band)
    pred = spec.ncell * np.sum(1.0 + rec[:, 2] / 2.0 ** 20 + rec[:, 3] / 2.0 ** 20)
    assert abs(seg_total - pred) < 0.02 * pred


def test_full_size_sum_ds_c3(orc):
    """Sum of ds per direction at a full benchmark size against the closed form N_m * L (P3)."""
    from rt_inputs import CONFIGS
    import paper_1410_0763_b200 as rt
    _torch()
    spec = CONFIGS["C3"]
    dirs = orc.healpix_dirs(spec.nside)[::24]          # 128 of the 3072 directions
    tr = rt.RayTracer(spec.dims, 1, dirs)
    try:
        s, mn, mx = tr.sum_ds()
        rec, L = tr.direction_records()
    finally:
        tr.close()
    assert np.abs(s / (spec.ncell * L) - 1).max() <= DS_TOL
    assert np.abs(mn / L - 1).max() <= 2e-6 and np.abs(mx / L - 1).max() <= 2e-6


# ---------------------------------------------------------------------------------------------
# edge cases
def _rand(dims, seed, nb=1):
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    return (rng.uniform(0.05, 2.0, (nb, nz, ny, nx)).astype(np.float32),
            rng.uniform(0.0, 1.0, (nb, nz, ny, nx)).astype(np.float32))


@pytest.mark.parametrize("dims", [(20, 12, 10), (33, 7, 5), (1, 1, 1), (64, 20, 12), (20, 64, 12)])
def test_generic_fallback_dims(orc, dims):
    """Small and odd mesh sizes: since rows are padded to 32/64/128/256/512 cells these all run on the owned kernel
    (R falls back to 1 for odd N_c; the 1 x 1 x 1 mesh too); only rows wider than 512 cells use the generic four-group
    kernel (test_padded_rows_take_the_owned_path covers (600, 8, 4)).  Same gates."""
    kap, S = _rand(dims, 5)
    dirs = orc.healpix_dirs(2)
    out = gpu_run(kap, S, dirs, count_dirs=range(0, 48, 5))
    ref = orc.sweep(kap, S, dirs, count_dirs=range(0, 48, 5))
    check_records(orc, dirs, out)
    check_full(orc, kap, S, dirs, out, ref)


@pytest.mark.parametrize("dims,nb", [((100, 60, 24), 1), ((130, 200, 8), 1), ((33, 7, 5), 2), ((250, 31, 9), 1), ((300, 16, 8), 1), ((512, 24, 8), 1), ((40, 500, 6), 1), ((600, 8, 4), 1)])
def test_padded_rows_take_the_owned_path(orc, dims, nb):
    """Row widths other than 32/64/128/256 are padded to the next such width (pad cells: kappa = 0, S = 0)
    and swept by the owned kernel (mirror pairs, reversed singles and counting modes all cross the pad);
    rows wider than 512 cells still fall back to the generic kernel for the layout they affect.  Same gates, with inflow."""
    kap, S = _rand(dims, 29, nb=nb)
    dirs = np.concatenate([orc.healpix_dirs(2), np.array([[1, 1, 1], [-1, 0.5, 0.25], [0.3, -1, 0]], dtype=np.float64)])
    Ibc = [0.4, 0.1][:nb]
    cd = [0, 7, 20, 33, 48, 49, 50]
    out = gpu_run(kap, S, dirs, Ibc=Ibc, count_dirs=cd)
    ref = orc.sweep(kap, S, dirs, Ibc=Ibc, count_dirs=cd)
    check_records(orc, dirs, out)
    layout_fast = {0: dims[0] <= 512, 1: dims[1] <= 512}
    for i in range(len(dirs)):
        assert out["rec"][i, 4] == (0 if layout_fast[1 if out["rec"][i, 0] == 0 else 0] else 1)
    check_full(orc, kap, S, dirs, out, ref)


@pytest.mark.parametrize("flags", [1, 2])
def test_ablation_variants_pass_the_same_gates(orc, flags):
    """RT_ATOMIC_ABLATION and RT_PAPER_GROUPS differ from the owned path only by summation order."""
    from rt_inputs import make_fields
    kap, S = make_fields("C1")
    dirs = orc.healpix_dirs(2)
    out = gpu_run(kap, S, dirs, flags=flags, count_dirs=range(0, 48, 7))
    ref = orc.sweep(kap, S, dirs, count_dirs=range(0, 48, 7))
    assert np.all(out["rec"][:, 4] == 1)
    check_full(orc, kap, S, dirs, out, ref)


@pytest.mark.parametrize("rows,stages,pair", [(1, 2, 1), (2, 2, 0), (2, 2, 1), (1, 3, 0), (2, 3, 1), (1, 3, 1), (4, 2, 1), (4, 2, 0), (4, 3, 1), (1, 4, 1), (2, 4, 0)])
def test_rows_per_warp_variants(orc, rows, stages, pair):
    kap, S = _rand((64, 32, 16), 9)
    dirs = orc.healpix_dirs(2)
    out = gpu_run(kap, S, dirs, rows=rows, stages=stages, pair=pair, slots=5, count_dirs=[0, 13, 47])
    ref = orc.sweep(kap, S, dirs, count_dirs=[0, 13, 47])
    check_full(orc, kap, S, dirs, out, ref)


@pytest.mark.parametrize("dims,rows,pair", [((64, 32, 16), 2, 1), ((128, 64, 40), 2, 1), ((32, 24, 64), 1, 0), ((256, 16, 6), 2, 1)])
def test_seam_handoff_ablation(orc, dims, rows, pair):
    """rt_tune("handoff"): seam partials go to the next warp of the CTA through shared memory instead of
    the seam accumulator; only the summation order within a cell changes.  Includes row counts that
    leave a CTA partly filled (Nc = 40, 6) and a single-warp CTA."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    kap, S = _rand(dims, 21, nb=2)
    dirs = orc.healpix_dirs(2)
    ref = orc.sweep(kap, S, dirs)
    nx, ny, nz = dims
    tr = rt.RayTracer(dims, 2, dirs, rows=rows, pair=pair, tune={"handoff": 1})
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        Jin2 = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        cnt = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
    finally:
        tr.close()
    assert np.array_equal(Jin, Jin2)
    assert np.array_equal(cnt, ref["cnt_sum"])
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL


def test_inflow_cellwidth_multibin(orc):
    kap, S = _rand((32, 64, 16), 11, nb=3)
    dirs = orc.healpix_dirs(2)
    Ibc = [0.5, 0.0, 2.0]
    out = gpu_run(kap, S, dirs, Ibc=Ibc, cell_width=0.7)
    ref = orc.sweep(kap, S, dirs, Ibc=Ibc, cell_width=0.7)
    check_full(orc, kap, S, dirs, out, ref, cell_width=0.7)


@pytest.mark.parametrize("name,dims,nside", [("C5", (64, 32, 48), 2), ("C2", (32, 32, 32), 2), ("C5", (20, 12, 10), 1),
                                             ("C5", (128, 130, 12), 1), ("C3", (192, 128, 8), 1)])   # the 64 x 64-tile epilogue
def test_rates_epilogue(orc, name, dims, nside):
    """rt_sweep_rates against the oracle's rates() of the oracle's J_in (eqs. 14-15, 20-23): 1e-5."""
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields
    torch = _torch()
    kap, S = make_fields(name, dims=dims)
    nb = kap.shape[0]
    dirs = orc.healpix_dirs(nside)
    rng = np.random.default_rng(3)
    w = rng.uniform(0.2, 3.0, (4, nb))
    ref = orc.sweep(kap, S, dirs, want_counts=False)
    Gr, Hr = orc.rates(ref["Jin"], S.astype(np.float64), w[0], w[1], w[2], w[3])
    tr = rt.RayTracer(dims, nb, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        G, H = tr.sweep_rates(w[0], w[1], w[2], w[3])
        G, H = G.cpu().numpy(), H.cpu().numpy()
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()      # the sweep is unchanged by the epilogue call
    finally:
        tr.close()
    assert rel_err(G, Gr).max() <= J_TOL and rel_err(H, Hr).max() <= J_TOL
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL


@pytest.mark.parametrize("world", [2, 3])
def test_direction_shards_combine(orc, world):
    """Direction sharding on one GPU: one context per share swept with RT_SUM_IN, the
    shares added (what the all-reduce does), rt_combine -> J of the whole set within 1e-5 of the oracle."""
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields
    torch = _torch()
    dims = (64, 32, 48)
    kap, S = make_fields("C3", dims=dims)
    dirs = orc.healpix_dirs(4)
    ref = orc.sweep(kap, S, dirs, want_counts=False)
    kd, sd = torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda()
    total = None
    trs = []
    try:
        for r in range(world):
            tr = rt.RayTracer(dims, 1, dirs[rt.shard_directions(dirs, world, r)])
            trs.append(tr)
            tr.set_fields(kd, sd)
            part = tr.sweep(what=rt.RT_SUM_IN)
            total = part if total is None else total + part
        Jin = trs[0].combine(total.clone(), len(dirs), what=rt.RT_J_IN).cpu().numpy()
        J = trs[-1].combine(total.clone(), len(dirs), what=rt.RT_J_TOTAL).cpu().numpy()
        one = rt.sweep_sharded(trs[0], len(trs[0].dirs), what=rt.RT_J_IN).cpu().numpy()   # world of 1: no collective
        ref0 = trs[0].sweep(what=rt.RT_J_IN).cpu().numpy()
    finally:
        for tr in trs:
            tr.close()
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL
    assert rel_err(J, ref["J"]).max() <= J_TOL
    assert rel_err(one, ref0).max() <= 1e-6


@pytest.mark.parametrize("dims,rays,flags", [((64, 32, 16), 2, 0), ((32, 64, 24), 4, 0), ((20, 12, 10), 2, 0), ((32, 32, 8), 2, 1)])
def test_rays_per_cell(orc, dims, rays, flags):
    """r > 1 rays per cell width (ray spacing dH / r; reading O3/A13): r^2 interleaved unit
    lattices.  Counts bit-exact (per direction and summed), sum ds = r^2 N_m L to 1e-6, J to 1e-5; owned
    (mirror-pair) path, generic path and the atomic ablation."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    kap, S = _rand(dims, 23, nb=2)
    dirs = np.concatenate([orc.healpix_dirs(1), np.array([[1, 1, 1], [1, 0.5, 0.25], [0, -1, 0], [0.3, 0.2, -1]], dtype=np.float64)])
    cd = [0, 5, 12, 13, 14, 15]
    ref = orc.sweep(kap, S, dirs, Ibc=[0.3, 0.0], count_dirs=cd, rays_per_cell=rays)
    tr = rt.RayTracer(dims, 2, dirs, flags=flags, rays_per_cell=rays)
    try:
        tr.set_inflow([0.3, 0.0])
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        J = tr.sweep(what=rt.RT_J_TOTAL).cpu().numpy()
        cnt = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
        cnt_d = np.stack([tr.segment_counts(i).cpu().numpy().astype(np.uint32) for i in cd])
        nseg = tr.total_segments()
        s, mn, mx = tr.sum_ds()
        rec, L = tr.direction_records()
    finally:
        tr.close()
    assert np.all(rec[:, 5] == rays)
    assert np.array_equal(cnt, ref["cnt_sum"]) and nseg == ref["seg_total"]
    assert np.array_equal(cnt_d, ref["cnt_dirs"])
    ncell = dims[0] * dims[1] * dims[2]
    assert np.abs(s / ref["sum_ds"] - 1).max() <= DS_TOL
    assert np.abs(s / (ncell * rays ** 2 * L) - 1).max() <= DS_TOL
    assert np.abs(mn / (rays ** 2 * L) - 1).max() <= 2e-6 and np.abs(mx / (rays ** 2 * L) - 1).max() <= 2e-6
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL
    assert rel_err(J, ref["J"]).max() <= J_TOL


@pytest.mark.parametrize("dims,flags,rays", [((64, 32, 16), 0, 1), ((100, 60, 24), 0, 1), ((32, 64, 24), 0, 2), ((20, 12, 10), 2, 1), ((32, 32, 8), 1, 1)])
def test_per_face_inflow(orc, dims, flags, rays):
    """rt_set_inflow_faces (boundary illumination; reading A10): the ray chains of the owned
    kernel (a-face at the start, b-face at the lane wrap - opposite faces for a mirror pair -, c-face at the
    row wrap) and the per-ray rule of the generic kernel against the oracle; includes exact diagonals, where
    a ray enters through an edge."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    kap, S = _rand(dims, 37, nb=2)
    kap *= 0.2                                           # thin enough that the inflow reaches every cell
    dirs = np.concatenate([orc.healpix_dirs(2), np.array([[1, 1, 1], [-1, 1, -1], [1, -1, 0], [0, 0, -1], [0.5, 1, 0.5]], dtype=np.float64)])
    faces = np.array([[0.1, 0.9, 0.3, 0.7, 0.5, 0.2], [1.5, 0.0, 0.0, 2.5, 0.25, 0.75]])
    ref = orc.sweep(kap, S, dirs, Ibc_faces=faces, rays_per_cell=rays, want_counts=False)
    tr = rt.RayTracer(dims, 2, dirs, flags=flags, rays_per_cell=rays)
    try:
        tr.set_inflow_faces(faces)
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        tr.set_inflow([0.4, 0.0])                        # back to one value per bin
        Jin_u = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
    finally:
        tr.close()
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL
    ref_u = orc.sweep(kap, S, dirs, Ibc=[0.4, 0.0], rays_per_cell=rays, want_counts=False)
    assert rel_err(Jin_u, ref_u["Jin"]).max() <= J_TOL


def test_degenerate_directions(orc):
    """Axis-aligned, exact diagonals, unit slopes, half slopes (crossings on slab planes), near-degenerate."""
    kap, S = _rand((32, 32, 32), 13)
    dirs = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1], [1, 1, 1], [-1, 1, -1],
                     [1, 1, 0], [0, -1, 1], [1, 0.5, 0.25], [0.5, -1, 0.5], [1, 0.999999, 1e-6], [0.25, 0.75, -1],
                     [1e-7, 1, 1e-7]], dtype=np.float64)
    out = gpu_run(kap, S, dirs, count_dirs=range(len(dirs)))
    ref = orc.sweep(kap, S, dirs, count_dirs=range(len(dirs)))
    check_records(orc, dirs, out)
    check_full(orc, kap, S, dirs, out, ref)


def test_kappa_zero_and_extremes(orc):
    """kappa = 0 (A7), tiny and huge optical depths: finite, and within tolerance (kappa floor 2^-60)."""
    kap, S = _rand((32, 32, 32), 17)
    kap[0, 8:12] = 0.0
    kap[0, 20:22] = 1e-6
    kap[0, 25:27] = 300.0
    dirs = orc.healpix_dirs(2)
    out = gpu_run(kap, S, dirs, want_ds=False)
    ref = orc.sweep(kap, S, dirs)
    assert np.all(np.isfinite(out["Jin"]))
    assert np.array_equal(out["cnt_sum"], ref["cnt_sum"])
    # behind 300 mean free paths per cell J_in of the far side underflows; A14 floor handles it
    assert rel_err(out["Jin"], ref["Jin"]).max() <= J_TOL
    assert rel_err(out["J"], ref["J"]).max() <= J_TOL


def test_error_codes():
    import paper_1410_0763_b200 as rt
    torch = _torch()
    d = rt.healpix_dirs(1)
    for bad in [dict(nx=0), dict(nbins=0), dict(nbins=17), dict(rays=3), dict(rays=32), dict(cw=0.0), dict(flags=7)]:
        with pytest.raises(rt.RtError) as ei:
            rt.rt_create(bad.get("nx", 8), 8, 8, bad.get("nbins", 1), d, bad.get("rays", 1), bad.get("cw", 1.0),
                         bad.get("flags", 0))
        assert ei.value.code == -1
    with pytest.raises(rt.RtError):
        rt.rt_create(8, 8, 8, 1, np.zeros((1, 3)))
    h = rt.rt_create(8, 8, 8, 1, d)
    try:
        J = torch.empty(512, dtype=torch.float32, device="cuda")
        with pytest.raises(rt.RtError) as ei:
            rt.rt_sweep(h, J, 512)                      # fields not set
        assert ei.value.code == -4
    finally:
        rt.rt_destroy(h)


def test_unsupported_tuning_is_refused_before_allocation(orc):
    """A ring of 4 TMA stages exists only for rows of <= 64 cells.  On 128-cell rows rt_set_fields refuses it with
    RT_EINVAL before any buffer exists, so that rt_tune can still correct the knob and the context then sweeps as usual."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    dims = (128, 16, 8)
    kap, S = _rand(dims, 5)
    dirs = rt.healpix_dirs(1)
    tr = rt.RayTracer(dims, 1, dirs, stages=4)
    try:
        kd, sd = torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda()
        with pytest.raises(rt.RtError) as ei:
            tr.set_fields(kd, sd)
        assert ei.value.code == -1
        rt.rt_tune(tr.h, "stages", 2)                   # still allowed: nothing was allocated
        tr.set_fields(kd, sd)
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
    finally:
        tr.close()
    ref = orc.sweep(kap, S, dirs)
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL


@pytest.mark.parametrize("tune", [{"overlap": 0}, {"overlap": 1, "graph": 0}, {"overlap": 1, "graph": 1}, {"overlap": 1, "wave_div": 4},
                                  {"overlap": 0, "graph": 1}])
def test_schedules_agree(orc, tune):
    """The overlapped schedule (classes on internal streams with slot ranges of their own), its CUDA-graph replay and
    the one-launch-after-the-other schedule sweep the same entries with the same arithmetic: all within 1e-5 of the
    oracle, repeated sweeps bitwise equal (the second and later ones are graph replays when the graph is on), on the
    caller's default stream and on a side stream."""
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields
    torch = _torch()
    dims = (64, 32, 48)
    kap, S = make_fields("C5", dims=dims)
    dirs = orc.healpix_dirs(4)
    ref = orc.sweep(kap, S, dirs, Ibc=[0.2, 0.0, 0.1], want_counts=False)
    tr = rt.RayTracer(dims, 3, dirs, tune=tune)
    try:
        tr.set_inflow([0.2, 0.0, 0.1])
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        out = torch.empty(tr.shape(), dtype=torch.float32, device="cuda")
        first = tr.sweep(out=out).clone()
        for _ in range(4):
            assert torch.equal(tr.sweep(out=out), first)
        Jtot = tr.sweep(what=rt.RT_J_TOTAL).cpu().numpy()
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for _ in range(3):
                side = tr.sweep(out=out, stream=st).clone()
        st.synchronize()
        assert torch.equal(side, first)
        kap2 = kap * np.float32(0.5)                         # new fields: the replayed graph must see them
        tr.set_fields(torch.from_numpy(kap2).cuda(), torch.from_numpy(S).cuda())
        again = tr.sweep(out=out).cpu().numpy()
    finally:
        tr.close()
    assert rel_err(first.cpu().numpy(), ref["Jin"]).max() <= J_TOL
    assert rel_err(Jtot, ref["J"]).max() <= J_TOL
    ref2 = orc.sweep(kap2, S, dirs, Ibc=[0.2, 0.0, 0.1], want_counts=False)
    assert rel_err(again, ref2["Jin"]).max() <= J_TOL


@pytest.mark.parametrize("tune", [{"overlap": 0}, {"overlap": 1}])
def test_sweep_inside_a_callers_stream_capture(tune):
    """A caller may capture rt_sweep into a CUDA graph of its own.  The library then records no timing events into that
    graph (rt_last_sweep_kernel_ms says "unavailable" instead of failing on events that were never executed) and does not
    start a graph of its own inside the capture; replays of the caller's graph give the bits of a plain sweep."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    dims = (64, 32, 16)
    kap, S = _rand(dims, 43)
    tr = rt.RayTracer(dims, 1, rt.healpix_dirs(2), tune=tune)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        plain = tr.sweep().clone()                       # also the first launch of every kernel, outside any capture
        assert tr.last_sweep_kernel_ms() > 0.0
        out = torch.zeros_like(plain)
        st = torch.cuda.Stream()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st, capture_error_mode="thread_local"):
            tr.sweep(out=out, stream=torch.cuda.current_stream())
        assert tr.last_sweep_kernel_ms() < 0.0 and not tr.last_sweep_was_graph()
        for _ in range(2):
            out.zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, plain)
        again = tr.sweep()                               # and the context still sweeps, and times, outside the capture
        assert torch.equal(again, plain) and tr.last_sweep_kernel_ms() > 0.0
    finally:
        tr.close()


@pytest.mark.parametrize("tune", [{"overlap": 1, "graph": 1}, {"overlap": 0, "graph": 0}])
def test_async_inflow_between_sweeps_on_a_side_stream(orc, tune):
    """rt_set_inflow_faces_async / rt_set_inflow_async are ordered by the stream they are enqueued on, with no device
    synchronisation (a boundary illumination that changes every iteration): sweeps, inflow updates and
    more sweeps (CUDA-graph replays when the graph is on) are all enqueued on a side stream before the host waits once;
    every sweep must carry the inflow that was current at its place in the stream."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    dims = (64, 32, 16)
    kap, S = _rand(dims, 41, nb=2)
    kap *= 0.2                                           # thin enough that the inflow reaches every cell
    dirs = orc.healpix_dirs(2)
    faces = np.array([[0.1, 0.9, 0.3, 0.7, 0.5, 0.2], [1.5, 0.0, 0.0, 2.5, 0.25, 0.75]])
    tr = rt.RayTracer(dims, 2, dirs, tune=tune)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        torch.cuda.synchronize()
        st = torch.cuda.Stream()
        out = torch.empty(tr.shape(), dtype=torch.float32, device="cuda")
        got = []
        with torch.cuda.stream(st):
            for _ in range(3):                           # inflow 0; from the second use on a graph replay
                tr.sweep(out=out, stream=st)
            got.append(out.clone())
            tr.set_inflow_faces_async(faces, stream=st)
            for _ in range(2):
                tr.sweep(out=out, stream=st)
            got.append(out.clone())
            tr.set_inflow_async([0.4, 0.0], stream=st)
            tr.sweep(out=out, stream=st)
            got.append(out.clone())
        st.synchronize()
        got = [g.cpu().numpy() for g in got]
        with pytest.raises(rt.RtError):
            tr.set_inflow_async([-1.0, 0.0])
    finally:
        tr.close()
    refs = [orc.sweep(kap, S, dirs, want_counts=False), orc.sweep(kap, S, dirs, Ibc_faces=faces, want_counts=False),
            orc.sweep(kap, S, dirs, Ibc=[0.4, 0.0], want_counts=False)]
    for g, r in zip(got, refs):
        assert rel_err(g, r["Jin"]).max() <= J_TOL


@pytest.mark.parametrize("dims,nb,rows,rays,nside", [
    ((32, 64, 16), 3, None, 1, 2),          # 32- and 64-cell rows, three bins in one group
    ((128, 64, 40), 3, 1, 1, 2),            # 128-cell rows (C5's width), one ray row per warp
    ((128, 128, 24), 3, 2, 1, 2),           # two ray rows per warp
    ((64, 32, 24), 6, None, 1, 2),          # two groups of three bins (grid.z = 2)
    ((100, 60, 24), 3, None, 1, 2),         # padded rows
    ((32, 64, 24), 3, None, 2, 1),          # r = 2 sub-lattices
])
def test_packed_bins(orc, dims, nb, rows, rays, nside):
    """rt_tune("binpack", 1): the multi-bin packed kernel (three bins of a cell row share the row: one bulk copy, one
    slab program, one set of addresses for three intensity recurrences) against the oracle, with
    per-face inflow that differs per bin (the b-handoff's carry restarts at every bin), plus everything that reads the
    packed layout: J total, the rates epilogue, rt_combine, point sources, counts, writer counts."""
    import paper_1410_0763_b200 as rt
    torch = _torch()
    kap, S = _rand(dims, 41, nb=nb)
    kap *= (0.3 + 0.5 * np.arange(nb, dtype=np.float32))[:, None, None, None]
    dirs = np.concatenate([orc.healpix_dirs(nside), np.array([[1, 1, 1], [-1, 0.5, 0.25], [0, 0, -1], [0.3, -1, 0]], dtype=np.float64)])
    rng = np.random.default_rng(5)
    faces = rng.uniform(0.0, 1.0, (nb, 6))
    w = rng.uniform(0.2, 3.0, (4, nb))
    ref = orc.sweep(kap, S, dirs, Ibc_faces=faces, rays_per_cell=rays)
    Gr, Hr = orc.rates(ref["Jin"], S.astype(np.float64), w[0], w[1], w[2], w[3])
    src = np.array([[0, 0, 0], [dims[0] * 128, dims[1] * 128 + 77, dims[2] * 256]], dtype=np.int32)
    lum = rng.uniform(0.5, 2.0, (2, nb))
    refQ = orc.point_sources(kap, src, lum, want_diag=False)
    tr = rt.RayTracer(dims, nb, dirs, rows=rows, rays_per_cell=rays, tune={"binpack": 1})
    try:
        tr.set_inflow_faces(faces)
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Jin = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        Jin2 = tr.sweep(what=rt.RT_J_IN).cpu().numpy()
        J = tr.sweep(what=rt.RT_J_TOTAL).cpu().numpy()
        G, H = tr.sweep_rates(w[0], w[1], w[2], w[3])
        G, H = G.cpu().numpy(), H.cpu().numpy()
        tot = tr.sweep(what=rt.RT_SUM_IN)
        Jc = tr.combine(tot, len(dirs), what=rt.RT_J_TOTAL).cpu().numpy()
        Q, _, steps = tr.point_sources(src, lum, want_steps=True)
        Q = Q.cpu().numpy()
        cnt = tr.segment_counts(-1).cpu().numpy().astype(np.uint32)
        wr = tr.debug_writer_counts()
    finally:
        tr.close()
    assert np.array_equal(Jin, Jin2)
    assert np.array_equal(cnt, ref["cnt_sum"])
    assert rel_err(Jin, ref["Jin"]).max() <= J_TOL and rel_err(J, ref["J"]).max() <= J_TOL
    assert rel_err(Jc, ref["J"]).max() <= J_TOL
    assert rel_err(G, Gr).max() <= J_TOL and rel_err(H, Hr).max() <= J_TOL
    assert steps == refQ["steps"] and rel_err(Q, refQ["Q"]).max() <= J_TOL
    assert wr["max_writers"] == 1 and wr["max_seam_writers"] <= 1 and wr["stores"] == wr["expected_stores"]


def test_sweep_is_deterministic_and_repeatable(orc):
    from rt_inputs import make_fields
    import paper_1410_0763_b200 as rt
    torch = _torch()
    kap, S = make_fields("C1")
    dirs = orc.healpix_dirs(2)
    tr = rt.RayTracer((32, 32, 32), 1, dirs)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        a = tr.sweep().clone()
        b = tr.sweep().clone()
        assert torch.equal(a, b)                       # atomic-free: bitwise reproducible
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            c = tr.sweep(stream=st).clone()
        st.synchronize()
        assert torch.equal(a, c)
        assert tr.last_launch_count() >= 2
    finally:
        tr.close()
