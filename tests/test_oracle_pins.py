"""Pins of the CPU oracle (oracle/oracle.c) against things other than itself.

Each test names the pin (P1..P11) and what mistake it would catch.
No GPU, no CUDA library: these run in the `-m "not gpu"` suite.
"""
import math
import os

import numpy as np
import pytest

from tests import bruteforce as bf

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


def rand_fields(dims, seed, kmin=0.05, kmax=2.0, nb=1):
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    kap = rng.uniform(kmin, kmax, size=(nb, nz, ny, nx)).astype(np.float32)
    S = rng.uniform(0.0, 1.0, size=(nb, nz, ny, nx)).astype(np.float32)
    return kap, S


# ---------------------------------------------------------------- P1: direction generator
@pytest.mark.parametrize("nside", [1, 2, 4, 8, 16])
def test_p1_healpix_count_norm_symmetry(orc, nside):
    d = orc.healpix_dirs(nside)
    assert d.shape == (12 * nside * nside, 3)                       # N_d = 12 Nside^2
    assert np.abs(np.linalg.norm(d, axis=1) - 1.0).max() < 1e-15
    assert np.abs(d.sum(axis=0)).max() < 1e-11                      # isotropic set: sum n = 0
    key = lambda a: sorted(map(tuple, np.round(a, 12) + 0.0))
    base = key(d)
    for ax in range(3):                                             # invariant under mirror of each axis
        m = d.copy()
        m[:, ax] *= -1
        assert key(m) == base
    assert key(d[:, [1, 0, 2]]) == base                             # and under x <-> y
    # RING order: z non-increasing
    assert np.all(np.diff(d[:, 2]) <= 1e-15)


def test_p1_healpix_nside1_base_pixels(orc):
    """Nside = 1: the 12 base-pixel centres: z = +-2/3 at phi = pi/4 + k pi/2, z = 0 at phi = k pi/2."""
    d = orc.healpix_dirs(1)
    z = d[:, 2]
    assert np.allclose(z[:4], 2.0 / 3.0, atol=1e-15) and np.allclose(z[8:], -2.0 / 3.0, atol=1e-15)
    assert np.allclose(z[4:8], 0.0, atol=1e-15)
    phi = np.mod(np.arctan2(d[:, 1], d[:, 0]), 2 * np.pi)
    assert np.allclose(np.sort(phi[:4]), np.pi / 4 + np.arange(4) * np.pi / 2, atol=1e-14)
    eq = {tuple(np.round(v, 12) + 0.0) for v in d[4:8]}
    assert eq == {(1.0, 0.0, 0.0), (-1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, -1.0, 0.0)}


@pytest.mark.parametrize("nside", [2, 4, 16])
def test_p1_healpix_equal_area_rings(orc, nside):
    """Equal-area pixels on iso-latitude rings: the pixels north of the boundary between ring i and
    ring i+1 tile a cap of area 2 pi (1 - z_edge); with equal areas their count fixes z_edge, and
    every ring centre must lie strictly between consecutive edges.  Also ring z from the closed form."""
    d = orc.healpix_dirs(nside)
    npix = d.shape[0]
    zs, counts = np.unique(np.round(d[:, 2], 13), return_counts=True)
    zs, counts = zs[::-1], counts[::-1]
    assert len(zs) == 4 * nside - 1
    assert abs(zs[0] - (1 - 1 / (3 * nside ** 2))) < 1e-12          # ring 1
    assert abs(zs[2 * nside - 1]) < 1e-12                           # ring 2 Nside is the equator
    cum = np.cumsum(counts)
    z_edge = 1.0 - 2.0 * cum / npix                                 # cap area fraction = (1 - z)/2
    upper = np.concatenate([[1.0], z_edge[:-1]])
    assert np.all(zs < upper + 1e-12) and np.all(zs > z_edge - 1e-12)


def test_p1_direction_record(orc):
    r = orc.dir_record([0.3, -0.9, 0.2])
    assert r["a"] == 1 and r["refl"] == (0, 1, 0)
    assert r["Mb"] == round(0.3 / 0.9 * 2 ** 20) and r["Mc"] == round(0.2 / 0.9 * 2 ** 20)
    assert abs(r["L"] - math.sqrt(1 + (r["Mb"] / 2 ** 20) ** 2 + (r["Mc"] / 2 ** 20) ** 2)) < 1e-15
    assert orc.dir_record([1.0, 1.0, 1.0])["a"] == 0                # ties -> lowest axis (A5)
    assert orc.dir_record([0.0, 1.0, 1.0])["a"] == 1
    assert orc.dir_record([6e-17, 1.0, 0.0])["Mb"] == 0             # cos(pi/2) noise quantises to 0 (A6)
    with pytest.raises(ValueError):
        orc.dir_record([0.0, 0.0, 0.0])
    # agreement with the brute-force module's separately written record
    rng = np.random.default_rng(5)
    for n in rng.normal(size=(50, 3)):
        a, b, c, refl, Mb, Mc, L = bf.dir_record(n)
        r = orc.dir_record(n)
        assert (r["a"], r["Mb"], r["Mc"]) == (a, Mb, Mc) and r["refl"] == tuple(int(x) for x in refl)


# ---------------------------------------------------------------- P2: axis-aligned hand enumeration
def test_p2_axis_aligned_4cubed(orc):
    """6 axis directions on a 4^3 mesh: every cell has one segment of length 1 per direction;
    along each row I follows the textbook recurrence; J_in = (1/6) sum_dir I_in f(kappa) (eqs. 7, 8, 13)."""
    dims = (4, 4, 4)
    kap, S = rand_fields(dims, 11)
    dirs = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=np.float64)
    r = orc.sweep(kap, S, dirs, count_dirs=range(6))
    assert r["seg_total"] == 6 * 64
    assert np.all(r["cnt_dirs"] == 1)
    assert np.allclose(r["sum_ds"], 64.0, rtol=0, atol=1e-12)
    k3, s3 = kap[0].astype(np.float64), S[0].astype(np.float64)
    expect = np.zeros((4, 4, 4))
    for axis in range(3):                      # numpy axis of [z][y][x]: 0=z,1=y,2=x
        for sign in (+1, -1):
            kk = np.moveaxis(k3, axis, 0)
            ss = np.moveaxis(s3, axis, 0)
            out = np.zeros_like(kk)
            order = range(4) if sign > 0 else range(3, -1, -1)
            I = np.zeros(kk.shape[1:])
            for i in order:
                tau = kk[i]
                out[i] = I * (1 - np.exp(-tau)) / tau
                I = I * np.exp(-tau) + ss[i] * (1 - np.exp(-tau))
            expect += np.moveaxis(out, 0, axis) / 6.0
    assert np.allclose(r["Jin"][0], expect, rtol=1e-13, atol=0)
    assert np.allclose(r["J"][0], expect + s3, rtol=1e-13, atol=0)          # eq. 12


# ---------------------------------------------------------------- P3 / P4: lattice invariants
@pytest.mark.parametrize("dims", [(8, 8, 8), (16, 8, 4), (4, 8, 16), (6, 5, 4)])
def test_p3_per_cell_sum_ds_equals_L(orc, dims):
    """Equally spaced rays: per cell and direction sum_j ds_j = L exactly, hence
    sum ds = N_m L = mesh volume / per-ray cross-section (north_star invariant)."""
    kap, S = rand_fields(dims, 3)
    dirs = np.array([[1, 0.4, 0], [1, 0.5, 0], [0.37, 1, 0.81], [1, 1, 1], [0.5, 0.25, 1], [0, 0, -1],
                     [0.3333, -1, 0.9], [-0.77, 0.12, -1], [1, 1, 0], [-1, -0.999999, 0.5]], dtype=np.float64)
    r = orc.sweep(kap, S, dirs)
    ncell = dims[0] * dims[1] * dims[2]
    for i, n in enumerate(dirs):
        L = orc.dir_record(n)["L"]
        assert abs(r["min_den"][i] - L) < 1e-12 * L and abs(r["max_den"][i] - L) < 1e-12 * L
        assert abs(r["sum_ds"][i] - ncell * L) < 1e-11 * ncell * L


def test_p3_healpix_set_sum_ds(orc):
    dims = (12, 10, 14)
    kap, S = rand_fields(dims, 4)
    dirs = orc.healpix_dirs(4)
    r = orc.sweep(kap, S, dirs)
    L = np.array([orc.dir_record(n)["L"] for n in dirs])
    assert np.allclose(r["min_den"], L, rtol=1e-12) and np.allclose(r["max_den"], L, rtol=1e-12)


def test_p4_segment_count_band(orc):
    """Segments per direction = N_m (1 + m_b + m_c) for generic slopes (cost model PAPER.md:177)."""
    dims = (32, 32, 32)
    kap, S = rand_fields(dims, 6)
    dirs = np.array([[1, 0.37, 0.81], [0.123, -1, 0.456]], dtype=np.float64)
    for n in dirs:
        r = orc.sweep(kap, S, n[None], want_counts=False)
        rec = orc.dir_record(n)
        pred = 32 ** 3 * (1 + rec["Mb"] / 2 ** 20 + rec["Mc"] / 2 ** 20)
        assert abs(r["seg_total"] - pred) < 0.02 * pred
    # rational-degenerate slopes from half-integer origins: every crossing lies on a slab plane
    r = orc.sweep(kap, S, np.array([[1, 0.5, 0.25]]), want_counts=False)
    assert r["seg_total"] == 32 ** 3


# ---------------------------------------------------------------- P5: uniform medium closed form
def test_p5_uniform_slab_closed_form(orc):
    """Uniform kappa, S, zero inflow: exit intensity = S (1 - exp(-kappa * chord)) for every ray (eq. 7
    is exact for piecewise-constant media), independent of the segmentation."""
    dims = (10, 12, 8)
    kap = np.full((1, 8, 12, 10), 0.3, dtype=np.float32)
    S = np.full_like(kap, 1.7)
    k64, s64 = float(kap.flat[0]), float(S.flat[0])
    for n in ([1, 0.37, 0.81], [-0.2, 0.5, -1], [0, 1, 0], [1, 1, 1]):
        t = orc.trace_direction(kap, S, n)
        expect = s64 * (1 - np.exp(-k64 * t["chord"]))
        assert np.allclose(t["exitI"][..., 0], expect, rtol=1e-13, atol=1e-15)
        assert t["chord"].max() > 5.0
    # with inflow I_bc: I = I_bc e^-tau + S (1 - e^-tau)
    t = orc.trace_direction(kap, S, [1, 0.37, 0.81], Ibc=[0.9])
    tau = k64 * t["chord"]
    assert np.allclose(t["exitI"][..., 0], 0.9 * np.exp(-tau) + s64 * (1 - np.exp(-tau)), rtol=1e-13)


def test_p5_pure_absorption_keeps_relative_accuracy(orc):
    """S = 0, inflow I_bc: exit intensity = I_bc exp(-kappa * chord) down to 1e-49 with full relative
    accuracy (eq. 7 evaluated term by term: the transmitted part must not be formed as 1 - (1 - e))."""
    kap = np.full((1, 8, 12, 10), 8.0, dtype=np.float32)
    S = np.zeros_like(kap)
    t = orc.trace_direction(kap, S, [1, 0.37, 0.81], Ibc=[1.0])
    expect = np.exp(-8.0 * t["chord"])
    inside = t["chord"] > 0
    assert expect[inside].min() < 1e-40
    assert np.allclose(t["exitI"][..., 0][inside], expect[inside], rtol=1e-12, atol=0)


def test_p5_chord_total_is_volume_over_cross_section(orc):
    dims = (10, 12, 8)
    kap, S = rand_fields(dims, 9)
    n = [0.3, -0.8, 0.5]
    t = orc.trace_direction(kap, S, n)
    assert abs(t["chord"].sum() - 10 * 12 * 8 * orc.dir_record(n)["L"]) < 1e-9


# ---------------------------------------------------------------- P8 / P6 / P11: rational brute force
BF_DIMS = (6, 5, 4)
BF_DIRS = [[0.37, 1, 0.81], [1, 0.5, 0.25], [-1, 1, 1], [0.2, -0.3, -1], [1, 0, 0.999999], [0, -1, 0]]


def test_p8_bruteforce_geometry_and_J(orc):
    """Independent algorithm (global event sort + midpoint classification, exact rationals): per-cell
    counts bit-exact, per-cell sum ds, per-ray chord and exit intensity, and J_in to 1e-12."""
    kap, S = rand_fields(BF_DIMS, 21)
    dirs = np.array(BF_DIRS, dtype=np.float64)
    ref = bf.sweep(kap[0], S[0], dirs, Ibc=0.25)
    r = orc.sweep(kap, S, dirs, Ibc=[0.25], count_dirs=range(len(dirs)))
    nx, ny, nz = BF_DIMS
    for i, n in enumerate(dirs):
        cnt = np.zeros((nz, ny, nx), dtype=np.uint32)
        for (x, y, z), c in ref["per_dir"][i]["cnt"].items():
            cnt[z, y, x] = c
        assert np.array_equal(cnt, r["cnt_dirs"][i])
        assert abs(sum(ref["per_dir"][i]["den"].values()) - r["sum_ds"][i]) < 1e-10
        t = orc.trace_direction(kap, S, n, Ibc=[0.25])
        for (p, q), (I, chord) in ref["per_dir"][i]["exits"].items():
            assert abs(t["chord"][q - t["qmin"], p - t["pmin"]] - chord) < 1e-12
            assert abs(t["exitI"][q - t["qmin"], p - t["pmin"], 0] - I) < 1e-12
    Jin = np.zeros((nz, ny, nx))
    for (x, y, z), v in ref["Jin"].items():
        Jin[z, y, x] = v
    assert np.allclose(r["Jin"][0], Jin, rtol=1e-12, atol=1e-15)
    assert r["seg_total"] == sum(ref["cnt"].values())


def test_p6_optically_thin_limit(orc):
    """kappa -> 0 at fixed emissivity eps = kappa S: J_in -> path-length-weighted mean of the linear
    emission integral (no exponentials), computed by the brute-force module with linear=True."""
    kap, S = rand_fields(BF_DIMS, 22)
    kap_thin = (kap.astype(np.float64) * 1e-8).astype(np.float32)
    S_big = (S.astype(np.float64) * 1e8).astype(np.float32)
    dirs = np.array(BF_DIRS[:4], dtype=np.float64)
    ref = bf.sweep(kap_thin[0], S_big[0], dirs, linear=True)
    r = orc.sweep(kap_thin, S_big, dirs)
    nx, ny, nz = BF_DIMS
    Jin = np.zeros((nz, ny, nx))
    for (x, y, z), v in ref["Jin"].items():
        Jin[z, y, x] = v
    assert Jin.max() > 0.1
    assert np.allclose(r["Jin"][0], Jin, rtol=1e-6, atol=1e-12)


def test_p11_optically_thick_limit(orc):
    """Uniform box with kappa dH = 60: every ray reaching an interior cell carries I_in = S, so
    J_in = S (1/N_d) sum_i sum_j (ds_j / L_i) f(kappa ds_j) from the segment lengths alone
    (checks the 1/N_d factor and the ds weighting of eqs. 10-13 together)."""
    dims = (7, 7, 7)
    kap = np.full((1, 7, 7, 7), 60.0, dtype=np.float32)
    S = np.full_like(kap, 0.8)
    dirs = np.array([[0.37, 1, 0.81], [1, 0.5, 0.25], [-1, 0.9, 0.3], [0.2, -0.3, -1]], dtype=np.float64)
    r = orc.sweep(kap, S, dirs)
    centre = (3, 3, 3)
    expect = 0.0
    for n in dirs:
        for (p, q) in bf.lattice(dims, n):
            iv, L = bf.ray_intervals(dims, n, p, q)
            for cell, frac in iv:
                if cell == centre:
                    expect += float(frac) * bf.f_of(60.0 * float(frac) * L)
    expect *= float(S.flat[0]) / len(dirs)
    assert abs(r["Jin"][0, 3, 3, 3] - expect) < 1e-12 * expect


# ---------------------------------------------------------------- P7: mirror / permutation symmetry
def test_p7_mirror_and_permutation(orc):
    dims = (6, 8, 10)
    kap, S = rand_fields(dims, 31)
    dirs = orc.healpix_dirs(2)[::3].copy()
    base = orc.sweep(kap, S, dirs, count_dirs=range(len(dirs)))
    for ax in range(3):                                   # numpy axis of [bin][z][y][x] for coordinate ax
        npax = 3 - ax
        d2 = dirs.copy()
        d2[:, ax] *= -1
        r2 = orc.sweep(np.flip(kap, npax), np.flip(S, npax), d2, count_dirs=range(len(dirs)))
        assert np.array_equal(np.flip(r2["cnt_dirs"], npax), base["cnt_dirs"])
        assert np.allclose(np.flip(r2["Jin"], npax), base["Jin"], rtol=1e-13, atol=1e-16)
    # cyclic permutation x->y->z->x of fields and directions together
    kp = np.ascontiguousarray(np.transpose(kap, (0, 2, 1, 3)))      # new [z'][y'][x'] = old [y][z][x]: swaps y,z
    sp = np.ascontiguousarray(np.transpose(S, (0, 2, 1, 3)))
    r3 = orc.sweep(kp, sp, dirs[:, [0, 2, 1]], count_dirs=range(len(dirs)))
    assert np.array_equal(np.transpose(r3["cnt_sum"], (1, 0, 2)), base["cnt_sum"])
    assert np.allclose(np.transpose(r3["Jin"], (0, 2, 1, 3)), base["Jin"], rtol=1e-12, atol=1e-16)


# ---------------------------------------------------------------- P9: ray groups
def test_p9_four_groups_never_share_a_cell(orc):
    """rays of one of the 4 interleaved groups never traverse the same mesh grid."""
    dims = (8, 6, 10)
    kap, S = rand_fields(dims, 41)
    for n in list(orc.healpix_dirs(2)) + [[1, 1, 1], [1, 0.5, 0.25], [0.999999, 1, 0.000001]]:
        assert orc.trace_direction(kap, S, n, check_groups=True)["conflicts"] == 0


# ---------------------------------------------------------------- P10: worked example
def test_p10_worked_example_golden(orc):
    gold = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    kap = np.zeros((1, 1, 2, 2), np.float32)
    S = np.zeros_like(kap)
    K = [[1.0, 0.5], [2.0, 0.25]]
    Sv = [[1.0, 0.25], [0.5, 2.0]]
    for k in range(2):
        for j in range(2):
            kap[0, 0, j, k] = K[k][j]
            S[0, 0, j, k] = Sv[k][j]
    n = np.array([[1.0, 0.375, 0.0]])
    r = orc.sweep(kap, S, n, count_dirs=[0])
    assert abs(orc.dir_record(n[0])["L"] - gold["L"]) < 1e-15
    assert r["seg_total"] == gold["total_segments"]
    assert abs(r["sum_ds"][0] - gold["sum_ds"]) < 1e-12
    for k in range(2):
        for j in range(2):
            assert r["cnt_dirs"][0, 0, j, k] == gold["count_%d%d" % (k, j)]
            assert abs(r["Jin"][0, 0, j, k] - gold["Jin_%d%d" % (k, j)]) < 1e-12
            assert abs(r["J"][0, 0, j, k] - (gold["Jin_%d%d" % (k, j)] + float(np.float32(Sv[k][j])))) < 1e-12
    t = orc.trace_direction(kap, S, n[0])
    ex = t["exitI"][0 - t["qmin"], :, 0]
    for name, p in (("pm1", -1), ("p0", 0), ("p1", 1)):
        assert abs(ex[p - t["pmin"]] - gold["exit_" + name]) < 1e-12


# ---------------------------------------------------------------- special cases and consistency
def test_kappa_zero_is_well_defined(orc):
    """A7: kappa = 0 cells: f(0) = 1, I unchanged; J_in stays finite."""
    dims = (6, 6, 6)
    kap, S = rand_fields(dims, 51)
    kap[0, 2:4] = 0.0
    r = orc.sweep(kap, S, orc.healpix_dirs(1))
    assert np.all(np.isfinite(r["Jin"])) and r["Jin"].min() >= 0.0


def test_multibin_bins_are_independent(orc):
    """A15 / eq. 22: bins share geometry and do not couple."""
    dims = (6, 5, 7)
    k1, s1 = rand_fields(dims, 61)
    k2, s2 = rand_fields(dims, 62)
    dirs = orc.healpix_dirs(1)
    both = orc.sweep(np.concatenate([k1, k2]), np.concatenate([s1, s2]), dirs, Ibc=[0.1, 0.7])
    a = orc.sweep(k1, s1, dirs, Ibc=[0.1])
    b = orc.sweep(k2, s2, dirs, Ibc=[0.7])
    assert np.allclose(both["Jin"][0], a["Jin"][0], rtol=1e-13) and np.allclose(both["Jin"][1], b["Jin"][0], rtol=1e-13)
    assert not np.allclose(both["Jin"][0], both["Jin"][1], rtol=1e-3)


@pytest.mark.parametrize("dims,nb,Ibc,nside,every", [
    ((12, 10, 9), 1, None, 2, False),
    ((12, 10, 9), 3, [0.4, 0.0, 1.5], 2, False),          # three bins, non-zero inflow
    ((9, 14, 6), 2, [0.25, 2.0], 1, True),                # every cell sampled: all candidate rays shared
    ((16, 5, 11), 3, [1.0, 0.5, 0.0], 2, True),
])
def test_sampled_cells_match_full_sweep(orc, dims, nb, Ibc, nside, every):
    """orc_sweep_cells (used for parity at full benchmark sizes) traces only the rays through the
    sampled cells with the same trace_ray: must reproduce the full sweep there (J_in, J and counts),
    for several bins and non-zero inflow, and when neighbouring samples share their candidate rays
    (axis lines, every cell)."""
    kap, S = rand_fields(dims, 71, nb=nb)
    dirs = np.concatenate([orc.healpix_dirs(nside), np.array([[1, 1, 1], [-1, 0.5, 0.25], [0, 0, -1]], dtype=np.float64)])
    full = orc.sweep(kap, S, dirs, Ibc=Ibc)
    if every:
        cells = np.stack(np.meshgrid(np.arange(dims[0]), np.arange(dims[1]), np.arange(dims[2]), indexing="ij"), -1).reshape(-1, 3)
    else:
        rng = np.random.default_rng(0)
        cells = np.stack([rng.integers(0, dims[0], 20), rng.integers(0, dims[1], 20), rng.integers(0, dims[2], 20)], 1)
        line = np.stack([np.arange(dims[0]), np.full(dims[0], 3), np.full(dims[0], 4)], 1)       # a full axis line
        cells = np.unique(np.concatenate([cells, line, [[0, 0, 0], [dims[0] - 1, dims[1] - 1, dims[2] - 1], [0, dims[1] - 1, 0]]]), axis=0)
    part = orc.sweep_cells(kap, S, dirs, cells, Ibc=Ibc)
    x, y, z = cells[:, 0], cells[:, 1], cells[:, 2]
    assert np.array_equal(part["cnt"], full["cnt_sum"][z, y, x])
    for b in range(nb):
        assert np.abs(part["Jin"][b] - full["Jin"][b, z, y, x]).max() <= 1e-13 * full["Jin"][b].max()
        assert np.all(np.abs(part["Jin"][b] - full["Jin"][b, z, y, x]) <= 1e-12 * full["Jin"][b, z, y, x] + 1e-300)
        assert np.all(np.abs(part["J"][b] - full["J"][b, z, y, x]) <= 1e-12 * full["J"][b, z, y, x])


def test_cell_width_scales_optical_depth(orc):
    """kappa is per unit length: (kappa, dH) and (kappa*dH, 1) give the same J_in."""
    dims = (5, 6, 4)
    kap, S = rand_fields(dims, 81)
    dirs = orc.healpix_dirs(1)
    a = orc.sweep(kap, S, dirs, cell_width=2.0)
    b = orc.sweep((kap * np.float32(2.0)), S, dirs, cell_width=1.0)
    assert np.allclose(a["Jin"], b["Jin"], rtol=1e-12)


# ---------------------------------------------------------------------------------------------
# Rates epilogue (eqs. 14-15, 20-23)
def _quad(f, a, b, n=20001):
    """Composite Simpson on [a, b] (n odd), plain numpy: the independent quadrature of the pins."""
    x = np.linspace(a, b, n)
    y = f(x)
    h = (b - a) / (n - 1)
    return h / 3.0 * (y[0] + y[-1] + 4.0 * y[1:-1:2].sum() + 2.0 * y[2:-1:2].sum())


def test_rates_one_bin_reproduces_eqs_20_21(orc):
    """One bin, S of eq. 18 and J_in flat in the band (eq. 19): the epilogue must give
    eq. 20 / eq. 21, i.e. the local terms  X/n_HI  and  X h dnu / (2 n_HI)  with
    X = delta_alpha n_e n_HII, and the J_in terms 4 pi J int sigma/(h nu) and 4 pi J int (1-nu0/nu) sigma.
    Weights come from numerical quadrature of eqs. 14-15 written out with S_nu(nu) of eq. 18."""
    h_pl, nu0, sig0 = 6.62607015e-27, 3.288e15, 6.3e-18
    dnu = 0.0262 * nu0                                     # k_B T / h at 1e4 K is about 2.08e14 Hz
    sigma = lambda nu: sig0 * (nu / nu0) ** -3.0
    rng = np.random.default_rng(5)
    X = rng.uniform(1e-14, 1e-12, (3, 4, 5))               # delta_alpha n_e n_HII per cell
    nHI = rng.uniform(1e-4, 1e-2, (3, 4, 5))
    Jin = rng.uniform(0.0, 1e-20, (1, 3, 4, 5))
    S_nu = lambda nu, c=1.0: c * h_pl * nu / (4 * math.pi * sigma(nu) * dnu)     # eq. 18 per unit X/n_HI
    S0 = (X / nHI * S_nu(nu0))[None]                       # the bin's stored S: eq. 18 at nu0
    shape = lambda nu: S_nu(nu) / S_nu(nu0)
    wG = 4 * math.pi * _quad(lambda nu: sigma(nu) / (h_pl * nu), nu0, nu0 + dnu)
    wH = 4 * math.pi * _quad(lambda nu: sigma(nu) * (1 - nu0 / nu), nu0, nu0 + dnu)
    lG = 4 * math.pi * _quad(lambda nu: shape(nu) * sigma(nu) / (h_pl * nu), nu0, nu0 + dnu)
    lH = 4 * math.pi * _quad(lambda nu: shape(nu) * sigma(nu) * (1 - nu0 / nu), nu0, nu0 + dnu)
    G, H = orc.rates(Jin, S0, [wG], [lG], [wH], [lH])
    G20 = wG * Jin[0] + X / nHI                                              # eq. 20
    H21 = wH * Jin[0] + X / (2 * nHI) * h_pl * dnu                           # eq. 21
    assert np.abs(G / G20 - 1).max() < 1e-10
    assert np.abs(H / H21 - 1).max() < 1e-10
    # closed forms of the power-law integrals (a dropped factor or a swapped weight fails here)
    assert abs(wG / (4 * math.pi * sig0 * nu0 ** 3 / (3 * h_pl) * (nu0 ** -3 - (nu0 + dnu) ** -3)) - 1) < 1e-10
    assert abs(lG / (4 * math.pi * sig0 * dnu / (h_pl * nu0)) - 1) < 1e-10


def test_rates_bins_are_additive_and_linear(orc):
    """Eq. 22: the spectrum is a sum of rectangular bins, so the rates are a plain sum over bins,
    linear in every weight; with lG = wG, lH = wH they are eq. 14-15 applied to J = J_in + S."""
    rng = np.random.default_rng(6)
    Jin = rng.uniform(0, 1, (3, 2, 3, 4))
    S = rng.uniform(0, 1, (3, 2, 3, 4))
    w = rng.uniform(0.1, 2.0, (4, 3))
    G, H = orc.rates(Jin, S, w[0], w[1], w[2], w[3])
    Gs = sum(orc.rates(Jin[b:b + 1], S[b:b + 1], w[0, b:b + 1], w[1, b:b + 1], w[2, b:b + 1], w[3, b:b + 1])[0] for b in range(3))
    assert np.allclose(G, Gs, rtol=1e-14, atol=0)
    G2, H2 = orc.rates(Jin, S, w[0], w[0], w[2], w[2])
    assert np.allclose(G2, np.tensordot(w[0], Jin + S, axes=(0, 0)), rtol=1e-14)
    assert np.allclose(H2, np.tensordot(w[2], Jin + S, axes=(0, 0)), rtol=1e-14)
    G3, _ = orc.rates(Jin, S, 2 * w[0], w[1], w[2], w[3])
    assert np.allclose(G3 - G, np.tensordot(w[0], Jin, axes=(0, 0)), rtol=1e-12)


# ---------------------------------------------------------------------------------------------
# r > 1 rays per cell width (O3, A13)
@pytest.mark.parametrize("rays", [2, 4])
def test_p12_rays_per_cell_bruteforce_and_closed_forms(orc, rays):
    """Lattice of spacing 1/r: independent exact-rational brute force (counts bit-exact, J_in to 1e-12),
    per cell and direction sum ds = r^2 L (pin P3 with r rays per cell width), hence
    sum ds = volume / per-ray cross-section, and the uniform-medium thick limit is unchanged."""
    dims = (5, 4, 3)
    kap, S = rand_fields(dims, 31)
    dirs = np.array([[0.37, 1, 0.81], [1, 0.5, 0.25], [-1, 1, 1], [0.2, -0.3, -1], [0, -1, 0]], dtype=np.float64)
    ref = bf.sweep(kap[0], S[0], dirs, Ibc=0.25, rays=rays)
    r = orc.sweep(kap, S, dirs, Ibc=[0.25], count_dirs=range(len(dirs)), rays_per_cell=rays)
    nx, ny, nz = dims
    for i, n in enumerate(dirs):
        cnt = np.zeros((nz, ny, nx), dtype=np.uint32)
        for (x, y, z), c in ref["per_dir"][i]["cnt"].items():
            cnt[z, y, x] = c
        assert np.array_equal(cnt, r["cnt_dirs"][i])
        L = orc.dir_record(n)["L"]
        assert abs(r["min_den"][i] / (rays ** 2 * L) - 1) < 1e-12 and abs(r["max_den"][i] / (rays ** 2 * L) - 1) < 1e-12
        assert abs(r["sum_ds"][i] / (nx * ny * nz * rays ** 2 * L) - 1) < 1e-12
    Jin = np.zeros((nz, ny, nx))
    for (x, y, z), v in ref["Jin"].items():
        Jin[z, y, x] = v
    assert np.allclose(r["Jin"][0], Jin, rtol=1e-12, atol=1e-15)
    assert r["seg_total"] == sum(ref["cnt"].values())


def test_p12_rays_per_cell_refines_the_same_quadrature(orc):
    """In a uniform medium J_in of an interior cell is a smooth function of the ray offset, so r = 1, 2, 4
    agree to the quadrature error and differences shrink with r; r is rejected unless a power of two."""
    kap = np.full((1, 12, 12, 12), 0.3, dtype=np.float32)
    S = np.ones_like(kap)
    dirs = orc.healpix_dirs(1)
    J = [orc.sweep(kap, S, dirs, rays_per_cell=r, want_counts=False)["Jin"][0, 6, 6, 6] for r in (1, 2, 4, 8)]
    assert abs(J[1] - J[3]) < abs(J[0] - J[3]) and abs(J[2] - J[3]) < abs(J[1] - J[3])
    assert abs(J[0] / J[3] - 1) < 0.05 and abs(J[2] / J[3] - 1) < 2e-3
    with pytest.raises(RuntimeError):
        orc.sweep(kap, S, dirs, rays_per_cell=3)


# ---------------------------------------------------------------------------------------------
# per-face inflow (A10)
def test_p13_per_face_inflow_bruteforce_and_vacuum(orc):
    """Inflow per entry face: (i) against the brute force, which finds the entry face from the exact
    entry point (the boundary plane it lies on); (ii) in vacuum (kappa = 0, S = 0) every ray keeps its
    inflow, so for one axis-aligned direction J_in is the inflow of the single upwind face everywhere;
    (iii) six equal faces = the uniform inflow."""
    dims = (5, 4, 3)
    kap, S = rand_fields(dims, 41)
    dirs = np.array([[0.37, 1, 0.81], [1, 0.5, 0.25], [-1, 1, 1], [0.2, -0.3, -1], [0, -1, 0], [-1, -0.999999, 0.5]], dtype=np.float64)
    faces = [0.1, 0.9, 0.3, 0.7, 0.5, 0.2]
    ref = bf.sweep(kap[0], S[0], [list(d) for d in dirs], Ibc_faces=faces)
    r = orc.sweep(kap, S, dirs, Ibc_faces=[faces])
    nx, ny, nz = dims
    Jin = np.zeros((nz, ny, nx))
    for (x, y, z), v in ref["Jin"].items():
        Jin[z, y, x] = v
    assert np.allclose(r["Jin"][0], Jin, rtol=1e-12, atol=1e-15)
    vac = np.zeros((1, 3, 4, 5), dtype=np.float32)
    for ax in range(3):
        for sgn in (1, -1):
            n = np.zeros((1, 3))
            n[0, ax] = sgn
            J = orc.sweep(vac, vac, n, Ibc_faces=[faces])["Jin"]
            assert np.allclose(J, faces[2 * ax + (1 if sgn < 0 else 0)], rtol=1e-14)
    a = orc.sweep(kap, S, dirs, Ibc=[0.6])["Jin"]
    b = orc.sweep(kap, S, dirs, Ibc_faces=[[0.6] * 6])["Jin"]
    assert np.allclose(a, b, rtol=1e-14, atol=0)            # (thread reduction order differs between runs)


def test_golden_count_hashes_are_the_oracles(orc):
    """tests/golden/segment_totals.txt (totals + SHA-256 of the direction-summed per-cell counts, the every-cell integer
    gate of the full-size GPU tests) is what oracle/ computes: re-derived here for the two configs that take seconds."""
    import hashlib
    from rt_inputs import CONFIGS
    rows = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "segment_totals.txt")):
        w = line.split()
        if w and not line.startswith("#"):
            rows[w[0]] = (int(w[1]), w[4])
    assert sorted(rows) == ["C1", "C2", "C3", "C4", "C5"] and all(len(v[1]) == 64 for v in rows.values())
    for name in ("C1", "C2"):
        spec = CONFIGS[name]
        nx, ny, nz = spec.dims
        r = orc.sweep(np.ones((1, nz, ny, nx), np.float32), np.zeros((1, nz, ny, nx), np.float32), orc.healpix_dirs(spec.nside))
        sha = hashlib.sha256(np.ascontiguousarray(r["cnt_sum"], dtype="<u4").tobytes()).hexdigest()
        assert (r["seg_total"], sha) == rows[name]
