"""Point radiation sources (Appendix 1): pins of the oracle (CPU) and parity of the CUDA
path against it (GPU)."""
import math
from fractions import Fraction

import numpy as np
import pytest

FIX = 256


def brute_ray(dims, kap, src_fix, tgt):
    """Independent algorithm: all plane crossings of the line source -> cell centre (and beyond) as exact
    rationals, sorted globally; every interval is classified by the cell its midpoint lies in.
    Returns (tau up to the target cell, r_in, r_out) with lengths in cell widths."""
    s = [Fraction(int(v), FIX) for v in src_fix]
    c = [Fraction(2 * t + 1, 2) for t in tgt]
    d = [ci - si for ci, si in zip(c, s)]
    ln = math.sqrt(float(sum(x * x for x in d)))
    if all(x == 0 for x in d):
        return 0.0, 0.0, 0.5
    ev = {Fraction(0)}
    for i in range(3):
        if d[i] != 0:
            for plane in range(0, dims[i] + 1):
                u = (Fraction(plane) - s[i]) / d[i]
                if u > 0:
                    ev.add(u)
    ev = sorted(ev)
    tau, r_in, r_out = 0.0, None, None
    for u0, u1 in zip(ev[:-1], ev[1:]):
        mid = (u0 + u1) / 2
        cell = tuple(math.floor(s[i] + d[i] * mid) for i in range(3))
        if cell == tuple(tgt):
            if r_in is None:
                r_in = float(u0) * ln
            r_out = float(u1) * ln
        elif r_in is None:
            if all(0 <= cell[i] < dims[i] for i in range(3)):
                tau += float(kap[cell[2], cell[1], cell[0]]) * float(u1 - u0) * ln
        else:
            break
    return tau, r_in, r_out


SOURCES = [[0, 0, 0], [5 * FIX, 4 * FIX, 3 * FIX], [2 * FIX + 128, 1 * FIX + 128, 1 * FIX + 128], [3 * FIX, 2 * FIX + 128, 77],
           [1 * FIX + 10, 3 * FIX + 200, 2 * FIX + 31], [0, 2 * FIX, 3 * FIX]]


def test_ps1_bruteforce_tau_and_radii(orc):
    """tau, r_in, r_out of every (source, cell) pair against the global event sort with exact rationals;
    sources at a box corner, the opposite corner, a cell centre, on a face, generic, on an edge."""
    dims = (5, 4, 3)
    rng = np.random.default_rng(51)
    kap = rng.uniform(0.05, 2.0, (1, 3, 4, 5)).astype(np.float32)
    for si, src in enumerate(SOURCES):
        r = orc.point_sources(kap, SOURCES, np.ones((len(SOURCES), 1)), diag=(si, 0))
        for z in range(3):
            for y in range(4):
                for x in range(5):
                    tau, r_in, r_out = brute_ray(dims, kap[0], src, (x, y, z))
                    assert abs(r["tau"][z, y, x] - tau) <= 1e-12 * max(1.0, tau)
                    assert abs(r["r_in"][z, y, x] - r_in) <= 1e-12 and abs(r["r_out"][z, y, x] - r_out) <= 1e-12
                    assert abs(r["dtau"][z, y, x] - float(kap[0, z, y, x]) * (r_out - r_in)) <= 1e-12


def test_ps2_uniform_medium_closed_forms(orc):
    """Uniform kappa: tau = kappa r_in exactly (eq. 4's optical depth of a straight path), and Q of a single
    source is L e^{-kappa r_in} (1 - e^{-kappa (r_out - r_in)}) / (4 pi/3 (r_out^3 - r_in^3)) (eqs. A1-A3);
    sources add linearly; cell_width scales lengths."""
    kap = np.full((2, 6, 7, 8), 0.3, dtype=np.float32)
    kap[1] = 1.7
    src = [[0, 0, 0], [8 * FIX, 3 * FIX + 128, 100]]
    lum = np.array([[2.0, 0.5], [1.0, 3.0]])
    for cw in (1.0, 0.4):
        ra = orc.point_sources(kap, src[:1], lum[:1], cell_width=cw)
        rb = orc.point_sources(kap, src[1:], lum[1:], cell_width=cw)
        rab = orc.point_sources(kap, src, lum, cell_width=cw, diag=(0, 1))
        assert np.allclose(rab["Q"], ra["Q"] + rb["Q"], rtol=1e-13)
        k1 = float(kap[1, 0, 0, 0])
        assert np.allclose(rab["tau"], k1 * rab["r_in"], rtol=1e-12, atol=1e-14)
        for b in range(2):
            k = float(kap[b, 0, 0, 0])
            q = lum[0, b] * np.exp(-k * ra["r_in"]) * (1 - np.exp(-k * (ra["r_out"] - ra["r_in"]))) / \
                (4 * math.pi / 3 * (ra["r_out"] ** 3 - ra["r_in"] ** 3))
            assert np.allclose(ra["Q"][b], q, rtol=1e-12)
    # geometry: the ray to a cell centre passes the centre between r_in and r_out, at distance |c - s|
    r = orc.point_sources(kap, src[:1], lum[:1])
    z, y, x = np.meshgrid(np.arange(6), np.arange(7), np.arange(8), indexing="ij")
    dist = np.sqrt((x + 0.5) ** 2 + (y + 0.5) ** 2 + (z + 0.5) ** 2)
    assert np.all(r["r_in"] < dist) and np.all(dist < r["r_out"])


def test_ps3_thin_limit_is_the_inverse_square_law(orc):
    """kappa -> 0: Q / kappa -> L / (4 pi/3 (r_out^2 + r_out r_in + r_in^2)), i.e. L / (4 pi r^2) (eq. 4) to
    O((dr/r)^2) far from the source."""
    kap = np.full((1, 16, 16, 16), 1e-9, dtype=np.float32)
    r = orc.point_sources(kap, [[0, 0, 0]], [[5.0]])
    k = float(kap[0, 0, 0, 0])
    exact = 5.0 / (4 * math.pi / 3 * (r["r_out"] ** 2 + r["r_out"] * r["r_in"] + r["r_in"] ** 2))
    assert np.allclose(r["Q"][0] / k, exact, rtol=1e-7)
    z, y, x = np.meshgrid(np.arange(16), np.arange(16), np.arange(16), indexing="ij")
    d2 = (x + 0.5) ** 2 + (y + 0.5) ** 2 + (z + 0.5) ** 2
    far = d2 > 100
    assert np.abs(r["Q"][0][far] / k / (5.0 / (4 * math.pi * d2[far])) - 1).max() < 0.02


def test_ps4_mirror_symmetry(orc):
    """Mirroring the field and the source along an axis mirrors Q."""
    rng = np.random.default_rng(52)
    kap = rng.uniform(0.05, 1.0, (1, 4, 5, 6)).astype(np.float32)
    src = np.array([[1 * FIX + 40, 2 * FIX, 3 * FIX + 128]])
    q = orc.point_sources(kap, src, [[1.0]], want_diag=False)["Q"]
    dims = (6, 5, 4)
    for ax in range(3):
        km = np.ascontiguousarray(np.flip(kap, axis=3 - ax))
        sm = src.copy()
        sm[0, ax] = dims[ax] * FIX - src[0, ax]
        qm = orc.point_sources(km, sm, [[1.0]], want_diag=False)["Q"]
        assert np.allclose(np.flip(qm, axis=3 - ax), q, rtol=1e-12)


def _species_case(rng, shape, nb, ns):
    """Seeded per-species cross sections and densities: kappa_i,b = n_i sigma_i,b, kappa_b = sum_i kappa_i,b."""
    n_sp = rng.uniform(0.1, 2.0, (ns,) + shape)
    sigma = rng.uniform(0.05, 0.6, (ns, nb))
    kappa_sp = n_sp[:, None] * sigma.reshape(ns, nb, *([1] * len(shape)))
    return n_sp, sigma, kappa_sp, kappa_sp.sum(axis=0)


def test_ps5_species_split_conserves_photons(orc):
    """A4 summed over the species is A3: with every threshold below every bin, sum_i n_i Gamma_i = sum_b Q_b / (h nu_b)
    (each absorbed photon ionises exactly one particle), and sum_i n_i Heat_i = sum_b sum_i share_i Q_b (1 - h nu_i / h nu_b)."""
    rng = np.random.default_rng(71)
    nb, ns, shape = 3, 3, (4, 5, 6)
    n_sp, sigma, kappa_sp, kappa = _species_case(rng, shape, nb, ns)
    Q = rng.uniform(0.0, 3.0, (nb,) + shape)
    hnu = np.array([1.0, 1.7, 3.2])
    thr = np.array([0.5, 0.8, 1.0])
    G, H = orc.point_source_rates(Q, kappa, kappa_sp, n_sp, hnu, thr)
    photons = sum(Q[b] / hnu[b] for b in range(nb))
    assert np.allclose((n_sp * G).sum(axis=0), photons, rtol=1e-13)
    heat = sum(kappa_sp[i, b] / kappa[b] * Q[b] * (1.0 - thr[i] / hnu[b]) for i in range(ns) for b in range(nb))
    assert np.allclose((n_sp * H).sum(axis=0), heat, rtol=1e-13)


def test_ps5_single_species_and_thresholds(orc):
    """One species carrying all the opacity: Gamma = sum_b Q_b / (n h nu_b) (A5 from A3).  A bin below a species'
    threshold contributes nothing to that species (the integrals of A5-A6 start at nu_i); n_i = 0 gives 0."""
    rng = np.random.default_rng(72)
    shape = (3, 4, 5)
    n = rng.uniform(0.5, 2.0, (1,) + shape)
    kap = rng.uniform(0.1, 1.0, (2,) + shape)
    Q = rng.uniform(0.0, 2.0, (2,) + shape)
    hnu = np.array([1.2, 2.5])
    G, H = orc.point_source_rates(Q, kap, kap[None], n, hnu, [1.0])
    assert np.allclose(G[0], (Q[0] / 1.2 + Q[1] / 2.5) / n[0], rtol=1e-14)
    assert np.allclose(H[0], (Q[0] * (0.2 / 1.2) + Q[1] * (1.5 / 2.5)) / n[0], rtol=1e-13)
    G2, H2 = orc.point_source_rates(Q, kap, kap[None], n, hnu, [2.0])          # bin 0 lies below the threshold
    assert np.allclose(G2[0], Q[1] / 2.5 / n[0], rtol=1e-14) and np.allclose(H2[0], Q[1] * (0.5 / 2.5) / n[0], rtol=1e-13)
    n0 = n.copy()
    n0[0, 0, 0, 0] = 0.0
    G3, H3 = orc.point_source_rates(Q, kap, kap[None], n0, hnu, [1.0])
    assert G3[0, 0, 0, 0] == 0.0 and H3[0, 0, 0, 0] == 0.0 and np.array_equal(G3[0].ravel()[1:], G[0].ravel()[1:])


def test_ps5_thin_limit_is_eqs_5_and_6(orc):
    """kappa -> 0: the photon-conserving rates reduce to eqs. 5-6 with the flux of eq. 4, bin by bin:
    Gamma_i -> sum_b L_b sigma_i,b / (4 pi r^2 h nu_b), Heat_i -> sum_b L_b sigma_i,b (h nu_b - h nu_i) / (4 pi r^2 h nu_b),
    with 1 / r^2 -> 3 / (r_out^2 + r_out r_in + r_in^2) for a shell of finite width (pin PS3)."""
    rng = np.random.default_rng(73)
    nb, ns, shape = 2, 2, (8, 8, 8)
    n_sp = rng.uniform(0.5, 2.0, (ns,) + shape) * 1e-9
    sigma = np.array([[0.3, 0.1], [0.0, 0.5]])                  # species 1 does not absorb in bin 0
    kappa_sp = n_sp[:, None] * sigma.reshape(ns, nb, 1, 1, 1)
    kappa = kappa_sp.sum(axis=0).astype(np.float32)             # the oracle's traversal takes fp32 kappa
    kappa_sp = kappa_sp * (kappa.astype(np.float64) / kappa_sp.sum(axis=0))[None]   # shares consistent with the rounded total
    lum = np.array([[4.0, 1.5]])
    hnu, thr = np.array([1.0, 2.0]), np.array([0.9, 1.6])
    r = orc.point_sources(kappa, [[0, 0, 0]], lum)
    G, H = orc.point_source_rates(r["Q"], kappa, kappa_sp, n_sp, hnu, thr)
    geom = 1.0 / (4 * math.pi / 3 * (r["r_out"] ** 2 + r["r_out"] * r["r_in"] + r["r_in"] ** 2))
    for i in range(ns):
        g = sum(lum[0, b] * sigma[i, b] / hnu[b] for b in range(nb) if hnu[b] >= thr[i]) * geom
        h = sum(lum[0, b] * sigma[i, b] * (hnu[b] - thr[i]) / hnu[b] for b in range(nb) if hnu[b] >= thr[i]) * geom
        assert np.allclose(G[i], g, rtol=1e-6) and np.allclose(H[i], h, rtol=1e-6)


# ---------------------------------------------------------------------------------------------
# CUDA path against the oracle
PS_TOL = 1e-5          # relative, with the A14 floor: fp32 output of fp64 path sums over fp32 kappa


def _ps_rel(got, ref):
    ref = np.asarray(ref, dtype=np.float64)
    floor = max(1e-30 * np.abs(ref).max(), 1e-300)
    return np.abs(np.asarray(got, dtype=np.float64) - ref) / np.maximum(np.abs(ref), floor)


@pytest.mark.gpu
@pytest.mark.parametrize("dims,nb,cw", [((5, 4, 3), 1, 1.0), ((33, 20, 17), 2, 0.7), ((64, 64, 64), 1, 1.0), ((100, 30, 12), 3, 1.0)])
def test_point_sources_parity(orc, dims, nb, cw):
    """rt_point_sources against the oracle: step count bit-exact (integer traversal data), tau and Q within
    1e-5 on every cell; sources on corners, faces, edges, cell centres and generic positions."""
    import torch
    import paper_1410_0763_b200 as rt
    assert torch.cuda.is_available()
    nx, ny, nz = dims
    rng = np.random.default_rng(61)
    kap = rng.uniform(0.02, 0.6, (nb, nz, ny, nx)).astype(np.float32)
    kap[:, nz // 2:, : ny // 2, :] *= 8.0                      # an opaque block: exp(-tau) spans many decades
    S = np.zeros_like(kap)
    src = np.array([[0, 0, 0], [nx * FIX, ny * FIX, nz * FIX], [(nx // 2) * FIX + 128, (ny // 2) * FIX + 128, (nz // 2) * FIX + 128],
                    [nx * FIX // 3, 0, nz * FIX // 2], [17, ny * FIX - 1, 3], [(nx // 2) * FIX, (ny // 2) * FIX, 77]], dtype=np.int32)
    lum = rng.uniform(0.5, 2.0, (len(src), nb))
    tr = rt.RayTracer(dims, nb, rt.healpix_dirs(1), cell_width=cw)
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        for diag in [(0, 0), (len(src) - 1, nb - 1), (2, 0)]:
            Q, tau, steps = tr.point_sources(src, lum, diag=diag, want_steps=True)
            ref = orc.point_sources(kap, src, lum, cell_width=cw, diag=diag)
            assert steps == ref["steps"]
            assert _ps_rel(tau.cpu().numpy(), ref["tau"]).max() <= PS_TOL
            assert _ps_rel(Q.cpu().numpy(), ref["Q"]).max() <= PS_TOL
        with pytest.raises(rt.RtError):
            tr.point_sources([[nx * FIX + 1, 0, 0]], np.ones((1, nb)))
    finally:
        tr.close()


@pytest.mark.gpu
def test_point_sources_two_streams():
    """rt_point_sources is asynchronous on the caller's stream, whichever stream that is: calls that alternate between two
    streams and between two source tables, with no host synchronisation in between, each give the result of their own
    tables (the device copy of the tables is shared by all calls of a context: a call with the same tables on another
    stream has to wait for the copy, a call with new tables for the kernels that still read the old ones)."""
    import torch
    import paper_1410_0763_b200 as rt
    dims, nb = (96, 96, 96), 1
    nx, ny, nz = dims
    rng = np.random.default_rng(62)
    kap = torch.from_numpy(rng.uniform(0.02, 0.6, (nb, nz, ny, nx)).astype(np.float32)).cuda()
    tables = []
    for t in range(2):
        src = np.stack([rng.integers(0, nx * FIX + 1, 12), rng.integers(0, ny * FIX + 1, 12), rng.integers(0, nz * FIX + 1, 12)], axis=1).astype(np.int32)
        tables.append((src, rng.uniform(0.5, 2.0, (12, nb))))
    tr = rt.RayTracer(dims, nb, rt.healpix_dirs(1))
    try:
        tr.set_fields(kap, torch.zeros_like(kap))
        ref = []
        for src, lum in tables:                                  # one stream, synchronised: the reference
            Q = torch.empty_like(kap)
            rt.rt_point_sources(tr.h, src, lum, Q, tr.numel, nb)
            torch.cuda.synchronize()
            ref.append(Q.clone())
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        order = [(0, 0), (1, 0), (0, 1), (1, 1), (1, 0), (0, 0), (1, 1), (0, 1), (0, 0), (1, 1)]      # (stream, table)
        outs = [torch.full_like(kap, -1.0) for _ in order]
        torch.cuda.synchronize()
        for (si, ti), Q in zip(order, outs):
            rt.rt_point_sources(tr.h, tables[ti][0], tables[ti][1], Q, tr.numel, nb, stream=streams[si])
        torch.cuda.synchronize()
        for (si, ti), Q in zip(order, outs):
            assert torch.equal(Q, ref[ti]), "call on stream %d with table %d" % (si, ti)
    finally:
        tr.close()


@pytest.mark.gpu
def test_point_sources_c3_sampled(orc):
    """128^3 (config C3's mesh and kappa), 4 sources: full oracle comparison (the oracle takes seconds)."""
    import torch
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields
    kap, S = make_fields("C3")
    src = np.array([[0, 0, 0], [64 * FIX + 128, 64 * FIX + 128, 64 * FIX + 128], [128 * FIX, 40 * FIX, 77], [10 * FIX + 5, 100 * FIX + 200, 50 * FIX]], dtype=np.int32)
    lum = np.array([[1.0], [2.0], [0.5], [1.5]])
    tr = rt.RayTracer((128, 128, 128), 1, rt.healpix_dirs(1))
    try:
        tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
        Q, tau, steps = tr.point_sources(src, lum, diag=(1, 0), want_steps=True)
        ref = orc.point_sources(kap, src, lum, diag=(1, 0))
    finally:
        tr.close()
    assert steps == ref["steps"]
    assert _ps_rel(tau.cpu().numpy(), ref["tau"]).max() <= PS_TOL
    assert _ps_rel(Q.cpu().numpy(), ref["Q"]).max() <= PS_TOL


@pytest.mark.gpu
@pytest.mark.parametrize("dims,nb,ns,binpack", [((33, 20, 17), 2, 3, 0), ((64, 40, 12), 3, 2, 0), ((64, 40, 12), 3, 8, 1), ((5, 4, 3), 1, 1, 0)])
def test_point_source_rates_parity(orc, dims, nb, ns, binpack):
    """rt_point_source_rates (eqs. A4-A6) against the oracle's per-species split of the oracle's own Q, on every cell;
    thresholds that cut bins off, a species with zero density somewhere, bins as planes and packed rows."""
    import torch
    import paper_1410_0763_b200 as rt
    nx, ny, nz = dims
    rng = np.random.default_rng(81)
    n_sp, sigma, kappa_sp, kappa = _species_case(rng, (nz, ny, nx), nb, ns)
    n_sp[0, 0, 0, : nx // 2] = 0.0
    kappa_sp = n_sp[:, None] * sigma.reshape(ns, nb, 1, 1, 1)
    kap32 = kappa_sp.sum(axis=0).astype(np.float32)
    ksp32, n32 = kappa_sp.astype(np.float32), n_sp.astype(np.float32)
    hnu = np.linspace(1.0, 3.0, nb) if nb > 1 else np.array([1.3])
    thr = np.linspace(0.8, 2.2, ns)
    src = np.array([[0, 0, 0], [(nx // 2) * FIX + 128, (ny // 2) * FIX + 128, (nz // 2) * FIX + 128]], dtype=np.int32)
    lum = rng.uniform(0.5, 2.0, (2, nb))
    tr = rt.RayTracer(dims, nb, rt.healpix_dirs(1), tune={"binpack": binpack})
    try:
        tr.set_fields(torch.from_numpy(kap32).cuda(), torch.zeros(kap32.shape, device="cuda"))
        Q, _, _ = tr.point_sources(src, lum)
        G, H = tr.point_source_rates(Q, torch.from_numpy(ksp32).cuda(), torch.from_numpy(n32).cuda(), hnu, thr)
        with pytest.raises(rt.RtError):
            tr.point_source_rates(Q, torch.from_numpy(ksp32).cuda(), torch.from_numpy(n32).cuda(), -hnu, thr)
    finally:
        tr.close()
    ref = orc.point_sources(kap32, src, lum, want_diag=False)
    Gr, Hr = orc.point_source_rates(ref["Q"], kap32, ksp32, n32, hnu, thr)
    assert _ps_rel(G.cpu().numpy(), Gr).max() <= PS_TOL
    assert _ps_rel(H.cpu().numpy(), Hr).max() <= PS_TOL
    assert np.all(G.cpu().numpy()[0, 0, 0, : nx // 2] == 0.0)
