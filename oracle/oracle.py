"""ctypes wrapper around oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It builds oracle/liboracle.so with gcc on first use (plain C, -O2,
OpenMP over directions) and exposes the oracle's entry points with numpy host arrays.
Nothing here touches CUDA or the paper_1410_0763_b200 package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so (idempotent)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp%d" % os.getpid()
            cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-std=c11", "-Wall", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, fp, ip = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
        up, i64p = C.POINTER(C.c_uint32), C.POINTER(C.c_int64)
        L.orc_healpix_dirs.argtypes = [C.c_int, dp]
        L.orc_healpix_dirs.restype = C.c_int
        L.orc_dir_record.argtypes = [dp, ip, ip, i64p, i64p, dp]
        L.orc_dir_record.restype = C.c_int
        L.orc_sweep.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, fp, dp, C.c_int, dp, C.c_double,
                                dp, dp, dp, C.POINTER(C.c_ulonglong), up, ip, C.c_int, up, dp, dp, C.c_int]
        L.orc_sweep.restype = C.c_int
        L.orc_sweep_rays.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, fp, dp, C.c_int, dp, C.c_double, C.c_int,
                                     dp, dp, dp, C.POINTER(C.c_ulonglong), up, ip, C.c_int, up, dp, dp, C.c_int]
        L.orc_sweep_rays.restype = C.c_int
        L.orc_sweep_faces.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, fp, dp, C.c_int, dp, dp, C.c_double, C.c_int,
                                      dp, dp, dp, C.POINTER(C.c_ulonglong), up, ip, C.c_int, up, dp, dp, C.c_int]
        L.orc_sweep_faces.restype = C.c_int
        L.orc_trace_direction.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, fp, dp, dp, C.c_double,
                                          ip, dp, dp, C.POINTER(C.c_long)]
        L.orc_trace_direction.restype = C.c_int
        L.orc_sweep_cells.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, fp, dp, C.c_int, dp, C.c_double,
                                      ip, C.c_int, dp, dp, up, C.c_int]
        L.orc_sweep_cells.restype = C.c_int
        L.orc_point_sources.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, fp, C.c_int, ip, dp, C.c_double, dp, C.c_int, C.c_int,
                                        dp, dp, dp, dp, C.POINTER(C.c_ulonglong), C.c_int]
        L.orc_point_sources.restype = C.c_int
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _fields(kappa, S):
    kappa = np.ascontiguousarray(kappa, dtype=np.float32)
    S = np.ascontiguousarray(S, dtype=np.float32)
    if kappa.ndim == 3:
        kappa, S = kappa[None], S[None]
    assert kappa.ndim == 4 and kappa.shape == S.shape, "fields must be [nbins][nz][ny][nx]"
    return kappa, S


def healpix_dirs(nside: int) -> np.ndarray:
    """HEALPix RING-order pixel centres, [12 nside^2][3] fp64 (oracle.c orc_healpix_dirs)."""
    out = np.empty((12 * nside * nside, 3), dtype=np.float64)
    n = lib().orc_healpix_dirs(nside, _p(out, C.c_double))
    assert n == out.shape[0]
    return out


def dir_record(n) -> dict:
    """Dominant axis, reflections, quantised slopes and slab length of one direction (O2)."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    a = C.c_int()
    refl = (C.c_int * 3)()
    Mb, Mc, L = C.c_int64(), C.c_int64(), C.c_double()
    rc = lib().orc_dir_record(_p(n, C.c_double), C.byref(a), refl, C.byref(Mb), C.byref(Mc), C.byref(L))
    if rc != 0:
        raise ValueError("zero direction vector")
    return {"a": a.value, "refl": tuple(refl), "Mb": Mb.value, "Mc": Mc.value, "L": L.value}


def sweep(kappa, S, dirs, Ibc=None, cell_width: float = 1.0, count_dirs=(), nthreads: int = 0,
          want_counts: bool = True, rays_per_cell: int = 1, Ibc_faces=None) -> dict:
    """Full sweep.  Returns dict(Jin, J, sum_ds, seg_total, cnt_sum, cnt_dirs, min_den, max_den).
    rays_per_cell = r: ray spacing = cell width / r in both transverse axes (O3, A13; a power of two).
    Ibc_faces [nbins][6]: inflow per bin and entry face (-x, +x, -y, +y, -z, +z), overrides Ibc (A10)."""
    kappa, S = _fields(kappa, S)
    nb, nz, ny, nx = kappa.shape
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    nd = dirs.shape[0]
    Jin = np.empty(kappa.shape, dtype=np.float64)
    J = np.empty(kappa.shape, dtype=np.float64)
    sum_ds = np.empty(nd, dtype=np.float64)
    min_den = np.empty(nd, dtype=np.float64)
    max_den = np.empty(nd, dtype=np.float64)
    seg = C.c_ulonglong(0)
    cnt_sum = np.empty((nz, ny, nx), dtype=np.uint32) if want_counts else None
    cd = np.ascontiguousarray(list(count_dirs), dtype=np.int32)
    cnt_out = np.zeros((len(cd), nz, ny, nx), dtype=np.uint32) if len(cd) else None
    ibc = None if Ibc is None else np.ascontiguousarray(Ibc, dtype=np.float64)
    ibc6 = None if Ibc_faces is None else np.ascontiguousarray(Ibc_faces, dtype=np.float64).reshape(nb, 6)
    rc = lib().orc_sweep_faces(nx, ny, nz, nb, _p(kappa, C.c_float), _p(S, C.c_float), _p(dirs, C.c_double), nd,
                         _p(ibc, C.c_double), _p(ibc6, C.c_double), float(cell_width), int(rays_per_cell), _p(Jin, C.c_double), _p(J, C.c_double),
                         _p(sum_ds, C.c_double), C.byref(seg), _p(cnt_sum, C.c_uint32),
                         _p(cd, C.c_int) if len(cd) else None, len(cd), _p(cnt_out, C.c_uint32),
                         _p(min_den, C.c_double), _p(max_den, C.c_double), int(nthreads))
    if rc != 0:
        raise RuntimeError("orc_sweep failed: %d" % rc)
    return {"Jin": Jin, "J": J, "sum_ds": sum_ds, "seg_total": int(seg.value), "cnt_sum": cnt_sum,
            "cnt_dirs": cnt_out, "min_den": min_den, "max_den": max_den}


def trace_direction(kappa, S, n, Ibc=None, cell_width: float = 1.0, check_groups: bool = False) -> dict:
    """One direction: per-ray exit intensity and in-box chord over the whole launch lattice (+ P9 check)."""
    kappa, S = _fields(kappa, S)
    nb, nz, ny, nx = kappa.shape
    n = np.ascontiguousarray(n, dtype=np.float64)
    lat = (C.c_int * 4)()
    ibc = None if Ibc is None else np.ascontiguousarray(Ibc, dtype=np.float64)
    L = lib()
    args = [nx, ny, nz, nb, _p(kappa, C.c_float), _p(S, C.c_float), _p(n, C.c_double), _p(ibc, C.c_double),
            float(cell_width), lat]
    rc = L.orc_trace_direction(*args, None, None, None)
    assert rc == 0
    pmin, qmin, np_, nq = lat
    exitI = np.zeros((nq, np_, nb), dtype=np.float64)
    chord = np.zeros((nq, np_), dtype=np.float64)
    conf = C.c_long(0)
    rc = L.orc_trace_direction(*args, _p(exitI, C.c_double), _p(chord, C.c_double),
                               C.byref(conf) if check_groups else None)
    if rc != 0:
        raise RuntimeError("orc_trace_direction failed: %d" % rc)
    return {"pmin": pmin, "qmin": qmin, "exitI": exitI, "chord": chord, "conflicts": int(conf.value)}


def sweep_cells(kappa, S, dirs, cells, Ibc=None, cell_width: float = 1.0, nthreads: int = 0) -> dict:
    """J_in / J at sampled cells (x,y,z), tracing only the rays that touch them."""
    kappa, S = _fields(kappa, S)
    nb, nz, ny, nx = kappa.shape
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    cells = np.ascontiguousarray(cells, dtype=np.int32).reshape(-1, 3)
    nc = cells.shape[0]
    Jin = np.empty((nb, nc), dtype=np.float64)
    J = np.empty((nb, nc), dtype=np.float64)
    cnt = np.empty(nc, dtype=np.uint32)
    ibc = None if Ibc is None else np.ascontiguousarray(Ibc, dtype=np.float64)
    rc = lib().orc_sweep_cells(nx, ny, nz, nb, _p(kappa, C.c_float), _p(S, C.c_float), _p(dirs, C.c_double),
                               dirs.shape[0], _p(ibc, C.c_double), float(cell_width), _p(cells, C.c_int), nc,
                               _p(Jin, C.c_double), _p(J, C.c_double), _p(cnt, C.c_uint32), int(nthreads))
    if rc != 0:
        raise RuntimeError("orc_sweep_cells failed: %d" % rc)
    return {"Jin": Jin, "J": J, "cnt": cnt}


def rates(Jin, S, wG, lG, wH, lH):
    """Rates epilogue, fp64 (eqs. 14-15 with the rectangular bins of eqs. 22-23,
    PAPER.md:163-175): per cell  Gamma = sum_b wG[b] Jin[b] + lG[b] S[b],  Heat = sum_b wH[b] Jin[b] + lH[b] S[b].
    wG, wH integrate a J_in that is flat inside the bin (eq. 19); lG, lH carry the shape of S_nu inside the
    bin, so that with one bin and S of eq. 18 the second terms are those of eqs. 20-21.
    Pinned by tests/test_oracle_pins.py::test_rates_* against numerical quadrature of eqs. 14-15."""
    Jin = np.asarray(Jin, dtype=np.float64)
    S = np.asarray(S, dtype=np.float64)
    if Jin.ndim == 3:
        Jin, S = Jin[None], S[None]
    G = np.zeros(Jin.shape[1:], dtype=np.float64)
    H = np.zeros(Jin.shape[1:], dtype=np.float64)
    for b in range(Jin.shape[0]):
        G += float(wG[b]) * Jin[b] + float(lG[b]) * S[b]
        H += float(wH[b]) * Jin[b] + float(lH[b]) * S[b]
    return G, H


PS_FIX = 256        # source positions are given in units of 1/256 cell (exact integer traversal)


def point_sources(kappa, src_fix, lum, cell_width: float = 1.0, diag=(0, 0), want_diag: bool = True, nthreads: int = 0) -> dict:
    """Point radiation sources (PAPER.md:64-82 and Appendix 1): photon-conserving absorption rate per unit
    shell volume Q [nbins][nz][ny][nx], and for source/bin `diag` the optical depth tau up to the target
    cell, dtau across it and the radii r_in, r_out of Appendix 1.  src_fix: int [nsrc][3] in 1/256 cells."""
    kappa = np.ascontiguousarray(kappa, dtype=np.float32)
    if kappa.ndim == 3:
        kappa = kappa[None]
    nb, nz, ny, nx = kappa.shape
    src = np.ascontiguousarray(src_fix, dtype=np.int32).reshape(-1, 3)
    lum = np.ascontiguousarray(lum, dtype=np.float64).reshape(src.shape[0], nb)
    Q = np.empty(kappa.shape, dtype=np.float64)
    d = [np.empty((nz, ny, nx), dtype=np.float64) if want_diag else None for _ in range(4)]
    steps = C.c_ulonglong(0)
    rc = lib().orc_point_sources(nx, ny, nz, nb, _p(kappa, C.c_float), src.shape[0], _p(src, C.c_int), _p(lum, C.c_double),
                                 float(cell_width), _p(Q, C.c_double), int(diag[0]), int(diag[1]),
                                 _p(d[0], C.c_double), _p(d[1], C.c_double), _p(d[2], C.c_double), _p(d[3], C.c_double),
                                 C.byref(steps), int(nthreads))
    if rc != 0:
        raise RuntimeError("orc_point_sources failed: %d" % rc)
    return {"Q": Q, "tau": d[0], "dtau": d[1], "r_in": d[2], "r_out": d[3], "steps": int(steps.value)}


def point_source_rates(Q, kappa, kappa_sp, n_sp, hnu, hnu_thr):
    """Per-species photo-ionisation and photo-heating rates of the point-source absorption, fp64 (Appendix 1,
    PAPER.md:378-388, eqs. A4-A6), written out per cell:
      absorbed photons per unit time and shell volume in bin b      Ndot_b   = Q_b / (h nu_b)              (A3)
      share of species i (dtau_i / dtau = kappa_i / kappa in a cell) Ndot_i,b = (kappa_i,b / kappa_b) Ndot_b (A4)
      Gamma_i = (1 / n_i) sum_{b: h nu_b >= h nu_i} Ndot_i,b                                               (A5)
      Heat_i  = (1 / n_i) sum_{b: h nu_b >= h nu_i} Ndot_i,b (h nu_b - h nu_i)                             (A6, reading PS-f)
    (N_i = n_i x shell volume; Q is per unit shell volume; the integrals are sums over rectangular bins, eqs. 22-23.)
    Q [nb][cells...], kappa [nb][...] total opacity, kappa_sp [ns][nb][...], n_sp [ns][...]; cells with n_i <= 0 get 0.
    Pinned by tests/test_point_sources.py::test_ps5_*."""
    Q = np.asarray(Q, dtype=np.float64)
    kappa = np.asarray(kappa, dtype=np.float64)
    kappa_sp = np.asarray(kappa_sp, dtype=np.float64)
    n_sp = np.asarray(n_sp, dtype=np.float64)
    ns, nb = kappa_sp.shape[0], kappa_sp.shape[1]
    G = np.zeros(n_sp.shape, dtype=np.float64)
    H = np.zeros(n_sp.shape, dtype=np.float64)
    for i in range(ns):
        for b in range(nb):
            if float(hnu[b]) < float(hnu_thr[i]):
                continue
            ndot_ib = kappa_sp[i, b] / kappa[b] * (Q[b] / float(hnu[b]))
            G[i] += ndot_ib
            H[i] += ndot_ib * (float(hnu[b]) - float(hnu_thr[i]))
        ok = n_sp[i] > 0
        G[i] = np.where(ok, G[i] / np.where(ok, n_sp[i], 1.0), 0.0)
        H[i] = np.where(ok, H[i] / np.where(ok, n_sp[i], 1.0), 0.0)
    return G, H


def num_threads() -> int:
    return int(lib().orc_num_threads())
