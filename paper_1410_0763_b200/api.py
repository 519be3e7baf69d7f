"""ctypes binding of include/rt.h.  Same names as the C ABI; argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

RT_OWNED, RT_ATOMIC_ABLATION, RT_PAPER_GROUPS = 0, 1, 2
RT_J_IN, RT_J_TOTAL, RT_SUM_IN = 0, 1, 2
RT_ELIMIT = -5
RT_STATIC_MAX_SOURCES, RT_STATIC_MAX_BINS = 1024, 16

EXPORTED_SYMBOLS = [
    "rt_healpix_dirs", "rt_create", "rt_set_fields", "rt_set_inflow", "rt_set_inflow_faces", "rt_set_inflow_async", "rt_set_inflow_faces_async", "rt_sweep", "rt_combine", "rt_sweep_rates", "rt_point_sources", "rt_point_sources_static", "rt_point_source_rates", "rt_segment_counts",
    "rt_sum_ds", "rt_total_segments", "rt_debug_writer_counts", "rt_working_set_bytes", "rt_probe_bandwidth", "rt_direction_records", "rt_tune", "rt_last_launch_count",
    "rt_last_sweep_kernel_ms", "rt_last_sweep_was_graph", "rt_destroy", "rt_strerror", "rt_last_cuda_error",
]

_lib = None


class RtError(RuntimeError):
    def __init__(self, code, where):
        L = load_library()
        msg = L.rt_strerror(code).decode()
        cuda = L.rt_last_cuda_error().decode()
        super().__init__("%s failed: %s (%d)%s" % (where, msg, code, (" [" + cuda + "]") if cuda and code == -3 else ""))
        self.code = code


def load_library():
    """Load (building if necessary) librt.so.  Raises if it cannot be built: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.needs_build():
        path = _build.build()
    L = C.CDLL(path)
    vp, dp, fp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_float)
    L.rt_healpix_dirs.argtypes = [C.c_int, dp]
    L.rt_healpix_dirs.restype = C.c_int
    L.rt_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, dp, C.c_int, C.c_int, C.c_double, C.c_uint]
    L.rt_create.restype = C.c_int
    L.rt_set_fields.argtypes = [vp, vp, vp, vp]
    L.rt_set_fields.restype = C.c_int
    L.rt_set_inflow.argtypes = [vp, fp]
    L.rt_set_inflow.restype = C.c_int
    L.rt_set_inflow_faces.argtypes = [vp, fp]
    L.rt_set_inflow_faces.restype = C.c_int
    L.rt_set_inflow_async.argtypes = [vp, fp, vp]
    L.rt_set_inflow_async.restype = C.c_int
    L.rt_set_inflow_faces_async.argtypes = [vp, fp, vp]
    L.rt_set_inflow_faces_async.restype = C.c_int
    L.rt_sweep.argtypes = [vp, vp, C.c_uint, vp]
    L.rt_sweep.restype = C.c_int
    L.rt_combine.argtypes = [vp, vp, C.c_longlong, C.c_uint, vp, vp]
    L.rt_combine.restype = C.c_int
    L.rt_sweep_rates.argtypes = [vp, vp, vp, dp, dp, dp, dp, vp]
    L.rt_sweep_rates.restype = C.c_int
    L.rt_point_sources.argtypes = [vp, C.POINTER(C.c_int), dp, C.c_int, vp, C.c_int, C.c_int, vp, C.POINTER(C.c_ulonglong), vp]
    L.rt_point_sources.restype = C.c_int
    L.rt_point_sources_static.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, C.POINTER(C.c_int), dp, C.c_int, vp,
                                          C.c_int, C.c_int, vp, C.POINTER(C.c_ulonglong), vp]
    L.rt_point_sources_static.restype = C.c_int
    L.rt_point_source_rates.argtypes = [vp, vp, vp, vp, C.c_int, dp, dp, vp, vp, vp]
    L.rt_point_source_rates.restype = C.c_int
    L.rt_segment_counts.argtypes = [vp, C.c_int, vp, vp]
    L.rt_segment_counts.restype = C.c_int
    L.rt_sum_ds.argtypes = [vp, dp, dp, dp, vp]
    L.rt_sum_ds.restype = C.c_int
    L.rt_total_segments.argtypes = [vp, C.POINTER(C.c_ulonglong), vp]
    L.rt_total_segments.restype = C.c_int
    L.rt_debug_writer_counts.argtypes = [vp, C.POINTER(C.c_ulonglong), vp]
    L.rt_debug_writer_counts.restype = C.c_int
    L.rt_working_set_bytes.argtypes = [vp, C.POINTER(C.c_ulonglong)]
    L.rt_working_set_bytes.restype = C.c_int
    L.rt_probe_bandwidth.argtypes = [C.c_ulonglong, C.c_int, C.c_int, dp, vp]
    L.rt_probe_bandwidth.restype = C.c_int
    L.rt_direction_records.argtypes = [vp, C.POINTER(C.c_longlong), dp]
    L.rt_direction_records.restype = C.c_int
    L.rt_tune.argtypes = [vp, C.c_char_p, C.c_int]
    L.rt_tune.restype = C.c_int
    L.rt_last_launch_count.argtypes = [vp]
    L.rt_last_launch_count.restype = C.c_int
    L.rt_last_sweep_kernel_ms.argtypes = [vp]
    L.rt_last_sweep_kernel_ms.restype = C.c_float
    L.rt_last_sweep_was_graph.argtypes = [vp]
    L.rt_last_sweep_was_graph.restype = C.c_int
    L.rt_destroy.argtypes = [vp]
    L.rt_destroy.restype = C.c_int
    L.rt_strerror.argtypes = [C.c_int]
    L.rt_strerror.restype = C.c_char_p
    L.rt_last_cuda_error.argtypes = []
    L.rt_last_cuda_error.restype = C.c_char_p
    _lib = L
    return L


def _check(rc, where):
    if rc != 0:
        raise RtError(rc, where)


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return C.c_void_p(stream)
    return C.c_void_p(stream.cuda_stream)


def _dev_ptr(t, dtype, numel, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype and t.numel() == numel):
        raise ValueError("%s must be a contiguous CUDA tensor of dtype %s with %d elements" % (name, dtype, numel))
    return C.c_void_p(t.data_ptr())


# ---- the C ABI, one function per entry point ------------------------------------------------------
def healpix_dirs(nside: int) -> np.ndarray:
    """rt_healpix_dirs: HEALPix RING pixel centres [12 nside^2][3] fp64 (host)."""
    out = np.empty((12 * nside * nside, 3), dtype=np.float64)
    n = load_library().rt_healpix_dirs(int(nside), out.ctypes.data_as(C.POINTER(C.c_double)))
    if n != out.shape[0]:
        raise RtError(n if n < 0 else -1, "rt_healpix_dirs")
    return out


def rt_create(nx, ny, nz, nbins, dirs, rays_per_cell=1, cell_width=1.0, flags=RT_OWNED):
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    h = C.c_void_p()
    rc = load_library().rt_create(C.byref(h), int(nx), int(ny), int(nz), int(nbins),
                                  dirs.ctypes.data_as(C.POINTER(C.c_double)), dirs.shape[0], int(rays_per_cell),
                                  float(cell_width), int(flags))
    _check(rc, "rt_create")
    return h


def rt_tune(h, key: str, value: int):
    _check(load_library().rt_tune(h, key.encode(), int(value)), "rt_tune(%s)" % key)


def rt_set_fields(h, kappa, S, numel, stream=None):
    import torch
    _check(load_library().rt_set_fields(h, _dev_ptr(kappa, torch.float32, numel, "kappa"),
                                        _dev_ptr(S, torch.float32, numel, "S"), _stream(stream)), "rt_set_fields")


def rt_set_inflow(h, Ibc):
    a = np.ascontiguousarray(Ibc, dtype=np.float32)
    _check(load_library().rt_set_inflow(h, a.ctypes.data_as(C.POINTER(C.c_float))), "rt_set_inflow")


def rt_set_inflow_faces(h, I_face, nbins):
    a = np.ascontiguousarray(I_face, dtype=np.float32).reshape(-1)
    if a.shape[0] != 6 * nbins:
        raise ValueError("I_face must be [nbins][6]")
    _check(load_library().rt_set_inflow_faces(h, a.ctypes.data_as(C.POINTER(C.c_float))), "rt_set_inflow_faces")


def rt_set_inflow_async(h, Ibc, stream=None):
    a = np.ascontiguousarray(Ibc, dtype=np.float32)
    _check(load_library().rt_set_inflow_async(h, a.ctypes.data_as(C.POINTER(C.c_float)), _stream(stream)), "rt_set_inflow_async")


def rt_set_inflow_faces_async(h, I_face, nbins, stream=None):
    a = np.ascontiguousarray(I_face, dtype=np.float32).reshape(-1)
    if a.shape[0] != 6 * nbins:
        raise ValueError("I_face must be [nbins][6]")
    _check(load_library().rt_set_inflow_faces_async(h, a.ctypes.data_as(C.POINTER(C.c_float)), _stream(stream)), "rt_set_inflow_faces_async")


def rt_sweep(h, J, numel, what=RT_J_IN, stream=None):
    import torch
    _check(load_library().rt_sweep(h, _dev_ptr(J, torch.float32, numel, "J"), int(what), _stream(stream)), "rt_sweep")


def rt_combine(h, total, ndirs_total, J, numel, what=RT_J_IN, stream=None):
    import torch
    _check(load_library().rt_combine(h, _dev_ptr(total, torch.float32, numel, "sum"), int(ndirs_total), int(what),
                                     _dev_ptr(J, torch.float32, numel, "J"), _stream(stream)), "rt_combine")


def rt_sweep_rates(h, Gamma, Heat, ncell, nbins, wG, lG, wH, lH, stream=None):
    import torch
    w = [np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in (wG, lG, wH, lH)]
    if any(a.shape[0] != nbins for a in w):
        raise ValueError("rate weights must have one entry per bin")
    p = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    _check(load_library().rt_sweep_rates(h, _dev_ptr(Gamma, torch.float32, ncell, "Gamma"),
                                         _dev_ptr(Heat, torch.float32, ncell, "Heat"), p(w[0]), p(w[1]), p(w[2]), p(w[3]),
                                         _stream(stream)), "rt_sweep_rates")


def rt_point_sources(h, src_fix, lum, Q, numel, nbins, tau=None, diag=(0, 0), want_steps=False, stream=None):
    import torch
    src = np.ascontiguousarray(src_fix, dtype=np.int32).reshape(-1, 3)
    lum = np.ascontiguousarray(lum, dtype=np.float64).reshape(src.shape[0], nbins)
    steps = C.c_ulonglong(0)
    _check(load_library().rt_point_sources(h, src.ctypes.data_as(C.POINTER(C.c_int)), lum.ctypes.data_as(C.POINTER(C.c_double)),
                                           src.shape[0], _dev_ptr(Q, torch.float32, numel, "Q"), int(diag[0]), int(diag[1]),
                                           None if tau is None else _dev_ptr(tau, torch.float32, numel // nbins, "tau"),
                                           C.byref(steps) if want_steps else None, _stream(stream)), "rt_point_sources")
    return int(steps.value)


def rt_point_sources_static(dims, nbins, kappa, src_fix, lum, Q, cell_width=1.0, tau=None, diag=(0, 0), want_steps=False, stream=None):
    """rt_point_sources_static: rt_point_sources without a context and without any allocation by the library, for
    callers whose device memory is spoken for (an arena that owns the GPU, a caching allocator, an MPS memory limit)
    or that cannot afford cudaMalloc's device-wide synchronisation.  kappa, Q (and tau) are the caller's CUDA tensors
    on the current device; the source tables go through a fixed 143,616-byte device array inside librt.so, which caps
    the call at RT_STATIC_MAX_SOURCES sources and RT_STATIC_MAX_BINS bins (RtError with code RT_ELIMIT beyond).  All
    calls on a device share that array: do not let two of them overlap on the GPU.  Returns the step count (0 unless
    want_steps)."""
    import torch
    nx, ny, nz = (int(v) for v in dims)
    numel = nx * ny * nz * int(nbins)
    src = np.ascontiguousarray(src_fix, dtype=np.int32).reshape(-1, 3)
    lum = np.ascontiguousarray(lum, dtype=np.float64).reshape(src.shape[0], nbins)
    steps = C.c_ulonglong(0)
    _check(load_library().rt_point_sources_static(nx, ny, nz, int(nbins), float(cell_width), _dev_ptr(kappa, torch.float32, numel, "kappa"),
                                                  src.ctypes.data_as(C.POINTER(C.c_int)), lum.ctypes.data_as(C.POINTER(C.c_double)),
                                                  src.shape[0], _dev_ptr(Q, torch.float32, numel, "Q"), int(diag[0]), int(diag[1]),
                                                  None if tau is None else _dev_ptr(tau, torch.float32, numel // nbins, "tau"),
                                                  C.byref(steps) if want_steps else None, _stream(stream)), "rt_point_sources_static")
    return int(steps.value)


def rt_point_source_rates(h, Q, kappa_sp, n_sp, hnu, hnu_thr, Gamma, Heat, ncell, nbins, stream=None):
    import torch
    hnu = np.ascontiguousarray(hnu, dtype=np.float64).reshape(-1)
    thr = np.ascontiguousarray(hnu_thr, dtype=np.float64).reshape(-1)
    ns = thr.shape[0]
    if hnu.shape[0] != nbins:
        raise ValueError("hnu must have one entry per bin")
    p = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    _check(load_library().rt_point_source_rates(h, _dev_ptr(Q, torch.float32, ncell * nbins, "Q"),
                                                _dev_ptr(kappa_sp, torch.float32, ns * nbins * ncell, "kappa_sp"),
                                                _dev_ptr(n_sp, torch.float32, ns * ncell, "n_sp"), ns, p(hnu), p(thr),
                                                _dev_ptr(Gamma, torch.float32, ns * ncell, "Gamma"),
                                                _dev_ptr(Heat, torch.float32, ns * ncell, "Heat"), _stream(stream)),
           "rt_point_source_rates")


def rt_segment_counts(h, dir_index, counts, numel, stream=None):
    import torch
    _check(load_library().rt_segment_counts(h, int(dir_index), _dev_ptr(counts, torch.int32, numel, "counts"),
                                            _stream(stream)), "rt_segment_counts")


def rt_sum_ds(h, ndirs, stream=None):
    s, mn, mx = (np.empty(ndirs, dtype=np.float64) for _ in range(3))
    p = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    _check(load_library().rt_sum_ds(h, p(s), p(mn), p(mx), _stream(stream)), "rt_sum_ds")
    return s, mn, mx


def rt_total_segments(h, stream=None) -> int:
    n = C.c_ulonglong(0)
    _check(load_library().rt_total_segments(h, C.byref(n), _stream(stream)), "rt_total_segments")
    return int(n.value)


def rt_debug_writer_counts(h, stream=None) -> dict:
    out = (C.c_ulonglong * 8)()
    _check(load_library().rt_debug_writer_counts(h, out, _stream(stream)), "rt_debug_writer_counts")
    keys = ("max_writers", "stores", "max_seam_writers", "seam_stores", "launches", "partial_launches", "expected_stores", "entries")
    return dict(zip(keys, (int(v) for v in out)))


def rt_working_set_bytes(h) -> int:
    n = C.c_ulonglong(0)
    _check(load_library().rt_working_set_bytes(h, C.byref(n)), "rt_working_set_bytes")
    return int(n.value)


def rt_probe_bandwidth(nbytes: int, mode: int = 0, iters: int = 5, stream=None) -> float:
    """GB/s of the streaming probe over a scratch buffer of nbytes (mode 0 read, 1 read-modify-write)."""
    g = C.c_double(0.0)
    _check(load_library().rt_probe_bandwidth(int(nbytes), int(mode), int(iters), C.byref(g), _stream(stream)), "rt_probe_bandwidth")
    return float(g.value)


def rt_direction_records(h, ndirs):
    rec = np.empty((ndirs, 6), dtype=np.int64)
    L = np.empty(ndirs, dtype=np.float64)
    _check(load_library().rt_direction_records(h, rec.ctypes.data_as(C.POINTER(C.c_longlong)),
                                               L.ctypes.data_as(C.POINTER(C.c_double))), "rt_direction_records")
    return rec, L


def rt_destroy(h):
    _check(load_library().rt_destroy(h), "rt_destroy")


# ---- convenience wrapper (still argument marshalling only) -----------------------------------------
class RayTracer:
    """Owns one rt_ctx.  Fields and outputs are torch CUDA tensors [nbins][nz][ny][nx] fp32."""

    def __init__(self, dims, nbins, dirs, cell_width=1.0, flags=RT_OWNED, slots=None, rows=None, stages=None, pair=None, tune=None,
                 rays_per_cell=1):
        self.nx, self.ny, self.nz = (int(v) for v in dims)
        self.nbins = int(nbins)
        self.dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
        self.ndirs = self.dirs.shape[0]
        self.numel = self.nx * self.ny * self.nz * self.nbins
        self.h = rt_create(self.nx, self.ny, self.nz, self.nbins, self.dirs, rays_per_cell, cell_width, flags)
        if slots is not None:
            rt_tune(self.h, "slots", slots)
        if rows is not None:
            rt_tune(self.h, "rows", rows)
        if stages is not None:
            rt_tune(self.h, "stages", stages)
        if pair is not None:
            rt_tune(self.h, "pair", int(pair))
        for k, v in (tune or {}).items():
            rt_tune(self.h, k, int(v))

    def shape(self):
        return (self.nbins, self.nz, self.ny, self.nx)

    def set_fields(self, kappa, S, stream=None):
        rt_set_fields(self.h, kappa, S, self.numel, stream)

    def set_inflow(self, Ibc):
        rt_set_inflow(self.h, Ibc)

    def set_inflow_faces(self, I_face):
        rt_set_inflow_faces(self.h, I_face, self.nbins)

    def set_inflow_async(self, Ibc, stream=None):
        if np.asarray(Ibc).reshape(-1).shape[0] != self.nbins:
            raise ValueError("Ibc must have one value per bin")
        rt_set_inflow_async(self.h, Ibc, stream)

    def set_inflow_faces_async(self, I_face, stream=None):
        rt_set_inflow_faces_async(self.h, I_face, self.nbins, stream)

    def sweep(self, out=None, what=RT_J_IN, stream=None):
        import torch
        if out is None:
            out = torch.empty(self.shape(), dtype=torch.float32, device="cuda")
        rt_sweep(self.h, out, self.numel, what, stream)
        return out

    def combine(self, total, ndirs_total, what=RT_J_IN, out=None, stream=None):
        """rt_combine: J from the all-reduced RT_SUM_IN results of a direction-sharded sweep."""
        if out is None:
            out = total
        rt_combine(self.h, total, ndirs_total, out, self.numel, what, stream)
        return out

    def sweep_rates(self, wG, lG, wH, lH, stream=None):
        """rt_sweep_rates: (Gamma, Heat), each [nz][ny][nx] fp32."""
        import torch
        G = torch.empty((self.nz, self.ny, self.nx), dtype=torch.float32, device="cuda")
        H = torch.empty_like(G)
        rt_sweep_rates(self.h, G, H, self.nx * self.ny * self.nz, self.nbins, wG, lG, wH, lH, stream)
        return G, H

    def point_sources(self, src_fix, lum, diag=None, want_steps=False, stream=None):
        """rt_point_sources: Q [nbins][nz][ny][nx] (+ tau of (source, bin) = diag, + the step count)."""
        import torch
        Q = torch.empty(self.shape(), dtype=torch.float32, device="cuda")
        tau = torch.empty((self.nz, self.ny, self.nx), dtype=torch.float32, device="cuda") if diag is not None else None
        n = rt_point_sources(self.h, src_fix, lum, Q, self.numel, self.nbins, tau, diag or (0, 0), want_steps, stream)
        return Q, tau, n

    def point_source_rates(self, Q, kappa_sp, n_sp, hnu, hnu_thr, stream=None):
        """rt_point_source_rates: per-species (Gamma, Heat), each [nspecies][nz][ny][nx] (eqs. A4-A6)."""
        import torch
        ns = int(n_sp.shape[0])
        G = torch.empty((ns, self.nz, self.ny, self.nx), dtype=torch.float32, device="cuda")
        H = torch.empty_like(G)
        rt_point_source_rates(self.h, Q, kappa_sp, n_sp, hnu, hnu_thr, G, H, self.nx * self.ny * self.nz, self.nbins, stream)
        return G, H

    def segment_counts(self, dir_index=-1, stream=None):
        import torch
        out = torch.empty((self.nz, self.ny, self.nx), dtype=torch.int32, device="cuda")
        rt_segment_counts(self.h, dir_index, out, self.nx * self.ny * self.nz, stream)
        return out

    def sum_ds(self, stream=None):
        return rt_sum_ds(self.h, self.ndirs, stream)

    def total_segments(self, stream=None) -> int:
        return rt_total_segments(self.h, stream)

    def debug_writer_counts(self, stream=None) -> dict:
        return rt_debug_writer_counts(self.h, stream)

    def working_set_bytes(self) -> int:
        return rt_working_set_bytes(self.h)

    def direction_records(self):
        return rt_direction_records(self.h, self.ndirs)

    def last_launch_count(self) -> int:
        return int(load_library().rt_last_launch_count(self.h))

    def last_sweep_kernel_ms(self) -> float:
        return float(load_library().rt_last_sweep_kernel_ms(self.h))

    def last_sweep_was_graph(self) -> bool:
        return int(load_library().rt_last_sweep_was_graph(self.h)) == 1

    def close(self):
        if self.h is not None:
            rt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
