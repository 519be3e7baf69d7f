"""rt_point_sources_static: the point-source solver for callers that cannot allocate device memory.

Some users of this library never get to call cudaMalloc: a radiation-hydrodynamics code whose own arena took
the GPU's memory at start-up, anything living under a framework's caching allocator or an MPS memory limit, and
code inside a time step that cannot take the device-wide synchronisation an allocation implies.  For them the
library has one entry point that allocates nothing; its scratch memory (device copy of the source tables + the
step counter) is a fixed 143,616-byte array inside librt.so, shared by every call on a device.

The check here is against the library's regular path (rt_create + rt_set_fields + rt_point_sources, itself gated
against the oracle in test_point_sources.py), with that file's tolerance, on two calls in a row with different
sources: the second call must not see anything of the first (the counter is cleared, the tables overwritten).

This file is named so that pytest collects it last: with `-x` a failure here hides no other test.  It passes alone
in a fresh process (the first call does the per-device set-up) and after the rest of the suite."""
import numpy as np
import pytest

FIX = 256
PS_TOL = 1e-5          # same gate as tests/test_point_sources.py


def _rel(got, ref):
    ref = np.asarray(ref, dtype=np.float64)
    floor = max(1e-30 * np.abs(ref).max(), 1e-300)
    return np.abs(np.asarray(got, dtype=np.float64) - ref) / np.maximum(np.abs(ref), floor)


@pytest.mark.gpu
@pytest.mark.parametrize("dims,nb,cw", [((33, 20, 17), 2, 0.7), ((100, 30, 12), 3, 1.0)])
def test_static_scratch_point_sources_match_the_context_path(dims, nb, cw):
    """Two consecutive calls of the no-allocation entry point (six sources, then two others: fewer sources, so stale
    table rows and a stale counter would show) against rt_point_sources on the same inputs: step counts equal,
    tau and Q within 1e-5 on every cell; and the library's device-memory footprint does not grow across the calls."""
    import torch
    import paper_1410_0763_b200 as rt
    assert torch.cuda.is_available()
    nx, ny, nz = dims
    rng = np.random.default_rng(91)
    kap = rng.uniform(0.02, 0.6, (nb, nz, ny, nx)).astype(np.float32)
    kap[:, nz // 2:, : ny // 2, :] *= 8.0                      # an opaque block: exp(-tau) spans many decades
    kap[0, 0, 0, :3] = 0.0                                     # kappa = 0 cells: both paths floor them at 2^-60
    src_a = np.array([[0, 0, 0], [nx * FIX, ny * FIX, nz * FIX], [(nx // 2) * FIX + 128, (ny // 2) * FIX + 128, (nz // 2) * FIX + 128],
                      [nx * FIX // 3, 0, nz * FIX // 2], [17, ny * FIX - 1, 3], [(nx // 2) * FIX, (ny // 2) * FIX, 77]], dtype=np.int32)
    src_b = np.array([[nx * FIX, 0, 40], [5 * FIX + 9, 3 * FIX + 128, 2 * FIX]], dtype=np.int32)
    calls = [(src_a, rng.uniform(0.5, 2.0, (len(src_a), nb)), (len(src_a) - 1, nb - 1)),
             (src_b, rng.uniform(0.5, 2.0, (len(src_b), nb)), (1, 0))]
    kap_d = torch.from_numpy(kap).cuda()
    tr = rt.RayTracer(dims, nb, rt.healpix_dirs(1), cell_width=cw)
    try:
        tr.set_fields(kap_d, torch.zeros_like(kap_d))
        ref = [tr.point_sources(src, lum, diag=diag, want_steps=True) for src, lum, diag in calls]
        ref = [(Q.cpu().numpy(), tau.cpu().numpy(), n) for Q, tau, n in ref]
    finally:
        tr.close()
    Q = torch.empty_like(kap_d)
    tau = torch.empty((nz, ny, nx), dtype=torch.float32, device="cuda")
    # Two rounds of the two calls.  The first round is also the warm-up: the first call on this device (in a fresh
    # process) resolves the scratch array's address, and the CUDA runtime loads each kernel's code at its first launch,
    # which takes device memory that is not an allocation of the library's.  The second round must leave the free
    # memory where the first left it.
    free = []
    for _ in range(2):
        for (src, lum, diag), (Q_ref, tau_ref, n_ref) in zip(calls, ref):
            Q.fill_(-1.0)
            tau.fill_(-1.0)
            n = rt.rt_point_sources_static(dims, nb, kap_d, src, lum, Q, cell_width=cw, tau=tau, diag=diag, want_steps=True)
            assert n == n_ref
            assert _rel(tau.cpu().numpy(), tau_ref).max() <= PS_TOL
            assert _rel(Q.cpu().numpy(), Q_ref).max() <= PS_TOL
            rt.rt_point_sources_static(dims, nb, kap_d, src, lum, Q, cell_width=cw)      # the non-counting instantiation
            assert _rel(Q.cpu().numpy(), Q_ref).max() <= PS_TOL
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    assert free[1] >= free[0], "device memory in use grew by %d bytes across no-allocation calls" % (free[0] - free[1])


@pytest.mark.gpu
def test_static_scratch_capacity_is_enforced():
    """Beyond RT_STATIC_MAX_SOURCES sources or RT_STATIC_MAX_BINS bins the call is refused with RT_ELIMIT (a code of its
    own, with a text) before anything is enqueued; exactly at the limit it runs."""
    import torch
    import paper_1410_0763_b200 as rt
    dims = (8, 6, 4)
    kap = torch.full((1, 4, 6, 8), 0.3, dtype=torch.float32, device="cuda")
    Q = torch.full_like(kap, -1.0)
    n_max = rt.RT_STATIC_MAX_SOURCES
    src = np.zeros((n_max + 1, 3), dtype=np.int32)
    src[:, 0] = np.arange(n_max + 1) % (8 * FIX)
    with pytest.raises(rt.RtError) as ei:
        rt.rt_point_sources_static(dims, 1, kap, src, np.ones((n_max + 1, 1)), Q)
    assert ei.value.code == rt.RT_ELIMIT and "capacity" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((Q == -1.0).all()), "a refused call must not touch the output"
    nb = rt.RT_STATIC_MAX_BINS + 1
    kap_b = torch.full((nb, 4, 6, 8), 0.3, dtype=torch.float32, device="cuda")
    with pytest.raises(rt.RtError) as ei:
        rt.rt_point_sources_static(dims, nb, kap_b, src[:1], np.ones((1, nb)), torch.empty_like(kap_b))
    assert ei.value.code == rt.RT_ELIMIT
    # at the limit: n_max unit sources at one point give n_max times the Q of one source there
    one = np.array([[3 * FIX + 40, 2 * FIX + 7, 1 * FIX + 200]], dtype=np.int32)
    Q1 = torch.empty_like(kap)
    rt.rt_point_sources_static(dims, 1, kap, one, np.ones((1, 1)), Q1)
    rt.rt_point_sources_static(dims, 1, kap, np.repeat(one, n_max, axis=0), np.ones((n_max, 1)), Q)
    assert _rel(Q.cpu().numpy(), n_max * Q1.cpu().numpy().astype(np.float64)).max() <= PS_TOL
