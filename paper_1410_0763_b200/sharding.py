"""Direction sharding across GPUs: the paper's multi-accelerator scheme (every
device holds the whole mesh and a share of the directions; the partial mean intensities are summed).

Host logic only.  `shard_directions` splits a direction set into `world` shares that (a) are a
partition of the set, (b) carry nearly equal work  sum_i (|n_x|+|n_y|+|n_z|)/max|n|  (segments per
cell of a direction) and (c) keep a direction together with its mirror images along
the two transverse axes, so that the sweep kernel's mirror pairs stay on one device.
`sweep_sharded` is the exchange step: each rank sweeps its share with RT_SUM_IN, one
all-reduce(sum) over `torch.distributed` (NCCL on GPUs), then rt_combine.  The data path has no
other collective.
"""
from __future__ import annotations

import numpy as np


def direction_work(dirs: np.ndarray) -> np.ndarray:
    """Segments per cell of each direction: 1 + m_b + m_c = (|nx|+|ny|+|nz|) / max|n|."""
    a = np.abs(np.asarray(dirs, dtype=np.float64).reshape(-1, 3))
    return a.sum(axis=1) / a.max(axis=1)


def shard_directions(dirs: np.ndarray, world: int, rank: int | None = None):
    """Partition of range(len(dirs)) into `world` index arrays (sorted ascending).  Returns the list of
    all shares, or the share of `rank` if given.  Deterministic: every rank computes the same plan."""
    d = np.asarray(dirs, dtype=np.float64).reshape(-1, 3)
    n = d.shape[0]
    if world < 1:
        raise ValueError("world must be >= 1")
    a = np.abs(d)
    dom = np.argmax(a, axis=1)                        # ties: lowest axis, like the library
    # group key: dominant axis, its sign, and the absolute direction rounded well above the
    # library's 2^-20 slope quantum -> a direction and its transverse mirrors share a key
    unit = a / np.linalg.norm(a, axis=1, keepdims=True)
    q = np.rint(unit * 2.0 ** 26).astype(np.int64)
    sgn = np.take_along_axis(d, dom[:, None], axis=1)[:, 0] < 0
    groups: dict = {}
    for i in range(n):
        groups.setdefault((int(dom[i]), bool(sgn[i]), int(q[i, 0]), int(q[i, 1]), int(q[i, 2])), []).append(i)
    work = direction_work(d)
    glist = sorted(groups.values(), key=lambda g: (-work[g].sum(), g[0]))
    load = np.zeros(world)
    shares = [[] for _ in range(world)]
    for g in glist:                                   # longest-processing-time first
        r = int(np.argmin(load))
        shares[r].extend(g)
        load[r] += work[g].sum()
    shares = [np.array(sorted(s), dtype=np.int64) for s in shares]
    return shares if rank is None else shares[rank]


def sweep_sharded(tracer, ndirs_total: int, what: int = 0, group=None, out=None, stream=None):
    """One direction-sharded sweep on this rank: `tracer` holds this rank's share of the directions.
    Returns J (RT_J_IN / RT_J_TOTAL) of the WHOLE direction set, identical on every rank."""
    import torch.distributed as dist
    from . import api
    total = tracer.sweep(out=out, what=api.RT_SUM_IN, stream=stream)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(total, op=dist.ReduceOp.SUM, group=group)
    return tracer.combine(total, ndirs_total, what=what, stream=stream)
