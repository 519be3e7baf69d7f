"""Direction sharding: the host-side plan, and the exchange step on two gloo ranks
on the CPU with the oracle standing in for the per-rank sweep (the GPU version of the same algebra is
tests/test_gpu_parity.py::test_direction_shards_combine)."""
import os
import socket

import numpy as np
import pytest


@pytest.mark.parametrize("nside,world", [(2, 2), (4, 3), (8, 8), (16, 8), (1, 5)])
def test_plan_is_a_balanced_partition_that_keeps_mirrors_together(orc, nside, world):
    from paper_1410_0763_b200.sharding import shard_directions, direction_work
    dirs = orc.healpix_dirs(nside)
    shares = shard_directions(dirs, world)
    allidx = np.concatenate(shares)
    assert sorted(allidx.tolist()) == list(range(len(dirs)))                  # partition
    for r in range(world):
        assert np.array_equal(shard_directions(dirs, world, r), shares[r])     # every rank computes the same plan
    w = direction_work(dirs)
    loads = np.array([w[s].sum() for s in shares])
    if len(dirs) >= 16 * world:
        assert loads.max() / loads.mean() < 1.05                               # balanced by segments per cell
    # a direction and its b-/c-mirror (same dominant axis and sense) sit in the same share
    owner = np.empty(len(dirs), dtype=int)
    for r, s in enumerate(shares):
        owner[s] = r
    recs = [orc.dir_record(d) for d in dirs]
    key = {}
    for i, rec in enumerate(recs):
        k = (rec["a"], rec["refl"][rec["a"]], rec["Mb"], rec["Mc"])
        key.setdefault(k, set()).add(owner[i])
    assert all(len(v) == 1 for v in key.values())


def test_work_is_segments_per_cell(orc):
    """direction_work = 1 + m_b + m_c: the exact per-cell segment count of a generic direction (pin P4)."""
    from paper_1410_0763_b200.sharding import direction_work
    dirs = np.array([[1.0, 0.37, 0.81], [0.3, -1.0, 0.2], [0, 0, 1]])
    w = direction_work(dirs)
    kap = np.ones((1, 16, 16, 16), dtype=np.float32)
    for i, d in enumerate(dirs):
        r = orc.sweep(kap, kap, d[None])
        assert abs(r["seg_total"] / 16 ** 3 - w[i]) < 0.02 * w[i]


def _rank_main(rank, world, port, tmpdir):
    import torch
    import torch.distributed as dist
    from oracle import oracle
    from paper_1410_0763_b200.sharding import shard_directions
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(11)
        kap = rng.uniform(0.05, 2.0, (2, 6, 8, 10)).astype(np.float32)
        S = rng.uniform(0.0, 1.0, (2, 6, 8, 10)).astype(np.float32)
        dirs = oracle.healpix_dirs(2)
        mine = shard_directions(dirs, world, rank)
        loc = oracle.sweep(kap, S, dirs[mine], nthreads=1, want_counts=False)
        total = torch.from_numpy(loc["Jin"] * len(mine))          # RT_SUM_IN of this share
        dist.all_reduce(total, op=dist.ReduceOp.SUM)               # the one exchange step
        Jin = total.numpy() / len(dirs)                            # rt_combine
        np.save(os.path.join(tmpdir, "jin_%d.npy" % rank), Jin)
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_full_sweep(orc, tmp_path):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_rank_main, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    rng = np.random.default_rng(11)
    kap = rng.uniform(0.05, 2.0, (2, 6, 8, 10)).astype(np.float32)
    S = rng.uniform(0.0, 1.0, (2, 6, 8, 10)).astype(np.float32)
    ref = orc.sweep(kap, S, orc.healpix_dirs(2), want_counts=False)["Jin"]
    j0 = np.load(tmp_path / "jin_0.npy")
    j1 = np.load(tmp_path / "jin_1.npy")
    assert np.array_equal(j0, j1)                                  # identical on every rank
    assert np.abs(j0 / ref - 1).max() < 1e-12


def _nccl_rank_main(rank, world, port, tmpdir):
    import torch
    import torch.distributed as dist
    import paper_1410_0763_b200 as rt
    from rt_inputs import make_fields
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        dims = (64, 32, 48)
        kap, S = make_fields("C3", dims=dims)
        dirs = rt.healpix_dirs(4)
        tr = rt.RayTracer(dims, 1, dirs[rt.shard_directions(dirs, world, rank)])
        try:
            tr.set_fields(torch.from_numpy(kap).cuda(), torch.from_numpy(S).cuda())
            Jin = rt.sweep_sharded(tr, len(dirs), what=rt.RT_J_IN).cpu().numpy()
        finally:
            tr.close()
        np.save(os.path.join(tmpdir, "nccl_jin_%d.npy" % rank), Jin)
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_two_nccl_ranks_sweep_sharded(orc, tmp_path):
    """sweep_sharded under NCCL on two devices of one node (one process per GPU): every rank sweeps its share with
    RT_SUM_IN, one all-reduce, rt_combine -> J_in of the whole set on both ranks.  Skipped with fewer than two GPUs."""
    import torch
    import torch.multiprocessing as mp
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    from rt_inputs import make_fields
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_nccl_rank_main, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    kap, S = make_fields("C3", dims=(64, 32, 48))
    ref = orc.sweep(kap, S, orc.healpix_dirs(4), want_counts=False)["Jin"]
    j0 = np.load(tmp_path / "nccl_jin_0.npy")
    j1 = np.load(tmp_path / "nccl_jin_1.npy")
    assert np.array_equal(j0, j1)
    floor = 1e-30 * np.abs(ref).max()
    assert (np.abs(j0 - ref) / np.maximum(np.abs(ref), floor)).max() <= 1e-5
