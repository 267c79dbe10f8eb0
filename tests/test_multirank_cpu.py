"""N > 1 host logic on CPU: world_size-2 gloo processes shard a ragged batch by replica, each evaluates
its shard (with the CPU oracle standing in for the GPU kernels -- tests may use it), the per-replica
observables are gathered, and the result must equal the unsharded evaluation.  No data-path collective
exists, so what is tested is the partition, the gather and the timing reduction."""
import os
import socket

import numpy as np
import pytest

from paper_1311_3890_b200 import sharding
from paper_1311_3890_b200 import workloads as W

torch = pytest.importorskip("torch")


def test_replica_range_is_a_balanced_contiguous_partition():
    for n in (0, 1, 5, 256, 2048, 2049):
        for world in (1, 2, 3, 8):
            edges = [sharding.replica_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.replica_range(4, 2, 2)


def test_shard_keeps_replica_metadata():
    w = W.config4(5, seed=9)
    got = []
    for rank in range(2):
        sub, (r0, r1) = sharding.shard_workload(w, rank, 2)
        assert np.array_equal(sub.seed, w.seed[r0:r1]) and np.array_equal(sub.T, w.T[r0:r1])
        assert np.array_equal(sub.pos4, w.pos4[w.offsets[r0]:w.offsets[r1]])
        assert sub.offsets[0] == 0 and sub.offsets[-1] == sub.n_atoms
        got.append(sub.n_atoms)
    assert sum(got) == w.n_atoms


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.config4(5, seed=9)                       # ragged: 5 replicas over 2 ranks -> 3 + 2
        sub, (r0, r1) = sharding.shard_workload(w, rank, world)
        o = oracle.compute(sub.x64(), sub.r_cut, offsets=sub.offsets, lo=sub.box_lo, hi=sub.box_hi,
                           periodic=sub.periodic, cells=True)
        local = np.concatenate([o["e_rep"][:, None], o["w_rep"]], axis=1)      # (r1 - r0, 7)
        full = sharding.gather_replica_values(local, w.n_replicas, rank, world, dist)
        t = sharding.max_over_ranks(10.0 + rank, world, dist)
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), full)
        with open(os.path.join(out_dir, f"t{rank}.txt"), "w") as f:
            f.write(repr(t))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_sharded_equals_unsharded(tmp_path):
    import torch.multiprocessing as mp
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = W.config4(5, seed=9)
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, periodic=w.periodic,
                       cells=True)
    want = np.concatenate([o["e_rep"][:, None], o["w_rep"]], axis=1)
    for rank in range(world):
        got = np.load(tmp_path / f"rank{rank}.npy")
        assert got.shape == want.shape
        # replicas are independent; only the OpenMP reduction order of the oracle differs run to run
        assert np.allclose(got, want, rtol=1e-12, atol=1e-9)
        assert float(open(tmp_path / f"t{rank}.txt").read()) == 11.0
