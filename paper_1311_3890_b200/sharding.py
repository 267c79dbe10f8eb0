"""Replica sharding across ranks: host logic only, no arithmetic of the method.

The path shards by replica and only by replica -- replicas never interact (the paper's campaign is
thousands of independent single-GPU runs) -- so there is NO data-path collective.
What remains is (i) a contiguous, balanced partition of the replica range, (ii) the gather of the
per-replica observables (a few doubles per replica per logged step) onto rank 0, and (iii) the
max-over-ranks of a timing.  (ii) and (iii) go through torch.distributed (nccl on GPUs, gloo in the
CPU tests).
"""
import numpy as np


def replica_range(n_replicas, rank, world):
    """Contiguous balanced partition: the first n_replicas % world ranks get one replica more."""
    if world < 1 or not (0 <= rank < world) or n_replicas < 0:
        raise ValueError("bad (n_replicas, rank, world)")
    base, extra = divmod(n_replicas, world)
    r0 = rank * base + min(rank, extra)
    return r0, r0 + base + (1 if rank < extra else 0)


def shard_workload(w, rank, world):
    """The sub-batch of `w` (workloads.Workload) that `rank` owns.  Seeds, temperatures, boxes and
    pulling rates travel with their replica, so a replica's trajectory does not depend on the
    sharding (Philox is keyed by the replica seed and the tag inside the replica)."""
    r0, r1 = replica_range(w.n_replicas, rank, world)
    return w.take(r0, r1, name=f"{w.name}[rank {rank}/{world}]"), (r0, r1)


def gather_replica_values(local, n_replicas, rank, world, dist=None, device=None):
    """Per-replica observables of every rank -> one (n_replicas, ...) array on every rank.
    `local` is this rank's (r1 - r0, ...) float64 array.  world == 1 needs no process group."""
    local = np.ascontiguousarray(local, dtype=np.float64)
    if world == 1:
        return local.copy()
    import torch
    counts = [replica_range(n_replicas, r, world) for r in range(world)]
    width = max(b - a for a, b in counts)
    tail = local.shape[1:]
    pad = np.zeros((width,) + tail)
    pad[:len(local)] = local
    t = torch.from_numpy(pad)
    if device is not None:
        t = t.to(device)
    out = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(out, t)
    parts = [o.cpu().numpy()[:b - a] for o, (a, b) in zip(out, counts)]
    return np.concatenate(parts, axis=0)


def max_over_ranks(x, world, dist=None, device=None):
    if world == 1:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
