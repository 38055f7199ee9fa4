"""Sharding of replicas (lattice copies / temperatures) over ranks -- the only way the path shards.

The paper runs several lattice copies in parallel and averages them; copies are independent, so a rank
owns a subset of them, no collective runs during sweeps, and one gather of the per-replica observables ends the job.
Host-side logic only (no kernels): works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""


def replica_shard(n_replicas, rank, world):
    """Indices of the replicas rank `rank` of `world` owns: round-robin, so neighbouring temperatures (similar cost)
    spread evenly.  Every replica is owned by exactly one rank."""
    if world < 1 or not (0 <= rank < world) or n_replicas < 0:
        raise ValueError("bad (n_replicas, rank, world)")
    return list(range(rank, n_replicas, world))


def gather_observables(local, n_replicas, rank=None, world=None, group=None):
    """local: {global replica index: observables dict} of this rank.  Returns the list of all n_replicas observables in
    replica order on every rank (one all_gather_object of about 100 B per replica)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        world = dist.get_world_size(group) if world is None else world
        parts = [None] * world
        dist.all_gather_object(parts, local, group=group)
    else:
        parts = [local]
    merged = {}
    for p in parts:
        for k, v in p.items():
            if k in merged:
                raise RuntimeError(f"replica {k} reported by two ranks")
            merged[int(k)] = v
    missing = [r for r in range(n_replicas) if r not in merged]
    if missing:
        raise RuntimeError(f"replicas without an owner: {missing[:8]}")
    return [merged[r] for r in range(n_replicas)]


def max_over_ranks(value, group=None):
    """Max of a host float over ranks (timing rule: a multi-rank time is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
