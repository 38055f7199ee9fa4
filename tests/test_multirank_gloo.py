"""world_size-2 gloo test of the replica sharding and the observable gather; CPU only."""
import importlib.util
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _shard_module():
    # loaded by path: importing the package would build and load the CUDA library, which this test does not need
    spec = importlib.util.spec_from_file_location("ic_shard", os.path.join(ROOT, "paper_2301_11735_b200", "shard.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def _worker(rank, world, port, n_replicas, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sh = _shard_module()
        mine = sh.replica_shard(n_replicas, rank, world)
        local = {r: {"replica": r, "T": 0.1 * (r + 1), "owner": rank} for r in mine}
        allobs = sh.gather_observables(local, n_replicas)
        slow = sh.max_over_ranks(10.0 + rank)
        q.put((rank, mine, [(o["replica"], o["owner"]) for o in allobs], slow))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_replicas", [1, 7, 16])
def test_replicas_shard_over_two_ranks(n_replicas):
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_replicas, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    got.sort()
    owned = sorted(r for _, mine, _, _ in got for r in mine)
    assert owned == list(range(n_replicas))                     # every replica has exactly one owner
    for rank, mine, allobs, slow in got:
        assert [r for r, _ in allobs] == list(range(n_replicas))  # gathered in replica order on every rank
        assert all(owner == r % world for r, owner in allobs)
        assert slow == 11.0                                     # max over ranks


def test_shard_argument_checks():
    sh = _shard_module()
    assert sh.replica_shard(5, 1, 2) == [1, 3]
    assert sh.replica_shard(0, 0, 1) == []
    with pytest.raises(ValueError):
        sh.replica_shard(4, 2, 2)
    assert sh.gather_observables({0: "a", 1: "b"}, 2) == ["a", "b"]
    with pytest.raises(RuntimeError):
        sh.gather_observables({0: "a"}, 2)
