"""N > 1 host logic (replicas) with world_size-2 gloo on the CPU: the systems are partitioned without
overlap, the timing is the max over ranks, scalars are gathered in rank order."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2307_14296_b200 import replicas
    lo, hi = replicas.shard(7, rank, world)
    tmax = replicas.max_over_ranks([10.0 + rank, 5.0 - rank])
    allv = replicas.gather_scalars([complex(rank, k) for k in range(lo, hi)][:3])
    q.put((rank, lo, hi, tmax, allv))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_two_shards_and_reductions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, t0, g0), (r1, lo1, hi1, t1, g1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 4, 4, 7)
    assert t0 == t1 == [11.0, 5.0]
    assert g0 == g1 == [0j, 1j, 2j, 1 + 4j, 1 + 5j, 1 + 6j]


def test_shard_partitions_every_size():
    from paper_2307_14296_b200 import replicas
    for n in range(0, 20):
        for w in range(1, 9):
            cuts = [replicas.shard(n, r, w) for r in range(w)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[k][1] == cuts[k + 1][0] for k in range(w - 1))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
