"""-m "not gpu": the N>1 host logic (barrier, max-over-ranks timing, whole-job aggregation,
replica inputs) under torch.distributed gloo with world_size 2, on the CPU."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

import workloads


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_1803_03498_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    replicas.barrier(world)
    t = replicas.max_over_ranks(1.0 + rank, world)           # rank 1 is the slow one
    agg = replicas.aggregate_throughput(100.0, 1.0 + rank, world)
    s0 = replicas.replica_sigma0(workloads.dimer(), rank)
    q.put((rank, t, agg, int(np.argmax(np.diag(s0).real))))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [o[1] for o in out] == [2.0, 2.0]                 # max over ranks on every rank
    assert [o[2] for o in out] == [100.0, 100.0]             # 2 ranks x 100 units / 2.0 s
    assert [o[3] for o in out] == [0, 1]                     # replicas start on different sites


def test_single_rank_passthrough():
    from paper_1803_03498_b200 import replicas
    assert replicas.max_over_ranks(3.5, 1) == 3.5
    replicas.barrier(1)
