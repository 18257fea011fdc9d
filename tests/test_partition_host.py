"""-m "not gpu": the host side of the sharded path (heom_create_partition): ownership, ghost sets, local link
tables against the oracle's global tables (bit-exact after the index maps), the exchange plan, and the exchange
itself under torch.distributed gloo with world_size 2 and 3 on integer payloads."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from oracle.oracle import Oracle
from paper_1803_03498_b200 import Heom, HeomError
from paper_1803_03498_b200.sharded import exchange_plan_check, slice_plan_check


def _parts(N, K, D, world, bath_state=None):
    H = np.zeros((N, N))
    return [Heom(H, 35.0, 0.02, 300.0, K, D, partition=(r, world), bath_state=bath_state) for r in range(world)]


@pytest.mark.parametrize("N,K,D,world", [(2, 1, 4, 2), (2, 1, 4, 3), (7, 1, 3, 4), (3, 2, 5, 8), (14, 0, 3, 5),
                                         (2, 0, 6, 7), (5, 0, 1, 2), (4, 1, 3, 1)])
def test_partition_tables_vs_oracle(N, K, D, world):
    o = Oracle(np.zeros((N, N)), 35.0, 0.02, 300.0, K, D)
    t, plus, minus = o.tables()
    parts = _parts(N, K, D, world)
    owned_all, plans = [], []
    for r, g in enumerate(parts):
        gid, sc, rc, idx = g.partition_plan()
        n_own = g.owned()
        assert g.nodes == gid.size and sc[r] == 0 and rc[r] == 0 and rc.sum() == g.nodes - n_own
        lt, lp, lm = g.tables()
        assert np.array_equal(lt, t[gid])                          # tuples of the local nodes
        for loc, glob in ((lp, plus), (lm, minus)):
            own = loc[:n_own]
            want = glob[gid[:n_own]]
            assert np.array_equal(own >= 0, want >= 0)             # every link of an owned node is local
            assert np.array_equal(gid[own[own >= 0]], want[want >= 0])
            assert np.all(loc[n_own:] == -1)                       # ghost rows are copies only
        # every ghost is the neighbour of an owned node; send rows are owned rows
        nb = np.concatenate([lp[:n_own].ravel(), lm[:n_own].ravel()])
        assert set(range(n_own, g.nodes)) <= set(nb[nb >= 0].tolist())
        assert idx.size == sc.sum() and (idx.size == 0 or (idx.min() >= 0 and idx.max() < n_own))
        owned_all.append(gid[:n_own])
        plans.append((gid, n_own, sc, rc, idx))
    allowned = np.concatenate(owned_all)
    assert np.array_equal(np.sort(allowned), np.arange(o.nodes))   # a partition of the node set
    sizes = [len(a) for a in owned_all]
    assert max(sizes) - min(sizes) <= 1                            # balanced
    assert exchange_plan_check(plans)
    assert sum(1 for g in parts if g.owned() and 0 in g.partition_plan()[0][:g.owned()]) == 1


@pytest.mark.parametrize("N,K,D,world,bath_state", [(2, 1, 4, 2, None), (7, 1, 3, 4, None), (3, 2, 5, 8, None),
                                                    (14, 0, 3, 5, None), (4, 1, 3, 3, [1, 2, 3])])
def test_slice_halo_plan(N, K, D, world, bath_state):
    """The slice halo: (ghost, state) pairs are exactly what the owned nodes' links read, each once; sender and
    receiver lists agree pair for pair; never more rows than whole ghost nodes would carry."""
    parts = _parts(N, K, D, world, bath_state=bath_state)
    M = K + 1
    states = list(range(N)) if bath_state is None else bath_state
    info = []
    for r, g in enumerate(parts):
        gid, sc, rc, idx = g.partition_plan()
        ps = g.partition_plan_slices()
        psc, prc, sn, ss, rn, rs = ps
        n_own = g.owned()
        lt, lp, lm = g.tables()
        want = set()
        for tab in (lp, lm):
            u, l = np.nonzero(tab[:n_own] >= n_own)                # links of owned nodes into the ghost region
            want |= set(zip(tab[u, l].tolist(), [states[x // M] for x in l.tolist()]))
        got = list(zip(rn.tolist(), rs.tolist()))
        assert len(got) == len(set(got)) and set(got) == want      # every pair once, nothing else
        assert psc[r] == 0 and prc[r] == 0
        assert sn.size == psc.sum() and (sn.size == 0 or (sn.min() >= 0 and sn.max() < n_own))
        assert rn.size == 0 or rn.min() >= n_own
        assert len(got) <= (g.nodes - n_own) * N                   # at most every row of every ghost
        info.append((gid, ps))
    assert slice_plan_check(info)


def test_partition_with_site_map_and_validation():
    parts = _parts(4, 1, 3, 2, bath_state=[1, 2, 3])
    o = Oracle(np.zeros((4, 4)), 35.0, 0.02, 300.0, 1, 3, bath_state=[1, 2, 3])
    assert sum(g.owned() for g in parts) == o.nodes
    for bad in ((2, 2), (-1, 2), (0, 0)):
        with pytest.raises(HeomError):
            Heom(np.zeros((2, 2)), 35.0, 0.02, 300.0, 1, 2, partition=bad)
    with pytest.raises(HeomError):
        Heom(np.zeros((2, 2)), 35.0, 0.02, 300.0, 0, 1, partition=(0, 9))      # more ranks than nodes
    with pytest.raises(HeomError):
        parts[0].set_option("order", 0)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from paper_1803_03498_b200.sharded import halo_all_to_all
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = Heom(np.zeros((3, 3)), 35.0, 0.02, 300.0, 1, 5, partition=(rank, world))
    gid, sc, rc, idx = g.partition_plan()
    n_own = g.owned()
    ok = True
    for rnd in range(2):                                            # two rounds: the plan is reusable
        buf = torch.full((g.nodes, 4), -1.0, dtype=torch.float64)
        buf[:n_own] = torch.from_numpy(gid[:n_own].astype(np.float64))[:, None] * (rnd + 1)
        send = buf[torch.from_numpy(idx.astype(np.int64))].contiguous() if idx.size else torch.empty((1, 4), dtype=torch.float64)
        halo_all_to_all(buf, send, n_own, sc, rc)
        ok = ok and bool(torch.equal(buf[:, 0], torch.from_numpy(gid.astype(np.float64)) * (rnd + 1)))
    # the slice halo through the same collective: payload = (global id, state) of every pair, twice per element
    from paper_1803_03498_b200.sharded import slice_all_to_all
    psc, prc, sn, ss, rn, rs = g.partition_plan_slices()
    per = 3                                                         # stands for N complex elements
    send = np.zeros((max(1, sn.size), per, 2))
    send[:sn.size, :, 0] = gid[sn][:, None]
    send[:sn.size, :, 1] = ss[:, None]
    recv = torch.full((max(1, rn.size) * per * 2,), -1.0, dtype=torch.float64)
    slice_all_to_all(recv, torch.from_numpy(send.reshape(-1)).contiguous(), per, psc, prc)
    got = recv.numpy().reshape(-1, per, 2)[:rn.size]
    ok = ok and np.array_equal(got[:, 0, 0], gid[rn].astype(np.float64)) and np.array_equal(got[:, 2, 1], rs.astype(np.float64))
    q.put((rank, bool(ok), int(g.nodes - n_own)))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_gloo(world):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=180) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(o[1] for o in out)
    assert all(o[2] > 0 for o in out)                               # every rank has ghosts
