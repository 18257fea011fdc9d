"""-m gpu: the sharded path (heom_create_partition + stage-wise stepping + halo exchange) on ONE GPU.

The `world` partition contexts live in one process and are advanced one after the other, stage by stage; the
exchange between them is the same pack kernel (heom_pack_halo) followed by device copies of exactly the rows
halo_all_to_all would move (no rank waits on another inside a kernel).  The union of the owned rows is compared
with the oracle's global state."""
import numpy as np
import pytest
import torch

import workloads
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu
STATE_TOL = 1e-10
RHS_TOL = 1e-13


def rel_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


class LocalWorld:
    def __init__(self, w, world, bath_state=None, halo="nodes", **opts):
        from paper_1803_03498_b200 import Heom
        self.world, self.halo = world, halo
        self.parts = [Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, partition=(r, world),
                           bath_state=bath_state, **opts).bind(poison=True) for r in range(world)]
        self.plans = [g.partition_plan() for g in self.parts]
        self.send = [torch.full((max(1, int(p[1].sum())), 2 * g.N * g.N), float("nan"), dtype=torch.float64, device="cuda")
                     for g, p in zip(self.parts, self.plans)]
        self.splans = [g.partition_plan_slices() for g in self.parts]
        self.ssend = [torch.full((max(1, int(p[0].sum())) * 4 * g.N,), float("nan"), dtype=torch.float64, device="cuda")
                      for g, p in zip(self.parts, self.splans)]
        self.srecv = [torch.full((max(1, int(p[1].sum())) * 4 * g.N,), float("nan"), dtype=torch.float64, device="cuda")
                      for g, p in zip(self.parts, self.splans)]

    def exchange_slices(self, ptrs):
        """What ShardedHeom.exchange does with halo="slices": pack, move exactly the packed pairs, unpack."""
        for g, s, p in zip(self.parts, self.ssend, ptrs):
            g.pack_halo_slices(p, s.data_ptr())
        torch.cuda.synchronize()
        for r, g in enumerate(self.parts):
            per = 2 * g.halo_slice_elements()                       # float64 per pair
            roff = 0
            for p in range(self.world):
                n = int(self.splans[r][1][p]) * per
                soff = int(self.splans[p][0][:r].sum()) * per
                assert n == int(self.splans[p][0][r]) * per
                self.srecv[r][roff:roff + n] = self.ssend[p][soff:soff + n]
                roff += n
            g.unpack_halo_slices(self.srecv[r].data_ptr(), ptrs[r])
        torch.cuda.synchronize()

    def exchange(self, ptrs):
        if self.halo == "slices":
            return self.exchange_slices(ptrs)
        for g, s, p in zip(self.parts, self.send, ptrs):
            if g.partition_plan()[1].sum():
                g.pack_halo(p, s.data_ptr())
        torch.cuda.synchronize()
        for r, g in enumerate(self.parts):
            buf = g.buffer_view(ptrs[r])
            goff = g.owned()
            for p in range(self.world):
                n = int(self.plans[r][2][p])                      # recv_counts[p]
                soff = int(self.plans[p][1][:r].sum())            # where p's rows for r start in p's send buffer
                assert n == int(self.plans[p][1][r])
                buf[goff:goff + n] = self.send[p][soff:soff + n]
                goff += n
        torch.cuda.synchronize()

    def set_state(self, s0):
        for g in self.parts:
            g.set_state(s0)

    def set_full_state(self, st):
        for g, p in zip(self.parts, self.plans):
            g.set_full_state(st[p[0]])

    def rk4_steps(self, dt, n):
        for _ in range(n):
            for stage in range(4):
                for g in self.parts:
                    g.rk4_stage(dt, stage)
                self.exchange([g.stage_output(stage) for g in self.parts])

    def gather(self, getter, total):
        out = None
        for g, p in zip(self.parts, self.plans):
            loc = getter(g)
            if out is None:
                out = np.empty((total,) + loc.shape[1:], dtype=loc.dtype)
            out[p[0][:g.owned()]] = loc[:g.owned()]
        return out


@pytest.mark.parametrize("name,D,steps,world", [("cfg2", 4, 100, 2), ("cfg2", 4, 60, 5), ("cfg3", 5, 60, 3),
                                                ("cfg4", 3, 60, 4), ("cfg5", 1, 20, 2), ("cfg5", 2, 2, 3),
                                                ("cfg1", 4, 200, 3)])
@pytest.mark.parametrize("herm,form,halo", [(1, -1, "slices"), (0, -1, "slices"), (1, 0, "nodes")])
def test_sharded_rk4_parity(name, D, steps, world, herm, form, halo):
    w = workloads.get(name).with_(D=D)
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
    lw = LocalWorld(w, world, halo=halo, hermitian=herm, rk4_form=form)
    assert sum(g.owned() for g in lw.parts) == o.nodes
    # a single right-hand side on a dense random state first (ghost rows of the result are not meaningful)
    st = workloads.random_state(o.nodes, w.N, seed=5)
    o.set_full_state(st); lw.set_full_state(st)
    assert rel_err(lw.gather(lambda g: g.rhs(), o.nodes), o.rhs()) < RHS_TOL
    o.set_state(w.sigma0()); lw.set_state(w.sigma0())
    o.rk4_steps(w.dt_fs, steps); lw.rk4_steps(w.dt_fs, steps)
    ref = o.get_full_state()
    got = lw.gather(lambda g: g.get_full_state(), o.nodes)
    assert rel_err(got, ref) < STATE_TOL
    pop, tr = lw.parts[0].populations()                             # rank 0 owns sigma_0
    assert abs(tr - 1.0) < 1e-11 and np.allclose(pop, np.diag(ref[0]).real, atol=1e-11)
    # ghost copies agree with their owners' rows after the last exchange (whole-node halo; the slice halo
    # refreshes only the rows and columns the gathers read)
    for g, p in zip(lw.parts, lw.plans):
        if halo == "nodes":
            loc = g.get_full_state()
            assert rel_err(loc, ref[p[0]]) < STATE_TOL
        assert g.workspace_guard_intact()                           # nothing wrote past the workspace


def test_sharded_world_1_equals_plain():
    from paper_1803_03498_b200 import Heom
    w = workloads.fmo_like().with_(D=3)
    a = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D).bind()
    b = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, partition=(0, 1)).bind()
    a.set_state(w.sigma0()); b.set_state(w.sigma0())
    a.rk4_steps(1.0, 50); b.rk4_steps(1.0, 50)                     # world 1: rk4_steps is allowed
    gid = b.partition_plan()[0]
    assert np.array_equal(b.get_full_state(), a.get_full_state()[gid])


def test_partition_refuses_unsplit_stepping():
    from paper_1803_03498_b200 import Heom, HeomError
    w = workloads.dimer()
    g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, partition=(1, 2)).bind()
    g.set_state(w.sigma0())
    with pytest.raises(HeomError) as e:
        g.rk4_steps(1.0, 1)
    assert e.value.status == -4


def test_sharded_class_nccl_world_1():
    """ShardedHeom end to end through torch.distributed NCCL with a one-rank group on the one GPU there is: the
    exchange call (views of the workspace tensor, split lists, in-place receive) is issued after every stage."""
    import os
    import socket
    import torch.distributed as dist
    from paper_1803_03498_b200.sharded import ShardedHeom
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        w = workloads.fmo_like().with_(D=3)
        o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
        sh = ShardedHeom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, 0, 1).bind()
        assert sh.n_owned == o.nodes and sh.send_counts.sum() == 0
        o.set_state(w.sigma0()); sh.set_state(w.sigma0())
        for _ in range(40):
            for stage in range(4):
                sh.g.rk4_stage(w.dt_fs, stage)
                sh.exchange(stage)                                  # nothing to move, but the collective runs
        o.rk4_steps(w.dt_fs, 40)
        got = sh.gather_state(o.nodes)
        assert rel_err(got, o.get_full_state()) < STATE_TOL
        pop, tr = sh.populations()
        assert abs(tr - 1.0) < 1e-12
    finally:
        dist.destroy_process_group()


def test_partition_launch_cost_follows_owned_rows():
    """A partition launches over its owned rows only: on config 2 split 4 ways, rank 2 (1.44 ghosts per owned node)
    must cost about a quarter of the full launch, not (1 + 1.44)/4 of it.  Prints the times."""
    from paper_1803_03498_b200 import Heom
    w = workloads.fmo_like()

    def stage_ms(g, reps=40):
        g.set_state(w.sigma0())
        for s in range(4):
            g.rk4_stage(w.dt_fs, s)                                 # warm-up (ghost rows stay as they are: timing only)
        g.sync()
        g.set_option("timing", 1); g.kernel_time()
        for _ in range(reps):
            for s in range(4):
                g.rk4_stage(w.dt_fs, s)
        ms, n = g.kernel_time()
        g.set_option("timing", 0)
        return ms / n

    full = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, ket=0).bind()
    t_full = stage_ms(full)
    full.close()
    out = []
    for world, rank in ((2, 1), (4, 2), (8, 4)):
        g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, partition=(rank, world)).bind()
        t = stage_ms(g)
        out.append((world, rank, g.owned(), g.nodes - g.owned(), t))
        g.close()
    print(f"\nPARTITION_COST cfg2 full launch {t_full*1e3:.1f} us; " +
          "; ".join(f"world {wd} rank {r}: owned {o} ghosts {gh} launch {t*1e3:.1f} us ({t/t_full:.2f} of full, ideal {1/wd:.2f})"
                    for wd, r, o, gh, t in out))
    for wd, r, o, gh, t in out:
        assert t < (1.0 / wd + 0.5 * gh / (o + gh) / wd + 0.12) * t_full


def _nccl_worker(rank, world, port, halo, q):
    """One rank of the multi-GPU parity run: its own GPU, NCCL, ShardedHeom against the oracle."""
    import os
    import torch
    import torch.distributed as dist
    from paper_1803_03498_b200.sharded import ShardedHeom
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        w = workloads.fmo_like().with_(D=4)
        sh = ShardedHeom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, rank, world, device=rank,
                         halo=halo).bind()
        sh.set_state(w.sigma0())
        sh.rk4_steps(w.dt_fs, 60)
        got = sh.gather_state(w.nodes)
        pop, tr = sh.populations() if rank == 0 else (None, None)
        if rank == 0:
            o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
            o.set_state(w.sigma0()); o.rk4_steps(w.dt_fs, 60)
            q.put((float(rel_err(got, o.get_full_state())), float(abs(tr - 1.0))))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("halo", ["slices", "nodes"])
def test_sharded_nccl_two_gpus(halo):
    """ONE hierarchy over two GPUs through NCCL (one process per GPU): stage-wise stepping with the halo exchange
    after every stage, final state of all ranks against the oracle.  Needs two GPUs: skipped on the one-GPU boxes
    this repository has been measured on (the exchange logic is covered there by the one-GPU emulation above and
    by the gloo world-size-2/3 tests of test_partition_host.py)."""
    import socket
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_nccl_worker, args=(r, 2, port, halo, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(600)
        assert p.exitcode == 0
    err, dtr = q.get(timeout=10)
    assert err < STATE_TOL and dtr < 1e-11
