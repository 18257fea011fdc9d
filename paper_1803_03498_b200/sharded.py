"""One hierarchy sharded over several GPUs: one process per GPU, halo exchange over NCCL.

The paper partitions the ADO graph into self-contained parts plus halo regions and exchanges the halos every
right-hand-side evaluation.  Here rank r owns a contiguous range of the lexicographic node order
(heom_create_partition); after every fused RHS + RK4-stage launch the rows other ranks hold as ghosts are packed by
a device kernel (heom_pack_halo) and sent with ONE all_to_all_single, received straight into the ghost rows of the
buffer the next stage reads (the local node order makes the ghost region the receive buffer: no unpack).
4 exchanges per RK4 step.  torch.distributed is plumbing only; every arithmetic step runs in the library's kernels.
"""
import numpy as np

from .binding import Heom


def halo_all_to_all(buf, send, n_owned, send_counts, recv_counts, group=None):
    """rows of `send` (grouped by destination rank) -> the ghost rows buf[n_owned:] of the peers (grouped by
    source rank): one all_to_all_single, received in place."""
    import torch.distributed as dist
    n_send = int(np.sum(send_counts))
    dist.all_to_all_single(buf[n_owned:], send[:n_send],
                           output_split_sizes=[int(c) for c in recv_counts],
                           input_split_sizes=[int(c) for c in send_counts], group=group)


def slice_all_to_all(recv, send, per, send_counts, recv_counts, group=None):
    """Slice halo: `per` complex128 per (node, state) pair; send / recv are flat float64 buffers of packed pairs
    grouped by destination / source rank.  One all_to_all_single."""
    import torch.distributed as dist
    n_send, n_recv = int(np.sum(send_counts)) * 2 * per, int(np.sum(recv_counts)) * 2 * per
    dist.all_to_all_single(recv[:n_recv], send[:n_send],
                           output_split_sizes=[int(c) * 2 * per for c in recv_counts],
                           input_split_sizes=[int(c) * 2 * per for c in send_counts], group=group)


class ShardedHeom:
    """Rank `rank` of `world`: a partition context + the exchange.  group=None: the default process group.
    halo = "slices" (default): only row s -- and column s for states that are not exactly Hermitian -- of every
    (ghost, state) pair a gather reads crosses the link (heom_pack_halo_slices / heom_unpack_halo_slices around one
    all_to_all_single); halo = "nodes": whole N x N ghost nodes, received in place (no unpack kernel)."""

    def __init__(self, H_cm, lambda_cm, nu_per_fs, T_kelvin, K, D, rank, world, device=0, bath_state=None,
                 group=None, halo="slices", **options):
        self.rank, self.world, self.group, self.halo = int(rank), int(world), group, halo
        self.g = Heom(H_cm, lambda_cm, nu_per_fs, T_kelvin, K, D, device=device, bath_state=bath_state,
                      partition=(rank, world), **options)
        self.n_owned = self.g.owned()
        self.global_ids, self.send_counts, self.recv_counts, self.send_idx = self.g.partition_plan()
        self.pair_send_counts, self.pair_recv_counts = self.g.partition_plan_slices()[:2]
        self._send = self._recv = None

    def bind(self, stream=None):
        import torch
        self.g.bind(stream=stream)
        dev = self.g._workspace.device
        if self.halo == "nodes":
            rows = max(1, int(self.send_counts.sum()))
            self._send = torch.empty((rows, 2 * self.g.N * self.g.N), dtype=torch.float64, device=dev)
        else:
            per = 2 * 2 * self.g.N          # float64 per pair at most (row + column, complex)
            self._send = torch.empty(max(1, int(self.pair_send_counts.sum())) * per, dtype=torch.float64, device=dev)
            self._recv = torch.empty(max(1, int(self.pair_recv_counts.sum())) * per, dtype=torch.float64, device=dev)
        return self

    def halo_bytes_per_stage(self):
        """Bytes this rank sends per stage with the halo in use (plan count, not a measurement)."""
        if self.halo == "nodes":
            return int(self.send_counts.sum()) * 16 * self.g.N * self.g.N
        return int(self.pair_send_counts.sum()) * 16 * self.g.halo_slice_elements()

    # -- state ----------------------------------------------------------------------------------
    def set_state(self, sigma0):
        self.g.set_state(sigma0)

    def owned_state(self):
        """(global pinned-order ids, states) of the nodes this rank owns."""
        full = self.g.get_full_state()
        return self.global_ids[:self.n_owned], full[:self.n_owned]

    def gather_state(self, total_nodes):
        """The whole state in the pinned order on every rank (small cases / tests): all_gather of the owned parts."""
        import torch.distributed as dist
        ids, st = self.owned_state()
        parts = [None] * self.world
        dist.all_gather_object(parts, (ids, st), group=self.group)
        out = np.empty((total_nodes, self.g.N, self.g.N), dtype=np.complex128)
        for i, s in parts:
            out[i] = s
        return out

    # -- propagation ----------------------------------------------------------------------------
    def exchange(self, stage):
        """Refresh the ghost rows of the buffer the next stage reads.  The library launches on the stream bound
        with heom_bind_workspace; torch.distributed orders the NCCL collective against torch's CURRENT stream --
        so the bound stream is made current here: the collective then runs after the pack kernel and before the
        next stage kernel, whatever stream the caller is on."""
        import torch
        with torch.cuda.stream(self.g._stream):
            ptr = self.g.stage_output(stage)
            if self.halo == "nodes":
                buf = self.g.buffer_view(ptr)
                if int(self.send_counts.sum()):
                    self.g.pack_halo(ptr, self._send.data_ptr())
                halo_all_to_all(buf, self._send, self.n_owned, self.send_counts, self.recv_counts, self.group)
            else:
                per = self.g.halo_slice_elements()
                self.g.pack_halo_slices(ptr, self._send.data_ptr())
                slice_all_to_all(self._recv, self._send, per, self.pair_send_counts, self.pair_recv_counts, self.group)
                self.g.unpack_halo_slices(self._recv.data_ptr(), ptr)

    def rk4_steps(self, dt_fs, nsteps):
        import torch
        with torch.cuda.stream(self.g._stream):
            for _ in range(int(nsteps)):
                for stage in range(4):
                    self.g.rk4_stage(dt_fs, stage)
                    if self.world > 1:
                        self.exchange(stage)

    def populations(self):
        """Eq. 26 from the rank's copy of sigma_0 (rank 0 owns it: the root is the first node of the order; ranks
        that hold neither it nor a ghost of it return zeros)."""
        from .binding import HeomError
        try:
            return self.g.populations()
        except HeomError as e:
            if e.status != -4:
                raise
            return np.zeros(self.g.N), 0j

    def __getattr__(self, name):
        # plumbing calls (sync, set_option, kernel_time, launch_count, kernel_name, ...) go to the partition context
        if name == "g":
            raise AttributeError(name)
        return getattr(self.g, name)


def slice_plan_check(parts):
    """Host-side consistency of the slice-halo plans (tests): the (node, state) pairs rank p sends to r are, pair
    for pair and in order, the pairs r expects from p.  parts[r] = (global_ids, plan_slices tuple)."""
    world = len(parts)
    for r in range(world):
        gid_r, (sc_r, rc_r, sn_r, ss_r, rn_r, rs_r) = parts[r]
        roff = 0
        for p in range(world):
            gid_p, (sc_p, rc_p, sn_p, ss_p, rn_p, rs_p) = parts[p]
            soff = int(sc_p[:r].sum())
            n = int(sc_p[r])
            if n != int(rc_r[p]):
                return False
            if not np.array_equal(gid_p[sn_p[soff:soff + n]], gid_r[rn_r[roff:roff + n]]):
                return False
            if not np.array_equal(ss_p[soff:soff + n], rs_r[roff:roff + n]):
                return False
            roff += n
    return True


def exchange_plan_check(plans):
    """Host-side consistency of the plans of all ranks (tests): what rank p sends to r is, node for node, what r
    expects from p.  plans[r] = (global_ids, n_owned, send_counts, recv_counts, send_idx)."""
    world = len(plans)
    for r in range(world):
        gid_r, own_r, sc_r, rc_r, idx_r = plans[r]
        goff = own_r
        for p in range(world):
            gid_p, own_p, sc_p, rc_p, idx_p = plans[p]
            soff = int(sc_p[:r].sum())
            sent = gid_p[idx_p[soff:soff + int(sc_p[r])]]
            want = gid_r[goff:goff + int(rc_r[p])]
            if sent.shape != want.shape or not np.array_equal(sent, want):
                return False
            goff += int(rc_r[p])
    return True
