"""Thin Python binding of include/heom.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libheom_b200.so; PyTorch is
used for the device workspace tensor and the stream, nothing else.  There is no CPU
fallback: if the library is missing or no GPU is present the calls raise.
This module never imports `oracle`.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libheom_b200.so")

HEOM_OK, HEOM_EINVAL, HEOM_ENOMEM, HEOM_ECUDA, HEOM_ESTATE = 0, -1, -2, -3, -4
_STATUS = {0: "HEOM_OK", -1: "HEOM_EINVAL", -2: "HEOM_ENOMEM", -3: "HEOM_ECUDA", -4: "HEOM_ESTATE"}

# every symbol include/heom.h declares (tests check the library exports all of them)
SYMBOLS = [
    "heom_create", "heom_create_sites", "heom_create_partition", "heom_partition_owned", "heom_partition_plan",
    "heom_rk4_stage", "heom_stage_output", "heom_pack_halo", "heom_num_baths", "heom_expectation", "heom_destroy", "heom_set_option", "heom_num_nodes", "heom_num_modes",
    "heom_get_tables", "heom_get_coefficients", "heom_workspace_bytes", "heom_bind_workspace",
    "heom_set_state", "heom_set_full_state", "heom_get_full_state", "heom_rhs", "heom_rk4_steps",
    "heom_sync", "heom_populations", "heom_launch_count", "heom_kernel_time", "heom_kernel_name",
    "heom_last_error", "heom_probe_peak", "heom_create_general", "heom_set_hamiltonian",
    "heom_level_max", "heom_partition_plan_slices", "heom_halo_slice_elements", "heom_pack_halo_slices", "heom_unpack_halo_slices",
    "heom_level_max_static", "heom_static_last_error",
]

_lib = None
import weakref  # noqa: E402
POISONED = weakref.WeakSet()   # contexts bound with poison=True (the test suite checks their guard bytes)


class HeomError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def load_library():
    """Load libheom_b200.so; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1803_03498_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    P, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.heom_create.argtypes = [C.POINTER(P), C.c_int, dp, dp, dp, C.c_double, C.c_int, C.c_int, C.c_int]
    lib.heom_create_sites.argtypes = [C.POINTER(P), C.c_int, dp, C.c_int, C.POINTER(C.c_int), dp, dp, C.c_double,
                                      C.c_int, C.c_int, C.c_int]
    lib.heom_create_partition.argtypes = [C.POINTER(P), C.c_int, dp, C.c_int, C.POINTER(C.c_int), dp, dp, C.c_double,
                                          C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
    lib.heom_create_general.argtypes = [C.POINTER(P), C.c_int, dp, dp, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                        dp, dp, C.c_double, C.c_int, C.c_int, C.c_int]
    lib.heom_set_hamiltonian.argtypes = [P, dp, dp]
    lib.heom_partition_owned.argtypes = [P]
    lib.heom_partition_owned.restype = C.c_int64
    lib.heom_partition_plan.argtypes = [P, P, P, P, P]
    lib.heom_level_max.argtypes = [P, P]
    lib.heom_partition_plan_slices.argtypes = [P, P, P, P, P, P, P]
    lib.heom_halo_slice_elements.argtypes = [P]
    lib.heom_pack_halo_slices.argtypes = [P, P, P]
    lib.heom_unpack_halo_slices.argtypes = [P, P, P]
    lib.heom_rk4_stage.argtypes = [P, C.c_double, C.c_int]
    lib.heom_stage_output.argtypes = [P, C.c_int, C.POINTER(P)]
    lib.heom_pack_halo.argtypes = [P, P, P]
    lib.heom_num_baths.argtypes = [P]
    lib.heom_expectation.argtypes = [P, P, P, P]
    lib.heom_destroy.argtypes = [P]
    lib.heom_destroy.restype = None
    lib.heom_set_option.argtypes = [P, C.c_char_p, C.c_int]
    lib.heom_num_nodes.argtypes = [P]
    lib.heom_num_nodes.restype = C.c_int64
    lib.heom_num_modes.argtypes = [P]
    lib.heom_get_tables.argtypes = [P, P, P, P]
    lib.heom_get_coefficients.argtypes = [P, P, P, P, P]
    lib.heom_workspace_bytes.argtypes = [P]
    lib.heom_workspace_bytes.restype = C.c_size_t
    lib.heom_bind_workspace.argtypes = [P, P, C.c_size_t, P]
    lib.heom_set_state.argtypes = [P, P]
    lib.heom_set_full_state.argtypes = [P, P]
    lib.heom_get_full_state.argtypes = [P, P]
    lib.heom_rhs.argtypes = [P, P]
    lib.heom_rk4_steps.argtypes = [P, C.c_double, C.c_int]
    lib.heom_sync.argtypes = [P]
    lib.heom_populations.argtypes = [P, P, P, P]
    lib.heom_launch_count.argtypes = [P]
    lib.heom_launch_count.restype = C.c_int64
    lib.heom_kernel_time.argtypes = [P, P, P]
    lib.heom_kernel_name.argtypes = [P]
    lib.heom_kernel_name.restype = C.c_char_p
    lib.heom_last_error.argtypes = [P]
    lib.heom_last_error.restype = C.c_char_p
    lib.heom_probe_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
    lib.heom_level_max_static.argtypes = [C.c_int, P, P, C.c_int64, C.c_int, C.c_int, P, P]
    lib.heom_static_last_error.argtypes = []
    lib.heom_static_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def probe_peak(kind, device=0):
    """heom_probe_peak: measured FP64 FMA ("dfma") / FP64 tensor-core ("dmma") peak in TFLOP/s, or HBM copy
    bandwidth ("hbm") in GB/s, of `device`."""
    lib = load_library()
    v = C.c_double()
    rc = lib.heom_probe_peak(int(device), {"dfma": 0, "dmma": 1, "hbm": 2}[kind], C.byref(v))
    if rc != 0:
        raise HeomError(rc, "heom_probe_peak failed (no CUDA device?)")
    return v.value


STATIC_MAX_DEPTH = 63   # HEOM_STATIC_MAX_DEPTH


def level_max_static(state_ptr, level_ptr, nodes, elems_per_node, depth, out_ptr, device=0, cuda_stream=0):
    """heom_level_max_static: the per-level growth monitor without any allocation (scratch in a static device
    array, depth <= STATIC_MAX_DEPTH).  All pointers are DEVICE addresses; stream-ordered, does not synchronise."""
    lib = load_library()
    rc = lib.heom_level_max_static(int(device), int(state_ptr), int(level_ptr), int(nodes), int(elems_per_node),
                                   int(depth), int(out_ptr), int(cuda_stream))
    if rc != 0:
        raise HeomError(rc, lib.heom_static_last_error().decode())


class Heom:
    """One truncated hierarchy bound to one GPU stream.  Mirrors include/heom.h one to one."""

    def __init__(self, H_cm, lambda_cm, nu_per_fs, T_kelvin, K, D, device=0, bath_state=None, partition=None,
                 bath_states=None, **options):
        """bath_state=None: heom_create (one bath per state); else heom_create_sites with the listed states
        (lambda_cm, nu_per_fs then have one entry per bath).  partition=(rank, world): heom_create_partition --
        this context holds rank's part of the hierarchy (owned + ghost nodes).
        bath_states = list of lists (bath b couples to every state of bath_states[b]) and/or a complex H_cm:
        heom_create_general."""
        self._lib = load_library()
        self._h = None
        Hc = np.asarray(H_cm)
        H = np.ascontiguousarray(Hc.real, dtype=np.float64)
        Him = np.ascontiguousarray(Hc.imag, dtype=np.float64) if np.iscomplexobj(Hc) else None
        if H.ndim != 2 or H.shape[0] != H.shape[1]:
            raise ValueError("H_cm must be square")
        self.N = H.shape[0]
        self.B = len(bath_states) if bath_states is not None else self.N if bath_state is None else len(bath_state)
        lam = np.ascontiguousarray(np.broadcast_to(lambda_cm, (self.B,)), dtype=np.float64)
        nu = np.ascontiguousarray(np.broadcast_to(nu_per_fs, (self.B,)), dtype=np.float64)
        h = C.c_void_p()
        self.partition = partition
        if bath_states is not None or Him is not None:
            if partition is not None:
                raise ValueError("general contexts are single-GPU")
            if bath_states is None:
                bath_states = [[b] for b in (range(self.N) if bath_state is None else bath_state)]
            ptr = np.concatenate([[0], np.cumsum([len(x) for x in bath_states])]).astype(np.int32)
            flat = np.array([int(q) for x in bath_states for q in x], dtype=np.int32)
            rc = self._lib.heom_create_general(C.byref(h), self.N, _dptr(H), _dptr(Him) if Him is not None else None,
                                               self.B, ptr.ctypes.data_as(C.POINTER(C.c_int)),
                                               flat.ctypes.data_as(C.POINTER(C.c_int)), _dptr(lam), _dptr(nu),
                                               float(T_kelvin), int(K), int(D), int(device))
        elif partition is not None:
            states = list(range(self.N)) if bath_state is None else bath_state
            bs = (C.c_int * self.B)(*[int(x) for x in states])
            rc = self._lib.heom_create_partition(C.byref(h), self.N, _dptr(H), self.B, bs, _dptr(lam), _dptr(nu),
                                                 float(T_kelvin), int(K), int(D), int(device),
                                                 int(partition[0]), int(partition[1]))
        elif bath_state is None:
            rc = self._lib.heom_create(C.byref(h), self.N, _dptr(H), _dptr(lam), _dptr(nu),
                                       float(T_kelvin), int(K), int(D), int(device))
        else:
            bs = (C.c_int * self.B)(*[int(x) for x in bath_state])
            rc = self._lib.heom_create_sites(C.byref(h), self.N, _dptr(H), self.B, bs, _dptr(lam), _dptr(nu),
                                             float(T_kelvin), int(K), int(D), int(device))
        if rc != 0:
            raise HeomError(rc, "heom_create rejected its arguments")
        self._h = h
        self.K, self.D, self.device = int(K), int(D), int(device)
        self.nodes = int(self._lib.heom_num_nodes(h))
        self.W = int(self._lib.heom_num_modes(h))
        self._workspace = None
        self._stream = None
        for k, v in options.items():
            self.set_option(k, v)

    # -- plumbing -------------------------------------------------------------------------
    def _ck(self, rc):
        if rc != 0:
            raise HeomError(rc, self._lib.heom_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.heom_destroy(self._h)
            self._h = None
        self._workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, name, value):
        self._ck(self._lib.heom_set_option(self._h, name.encode(), int(value)))

    # -- host tables ----------------------------------------------------------------------
    def tables(self):
        t = np.empty((self.nodes, self.W), dtype=np.uint8)
        p = np.empty((self.nodes, self.W), dtype=np.int32)
        m = np.empty((self.nodes, self.W), dtype=np.int32)
        self._ck(self._lib.heom_get_tables(self._h, t.ctypes.data, p.ctypes.data, m.ctypes.data))
        return t, p, m

    def coefficients(self):
        g = np.empty(self.W); cr = np.empty(self.W); ci = np.empty(self.W); d = np.empty(self.B)
        self._ck(self._lib.heom_get_coefficients(self._h, g.ctypes.data, cr.ctypes.data,
                                                 ci.ctypes.data, d.ctypes.data))
        return g, cr, ci, d

    # -- device workspace -----------------------------------------------------------------
    def workspace_bytes(self):
        return int(self._lib.heom_workspace_bytes(self._h))

    def bind(self, stream=None, poison=False):
        """Allocate the workspace as a torch tensor on `device` and bind it (PyTorch = memory + stream).
        poison=True fills it with 0xFF bytes (NaNs, index -1) first, so that a read of memory the library never
        wrote shows up in the results (tests)."""
        import torch
        if not torch.cuda.is_available():
            raise HeomError(HEOM_ECUDA, "no CUDA device: the HEOM path has no CPU fallback")
        dev = torch.device("cuda", self.device)
        nbytes = self.workspace_bytes()
        self._workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        if poison:
            self._workspace.fill_(255)
            torch.cuda.synchronize(dev)
            POISONED.add(self)
        ptr = (self._workspace.data_ptr() + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(dev)
        self._ws_end = ptr - self._workspace.data_ptr() + nbytes
        self._ck(self._lib.heom_bind_workspace(self._h, ptr, nbytes, self._stream.cuda_stream))
        return self

    def workspace_guard_intact(self):
        """After bind(poison=True): the slack bytes behind heom_workspace_bytes() still hold the poison pattern,
        i.e. nothing wrote past the end of the workspace (tests)."""
        import torch
        if self._workspace is None:
            return True
        torch.cuda.synchronize(self._workspace.device)
        tail = self._workspace[self._ws_end:]
        return bool(tail.numel() > 0 and (tail == 255).all().item())

    def bind_raw(self, dev_ptr, nbytes, cuda_stream=0):
        self._ck(self._lib.heom_bind_workspace(self._h, dev_ptr, nbytes, cuda_stream))

    # -- state ----------------------------------------------------------------------------
    def set_state(self, sigma0):
        s = np.ascontiguousarray(sigma0, dtype=np.complex128)
        if s.shape != (self.N, self.N):
            raise ValueError("sigma0 must be N x N")
        self._ck(self._lib.heom_set_state(self._h, s.ctypes.data))

    def set_full_state(self, sigma):
        s = np.ascontiguousarray(sigma, dtype=np.complex128)
        if s.shape != (self.nodes, self.N, self.N):
            raise ValueError("sigma must be [nodes][N][N]")
        self._ck(self._lib.heom_set_full_state(self._h, s.ctypes.data))

    def get_full_state(self, out=None):
        if out is None:
            out = np.empty((self.nodes, self.N, self.N), dtype=np.complex128)
        self._ck(self._lib.heom_get_full_state(self._h, out.ctypes.data))
        return out

    def rhs(self, out=None):
        if out is None:
            out = np.empty((self.nodes, self.N, self.N), dtype=np.complex128)
        self._ck(self._lib.heom_rhs(self._h, out.ctypes.data))
        return out

    def rk4_steps(self, dt_fs, nsteps):
        self._ck(self._lib.heom_rk4_steps(self._h, float(dt_fs), int(nsteps)))

    def set_hamiltonian(self, H_cm):
        """heom_set_hamiltonian: replace H (complex Hermitian allowed on contexts created with a complex H)."""
        Hc = np.asarray(H_cm)
        re = np.ascontiguousarray(Hc.real, dtype=np.float64)
        im = np.ascontiguousarray(Hc.imag, dtype=np.float64) if np.iscomplexobj(Hc) else None
        self._ck(self._lib.heom_set_hamiltonian(self._h, _dptr(re), _dptr(im) if im is not None else None))

    def rk4_step_td(self, dt_fs, H0, Hm, H1):
        """One RK4 step with a time-dependent Hamiltonian H(t) = H0, H(t + dt/2) = Hm, H(t + dt) = H1 (heom.h:
        heom_set_hamiltonian + heom_rk4_stage; needs option rk4_form = 0).  Argument marshalling only."""
        self.set_hamiltonian(H0); self.rk4_stage(dt_fs, 0)
        self.set_hamiltonian(Hm); self.rk4_stage(dt_fs, 1); self.rk4_stage(dt_fs, 2)
        self.set_hamiltonian(H1); self.rk4_stage(dt_fs, 3)

    def sync(self):
        self._ck(self._lib.heom_sync(self._h))

    def populations(self):
        pop = np.empty(self.N)
        tr = C.c_double(), C.c_double()
        self._ck(self._lib.heom_populations(self._h, pop.ctypes.data, C.addressof(tr[0]),
                                            C.addressof(tr[1])))
        return pop, complex(tr[0].value, tr[1].value)

    # -- partitions (one hierarchy over several GPUs) -----------------------------------------
    def owned(self):
        return int(self._lib.heom_partition_owned(self._h))

    def partition_plan(self):
        """(global_ids [local nodes], send_counts [world], recv_counts [world], send_idx [sum send_counts])."""
        world = self.partition[1]
        gid = np.empty(self.nodes, dtype=np.int64)
        sc = np.empty(world, dtype=np.int64); rc_ = np.empty(world, dtype=np.int64)
        self._ck(self._lib.heom_partition_plan(self._h, gid.ctypes.data, sc.ctypes.data, rc_.ctypes.data, None))
        idx = np.empty(int(sc.sum()), dtype=np.int32)
        self._ck(self._lib.heom_partition_plan(self._h, None, None, None, idx.ctypes.data if idx.size else None))
        return gid, sc, rc_, idx

    def partition_plan_slices(self):
        """(send_counts, recv_counts, send_node, send_state, recv_node, recv_state) of the slice halo."""
        world = self.partition[1]
        sc = np.empty(world, dtype=np.int64); rc_ = np.empty(world, dtype=np.int64)
        self._ck(self._lib.heom_partition_plan_slices(self._h, sc.ctypes.data, rc_.ctypes.data, None, None, None, None))
        sn = np.empty(int(sc.sum()), dtype=np.int32); ss = np.empty_like(sn)
        rn = np.empty(int(rc_.sum()), dtype=np.int32); rs = np.empty_like(rn)
        self._ck(self._lib.heom_partition_plan_slices(self._h, None, None, sn.ctypes.data if sn.size else None,
                                                      ss.ctypes.data if ss.size else None,
                                                      rn.ctypes.data if rn.size else None,
                                                      rs.ctypes.data if rs.size else None))
        return sc, rc_, sn, ss, rn, rs

    def halo_slice_elements(self):
        return int(self._lib.heom_halo_slice_elements(self._h))

    def pack_halo_slices(self, src_ptr, dst_ptr):
        self._ck(self._lib.heom_pack_halo_slices(self._h, int(src_ptr), int(dst_ptr)))

    def unpack_halo_slices(self, src_ptr, state_ptr):
        self._ck(self._lib.heom_unpack_halo_slices(self._h, int(src_ptr), int(state_ptr)))

    def rk4_stage(self, dt_fs, stage):
        self._ck(self._lib.heom_rk4_stage(self._h, float(dt_fs), int(stage)))

    def stage_output(self, stage):
        """Device pointer of the buffer whose ghost rows must be refreshed after `stage`."""
        ptr = C.c_void_p()
        self._ck(self._lib.heom_stage_output(self._h, int(stage), C.byref(ptr)))
        return int(ptr.value)

    def pack_halo(self, src_ptr, dst_ptr):
        self._ck(self._lib.heom_pack_halo(self._h, int(src_ptr), int(dst_ptr)))

    def buffer_view(self, dev_ptr):
        """torch view [local nodes][2 N N] float64 of a state buffer inside the bound workspace tensor."""
        import torch
        off = int(dev_ptr) - self._workspace.data_ptr()
        nbytes = self.nodes * self.N * self.N * 16
        return self._workspace[off:off + nbytes].view(torch.float64).view(self.nodes, 2 * self.N * self.N)

    def level_max(self):
        """heom_level_max: max(|Re|, |Im|) over the nodes of every hierarchy level, L = 0..D."""
        out = np.zeros(self.D + 1)
        self._ck(self._lib.heom_level_max(self._h, out.ctypes.data))
        return out

    def expectation(self, A):
        """Tr(A sigma_0) (heom_expectation)."""
        a = np.ascontiguousarray(A, dtype=np.complex128)
        if a.shape != (self.N, self.N):
            raise ValueError("A must be N x N")
        v = C.c_double(), C.c_double()
        self._ck(self._lib.heom_expectation(self._h, a.ctypes.data, C.addressof(v[0]), C.addressof(v[1])))
        return complex(v[0].value, v[1].value)

    # -- introspection --------------------------------------------------------------------
    def launch_count(self):
        return int(self._lib.heom_launch_count(self._h))

    def kernel_time(self):
        ms, n = C.c_double(), C.c_int64()
        self._ck(self._lib.heom_kernel_time(self._h, C.addressof(ms), C.addressof(n)))
        return ms.value, n.value

    def kernel_name(self):
        return self._lib.heom_kernel_name(self._h).decode()
