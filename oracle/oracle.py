"""ctypes binding of the CPU oracle (oracle/libheom_oracle.so).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports
nothing from the CUDA package.
"""
import ctypes as C
import os

import numpy as np

from . import build_oracle

_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    path = build_oracle.build()
    lib = C.CDLL(path)
    P = C.c_void_p
    dp = C.POINTER(C.c_double)
    lib.oracle_create.argtypes = [C.POINTER(P), C.c_int, dp, dp, dp, C.c_double, C.c_int, C.c_int]
    lib.oracle_create.restype = C.c_int
    lib.oracle_create_sites.argtypes = [C.POINTER(P), C.c_int, dp, C.c_int, C.POINTER(C.c_int), dp, dp,
                                        C.c_double, C.c_int, C.c_int]
    lib.oracle_create_sites.restype = C.c_int
    lib.oracle_create_general.argtypes = [C.POINTER(P), C.c_int, dp, dp, C.c_int, C.POINTER(C.c_int),
                                          C.POINTER(C.c_int), dp, dp, C.c_double, C.c_int, C.c_int]
    lib.oracle_create_general.restype = C.c_int
    lib.oracle_set_hamiltonian.argtypes = [P, dp, dp]
    lib.oracle_rk4_step_td.argtypes = [P, C.c_double, dp, dp, dp, dp, dp, dp]
    lib.oracle_destroy.argtypes = [P]
    lib.oracle_destroy.restype = None
    lib.oracle_set_option.argtypes = [P, C.c_char_p, C.c_int]
    lib.oracle_num_nodes.argtypes = [P]
    lib.oracle_num_nodes.restype = C.c_int64
    lib.oracle_num_modes.argtypes = [P]
    lib.oracle_num_threads.argtypes = [P]
    lib.oracle_get_tables.argtypes = [P, P, P, P]
    lib.oracle_get_coefficients.argtypes = [P, P, P, P, P]
    lib.oracle_set_state.argtypes = [P, P]
    lib.oracle_set_full_state.argtypes = [P, P]
    lib.oracle_get_full_state.argtypes = [P, P]
    lib.oracle_rhs.argtypes = [P, P]
    lib.oracle_rhs_nodes.argtypes = [P, P, C.c_int64, P]
    lib.oracle_rk4_steps.argtypes = [P, C.c_double, C.c_int]
    lib.oracle_populations.argtypes = [P, P, P, P]
    lib.oracle_pade_poles.argtypes = [C.c_int, P, P]
    _lib = lib
    return lib


def pade_poles(K):
    """(xi, eta) of the [K-1/K] Pade decomposition of the Bose function (heom_oracle.h)."""
    lib = _load()
    xi = np.empty(K); eta = np.empty(K)
    if lib.oracle_pade_poles(int(K), xi.ctypes.data, eta.ctypes.data) != 0:
        raise ValueError("oracle_pade_poles failed")
    return xi, eta


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """One truncated hierarchy on the CPU.  Arguments as heom_oracle.h."""

    def __init__(self, H_cm, lambda_cm, nu_per_fs, T_kelvin, K, D, scaling=1, terminator=1,
                 threads=0, pade=0, bath_state=None, bath_states=None, terminator_form=0):
        """bath_state=None: one bath per state (oracle_create); else a list of the states the baths couple
        to (oracle_create_sites), lambda_cm / nu_per_fs then have one entry per bath.
        bath_states = list of lists: bath b couples to every state of bath_states[b] (oracle_create_general);
        H_cm may then be complex Hermitian."""
        lib = _load()
        Hc = np.asarray(H_cm)
        H = np.ascontiguousarray(Hc.real, dtype=np.float64)
        Him = np.ascontiguousarray(Hc.imag, dtype=np.float64) if np.iscomplexobj(Hc) else None
        self.N = H.shape[0]
        self.B = len(bath_states) if bath_states is not None else self.N if bath_state is None else len(bath_state)
        lam = np.ascontiguousarray(np.broadcast_to(lambda_cm, (self.B,)), dtype=np.float64)
        nu = np.ascontiguousarray(np.broadcast_to(nu_per_fs, (self.B,)), dtype=np.float64)
        h = C.c_void_p()
        if bath_states is not None or Him is not None:
            if bath_states is None:
                bath_states = [[b] for b in (range(self.N) if bath_state is None else bath_state)]
            ptr = np.concatenate([[0], np.cumsum([len(x) for x in bath_states])]).astype(np.int32)
            flat = np.array([s for x in bath_states for s in x], dtype=np.int32)
            rc = lib.oracle_create_general(C.byref(h), self.N, _dptr(H), _dptr(Him) if Him is not None else None,
                                           self.B, ptr.ctypes.data_as(C.POINTER(C.c_int)),
                                           flat.ctypes.data_as(C.POINTER(C.c_int)), _dptr(lam), _dptr(nu),
                                           float(T_kelvin), int(K), int(D))
        elif bath_state is None:
            rc = lib.oracle_create(C.byref(h), self.N, _dptr(H), _dptr(lam), _dptr(nu),
                                   float(T_kelvin), int(K), int(D))
        else:
            bs = (C.c_int * self.B)(*[int(x) for x in bath_state])
            rc = lib.oracle_create_sites(C.byref(h), self.N, _dptr(H), self.B, bs, _dptr(lam), _dptr(nu),
                                         float(T_kelvin), int(K), int(D))
        if rc != 0:
            raise ValueError(f"oracle_create failed with status {rc}")
        self._h = h
        self._lib = lib
        self.K, self.D = int(K), int(D)
        self.nodes = int(lib.oracle_num_nodes(h))
        self.W = int(lib.oracle_num_modes(h))
        for name, v in (("scaling", scaling), ("terminator", terminator), ("threads", threads), ("pade", pade),
                        ("terminator_form", terminator_form)):
            self._ck(lib.oracle_set_option(h, name.encode(), int(v)))

    def _ck(self, rc):
        if rc != 0:
            raise RuntimeError(f"oracle call failed with status {rc}")

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    @property
    def threads(self):
        return int(self._lib.oracle_num_threads(self._h))

    def tables(self):
        t = np.empty((self.nodes, self.W), dtype=np.uint8)
        p = np.empty((self.nodes, self.W), dtype=np.int32)
        m = np.empty((self.nodes, self.W), dtype=np.int32)
        self._ck(self._lib.oracle_get_tables(self._h, t.ctypes.data, p.ctypes.data, m.ctypes.data))
        return t, p, m

    def coefficients(self):
        g = np.empty(self.W); cr = np.empty(self.W); ci = np.empty(self.W); d = np.empty(self.B)
        self._ck(self._lib.oracle_get_coefficients(self._h, g.ctypes.data, cr.ctypes.data,
                                                   ci.ctypes.data, d.ctypes.data))
        return g, cr, ci, d

    def set_state(self, sigma0):
        s = np.ascontiguousarray(sigma0, dtype=np.complex128)
        assert s.shape == (self.N, self.N)
        self._ck(self._lib.oracle_set_state(self._h, s.ctypes.data))

    def set_full_state(self, sigma):
        s = np.ascontiguousarray(sigma, dtype=np.complex128)
        assert s.shape == (self.nodes, self.N, self.N)
        self._ck(self._lib.oracle_set_full_state(self._h, s.ctypes.data))

    def get_full_state(self):
        out = np.empty((self.nodes, self.N, self.N), dtype=np.complex128)
        self._ck(self._lib.oracle_get_full_state(self._h, out.ctypes.data))
        return out

    def rhs(self):
        out = np.empty((self.nodes, self.N, self.N), dtype=np.complex128)
        self._ck(self._lib.oracle_rhs(self._h, out.ctypes.data))
        return out

    def rhs_nodes(self, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        out = np.empty((ids.size, self.N, self.N), dtype=np.complex128)
        self._ck(self._lib.oracle_rhs_nodes(self._h, ids.ctypes.data, ids.size, out.ctypes.data))
        return out

    def rk4_steps(self, dt_fs, nsteps):
        self._ck(self._lib.oracle_rk4_steps(self._h, float(dt_fs), int(nsteps)))

    @staticmethod
    def _parts(H):
        Hc = np.asarray(H)
        re = np.ascontiguousarray(Hc.real, dtype=np.float64)
        im = np.ascontiguousarray(Hc.imag, dtype=np.float64) if np.iscomplexobj(Hc) else None
        return re, im

    def set_hamiltonian(self, H):
        re, im = self._parts(H)
        self._ck(self._lib.oracle_set_hamiltonian(self._h, _dptr(re), _dptr(im) if im is not None else None))

    def rk4_step_td(self, dt_fs, H0, Hm, H1):
        """One classical RK4 step with H(t) = H0, H(t + dt/2) = Hm, H(t + dt) = H1."""
        parts = [self._parts(H) for H in (H0, Hm, H1)]
        args = []
        for re, im in parts:
            args += [_dptr(re), _dptr(im) if im is not None else None]
        self._ck(self._lib.oracle_rk4_step_td(self._h, float(dt_fs), *args))

    def populations(self):
        pop = np.empty(self.N)
        tr = C.c_double(), C.c_double()
        self._ck(self._lib.oracle_populations(self._h, pop.ctypes.data, C.byref(tr[0]),
                                              C.byref(tr[1])))
        return pop, complex(tr[0].value, tr[1].value)

    def sigma0(self):
        """rho = sigma_0 (Eq. 26) as an N x N array (reads the full state; small cases)."""
        return self.get_full_state()[0]
