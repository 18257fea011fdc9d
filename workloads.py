"""Seeded synthetic inputs shaped like the paper's light-harvesting complexes.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path
(tests, bench.py).  It holds none of the method's arithmetic: it only draws
Hamiltonians, bath parameters, initial matrices and random test states.  It
imports neither `oracle` nor `paper_1803_03498_b200`.

The five configurations are BASELINE.json's `configs[0..4]`, stand-ins for the
paper's FMO workloads (Eq. 78: 7 sites, couplings 1-100 cm^-1, energy
spread ~400 cm^-1; Table 1: lambda = 35 cm^-1, 1/nu = 50 fs, Omega = 0;
P:443: T = 30..300 K; "more than 100 states" for supercomplexes).
Generator recipe: numpy PCG64 `default_rng(seed)`, draws in the
order written below, upper triangle row-major, then symmetrised.
"""
from dataclasses import dataclass, replace
from math import comb

import numpy as np

SEED_FMO = 1803034982      # configs 2 and 3 share one H (BASELINE.json)
SEED_LHCII = 1803034983
SEED_LARGE = 1803034984


@dataclass(frozen=True)
class Workload:
    name: str
    H_cm: np.ndarray          # [N][N] real symmetric, cm^-1
    lambda_cm: float          # reorganisation energy of every site's bath
    inv_nu_fs: float          # bath correlation time 1/nu_b, fs
    T_kelvin: float
    K: int                    # Matsubara terms beyond the Drude pole
    D: int                    # truncation depth
    dt_fs: float
    steps: int
    bath_state: tuple = None      # None: one bath per state; else the states the baths couple to (heom_create_sites)
    sigma0_matrix: np.ndarray = None   # None: |1><1|
    bath_states: tuple = None     # lists of states per bath (heom_create_general): S(b) >= 1, shared states

    @property
    def N(self):
        return self.H_cm.shape[0]

    @property
    def B(self):
        if self.bath_states is not None:
            return len(self.bath_states)
        return self.N if self.bath_state is None else len(self.bath_state)

    @property
    def W(self):
        return self.B * (self.K + 1)

    @property
    def nodes(self):
        return comb(self.W + self.D, self.D)

    @property
    def nu_per_fs(self):
        return 1.0 / self.inv_nu_fs

    @property
    def state_bytes(self):
        return 16 * self.N * self.N * self.nodes

    def with_(self, **kw):
        return replace(self, **kw)

    def sigma0(self):
        """sigma_0(0) = |1><1| (BASELINE.json: all configs)."""
        if self.sigma0_matrix is not None:
            return self.sigma0_matrix.astype(np.complex128)
        s = np.zeros((self.N, self.N), dtype=np.complex128)
        s[0, 0] = 1.0
        return s


def _symmetric_from_upper(N, diag, upper):
    H = np.zeros((N, N))
    iu = np.triu_indices(N, k=1)
    H[iu] = upper
    H = H + H.T
    H[np.diag_indices(N)] = diag
    return H


def dimer():
    H = np.array([[100.0, 100.0], [100.0, 0.0]])
    return Workload("cfg1_dimer", H, 35.0, 50.0, 300.0, 1, 4, 1.0, 1000)


def _fmo_like_H():
    rng = np.random.default_rng(SEED_FMO)
    eps = rng.uniform(0.0, 500.0, size=7)
    J = rng.normal(0.0, 40.0, size=7 * 6 // 2)
    return _symmetric_from_upper(7, eps, J)


def fmo_like():
    return Workload("cfg2_fmo7", _fmo_like_H(), 35.0, 50.0, 77.0, 1, 8, 1.0, 1000)


def deep():
    return Workload("cfg3_deep7", _fmo_like_H(), 35.0, 50.0, 300.0, 1, 12, 1.0, 200)


def lhcii_like():
    N = 14
    rng = np.random.default_rng(SEED_LHCII)
    eps = rng.uniform(0.0, 600.0, size=N)
    sign = rng.choice([-1.0, 1.0], size=N * (N - 1) // 2)
    iu = np.triu_indices(N, k=1)
    J = 80.0 * np.exp(-np.abs(iu[0] - iu[1]) / 3.0) * sign
    return Workload("cfg4_lhcii14", _symmetric_from_upper(N, eps, J), 37.0, 40.0, 300.0, 0, 8,
                    0.5, 500)


def large():
    N = 96
    rng = np.random.default_rng(SEED_LARGE)
    eps = rng.uniform(0.0, 800.0, size=N)
    pos = rng.uniform(0.0, 6.0, size=(N, 3))
    iu = np.triu_indices(N, k=1)
    d = np.linalg.norm(pos[iu[0]] - pos[iu[1]], axis=1)
    J = 300.0 / (1.0 + d ** 3)
    return Workload("cfg5_large96", _symmetric_from_upper(N, eps, J), 35.0, 50.0, 300.0, 0, 3,
                    0.5, 50)


def absorption_fmo(p=2):
    """Not a BASELINE config: the paper's linear-absorption use (Fig. 5: FMO at 77 K) on the FMO-like
    stand-in.  cfg2's H with the ground state as state 0, its 7 baths on states 1..7, sigma_0(0) = mu_p |0><0|
    (p = 0, 1, 2: the polarisation directions of Eq. 55, independent replicas; default z), a non-Hermitian
    single-column state, N = 8, W = 14, D = 8, the same 319 770 nodes."""
    w = fmo_like()
    H, bath_state, dip = with_ground_state(w)
    mu = dipole_operator(dip, int(p) % 3)
    s0 = np.zeros((8, 8), dtype=np.complex128)
    s0[:, 0] = mu[:, 0]
    return Workload("absorb_fmo8", H, 35.0, 50.0, 77.0, 1, 8, 1.0, 1000, tuple(bath_state), s0)


def two_exciton_fmo(D=5, K=1, T=77.0):
    """Not a BASELINE config: the paper's transient-absorption state space (ground state, 7 one-exciton
    and 21 two-exciton states of FMO = 29 states, Eq. 54) on the FMO-like stand-in H of cfg2; bath a couples to |a>
    and to the six |ab>.  sigma_0(0) = |1><1| (one-exciton state of site 1).  Defaults: 7 baths x 2 modes,
    D = 5: 11 628 nodes of 29 x 29 (156 MB per state buffer)."""
    H, S, _ = two_exciton_manifold(_fmo_like_H())
    s0 = np.zeros(H.shape, dtype=np.complex128)
    s0[1, 1] = 1.0
    return Workload("twoex_fmo29", H, 35.0, 50.0, T, K, D, 0.2, 200, None, s0, tuple(tuple(x) for x in S))


def mid_size(N=24, D=5):
    """Not a BASELINE config: a mid-size site-map system (N between the small-N and the N = 32/64/96 kernels; the
    paper's "larger state spaces") with cfg4's generator (LHCII-like couplings), K = 0, one bath per
    site.  Defaults: 24 sites, D = 5: 118 755 nodes of 24 x 24 (1.09 GB per state buffer)."""
    rng = np.random.default_rng(SEED_LHCII + 7)
    eps = rng.uniform(0.0, 600.0, size=N)
    sign = rng.choice([-1.0, 1.0], size=N * (N - 1) // 2)
    iu = np.triu_indices(N, k=1)
    J = 80.0 * np.exp(-np.abs(iu[0] - iu[1]) / 3.0) * sign
    return Workload(f"mid_sites{N}", _symmetric_from_upper(N, eps, J), 37.0, 40.0, 300.0, 0, D, 0.5, 200)


CONFIGS = {
    "cfg1": dimer, "cfg2": fmo_like, "cfg3": deep, "cfg4": lhcii_like, "cfg5": large,
}
EXTRA = {"absorb": absorption_fmo, "twoex": two_exciton_fmo, "mid24": mid_size}


def get(name):
    return (CONFIGS.get(name) or EXTRA[name])()


def random_state(nodes, N, seed, hermitian=False, tile=0):
    """A dense seeded test state [nodes][N][N] complex128 with O(1) entries
    (for single-RHS parity, where every term of the equation must be exercised).
    tile > 0 (very large states): `tile` random nodes repeated, node u scaled by 1 + (u mod 97)/100 -- every node
    still differs from its neighbours, at a fraction of the generation time."""
    rng = np.random.default_rng(seed)
    out = np.empty((nodes, N, N), dtype=np.complex128)
    if tile > 0:
        blk = rng.standard_normal((tile, N, N)) + 1j * rng.standard_normal((tile, N, N))
        if hermitian:
            blk = 0.5 * (blk + np.conj(np.swapaxes(blk, 1, 2)))
        for a in range(0, nodes, tile):
            b = min(nodes, a + tile)
            out[a:b] = blk[:b - a] * (1.0 + (np.arange(a, b) % 97) / 100.0)[:, None, None]
        return out
    chunk = max(1, (1 << 22) // (N * N))
    for a in range(0, nodes, chunk):
        b = min(nodes, a + chunk)
        blk = rng.standard_normal((b - a, N, N)) + 1j * rng.standard_normal((b - a, N, N))
        if hermitian:
            blk = 0.5 * (blk + np.conj(np.swapaxes(blk, 1, 2)))
        out[a:b] = blk
    return out


def random_density(N, seed):
    """A seeded random density matrix (Hermitian, positive, trace 1)."""
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    rho = A @ A.conj().T
    return rho / np.trace(rho).real


def with_ground_state(w, seed=1803034990):
    """Linear-absorption stand-in (Eq. 53, 56): the workload's H with the electronic ground state
    prepended as state 0 (energy 0, uncoupled: Eq. 48's block form), bath b on state b+1, and one seeded
    transition dipole d_m per site (unit vectors, like the BChl Q_y dipoles the paper takes from the
    crystal structure).  Returns (H_ext [N+1][N+1], bath_state [N], dipoles [N][3])."""
    N = w.N
    H = np.zeros((N + 1, N + 1))
    H[1:, 1:] = w.H_cm
    rng = np.random.default_rng(seed)
    d = rng.standard_normal((N, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    return H, list(range(1, N + 1)), d


def dipole_operator(dipoles, p):
    """mu_p = mu_p^+ + mu_p^- with mu_p^+ = sum_m (e_p . d_m) |m><0| (Eq. 53), e_p the p-th Cartesian unit vector (Eq. 55)."""
    N = dipoles.shape[0]
    mu = np.zeros((N + 1, N + 1))
    mu[1:, 0] = dipoles[:, p]
    mu[0, 1:] = dipoles[:, p]
    return mu


def two_exciton_manifold(H_sites):
    """Input construction for the paper's two-exciton space (Eq. 54: N_states = 1 + N + N(N-1)/2; P:84:
    "a two-exciton state is coupled to two sites"): states 0 = ground, 1..N = |a>, then |ab> (a < b) in
    row-major pair order.  Frenkel-exciton matrix elements: <ab|H|ab> = eps_a + eps_b, <ab|H|ac> = J_bc for pairs
    that share one site, zero otherwise; the manifolds are not coupled by the field-free H.  Bath a (site a's
    bath) couples to |a> and to every |ab>.  Returns (H [Ns][Ns], bath_states list of lists, pair index list)."""
    N = H_sites.shape[0]
    pairs = [(a, b) for a in range(N) for b in range(a + 1, N)]
    Ns = 1 + N + len(pairs)
    H = np.zeros((Ns, Ns))
    H[1:N + 1, 1:N + 1] = H_sites
    for p, (a, b) in enumerate(pairs):
        for q, (c, d) in enumerate(pairs):
            if p == q:
                H[1 + N + p, 1 + N + q] = H_sites[a, a] + H_sites[b, b]
            else:
                shared = {a, b} & {c, d}
                if len(shared) == 1:
                    (x,) = {a, b} - shared
                    (y,) = {c, d} - shared
                    H[1 + N + p, 1 + N + q] = H_sites[x, y]
    bath_states = [[1 + a] + [1 + N + p for p, pr in enumerate(pairs) if a in pr] for a in range(N)]
    return H, bath_states, pairs


def rwa_field_hamiltonian(H0, mu_plus, field):
    """H(t) of Eq. 51 for one polarisation: H0 - (mu^+ E^-(t) + mu^- E^+(t)), E^- = conj(E^+); `field` = E^+(t) as a
    complex number (envelope times carrier phase, Eq. 50), mu_plus = sum_a d_a |a><0| (Eq. 48), real."""
    return H0.astype(np.complex128) - (mu_plus * np.conj(field) + mu_plus.T * field)
