"""Pins for the oracle's bath -> state map (oracle_create_sites): systems in which not every state carries a
bath -- the ground state |0> of linear absorption (Eq. 53, 56).

Expected values come from outside the new code: the cumulant closed form of a two-level absorber, the already
pinned per-site path (a bath with lambda = 0 is no bath), and the block structure of Eq. 48.
"""
import numpy as np
import pytest

import workloads
from oracle.oracle import Oracle
from test_oracle_physics import HBAR, lineshape_from_modes


@pytest.mark.parametrize("T,K,D,tol", [(77.0, 2, 10, 1e-10), (300.0, 1, 10, 5e-6)])
def test_monomer_optical_coherence_closed_form(T, K, D, tol):
    """States (g, e), bath on e only.  mu^+ rho(0) = |e><g| evolves as exp(-i eps t/hbar - g(t)) (textbook
    cumulant, exact for a Gaussian bath), the conjugate element |g><e| as exp(+i eps t/hbar - conj g(t)).
    A map that put the bath on the wrong state, or on both, fails: both give other exponents."""
    eps, lam, nu, t_end, dt = 120.0, 35.0, 0.02, 200.0, 0.25
    H = np.diag([0.0, eps])
    g = lineshape_from_modes(t_end, lam, nu, T, K)
    for (i, j), expect in (((1, 0), np.exp(-1j * eps * t_end / HBAR - g)),
                           ((0, 1), np.exp(+1j * eps * t_end / HBAR - np.conj(g)))):
        o = Oracle(H, lam, nu, T, K, D, bath_state=[1])
        assert o.W == K + 1 and o.B == 1
        s0 = np.zeros((2, 2), dtype=complex)
        s0[i, j] = 1.0
        o.set_state(s0)
        o.rk4_steps(dt, int(t_end / dt))
        rho = o.sigma0()
        assert abs(rho[i, j] - expect) < tol
        rho[i, j] = 0.0
        assert np.abs(rho).max() == 0.0


def test_bath_on_state_zero_instead():
    """The same absorber with the states swapped (bath_state = [0]) gives the transposed picture."""
    eps, lam, nu, T, K, D = 120.0, 35.0, 0.02, 77.0, 2, 10
    a = Oracle(np.diag([0.0, eps]), lam, nu, T, K, D, bath_state=[1])
    b = Oracle(np.diag([eps, 0.0]), lam, nu, T, K, D, bath_state=[0])
    sa = np.array([[0, 0], [1, 0]], dtype=complex)
    a.set_state(sa); b.set_state(sa.T.copy())
    a.rk4_steps(0.25, 400); b.rk4_steps(0.25, 400)
    assert abs(a.sigma0()[1, 0] - b.sigma0()[0, 1]) < 1e-15


def test_map_equals_decoupled_bath_of_the_per_site_path():
    """A state without a bath == a per-site bath with lambda = 0 (every coupling factor of that bath
    vanishes, R5).  The per-site path is pinned in test_oracle_physics.py; the hierarchy of the
    mapped system is the sub-hierarchy with n = 0 in the dead modes."""
    w = workloads.fmo_like()
    H, bath_state, dip = workloads.with_ground_state(w.with_(H_cm=w.H_cm[:3, :3]))
    K, D, T = 1, 3, 77.0
    mapped = Oracle(H, 35.0, 0.02, T, K, D, bath_state=bath_state)
    per_site = Oracle(H, [0.0, 35.0, 35.0, 35.0], 0.02, T, K, D)
    s0 = workloads.dipole_operator(dip, 1).astype(complex) @ np.diag([1.0, 0, 0, 0]).astype(complex)
    s0 = s0 + 0.3 * workloads.random_density(4, 5)          # coherences, populations, everything
    mapped.set_state(s0); per_site.set_state(s0)
    mapped.rk4_steps(0.5, 200); per_site.rk4_steps(0.5, 200)
    full_m, full_p = mapped.get_full_state(), per_site.get_full_state()
    tm, _, _ = mapped.tables()
    tp, _, _ = per_site.tables()
    M = K + 1
    index = {tuple(t): u for u, t in enumerate(map(tuple, tp))}
    for u, t in enumerate(map(tuple, tm)):
        v = index[(0,) * M + t]
        assert np.abs(full_m[u] - full_p[v]).max() < 1e-14
    dead = [v for v, t in enumerate(tp) if any(t[:M])]
    assert np.abs(full_p[dead]).max() == 0.0


def test_excited_block_equals_the_system_without_ground_state():
    """Eq. 48: H is block diagonal in (ground, one-exciton).  A state inside the one-exciton block evolves as in
    the N-site system; the ground-state row and column stay zero."""
    w = workloads.fmo_like()
    Hs = w.H_cm[:3, :3]
    H, bath_state, _ = workloads.with_ground_state(w.with_(H_cm=Hs))
    rho = workloads.random_density(3, 11)
    big = np.zeros((4, 4), dtype=complex); big[1:, 1:] = rho
    a = Oracle(H, 35.0, 0.02, 77.0, 1, 4, bath_state=bath_state)
    b = Oracle(Hs, 35.0, 0.02, 77.0, 1, 4)
    a.set_state(big); b.set_state(rho)
    a.rk4_steps(1.0, 100); b.rk4_steps(1.0, 100)
    fa, fb = a.get_full_state(), b.get_full_state()
    assert np.array_equal(a.tables()[0], b.tables()[0])
    assert np.abs(fa[:, 1:, 1:] - fb).max() < 1e-15
    assert np.abs(fa[:, 0, :]).max() == 0.0 and np.abs(fa[:, :, 0]).max() == 0.0


def test_identity_map_is_the_per_site_constructor():
    w = workloads.dimer()
    a = Oracle(w.H_cm, 35.0, 0.02, 300.0, 1, 4)
    b = Oracle(w.H_cm, 35.0, 0.02, 300.0, 1, 4, bath_state=[0, 1])
    st = workloads.random_state(a.nodes, 2, 3)
    a.set_full_state(st); b.set_full_state(st)
    assert np.array_equal(a.rhs(), b.rhs())
    # a permuted map is a different system: mode block 0 now belongs to state 1
    c = Oracle(w.H_cm, [35.0, 10.0], 0.02, 300.0, 1, 4, bath_state=[1, 0])
    d = Oracle(w.H_cm, [10.0, 35.0], 0.02, 300.0, 1, 4)
    s0 = workloads.random_density(2, 1)
    c.set_state(s0); d.set_state(s0)
    c.rk4_steps(1.0, 50); d.rk4_steps(1.0, 50)
    assert np.abs(c.sigma0() - d.sigma0()).max() < 1e-15


def test_site_map_validation():
    H = np.zeros((3, 3))
    for bad in ([1, 1], [3], [-1], [0, 1, 2, 0]):
        with pytest.raises(ValueError):
            Oracle(H, 35.0, 0.02, 300.0, 0, 2, bath_state=bad)
