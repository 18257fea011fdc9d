"""Pins for the oracle's general system-bath operators (oracle_create_general: S(b) >= 1 states per bath, several
baths per state -- the sums over s of Eq. 14-17; the two-exciton manifold of Eq. 54)
and for complex / time-dependent Hamiltonians (Eq. 51).  SURVEY.md 8(f) next #4.

Expected values come from outside the new code: the cumulant line shape of a Gaussian bath for diagonal couplings
(every coherence of a J = 0 system is a closed form), the matrix-algebra form of the equations with projector sums,
the gauge covariance of the equations under diagonal unitaries (which maps a complex H onto the already pinned
real-H path), scipy's expm, and the rotating-frame Rabi formula of a resonantly driven two-level system.
"""
import numpy as np
import pytest
import scipy.linalg

import workloads
from oracle.oracle import Oracle
from test_oracle_physics import HBAR, KB


def mode_lineshape(t, lam, nu, T, K):
    """(g_modes(t), Delta): g of the K+1 exponential modes alone (complex c_0), and the Eq. 14 bracket."""
    bh = HBAR / (KB * T)
    lam_h = lam / HBAR
    gam = [nu] + [2 * np.pi * k / bh for k in range(1, K + 1)]
    c = [lam_h * nu * (1 / np.tan(bh * nu / 2) - 1j)]
    c += [4 * lam_h * nu * g / (bh * (g * g - nu * nu)) for g in gam[1:]]
    Delta = 2 * lam_h / (bh * nu) - sum(ck.real / g for ck, g in zip(c, gam))
    return sum(ck / g ** 2 * (np.exp(-g * t) + g * t - 1) for ck, g in zip(c, gam)), Delta


def coherence_closed_form(t, eps, bath_states, lam, nu, T, K, form):
    """rho_ij(t)/rho_ij(0) for H = diag(eps) and baths coupling through V_b = sum_{s in S_b} |s><s| (q_b = the 0/1
    membership): exp(-i (eps_i - eps_j) t/hbar - sum_b [(q_i - q_j)^2 Re g_b + i (q_i^2 - q_j^2) Im g_b
    + mask_b(i,j) Delta_b t]) -- textbook second cumulant, exact for a Gaussian bath; the delta-correlated tail the
    terminator stands for adds mask * Delta * t with mask = (q_i - q_j)^2 for the operator form of Eq. 14 and
    (1 - delta_ij)(q_i + q_j) for the sum as printed (R12)."""
    N = len(eps)
    out = np.zeros((N, N), dtype=complex)
    for i in range(N):
        for j in range(N):
            ex = -1j * (eps[i] - eps[j]) * t / HBAR
            for b, S in enumerate(bath_states):
                qi, qj = float(i in S), float(j in S)
                g, Delta = mode_lineshape(t, lam[b], nu[b], T, K)
                mask = (qi - qj) ** 2 if form == 1 else (i != j) * (qi + qj)
                ex -= (qi - qj) ** 2 * g.real + 1j * (qi * qi - qj * qj) * g.imag + mask * Delta * t
            out[i, j] = np.exp(ex)
    return out


@pytest.mark.parametrize("form", [0, 1])
def test_two_exciton_manifold_at_zero_coupling(form):
    """Two sites a, b with J = 0 and the two-exciton state (Eq. 54: N_states = 1 + 2 + 1): states 0 = ground,
    1 = |a>, 2 = |b>, 3 = |ab>; bath A couples to {|a>, |ab>}, bath B to {|b>, |ab>}.  Every coherence is a
    closed form; in particular <ab|rho|0> = <a|rho|0> <b|rho|0> (two independent one-exciton line shapes), and in
    <ab|rho|a> the shared bath A cancels."""
    eps = np.array([0.0, 120.0, 45.0, 165.0])
    lam, nu, T, K, D = [35.0, 20.0], [0.02, 0.03], 77.0, 2, 9
    S = [[1, 3], [2, 3]]
    o = Oracle(np.diag(eps), lam, nu, T, K, D, bath_states=S, terminator_form=form)
    assert o.B == 2 and o.W == 2 * (K + 1)
    s0 = np.full((4, 4), 0.25, dtype=complex)
    o.set_state(s0)
    t_end, dt = 150.0, 0.25
    o.rk4_steps(dt, int(t_end / dt))
    rho = o.sigma0()
    expect = 0.25 * coherence_closed_form(t_end, eps, S, lam, nu, T, K, form)
    assert np.max(np.abs(rho - expect)) < 2e-8
    # the product structure, from the propagated numbers alone
    assert abs(rho[3, 0] / 0.25 - (rho[1, 0] / 0.25) * (rho[2, 0] / 0.25)) < 1e-7
    # populations do not move under pure dephasing
    assert np.max(np.abs(np.diag(rho) - 0.25)) < 1e-14


def test_shared_bath_printed_and_operator_form_differ_by_the_terminator_only():
    """One bath coupled to states {0, 1} of a three-state system, J = 0.  The coupling is the same for both, so the
    bath drops out of their coherence -- except for Eq. 14 as printed, whose sum over s leaves (1 - delta_ij) * 2
    there: rho_01 decays with exp(-2 Delta t), the operator form (sum_s V_s^x)^2 gives none (R12).  The
    coherences with the uncoupled state 2 are the one-bath line shape in both forms."""
    eps = np.array([10.0, 70.0, 0.0])
    lam, nu, T, K, D, t_end, dt = 35.0, 0.02, 77.0, 1, 10, 120.0, 0.25
    g, Delta = mode_lineshape(t_end, lam, nu, T, K)
    res = {}
    for form in (0, 1):
        o = Oracle(np.diag(eps), [lam], [nu], T, K, D, bath_states=[[0, 1]], terminator_form=form)
        o.set_state(np.full((3, 3), 1 / 3, dtype=complex))
        o.rk4_steps(dt, int(t_end / dt))
        res[form] = o.sigma0() * 3
    free01 = np.exp(-1j * (eps[0] - eps[1]) * t_end / HBAR)
    assert abs(res[1][0, 1] - free01) < 1e-9
    assert abs(res[0][0, 1] - free01 * np.exp(-2 * Delta * t_end)) < 1e-9
    for form in (0, 1):
        assert abs(res[form][0, 2] - np.exp(-1j * (eps[0] - eps[2]) * t_end / HBAR - g - Delta * t_end)) < 1e-7
        assert abs(res[form][2, 1] - np.exp(-1j * (eps[2] - eps[1]) * t_end / HBAR - np.conj(g) - Delta * t_end)) < 1e-7


def general_operator_form_rhs(H, bath_states, lam, nu, T, K, state, tuples, form):
    """Eq. 12-17 (unscaled) with matrix (anti)commutators of the projector sums V_b = sum_s P_s (linear terms) and
    Eq. 14 either as printed (sum_s [P_s, [P_s, .]]) or as [V_b, [V_b, .]]: a different route to the same numbers
    than the oracle's elementwise masks."""
    N = H.shape[0]
    M = K + 1
    bh = HBAR / (KB * T)
    idx = {tuple(int(v) for v in n): u for u, n in enumerate(tuples)}
    out = np.zeros_like(state)
    P = [np.diag((np.arange(N) == s).astype(float)) for s in range(N)]
    comm = lambda A, B: A @ B - B @ A
    acomm = lambda A, B: A @ B + B @ A
    for n, u in idx.items():
        s = state[u]
        r = -1j / HBAR * comm(H, s)
        for b, S in enumerate(bath_states):
            V = sum(P[q] for q in S)
            lam_h = lam[b] / HBAR
            gam = [nu[b]] + [2 * np.pi * k / bh for k in range(1, M)]
            c = [lam_h * nu[b] / np.tan(bh * nu[b] / 2)] + \
                [4 * lam_h * nu[b] * g / (bh * (g * g - nu[b] ** 2)) for g in gam[1:]]
            Delta = 2 * lam_h / (bh * nu[b]) - sum(ck / g for ck, g in zip(c, gam))
            if form == 1:
                r = r - Delta * comm(V, comm(V, s))
            else:
                r = r - Delta * sum(comm(P[q], comm(P[q], s)) for q in S)
            for k in range(M):
                l = b * M + k
                r = r - n[l] * gam[k] * s
                up = tuple(v + (i == l) for i, v in enumerate(n))
                dn = tuple(v - (i == l) for i, v in enumerate(n))
                if up in idx:
                    r = r + 1j * comm(V, state[idx[up]])
                if n[l] > 0:
                    th = 1j * c[k] * comm(V, state[idx[dn]])
                    if k == 0:
                        th = th + lam_h * nu[b] * acomm(V, state[idx[dn]])
                    r = r + n[l] * th
        out[u] = r
    return out


@pytest.mark.parametrize("form", [0, 1])
@pytest.mark.parametrize("N,S,K,D", [(4, [[1, 3], [2, 3]], 1, 3), (5, [[0, 1, 2], [2, 3], [4], [0, 4]], 0, 3),
                                     (3, [[0, 1, 2]], 2, 3)])
def test_general_rhs_against_operator_form(N, S, K, D, form):
    """Random complex Hermitian H, dense random state: every term, sign and index of the generalised sums."""
    rng = np.random.default_rng(200 + N + K + D)
    A = rng.normal(0, 80, (N, N)) + 1j * rng.normal(0, 80, (N, N))
    H = A + A.conj().T
    lam = rng.uniform(10, 50, len(S)); nu = rng.uniform(0.01, 0.04, len(S))
    o = Oracle(H, lam, nu, 140.0, K, D, scaling=0, bath_states=S, terminator_form=form)
    t, _, _ = o.tables()
    st = workloads.random_state(o.nodes, N, seed=6)
    o.set_full_state(st)
    ref = general_operator_form_rhs(H, S, lam, nu, 140.0, K, st, t, form)
    got = o.rhs()
    assert np.max(np.abs(got - ref)) < 1e-14 * np.abs(ref).max() + 1e-16


def test_general_with_singletons_is_the_site_map_path():
    w = workloads.fmo_like()
    H = w.H_cm[:4, :4]
    a = Oracle(H, [35.0, 20.0, 10.0], 0.02, 77.0, 1, 3, bath_state=[2, 0, 3])
    b = Oracle(H, [35.0, 20.0, 10.0], 0.02, 77.0, 1, 3, bath_states=[[2], [0], [3]])
    s0 = workloads.random_density(4, 3)
    a.set_state(s0); b.set_state(s0)
    a.rk4_steps(0.5, 50); b.rk4_steps(0.5, 50)
    assert np.array_equal(a.get_full_state(), b.get_full_state())


def test_complex_hamiltonian_gauge_covariance():
    """H' = U H U^dagger with U = diag(exp(i phi)) is complex Hermitian; every projector sum commutes with U, so the
    whole hierarchy transforms covariantly: sigma'_u(t) = U sigma_u(t) U^dagger for the state started at
    U sigma(0) U^dagger.  The right-hand side is the already pinned real-H path."""
    rng = np.random.default_rng(11)
    N, S = 4, [[1, 3], [2, 3], [0]]
    H = rng.normal(0, 60, (N, N)); H = (H + H.T) / 2
    U = np.diag(np.exp(1j * rng.uniform(0, 2 * np.pi, N)))
    Hc = U @ H @ U.conj().T
    Hc = (Hc + Hc.conj().T) / 2
    assert np.abs(Hc.imag).max() > 1.0
    lam, nu, T, K, D = [35.0, 20.0, 50.0], [0.02, 0.03, 0.025], 150.0, 1, 4
    a = Oracle(H, lam, nu, T, K, D, bath_states=S)
    b = Oracle(Hc, lam, nu, T, K, D, bath_states=S)
    s0 = workloads.random_density(N, 7)
    a.set_state(s0); b.set_state(U @ s0 @ U.conj().T)
    a.rk4_steps(0.5, 300); b.rk4_steps(0.5, 300)
    sa, sb = a.get_full_state(), b.get_full_state()
    assert np.max(np.abs(sb - U[None] @ sa @ U.conj().T[None])) < 1e-12
    assert abs(np.trace(sb[0]) - 1) < 1e-12


def test_complex_hamiltonian_without_bath_against_expm():
    rng = np.random.default_rng(12)
    N = 5
    A = rng.normal(0, 50, (N, N)) + 1j * rng.normal(0, 50, (N, N))
    H = (A + A.conj().T) / 2
    o = Oracle(H, 0.0, 0.02, 300.0, 1, 2, bath_states=[[i] for i in range(N)])
    rho0 = workloads.random_density(N, 4)
    o.set_state(rho0)
    t_end, dt = 100.0, 0.05
    o.rk4_steps(dt, int(t_end / dt))
    Ut = scipy.linalg.expm(-1j * H * t_end / HBAR)
    assert np.max(np.abs(o.sigma0() - Ut @ rho0 @ Ut.conj().T)) < 1e-9


def test_time_dependent_hamiltonian_resonant_rabi():
    """Ground and excited state, RWA field coupling (Eq. 51): H(t) = [[0, W e^{+i w t}], [W e^{-i w t}, eps]] with
    hbar w = eps (resonance).  In the frame rotating with w the Hamiltonian is the constant [[0, W], [W, 0]]:
    P_e(t) = sin^2(W t/hbar), whatever eps.  Pins oracle_rk4_step_td (H at t, t + dt/2, t + dt) and the complex H."""
    eps, Wc = 400.0, 60.0
    om = eps / HBAR

    def H(t):
        return np.array([[0.0, Wc * np.exp(1j * om * t)], [Wc * np.exp(-1j * om * t), eps]])

    errs = []
    for dt in (0.2, 0.1):
        o = Oracle(H(0.0), 0.0, 0.02, 300.0, 0, 1, bath_states=[[1]])
        o.set_state(np.diag([1.0, 0.0]).astype(complex))
        n = int(round(60.0 / dt))
        for q in range(n):
            o.rk4_step_td(dt, H(q * dt), H((q + 0.5) * dt), H((q + 1) * dt))
        pe = o.sigma0()[1, 1].real
        errs.append(abs(pe - np.sin(Wc * n * dt / HBAR) ** 2))
    assert errs[0] < 1e-7 and errs[1] < errs[0] / 12        # dt^4
    # with the field frozen at t = 0 the step reduces to oracle_rk4_steps
    a = Oracle(H(0.0), 35.0, 0.02, 300.0, 1, 3, bath_states=[[1]])
    b = Oracle(H(0.0), 35.0, 0.02, 300.0, 1, 3, bath_states=[[1]])
    s0 = workloads.random_density(2, 1)
    a.set_state(s0); b.set_state(s0)
    a.rk4_steps(0.5, 3)
    for _ in range(3):
        b.rk4_step_td(0.5, H(0.0), H(0.0), H(0.0))
    assert np.array_equal(a.get_full_state(), b.get_full_state())


def test_general_argument_validation():
    H = np.zeros((3, 3))
    with pytest.raises(ValueError):
        Oracle(H, [35.0], [0.02], 300.0, 1, 2, bath_states=[[0, 0]])        # a state twice in one bath
    with pytest.raises(ValueError):
        Oracle(H, [35.0], [0.02], 300.0, 1, 2, bath_states=[[3]])           # state out of range
    with pytest.raises(ValueError):
        Oracle(H, [35.0, 1.0], [0.02, 0.02], 300.0, 1, 2, bath_states=[[0], []])   # S(b) = 0
    Hbad = np.array([[0, 1j, 0], [1j, 0, 0], [0, 0, 0]])
    with pytest.raises(ValueError):
        Oracle(Hbad, [35.0], [0.02], 300.0, 1, 2, bath_states=[[0]])        # not Hermitian
