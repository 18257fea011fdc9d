"""-m "not gpu": the Pade decomposition (S section 8(f) next #1; Eq. 27-33, R11) in the oracle,
pinned by what the mathematics fixes, and the library's independent implementation (Sturm bisection instead of
Jacobi rotations) against it."""
import numpy as np
import pytest

import workloads
from oracle.oracle import Oracle, pade_poles
from paper_1803_03498_b200 import Heom

HBAR = 5308.8
KB = 0.6950348


def test_k1_closed_form():
    """[0/1]: Lambda is 2x2 with off-diagonal 1/sqrt(15) -> xi = 2 sqrt(15); Eq. 29 with empty products ->
    eta = 1 + 3/2; and 2 eta/xi^2 = 1/12 is the x/12 term of the Bose function."""
    xi, eta = pade_poles(1)
    assert abs(xi[0] - 2.0 * np.sqrt(15.0)) < 1e-13
    assert abs(eta[0] - 2.5) < 1e-13


@pytest.mark.parametrize("K", [1, 2, 3, 4, 6, 10, 16])
def test_taylor_sum_rules(K):
    """1/(1-e^-x) = 1/x + 1/2 + x/12 - x^3/720 + x^5/30240 - ...; the [K-1/K] approximant matches the first
    2K orders, i.e. sum_j eta_j/xi_j^(2p) = |B_2p|/(2 (2p)!) for p <= K."""
    xi, eta = pade_poles(K)
    assert np.all(np.diff(xi) > 0) and np.all(eta > 0)
    assert abs(24.0 * np.sum(eta / xi ** 2) - 1.0) < 1e-12
    if K >= 2:
        assert abs(1440.0 * np.sum(eta / xi ** 4) - 1.0) < 1e-11
    if K >= 3:
        assert abs(60480.0 * np.sum(eta / xi ** 6) - 1.0) < 1e-10


def test_bose_function_error_decreases_with_k():
    x = np.array([0.5, 2.0, 5.0, 10.0])
    exact = 1.0 / (1.0 - np.exp(-x))
    prev = None
    for K in (1, 2, 3, 5, 8):
        xi, eta = pade_poles(K)
        f = 1.0 / x + 0.5 + np.sum(2.0 * eta[None, :] * x[:, None] / (x[:, None] ** 2 + xi[None, :] ** 2), axis=1)
        err = np.abs(f - exact)
        if prev is not None:
            assert np.all(err <= prev + 1e-15)
        prev = err
    assert np.all(prev < 1e-9)


def test_lowest_poles_approach_matsubara():
    xi, eta = pade_poles(8)
    assert np.allclose(xi[:3], 2.0 * np.pi * np.arange(1, 4), rtol=1e-6)
    assert np.allclose(eta[:3], 1.0, rtol=1e-5)


@pytest.mark.parametrize("T", [300.0, 77.0, 30.0])
def test_coefficients_converge_to_exact_drude_term_and_zero_terminator(T):
    """Eq. 33, k = 0 tends to the exact lambda nu cot(beta hbar nu / 2) (Eq. 20) much faster than it would by
    truncating the Matsubara series, and the Eq. 14 bracket vanishes identically: the approximant reproduces the
    x -> 0 behaviour of coth exactly."""
    H = np.zeros((1, 1))
    lam, nu = 35.0, 0.02
    bh = HBAR / (KB * T)
    exact = lam / HBAR * nu / np.tan(bh * nu / 2.0)
    errs = []
    for K in (1, 2, 4, 8):
        g, cr, ci, d = Oracle(H, lam, nu, T, K, 1, pade=1).coefficients()
        assert abs(d[0]) < 1e-15
        assert ci[0] == -lam / HBAR * nu
        assert np.allclose(g[1:], pade_poles(K)[0] / bh, rtol=1e-14)
        errs.append(abs(cr[0] - exact) / abs(exact))
    assert errs[-1] < 1e-10 and all(b <= a + 1e-13 for a, b in zip(errs, errs[1:]))


def test_pade_converges_faster_than_matsubara_on_the_dimer():
    """P:148 "a faster converging Pade expansion": low-temperature dimer (77 K), rho_11(t = 300 fs) as a function
    of the number of poles K.  The Pade sequence is Cauchy with quickly shrinking increments; the Matsubara
    sequence (with the Eq. 14 terminator) creeps monotonically towards the same limit."""
    w = workloads.dimer().with_(T_kelvin=77.0, D=4)

    def rho11(K, pade):
        o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, K, w.D, pade=pade)
        o.set_state(w.sigma0())
        o.rk4_steps(0.5, 600)
        return o.populations()[0][0]

    P = {K: rho11(K, 1) for K in (2, 3, 4, 6)}
    M = {K: rho11(K, 0) for K in (2, 4, 6, 8)}
    assert abs(P[3] - P[2]) > abs(P[4] - P[3]) > abs(P[6] - P[4])
    assert abs(P[6] - P[4]) < 0.25 * abs(M[6] - M[4])
    gaps = [abs(M[K] - P[6]) for K in (2, 4, 6, 8)]
    assert all(b < a for a, b in zip(gaps, gaps[1:])) and gaps[-1] < 2e-5


@pytest.mark.parametrize("T,K", [(300.0, 1), (77.0, 3), (30.0, 6), (77.0, 0)])
def test_library_pade_matches_oracle(T, K):
    H = np.zeros((3, 3))
    lam, nu = [35.0, 0.0, 12.5], [0.02, 0.025, 0.01]
    o = Oracle(H, lam, nu, T, K, 2, pade=1)
    g = Heom(H, lam, nu, T, K, 2, pade=1)
    for q, (a, b) in enumerate(zip(g.coefficients(), o.coefficients())):
        if q == 3:
            assert np.all(np.abs(a) < 1e-15) and np.all(np.abs(b) < 1e-15)
        else:
            assert np.allclose(a, b, rtol=1e-12, atol=1e-300)
    g.set_option("pade", 0)                                   # switching back restores the Matsubara set
    g0 = Heom(H, lam, nu, T, K, 2)
    for a, b in zip(g.coefficients(), g0.coefficients()):
        assert np.array_equal(a, b)
