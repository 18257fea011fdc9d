"""-m gpu: systems in which not every state carries a bath (heom_create_sites; the ground state of linear
absorption) on every kernel family, against the oracle."""
import numpy as np
import pytest

import workloads
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-13
STATE_TOL = 1e-10


def rel_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def _system(N, bath_state, seed):
    rng = np.random.default_rng(4000 + seed)
    H = rng.normal(0.0, 80.0, (N, N)); H = (H + H.T) / 2
    B = len(bath_state)
    return H, rng.uniform(20.0, 45.0, B), rng.uniform(0.015, 0.03, B)


def _pair(H, lam, nu, T, K, D, bath_state, **opts):
    from paper_1803_03498_b200 import Heom
    o = Oracle(H, lam, nu, T, K, D, bath_state=bath_state)
    g = Heom(H, lam, nu, T, K, D, bath_state=bath_state, **opts).bind()
    return o, g


# N, bath_state, K, D: tiny kernel (N = 2, 3), pipelined small-N kernel, generic (N = 20, 33), tensor-core (N = 32)
CASES = [(2, [1], 1, 4), (3, [1, 2], 1, 3), (8, [1, 2, 3, 4, 5, 6, 7], 1, 3), (8, [1, 2, 3, 4, 5, 6, 7], 0, 5),
         (5, [3, 0], 2, 4), (15, list(range(1, 15)), 0, 2), (16, [15, 2, 7], 1, 3), (20, list(range(1, 20)), 0, 2),
         (32, list(range(1, 32)), 0, 2), (32, [5, 31, 0], 1, 3), (33, list(range(1, 33)), 0, 1), (4, [3, 2, 1, 0], 1, 3)]


@pytest.mark.parametrize("N,bath_state,K,D", CASES)
@pytest.mark.parametrize("order,kernel", [(0, 1), (1, 1), (1, 2), (1, 0)])
def test_rhs_parity_site_map_random_state(N, bath_state, K, D, order, kernel):
    H, lam, nu = _system(N, bath_state, N + K + D)
    o, g = _pair(H, lam, nu, 150.0, K, D, bath_state, order=order, kernel=kernel)
    for a, b in zip(g.tables(), o.tables()):
        assert np.array_equal(a, b)
    st = workloads.random_state(o.nodes, N, seed=77 + N)
    o.set_full_state(st); g.set_full_state(st)
    assert rel_err(g.rhs(), o.rhs()) < RHS_TOL
    sth = workloads.random_state(o.nodes, N, seed=78 + N, hermitian=True)
    o.set_full_state(sth); g.set_full_state(sth)
    got = g.rhs()
    assert rel_err(got, o.rhs()) < RHS_TOL
    if g.kernel_name() in ("rhs_hpipe_kernel", "rhs_herm_kernel"):
        assert np.array_equal(got, np.conj(np.swapaxes(got, 1, 2)))


@pytest.mark.parametrize("form", [-1, 0])
@pytest.mark.parametrize("sites,K,D,steps", [(1, 2, 6, 400), (2, 1, 4, 1000), (7, 1, 4, 300), (7, 0, 5, 300)])
def test_absorption_propagation_parity(sites, K, D, steps, form):
    """mu_p rho(0) with rho(0) = |0><0|, a non-Hermitian state, propagated with the ground state in the
    basis; every node compared, and Tr(mu_p sigma_0(t)) (heom_expectation) against the oracle's sigma_0."""
    w = workloads.fmo_like()
    w = w.with_(H_cm=w.H_cm[:sites, :sites])
    H, bath_state, dip = workloads.with_ground_state(w)
    o, g = _pair(H, w.lambda_cm, w.nu_per_fs, 77.0, K, D, bath_state, rk4_form=form)
    mu = workloads.dipole_operator(dip, 2).astype(complex)
    rho0 = np.zeros_like(mu); rho0[0, 0] = 1.0
    s0 = mu @ rho0
    o.set_state(s0); g.set_state(s0)
    assert abs(g.expectation(mu) - np.trace(mu @ s0)) < 1e-15
    o.rk4_steps(1.0, steps); g.rk4_steps(1.0, steps)
    ref, got = o.get_full_state(), g.get_full_state()
    assert rel_err(got, ref) < STATE_TOL
    c_ref = np.trace(mu @ ref[0])
    assert abs(g.expectation(mu) - c_ref) < 1e-12 * max(1.0, abs(c_ref))
    # only the (site, ground) column is populated (Eq. 48 block structure)
    assert np.abs(got[:, :, 1:]).max() == 0.0


def test_linear_absorption_spectrum_matches_oracle():
    """Eq. 56 end to end on a dimer + ground state: the library's correlation function and spectrum against the
    same quantities from oracle-propagated states."""
    from paper_1803_03498_b200.spectra import linear_absorption
    w = workloads.dimer()
    H, bath_state, dip = workloads.with_ground_state(w)
    K, D, T, dt, steps = 1, 4, 300.0, 1.0, 256
    t, corr, omega, spec = linear_absorption(H, bath_state, dip, w.lambda_cm, w.nu_per_fs, T, K, D, dt, steps, pad=4)
    ref = np.zeros(steps + 1, dtype=complex)
    for p in range(3):
        mu = workloads.dipole_operator(dip, p).astype(complex)
        o = Oracle(H, w.lambda_cm, w.nu_per_fs, T, K, D, bath_state=bath_state)
        s0 = np.zeros_like(mu); s0[:, 0] = mu[:, 0]
        o.set_state(s0)
        ref[0] += np.trace(mu @ s0)
        for n in range(1, steps + 1):
            o.rk4_steps(dt, 1)
            ref[n] += np.trace(mu @ o.sigma0())
    assert np.max(np.abs(corr - ref)) < 1e-11
    assert abs(corr[0] - np.sum(dip ** 2)) < 1e-14            # C(0) = sum_p Tr(mu_p mu_p rho(0)) = sum_m |d_m|^2
    # the spectrum peaks near the exciton energies of the dimer (eigenvalues of H_sites, shifted by the bath)
    peak = omega[np.argmax(spec)]
    ev = np.linalg.eigvalsh(w.H_cm)
    assert np.min(np.abs(peak - ev)) < 60.0
