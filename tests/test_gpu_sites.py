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
    g = Heom(H, lam, nu, T, K, D, bath_state=bath_state, **opts).bind(poison=True)
    return o, g


# N, bath_state, K, D: tiny kernel (N = 2, 3), pipelined small-N kernel, generic (N = 20, 33), tensor-core (N = 32)
CASES = [(2, [1], 1, 4), (3, [1, 2], 1, 3), (8, [1, 2, 3, 4, 5, 6, 7], 1, 3), (8, [1, 2, 3, 4, 5, 6, 7], 0, 5),
         (5, [3, 0], 2, 4), (15, list(range(1, 15)), 0, 2), (16, [15, 2, 7], 1, 3), (20, list(range(1, 20)), 0, 2),
         (32, list(range(1, 32)), 0, 2), (32, [5, 31, 0], 1, 3), (33, list(range(1, 33)), 0, 1), (4, [3, 2, 1, 0], 1, 3)]


@pytest.mark.parametrize("N,bath_state,K,D", CASES)
@pytest.mark.parametrize("order,kernel", [(0, 1), (1, 1), (1, 0)])
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
    if g.kernel_name() == "rhs_hpipe_kernel":
        assert np.array_equal(got, np.conj(np.swapaxes(got, 1, 2)))


@pytest.mark.parametrize("form", [-1, 0])
@pytest.mark.parametrize("sites,K,D,steps", [(1, 2, 6, 400), (2, 1, 4, 1000), (7, 1, 4, 300), (7, 0, 5, 300)])
def test_absorption_propagation_parity(sites, K, D, steps, form):
    """mu_p rho(0) with rho(0) = |0><0|, a non-Hermitian state, propagated with the ground state in the
    basis; every node compared, and Tr(mu_p sigma_0(t)) (heom_expectation) against the oracle's sigma_0."""
    w = workloads.fmo_like()
    w = w.with_(H_cm=w.H_cm[:sites, :sites])
    H, bath_state, dip = workloads.with_ground_state(w)
    o, g = _pair(H, w.lambda_cm, w.nu_per_fs, 77.0, K, D, bath_state, rk4_form=form, ket=0 if form == 0 else 1)
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


# ------------------------------------------------------------- column-sparse states (kernels_ket.cu)
def _ket_system(N, col, seed):
    """Random H with state `col` uncoupled (Eq. 48 block form), baths on every other state."""
    rng = np.random.default_rng(5000 + seed)
    H = rng.normal(0.0, 80.0, (N, N)); H = (H + H.T) / 2
    H[col, :] = 0.0; H[:, col] = 0.0; H[col, col] = rng.normal(0.0, 50.0)
    bath_state = [s for s in range(N) if s != col]
    B = N - 1
    return H, bath_state, rng.uniform(20.0, 45.0, B), rng.uniform(0.015, 0.03, B)


@pytest.mark.parametrize("N,col,K,D,steps", [(8, 0, 1, 4, 200), (8, 7, 0, 5, 200), (5, 2, 2, 4, 150), (3, 1, 3, 5, 100),
                                             (16, 0, 0, 3, 100), (13, 12, 1, 2, 100), (2, 0, 1, 9, 100), (9, 4, 0, 4, 100)])
@pytest.mark.parametrize("order", [1, 0])
def test_ket_kernel_parity(N, col, K, D, steps, order):
    """sigma_0(0) with one non-zero column on an unbathed, uncoupled state: held as kets; the RHS, the RK4 run on
    every node, the populations and Tr(A sigma_0) all against the oracle's full matrices."""
    H, bath_state, lam, nu = _ket_system(N, col, N + K + D)
    o, g = _pair(H, lam, nu, 120.0, K, D, bath_state, order=order)
    rng = np.random.default_rng(N)
    s0 = np.zeros((N, N), dtype=complex)
    s0[:, col] = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    o.set_state(s0); g.set_state(s0)
    if g.nodes * N * N > 2048:
        assert g.kernel_name() == "rhs_ket_kernel"
    assert np.array_equal(g.get_full_state(), o.get_full_state())
    assert rel_err(g.rhs(), o.rhs()) < RHS_TOL
    o.rk4_steps(0.5, steps); g.rk4_steps(0.5, steps)
    ref, got = o.get_full_state(), g.get_full_state()
    assert rel_err(got, ref) < STATE_TOL
    mask = np.ones(N, bool); mask[col] = False
    assert np.abs(got[:, :, mask]).max() == 0.0
    A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    c_ref = np.trace(A @ ref[0])
    assert abs(g.expectation(A) - c_ref) < 1e-11 * max(1.0, abs(c_ref))
    pop, tr = g.populations()
    assert np.allclose(pop, np.diag(ref[0]).real, atol=1e-11) and abs(tr - np.trace(ref[0])) < 1e-11
    # the same run with full matrices (option ket = 0) agrees too, and a later full-state upload leaves ket mode
    g.set_option("ket", 0)
    g.set_state(s0)
    assert g.kernel_name() != "rhs_ket_kernel"
    g.rk4_steps(0.5, steps)
    assert rel_err(g.get_full_state(), ref) < STATE_TOL
    g.set_option("ket", 1)
    g.set_state(s0)
    st = workloads.random_state(o.nodes, N, seed=3)
    o.set_full_state(st); g.set_full_state(st)
    assert g.kernel_name() != "rhs_ket_kernel"
    assert rel_err(g.rhs(), o.rhs()) < RHS_TOL


def test_ket_kernel_not_taken_when_conditions_fail():
    """One non-zero column is not enough: the state of that column must be unbathed AND uncoupled in H."""
    N, K, D = 6, 1, 4
    H, bath_state, lam, nu = _ket_system(N, 0, 1)
    s0 = np.zeros((N, N), dtype=complex); s0[:, 0] = np.arange(1, N + 1)
    # (a) column of a bathed state
    o, g = _pair(H, lam, nu, 120.0, K, D, bath_state)
    s1 = np.zeros((N, N), dtype=complex); s1[:, 2] = np.arange(1, N + 1)
    o.set_state(s1); g.set_state(s1)
    assert g.kernel_name() != "rhs_ket_kernel"
    o.rk4_steps(0.5, 50); g.rk4_steps(0.5, 50)
    assert rel_err(g.get_full_state(), o.get_full_state()) < STATE_TOL
    # (b) unbathed state coupled in H: the other columns fill in
    H2 = H.copy(); H2[0, 3] = H2[3, 0] = 25.0
    o, g = _pair(H2, lam, nu, 120.0, K, D, bath_state)
    o.set_state(s0); g.set_state(s0)
    assert g.kernel_name() != "rhs_ket_kernel"
    o.rk4_steps(0.5, 50); g.rk4_steps(0.5, 50)
    ref = o.get_full_state()
    assert np.abs(ref[:, :, 1:]).max() > 0.0
    assert rel_err(g.get_full_state(), ref) < STATE_TOL
    # (c) two non-zero columns
    o, g = _pair(H, lam, nu, 120.0, K, D, bath_state)
    s2 = s0.copy(); s2[1, 1] = 1.0
    o.set_state(s2); g.set_state(s2)
    assert g.kernel_name() != "rhs_ket_kernel"
