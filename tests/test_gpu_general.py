"""-m gpu: general system-bath operators (heom_create_general: S(b) >= 1 states per bath, several baths per state,
P:84 and the sums over s of Eq. 14-17; two-exciton manifold, Eq. 54) and complex / time-dependent Hamiltonians
(Eq. 51) on the CUDA path, against the oracle, element by element.  SURVEY.md 8(f) next #4."""
import numpy as np
import pytest

import workloads
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-13
STATE_TOL = 1e-10


def rel_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def _pair(H, S, lam, nu, T, K, D, form=0, **opts):
    from paper_1803_03498_b200 import Heom
    o = Oracle(H, lam, nu, T, K, D, bath_states=S, terminator_form=form)
    g = Heom(H, lam, nu, T, K, D, bath_states=S, terminator_form=form, **opts).bind(poison=True)
    return o, g


def _two_exciton(n_sites, seed=0, cplx=False):
    rng = np.random.default_rng(4000 + seed)
    Hs = rng.normal(0.0, 60.0, (n_sites, n_sites)); Hs = (Hs + Hs.T) / 2 + np.diag(rng.uniform(0, 400, n_sites))
    H, S, pairs = workloads.two_exciton_manifold(Hs)
    if cplx:
        A = rng.normal(0.0, 20.0, H.shape)
        H = H + 1j * (A - A.T)
    return H, S


# (n_states, bath lists) of small hand-made systems: shared baths, several baths on one state, unbathed states
HAND = [(4, [[1, 3], [2, 3]]), (5, [[0, 1, 2], [2, 3], [4], [0, 4]]), (3, [[0, 1, 2]]), (6, [[5], [5], [0, 1]])]


@pytest.mark.parametrize("case", range(len(HAND)))
@pytest.mark.parametrize("K,D", [(1, 3), (0, 4)])
@pytest.mark.parametrize("form,order,cplx", [(0, 1, False), (1, 0, False), (0, 1, True)])
def test_general_rhs_parity_small(case, K, D, form, order, cplx):
    N, S = HAND[case]
    rng = np.random.default_rng(500 + case)
    H = rng.normal(0.0, 80.0, (N, N)); H = (H + H.T) / 2
    if cplx:
        A = rng.normal(0.0, 40.0, (N, N)); H = H + 1j * (A - A.T)
    lam = rng.uniform(10, 50, len(S)); nu = rng.uniform(0.01, 0.04, len(S))
    o, g = _pair(H, S, lam, nu, 150.0, K, D, form=form, order=order)
    for a, b in zip(g.tables(), o.tables()):
        assert np.array_equal(a, b)
    for q, (a, b) in enumerate(zip(g.coefficients(), o.coefficients())):
        assert np.allclose(a, b, rtol=1e-11 if q == 3 else 1e-15, atol=1e-300)
    st = workloads.random_state(o.nodes, N, seed=40 + case)
    o.set_full_state(st); g.set_full_state(st)
    assert rel_err(g.rhs(), o.rhs()) < RHS_TOL


@pytest.mark.parametrize("n_sites,K,D,cplx", [(3, 1, 3, False), (4, 0, 3, True), (7, 0, 2, False), (7, 0, 2, True),
                                              (6, 1, 1, False), (9, 0, 1, False), (13, 0, 1, True)])
@pytest.mark.parametrize("form", [0, 1])
def test_two_exciton_rhs_and_rk4_parity(n_sites, K, D, cplx, form):
    """The two-exciton space of Eq. 54 (n_sites = 7 is the paper's FMO case: 29 states): RHS on a dense
    random state, then an RK4 run from a mixed state, every node compared."""
    H, S = _two_exciton(n_sites, seed=n_sites + K, cplx=cplx)
    N = H.shape[0]
    assert N == 1 + n_sites + n_sites * (n_sites - 1) // 2
    o, g = _pair(H, S, 35.0, 0.02, 150.0, K, D, form=form)
    st = workloads.random_state(o.nodes, N, seed=7 + n_sites)
    o.set_full_state(st); g.set_full_state(st)
    assert rel_err(g.rhs(), o.rhs()) < RHS_TOL
    if form == 1 and n_sites > 7:
        return
    s0 = workloads.random_density(N, 3)
    s0 = 0.5 * (s0 + s0.conj().T)                 # Hermitian bit for bit (a matrix product need not be)
    o.set_state(s0); g.set_state(s0)
    steps = 40 if N <= 29 else 10
    o.rk4_steps(0.25, steps); g.rk4_steps(0.25, steps)
    ref, got = o.get_full_state(), g.get_full_state()
    assert rel_err(got, ref) < STATE_TOL
    pop, tr = g.populations()
    assert abs(tr - 1.0) < 1e-12
    if N >= 17 and not (cplx and N > 80):             # (Re H, Im H and sigma of N > 80 do not fit one SM: generic kernel)
        # a density matrix is exactly Hermitian: the one-product variant ran and kept every ADO exactly Hermitian
        assert g.kernel_name() == "rhs_mma_herm_kernel"
        assert np.array_equal(got, np.conj(np.swapaxes(got, 1, 2)))
        # the same run through the general (two-product) variant
        g.set_option("hermitian", 0)
        g.set_state(s0); g.rk4_steps(0.25, steps)
        assert g.kernel_name() == "rhs_mma_kernel"
        assert rel_err(g.get_full_state(), ref) < STATE_TOL


@pytest.mark.parametrize("n_sites,K,D", [(2, 1, 3), (7, 0, 2)])
def test_time_dependent_field_parity(n_sites, K, D):
    """H(t) of Eq. 51 (RWA, Gaussian pulse on a carrier, Eq. 50) on the ground + one-exciton + two-exciton space:
    heom_set_hamiltonian + heom_rk4_stage against oracle_rk4_step_td, every node."""
    H0, S = _two_exciton(n_sites, seed=2)
    N = H0.shape[0]
    rng = np.random.default_rng(9)
    mu = np.zeros((N, N))
    mu[1:n_sites + 1, 0] = rng.normal(0, 1, n_sites)                     # |a><0|
    pairs = [(a, b) for a in range(n_sites) for b in range(a + 1, n_sites)]
    for p, (a, b) in enumerate(pairs):                                   # |ab><a|, |ab><b|
        mu[1 + n_sites + p, 1 + a] = mu[1 + b, 0]
        mu[1 + n_sites + p, 1 + b] = mu[1 + a, 0]
    om = 300.0 / 5308.8

    def Ht(t):
        field = 25.0 * np.exp(-((t - 10.0) / 6.0) ** 2) * np.exp(1j * om * t)
        return workloads.rwa_field_hamiltonian(H0, mu, field)

    o, g = _pair(Ht(0.0), S, 35.0, 0.02, 150.0, K, D, rk4_form=0)
    s0 = np.zeros((N, N), dtype=complex); s0[0, 0] = 1.0
    o.set_state(s0); g.set_state(s0)
    dt = 0.25
    for q in range(80):
        Hs = Ht(q * dt), Ht((q + 0.5) * dt), Ht((q + 1) * dt)
        o.rk4_step_td(dt, *Hs); g.rk4_step_td(dt, *Hs)
    ref, got = o.get_full_state(), g.get_full_state()
    assert np.abs(ref[0][1:, 1:]).max() > 1e-3                           # the pulse did excite the system
    assert rel_err(got, ref) < STATE_TOL
    # a real Hamiltonian on a context created with a real one: the same entry point, hpipe / tiny kernels
    from paper_1803_03498_b200 import Heom
    w = workloads.fmo_like().with_(D=2)
    o2 = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
    g2 = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, rk4_form=0).bind()
    o2.set_state(w.sigma0()); g2.set_state(w.sigma0())
    for q in range(20):
        Hs = [w.H_cm * (1.0 + 0.01 * np.sin(0.1 * (q + f))) for f in (0.0, 0.5, 1.0)]
        o2.rk4_step_td(0.5, *Hs); g2.rk4_step_td(0.5, *Hs)
    assert rel_err(g2.get_full_state(), o2.get_full_state()) < STATE_TOL


def test_general_argument_errors_on_gpu():
    from paper_1803_03498_b200 import Heom, HeomError
    H = np.zeros((3, 3))
    g = Heom(H, [35.0], [0.02], 300.0, 1, 2, bath_states=[[0, 1]]).bind()
    with pytest.raises(HeomError):
        g.set_hamiltonian(np.array([[0, 1j, 0], [-1j, 0, 0], [0, 0, 0]]))     # context was created with a real H
    with pytest.raises(HeomError):
        g.set_hamiltonian(np.array([[0, 1.0, 0], [2.0, 0, 0], [0, 0, 0]]))    # not symmetric
    assert g.kernel_name() in ("rhs_generic_kernel", "rhs_mma_kernel", "rhs_mma_herm_kernel")
