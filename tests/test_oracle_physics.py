"""Pins for the oracle's arithmetic: what the paper and the physics fix.

Every expected value below comes from outside the oracle: a textbook closed
form, a library routine (scipy expm, numerical quadrature of the spectral
density), an invariant, or an operator-form brute force on a tiny hierarchy.
Chosen so that a dropped term, a wrong sign or index, a transposed operand or a
misplaced hbar fails at least one test.
"""
import itertools
from math import comb

import numpy as np
import pytest
import scipy.linalg

import workloads
from oracle.oracle import Oracle

HBAR = 5308.8          # cm^-1 fs (BASELINE.json config 1)
KB = 0.6950348         # cm^-1 / K (R3)


def dimer_oracle(**kw):
    w = workloads.dimer()
    args = dict(H=w.H_cm, lam=w.lambda_cm, nu=w.nu_per_fs, T=w.T_kelvin, K=w.K, D=w.D)
    opts = {}
    for k, v in kw.items():
        (args if k in args else opts)[k] = v
    o = Oracle(args["H"], args["lam"], args["nu"], args["T"], args["K"], args["D"], **opts)
    return o


# ------------------------------------------------------------------ coefficients
def test_cot_series_terminator_vanishes():
    """Mittag-Leffler: sum_{k>=0} Re c_k/gamma_k = 2 lambda/(beta hbar^2 nu)
    => the Eq. 14 bracket Delta_b decreases monotonically to 0+ as K grows."""
    H = np.zeros((1, 1))
    prev = None
    for K in (0, 1, 2, 5, 20, 200, 5000):
        o = Oracle(H, 35.0, 0.02, 77.0, K, 0)
        _, _, _, d = o.coefficients()
        assert d[0] > 0.0
        if prev is not None:
            assert d[0] < prev
        prev = d[0]
    # tail of the series ~ sum_{k>K} 4 lam nu/(beta_hbar gamma_k^2) ~ lam nu beta_hbar/(pi^2 K)
    bh = HBAR / (KB * 77.0)
    est = (35.0 / HBAR) * 0.02 * bh / (np.pi ** 2 * 5000)
    assert abs(prev - est) / est < 0.01


def test_high_temperature_limit_of_c0():
    """beta -> 0:  nu lambda cot(beta hbar nu/2) -> 2 lambda/(beta hbar)  (Eq. 20 vs Eq. 14's first term)."""
    H = np.zeros((1, 1))
    T = 3.0e6
    o = Oracle(H, 35.0, 0.02, T, 0, 0)
    g, cr, ci, d = o.coefficients()
    bh = HBAR / (KB * T)
    assert g[0] == 0.02
    assert abs(cr[0] / (2 * (35.0 / HBAR) / bh) - 1) < 1e-6
    assert abs(ci[0] + (35.0 / HBAR) * 0.02) < 1e-18
    assert abs(d[0]) < 1e-6 * cr[0] / 0.02


def test_mode_layout_and_matsubara_frequencies():
    o = Oracle(np.zeros((3, 3)), [10.0, 20.0, 30.0], [0.02, 0.03, 0.04], 150.0, 2, 1)
    g, cr, ci, d = o.coefficients()
    bh = HBAR / (KB * 150.0)
    # l = b*M + k (Eq. 10), gamma(b,0) = nu_b, gamma(b,k) = 2 pi k/(beta hbar) (Eq. 19)
    assert np.allclose(g.reshape(3, 3)[:, 0], [0.02, 0.03, 0.04], rtol=0, atol=0)
    assert np.allclose(g.reshape(3, 3)[:, 1], 2 * np.pi / bh, rtol=1e-15)
    assert np.allclose(g.reshape(3, 3)[:, 2], 4 * np.pi / bh, rtol=1e-15)
    assert np.all(ci.reshape(3, 3)[:, 1:] == 0)
    # c scales linearly with lambda_b
    o2 = Oracle(np.zeros((3, 3)), [20.0, 40.0, 60.0], [0.02, 0.03, 0.04], 150.0, 2, 1)
    assert np.allclose(o2.coefficients()[1], 2 * cr, rtol=1e-14)


# ------------------------------------------------------- commutator, hbar, RK4
def rabi_rho11(t):
    # two-level Rabi formula for H = [[100,100],[100,0]] cm^-1, rho(0) = |1><1|
    Om = np.sqrt(100.0 ** 2 + 4 * 100.0 ** 2)
    return 1.0 - (4 * 100.0 ** 2 / Om ** 2) * np.sin(Om * t / (2 * HBAR)) ** 2


def test_lambda_zero_rabi_and_dt4():
    errs = []
    for dt in (1.0, 0.5, 0.25):
        o = dimer_oracle(lam=0.0)
        o.set_state(workloads.dimer().sigma0())
        o.rk4_steps(dt, int(round(1000 / dt)))
        st = o.get_full_state()
        assert np.all(st[1:] == 0)                       # hierarchy decouples
        rho = st[0]
        errs.append(abs(rho[0, 0].real - rabi_rho11(1000.0)))
        assert abs(np.trace(rho) - 1) < 1e-13
    assert abs(rabi_rho11(1000.0) - 0.485054206890) < 1e-11   # SURVEY 8(c) value of the closed form
    assert errs[0] < 1e-6
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 14.0 < r1 < 18.0 and 14.0 < r2 < 18.0          # global error ~ dt^4


def test_rabi_full_density_matrix():
    """All four elements against expm(-iHt/hbar) rho expm(+iHt/hbar) (library routine)."""
    w = workloads.dimer()
    o = dimer_oracle(lam=0.0)
    rho0 = workloads.random_density(2, 7)
    o.set_state(rho0)
    o.rk4_steps(0.1, 2000)
    U = scipy.linalg.expm(-1j * w.H_cm * 200.0 / HBAR)
    assert np.max(np.abs(o.sigma0() - U @ rho0 @ U.conj().T)) < 1e-10


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("cfg", ["dimer", "trimer_lowT"])
def test_trace_and_hermiticity(cfg):
    if cfg == "dimer":
        o = dimer_oracle()
        rho0 = workloads.dimer().sigma0()
        dt = 1.0
    else:
        rng = np.random.default_rng(3)
        H = rng.normal(0, 60, (3, 3)); H = H + H.T
        o = Oracle(H, [35.0, 20.0, 50.0], [0.02, 0.01, 0.03], 77.0, 2, 3)
        rho0 = workloads.random_density(3, 11)
        dt = 0.5
    o.set_state(rho0)
    # Tr k_0 = 0 identically: commutator traceless, V^x mask vanishes on the diagonal
    k = o.rhs()
    assert abs(np.trace(k[0])) < 1e-18
    o.rk4_steps(dt, 400)
    st = o.get_full_state()
    assert abs(np.trace(st[0]) - 1.0) < 1e-13
    # Hermitian initial data stay Hermitian (all Re c, gamma real)
    assert np.max(np.abs(st - np.conj(np.swapaxes(st, 1, 2)))) < 1e-15
    ev = np.linalg.eigvalsh(st[0])
    assert ev.min() > -1e-6


def test_relaxes_towards_boltzmann():
    """Pins the sign of the V^o (Im c_0) term: populations thermalise, not invert."""
    w = workloads.dimer()
    o = dimer_oracle()
    o.set_state(w.sigma0())
    o.rk4_steps(1.0, 1000)
    pop, tr = o.populations()
    e = np.linalg.eigvalsh(w.H_cm)
    U = np.linalg.eigh(w.H_cm)[1]
    p = np.exp(-e / (KB * w.T_kelvin)); p /= p.sum()
    boltz = (U * p) @ U.T
    assert abs(pop[0] - boltz[0, 0]) < 5e-3       # SURVEY probe: 0.39034 vs 0.39041
    assert pop[0] < 0.45 < 0.55 < pop[1]


# --------------------------------------------------- pure dephasing line shape
def lineshape_from_modes(t, lam, nu, T, K):
    """g(t) for C(t) = sum_k c_k exp(-gamma_k t) + 2 Delta delta(t), complex c_0 (textbook cumulant)."""
    bh = HBAR / (KB * T)
    lam_h = lam / HBAR
    gam = [nu] + [2 * np.pi * k / bh for k in range(1, K + 1)]
    c = [lam_h * nu * (1 / np.tan(bh * nu / 2) - 1j)]
    c += [4 * lam_h * nu * g / (bh * (g * g - nu * nu)) for g in gam[1:]]
    Delta = 2 * lam_h / (bh * nu) - sum(ck.real / g for ck, g in zip(c, gam))
    return sum(ck / g ** 2 * (np.exp(-g * t) + g * t - 1) for ck, g in zip(c, gam)) + Delta * t


def lineshape_from_spectral_density(t, lam, nu, T):
    """g(t) = (1/pi) int_0^inf dw J(w)/w^2 [coth(beta hbar w/2)(1-cos wt) + i(sin wt - wt)],
    J(w) = 2 lam w nu/(w^2+nu^2) (Eq. 6 with Omega = 0), by composite Simpson quadrature.
    Independent of the Matsubara decomposition of Eq. 19-20."""
    bh = HBAR / (KB * T)
    lam_h = lam / HBAR
    wmax = 80.0
    n = int(wmax / (2 * np.pi / t / 64)) // 2 * 2
    w = np.linspace(0.0, wmax, n + 1)
    with np.errstate(divide="ignore", invalid="ignore"):
        pref = 2 * lam_h * nu / (w * (w * w + nu * nu)) / np.pi     # J/(pi w^2)
        re = pref / np.tanh(bh * w / 2) * (1 - np.cos(w * t))
        im = pref * (np.sin(w * t) - w * t)
    re[0] = 2 * lam_h * nu / (np.pi * nu * nu) * (2 / bh) * t * t / 2
    im[0] = 0.0
    h = w[1] - w[0]
    simpson = lambda f: h / 3 * (f[0] + f[-1] + 4 * f[1:-1:2].sum() + 2 * f[2:-1:2].sum())
    tail_re = lam_h * nu / (np.pi * wmax ** 2)           # int 2 lam nu/(pi w^3) dw
    tail_im = -2 * lam_h * nu * t / (np.pi * wmax)       # int -2 lam nu t/(pi w^2) dw
    return simpson(re) + tail_re + 1j * (simpson(im) + tail_im)


@pytest.mark.parametrize("T,K,D,tol", [(77.0, 2, 10, 1e-10), (300.0, 1, 10, 5e-6), (300.0, 1, 6, 2e-3)])
def test_pure_dephasing_closed_form(T, K, D, tol):
    """J = 0: populations constant; rho_12(t) = rho_12(0) exp(-i(e1-e2)t/hbar - g_1(t) - conj(g_2(t))),
    exact as D -> inf (the line-shape function HEOM encodes, P:194 / ref 33).  Pins V^x and V^o
    signs, the complex c_0, the terminator and the Matsubara terms together."""
    H = np.diag([100.0, 0.0])
    lam, nu, t_end, dt = 35.0, 0.02, 200.0, 0.25
    o = Oracle(H, lam, nu, T, K, D)
    rho0 = np.full((2, 2), 0.5, dtype=complex)
    o.set_state(rho0)
    o.rk4_steps(dt, int(t_end / dt))
    rho = o.sigma0()
    g = lineshape_from_modes(t_end, lam, nu, T, K)
    expect = 0.5 * np.exp(-1j * 100.0 * t_end / HBAR - g - np.conj(g))
    assert abs(rho[0, 0] - 0.5) < 1e-13 and abs(rho[1, 1] - 0.5) < 1e-13
    assert abs(rho[0, 1] - expect) < tol
    assert abs(rho[1, 0] - np.conj(expect)) < tol


def test_pure_dephasing_different_baths():
    """Two different baths: distinguishes g_1 from g_2 (site index of V_b) and conj placement."""
    H = np.diag([40.0, -25.0])
    lam, nu, T, K, D = [35.0, 12.0], [0.02, 0.035], 120.0, 2, 9
    o = Oracle(H, lam, nu, T, K, D)
    rho0 = np.array([[0.3, 0.2 - 0.1j], [0.2 + 0.1j, 0.7]])
    o.set_state(rho0)
    o.rk4_steps(0.25, 600)
    rho = o.sigma0()
    g1 = lineshape_from_modes(150.0, lam[0], nu[0], T, K)
    g2 = lineshape_from_modes(150.0, lam[1], nu[1], T, K)
    expect = rho0[0, 1] * np.exp(-1j * 65.0 * 150.0 / HBAR - g1 - np.conj(g2))
    assert abs(rho[0, 1] - expect) < 1e-8
    assert abs(rho[0, 0] - 0.3) < 1e-13


def test_lineshape_against_spectral_density_quadrature():
    """The Matsubara coefficients (Eq. 19-20) + terminator reproduce the line-shape function
    computed straight from the Drude-Lorentz spectral density (Eq. 6), up to the truncated
    Matsubara tail; the oracle's HEOM run matches that same function."""
    lam, nu, T, t_end = 35.0, 0.02, 300.0, 200.0
    g_exact = lineshape_from_spectral_density(t_end, lam, nu, T)
    bh = HBAR / (KB * T)
    for K in (1, 4):
        # what the terminator's delta(t) approximation drops: sum_{k>K} c_k/gamma_k^2 (1 - e^{-gamma_k t})
        gk = 2 * np.pi * np.arange(K + 1, 200000) / bh
        tail = np.sum(4 * (lam / HBAR) * nu / (bh * (gk * gk - nu * nu) * gk) * (1 - np.exp(-gk * t_end)))
        diff = lineshape_from_modes(t_end, lam, nu, T, K) - g_exact
        assert abs(diff.imag) < 1e-9
        assert abs(diff.real - tail) < 0.02 * tail
        assert tail < (3e-4 if K == 1 else 4e-5)
    H = np.diag([100.0, 0.0])
    o = Oracle(H, lam, nu, T, 2, 10)
    o.set_state(np.full((2, 2), 0.5, dtype=complex))
    o.rk4_steps(0.2, 1000)
    rho = o.sigma0()
    expect = 0.5 * np.exp(-1j * 100.0 * t_end / HBAR - g_exact - np.conj(g_exact))
    assert abs(rho[0, 1] - expect) < 2e-4 * abs(expect) + 1e-6


# ------------------------------------------------ rescaling (Eq. 35-36) invariance
def test_sigma0_independent_of_rescaling():
    """Eq. 35-36 is a similarity transform: sigma_0 identical, ADOs related by
    sigma~_n = sigma_n / prod_l sqrt(n_l! s_l^{n_l})."""
    w = workloads.dimer()
    res = {}
    for sc in (0, 1, 2):
        o = dimer_oracle(scaling=sc)
        o.set_state(w.sigma0())
        o.rk4_steps(1.0, 300)
        res[sc] = o.get_full_state()
        if sc == 1:
            t, _, _ = o.tables()
            _, cr, ci, _ = o.coefficients()
    for sc in (1, 2):
        assert np.max(np.abs(res[sc][0] - res[0][0])) < 5e-15
    from math import factorial
    for s, sc in ((np.abs(cr), 1), (np.hypot(cr, ci), 2)):
        scale = np.array([np.prod([np.sqrt(factorial(n) * s[l] ** n) for l, n in enumerate(tt)])
                          for tt in t.astype(int)])
        assert np.max(np.abs(res[sc] * scale[:, None, None] - res[0])) < 1e-13 * np.abs(res[0]).max() + 1e-18


# ------------------------------------------------------------- depth convergence
def test_depth_convergence():
    w = workloads.dimer()
    vals = []
    for D in (2, 4, 6, 8, 10):
        o = dimer_oracle(D=D)
        o.set_state(w.sigma0())
        o.rk4_steps(1.0, 1000)
        vals.append(o.populations()[0][0])
    d = np.abs(np.diff(vals))
    assert np.all(d[1:] < d[:-1]) and d[-1] < 1e-7
    # SURVEY 8(c) probe values (independent survey-time evaluation, not from the paper)
    probe = [0.390429520, 0.390339686, 0.390314975, 0.390313999, 0.390313979]
    assert np.max(np.abs(np.array(vals) - probe)) < 1e-9


# --------------------------------------- operator-form brute force on a tiny hierarchy
def operator_form_rhs(H, lam, nu, T, K, D, state, tuples):
    """The hierarchy written with projectors P_b = |b><b| and matrix (anti)commutators
    (V^x A = [P,A], V^o A = {P,A}; unscaled Eq. 12-17), nodes found through a dict.
    A different route to the same numbers than the oracle's elementwise masks."""
    N = H.shape[0]
    M = K + 1
    bh = HBAR / (KB * T)
    idx = {tuple(int(v) for v in n): u for u, n in enumerate(tuples)}
    out = np.zeros_like(state)
    P = [np.diag((np.arange(N) == b).astype(float)) for b in range(N)]
    comm = lambda A, B: A @ B - B @ A
    acomm = lambda A, B: A @ B + B @ A
    for n, u in idx.items():
        s = state[u]
        r = -1j / HBAR * comm(H, s)
        for b in range(N):
            lam_h = lam[b] / HBAR
            gam = [nu[b]] + [2 * np.pi * k / bh for k in range(1, M)]
            c = [lam_h * nu[b] / np.tan(bh * nu[b] / 2)] + \
                [4 * lam_h * nu[b] * g / (bh * (g * g - nu[b] ** 2)) for g in gam[1:]]
            Delta = 2 * lam_h / (bh * nu[b]) - sum(ck / g for ck, g in zip(c, gam))
            r = r - Delta * comm(P[b], comm(P[b], s))
            for k in range(M):
                l = b * M + k
                r = r - n[l] * gam[k] * s
                up = tuple(v + (i == l) for i, v in enumerate(n))
                dn = tuple(v - (i == l) for i, v in enumerate(n))
                if up in idx:
                    r = r + 1j * comm(P[b], state[idx[up]])
                if n[l] > 0:
                    th = 1j * c[k] * comm(P[b], state[idx[dn]])
                    if k == 0:
                        th = th + lam_h * nu[b] * acomm(P[b], state[idx[dn]])
                    r = r + n[l] * th
        out[u] = r
    return out


@pytest.mark.parametrize("N,K,D", [(2, 1, 3), (3, 0, 3), (3, 2, 2)])
def test_rhs_against_operator_form(N, K, D):
    rng = np.random.default_rng(100 + N + K + D)
    H = rng.normal(0, 80, (N, N)); H = H + H.T
    lam = rng.uniform(10, 50, N); nu = rng.uniform(0.01, 0.04, N)
    o = Oracle(H, lam, nu, 140.0, K, D, scaling=0)
    t, _, _ = o.tables()
    st = workloads.random_state(o.nodes, N, seed=5)
    o.set_full_state(st)
    ref = operator_form_rhs(H, lam, nu, 140.0, K, D, st, t)
    got = o.rhs()
    assert np.max(np.abs(got - ref)) < 1e-14 * np.abs(ref).max() + 1e-16
    # sampled-node entry point agrees with the full sweep
    ids = np.array([0, o.nodes - 1, o.nodes // 2])
    assert np.array_equal(o.rhs_nodes(ids), got[ids])


# ------------------------------------------------- whole pipeline vs dense expm
def test_dense_liouvillian_expm():
    """Build the 280 x 280 Liouvillian of the dimer config column by column from rhs();
    1000 RK4 steps must equal (I + dtL + (dtL)^2/2 + (dtL)^3/6 + (dtL)^4/24)^1000 to rounding
    (pins the RK4 tableau) and expm(1000 dt L) (scipy) to O(dt^4)."""
    w = workloads.dimer()
    o = dimer_oracle()
    n = o.nodes * 4
    L = np.zeros((n, n), dtype=complex)
    for q in range(n):
        e = np.zeros(n, dtype=complex); e[q] = 1.0
        o.set_full_state(e.reshape(o.nodes, 2, 2))
        L[:, q] = o.rhs().reshape(-1)
    y0 = np.zeros(n, dtype=complex); y0[0] = 1.0
    o.set_state(w.sigma0())
    o.rk4_steps(1.0, 1000)
    y = o.get_full_state().reshape(-1)
    A = np.eye(n) + L + L @ L / 2 + L @ L @ L / 6 + L @ L @ L @ L / 24
    y_poly = np.linalg.matrix_power(A, 1000) @ y0
    assert np.max(np.abs(y - y_poly)) < 1e-12
    y_exp = scipy.linalg.expm(1000.0 * L) @ y0
    assert np.max(np.abs(y - y_exp)) < 2e-6
    # and with dt halved the distance to expm drops ~16x
    o.set_state(w.sigma0()); o.rk4_steps(0.5, 2000)
    y2 = o.get_full_state().reshape(-1)
    ratio = np.max(np.abs(y - y_exp)) / np.max(np.abs(y2 - y_exp))
    assert 12.0 < ratio < 20.0


def test_golden_dimer_trajectory():
    """SURVEY.md 8(c) cross-check trajectory of BASELINE config 1 (independent survey-time probe)."""
    w = workloads.dimer()
    o = dimer_oracle()
    o.set_state(w.sigma0())
    expect = {1: (0.999645320015321, 0.000176459621133 + 0.018823291055129j, 1.000134329431380),
              10: (0.965396598401502, 0.016247706727028 + 0.179312925292194j, 1.010740838957410),
              100: (0.433607186172902, -0.018148894890768 - 0.146257030921921j, 0.646195611503115),
              1000: (0.390339686027749, -0.208198771289495 + 0.000096617121423j, 0.827715714127886)}
    done = 0
    for s in sorted(expect):
        o.rk4_steps(1.0, s - done); done = s
        st = o.get_full_state()
        r11, r12, nrm = expect[s]
        assert abs(st[0][0, 0].real - r11) < 2e-13
        assert abs(st[0][0, 1] - r12) < 2e-13
        assert abs((np.abs(st) ** 2).sum() - nrm) < 2e-12


def test_terminator_switch_identifies_variant():
    """rho_11 with the Eq. 14 terminator off (independent probe values)."""
    w = workloads.dimer()
    o = dimer_oracle(terminator=0)
    o.set_state(w.sigma0())
    o.rk4_steps(1.0, 1000)
    assert abs(o.populations()[0][0] - 0.385853809100661) < 2e-13


def test_argument_validation():
    H = np.array([[0.0, 1.0], [2.0, 0.0]])
    with pytest.raises(ValueError):
        Oracle(H, 35.0, 0.02, 300.0, 1, 2)              # not symmetric
    with pytest.raises(ValueError):
        Oracle(np.zeros((2, 2)), 35.0, 0.02, -1.0, 1, 2)
    with pytest.raises(ValueError):
        Oracle(np.zeros((2, 2)), 35.0, 0.0, 300.0, 1, 2)
    assert comb(8, 4) == Oracle(np.zeros((2, 2)), 35.0, 0.02, 300.0, 1, 4).nodes
