"""-m "not gpu": the C-ABI library loads, exports every declared symbol, and its host-side
hierarchy / coefficient builder (closed-form ranks) matches the oracle's tables bit for bit
(enumeration + bisection) and its coefficients to rounding.  No compute call is made."""
import re
import os

import numpy as np
import pytest

import workloads
from oracle.oracle import Oracle
from paper_1803_03498_b200 import Heom, HeomError, load_library, SYMBOLS
from paper_1803_03498_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    libbuild.build()


def test_exports_every_declared_symbol():
    lib = load_library()
    hdr = open(os.path.join(ROOT, "include", "heom.h")).read()
    declared = sorted(set(re.findall(r"\b(heom_[a-z0-9_]+)\s*\(", hdr)))
    assert declared == sorted(SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


CASES = [(2, 1, 4), (7, 1, 4), (7, 0, 5), (3, 2, 6), (14, 0, 4), (96, 0, 2), (1, 0, 3), (2, 0, 0),
         (5, 3, 3)]


@pytest.mark.parametrize("N,K,D", CASES)
@pytest.mark.parametrize("order", [0, 1])
def test_tables_bit_exact_vs_oracle(N, K, D, order):
    H = np.zeros((N, N))
    o = Oracle(H, 35.0, 0.02, 300.0, K, D)
    g = Heom(H, 35.0, 0.02, 300.0, K, D, order=order)
    assert g.nodes == o.nodes and g.W == o.W
    for a, b in zip(g.tables(), o.tables()):
        assert a.dtype == b.dtype and np.array_equal(a, b)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_tables_bit_exact_baseline_configs(name):
    w = workloads.get(name)
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
    g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D)
    assert g.nodes == w.nodes == o.nodes
    for a, b in zip(g.tables(), o.tables()):
        assert np.array_equal(a, b)
    for q, (a, b) in enumerate(zip(g.coefficients(), o.coefficients())):
        # delta (q == 3) is a difference of nearly equal terms: rounding amplified ~100x
        assert np.allclose(a, b, rtol=1e-12 if q == 3 else 4e-16, atol=0)


@pytest.mark.parametrize("T,K", [(300.0, 1), (77.0, 3), (30.0, 6)])
def test_coefficients_vs_oracle(T, K):
    H = np.zeros((3, 3))
    lam, nu = [35.0, 0.0, 12.5], [0.02, 0.025, 0.01]
    o = Oracle(H, lam, nu, T, K, 2)
    g = Heom(H, lam, nu, T, K, 2)
    for q, (a, b) in enumerate(zip(g.coefficients(), o.coefficients())):
        assert np.allclose(a, b, rtol=1e-11 if q == 3 else 1e-15, atol=1e-300)


def test_argument_validation_without_gpu():
    with pytest.raises(HeomError):
        Heom(np.array([[0.0, 1.0], [2.0, 0.0]]), 35.0, 0.02, 300.0, 1, 2)     # not symmetric
    with pytest.raises(HeomError):
        Heom(np.zeros((2, 2)), 35.0, 0.02, 0.0, 1, 2)                          # T = 0
    with pytest.raises(HeomError):
        Heom(np.zeros((2, 2)), -1.0, 0.02, 300.0, 1, 2)                        # lambda < 0
    with pytest.raises(HeomError):
        Heom(np.zeros((2, 2)), 35.0, float("nan"), 300.0, 1, 2)
    g = Heom(np.zeros((2, 2)), 35.0, 0.02, 300.0, 1, 2)
    assert g.workspace_bytes() >= 4 * 16 * 4 * g.nodes
    with pytest.raises(HeomError) as e:
        g.set_state(np.eye(2))                       # no workspace bound
    assert e.value.status == -4
    with pytest.raises(HeomError):
        g.set_option("no_such_option", 1)


def test_option_validation_without_gpu():
    g = Heom(np.zeros((3, 3)), 35.0, 0.02, 300.0, 2, 2)
    for name, good, bad in [("order", 0, 2), ("kernel", 2, 3), ("rk4_form", 0, 2), ("l2_fetch", 64, 48),
                            ("warps_per_cta", 4, 99)]:
        g.set_option(name, good)
        with pytest.raises(HeomError) as e:
            g.set_option(name, bad)
        assert e.value.status == -1
    for name in ("timing", "hermitian", "ket", "pade"):
        g.set_option(name, 1)
        g.set_option(name, 0)


def test_no_cpu_fallback():
    """Without a GPU the compute path must fail loudly, never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = Heom(np.zeros((2, 2)), 35.0, 0.02, 300.0, 1, 2)
    with pytest.raises(HeomError) as e:
        g.bind()
    assert e.value.status == -3
    # raw bind with a fake pointer must report the missing device too
    with pytest.raises(HeomError) as e:
        g.bind_raw(256, g.workspace_bytes())
    assert e.value.status == -3


# ------------------------------------------------ bath -> state map (heom_create_sites)
@pytest.mark.parametrize("N,bath_state,K,D", [(2, [1], 2, 5), (8, [1, 2, 3, 4, 5, 6, 7], 1, 3), (4, [3, 0], 1, 4),
                                               (33, list(range(1, 33)), 0, 2), (3, [2, 1, 0], 0, 3)])
def test_site_map_tables_and_coefficients_vs_oracle(N, bath_state, K, D):
    H = np.zeros((N, N))
    B = len(bath_state)
    lam = np.linspace(20.0, 40.0, B); nu = np.linspace(0.02, 0.03, B)
    o = Oracle(H, lam, nu, 150.0, K, D, bath_state=bath_state)
    g = Heom(H, lam, nu, 150.0, K, D, bath_state=bath_state)
    assert g.nodes == o.nodes and g.W == o.W == B * (K + 1) and g.B == B
    for a, b in zip(g.tables(), o.tables()):
        assert a.dtype == b.dtype and np.array_equal(a, b)
    for q, (a, b) in enumerate(zip(g.coefficients(), o.coefficients())):
        assert a.shape == b.shape
        assert np.allclose(a, b, rtol=1e-11 if q == 3 else 1e-15, atol=1e-300)
    # workspace: 4 state buffers of n_states x n_states matrices
    assert g.workspace_bytes() >= 4 * 16 * N * N * g.nodes


def test_site_map_validation():
    H = np.zeros((3, 3))
    for bad in ([1, 1], [3], [-1], [0, 1, 2, 0], []):
        with pytest.raises(HeomError):
            Heom(H, 35.0, 0.02, 300.0, 0, 2, bath_state=bad)


def test_general_create_validation_without_gpu():
    """heom_create_general argument checking and host tables (no CUDA call)."""
    H = np.zeros((4, 4))
    g = Heom(H, [35.0, 20.0], [0.02, 0.03], 300.0, 1, 3, bath_states=[[1, 3], [2, 3]])
    o = Oracle(H, [35.0, 20.0], [0.02, 0.03], 300.0, 1, 3, bath_states=[[1, 3], [2, 3]])
    assert g.nodes == o.nodes and g.W == o.W == 4
    for a, b in zip(g.tables(), o.tables()):
        assert np.array_equal(a, b)
    for bad in ([[1, 1]], [[4]], [[0], []]):
        with pytest.raises(HeomError):
            Heom(H, [35.0] * len(bad), [0.02] * len(bad), 300.0, 1, 2, bath_states=bad)
    with pytest.raises(HeomError):
        Heom(np.array([[0, 1j], [1j, 0]]), [35.0], [0.02], 300.0, 1, 2, bath_states=[[0]])   # not Hermitian
    for name, good, bad in [("terminator_form", 1, 2)]:
        g.set_option(name, good)
        with pytest.raises(HeomError):
            g.set_option(name, bad)


def test_level_max_static_rejects_bad_arguments_without_a_gpu():
    """heom_level_max_static checks its arguments before any CUDA call: depth beyond HEOM_STATIC_MAX_DEPTH, NULL
    pointers and sizes out of range return HEOM_EINVAL with a message, with or without a device."""
    import ctypes as C
    from paper_1803_03498_b200 import STATIC_MAX_DEPTH
    lib = load_library()
    hdr = open(os.path.join(ROOT, "include", "heom.h")).read()
    assert f"#define HEOM_STATIC_MAX_DEPTH {STATIC_MAX_DEPTH}" in hdr
    fake = 0x1000                                   # never dereferenced: the call fails before touching memory
    assert lib.heom_level_max_static(0, fake, fake, 3, 4, STATIC_MAX_DEPTH + 1, fake, None) == -1
    assert b"outside 0..63" in lib.heom_static_last_error()
    assert lib.heom_level_max_static(0, None, fake, 3, 4, 2, fake, None) == -1
    assert b"NULL" in lib.heom_static_last_error()
    assert lib.heom_level_max_static(0, fake, fake, -1, 4, 2, fake, None) == -1
    assert lib.heom_level_max_static(-1, fake, fake, 3, 4, 2, fake, None) == -1
    assert b"device" in lib.heom_static_last_error()
