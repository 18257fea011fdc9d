"""Pins for the oracle's hierarchy enumeration and +/- link tables.

Nothing here compares the oracle with itself: the expected values are closed
forms (Eq. 9), numbers printed in the paper (tests/golden/paper_values.txt),
structural identities, and a brute-force enumeration with itertools.
"""
import itertools
import os
from math import comb

import numpy as np
import pytest

from oracle.oracle import Oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val, _cite = [s.strip() for s in line.split("|", 2)]
            out[name] = float(val)
    return out


def make(N, K, D):
    H = np.zeros((N, N))
    return Oracle(H, 35.0, 0.02, 300.0, K, D)


def test_paper_printed_counts():
    g = golden()
    # Eq. 9 at the paper's reference hierarchy: W = 7*6 = 42, D = 6.
    assert comb(42 + 6, 6) == int(g["n_matrices_B7_K6_D6"])
    # the printed 44964388 is a typo; C(41,6) = 4496388 reproduces "3.3 GiB".
    n = comb(35 + 6, 6)
    assert n == 4496388 and n != int(g["n_matrices_B7_K5_D6_printed"])
    gib = n * 49 * 16 / 2 ** 30
    assert abs(gib - g["gib_per_copy_B7_K5_D6"]) < 0.05
    assert abs(int(g["n_matrices_B7_K5_D6_printed"]) * 49 * 16 / 2 ** 30 - 3.3) > 20


@pytest.mark.parametrize("N,K,D", [(2, 1, 4), (7, 0, 3), (7, 1, 4), (7, 5, 3), (7, 4, 4),
                                   (3, 2, 6), (1, 0, 5), (2, 0, 0), (14, 0, 5), (96, 0, 2)])
def test_count_and_link_closed_forms(N, K, D):
    o = make(N, K, D)
    W = N * (K + 1)
    assert o.W == W
    assert o.nodes == comb(W + D, W)                      # Eq. 9
    t, p, m = o.tables()
    lev = t.sum(axis=1)
    # level-major with level sizes C(L+W-1, W-1)
    assert np.all(np.diff(lev.astype(int)) >= 0)
    for L in range(D + 1):
        assert int((lev == L).sum()) == comb(L + W - 1, W - 1)
    valid = W * comb(W + D - 1, D - 1) if D > 0 else 0
    assert int((p >= 0).sum()) == valid
    assert int((m >= 0).sum()) == valid
    # P:90 validity rules
    assert np.array_equal(p >= 0, np.repeat((lev < D)[:, None], W, axis=1))
    assert np.array_equal(m >= 0, t > 0)
    # link symmetry and tuple arithmetic
    u, l = np.nonzero(p >= 0)
    assert np.array_equal(m[p[u, l], l], u)
    e = np.zeros_like(t[u]); e[np.arange(u.size), l] = 1
    assert np.array_equal(t[p[u, l]], t[u] + e)
    u, l = np.nonzero(m >= 0)
    assert np.array_equal(p[m[u, l], l], u)
    # first nodes: u(0) = 0, u(e_l) = 1 + l, last node (0,..,0,D)
    assert not t[0].any()
    if D >= 1:
        assert np.array_equal(p[0], 1 + np.arange(W))
    assert t[-1, -1] == D and t[-1].sum() == D


@pytest.mark.parametrize("W,D", [(1, 6), (2, 5), (3, 4), (4, 6), (4, 4)])
def test_brute_force_small(W, D):
    # N = W sites with K = 0 gives a tuple of length W.
    o = make(W, 0, D)
    t, p, m = o.tables()
    allt = [n for n in itertools.product(range(D + 1), repeat=W) if sum(n) <= D]
    # pinned order: level ascending, inside a level descending lexicographic
    allt.sort(key=lambda n: (sum(n), tuple(-x for x in n)))
    assert len(allt) == o.nodes
    assert np.array_equal(t, np.array(allt, dtype=np.uint8).reshape(-1, W))
    idx = {n: u for u, n in enumerate(allt)}
    for u, n in enumerate(allt):
        for l in range(W):
            up = tuple(x + (i == l) for i, x in enumerate(n))
            dn = tuple(x - (i == l) for i, x in enumerate(n))
            assert p[u, l] == idx.get(up, -1)
            assert m[u, l] == (idx[dn] if n[l] > 0 else -1)


def _checksums(T):
    """h1 = sum (T+1)(l+1), h2 = sum (T+1)((u mod 65521)+1), both mod 2^64."""
    nodes, W = T.shape
    Tp = (T.astype(np.int64) + 1).astype(np.uint64)
    lw = (np.arange(W, dtype=np.uint64) + np.uint64(1))[None, :]
    uw = ((np.arange(nodes, dtype=np.uint64) % np.uint64(65521)) + np.uint64(1))[:, None]
    with np.errstate(over="ignore"):
        h1 = int((Tp * lw).sum(dtype=np.uint64))
        h2 = int((Tp * uw).sum(dtype=np.uint64))
    return int(T[T >= 0].astype(np.int64).sum()), h1, h2


# Cross-check values from an independent survey-time enumeration (
# NOT from the paper and not from any code in this repository).
SURVEY_CHECKS = {
    (2, 1, 4): (5246, 2380, 13976, 122561, 6300, 122561),
    (7, 1, 8): (266843672200, 94646454840, 2067401366940, 8701842624013419,
                709860620700, 3163845708648120),
    (7, 1, 12): (307620673231800, 139078872118200, 2351115053793228, 10115670477738734324,
                 1043092008913500, 4550830205369578669),          # cfg3: W = 14, D = 12, 9 657 700 nodes
    (96, 0, 3): (36002339968, 1084140288, 1983102012080, 107104809694540,
                 52602933936, 32955572434587),
}


@pytest.mark.parametrize("cfg", list(SURVEY_CHECKS))
def test_survey_cross_check_values(cfg):
    N, K, D = cfg
    o = make(N, K, D)
    _, p, m = o.tables()
    sp, h1p, h2p = _checksums(p)
    sm, h1m, h2m = _checksums(m)
    assert (sp, sm, h1p, h2p, h1m, h2m) == SURVEY_CHECKS[cfg]


def test_dimer_first_rows():
    # SURVEY.md section 8(c) C1 "cfg1 first rows" (independent survey-time enumeration).
    o = make(2, 1, 4)
    t, p, m = o.tables()
    assert list(p[0]) == [1, 2, 3, 4]
    assert list(t[1]) == [1, 0, 0, 0] and list(p[1]) == [5, 6, 7, 8] and list(m[1]) == [0, -1, -1, -1]
    assert list(t[4]) == [0, 0, 0, 1] and list(p[4]) == [8, 11, 13, 14] and list(m[4]) == [-1, -1, -1, 0]
    assert list(t[14]) == [0, 0, 0, 2] and list(p[14]) == [24, 30, 33, 34] and list(m[14]) == [-1, -1, -1, 4]
    assert list(t[35]) == [4, 0, 0, 0] and list(p[35]) == [-1] * 4 and list(m[35]) == [15, -1, -1, -1]
    assert list(t[69]) == [0, 0, 0, 4] and list(m[69]) == [-1, -1, -1, 34]
