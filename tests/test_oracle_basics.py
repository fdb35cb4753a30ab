"""Pins for the oracle's Philox, sort and potential (CPU only)."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_1206_5878_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- Philox
def test_philox_known_answers(oracle):
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for row in rows:
        w = [int(x, 16) for x in row]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]


def test_philox_counter_and_key_sensitivity(oracle):
    base = oracle.philox4x32_10([5, 0, 7, 9], [1, 2])
    seen = {tuple(base)}
    for pos in range(4):
        c = [5, 0, 7, 9]
        c[pos] += 1
        seen.add(tuple(oracle.philox4x32_10(c, [1, 2])))
    seen.add(tuple(oracle.philox4x32_10([5, 0, 7, 9], [2, 2])))
    seen.add(tuple(oracle.philox4x32_10([5, 0, 7, 9], [1, 3])))
    assert len(seen) == 7


def test_philox_words_uniform(oracle):
    # 4 x 4096 words: mean of the top bit and of the word value
    w = np.array([oracle.philox4x32_10([i, 0, 0, 0], [42, 0]) for i in range(4096)], dtype=np.float64)
    assert abs(w.mean() / 2 ** 32 - 0.5) < 0.01
    assert abs((w >= 2 ** 31).mean() - 0.5) < 0.02


# ----------------------------------------------------------------------------- sort
def _check_sort(oracle, r):
    n = len(r)
    a = np.arange(n, dtype=np.float64) * 3.0
    ids = np.arange(n, dtype=np.uint32)[::-1].copy()
    rs, perm, (a_s,), id_s = oracle.sort_by_radius(r, (a,), ids)
    ref = np.argsort(r, kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(perm, np.lexsort((np.arange(n), r)).astype(np.uint32))
    assert np.array_equal(rs, r[ref])
    assert np.array_equal(a_s, a[ref])
    assert np.array_equal(id_s, ids[ref])
    assert np.all(np.diff(rs) >= 0)


def test_sort_random_and_ties(oracle):
    g = np.random.default_rng(0)
    _check_sort(oracle, g.random(10007) + 1e-3)
    _check_sort(oracle, np.floor(g.random(5000) * 50) + 1.0)          # many exact ties
    _check_sort(oracle, np.full(1000, 2.5))                            # all equal
    _check_sort(oracle, np.sort(g.random(3000) + 1.0))                 # already sorted
    _check_sort(oracle, np.sort(g.random(3000) + 1.0)[::-1].copy())    # reversed
    _check_sort(oracle, 10.0 ** g.uniform(-300, 300, 4000))            # extreme range
    _check_sort(oracle, np.array([1.5]))
    _check_sort(oracle, np.array([2.0, 1.0]))


def test_sort_empty(oracle):
    rs, perm, outs, ids = oracle.sort_by_radius(np.empty(0), (), None)
    assert rs.size == 0 and perm.size == 0


# ----------------------------------------------------------------------------- potential
def _exact_sums(r, m):
    """Exact rational prefix sums of m and suffix sums of fl(m/r), rounded once."""
    n = len(r)
    M = np.empty(n)
    acc = Fraction(0)
    for i in range(n):
        acc += Fraction(float(m[i]))
        M[i] = float(acc)                 # float(Fraction) rounds to nearest-even
    S = np.empty(n)
    acc = Fraction(0)
    for i in range(n - 1, -1, -1):
        S[i] = float(acc)
        acc += Fraction(float(m[i]) / float(r[i]))
    return M, S


@pytest.mark.parametrize("masses", ["equal", "salpeter"])
def test_potential_sums_are_correctly_rounded_exact_sums(oracle, masses):
    c = inputs.plummer(1500, 11, masses)
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    phi, mc = oracle.potential(r, m)
    M, S = _exact_sums(r, m)
    assert np.array_equal(mc, M)
    assert np.array_equal(phi, -(1.0 * (M / r + S)))


@pytest.mark.parametrize("masses", ["equal", "salpeter"])
def test_potential_vs_shell_theorem_brute_force(oracle, masses):
    # Phi_k = -G sum_j m_j / max(r_j, r_k): needs no sort and no prefix sums (O(N^2), N = 2000).
    n, G = 2000, 1.7
    c = inputs.plummer(n, 12, masses)
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    phi, mc = oracle.potential(r, m, G)
    bf = np.array([-G * math.fsum(m / np.maximum(r, rk)) for rk in r])
    assert np.max(np.abs(phi - bf) / np.abs(bf)) < 4e-16 * 3


def test_potential_recursion_eq2_to_eq5(oracle):
    # Phi_{N+1}=0, M_N = sum m, Phi_k = Phi_{k+1} - G M_k (1/r_k - 1/r_{k+1}), M_{k-1} = M_k - m_k
    n = 2000
    c = inputs.plummer(n, 13)
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    phi, mc = oracle.potential(r, m)
    ld = np.longdouble
    rr = np.concatenate([r.astype(ld), [ld(np.inf)]])
    ph = np.zeros(n + 1, dtype=ld)
    Mk = np.sum(m.astype(ld))
    for k in range(n - 1, -1, -1):
        ph[k] = ph[k + 1] - Mk * (1 / rr[k] - 1 / rr[k + 1])
        Mk -= ld(m[k])
    assert np.max(np.abs(ph[:n].astype(np.float64) - phi) / np.abs(phi)) < 1e-13
    # local identity Eq. 4 on the oracle's own output and monotonicity
    lhs = phi[:-1] - phi[1:]
    rhs = -mc[:-1] * (1 / r[:-1] - 1 / r[1:])
    assert np.max(np.abs(lhs - rhs)) < 1e-14
    assert np.all(np.diff(phi) >= 0)
    assert abs(phi[-1] + mc[-1] / r[-1]) <= 2e-16 * abs(phi[-1])     # Phi_N = -G M_N / r_N


def test_potential_hand_cases(oracle):
    phi, mc = oracle.potential([2.0], [3.0], 1.0)
    assert phi[0] == -1.5 and mc[0] == 3.0
    # two stars: Phi_1 = -(m1/r1 + m2/r2), Phi_2 = -(m1+m2)/r2
    phi, mc = oracle.potential([1.0, 4.0], [2.0, 8.0], 0.5)
    assert phi[0] == -0.5 * (2.0 / 1.0 + 8.0 / 4.0)
    assert phi[1] == -0.5 * (10.0 / 4.0)
    assert list(mc) == [2.0, 10.0]
    # exact ties: equal radii give equal potentials
    phi, mc = oracle.potential([1.0, 2.0, 2.0, 2.0, 8.0], [1.0, 1.0, 1.0, 1.0, 4.0])
    assert phi[1] == phi[2] == phi[3] == -(4.0 / 2.0 + 4.0 / 8.0)
    # massless stars do not change anyone's potential
    phi2, _ = oracle.potential([1.0, 1.5, 2.0, 2.0, 2.0, 8.0], [1.0, 0.0, 1.0, 1.0, 1.0, 4.0])
    assert np.array_equal(phi2[[0, 2, 3, 4, 5]], phi)


def test_potential_plummer_closed_form_statistical(oracle):
    # Phi(r) = -1/sqrt(r^2 + a^2), a = 3 pi/16 in N-body units (BASELINE.json: -1/sqrt(1+r^2) in a=1 units).
    n = 200_000
    c = inputs.plummer(n, 14)
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    phi, mc = oracle.potential(r, m)
    a = inputs.A_NBODY
    dev = np.abs(phi + 1.0 / np.sqrt(r * r + a * a))
    assert dev[r > 0.1 * a].max() < 5.0 / math.sqrt(n)
    assert dev.max() < 20.0 / math.sqrt(n)
    # virial sanity: W = 1/2 sum m Phi = -1/2, T = 1/4
    W = 0.5 * np.sum(m * phi)
    T = 0.5 * np.sum(c["m"] * (c["v_r"] ** 2 + c["v_t"] ** 2))
    assert abs(W + 0.5) < 0.01 and abs(T - 0.25) < 0.005


def test_potential_summation_accuracy_at_scale(oracle):
    # R1p: a plain binary64 running sum of N equal masses drifts by ~1e-11 relative at N = 1e6;
    # the oracle's M_k must equal the correctly rounded k/N product-free exact sum.
    n = 1_000_000
    m = np.full(n, 1.0 / n)
    r = np.linspace(1.0, 2.0, n)
    phi, mc = oracle.potential(r, m)
    x = Fraction(1.0 / n)
    for k in (1, 2, 3, 1000, 333_333, 999_999, 1_000_000):
        assert mc[k - 1] == float(x * k)
    naive = np.cumsum(m)
    assert np.max(np.abs(naive - mc) / mc) > 1e-13     # the naive sum really is worse
