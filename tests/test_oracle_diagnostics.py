"""Pins for the oracle's diagnostics (CPU only): half-mass and Lagrange radii, kinetic and
potential energy, virial ratio, half-mass relaxation time (PAPER.md:140, :346 Eq. 20, :354;
DESIGN.md R15-R17).  Each pin is something other than the oracle's own formula: exact rational
pair sums, numpy's searchsorted, Plummer closed forms, scaling laws."""
import math
from fractions import Fraction

import numpy as np
import pytest

from paper_1206_5878_b200 import inputs


def sorted_cluster(oracle, n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    phi, mc = oracle.potential(rs, ms)
    return rs, vrs, vts, ms, phi, mc


def test_energies_against_exact_pair_sums(oracle):
    """W = 1/2 sum m_k Phi_k must equal the pair sum -G [sum_{i<j} m_i m_j / max(r_i, r_j) + 1/2 sum m_i^2 / r_i]
    (shell theorem; the second term is the self term Eq. 1 contains at r = r_k), T = 1/2 sum m v^2: both in
    exact rational arithmetic from the inputs, to a few ulps (the oracle rounds each term, then sums exactly)."""
    g = np.random.default_rng(2)
    n = 300
    r = np.sort(g.uniform(0.1, 5.0, n))
    m = g.uniform(0.5, 2.0, n) / n
    vr, vt = g.normal(0, 0.5, n), g.normal(0, 0.5, n)
    phi, mc = oracle.potential(r, m)
    d = oracle.diagnostics(r, vr, vt, m, phi, mc)
    F = Fraction
    R, M = [F(float(x)) for x in r], [F(float(x)) for x in m]
    W = F(0)
    for i in range(n):
        W -= M[i] * M[i] / R[i] / 2
        for j in range(i + 1, n):
            W -= M[i] * M[j] / R[j]                      # r sorted: max(r_i, r_j) = r_j
    T = sum(M[i] * (F(float(vr[i])) ** 2 + F(float(vt[i])) ** 2) / 2 for i in range(n))
    assert abs(d["W"] - float(W)) <= 1e-14 * abs(float(W))
    assert abs(d["T"] - float(T)) <= 1e-15 * float(T)
    assert d["E_tot"] == d["T"] + d["W"]
    assert abs(d["virial_ratio"] - float(2 * T / -W)) <= 1e-14 * float(2 * T / -W)
    assert d["M"] == mc[-1]


def test_lagrange_radii_against_searchsorted(oracle):
    rs, vrs, vts, ms, phi, mc = sorted_cluster(oracle, 20_000, 5, "salpeter")
    fr = np.array([1e-9, 0.001, 0.01, 0.1, 0.25, 0.5, 0.75, 0.9, 0.99, 1.0])
    d = oracle.diagnostics(rs, vrs, vts, ms, phi, mc, fr)
    k = np.minimum(np.searchsorted(mc, fr * mc[-1], side="left"), len(rs) - 1)
    assert np.array_equal(d["lagrange"], rs[k])
    assert d["lagrange"][0] == rs[0] and d["lagrange"][-1] == rs[-1]
    assert np.all(np.diff(d["lagrange"]) >= 0)
    assert d["r_h"] == d["lagrange"][5]
    # more than the whole mass asked for: the outermost star
    assert oracle.diagnostics(rs, vrs, vts, ms, phi, mc, [1.5])["lagrange"][0] == rs[-1]


def test_two_star_hand_case(oracle):
    """m = (1/4, 3/4) at r = (1, 2): M_1 = 1/4 < 1/2 <= M_2, so r_h = 2; Phi_1 = -(1/4 + 3/8), Phi_2 = -1/2;
    W = 1/2 (1/4 * -5/8 + 3/4 * -1/2) = -17/64; T = 1/2 (1/4 * 1 + 3/4 * 4) = 13/8; all exact in binary64."""
    r, m = np.array([1.0, 2.0]), np.array([0.25, 0.75])
    vr, vt = np.array([1.0, 0.0]), np.array([0.0, 2.0])
    phi, mc = oracle.potential(r, m)
    d = oracle.diagnostics(r, vr, vt, m, phi, mc, [0.25, 0.26])
    assert d["r_h"] == 2.0 and d["M"] == 1.0
    assert d["W"] == -17.0 / 64.0 and d["T"] == 13.0 / 8.0 and d["E_tot"] == 13.0 / 8.0 - 17.0 / 64.0
    assert d["virial_ratio"] == (13.0 / 4.0) / (17.0 / 64.0)
    assert list(d["lagrange"]) == [1.0, 2.0]              # M_1 = 1/4 reaches the fraction 1/4 exactly
    assert d["t_rh"] == pytest.approx(0.138 * 2 / math.log(0.2) * math.sqrt(8.0), rel=1e-15)


def test_plummer_closed_forms(oracle):
    """Plummer sphere in N-body units (G = M = 1, a = 3 pi / 16): r_h = a / sqrt(2^(2/3) - 1), T = 1/4, W = -1/2,
    virial ratio 1, E = -1/4 -- statistically, to a few / sqrt(N); t_rh from Eq. 20 with that r_h."""
    n = 200_000
    rs, vrs, vts, ms, phi, mc = sorted_cluster(oracle, n, 8)
    d = oracle.diagnostics(rs, vrs, vts, ms, phi, mc)
    a = 3 * math.pi / 16
    tol = 5 / math.sqrt(n)
    assert abs(d["r_h"] / (a / math.sqrt(2 ** (2 / 3) - 1)) - 1) < tol
    assert abs(d["T"] / 0.25 - 1) < tol and abs(d["W"] / -0.5 - 1) < tol
    assert abs(d["virial_ratio"] - 1) < 2 * tol and abs(d["E_tot"] / -0.25 - 1) < 2 * tol
    assert abs(d["M"] - 1) < 1e-12
    assert d["t_rh"] == pytest.approx(0.138 * n / math.log(0.1 * n) * math.sqrt(d["r_h"] ** 3), rel=1e-14)


def test_scaling_laws(oracle):
    """Radii x4, masses x2 (powers of two: exact): T x2, W x(4/4) = x1 ... precisely: Phi ~ M / r scales by 2/4,
    so W ~ M Phi by 2 * 1/2 = 1, T ~ M v^2 by 2; r_h x4; t_rh ~ (r_h^3 / (G M))^(1/2) by (64 / 2)^(1/2);
    doubling G instead scales W by 2 and t_rh by 2^(-1/2)."""
    rs, vrs, vts, ms, phi, mc = sorted_cluster(oracle, 5_000, 3)
    d0 = oracle.diagnostics(rs, vrs, vts, ms, phi, mc, [0.1, 0.9])
    r2, m2 = rs * 4.0, ms * 2.0
    phi2, mc2 = oracle.potential(r2, m2)
    d1 = oracle.diagnostics(r2, vrs, vts, m2, phi2, mc2, [0.1, 0.9])
    assert d1["T"] == 2.0 * d0["T"] and d1["W"] == d0["W"] and d1["r_h"] == 4.0 * d0["r_h"]
    assert np.array_equal(d1["lagrange"], 4.0 * d0["lagrange"])
    assert d1["t_rh"] == pytest.approx(d0["t_rh"] * math.sqrt(32.0), rel=1e-15)
    phi3, mc3 = oracle.potential(rs, ms, G=2.0)
    d2 = oracle.diagnostics(rs, vrs, vts, ms, phi3, mc3, G=2.0)
    assert d2["W"] == 2.0 * d0["W"] and d2["T"] == d0["T"]
    assert d2["t_rh"] == pytest.approx(d0["t_rh"] / math.sqrt(2.0), rel=1e-15)
