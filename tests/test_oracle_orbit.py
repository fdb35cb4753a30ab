"""Pins for the oracle's turning points (S3) and new-radius draw (S4), CPU only.

Every expected value here comes from a closed form, a brute force written differently from
the oracle (literal Eq. 12 with the division, linear scans, shell-theorem sums without
prefix sums) or a statistical law -- never from the CUDA path.
"""
import math

import numpy as np
import pytest
from scipy import stats

from paper_1206_5878_b200 import inputs


def sorted_cluster(n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    o = np.argsort(c["r"], kind="stable")
    return {k: v[o] for k, v in c.items() if isinstance(v, np.ndarray)}


def phi_brute(r, m, x, G=1.0):
    """Shell theorem at an arbitrary radius: Phi(x) = -G sum_j m_j / max(r_j, x)  (== Eq. 1)."""
    return -G * math.fsum(m / np.maximum(r, x))


def kepler_table(n=4000, rlo=1e-2, rhi=1e2):
    """Unit point mass at tiny radius plus massless tracers: Phi = -1/r on the whole grid."""
    r = np.concatenate([[1e-9], np.geomspace(rlo, rhi, n - 1)])
    m = np.zeros(n)
    m[0] = 1.0
    return r, m


# ----------------------------------------------------------------------------- S3
@pytest.mark.parametrize("masses,seed", [("equal", 21), ("salpeter", 22)])
def test_brackets_vs_linear_scan_of_literal_eq12(oracle, masses, seed):
    n = 2000
    c = sorted_cluster(n, seed, masses)
    phi, mc = oracle.potential(c["r"], c["m"])
    tp = oracle.orbit_turning_points(c["r"], c["v_r"], c["v_t"], phi, mc)
    assert np.all(tp["status"] == 0)
    # node arrays with sentinels, paper numbering 0..N+1
    R = np.concatenate([[0.0], c["r"], [np.inf]])
    PH = np.concatenate([[phi[0]], phi, [0.0]])
    kmin = np.empty(n, np.int64)
    kmax = np.empty(n, np.int64)
    contiguous = 0
    for a in range(n):
        k = a + 1
        E = phi[a] + 0.5 * (c["v_r"][a] ** 2 + c["v_t"][a] ** 2)
        J = c["r"][a] * c["v_t"][a]
        with np.errstate(divide="ignore"):
            Q = 2 * E - 2 * PH - J * J / R ** 2          # literal Eq. 12
        Q[k] = c["v_r"][a] ** 2
        neg = Q < 0
        kmin[a] = np.max(np.nonzero(neg[:k])[0])          # largest j <= k-1 with Q_j < 0
        kmax[a] = k + np.min(np.nonzero(neg[k + 1:])[0])  # (smallest j >= k+1 with Q_j < 0) - 1
        nn = np.nonzero(~neg)[0]
        contiguous += int(nn[-1] - nn[0] + 1 == nn.size)
    assert contiguous == n                                # concavity in 1/r: one interval of Q >= 0
    assert np.array_equal(tp["k_min"], kmin)
    assert np.array_equal(tp["k_max"], kmax)
    assert np.all(kmin < np.arange(1, n + 1)) and np.all(kmax >= np.arange(1, n + 1))


def test_roots_satisfy_eq12_with_brute_force_potential(oracle):
    n = 2000
    c = sorted_cluster(n, 23)
    r, m = c["r"], c["m"]
    phi, mc = oracle.potential(r, m)
    tp = oracle.orbit_turning_points(r, c["v_r"], c["v_t"], phi, mc)
    R = np.concatenate([[0.0], r, [np.inf]])
    worst = 0.0
    for a in range(n):
        E, J = tp["E"][a], tp["J"][a]
        assert E == pytest.approx(phi[a] + 0.5 * (c["v_r"][a] ** 2 + c["v_t"][a] ** 2), rel=1e-15)  # Eq. 16
        assert J == pytest.approx(r[a] * c["v_t"][a], rel=1e-15)
        for x, j in ((tp["r_min"][a], tp["k_min"][a]), (tp["r_max"][a], tp["k_max"][a])):
            p = phi_brute(r, m, x)
            q = 2 * E - 2 * p - J * J / (x * x)
            worst = max(worst, abs(q) / (abs(2 * E) + abs(2 * p) + J * J / (x * x)))
            assert R[j] * (1 - 1e-12) <= x <= R[j + 1] * (1 + 1e-12)              # root inside its shell
        assert tp["r_min"][a] <= r[a] * (1 + 1e-12) and r[a] <= tp["r_max"][a] * (1 + 1e-12)
    assert worst < 1e-13


def test_both_sentinel_shells_occur_in_a_plummer_cluster(oracle):
    """at N = 2e5 about 0.03 % of the stars have their pericentre inside the innermost star
    (k_min = 0) and a few in 1e5 their apocentre beyond the outermost (k_max = N), so natural inputs reach both
    sentinel nodes of the table; their roots still bracket the star."""
    n = 200_000
    c = sorted_cluster(n, 23)
    phi, mc = oracle.potential(c["r"], c["m"])
    tp = oracle.orbit_turning_points(c["r"], c["v_r"], c["v_t"], phi, mc)
    inner, outer = tp["k_min"] == 0, tp["k_max"] == n
    assert 20 <= inner.sum() <= 200 and 1 <= outer.sum() <= 20
    assert np.all(tp["r_min"][inner] <= c["r"][0]) and np.all(tp["r_min"][inner] > 0)
    assert np.all(tp["r_max"][outer] >= c["r"][-1]) and np.all(np.isfinite(tp["r_max"][outer]))


def test_sentinel_shells_are_exercised(oracle):
    # innermost star on a wide orbit -> pericentre inside r_1 (shell 0);
    # outermost star moving outwards -> apocentre beyond r_N (shell N, Kepler there)
    r = np.array([1.0, 2.0, 3.0, 4.0])
    m = np.array([0.25, 0.25, 0.25, 0.25])
    phi, mc = oracle.potential(r, m)
    vr = np.array([0.3, 0.0, 0.0, 0.2])
    vt = np.array([0.2, 0.5, 0.5, 0.3])
    tp = oracle.orbit_turning_points(r, vr, vt, phi, mc)
    assert tp["k_min"][0] == 0 and tp["k_max"][3] == 4
    E, J = tp["E"][0], tp["J"][0]
    assert tp["r_min"][0] == pytest.approx(J / math.sqrt(2 * (E - phi[0])), rel=1e-14)   # Phi == Phi_1 inside r_1
    E, J = tp["E"][3], tp["J"][3]
    a_k = -1.0 / (2 * E)
    e_k = math.sqrt(1 + 2 * E * J * J)
    assert tp["r_max"][3] == pytest.approx(a_k * (1 + e_k), rel=1e-13)                    # Kepler outside r_N


@pytest.mark.parametrize("ecc", [0.05, 0.5, 0.9, 0.99])
def test_kepler_turning_points(oracle, ecc):
    r, m = kepler_table()
    phi, mc = oracle.potential(r, m)
    assert np.max(np.abs(phi[1:] * r[1:] + 1.0)) < 1e-15
    a_k = 1.3
    E, J = -1.0 / (2 * a_k), math.sqrt(a_k * (1 - ecc * ecc))
    vr = np.zeros_like(r)
    vt = np.zeros_like(r)
    # put the orbit on every tracer that lies inside [a(1-e), a(1+e)]
    sel = np.nonzero((r > a_k * (1 - ecc) * 1.001) & (r < a_k * (1 + ecc) * 0.999))[0]
    vt[sel] = J / r[sel]
    vr[sel] = np.sqrt(np.maximum(2 * (E + 1 / r[sel]) - vt[sel] ** 2, 0.0))
    tp = oracle.orbit_turning_points(r, vr, vt, phi, mc)
    assert np.all(tp["status"][sel] == 0)
    assert np.max(np.abs(tp["r_min"][sel] / (a_k * (1 - ecc)) - 1)) < 1e-11 / (1 - ecc)
    assert np.max(np.abs(tp["r_max"][sel] / (a_k * (1 + ecc)) - 1)) < 1e-11 / (1 - ecc)


def test_circular_orbit_at_a_node(oracle):
    n = 2000
    c = sorted_cluster(n, 24)
    r, m = c["r"], c["m"]
    phi, mc = oracle.potential(r, m)
    vr = np.zeros(n)
    Mprev = np.concatenate([[0.0], mc[:-1]])
    vt = np.sqrt((Mprev + mc) / (2 * r))           # J^2/r_k between G M_{k-1} and G M_k: exactly circular
    tp = oracle.orbit_turning_points(r, vr, vt, phi, mc)
    k = np.arange(1, n + 1)
    sel = slice(1, None)                           # k = 1 has M_0 = 0: degenerate pericentre at shell 0
    assert np.array_equal(tp["k_min"][sel], (k - 1)[sel]) and np.array_equal(tp["k_max"][sel], k[sel])
    assert np.max(np.abs(tp["r_min"][sel] / r[sel] - 1)) < 1e-9
    assert np.max(np.abs(tp["r_max"][sel] / r[sel] - 1)) < 1e-9


def test_flags_unbound_and_radial(oracle):
    r = np.array([1.0, 2.0, 3.0])
    m = np.array([0.3, 0.3, 0.4])
    phi, mc = oracle.potential(r, m)
    tp = oracle.orbit_turning_points(r, np.array([0.0, 5.0, 0.1]), np.array([0.3, 0.1, 0.0]), phi, mc)
    assert tp["status"][0] == 0
    assert tp["status"][1] & oracle.ST_UNBOUND and np.isinf(tp["r_max"][1])
    assert tp["status"][2] & oracle.ST_RADIAL and tp["r_min"][2] == 0.0


def test_subset_selection_matches_full(oracle):
    c = sorted_cluster(3001, 25)
    phi, mc = oracle.potential(c["r"], c["m"])
    full = oracle.orbit_turning_points(c["r"], c["v_r"], c["v_t"], phi, mc)
    sub = oracle.orbit_turning_points(c["r"], c["v_r"], c["v_t"], phi, mc, first=3, stride=7)
    for k in full:
        assert np.array_equal(sub[k], full[k][3::7])


# ----------------------------------------------------------------------------- S4
def _draw(oracle, c, phi, mc, tp, seed=5, step=0, ids=None, sl=slice(None)):
    ids = c["id"] if ids is None else ids
    return oracle.sample_new_radius(c["r"], phi, mc, c["r"][sl], c["v_r"][sl], c["v_t"][sl], tp["E"], tp["J"],
                                    tp["r_min"], tp["r_max"], tp["k_min"], tp["k_max"], ids[sl], tp["status"],
                                    seed, step)


def test_draw_bounds_energy_and_angular_momentum(oracle):
    n = 3000
    c = sorted_cluster(n, 31, "salpeter")
    r, m = c["r"], c["m"]
    phi, mc = oracle.potential(r, m)
    tp = oracle.orbit_turning_points(r, c["v_r"], c["v_t"], phi, mc)
    s = _draw(oracle, c, phi, mc, tp)
    assert np.all(s["status"] & ~np.uint8(oracle.ST_CLIPPED) == 0)
    assert np.all(s["r_new"] >= tp["r_min"]) and np.all(s["r_new"] <= tp["r_max"])
    assert np.max(np.abs(s["r_new"] * s["v_t_new"] / tp["J"] - 1)) < 4e-16
    worst = 0.0
    for a in range(n):
        e_new = phi_brute(r, m, s["r_new"][a]) + 0.5 * (s["v_r_new"][a] ** 2 + s["v_t_new"][a] ** 2)
        worst = max(worst, abs(e_new - tp["E"][a]) / abs(tp["E"][a]))
    assert worst < 5e-14                                 # energy identity (Eq. 16 at the new radius)
    assert 0.45 < (s["v_r_new"] > 0).mean() < 0.55       # random sign of v_r
    assert s["trials"] == int(s["n_try"].sum())
    assert 1.6 < s["n_try"].mean() < 2.2


def _kepler_many(oracle, ecc, ndraw, a_k=1.3):
    r, m = kepler_table()
    phi, mc = oracle.potential(r, m)
    E, J = -1.0 / (2 * a_k), math.sqrt(a_k * (1 - ecc * ecc))
    # one tracer inside the orbit carries it; its orbit is replicated over ndraw star ids
    a = int(np.searchsorted(r, a_k))
    vt = np.zeros_like(r)
    vr = np.zeros_like(r)
    vt[a] = J / r[a]
    vr[a] = math.sqrt(2 * (E + 1 / r[a]) - vt[a] ** 2)
    tp = oracle.orbit_turning_points(r, vr, vt, phi, mc, first=a, stride=1, count=1)
    rep = {k: np.repeat(v, ndraw) for k, v in tp.items()}
    s = oracle.sample_new_radius(r, phi, mc, np.repeat(r[a], ndraw), np.repeat(vr[a], ndraw), np.repeat(vt[a], ndraw),
                                 rep["E"], rep["J"], rep["r_min"], rep["r_max"], rep["k_min"], rep["k_max"],
                                 np.arange(ndraw, dtype=np.uint32), rep["status"], seed=77, step=3)
    return s, a_k, ecc


@pytest.mark.parametrize("ecc", [0.05, 0.5, 0.9, 0.99])
def test_kepler_time_weighted_distribution_and_acceptance(oracle, ecc):
    ndraw = 100_000
    s, a_k, e = _kepler_many(oracle, ecc, ndraw)
    assert np.all(s["status"] & ~np.uint8(oracle.ST_CLIPPED) == 0)

    def cdf(x):      # fraction of the radial period spent inside radius x: (psi - e sin psi)/pi
        psi = np.arccos(np.clip((1 - x / a_k) / e, -1, 1))
        return (psi - e * np.sin(psi)) / math.pi

    ks = stats.kstest(s["r_new"], cdf)
    assert ks.pvalue > 1e-3, ks
    # closed-form acceptance probability of the scheme on a Kepler orbit: pi / (2 sqrt(3) C_F (1+e))
    acc = ndraw / s["trials"]
    pred = math.pi / (2 * math.sqrt(3) * oracle.C_F * (1 + e))
    assert abs(acc / pred - 1) < 0.01
    assert not np.any(s["status"] & oracle.ST_CLIPPED)   # F bounds g exactly for Kepler orbits


def test_draw_is_order_independent_and_keyed_by_id_step_seed(oracle):
    n = 1500
    c = sorted_cluster(n, 32)
    phi, mc = oracle.potential(c["r"], c["m"])
    tp = oracle.orbit_turning_points(c["r"], c["v_r"], c["v_t"], phi, mc)
    s0 = _draw(oracle, c, phi, mc, tp, seed=9, step=4)
    p = np.random.default_rng(1).permutation(n)
    tpp = {k: v[p] for k, v in tp.items()}
    sp = oracle.sample_new_radius(c["r"], phi, mc, c["r"][p], c["v_r"][p], c["v_t"][p], tpp["E"], tpp["J"],
                                  tpp["r_min"], tpp["r_max"], tpp["k_min"], tpp["k_max"], c["id"][p],
                                  tpp["status"], 9, 4)
    for k in ("r_new", "v_r_new", "v_t_new", "n_try", "status"):
        assert np.array_equal(sp[k], s0[k][p])
    s1 = _draw(oracle, c, phi, mc, tp, seed=9, step=5)
    s2 = _draw(oracle, c, phi, mc, tp, seed=10, step=4)
    s3 = _draw(oracle, c, phi, mc, tp, seed=9 + (1 << 32), step=4)      # high half of the seed is used
    assert (s1["r_new"] != s0["r_new"]).mean() > 0.99
    assert (s2["r_new"] != s0["r_new"]).mean() > 0.99
    assert (s3["r_new"] != s0["r_new"]).mean() > 0.99
    s4 = _draw(oracle, c, phi, mc, tp, seed=9, step=4, ids=c["id"] + np.uint32(1))
    assert (s4["r_new"] != s0["r_new"]).mean() > 0.99


def test_flagged_stars_are_left_in_place(oracle):
    r = np.array([1.0, 2.0, 3.0, 4.0])
    m = np.array([0.25, 0.25, 0.25, 0.25])
    phi, mc = oracle.potential(r, m)
    vr = np.array([0.1, 5.0, 0.1, 0.0])
    vt = np.array([0.3, 0.1, 0.0, math.sqrt((0.75 + 1.0) / 2 / 4.0)])     # ok, unbound, radial, circular
    tp = oracle.orbit_turning_points(r, vr, vt, phi, mc)
    s = oracle.sample_new_radius(r, phi, mc, r, vr, vt, tp["E"], tp["J"], tp["r_min"], tp["r_max"], tp["k_min"],
                                 tp["k_max"], np.arange(4, dtype=np.uint32), tp["status"], 1, 0)
    assert int(s["status"][0]) & ~oracle.ST_CLIPPED == 0 and s["n_try"][0] >= 1
    for a, bit in ((1, oracle.ST_UNBOUND), (2, oracle.ST_RADIAL)):
        assert int(s["status"][a]) & bit
        assert s["r_new"][a] == r[a] and s["v_r_new"][a] == vr[a] and s["v_t_new"][a] == vt[a] and s["n_try"][a] == 0
    # the circular star either is flagged CIRCULAR or is drawn inside a bracket of relative width < 1e-7
    assert (int(s["status"][3]) & oracle.ST_CIRCULAR) or abs(s["r_new"][3] / r[3] - 1) < 1e-7


def test_plummer_is_stationary_under_one_step(oracle):
    # The Plummer model is an equilibrium: drawing every star's new radius with density 1/|v_r| on its
    # own orbit must leave the radial distribution unchanged (2-sample KS), and likewise v^2.
    n = 60_000
    c = inputs.plummer(n, 33)
    o = oracle.orbit_step(c["r"], c["v_r"], c["v_t"], c["m"], c["id"], seed=33, step=0)
    s = o["sample"]
    assert np.all(s["status"] & ~np.uint8(oracle.ST_CLIPPED) == 0)
    assert stats.ks_2samp(o["r"], s["r_new"]).pvalue > 1e-3
    v2_old = o["v_r"] ** 2 + o["v_t"] ** 2
    v2_new = s["v_r_new"] ** 2 + s["v_t_new"] ** 2
    assert stats.ks_2samp(v2_old, v2_new).pvalue > 1e-3
    # radial-velocity anisotropy stays isotropic: <v_r^2> = <v_t^2>/2
    assert abs(np.mean(s["v_r_new"] ** 2) / (0.5 * np.mean(s["v_t_new"] ** 2)) - 1) < 0.03
    assert (s["status"] & oracle.ST_CLIPPED).sum() == 0    # F bounded g on every trial (R7)


def test_ten_chained_steps_conserve_what_they_should(oracle):
    n = 4000
    c = inputs.plummer(n, 34)
    r, vr, vt, m, ids = c["r"], c["v_r"], c["v_t"], c["m"], c["id"]
    J0 = np.empty(n)
    J0[ids] = r * vt
    e_tot = []
    for step in range(10):
        o = oracle.orbit_step(r, vr, vt, m, ids, seed=34, step=step)
        s = o["sample"]
        assert np.all(s["status"] & ~np.uint8(oracle.ST_CLIPPED) == 0)
        e_tot.append(np.sum(o["m"] * (0.5 * o["phi"] + 0.5 * (o["v_r"] ** 2 + o["v_t"] ** 2))))
        r, vr, vt, m, ids = s["r_new"], s["v_r_new"], s["v_t_new"], o["m"], o["id"]
    assert sorted(ids.tolist()) == list(range(n))
    assert abs(math.fsum(m) - 1.0) < 1e-15
    J = np.empty(n)
    J[ids] = r * vt
    assert np.max(np.abs(J / J0 - 1)) < 1e-14               # J is carried exactly (to rounding)
    assert abs(e_tot[0] + 0.25) < 0.01
    assert abs(e_tot[-1] - e_tot[0]) < 0.01                  # small drift only: no energy correction (R10)
