"""Pins for the oracle's energy correction for the time-varying potential (R18), CPU only.

The formula is not in the paper's text; the reading is dE = 1/2 [dPhi(r_old) + dPhi(r_new)].  What pins it is a
theorem, not the formula retyped: with the shell potential, sum_i m_i Phi'(r_old,i) and sum_i m_i Phi(r_new,i) are the
same double sum over pairs, so T + W of the whole cluster must come out of a corrected step exactly as it went in --
to rounding, for any masses and any displacement.  A wrong sign, a dropped term, the wrong table or the wrong position
breaks that by the size of the potential change itself (1e-4 relative per step on these models)."""
import numpy as np

from paper_1206_5878_b200 import inputs


def oracle_step_with_correction(oracle, state, seed, step, correct=True):
    """state = dict(r, v_r, v_t, m, id [, E, r_old, p_old]); returns (new state, diagnostics of the configuration the
    step started from, in that step's potential, after the correction if one was applied)."""
    have_old = "E" in state
    cols = [state["v_r"], state["v_t"], state["m"]] + ([state["E"], state["r_old"], state["p_old"]] if have_old else [])
    rs, perm, cs, ids = oracle.sort_by_radius(state["r"], tuple(cols), state["id"])
    vrs, vts, ms = cs[0], cs[1], cs[2]
    phi, mc = oracle.potential(rs, ms)
    nok = 0
    if have_old and correct:
        vrs, vts, st = oracle.energy_correction(rs, phi, mc, cs[3], cs[4], cs[5], vrs, vts)
        nok = int((st != 0).sum())
    diag = oracle.diagnostics(rs, vrs, vts, ms, phi, mc)
    tp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    sm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, tp["E"], tp["J"], tp["r_min"], tp["r_max"], tp["k_min"],
                                  tp["k_max"], ids, tp["status"], seed, step)
    new = dict(r=sm["r_new"], v_r=sm["v_r_new"], v_t=sm["v_t_new"], m=ms, id=ids, E=tp["E"], r_old=rs, p_old=phi)
    return new, diag, nok


def start(n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    return {k: c[k] for k in ("r", "v_r", "v_t", "m", "id")}


def test_total_energy_is_exactly_invariant_over_a_corrected_step(oracle):
    """A few stars per 10^4 sit so close to a turning point that the corrected kinetic energy would be negative; they
    keep their velocities and are flagged.  Their shortfall is put back here from a brute-force shell-theorem
    potential (numpy, all stars) before the invariance is asserted."""
    for masses, seed in (("equal", 12), ("salpeter", 13)):
        s0 = start(20_000, seed, masses)
        s1, d0, _ = oracle_step_with_correction(oracle, s0, seed, 0)
        # the corrected second configuration, by hand, to see the flags
        rs, perm, cs, ids = oracle.sort_by_radius(s1["r"], (s1["v_r"], s1["v_t"], s1["m"], s1["E"], s1["r_old"], s1["p_old"]), s1["id"])
        vrs, vts, ms, E, r_old, p_old = cs
        phi, mc = oracle.potential(rs, ms)
        vro, vto, st = oracle.energy_correction(rs, phi, mc, E, r_old, p_old, vrs, vts)
        d1 = oracle.diagnostics(rs, vro, vto, ms, phi, mc)
        d1u = oracle.diagnostics(rs, vrs, vts, ms, phi, mc)
        flagged = np.nonzero(st)[0]
        assert len(flagged) < 20 and set(st[flagged]) <= {64}
        shortfall = 0.0
        for a in flagged:
            K = 0.5 * (vrs[a] ** 2 + vts[a] ** 2)
            phi_new_at_old = -np.sum(ms / np.maximum(rs, r_old[a]))            # shell theorem, every star
            dE = 0.5 * ((phi_new_at_old - p_old[a]) + (phi[a] - (E[a] - K)))
            Kp = E[a] + dE - phi[a]
            assert Kp <= 0.0
            shortfall += ms[a] * (K - Kp)
        assert abs((d1["E_tot"] - shortfall) - d0["E_tot"]) <= 1e-12 * abs(d0["E_tot"]), (d0["E_tot"], d1["E_tot"], shortfall)
        assert abs(d1u["E_tot"] - d0["E_tot"]) >= 1e-6 * abs(d0["E_tot"])          # uncorrected: a visible jump
        assert d1["W"] == d1u["W"] and d1["r_h"] == d1u["r_h"]                      # positions are untouched


def test_ten_step_drift_with_and_without_correction(oracle):
    s, su = start(4_000, 7), start(4_000, 7)
    e0, flagged = None, 0
    for step in range(10):
        s, d, nok = oracle_step_with_correction(oracle, s, 7, step)
        su, du, _ = oracle_step_with_correction(oracle, su, 7, step, correct=False)
        flagged += nok
        e0 = d["E_tot"] if e0 is None else e0
    assert flagged <= 40                                                            # of 36 000 corrections
    # what is left is the flagged stars' shortfall (they keep more kinetic energy than the formula allows):
    # measured 1.2e-4 against 3.3e-3 without the correction
    assert abs(d["E_tot"] - e0) <= 3e-4 * abs(e0)
    assert abs(du["E_tot"] - e0) >= 10 * abs(d["E_tot"] - e0)


def test_no_change_of_potential_means_no_change_of_velocity(oracle):
    """New table = old table, r_old = own radius, E = Phi_k + K: every bracket of the formula vanishes."""
    c = inputs.plummer(5_000, 4)
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    phi, mc = oracle.potential(rs, ms)
    E = phi + 0.5 * (vrs * vrs + vts * vts)
    vro, vto, st = oracle.energy_correction(rs, phi, mc, E, rs, phi, vrs, vts)
    assert not st.any()
    assert np.max(np.abs(vro - vrs) / np.abs(vrs)) <= 1e-13 and np.max(np.abs(vto - vts) / np.abs(vts)) <= 1e-13


def test_ratio_and_signs_are_preserved_and_flags(oracle):
    s0 = start(10_000, 21)
    s1, _, _ = oracle_step_with_correction(oracle, s0, 21, 0)
    rs, perm, cs, ids = oracle.sort_by_radius(s1["r"], (s1["v_r"], s1["v_t"], s1["m"], s1["E"], s1["r_old"], s1["p_old"]), s1["id"])
    phi, mc = oracle.potential(rs, cs[2])
    vro, vto, st = oracle.energy_correction(rs, phi, mc, cs[3], cs[4], cs[5], cs[0], cs[1])
    ok = st == 0
    assert ok.mean() > 0.999
    assert np.array_equal(np.sign(vro), np.sign(cs[0])) and np.all(vto > 0)
    assert np.max(np.abs(vro / vto - cs[0] / cs[1]) / np.abs(cs[0] / cs[1])) <= 1e-15 * 4
    lam = vto / cs[1]
    assert abs(np.median(lam) - 1) < 1e-2 and np.percentile(np.abs(lam - 1), 99) < 0.1 and lam.std() > 1e-7   # small, non-trivial
    # a star whose corrected kinetic energy would be negative keeps its velocities and is flagged (bit 64)
    E_bad = cs[3].copy(); E_bad[5] = phi[5] - 1.0
    v_bad = cs[0].copy(); v_bad[5] = 1e-3
    vro2, vto2, st2 = oracle.energy_correction(rs, phi, mc, E_bad, cs[4], cs[5], v_bad, cs[1])
    assert st2[5] == 64 and vro2[5] == v_bad[5] and vto2[5] == cs[1][5]
