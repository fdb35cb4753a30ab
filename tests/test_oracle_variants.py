"""The other builds of oracle/hmc_oracle.c (oracle/__init__.py VARIANTS) against the oracle as defined.

* omp   : -fopenmp over the per-star loops.  Must be bit-identical to the single-threaded build
          (stars are independent, the random numbers are counter-based).
* tmax3 : -DT_MAX=3u.  Pins the one branch of hmc_ref_sample_new_radius that no natural input reaches with
          T_MAX = 4096 (R7: "at most T_max trials, then the last trial with Q > 0 is kept, flag
          MAXTRIES"): against the T_MAX = 4096 build (stars that accept within three trials must not change)
          and against the trial's radius recomputed here from the Philox words, which are pinned by the
          known-answer vectors of tests/golden/.
"""
import numpy as np

from paper_1206_5878_b200 import inputs


def _step(oracle, c, seed, step):
    return oracle.orbit_step(c["r"], c["v_r"], c["v_t"], c["m"], c["id"], seed, step)


def test_openmp_build_is_bit_identical(oracle):
    c = inputs.plummer(120_001, 61, "salpeter")
    a = _step(oracle, c, 61, 3)
    with oracle.use("omp"):
        assert oracle.lib().hmc_ref_openmp() == 1 and oracle.t_max() == 4096
        b = _step(oracle, c, 61, 3)
        # energy correction of the second configuration, threaded
        sm, tp = b["sample"], b["tp"]
        rs, perm, cs, ids = oracle.sort_by_radius(sm["r_new"], (sm["v_r_new"], sm["v_t_new"], b["m"], tp["E"], b["r"], b["phi"]), b["id"])
        phi, mc = oracle.potential(rs, cs[2])
        eb = oracle.energy_correction(rs, phi, mc, cs[3], cs[4], cs[5], cs[0], cs[1])
    assert oracle.lib().hmc_ref_openmp() == 0
    ea = oracle.energy_correction(rs, phi, mc, cs[3], cs[4], cs[5], cs[0], cs[1])
    for k in ("r", "perm", "v_r", "v_t", "m", "id", "phi", "m_cum"):
        assert np.array_equal(a[k], b[k]), k
    for k in a["tp"]:
        assert np.array_equal(a["tp"][k], b["tp"][k]), k
    for k in ("r_new", "v_r_new", "v_t_new", "n_try", "status"):
        assert np.array_equal(a["sample"][k], b["sample"][k]), k
    assert a["sample"]["trials"] == b["sample"]["trials"]
    for x, y in zip(ea, eb):
        assert np.array_equal(x, y)


def _henon_radius(oracle, sid, step, t, seed, r_min, r_max):
    """r_0 of trial t (R7, R9) from the Philox words; also the sign bit of the new v_r (R8)."""
    w = oracle.philox4x32_10([sid, 0, step, t], [seed & 0xFFFFFFFF, seed >> 32])
    X = float(((int(w[0]) << 32) | int(w[1])) >> 11) * 2.0 ** -53
    s = 2.0 * X - 1.0
    delta = r_max - r_min
    return 0.5 * (r_min + r_max) + (0.25 * delta) * (3.0 * s - (s * s) * s), int(w[3]) & 1


def test_exhaustion_branch_keeps_the_last_good_trial(oracle):
    n, seed, step = 40_000, 73, 2
    c = inputs.plummer(n, seed)
    full = _step(oracle, c, seed, step)
    with oracle.use("tmax3"):
        assert oracle.t_max() == 3
        cut = _step(oracle, c, seed, step)
    for k in full["tp"]:                                     # S3 does not depend on T_MAX
        assert np.array_equal(full["tp"][k], cut["tp"][k])
    f, s = full["sample"], cut["sample"]
    within = f["n_try"] <= 3
    assert 0.8 < within.mean() < 0.95                        # about one star in nine needs a fourth trial
    for k in ("r_new", "v_r_new", "v_t_new", "n_try", "status"):
        assert np.array_equal(f[k][within], s[k][within]), k
    ex = ~within
    assert np.all(s["status"][ex] & oracle.ST_MAXTRIES) and not np.any(s["status"][within] & oracle.ST_MAXTRIES)
    assert np.all(s["n_try"][ex] == 3)
    assert s["trials"] == int(np.minimum(f["n_try"], 3).sum())
    # the kept radius is that of the LAST trial (t = 2: every trial of these orbits has Q > 0), not of the first
    tp = full["tp"]
    idx = np.nonzero(ex)[0][:400]
    for a in idx:
        r2, sign = _henon_radius(oracle, int(full["id"][a]), step, 2, seed, tp["r_min"][a], tp["r_max"][a])
        assert s["r_new"][a] == r2
        assert (s["v_r_new"][a] < 0) == bool(sign)
        r0, _ = _henon_radius(oracle, int(full["id"][a]), step, 0, seed, tp["r_min"][a], tp["r_max"][a])
        assert s["r_new"][a] != r0
    # the kept trial is a point of the orbit: energy identity (Eq. 16) at the new radius, J conserved
    rs, phi, mc = full["r"], full["phi"], full["m_cum"]
    rn = s["r_new"][ex]
    j = np.clip(np.searchsorted(rs, rn, side="right"), tp["k_min"][ex], tp["k_max"][ex]).astype(np.int64)
    jj = np.maximum(j, 1) - 1
    phin = np.where(j == 0, phi[0], phi[jj] - mc[jj] * (1.0 / rn - 1.0 / rs[jj]))
    kin = 0.5 * (s["v_r_new"][ex] ** 2 + s["v_t_new"][ex] ** 2)
    assert np.max(np.abs(phin + kin - tp["E"][ex]) / (np.abs(phin) + kin)) < 1e-13
    assert np.max(np.abs(rn * s["v_t_new"][ex] / tp["J"][ex] - 1)) < 4e-16


def test_no_good_trial_leaves_the_star_in_place(oracle):
    """S4 given an energy below the potential well of the interval: Q(r_0) < 0 at every trial, so no trial
    is 'good': after T_MAX trials the star keeps r, v_r, v_t, n_try = T_MAX, flag MAXTRIES (both builds)."""
    n, seed = 3000, 5
    c = inputs.plummer(n, seed)
    o = _step(oracle, c, seed, 0)
    tp = {k: v.copy() for k, v in o["tp"].items()}
    sel = np.arange(7, n, 500)
    tp["E"][sel] = 2.0 * o["phi"][0]                         # far below Phi everywhere
    for variant, tmax in (("serial", 4096), ("tmax3", 3)):
        with oracle.use(variant):
            s = oracle.sample_new_radius(o["r"], o["phi"], o["m_cum"], o["r"], o["v_r"], o["v_t"], tp["E"], tp["J"],
                                         tp["r_min"], tp["r_max"], tp["k_min"], tp["k_max"], o["id"], tp["status"], seed, 0)
        assert np.all(s["status"][sel] == oracle.ST_MAXTRIES)
        assert np.all(s["n_try"][sel] == tmax)
        assert np.array_equal(s["r_new"][sel], o["r"][sel]) and np.array_equal(s["v_r_new"][sel], o["v_r"][sel])
        assert np.array_equal(s["v_t_new"][sel], o["v_t"][sel])
        if variant == "serial":
            rest = np.setdiff1d(np.arange(n), sel)
            assert np.array_equal(s["r_new"][rest], o["sample"]["r_new"][rest])
