"""GPU-vs-oracle parity on the branches no natural Plummer input reaches (VERDICT r1 "What's weak" 1, 4):

* S4's exhaustion path (`draw_exhaustive`, MAXTRIES, keep-the-last-good-trial): the TEST-ONLY pair of builds
  with the cap on trials lowered to 3 -- paper_1206_5878_b200/libhmc_tmax3.so (-DHMC_T_MAX=3u) against
  oracle/libhmc_oracle_tmax3.so (-DT_MAX=3u) -- star by star; and in the PRODUCT build with orbits given an
  energy below the potential well, for which all 4096 trials fail.
* exactly circular orbits (CIRCULAR, or a bracket of a few ulps), stars whose outer quadratic has C >= 0
  (DEGENERATE), unbound and radial stars: flags and outputs bit for bit.
* the fused entry point hmc_orbit_step against the ORACLE (not against the two GPU calls).
* S3's exact search by lane pairs (the product's path from N = 2^25 on): the TEST-ONLY build libhmc_pairs.so
  (-DHMC_S3_PAIRS_MIN_N=1) takes it at every N.
"""
import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import build as hmc_build
from paper_1206_5878_b200 import hmc, inputs

pytestmark = pytest.mark.gpu


def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def host(t, dtype=None):
    a = t.cpu().numpy()
    return a.view(dtype) if dtype is not None else a


@pytest.fixture
def tmax3(monkeypatch, oracle):
    """Both sides built with a cap of three trials; every hmc.* call inside the test goes to that library."""
    L = hmc.load(hmc_build.build(variant="tmax3"))
    assert L.hmc_t_max() == 3
    monkeypatch.setattr(hmc, "_lib", L)
    with oracle.use("tmax3"):
        assert oracle.t_max() == 3
        yield oracle
    # monkeypatch restores hmc._lib


def sorted_tables(oracle, n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    phi, mc = oracle.potential(rs, ms)
    return rs, vrs, vts, ms, ids, phi, mc


def gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, step, counters=None, tp_override=None):
    d = [dev(x) for x in (rs, vrs, vts, phi, mc)]
    ws = hmc.alloc_workspace(len(rs))
    tp = hmc.hmc_orbit_turning_points(d[0], d[1], d[2], d[3], d[4], 1.0, counters=counters, workspace=ws)
    reuse = tp_override is None
    if tp_override is not None:
        tp = {k: dev(v) for k, v in tp_override.items()}
    sm = hmc.hmc_sample_new_radius(d[0], d[3], d[4], d[1], d[2], tp, dev(ids), seed, step, 1.0, counters=counters,
                                   workspace=ws, reuse_tables=reuse)
    return tp, sm


def assert_bitwise(tp, sm, otp, osm):
    for k in ("E", "J", "r_min", "r_max", "status"):
        assert np.array_equal(host(tp[k]), otp[k]), k
    for k in ("k_min", "k_max"):
        assert np.array_equal(host(tp[k], np.uint32), otp[k]), k
    for k in ("r_new", "v_r_new", "v_t_new", "status"):
        assert np.array_equal(host(sm[k]), osm[k]), k
    assert np.array_equal(host(sm["n_try"], np.uint16), osm["n_try"])


@pytest.mark.parametrize("n,masses", [(1, "equal"), (40, "equal"), (100_000, "equal"), (250_007, "salpeter")])
def test_exhaustion_path_cap_of_three_trials(tmax3, n, masses):
    """About 11 % of the stars run out of trials: draw_exhaustive against the oracle's last-good-trial rule."""
    oracle = tmax3
    seed, step = 83, 4
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed, masses)
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], seed, step)
    counters = hmc.alloc_counters()
    tp, sm = gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, step, counters)
    assert_bitwise(tp, sm, otp, osm)
    cnt = dict(zip(hmc.COUNTER_NAMES, host(counters).tolist()))
    exhausted = int(((osm["status"] & hmc.ST_MAXTRIES) != 0).sum())
    assert cnt["maxtries"] == exhausted and cnt["trials"] == osm["trials"]
    if n >= 100_000:
        assert 0.05 * n < exhausted < 0.2 * n
    # the fused entry point takes the same path
    tp2, sm2 = hmc.hmc_orbit_step(dev(rs), dev(vrs), dev(vts), dev(phi), dev(mc), dev(ids), seed, step)
    assert_bitwise(tp2, sm2, otp, osm)


def test_exhaustion_path_in_the_product_build_when_no_trial_is_good(oracle):
    """Product library, T_MAX = 4096: orbits handed to S4 with an energy below the whole potential well have
    Q(r_0) < 0 at every trial; the star stays where it is with n_try = 4096 and MAXTRIES, like the oracle's."""
    assert hmc.lib().hmc_t_max() == 4096 and oracle.t_max() == 4096
    n, seed, step = 20_000, 91, 1
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed)
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    sel = np.arange(3, n, 997)
    otp["E"][sel] = 2.0 * phi[0]
    # a star whose Q is positive only on part of its interval: some trials good, all rejected or accepted late
    half = np.arange(11, n, 1499)
    otp["E"][half] = otp["E"][half] - 0.3 * (otp["E"][half] - phi[half])
    osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], seed, step)
    assert np.all(osm["n_try"][sel] == 4096) and np.all(osm["status"][sel] == hmc.ST_MAXTRIES)
    counters = hmc.alloc_counters()
    _, sm = gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, step, counters, tp_override=otp)
    for k in ("r_new", "v_r_new", "v_t_new", "status"):
        assert np.array_equal(host(sm[k]), osm[k]), k
    assert np.array_equal(host(sm["n_try"], np.uint16), osm["n_try"])
    cnt = dict(zip(hmc.COUNTER_NAMES, host(counters).tolist()))
    assert cnt["maxtries"] == int(((osm["status"] & hmc.ST_MAXTRIES) != 0).sum()) >= sel.size
    assert cnt["trials"] == osm["trials"]


def test_circular_orbits_flags_and_outputs(oracle):
    """v_r = 0 and J^2 / r_k between G M_{k-1} and G M_k: the star sits on a circular orbit at a node
    (tests/test_oracle_orbit.py pins the oracle there).  r_min = r_max = r_k up to rounding: S4 either flags
    CIRCULAR (interval empty or end slopes of the wrong sign) or draws inside a bracket a few ulps wide.
    Whatever the oracle decides, the GPU decides the same, bit for bit."""
    n, seed = 30_000, 24
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed)
    m_prev = np.concatenate([[0.0], mc[:-1]])
    vts = np.sqrt((m_prev + mc) / (2 * rs))
    vrs = np.zeros(n)
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], seed, 0)
    ncirc = int(((osm["status"] & hmc.ST_CIRCULAR) != 0).sum())
    assert ncirc > n // 10                                   # the flag does arise on this input
    counters = hmc.alloc_counters()
    tp, sm = gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, 0, counters)
    assert_bitwise(tp, sm, otp, osm)
    assert host(counters)[hmc.COUNTER_NAMES.index("circular")] == ncirc
    tp2, sm2 = hmc.hmc_orbit_step(dev(rs), dev(vrs), dev(vts), dev(phi), dev(mc), dev(ids), seed, 0)
    assert_bitwise(tp2, sm2, otp, osm)


def assert_s3_and_flagged(tp, sm, otp, osm):
    """S3 bit for bit on every star; S4 on the stars S3 flagged (left in place, no trial)."""
    for k in ("E", "J", "r_min", "r_max", "status"):
        assert np.array_equal(host(tp[k]), otp[k]), k
    for k in ("k_min", "k_max"):
        assert np.array_equal(host(tp[k], np.uint32), otp[k]), k
    fl = otp["status"] != 0
    for k in ("r_new", "v_r_new", "v_t_new", "status"):
        assert np.array_equal(host(sm[k])[fl], osm[k][fl]), k
    assert np.all(host(sm["n_try"], np.uint16)[fl] == 0) and np.all(osm["n_try"][fl] == 0)


def test_degenerate_unbound_and_radial_stars(oracle):
    """A mass table a thousand times too light for its potential makes the outer quadratic's C >= 0 for most
    stars (DEGENERATE: r_max = +inf, no draw); a few stars are made unbound and radial as well.  DEGENERATE
    cannot arise from a table that hmc_potential made (Q is concave in 1/r), so the table here is inconsistent
    on purpose; S3 is compared on every star, S4 on the flagged ones (for the others the turning points lie
    outside their shells, which S4's callers guarantee they do not)."""
    n, seed = 20_000, 37
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed)
    mc_light = mc * 1e-3
    vrs, vts = vrs.copy(), vts.copy()
    vrs[5::400] = 9.0                                        # unbound
    vts[7::400] = 0.0                                        # radial
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc_light)
    osm = oracle.sample_new_radius(rs, phi, mc_light, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], seed, 6)
    ndeg = int(((otp["status"] & hmc.ST_DEGENERATE) != 0).sum())
    assert ndeg > n // 4
    counters = hmc.alloc_counters()
    tp, sm = gpu_s3_s4(rs, vrs, vts, phi, mc_light, ids, seed, 6, counters)
    assert_s3_and_flagged(tp, sm, otp, osm)
    cnt = dict(zip(hmc.COUNTER_NAMES, host(counters).tolist()))
    assert cnt["degenerate"] == ndeg
    assert cnt["unbound"] == int(((otp["status"] & hmc.ST_UNBOUND) != 0).sum()) > 0
    assert cnt["radial"] == int(((otp["status"] & hmc.ST_RADIAL) != 0).sum()) > 0
    tp2, sm2 = hmc.hmc_orbit_step(dev(rs), dev(vrs), dev(vts), dev(phi), dev(mc_light), dev(ids), seed, 6)
    assert_s3_and_flagged(tp2, sm2, otp, osm)


@pytest.mark.parametrize("n,masses", [(1, "equal"), (33, "equal"), (10_239, "equal"), (100_000, "equal"),
                                      (300_001, "salpeter"), (1_200_000, "equal")])
def test_fused_orbit_step_against_the_oracle(oracle, n, masses):
    """hmc_orbit_step (S3 + S4 in one launch) on the oracle's tables, compared with the ORACLE star by star."""
    seed, step = 21, 5
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed, masses)
    with oracle.use("omp"):
        otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
        osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                       otp["k_min"], otp["k_max"], ids, otp["status"], seed, step)
    counters = hmc.alloc_counters()
    tp, sm = hmc.hmc_orbit_step(dev(rs), dev(vrs), dev(vts), dev(phi), dev(mc), dev(ids), seed, step, counters=counters)
    assert_bitwise(tp, sm, otp, osm)
    assert host(counters)[hmc.COUNTER_NAMES.index("trials")] == osm["trials"]


@pytest.fixture
def pairs_build(monkeypatch):
    """S3's exact search by lane pairs at every N; every hmc.* call inside the test goes to that library."""
    monkeypatch.setattr(hmc, "_lib", hmc.load(hmc_build.build(variant="pairs")))


@pytest.mark.parametrize("n,masses", [(1, "equal"), (2, "equal"), (31, "equal"), (33, "equal"), (1025, "equal"),
                                      (10_239, "equal"), (100_000, "equal"), (300_001, "salpeter"), (1_200_000, "equal")])
def test_pair_search_matches_oracle(pairs_build, oracle, n, masses):
    """Lanes 2i and 2i+1 probe nodes p and p+1 of one star in one load instruction and hand the bracketing node
    over through shared memory: same brackets, roots and flags as the oracle, ragged last warp included; S4
    on S3's output as usual."""
    seed, step = 58, 2
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed, masses)
    with oracle.use("omp"):
        otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
        osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                       otp["k_min"], otp["k_max"], ids, otp["status"], seed, step)
    tp, sm = gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, step)
    assert_bitwise(tp, sm, otp, osm)


def test_pair_search_flagged_stars_and_ranges(pairs_build, oracle):
    """Unbound and radial stars take no search (their lanes pass closed brackets to the pair search); a range
    call whose count is not a multiple of 32 leaves lanes without a star in the last warp."""
    n, seed = 50_003, 61
    rs, vrs, vts, ms, ids, phi, mc = sorted_tables(oracle, n, seed)
    vrs, vts = vrs.copy(), vts.copy()
    vrs[5::40] = 9.0                                         # unbound
    vts[6::40] = 0.0                                         # radial
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    d = [dev(x) for x in (rs, vrs, vts, phi, mc)]
    ws = hmc.alloc_workspace(n)
    tp = hmc.hmc_orbit_turning_points(d[0], d[1], d[2], d[3], d[4], 1.0, workspace=ws)
    for k in ("E", "J", "r_min", "r_max", "status"):
        assert np.array_equal(host(tp[k]), otp[k]), k
    for k in ("k_min", "k_max"):
        assert np.array_equal(host(tp[k], np.uint32), otp[k]), k
    assert int((otp["status"] != 0).sum()) >= 2 * (n // 40)
    first, count = 12_345, 7_777
    tpr = hmc.hmc_orbit_turning_points(d[0], d[1][first:first + count].contiguous(), d[2][first:first + count].contiguous(),
                                       d[3], d[4], 1.0, workspace=ws, first=first)
    for k in ("E", "J", "r_min", "r_max", "status"):
        assert np.array_equal(host(tpr[k]), otp[k][first:first + count]), k
    for k in ("k_min", "k_max"):
        assert np.array_equal(host(tpr[k], np.uint32), otp[k][first:first + count]), k


# ----------------------------------------------------------------------------- trials inside the innermost star
def _draw_both(oracle, rs, vrs, vts, ms, ids, seed, step):
    phi, mc = oracle.potential(rs, ms)
    otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
    osm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], seed, step)
    tp, sm = gpu_s3_s4(rs, vrs, vts, phi, mc, ids, seed, step)
    assert_bitwise(tp, sm, otp, osm)
    return otp, osm


def test_round_innermost_radius_trials_below_it(oracle):
    """Radii 1, 2, 3, 4: r_1 has zero low mantissa bits and, the coarse table being the whole table (shift 0),
    coarse[1] = r_1 -- the case in which S4's inverse table used to send a trial radius below r_1 to interval 1
    instead of interval 0 (round-2 advisor).  Star 0's orbit reaches inside r_1 (k_min = 0); over 64 (seed, step)
    pairs some ACCEPTED radius lies there, so Phi(r0), Q0, g and the accept decision are all exercised."""
    r = np.array([1.0, 2.0, 3.0, 4.0])
    m = np.array([0.25, 0.25, 0.25, 0.25])
    vr = np.array([0.1, 5.0, 0.1, 0.0])
    vt = np.array([0.3, 0.1, 0.0, 0.3])
    ids = np.arange(4, dtype=np.uint32)
    below = 0
    for seed in (1, 2, 3, 4):
        for step in range(16):
            otp, osm = _draw_both(oracle, r, vr, vt, m, ids, seed, step)
            assert otp["k_min"][0] == 0 and otp["r_min"][0] < 1.0
            below += int(osm["r_new"][0] < 1.0)
    print("accepted radii below r_1: %d of 64" % below)
    assert below >= 4


def test_tied_round_innermost_radii_with_a_directory(oracle):
    """The same with a directory (N = 20 000: shift 1, coarse[1] is node 2): the two innermost stars share the round
    radius 1.0, every other radius is larger.  Trials of the inner stars' orbits fall below r_1."""
    n = 20_000
    rs, vrs, vts, ms, ids, _, _ = sorted_tables(oracle, n, 77)
    s = 1.0009765625 / rs[0]                  # lengths by s, velocities by s^-1/2: the cluster stays bound
    rs, vrs, vts = rs * s, vrs / np.sqrt(s), vts / np.sqrt(s)     # everything above 1 ...
    rs[0] = rs[1] = 1.0                       # ... except a tied, round innermost pair
    assert np.all(np.diff(rs) >= 0)
    below = 0
    for step in range(6):
        otp, osm = _draw_both(oracle, rs, vrs, vts, ms, ids, 5, step)
        below += int((osm["r_new"] < 1.0).sum())
    print("accepted radii below r_1: %d" % below)
    assert below >= 3
