"""Parity of the CUDA path (through the C ABI, via the thin binding) with the CPU oracle.

Bars (BASELINE.json north_star):
  * sort permutation and bracket indices k_min / k_max: bit-exact
  * Phi, r_min, r_max: <= 1e-12 relative
  * new radii: <= 1e-10 relative for >= 99.999 % of the stars; rejection-branch flips
    (different trial count than the oracle) counted and reported
Because both sides evaluate the same binary64 expressions without FMA (R2) the
observed differences are normally exactly zero; the tests print the counts.
"""
import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import hmc, inputs

pytestmark = pytest.mark.gpu

TOL_PHI = 1e-12
TOL_ROOT = 1e-12
TOL_RNEW = 1e-10
FRAC_RNEW = 0.99999


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    elif t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def host(t, dtype=None):
    a = t.cpu().numpy()
    if dtype is not None:
        a = a.view(dtype)
    return a


def rel(a, b):
    with np.errstate(divide="ignore", invalid="ignore"):
        d = np.abs(a - b) / np.maximum(np.abs(b), 1e-300)
    d[(a == b)] = 0.0           # also covers inf == inf
    return d


def gpu_sort(c):
    ids = dev(c["id"].view(np.int32))
    rs, perm, cols, ids_s = hmc.hmc_sort_by_radius(dev(c["r"]), (dev(c["v_r"]), dev(c["v_t"]), dev(c["m"])), ids)
    return rs, perm, cols, ids_s


# ----------------------------------------------------------------------------- S1
@pytest.mark.parametrize("n", [1, 2, 31, 4095, 4096, 4097, 100_000, 1_000_003])
def test_sort_matches_oracle(oracle, n):
    c = inputs.plummer(n, 100 + n % 97)
    rs, perm, cols, ids_s = gpu_sort(c)
    o_rs, o_perm, o_cols, o_ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    assert np.array_equal(host(perm, np.uint32), o_perm)
    assert np.array_equal(host(rs), o_rs)
    for g, o in zip(cols, o_cols):
        assert np.array_equal(host(g), o)
    assert np.array_equal(host(ids_s, np.uint32), o_ids)


@pytest.mark.parametrize("kind", ["ties", "all_equal", "sorted", "reversed", "extreme", "two_values", "denormal", "narrow",
                                  "narrow_span", "wide_runs"])
def test_sort_adversarial_keys(oracle, kind):
    g = np.random.default_rng(5)
    n = 50_001
    r = dict(
        ties=np.floor(g.random(n) * 40) + 1.0,
        all_equal=np.full(n, 0.75),
        sorted=np.sort(g.random(n) + 0.5),
        reversed=np.sort(g.random(n) + 0.5)[::-1].copy(),
        extreme=10.0 ** g.uniform(-300, 300, n),
        two_values=np.where(g.random(n) < 0.5, 1.0, 2.0),
        denormal=np.where(g.random(n) < 0.5, g.integers(1, 1 << 40, n).astype(np.uint64).view(np.float64), 10.0 ** g.uniform(-310, -300, n)),
        narrow=1.0 + g.integers(0, 1000, n) * 2.0 ** -52,        # a thousand adjacent doubles: long runs of exact ties
        narrow_span=1.0 + g.integers(0, 1 << 30, n) * 2.0 ** -52,  # keys spanning 30 bits: shifted up to fill the kept key bits
        wide_runs=np.repeat(10.0 ** g.uniform(-200, 200, n // 40 + 1), 40)[:n] * (1.0 + g.integers(0, 8, n) * 2.0 ** -52),
    )[kind]
    rs, perm, _, _ = hmc.hmc_sort_by_radius(dev(r))
    o_rs, o_perm, _, _ = oracle.sort_by_radius(r)
    assert np.array_equal(host(perm, np.uint32), o_perm)
    assert np.array_equal(host(rs), o_rs)


def _clustered_keys(n, cluster, g):
    """Radii over ~8 binades in which groups of `cluster` stars differ only in their lowest
    mantissa bits (and some are exactly equal): the packed-word fast path cannot separate them
    by its leading key bits and has to resolve each run from the full keys."""
    base = np.exp(g.uniform(np.log(0.01), np.log(3.0), n // cluster + 1))
    r = np.repeat(base, cluster)[:n].copy()
    bits = r.view(np.uint64)
    bits += g.integers(0, 6, n).astype(np.uint64)          # 0..5 ulps: near-ties and exact ties
    g.shuffle(r)
    return r


@pytest.mark.parametrize("cluster", [2, 7, 32, 33, 63, 64, 65, 66, 200])
def test_sort_runs_of_near_equal_keys(oracle, cluster):
    """Runs of up to 64 stars that agree in the bits the passes sorted are ranked inside the fast path (from the
    packed words, or from the full keys where even the kept bits agree); longer ones make the guarded general sort
    redo the call."""
    g = np.random.default_rng(11 + cluster)
    n = 300_017
    r = _clustered_keys(n, cluster, g)
    v = g.random(n)
    ids = np.arange(n, dtype=np.uint32)[::-1].copy()
    rs, perm, cols, ids_s = hmc.hmc_sort_by_radius(dev(r), (dev(v),), dev(ids.view(np.int32)))
    o_rs, o_perm, o_cols, o_ids = oracle.sort_by_radius(r, (v,), ids)
    assert np.array_equal(host(perm, np.uint32), o_perm)
    assert np.array_equal(host(rs), o_rs)
    assert np.array_equal(host(cols[0]), o_cols[0])
    assert np.array_equal(host(ids_s, np.uint32), o_ids)


@pytest.mark.parametrize("ncols,with_id", [(0, False), (0, True), (1, False), (6, True), (7, True), (8, False)])
def test_sort_column_counts(oracle, ncols, with_id):
    """0..8 record columns, with and without the id column (up to 6 columns travel as 64-byte records,
    more are gathered column by column)."""
    g = np.random.default_rng(3 + ncols)
    n = 70_001
    r = np.exp(g.uniform(-5, 5, n))
    cols = [g.random(n) for _ in range(ncols)]
    ids = g.permutation(n).astype(np.uint32)
    rs, perm, cols_s, ids_s = hmc.hmc_sort_by_radius(dev(r), [dev(c) for c in cols],
                                                     dev(ids.view(np.int32)) if with_id else None)
    o_rs, o_perm, o_cols, o_ids = oracle.sort_by_radius(r, tuple(cols), ids if with_id else None)
    assert np.array_equal(host(perm, np.uint32), o_perm)
    assert np.array_equal(host(rs), o_rs)
    for a, b in zip(cols_s, o_cols):
        assert np.array_equal(host(a), b)
    if with_id:
        assert np.array_equal(host(ids_s, np.uint32), o_ids)


def test_sort_empty_and_errors():
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    rs, perm, _, _ = hmc.hmc_sort_by_radius(e)
    assert rs.numel() == 0
    r = torch.ones(8, dtype=torch.float64, device="cuda")
    with pytest.raises(hmc.HmcError):
        hmc.hmc_sort_by_radius(r, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))   # too small
    with pytest.raises(hmc.HmcError):
        hmc.hmc_sort_by_radius(r.float())


# ----------------------------------------------------------------------------- S2
@pytest.mark.parametrize("n,masses", [(1, "equal"), (2047, "equal"), (2048, "equal"), (2049, "salpeter"),
                                      (100_000, "equal"), (1_000_003, "salpeter")])
def test_potential_matches_oracle(oracle, n, masses):
    c = inputs.plummer(n, 200 + n % 89, masses)
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    phi, mc = hmc.hmc_potential(dev(r), dev(m), 1.0)
    o_phi, o_mc = oracle.potential(r, m, 1.0)
    phi, mc = host(phi), host(mc)
    assert rel(phi, o_phi).max() <= TOL_PHI
    assert rel(mc, o_mc).max() <= TOL_PHI
    nbit = int((phi != o_phi).sum() + (mc != o_mc).sum())
    print("potential n=%d: %d of %d values not bit-identical" % (n, nbit, 2 * n))
    assert nbit <= max(2, n // 100_000)        # both sides round the exact sums once (R1p)


def test_potential_with_ties_and_G(oracle):
    r = np.sort(np.floor(np.random.default_rng(1).random(5000) * 100) + 1.0)
    m = np.random.default_rng(2).random(5000)
    phi, mc = hmc.hmc_potential(dev(r), dev(m), 2.5)
    o_phi, o_mc = oracle.potential(r, m, 2.5)
    assert np.array_equal(host(phi), o_phi) and np.array_equal(host(mc), o_mc)


# ----------------------------------------------------------------------------- S3 + S4
def oracle_chain(oracle, c, seed, step, sample=None):
    return oracle.orbit_step(c["r"], c["v_r"], c["v_t"], c["m"], c["id"], seed, step, sample=sample)


def check_orbit_against(oracle, o, tp, sm, sl=slice(None), report=""):
    otp, osm = o["tp"], o["sample"]
    kmin, kmax = host(tp["k_min"], np.uint32)[sl], host(tp["k_max"], np.uint32)[sl]
    assert np.array_equal(kmin, otp["k_min"]) and np.array_equal(kmax, otp["k_max"])
    assert np.array_equal(host(tp["status"])[sl], otp["status"])
    for key in ("E", "J", "r_min", "r_max"):
        assert rel(host(tp[key])[sl], otp[key]).max() <= TOL_ROOT, key
    assert np.array_equal(host(sm["status"])[sl], osm["status"])
    d = rel(host(sm["r_new"])[sl], osm["r_new"])
    flips = int((host(sm["n_try"], np.uint16)[sl] != osm["n_try"]).sum())
    frac = float((d <= TOL_RNEW).mean())
    nbit = int((host(sm["r_new"])[sl] != osm["r_new"]).sum())
    print("%s stars=%d  r_new within 1e-10: %.6f%%  not bit-identical: %d  rejection flips: %d"
          % (report, d.size, 100 * frac, nbit, flips))
    assert frac >= FRAC_RNEW
    assert flips <= max(1, d.size // 100_000)
    ok = d <= TOL_RNEW
    assert rel(host(sm["v_t_new"])[sl][ok], osm["v_t_new"][ok]).max() <= 1e-9
    assert rel(np.abs(host(sm["v_r_new"])[sl][ok]), np.abs(osm["v_r_new"][ok])).max() <= 1e-6
    return flips


@pytest.mark.parametrize("n,masses,seed", [(1, "equal", 3), (2, "equal", 4), (1000, "equal", 5), (100_000, "equal", 1),
                                           (250_007, "salpeter", 9)])
def test_orbit_stage_isolation_on_oracle_tables(oracle, n, masses, seed):
    """S3 and S4 fed the ORACLE's sorted arrays and potential (stage isolation)."""
    c = inputs.plummer(n, seed, masses)
    o = oracle_chain(oracle, c, seed, 2)
    rs, vrs, vts, phi, mc = (dev(o[k]) for k in ("r", "v_r", "v_t", "phi", "m_cum"))
    counters = hmc.alloc_counters()
    tp = hmc.hmc_orbit_turning_points(rs, vrs, vts, phi, mc, 1.0, counters=counters)
    sm = hmc.hmc_sample_new_radius(rs, phi, mc, vrs, vts, tp, dev(o["id"].view(np.int32)), seed, 2, 1.0,
                                   counters=counters)
    check_orbit_against(oracle, o, tp, sm, report="isolated n=%d" % n)
    cnt = host(counters)
    assert cnt[hmc.COUNTER_NAMES.index("trials")] == o["sample"]["trials"]
    # the same two calls sharing one workspace, S4 reusing S3's tables and per-star bound F
    ws = hmc.alloc_workspace(n)
    tp2 = hmc.hmc_orbit_turning_points(rs, vrs, vts, phi, mc, 1.0, workspace=ws)
    sm2 = hmc.hmc_sample_new_radius(rs, phi, mc, vrs, vts, tp2, dev(o["id"].view(np.int32)), seed, 2, 1.0,
                                    workspace=ws, reuse_tables=True)
    for key in ("r_new", "v_r_new", "v_t_new", "n_try", "status"):
        assert torch.equal(sm[key], sm2[key]), key


@pytest.mark.parametrize("n,masses", [(1, "equal"), (33, "equal"), (100_000, "equal"), (300_001, "salpeter")])
def test_fused_orbit_step_equals_the_two_calls(n, masses):
    """hmc_orbit_step (S3 + S4 in one launch) writes bit for bit what the two calls write, counters included."""
    c = inputs.plummer(n, 21, masses)
    rs, perm, (vrs, vts, ms), ids = hmc.hmc_sort_by_radius(dev(c["r"]), (dev(c["v_r"]), dev(c["v_t"]), dev(c["m"])),
                                                           dev(c["id"].view(np.int32)))
    phi, mc = hmc.hmc_potential(rs, ms)
    c1, c2 = hmc.alloc_counters(), hmc.alloc_counters()
    ws = hmc.alloc_workspace(n)
    tp = hmc.hmc_orbit_turning_points(rs, vrs, vts, phi, mc, counters=c1, workspace=ws)
    sm = hmc.hmc_sample_new_radius(rs, phi, mc, vrs, vts, tp, ids, 21, 5, counters=c1, workspace=ws, reuse_tables=True)
    tp2, sm2 = hmc.hmc_orbit_step(rs, vrs, vts, phi, mc, ids, 21, 5, counters=c2)
    for key in tp:
        assert torch.equal(tp[key], tp2[key]), key
    for key in sm:
        assert torch.equal(sm[key], sm2[key]), key
    assert torch.equal(c1, c2)


def test_config1_whole_step_chained(oracle):
    """BASELINE.json configs[0]: Plummer N = 1e5, seed 1, one orbit step -- all four GPU stages chained."""
    cfg = inputs.config(0)
    c = {k: cfg[k] for k in ("r", "v_r", "v_t", "m", "id")}
    o = oracle_chain(oracle, c, cfg["seed"], 0)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)),
                          cfg["seed"])
    st.step()
    assert np.array_equal(host(st.sorted["perm"], np.uint32), o["perm"])
    assert rel(host(st.phi), o["phi"]).max() <= TOL_PHI
    # after the step the carried state holds r_new etc.; the sample dict holds the swapped-out buffers
    sm = dict(st.sample)
    sm["r_new"], sm["v_r_new"], sm["v_t_new"] = st.state["r"], st.state["v_r"], st.state["v_t"]
    check_orbit_against(oracle, o, st.tp, sm, report="config1")
    assert np.array_equal(host(st.state["id"], np.uint32), o["id"])
    assert np.array_equal(host(st.state["m"]), o["m"])


def test_config2_eleven_chained_steps(oracle):
    """A quick version of BASELINE.json configs[1] at N = 60 000 (same recipe, seed 2): 1 + 10 steps re-sorting each
    step; tests/test_gpu_fullsize.py::test_config2_1e6_eleven_steps runs the config itself at its full N = 1e6.
    The oracle is fed its own previous output; the GPU its own.  Any divergence would compound."""
    cfg = inputs.config(1, n_override=60_000)
    c = {k: cfg[k] for k in ("r", "v_r", "v_t", "m", "id")}
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)),
                          cfg["seed"])
    r, vr, vt, m, ids = c["r"], c["v_r"], c["v_t"], c["m"], c["id"]
    total_flips = 0
    for step in range(11):
        o = oracle.orbit_step(r, vr, vt, m, ids, cfg["seed"], step)
        st.step()
        sm = dict(st.sample)
        sm["r_new"], sm["v_r_new"], sm["v_t_new"] = st.state["r"], st.state["v_r"], st.state["v_t"]
        assert np.array_equal(host(st.sorted["perm"], np.uint32), o["perm"])
        total_flips += check_orbit_against(oracle, o, st.tp, sm, report="config2 step %d" % step)
        s = o["sample"]
        r, vr, vt, m, ids = s["r_new"], s["v_r_new"], s["v_t_new"], o["m"], o["id"]
    assert total_flips == 0
    cnt = host(st.counters)
    assert cnt[:5].sum() == 0                     # no unbound / radial / degenerate / circular / maxtries


def test_order_independence_of_the_draw(oracle):
    """Permuting the stars of S4's per-star inputs permutes its outputs exactly (Philox keyed by id)."""
    c = inputs.plummer(30_000, 77)
    o = oracle_chain(oracle, c, 77, 0)
    rs, vrs, vts, phi, mc = (dev(o[k]) for k in ("r", "v_r", "v_t", "phi", "m_cum"))
    ids = dev(o["id"].view(np.int32))
    tp = hmc.hmc_orbit_turning_points(rs, vrs, vts, phi, mc)
    a = hmc.hmc_sample_new_radius(rs, phi, mc, vrs, vts, tp, ids, 77, 0)
    p = torch.randperm(30_000, device="cuda", generator=torch.Generator("cuda").manual_seed(0))
    tpp = {k: v[p].contiguous() for k, v in tp.items()}
    # tables stay in sorted order; only the per-star arrays are permuted.  v_r / v_t pass-through columns too.
    b = hmc.hmc_sample_new_radius(rs, phi, mc, vrs[p].contiguous(), vts[p].contiguous(), tpp, ids[p].contiguous(), 77, 0)
    # r pass-through uses r_sorted[a] for flagged stars only; none are flagged here
    assert int(a["status"].sum()) == 0
    for key in ("r_new", "v_r_new", "v_t_new", "n_try"):
        assert torch.equal(b[key], a[key][p])


def test_flagged_stars(oracle):
    r = np.array([1.0, 2.0, 3.0, 4.0])
    m = np.array([0.25, 0.25, 0.25, 0.25])
    vr = np.array([0.1, 5.0, 0.1, 0.0])
    vt = np.array([0.3, 0.1, 0.0, 0.3])
    phi, mc = oracle.potential(r, m)
    otp = oracle.orbit_turning_points(r, vr, vt, phi, mc)
    ids = np.arange(4, dtype=np.uint32)
    osm = oracle.sample_new_radius(r, phi, mc, r, vr, vt, otp["E"], otp["J"], otp["r_min"], otp["r_max"],
                                   otp["k_min"], otp["k_max"], ids, otp["status"], 1, 0)
    counters = hmc.alloc_counters()
    tp = hmc.hmc_orbit_turning_points(dev(r), dev(vr), dev(vt), dev(phi), dev(mc), counters=counters)
    sm = hmc.hmc_sample_new_radius(dev(r), dev(phi), dev(mc), dev(vr), dev(vt), tp, dev(ids.view(np.int32)), 1, 0,
                                   counters=counters)
    assert np.array_equal(host(tp["status"]), otp["status"])
    assert np.array_equal(host(sm["status"]), osm["status"])
    for key in ("r_new", "v_r_new", "v_t_new"):
        assert np.array_equal(host(sm[key]), osm[key])
    assert np.array_equal(host(tp["r_max"]), otp["r_max"]) and np.array_equal(host(tp["r_min"]), otp["r_min"])
    cnt = host(counters)
    assert cnt[0] == 1 and cnt[1] == 1


def test_host_buffer_step_matches_device_step(oracle):
    n = 50_000
    c = inputs.plummer(n, 55)
    o = oracle_chain(oracle, c, 55, 7)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = dict(r_new=torch.empty(n, dtype=torch.float64).pin_memory(), v_r_new=torch.empty(n, dtype=torch.float64).pin_memory(),
               v_t_new=torch.empty(n, dtype=torch.float64).pin_memory(), m=torch.empty(n, dtype=torch.float64).pin_memory(),
               id=torch.empty(n, dtype=torch.int32).pin_memory())
    arena = torch.empty(hmc.step_host_arena_bytes(n), dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(hmc.NCOUNTERS, dtype=torch.int64).pin_memory()
    hmc.hmc_step_host(pin(c["r"]), pin(c["v_r"]), pin(c["v_t"]), pin(c["m"]), pin(c["id"].view(np.int32)), out, 55, 7,
                      arena=arena, counters_host=cnt)
    torch.cuda.synchronize()
    assert np.array_equal(out["id"].numpy().view(np.uint32), o["id"])
    assert np.array_equal(out["m"].numpy(), o["m"])
    d = rel(out["r_new"].numpy(), o["sample"]["r_new"])
    assert (d <= TOL_RNEW).mean() >= FRAC_RNEW
    assert int(cnt[hmc.COUNTER_NAMES.index("trials")]) == o["sample"]["trials"]


# ----------------------------------------------------------------------------- diagnostics
@pytest.mark.parametrize("n,masses", [(1, "equal"), (2, "equal"), (255, "equal"), (100_000, "equal"), (1_000_003, "salpeter")])
def test_diagnostics_match_oracle(oracle, n, masses):
    """M, T, W, E_tot, virial ratio, r_h and the Lagrange radii bit for bit (exact sums rounded once on both sides,
    index work for the radii); t_rh to 1e-14 (one logarithm from two different math libraries)."""
    c = inputs.plummer(n, 31, masses)
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    phi, mc = oracle.potential(rs, ms)
    fr = [1e-6, 0.01, 0.1, 0.25, 0.5, 0.75, 0.9, 0.99, 1.0]
    o = oracle.diagnostics(rs, vrs, vts, ms, phi, mc, fr)
    out = host(hmc.hmc_diagnostics(dev(rs), dev(vrs), dev(vts), dev(ms), dev(phi), dev(mc), fr))
    for i, name in enumerate(hmc.DIAG_NAMES):
        if name == "t_rh":
            assert out[i] == o[name] or abs(out[i] - o[name]) <= 1e-14 * abs(o[name]) or (np.isnan(out[i]) and np.isnan(o[name])), name
        else:
            assert out[i] == o[name] or (np.isnan(out[i]) and np.isnan(o[name])), (name, out[i], o[name])
    assert np.array_equal(out[7:], o["lagrange"])
    # no fractions asked for
    out0 = host(hmc.hmc_diagnostics(dev(rs), dev(vrs), dev(vts), dev(ms), dev(phi), dev(mc)))
    assert np.array_equal(out0[:6], out[:6])


def test_diagnostics_errors():
    z = torch.ones(4, dtype=torch.float64, device="cuda")
    with pytest.raises(hmc.HmcError):
        hmc.hmc_diagnostics(z, z, z, z, z, z, [0.5] * 17)          # more than HMC_DIAG_MAX_FRACTIONS


def test_stepper_diagnostics_after_a_step(oracle):
    c = inputs.plummer(50_000, 17)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)), 17)
    st.step()
    o = oracle_chain(oracle, c, 17, 0)
    od = oracle.diagnostics(o["r"], o["v_r"], o["v_t"], o["m"], o["phi"], o["m_cum"], [0.1, 0.5])
    out = host(st.diagnostics([0.1, 0.5]))
    assert [out[i] for i in range(6)] == [od[k] for k in hmc.DIAG_NAMES[:6]]
    assert np.array_equal(out[7:], od["lagrange"])


# ----------------------------------------------------------------------------- energy correction
def _second_configuration(oracle, n, seed, masses):
    """Oracle: one step, then sort + potential of the new configuration, with the three carried columns."""
    c = inputs.plummer(n, seed, masses)
    o = oracle_chain(oracle, c, seed, 0)
    sm, tp = o["sample"], o["tp"]
    rs, perm, cs, ids = oracle.sort_by_radius(sm["r_new"], (sm["v_r_new"], sm["v_t_new"], o["m"], tp["E"], o["r"], o["phi"]), o["id"])
    phi, mc = oracle.potential(rs, cs[2])
    return rs, phi, mc, cs


@pytest.mark.parametrize("n,masses", [(1, "equal"), (3, "equal"), (100_000, "equal"), (250_007, "salpeter")])
def test_energy_correction_matches_oracle(oracle, n, masses):
    """Same expressions, correctly rounded operations: the corrected velocities and the flags are bit-identical."""
    rs, phi, mc, (vrs, vts, ms, E, r_old, p_old) = _second_configuration(oracle, n, 23, masses)
    o_vr, o_vt, o_st = oracle.energy_correction(rs, phi, mc, E, r_old, p_old, vrs, vts)
    counters = hmc.alloc_counters()
    vr, vt, st = hmc.hmc_energy_correction(dev(rs), dev(phi), dev(mc), dev(E), dev(r_old), dev(p_old), dev(vrs), dev(vts),
                                           counters=counters)
    assert np.array_equal(host(st), o_st)
    assert np.array_equal(host(vr), o_vr) and np.array_equal(host(vt), o_vt)
    assert host(counters)[hmc.COUNTER_NAMES.index("nokinetic")] == int((o_st != 0).sum())
    # r_old inside the innermost star and beyond the outermost one (shells 0 and N of the new table)
    if n >= 3:
        r_old2 = r_old.copy(); r_old2[0] = rs[0] * 0.5; r_old2[-1] = rs[-1] * 3.0
        o2 = oracle.energy_correction(rs, phi, mc, E, r_old2, p_old, vrs, vts)
        g2 = hmc.hmc_energy_correction(dev(rs), dev(phi), dev(mc), dev(E), dev(r_old2), dev(p_old), dev(vrs), dev(vts))
        assert np.array_equal(host(g2[0]), o2[0]) and np.array_equal(host(g2[1]), o2[1]) and np.array_equal(host(g2[2]), o2[2])


def test_stepper_with_energy_correction_conserves_total_energy(oracle):
    """Three chained steps with the correction on: T + W from hmc_diagnostics stays put (to the shortfall of the
    few flagged stars), and the state equals an oracle chain of the same calls."""
    n, seed = 60_000, 29
    c = inputs.plummer(n, seed)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)), seed,
                          energy_correction=True)
    state = {k: c[k] for k in ("r", "v_r", "v_t", "m", "id")}
    e = []
    for step in range(3):
        st.step()
        e.append(host(st.diagnostics())[3])
        # oracle: the same step
        have = "E" in state
        cols = [state["v_r"], state["v_t"], state["m"]] + ([state["E"], state["r_old"], state["p_old"]] if have else [])
        rs, perm, cs, ids = oracle.sort_by_radius(state["r"], tuple(cols), state["id"])
        vrs, vts, ms = cs[0], cs[1], cs[2]
        phi, mc = oracle.potential(rs, ms)
        if have:
            vrs, vts, _ = oracle.energy_correction(rs, phi, mc, cs[3], cs[4], cs[5], vrs, vts)
        tp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
        sm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, tp["E"], tp["J"], tp["r_min"], tp["r_max"], tp["k_min"],
                                      tp["k_max"], ids, tp["status"], seed, step)
        state = dict(r=sm["r_new"], v_r=sm["v_r_new"], v_t=sm["v_t_new"], m=ms, id=ids, E=tp["E"], r_old=rs, p_old=phi)
        assert np.array_equal(host(st.state["r"]), state["r"]) and np.array_equal(host(st.state["v_r"]), state["v_r"])
        assert np.array_equal(host(st.state["v_t"]), state["v_t"])
    nok = int(host(st.counters)[hmc.COUNTER_NAMES.index("nokinetic")])
    assert nok < 40
    assert abs(e[2] - e[0]) <= 2e-5 * abs(e[0])            # uncorrected: about 1e-4 per step at this N


def test_energy_correction_steps_replayed_from_a_graph_equal_eager_steps():
    """The correction's three extra columns are handed from step to step by exchanging buffers (no copies), so this
    mode can be captured too: six steps through run_graph (two eager, two captured, replayed twice) leave the same
    bits as six eager steps, in the state and in what the last step's S1-S3 produced."""
    n, seed = 100_000, 31
    c = inputs.plummer(n, seed)
    mk = lambda: hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)), seed,
                                  energy_correction=True)
    eager, graph = mk(), mk()
    for _ in range(6):
        eager.step()
    graph.run_graph(6)
    torch.cuda.synchronize()
    assert graph.step_index == eager.step_index == 6
    for k in ("r", "v_r", "v_t", "m", "id"):
        assert torch.equal(graph.state[k], eager.state[k]), k
    assert torch.equal(graph.sorted["r"], eager.sorted["r"]) and torch.equal(graph.phi, eager.phi)
    assert torch.equal(graph.tp["E"], eager.tp["E"])
    assert torch.equal(graph.counters, eager.counters)
    eager.step(); graph.step()                      # and an eager step after the replays picks up where they left
    assert torch.equal(graph.state["r"], eager.state["r"])


def test_twenty_step_soak_properties():
    """Twenty chained steps of a 10^6-star cluster with the energy correction on: properties that hold at any size
    and step (no oracle): sorted radii, the ids stay a permutation, no star flagged by S3/S4, the cluster stays in
    virial equilibrium with a stable half-mass radius, and T + W moves only by the flagged stars' shortfall."""
    n, seed = 1_000_000, 41
    c = inputs.plummer(n, seed)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)), seed,
                          energy_correction=True)
    e, rh = [], []
    for step in range(20):
        st.step()
        r = st.sorted["r"]
        assert bool((r[1:] >= r[:-1]).all())
        dg = host(st.diagnostics())
        e.append(dg[3]); rh.append(dg[5])
        assert abs(dg[4] - 1.0) < 0.01
    assert torch.equal(torch.sort(st.state["id"].long())[0], torch.arange(n, device="cuda"))
    cnt = dict(zip(hmc.COUNTER_NAMES, host(st.counters).tolist()))
    assert cnt["unbound"] == cnt["radial"] == cnt["degenerate"] == cnt["circular"] == cnt["maxtries"] == 0
    assert cnt["nokinetic"] < 20 * n * 1e-4 and 1.5 * 20 * n < cnt["trials"] < 2.5 * 20 * n
    assert abs(e[-1] - e[0]) <= 2e-6 * abs(e[0])
    assert max(rh) / min(rh) < 1.01


def test_empty_inputs_are_no_ops():
    """n = 0: every call returns HMC_OK without touching anything (include/hmc.h conventions)."""
    f = torch.empty(0, dtype=torch.float64, device="cuda")
    i = torch.empty(0, dtype=torch.int32, device="cuda")
    ws = hmc.alloc_workspace(0)
    phi, mc = hmc.hmc_potential(f, f, workspace=ws)
    assert phi.numel() == 0 and mc.numel() == 0
    tp = hmc.hmc_orbit_turning_points(f, f, f, f, f, workspace=ws)
    sm = hmc.hmc_sample_new_radius(f, f, f, f, f, tp, i, 1, 0, workspace=ws)
    assert sm["r_new"].numel() == 0
    tp2, sm2 = hmc.hmc_orbit_step(f, f, f, f, f, i, 1, 0, workspace=ws)
    assert sm2["r_new"].numel() == 0
    vr, vt, st = hmc.hmc_energy_correction(f, f, f, f, f, f, f, f, workspace=ws)
    assert vr.numel() == 0
    with pytest.raises(hmc.HmcError):                      # the diagnostics of nothing are not defined
        hmc.hmc_diagnostics(f, f, f, f, f, f, workspace=ws)
    torch.cuda.synchronize()


@pytest.mark.parametrize("n", [10_238, 10_239, 20_476, 20_477, 40_957])
def test_sizes_around_the_coarse_table_capacity(oracle, n):
    """The coarse table holds every 2^shift-th node and at most 10 240 entries: n = 10 238 is the last size
    with the whole table in shared memory (shift 0), 10 239 the first with a directory (shift 1), and so on."""
    c = inputs.plummer(n, 5)
    o = oracle_chain(oracle, c, 5, 0)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32)), 5)
    st.step()
    assert np.array_equal(host(st.sorted["perm"], np.uint32), o["perm"])
    assert np.array_equal(host(st.phi), o["phi"])
    sm = dict(r_new=st.state["r"], v_r_new=st.state["v_r"], v_t_new=st.state["v_t"], n_try=st.sample["n_try"],
              status=st.sample["status"])                  # step() swapped the new coordinates into the state
    check_orbit_against(oracle, o, st.tp, sm, report="n=%d" % n)
    assert np.array_equal(host(st.state["r"]), o["sample"]["r_new"])


@pytest.mark.parametrize("copies", [2, 5])
def test_orbit_stages_with_tied_radii(oracle, copies):
    """Every radius occurs `copies` times (distinct velocities and masses): nodes of equal radius, zero-width
    shells, directory buckets holding several identical radii.  Brackets bit-exact, the rest as usual."""
    g = np.random.default_rng(77)
    base = inputs.plummer(60_000 // copies, 19)
    r = np.repeat(base["r"], copies)
    n = r.shape[0]
    vr, vt = g.permutation(np.repeat(base["v_r"], copies)), np.abs(g.permutation(np.repeat(base["v_t"], copies))) + 1e-3
    m = g.uniform(0.5, 1.5, n); m /= m.sum()
    c = dict(r=r, v_r=vr, v_t=vt, m=m, id=np.arange(n, dtype=np.uint32))
    o = oracle_chain(oracle, c, 19, 3)
    rs, vrs, vts, phi, mc = (dev(o[k]) for k in ("r", "v_r", "v_t", "phi", "m_cum"))
    ws = hmc.alloc_workspace(n)
    tp = hmc.hmc_orbit_turning_points(rs, vrs, vts, phi, mc, workspace=ws)
    sm = hmc.hmc_sample_new_radius(rs, phi, mc, vrs, vts, tp, dev(o["id"].view(np.int32)), 19, 3, workspace=ws,
                                   reuse_tables=True)
    check_orbit_against(oracle, o, tp, sm, report="ties x%d" % copies)
    assert np.array_equal(host(hmc.hmc_sort_by_radius(dev(r))[1], np.uint32), o["perm"])


def test_repeated_steps_are_bit_reproducible():
    """The same step run ten times from the same state writes the same bits every time, every array.  The sort's
    decoupled look-back, the sampler's dynamic batches and the shared-memory parking all order their work
    differently from run to run; a data race would show as a difference (compute-sanitizer is closed on this pool:
    profiles/r2b.md).  Covers the fast sort path, the fallback sort (runs of 200 near-equal keys) and the fused call."""
    n, seed = 400_003, 61
    c = inputs.plummer(n, seed, "salpeter")
    r = c["r"].copy()
    r[:60_000] = _clustered_keys(60_000, 200, np.random.default_rng(2))       # long runs: the guarded general sort runs
    d = [dev(r), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32))]
    first = None
    for rep in range(10):
        st = hmc.OrbitStepper(*d, seed)
        st.step()
        st.step(fused=(rep % 2 == 1))
        got = dict(perm=st.sorted["perm"], phi=st.phi, m_cum=st.m_cum, r=st.state["r"], v_r=st.state["v_r"], v_t=st.state["v_t"],
                   id=st.state["id"], n_try=st.sample["n_try"], status=st.sample["status"], counters=st.counters,
                   **{"tp_" + k: v for k, v in st.tp.items()})
        got = {k: v.clone() for k, v in got.items()}
        if first is None:
            first = got
        else:
            for k in first:
                assert torch.equal(first[k], got[k]), (rep, k)


@pytest.mark.parametrize("n", [1, 5_000, 100_000, 400_003])
def test_graph_replay_equals_eager_steps(oracle, n):
    """OrbitStepper.run_graph: a CUDA graph of two steps, the Philox step number kept on the device
    (hmc_sample_new_radius_dstep / hmc_add_u32).  Eight steps by replay leave the same bits as eight eager steps,
    and the last one is compared with the oracle (so the step numbers really advanced); eager steps and replays
    can be mixed."""
    seed = 77
    c = inputs.plummer(n, seed)
    d = [dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"].view(np.int32))]
    eager = hmc.OrbitStepper(*d, seed)
    for _ in range(7):
        eager.step()
    before = {k: host(eager.state[k]) for k in ("r", "v_r", "v_t", "m")}
    before["id"] = host(eager.state["id"], np.uint32)
    eager.step()
    g = hmc.OrbitStepper(*d, seed)
    g.run_graph(4)                        # two eager steps (first launches), capture, one replay
    g.step()
    g.step()
    g.run_graph(2)
    torch.cuda.synchronize()
    assert g.step_index == eager.step_index == 8
    for k in ("r", "v_r", "v_t", "m", "id"):
        assert torch.equal(g.state[k], eager.state[k]), k
    for k in ("n_try", "status"):
        assert torch.equal(g.sample[k], eager.sample[k]), k
    assert torch.equal(g.counters, eager.counters)
    g.step()                              # an odd number of eager steps leaves the other buffer arrangement:
    with pytest.raises(hmc.HmcError):     # the captured graph must refuse to run from it
        g.run_graph(2)
    o = oracle.orbit_step(before["r"], before["v_r"], before["v_t"], before["m"], before["id"], seed, 7)
    assert np.array_equal(host(eager.state["r"]), o["sample"]["r_new"])
    assert np.array_equal(host(eager.sample["n_try"], np.uint16), o["sample"]["n_try"])


@pytest.mark.parametrize("n", [1, 40, 100_003, 1_200_000])
def test_prebuilt_tables_equal_the_one_call(oracle, n):
    """hmc_orbit_build_tables + hmc_orbit_turning_points_prebuilt (whole table, and a range of it) against
    hmc_orbit_turning_points: the same two launches, the same bits; one case against the oracle as well."""
    seed = 31
    c = inputs.plummer(n, seed)
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(c["r"], (c["v_r"], c["v_t"], c["m"]), c["id"])
    phi, mc = oracle.potential(rs, ms)
    d = [dev(x) for x in (rs, vrs, vts, phi, mc)]
    ws = hmc.alloc_workspace(n)
    one = hmc.hmc_orbit_turning_points(*d, 1.0, workspace=ws)
    one = {k: v.clone() for k, v in one.items()}
    ws2 = hmc.alloc_workspace(n)
    hmc.hmc_orbit_build_tables(d[0], d[3], d[4], 1.0, workspace=ws2)
    two = hmc.hmc_orbit_turning_points(*d, 1.0, workspace=ws2, prebuilt=True)
    for k in one:
        assert torch.equal(one[k], two[k]), k
    first, count = n // 3, max(1, n // 5)
    part = hmc.hmc_orbit_turning_points(d[0], d[1][first:first + count].contiguous(), d[2][first:first + count].contiguous(),
                                        d[3], d[4], 1.0, workspace=ws2, first=first, prebuilt=True)
    for k in one:
        assert torch.equal(one[k][first:first + count], part[k]), k
    if n <= 100_003:
        otp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
        assert np.array_equal(host(two["k_min"], np.uint32), otp["k_min"]) and np.array_equal(host(two["r_max"]), otp["r_max"])
