"""Parity on BASELINE.json's five configs at their stated sizes and step counts, in the launch configuration
bench.py times (hmc.OrbitStepper: the four C-ABI calls chained on one stream).

configs[0..3] (N = 1e5, 1e6, 1e7, 1e7 Salpeter; 1, 1 + 10, 10, 10 steps): the oracle runs its OWN chain (fed its
own previous output) and the GPU its own; after every step EVERY star is compared: permutation, sorted columns
and brackets bit for bit, Phi / M / E / J / r_min / r_max to 1e-12, new radii to 1e-10 with rejection flips
counted.  Any divergence would compound over the steps.  The oracle is the -fopenmp build of the same source
(bit-identical to the single-threaded one, tests/test_oracle_variants.py), or a step at N = 1e7 would take 30 s.

configs[4] (N = 1e8, 5 steps): the oracle cannot draw 1e8 stars in the time there is (about 10 min per step);
it follows the GPU's carried state: S1 and S2 on EVERY star of every step, S3 / S4 on every 16th star of the
sorted order against the full table ("S1/S2 on all 1e8 stars and S3/S4 on every 16th star"),
the offset moving with the step.  The five steps are checked concurrently (the oracle's Quicksort of 1e8 keys is
serial and takes most of a minute).  Properties that hold at any size are checked on every star of every step.
"""
import concurrent.futures as cf

import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import hmc, inputs

pytestmark = pytest.mark.gpu

TOL = 1e-12
TOL_RNEW = 1e-10


def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def host(t, dtype=None):
    a = t.cpu().numpy()
    return a.view(dtype) if dtype is not None else a


def rel(a, b):
    with np.errstate(divide="ignore", invalid="ignore"):
        d = np.abs(a - b) / np.maximum(np.abs(b), 1e-300)
    d[a == b] = 0.0
    return d


def need_memory(n):
    free, _ = torch.cuda.mem_get_info()
    if free < 300 * n:
        pytest.skip("needs %.0f GB of device memory" % (300 * n / 1e9))


def make_stepper(cfg):
    return hmc.OrbitStepper(dev(cfg["r"]), dev(cfg["v_r"]), dev(cfg["v_t"]), dev(cfg["m"]), dev(cfg["id"].view(np.int32)),
                            cfg["seed"])


def properties_on_every_star(st, n):
    """Checked on the device (torch as plumbing): sorted radii, r_min <= r_new <= r_max, J = r v_t carried,
    the energy identity at the new radius through Eq. 16 with Phi(r_new) bounded by the bracket."""
    rs, tp = st.sorted["r"], st.tp
    assert bool((rs[1:] >= rs[:-1]).all())
    status = st.sample["status"]
    drawn = (status & (255 - hmc.ST_CLIPPED)) == 0
    assert float(drawn.double().mean()) > 0.999
    r_new, vr_new, vt_new = st.state["r"], st.state["v_r"], st.state["v_t"]       # step() swapped them in
    assert bool(((r_new >= tp["r_min"]) & (r_new <= tp["r_max"]))[drawn].all())
    j_new = r_new * vt_new
    assert float(((j_new - tp["J"]).abs() / tp["J"].abs())[drawn].max()) <= 5e-16
    # Q(r_new) = v_r'^2 >= 0 and E = Phi(r_new) + K  =>  Phi(r_new) = E - K must lie within the potential's
    # range over the orbit, [Phi(r_min), Phi(r_max)] subset of [Phi_1, 0]
    phi_new = tp["E"] - 0.5 * (vr_new * vr_new + vt_new * vt_new)
    assert bool(((phi_new >= st.phi[0] * (1 + 1e-12)) & (phi_new <= 0.0))[drawn].all())


def compare_step(oracle, o, g, sl, label):
    """o: oracle.orbit_step output (S3/S4 compact over the slice sl); g: host copies of the GPU's arrays."""
    n = o["r"].shape[0]
    assert np.array_equal(g["perm"], o["perm"]), "permutation"
    for k in ("r", "v_r", "v_t", "m"):
        assert np.array_equal(g[k], o[k]), k
    assert np.array_equal(g["id"], o["id"])
    assert rel(g["phi"], o["phi"]).max() <= TOL and rel(g["m_cum"], o["m_cum"]).max() <= TOL
    nbit = int((g["phi"] != o["phi"]).sum() + (g["m_cum"] != o["m_cum"]).sum())
    assert nbit <= max(2, n // 100_000), "Phi / M values not bit-identical: %d" % nbit      # R1p: both round the exact sums once
    otp, osm = o["tp"], o["sample"]
    assert np.array_equal(g["k_min"], otp["k_min"]) and np.array_equal(g["k_max"], otp["k_max"])
    assert np.array_equal(g["tp_status"], otp["status"])
    for k in ("E", "J", "r_min", "r_max"):
        assert rel(g[k], otp[k]).max() <= TOL, k
    assert np.array_equal(g["status"], osm["status"])
    d = rel(g["r_new"], osm["r_new"])
    flips = int((g["n_try"] != osm["n_try"]).sum())
    frac = float((d <= TOL_RNEW).mean())
    nbit_r = int((g["r_new"] != osm["r_new"]).sum())
    print("%s: N=%d, %d stars of S3/S4 compared; Phi/M not bit-identical: %d; r_new within 1e-10: %.6f%%, "
          "not bit-identical: %d, rejection flips: %d" % (label, n, d.size, nbit, 100 * frac, nbit_r, flips))
    assert frac >= 0.99999 and flips <= max(1, d.size // 100_000)
    ok = d <= TOL_RNEW
    assert rel(g["v_t_new"][ok], osm["v_t_new"][ok]).max() <= 1e-9
    assert rel(np.abs(g["v_r_new"][ok]), np.abs(osm["v_r_new"][ok])).max() <= 1e-6
    return flips, nbit_r


def gpu_arrays(st, sl):
    """Host copies of what a step produced; the per-star S3/S4 arrays restricted to the slice sl."""
    so, tp, sm = st.sorted, st.tp, st.sample
    cut = (lambda t: t) if sl == slice(None) else (lambda t: t[sl].contiguous())
    g = dict(perm=host(so["perm"], np.uint32), r=host(so["r"]), v_r=host(so["v_r"]), v_t=host(so["v_t"]),
             m=host(st.state["m"]), id=host(st.state["id"], np.uint32), phi=host(st.phi), m_cum=host(st.m_cum))
    g.update(k_min=host(cut(tp["k_min"]), np.uint32), k_max=host(cut(tp["k_max"]), np.uint32), tp_status=host(cut(tp["status"])))
    for k in ("E", "J", "r_min", "r_max"):
        g[k] = host(cut(tp[k]))
    g.update(status=host(cut(sm["status"])), n_try=host(cut(sm["n_try"]), np.uint16),
             r_new=host(cut(st.state["r"])), v_r_new=host(cut(st.state["v_r"])), v_t_new=host(cut(st.state["v_t"])))
    return g


def run_self_chained(oracle, index, n_override=None, steps=None):
    """Oracle and GPU each run their own chain; every star compared after every step."""
    cfg = inputs.config(index, n_override)
    n, seed = cfg["n"], cfg["seed"]
    steps = cfg["steps"] if steps is None else steps
    need_memory(n)
    st = make_stepper(cfg)
    r, vr, vt, m, ids = cfg["r"], cfg["v_r"], cfg["v_t"], cfg["m"], cfg["id"]
    flips = nbit = 0
    with oracle.use("omp"):
        for step in range(steps):
            o = oracle.orbit_step(r, vr, vt, m, ids, seed, step)
            st.step()
            torch.cuda.synchronize()
            properties_on_every_star(st, n)
            f, b = compare_step(oracle, o, gpu_arrays(st, slice(None)), slice(None), "config[%d] step %d" % (index, step))
            flips += f
            nbit += b
            s = o["sample"]
            r, vr, vt, m, ids = s["r_new"], s["v_r_new"], s["v_t_new"], o["m"], o["id"]
    cnt = dict(zip(hmc.COUNTER_NAMES, host(st.counters).tolist()))
    print("counters:", cnt)
    assert cnt["unbound"] == cnt["radial"] == cnt["degenerate"] == cnt["circular"] == cnt["maxtries"] == 0
    assert flips == 0
    return nbit


def test_config1_1e5_one_step(oracle):
    """BASELINE.json configs[0]: N = 1e5 equal-mass, seed 1, one orbit step."""
    run_self_chained(oracle, 0)


def test_config2_1e6_eleven_steps(oracle):
    """BASELINE.json configs[1]: N = 1e6 equal-mass, seed 2, one orbit step plus 10 repeated steps re-sorting
    each step, at its own size (round 1 ran it at N = 60 000)."""
    run_self_chained(oracle, 1)


def test_config3_headline_1e7_ten_steps(oracle):
    """BASELINE.json configs[2]: N = 1e7 equal-mass, seed 3 (the bench workload), 10 chained steps, every star."""
    run_self_chained(oracle, 2)


def test_config4_salpeter_1e7_ten_steps(oracle):
    """BASELINE.json configs[3]: N = 1e7, Salpeter masses, seed 4, 10 chained steps, every star."""
    run_self_chained(oracle, 3)


def test_second_search_table_just_above_the_coarse_capacity(oracle):
    """N = 1.2e7 (recipe of configs[2]): the coarse table's spacing becomes 2048 nodes, so S3's second
    table (every 1024-th node, in L2) does one bisection step -- the smallest case of the large-N path."""
    run_self_chained(oracle, 2, n_override=12_000_000, steps=1)


def test_second_search_table_with_the_pair_search(oracle, monkeypatch):
    """The same case in the test-only build whose S3 searches by lane pairs at every N: the second table and the
    pair search together, on every star (the product build combines them from N = 2^25 on, where the oracle
    follows on every 16th star only)."""
    from paper_1206_5878_b200 import build as hmc_build
    monkeypatch.setattr(hmc, "_lib", hmc.load(hmc_build.build(variant="pairs")))
    run_self_chained(oracle, 2, n_override=12_000_000, steps=1)


def test_product_large_n_path_on_every_star_at_2_to_the_25(oracle):
    """N = 2^25 = 33 554 432 (recipe of configs[2]) is where the PRODUCT build switches to its large-N path: S3's exact
    search by lane pairs, the second search table doing several bisection steps (coarse spacing 2^12), the four-pass
    sort.  One step, every star, against the oracle's -fopenmp build (about half a minute): the paper's own bar,
    "matching ... to the last significant digit", on the path that N = 1e8 is only sampled on."""
    run_self_chained(oracle, 2, n_override=1 << 25, steps=1)


STRIDE_1E8 = 16


def test_config5_1e8_five_steps(oracle):
    """BASELINE.json configs[4]: N = 1e8 equal-mass, seed 5, 5 chained steps (tables far beyond L2, coarse
    spacing 2^14).  S1 / S2 on every star of every step, S3 / S4 on every 16th star (see the module docstring)."""
    cfg = inputs.config(4)
    n, seed, steps = cfg["n"], cfg["seed"], cfg["steps"]
    need_memory(n)
    st = make_stepper(cfg)
    state = {k: cfg[k] for k in ("r", "v_r", "v_t", "m", "id")}
    del cfg

    def check(step, inp, g, sl):
        o = oracle.orbit_step(inp["r"], inp["v_r"], inp["v_t"], inp["m"], inp["id"], seed, step, sample=(sl.start, sl.step))
        return compare_step(oracle, o, g, sl, "config[4] step %d" % step)

    jobs = []
    with cf.ThreadPoolExecutor(max_workers=steps) as pool:       # the serial oracle releases the GIL inside ctypes
        for step in range(steps):
            sl = slice(step % STRIDE_1E8, None, STRIDE_1E8)
            st.step()
            torch.cuda.synchronize()
            properties_on_every_star(st, n)
            g = gpu_arrays(st, sl)
            jobs.append(pool.submit(check, step, state, g, sl))
            if step + 1 < steps:                                  # the oracle follows the GPU's carried state
                state = dict(r=host(st.state["r"]), v_r=host(st.state["v_r"]), v_t=host(st.state["v_t"]), m=g["m"], id=g["id"])
        results = [j.result() for j in jobs]
    assert sum(f for f, _ in results) <= 1
    cnt = dict(zip(hmc.COUNTER_NAMES, host(st.counters).tolist()))
    print("counters:", cnt)
    assert cnt["unbound"] == cnt["radial"] == cnt["degenerate"] == cnt["circular"] == cnt["maxtries"] == 0


def test_potential_at_the_largest_n_the_header_allows():
    """hmc_potential at n = HMC_MAX_N = 2^28 (round-2 advisor: the launch plan wanted 296 tiles per chunk there and
    the call returned HMC_ERR_SIZE; the largest n any other test reaches is 1e8).  No oracle run at this size: the
    input is chosen so that Eq. 1 has an exact value that Python's rational arithmetic gives at any star --
    m_i = 2^-28, r_i = 2^(i >> 22) (64 blocks of tied radii 1, 2, 4, ... 2^63).  Then M_k = (k + 1) 2^-28 exactly,
    S_k = sum_{i > k} m_i / r_i is a dyadic rational, and the call must return both rounded once (R1p),
    so Phi_k = -(G (M_k / r_k + S_k)) is compared bit for bit on 20 000 sampled stars, the first, the last, and
    the stars on either side of every block edge."""
    from fractions import Fraction
    n = hmc.MAX_N
    free, _ = torch.cuda.mem_get_info()
    if free < 4 * 8 * n + hmc.workspace_bytes(n) + (1 << 30):
        pytest.skip("needs %.0f GB of device memory" % ((32 * n + hmc.workspace_bytes(n)) / 1e9))
    blk = 22
    i = torch.arange(n, dtype=torch.int64, device="cuda")
    r = (((i >> blk) + 1023) << 52).view(torch.float64)          # bit pattern of 2^(i >> 22)
    del i
    m = torch.full((n,), 2.0 ** -28, dtype=torch.float64, device="cuda")
    G = 3.0
    phi, mc = hmc.hmc_potential(r, m, G)
    torch.cuda.synchronize()
    rng = np.random.default_rng(28)
    edges = np.arange(1, 64, dtype=np.int64) << blk
    ks = np.unique(np.concatenate([rng.integers(0, n, 20_000), [0, 1, n - 2, n - 1], edges - 1, edges, edges + 2047, edges + 2048]))
    ks = ks[(ks >= 0) & (ks < n)]
    sel = torch.from_numpy(ks).cuda()
    g_phi, g_mc, g_r = phi[sel].cpu().numpy(), mc[sel].cpu().numpy(), r[sel].cpu().numpy()
    tail = [Fraction(0)] * 65                                     # tail[j] = sum over blocks j' >= j of 2^22 * 2^-j'
    for j in range(63, -1, -1):
        tail[j] = tail[j + 1] + Fraction(1 << blk, 1 << j)
    want_phi, want_mc = np.empty(ks.size), np.empty(ks.size)
    for a, k in enumerate(ks.tolist()):
        j = k >> blk
        rest = ((j + 1) << blk) - 1 - k                           # stars after k inside its own block
        S = float((Fraction(rest, 1 << j) + tail[j + 1]) / (1 << 28))      # exact sum, rounded once
        M = (k + 1) * 2.0 ** -28                                  # exact
        assert g_r[a] == 2.0 ** j
        want_mc[a] = M
        want_phi[a] = -(G * (M / 2.0 ** j + S))
    assert np.array_equal(g_mc, want_mc)
    assert np.array_equal(g_phi, want_phi)
    # every star: M is the exact ramp; Phi is constant inside a block of tied radii (what M_k / r gains, S_k loses)
    assert bool((mc == torch.arange(1, n + 1, dtype=torch.float64, device="cuda") * 2.0 ** -28).all())
    const = [-(G * float((Fraction((j + 1) << blk, 1 << j) + tail[j + 1]) / (1 << 28))) for j in range(64)]
    want_all = torch.tensor(const, dtype=torch.float64, device="cuda").repeat_interleave(1 << blk)
    assert bool(((phi - want_all).abs() <= 4e-16 * want_all.abs()).all())
