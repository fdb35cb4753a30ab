"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(hmc.OrbitStepper: the four C-ABI calls chained on one stream).

The oracle runs S1 and S2 on ALL stars (permutation compared bit for bit, Phi and M on every
star) and S3 / S4 on every STRIDE-th star of the sorted order against the full table (brackets
bit-exact, turning points to 1e-12, new radii to 1e-10, rejection flips counted) -- the "sampled
outputs the oracle can compute one by one" of the task statement.  Properties that hold at any
size are checked on every star: sortedness, permutation validity, r_min <= r_new <= r_max, the
energy identity at the new radius in this step's potential, conservation of J.
"""
import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import hmc, inputs

pytestmark = pytest.mark.gpu

STRIDE = 997


def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def rel(a, b):
    with np.errstate(divide="ignore", invalid="ignore"):
        d = np.abs(a - b) / np.maximum(np.abs(b), 1e-300)
    d[a == b] = 0.0
    return d


def run_fullsize(oracle, index, steps=1, n_override=None):
    cfg = inputs.config(index, n_override)
    n, seed = cfg["n"], cfg["seed"]
    free, _ = torch.cuda.mem_get_info()
    if free < 260 * n:
        pytest.skip("needs %.0f GB of device memory" % (260 * n / 1e9))
    st = hmc.OrbitStepper(dev(cfg["r"]), dev(cfg["v_r"]), dev(cfg["v_t"]), dev(cfg["m"]), dev(cfg["id"].view(np.int32)),
                          seed)
    r, vr, vt, m, ids = cfg["r"], cfg["v_r"], cfg["v_t"], cfg["m"], cfg["id"]
    for step in range(steps):
        if step > 0:       # the oracle follows the GPU's carried state (it cannot afford all stars of S3/S4)
            r, vr, vt = (st.state[k].cpu().numpy() for k in ("r", "v_r", "v_t"))
            m, ids = st.state["m"].cpu().numpy(), st.state["id"].cpu().numpy().view(np.uint32)
        o = oracle.orbit_step(r, vr, vt, m, ids, seed, step, sample=(step % STRIDE, STRIDE))
        st.step()
        torch.cuda.synchronize()
        sl = slice(step % STRIDE, None, STRIDE)
        # ---- S1: every star, bit-exact
        perm = st.sorted["perm"].cpu().numpy().view(np.uint32)
        assert np.array_equal(perm, o["perm"])
        assert np.array_equal(st.sorted["r"].cpu().numpy(), o["r"])
        assert np.array_equal(st.state["id"].cpu().numpy().view(np.uint32), o["id"])
        assert np.array_equal(st.sorted["v_t"].cpu().numpy(), o["v_t"])
        del perm
        # ---- S2: every star
        phi, mc = st.phi.cpu().numpy(), st.m_cum.cpu().numpy()
        assert rel(phi, o["phi"]).max() <= 1e-12
        assert rel(mc, o["m_cum"]).max() <= 1e-12
        nbit = int((phi != o["phi"]).sum() + (mc != o["m_cum"]).sum())
        # ---- S3 / S4: sampled stars against the oracle, star by star
        tp = {k: v.cpu().numpy() for k, v in st.tp.items()}
        otp, osm = o["tp"], o["sample"]
        assert np.array_equal(tp["k_min"].view(np.uint32)[sl], otp["k_min"])
        assert np.array_equal(tp["k_max"].view(np.uint32)[sl], otp["k_max"])
        assert np.array_equal(tp["status"][sl], otp["status"])
        for key in ("E", "J", "r_min", "r_max"):
            assert rel(tp[key][sl], otp[key]).max() <= 1e-12, key
        r_new, vr_new, vt_new = (st.state[k].cpu().numpy() for k in ("r", "v_r", "v_t"))
        d = rel(r_new[sl], osm["r_new"])
        flips = int((st.sample["n_try"].cpu().numpy().view(np.uint16)[sl] != osm["n_try"]).sum())
        status = st.sample["status"].cpu().numpy()
        assert np.array_equal(status[sl], osm["status"])
        frac = float((d <= 1e-10).mean())
        print("config %d step %d: N=%d, %d sampled stars; Phi/M not bit-identical: %d; r_new within 1e-10: %.6f%%, "
              "not bit-identical: %d, rejection flips: %d"
              % (index, step, n, d.size, nbit, 100 * frac, int((r_new[sl] != osm["r_new"]).sum()), flips))
        assert frac >= 0.99999 and flips <= max(1, d.size // 100_000)
        # ---- properties on every star
        rs = o["r"]
        assert np.all(rs[1:] >= rs[:-1])
        drawn = (status & ~np.uint8(hmc.ST_CLIPPED)) == 0
        assert drawn.mean() > 0.999
        assert np.all(r_new[drawn] >= tp["r_min"][drawn]) and np.all(r_new[drawn] <= tp["r_max"][drawn])
        assert rel((r_new * vt_new)[drawn], tp["J"][drawn]).max() <= 1e-15 * 4       # J = r v_t conserved
        # energy identity at the new radius in this step's potential (Eq. 16), Phi(r_new) by Eq. 6
        j = np.searchsorted(rs, r_new, side="right")                                 # shell number, 0..N
        j = np.clip(j, tp["k_min"].view(np.uint32), tp["k_max"].view(np.uint32)).astype(np.int64)
        jj = np.maximum(j, 1) - 1
        phi_new = np.where(j == 0, phi[0], phi[jj] - mc[jj] * (1.0 / r_new - 1.0 / rs[jj]))
        e_new = phi_new + 0.5 * (vr_new * vr_new + vt_new * vt_new)
        scale = np.abs(phi_new) + 0.5 * (vr_new * vr_new + vt_new * vt_new)
        assert (np.abs(e_new - tp["E"])[drawn] / scale[drawn]).max() <= 1e-13
    cnt = st.counters.cpu().numpy()
    print("counters:", dict(zip(hmc.COUNTER_NAMES, cnt.tolist())))
    assert cnt[:5].sum() == 0


def test_config3_headline_1e7_two_steps(oracle):
    """BASELINE.json configs[2]: N = 1e7 equal-mass, seed 3 (the bench workload), two chained steps."""
    run_fullsize(oracle, 2, steps=2)


def test_config4_salpeter_1e7(oracle):
    """BASELINE.json configs[3]: N = 1e7, Salpeter masses, seed 4."""
    run_fullsize(oracle, 3, steps=1)


def test_second_search_table_just_above_the_coarse_capacity(oracle):
    """N = 1.2e7 (recipe of configs[2]): the coarse table's spacing becomes 2048 nodes, so S3's second
    table (every 1024-th node, in L2) does one bisection step -- the smallest case of the large-N path."""
    run_fullsize(oracle, 2, steps=1, n_override=12_000_000)


def test_config5_1e8(oracle):
    """BASELINE.json configs[4]: N = 1e8 equal-mass, seed 5 (tables far beyond L2, coarse spacing 2^14)."""
    run_fullsize(oracle, 4, steps=1)
