"""GPU-vs-oracle parity of the relaxation stage: Eq. 7 per bin of 20 stars and its minimum,
and the representative two-body encounter of every neighbour pair.  Both sides evaluate the same binary64 expressions
(+, -, *, /, sqrt; no FMA; no trigonometric functions), so the bar is bit for bit."""
import math

import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import hmc, inputs

pytestmark = pytest.mark.gpu


def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def sorted_cluster(n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    o = np.argsort(c["r"], kind="stable")
    return {k: v[o] for k, v in c.items() if isinstance(v, np.ndarray)}


@pytest.mark.parametrize("n,masses", [(1, "equal"), (2, "equal"), (19, "equal"), (20, "equal"), (45, "salpeter"),
                                      (100_000, "equal"), (1_000_003, "salpeter")])
def test_relaxation_timestep_matches_oracle(oracle, n, masses):
    c = sorted_cluster(n, 41, masses)
    o_bin, o_min = oracle.relaxation_timestep(c["r"], c["v_r"], c["v_t"], c["m"], gamma=0.1, theta_max=1.3, G=1.0)
    t_bin, t_min = hmc.hmc_relaxation_timestep(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), 0.1, 1.3, 1.0)
    assert np.array_equal(t_bin.cpu().numpy(), o_bin)
    assert float(t_min.cpu()[0]) == o_min
    # without the per-bin output
    lib_min = torch.empty(1, dtype=torch.float64, device="cuda")
    hmc.lib().hmc_relaxation_timestep  # (binding always passes t_rel_bin; NULL is exercised through ctypes below)
    import ctypes
    ws = hmc.alloc_workspace(n)
    d = [dev(c[k]) for k in ("r", "v_r", "v_t", "m")]
    rc = hmc.lib().hmc_relaxation_timestep(ctypes.c_uint64(n), ctypes.c_double(1.0), ctypes.c_double(0.1), ctypes.c_double(1.3),
                                           *[ctypes.c_void_p(t.data_ptr()) for t in d], ctypes.c_void_p(0),
                                           ctypes.c_void_p(lib_min.data_ptr()), ctypes.c_void_p(ws.data_ptr()),
                                           ctypes.c_size_t(ws.numel()), ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0 and float(lib_min.cpu()[0]) == o_min


def test_relaxation_timestep_with_tied_radii(oracle):
    """A bin whose shell has zero volume (its last star and the previous bin's last star at the same radius): the
    density is infinite and the bin's T is 0, on both sides."""
    c = sorted_cluster(400, 42)
    r = c["r"].copy()
    r[19:40] = r[19]
    o_bin, o_min = oracle.relaxation_timestep(r, c["v_r"], c["v_t"], c["m"])
    t_bin, t_min = hmc.hmc_relaxation_timestep(dev(r), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]))
    assert o_bin[1] == 0.0 and o_min == 0.0
    assert np.array_equal(t_bin.cpu().numpy(), o_bin) and float(t_min.cpu()[0]) == o_min


@pytest.mark.parametrize("n,masses", [(1, "equal"), (2, "equal"), (3, "equal"), (41, "salpeter"), (100_000, "equal"),
                                      (1_000_003, "salpeter")])
def test_two_body_relaxation_matches_oracle(oracle, n, masses):
    c = sorted_cluster(n, 43, masses)
    _, tmin = oracle.relaxation_timestep(c["r"], c["v_r"], c["v_t"], c["m"])
    d = [dev(c[k]) for k in ("r", "v_r", "v_t", "m")]
    ids = dev(c["id"])
    for dt in ((tmin if math.isfinite(tmin) else 1.0), 0.0, 1e30):
        o_vr, o_vt = oracle.two_body_relaxation(c["r"], c["v_r"], c["v_t"], c["m"], c["id"], dt, seed=9 + (3 << 32), step=4)
        vr, vt = hmc.hmc_two_body_relaxation(d[0], d[1], d[2], d[3], ids, dt, 9 + (3 << 32), 4)
        assert np.array_equal(vr.cpu().numpy(), o_vr), dt
        assert np.array_equal(vt.cpu().numpy(), o_vt), dt


def test_two_body_relaxation_degenerate_pairs(oracle):
    """Massless pairs, identical velocities (w = 0), purely radial relative motion (w along z), zero-volume bins."""
    n = 200
    c = sorted_cluster(n, 44)
    r, vr, vt, m = c["r"].copy(), c["v_r"].copy(), c["v_t"].copy(), c["m"].copy()
    m[0:2] = 0.0                                  # massless pair
    vr[2], vr[3], vt[2], vt[3] = 0.25, 0.25, 0.0, 0.0          # w = 0
    vt[4], vt[5] = 0.0, 0.0                       # w along z
    m[7] = 0.0                                    # massless partner
    r[59:80] = r[59]                              # bin 3 has zero volume: sin^2(beta/2) capped at 1
    o_vr, o_vt = oracle.two_body_relaxation(r, vr, vt, m, c["id"], 3.0, seed=1, step=0)
    g_vr, g_vt = hmc.hmc_two_body_relaxation(dev(r), dev(vr), dev(vt), dev(m), dev(c["id"]), 3.0, 1, 0)
    assert np.array_equal(g_vr.cpu().numpy(), o_vr) and np.array_equal(g_vt.cpu().numpy(), o_vt)
    assert o_vr[2] == 0.25 and o_vr[0] == vr[0]


def test_zero_length_step_with_a_zero_volume_bin(oracle):
    """DESIGN.md R20a on the device, driven the way OrbitStepper(relaxation=True) drives it: the step is T_rel's minimum,
    read from device memory; with a zero-volume bin that minimum is 0 and nothing may move.  Also dt = +inf."""
    c = sorted_cluster(400, 42)
    r = c["r"].copy()
    r[19:40] = r[19]
    d = [dev(x) for x in (r, c["v_r"], c["v_t"], c["m"])]
    _, t_min = hmc.hmc_relaxation_timestep(*d)
    assert float(t_min.cpu()[0]) == 0.0
    vr, vt = hmc.hmc_two_body_relaxation(d[0], d[1], d[2], d[3], dev(c["id"]), 1.0, 1, 0, dt_device=t_min)
    assert np.max(np.abs(vr.cpu().numpy() - c["v_r"])) < 1e-15 and np.max(np.abs(vt.cpu().numpy() - c["v_t"])) < 1e-15
    for dt in (0.0, math.inf, 1e-300):
        o_vr, o_vt = oracle.two_body_relaxation(r, c["v_r"], c["v_t"], c["m"], c["id"], dt, seed=1, step=0)
        vr, vt = hmc.hmc_two_body_relaxation(d[0], d[1], d[2], d[3], dev(c["id"]), dt, 1, 0)
        assert np.array_equal(vr.cpu().numpy(), o_vr) and np.array_equal(vt.cpu().numpy(), o_vt), dt


def test_relaxation_inside_the_step_loop(oracle):
    """Potential -> timestep -> relaxation -> new orbits -> sort, three times, GPU chain against oracle chain
    (the paper's order of steps 1-6)."""
    n, seed = 60_000, 45
    c = inputs.plummer(n, seed)
    st = hmc.OrbitStepper(dev(c["r"]), dev(c["v_r"]), dev(c["v_t"]), dev(c["m"]), dev(c["id"]), seed, relaxation=True)
    r, vr, vt, m, ids = c["r"], c["v_r"], c["v_t"], c["m"], c["id"]
    for step in range(3):
        st.step()
        rs, perm, (vrs, vts, ms), ids_s = oracle.sort_by_radius(r, (vr, vt, m), ids)
        phi, mc = oracle.potential(rs, ms)
        _, tmin = oracle.relaxation_timestep(rs, vrs, vts, ms)
        vrs, vts = oracle.two_body_relaxation(rs, vrs, vts, ms, ids_s, tmin, seed, step)
        tp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc)
        sm = oracle.sample_new_radius(rs, phi, mc, rs, vrs, vts, tp["E"], tp["J"], tp["r_min"], tp["r_max"], tp["k_min"],
                                      tp["k_max"], ids_s, tp["status"], seed, step)
        assert float(st.t_rel_min.cpu()[0]) == tmin
        assert np.array_equal(st.state["r"].cpu().numpy(), sm["r_new"])
        assert np.array_equal(st.state["v_r"].cpu().numpy(), sm["v_r_new"])
        assert np.array_equal(st.state["v_t"].cpu().numpy(), sm["v_t_new"])
        r, vr, vt, m, ids = sm["r_new"], sm["v_r_new"], sm["v_t_new"], ms, ids_s
