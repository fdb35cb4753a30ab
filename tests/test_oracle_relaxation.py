"""Pins for the oracle's relaxation timestep (Eq. 7; bins of 20, :194) and two-body relaxation on
neighbour pairs (R19, R20).  CPU only.  Nothing expected here comes from the CUDA path:
closed forms on hand-made inputs, exact scaling laws of Eq. 7, conservation theorems of an elastic encounter, and
the first two moments of the deflection over the random angles."""
import math

import numpy as np
import pytest

from paper_1206_5878_b200 import inputs


def sorted_cluster(n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    o = np.argsort(c["r"], kind="stable")
    return {k: v[o] for k, v in c.items() if isinstance(v, np.ndarray)}


# ----------------------------------------------------------------------------- Eq. 7
def test_timestep_hand_case(oracle):
    """20 unit masses in a sphere of unit number density, every pair with relative speed c along the radius:
    <v_rel> = c, <(M1+M2)^2> = 4, n = 1  =>  T = (theta/(pi/2)) (pi/32) c^3 / (4 ln(gamma N) G^2)."""
    n, cspeed, theta, G = 20, 0.75, 1.25, 2.0
    R = (20 / (4 * math.pi / 3)) ** (1 / 3)                    # 20 stars inside R: density one star per unit volume
    r = np.linspace(0.1, 1.0, n) * R
    vr = np.where(np.arange(n) % 2 == 0, 0.5 * cspeed, -0.5 * cspeed)
    tb, tmin = oracle.relaxation_timestep(r, vr, np.zeros(n), np.ones(n), gamma=0.1, theta_max=theta, G=G,
                                          ln_gamma_n=3.0)
    want = (theta / (math.pi / 2)) * (math.pi / 32) * cspeed ** 3 / (3.0 * G * G * 1.0 * 4.0)
    assert tb.shape == (1,) and tb[0] == pytest.approx(want, rel=1e-14) and tmin == tb[0]
    # the transverse velocities enter through their squares (rms over the unknown angle between them)
    vt = np.full(n, 0.3)
    tb2, _ = oracle.relaxation_timestep(r, vr, vt, np.ones(n), theta_max=theta, G=G, ln_gamma_n=3.0)
    assert tb2[0] == pytest.approx(want * ((cspeed ** 2 + 2 * 0.09) ** 1.5) / cspeed ** 3, rel=1e-14)
    # default Coulomb logarithm: ln(0.1 N)
    tb3, _ = oracle.relaxation_timestep(r, vr, np.zeros(n), np.ones(n), theta_max=theta, G=G)
    assert tb3[0] == pytest.approx(want * 3.0 / math.log(0.1 * n), rel=1e-14)


def test_timestep_scaling_laws_are_exact(oracle):
    """Eq. 7 under r -> 4 r (n -> n / 64), m -> 2 m, v -> 2 v, G -> 2 G, theta -> 2 theta: powers of two, so the
    results scale exactly (bit for bit): x 64, / 4, x 8, / 4, x 2."""
    c = sorted_cluster(4000, 51, "salpeter")
    r, vr, vt, m = c["r"], c["v_r"], c["v_t"], c["m"]
    lg = math.log(0.1 * 4000)
    tb, tmin = oracle.relaxation_timestep(r, vr, vt, m, ln_gamma_n=lg)
    assert np.all(np.isfinite(tb)) and np.all(tb > 0) and tmin == tb.min()
    assert np.array_equal(oracle.relaxation_timestep(4 * r, vr, vt, m, ln_gamma_n=lg)[0], 64 * tb)
    assert np.array_equal(oracle.relaxation_timestep(r, vr, vt, 2 * m, ln_gamma_n=lg)[0], tb / 4)
    assert np.array_equal(oracle.relaxation_timestep(r, 2 * vr, 2 * vt, m, ln_gamma_n=lg)[0], 8 * tb)
    assert np.array_equal(oracle.relaxation_timestep(r, vr, vt, m, G=2.0, ln_gamma_n=lg)[0], tb / 4)
    assert np.array_equal(oracle.relaxation_timestep(r, vr, vt, m, theta_max=2.0, ln_gamma_n=lg)[0], 2 * tb)
    assert np.array_equal(oracle.relaxation_timestep(4 * r, 2 * vr, 2 * vt, 2 * m, ln_gamma_n=lg)[0], 128 * tb)


def test_timestep_bins_and_density(oracle):
    """45 stars: bins [0, 20) and [20, 45) (the 5 left over join the last bin; its last star has no partner).
    A star's velocity moves only its own bin's T; the density of a bin is its star count over the volume of the
    shell that ends at its last star and begins at the previous bin's last star."""
    n = 45
    g = np.random.default_rng(1)
    r = np.sort(g.uniform(0.5, 2.0, n))
    vr, vt, m = g.normal(size=n), np.abs(g.normal(size=n)), g.uniform(0.5, 1.5, n)
    tb, tmin = oracle.relaxation_timestep(r, vr, vt, m, ln_gamma_n=1.0)
    assert tb.shape == (2,)
    for star, bins in ((3, [0]), (19, [0]), (20, [1]), (43, [1])):
        v2 = vr.copy(); v2[star] += 1.0
        t2, _ = oracle.relaxation_timestep(r, v2, vt, m, ln_gamma_n=1.0)
        assert [b for b in range(2) if t2[b] != tb[b]] == bins
    v2 = vr.copy(); v2[44] += 1.0                                # the odd star out is in no pair ...
    assert np.array_equal(oracle.relaxation_timestep(r, v2, vt, m, ln_gamma_n=1.0)[0], tb)
    r2 = r.copy(); r2[44] *= 2.0                                 # ... but it closes the last bin's shell
    t3, _ = oracle.relaxation_timestep(r2, vr, vt, m, ln_gamma_n=1.0)
    ratio = ((2 * r[44]) ** 3 - r[19] ** 3) / (r[44] ** 3 - r[19] ** 3)
    assert t3[0] == tb[0] and t3[1] == pytest.approx(tb[1] * ratio, rel=1e-13)
    # first bin: the shell starts at r = 0
    r4 = r.copy(); r4[:19] *= 0.5
    assert np.array_equal(oracle.relaxation_timestep(r4, vr, vt, m, ln_gamma_n=1.0)[0], tb)
    # fewer than 20 stars: one bin; 0 or 1 star: no pair, no constraint
    assert oracle.relaxation_timestep(r[:19], vr[:19], vt[:19], m[:19], ln_gamma_n=1.0)[0].shape == (1,)
    assert oracle.relaxation_timestep(r[:1], vr[:1], vt[:1], m[:1], ln_gamma_n=1.0)[1] == math.inf


def test_timestep_is_shortest_in_the_core(oracle):
    """Plummer model: the local relaxation time grows outwards by orders of magnitude, so the minimum of Eq. 7
    sits in the core, and it is a small fraction of the half-mass relaxation time of Eq. 20."""
    n = 100_000
    c = sorted_cluster(n, 52)
    tb, tmin = oracle.relaxation_timestep(c["r"], c["v_r"], c["v_t"], c["m"])
    inner, outer = np.median(tb[: len(tb) // 10]), np.median(tb[-len(tb) // 10:])
    assert outer > 100 * inner
    assert np.argmin(tb) < len(tb) // 5
    phi, mc = oracle.potential(c["r"], c["m"])
    t_rh = oracle.diagnostics(c["r"], c["v_r"], c["v_t"], c["m"], phi, mc)["t_rh"]
    assert 0.01 * t_rh < tmin < 0.5 * t_rh


# ----------------------------------------------------------------------------- representative encounter
def test_encounter_conserves_pair_energy_and_radial_momentum(oracle):
    n = 50_001                                                   # odd: the last star has no partner
    c = sorted_cluster(n, 53, "salpeter")
    r, vr, vt, m, ids = c["r"], c["v_r"], c["v_t"], c["m"], c["id"]
    _, tmin = oracle.relaxation_timestep(r, vr, vt, m)
    for dt in (tmin, 30 * tmin):
        a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, dt, seed=5, step=2)
        assert a[-1] == vr[-1] and b[-1] == vt[-1]
        e0 = (m * (vr ** 2 + vt ** 2))[:-1].reshape(-1, 2).sum(1)
        e1 = (m * (a ** 2 + b ** 2))[:-1].reshape(-1, 2).sum(1)
        assert np.max(np.abs(e1 / e0 - 1)) < 4e-15                # kinetic energy of every pair
        p0 = (m * vr)[:-1].reshape(-1, 2).sum(1)
        p1 = (m * a)[:-1].reshape(-1, 2).sum(1)
        scale = (m * np.sqrt(vr ** 2 + vt ** 2))[:-1].reshape(-1, 2).sum(1)
        assert np.max(np.abs(p1 - p0) / scale) < 4e-15            # radial momentum of every pair
        assert np.all(b >= 0)
        assert (np.abs(a - vr) > 1e-6).mean() > 0.95              # and something did happen
    # other seed, step or id: other angles
    a0, _ = oracle.two_body_relaxation(r, vr, vt, m, ids, tmin, seed=5, step=2)
    for kw in (dict(seed=6, step=2), dict(seed=5, step=3), dict(seed=5 + (1 << 32), step=2)):
        a1, _ = oracle.two_body_relaxation(r, vr, vt, m, ids, tmin, **kw)
        assert (a1 != a0).mean() > 0.99
    a2, _ = oracle.two_body_relaxation(r, vr, vt, m, ids + np.uint32(1), tmin, seed=5, step=2)
    assert (a2 != a0).mean() > 0.99


def test_encounter_limits(oracle):
    c = sorted_cluster(2000, 54)
    r, vr, vt, m, ids = c["r"], c["v_r"], c["v_t"], c["m"], c["id"]
    # dt = 0: no deflection
    a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, 0.0, seed=1, step=0)
    assert np.max(np.abs(a - vr)) < 1e-15 and np.max(np.abs(b - vt)) < 1e-15
    # dt huge: sin^2(beta/2) capped at 1, beta = pi, w' = -w: equal masses swap their velocities
    a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, 1e30, seed=1, step=0)
    sw = lambda x: x.reshape(-1, 2)[:, ::-1].reshape(-1)
    assert np.max(np.abs(a - sw(vr))) < 1e-15 and np.max(np.abs(b - sw(vt))) < 1e-15
    # a massless partner does not move the massive star
    m2 = m.copy(); m2[1::2] = 0.0
    a, b = oracle.two_body_relaxation(r, vr, vt, m2, ids, 1e30, seed=1, step=0)
    assert np.max(np.abs(a[0::2] - vr[0::2])) < 1e-15 and np.max(np.abs(b[0::2] - vt[0::2])) < 1e-15


def _replicas(k, m1, m2, v1, v2):
    """k identical pairs at unit number density: star j sits where the sphere inside it holds a volume of j."""
    n = 2 * k
    r = (np.arange(1, n + 1) / (4 * math.pi / 3)) ** (1 / 3)
    m = np.where(np.arange(n) % 2 == 0, m1, m2).astype(float)
    vr = np.where(np.arange(n) % 2 == 0, v1[0], v2[0]).astype(float)
    vt = np.where(np.arange(n) % 2 == 0, v1[1], v2[1]).astype(float)
    return r, vr, vt, m, np.arange(n, dtype=np.uint32)


def test_deflection_angle_and_azimuth_statistics(oracle):
    """Star 2 moves radially (no angle phi involved): w and V are fixed vectors, and over the uniform azimuth psi
       <|v1'|^2> = V^2 + f^2 w^2 + 2 f cos(beta) V.w,   var = 2 f^2 w^2 sin^2(beta) (V^2 - (V.w)^2 / w^2),
       <v_r1'>  = V_z + f cos(beta) w_z,                 f = m2 / M,
    with sin^2(beta / 2) = 2 pi G^2 M^2 n ln(gamma N) dt / w^3 (n = 1 here).  Pins the constant and the exponent of
    w in the deflection, the rotation about w, and the uniformity of psi."""
    k, m1, m2, G, lg = 200_000, 1.0, 3.0, 1.5, 2.0
    v1, v2 = (0.3, 0.8), (-0.5, 0.0)                                           # (v_r, v_t)
    r, vr, vt, m, ids = _replicas(k, m1, m2, v1, v2)
    w = np.array([v1[1], 0.0, v1[0] - v2[0]])
    M = m1 + m2
    V = np.array([m1 * v1[1] / M, 0.0, (m1 * v1[0] + m2 * v2[0]) / M])
    wn = np.linalg.norm(w)
    f = m2 / M
    for S in (0.02, 0.3, 0.5, 0.9):
        dt = S * wn ** 3 / (2 * math.pi * G * G * M * M * 1.0 * lg)
        a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, dt, seed=11, step=1, G=G, ln_gamma_n=lg)
        cb, sb2 = 1 - 2 * S, 4 * S * (1 - S)
        sq = (a ** 2 + b ** 2)[0::2]
        mean = V @ V + f * f * wn ** 2 + 2 * f * cb * (V @ w)
        var = 2 * f * f * wn ** 2 * sb2 * (V @ V - (V @ w) ** 2 / wn ** 2)
        assert abs(sq.mean() - mean) < 5 * math.sqrt(var / k) + 1e-12
        assert abs(sq.var() / var - 1) < 0.02
        zmean, zvar = V[2] + f * cb * w[2], 0.5 * f * f * wn ** 2 * sb2 * (1 - w[2] ** 2 / wn ** 2)
        assert abs(a[0::2].mean() - zmean) < 5 * math.sqrt(zvar / k) + 1e-12
        assert abs(a[0::2].var() / zvar - 1) < 0.02


def test_orientation_angle_statistics(oracle):
    """Head-on limit (beta = pi, w' = -w) with unequal masses: v1' = ((m1 - m2) v1 + 2 m2 v2) / M, so |v1'|^2 depends
    on v1.v2 = v_t1 v_t2 cos(phi) + v_r1 v_r2: its mean and variance over phi pin <cos> = 0 and <cos^2> = 1/2."""
    k, m1, m2 = 200_000, 1.0, 3.0
    v1, v2 = (0.3, 0.8), (-0.5, 0.6)
    r, vr, vt, m, ids = _replicas(k, m1, m2, v1, v2)
    a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, 1e30, seed=12, step=0)
    M = m1 + m2
    c1, c2 = (m1 - m2) / M, 2 * m2 / M
    s1, s2 = v1[0] ** 2 + v1[1] ** 2, v2[0] ** 2 + v2[1] ** 2
    mean = c1 * c1 * s1 + c2 * c2 * s2 + 2 * c1 * c2 * v1[0] * v2[0]
    var = (2 * c1 * c2 * v1[1] * v2[1]) ** 2 / 2
    sq = (a ** 2 + b ** 2)[0::2]
    assert abs(sq.mean() - mean) < 5 * math.sqrt(var / k)
    assert abs(sq.var() / var - 1) < 0.02
    # cos(phi) is symmetric about 0: the third central moment vanishes
    assert abs(((sq - mean) ** 3).mean()) < 0.05 * var ** 1.5


def test_relaxation_drives_energy_equipartition(oracle):
    """Physics check of the whole scheme: repeated encounters between a heavy and a light population at the same
    place exchange energy from the heavy to the light stars (dynamical friction / equipartition)."""
    k = 20_000
    g = np.random.default_rng(3)
    n = 2 * k
    r = (np.arange(1, n + 1) / (4 * math.pi / 3)) ** (1 / 3)
    m = np.where(np.arange(n) % 2 == 0, 4.0, 1.0)
    vr, vt = g.normal(0, 0.5, n), np.abs(g.normal(0, 0.7, n))       # same velocity distribution: heavies carry 4x the energy
    ids = np.arange(n, dtype=np.uint32)
    e_heavy0 = (m * (vr ** 2 + vt ** 2))[0::2].mean()
    e_light0 = (m * (vr ** 2 + vt ** 2))[1::2].mean()
    for step in range(5):
        _, tmin = oracle.relaxation_timestep(r, vr, vt, m, ln_gamma_n=3.0)
        vr, vt = oracle.two_body_relaxation(r, vr, vt, m, ids, 20 * tmin, seed=21, step=step, ln_gamma_n=3.0)
    e_heavy, e_light = (m * (vr ** 2 + vt ** 2))[0::2].mean(), (m * (vr ** 2 + vt ** 2))[1::2].mean()
    assert e_heavy < 0.97 * e_heavy0 and e_light > 1.05 * e_light0
    assert abs((e_heavy + e_light) / (e_heavy0 + e_light0) - 1) < 1e-12


def test_openmp_build_of_the_relaxation_is_bit_identical(oracle):
    c = sorted_cluster(30_001, 55, "salpeter")
    args = (c["r"], c["v_r"], c["v_t"], c["m"], c["id"], 25.0)
    a = oracle.two_body_relaxation(*args, seed=3, step=1)
    with oracle.use("omp"):
        b = oracle.two_body_relaxation(*args, seed=3, step=1)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_zero_length_step_with_a_zero_volume_bin_moves_nothing(oracle):
    """DESIGN.md R20a.  Twenty-one tied radii give bin 1 zero volume: its T_rel is 0, so the global step is 0, and a
    step of zero length must leave every velocity as it was -- also in the tied bin, where sin^2(beta/2) is
    infinity times zero.  Likewise an infinite step (what T_rel's minimum is when no bin holds a pair) moves nothing,
    while a finite positive step still turns the pairs of the infinitely dense bin head-on (equal masses swap)."""
    c = sorted_cluster(400, 42)
    r, vr, vt, m, ids = c["r"].copy(), c["v_r"], c["v_t"], c["m"], c["id"]
    r[19:40] = r[19]
    t_bin, t_min = oracle.relaxation_timestep(r, vr, vt, m)
    assert t_bin[1] == 0.0 and t_min == 0.0
    for dt in (t_min, math.inf):
        a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, dt, seed=1, step=0)
        assert np.max(np.abs(a - vr)) < 1e-15 and np.max(np.abs(b - vt)) < 1e-15, dt     # up to the rounding of V +- f w
    a, b = oracle.two_body_relaxation(r, vr, vt, m, ids, 1e-300, seed=1, step=0)
    sw = lambda x: x.reshape(-1, 2)[:, ::-1].reshape(-1)
    assert np.max(np.abs(a[20:40] - sw(vr)[20:40])) < 1e-15 and np.max(np.abs(b[20:40] - sw(vt)[20:40])) < 1e-15
    assert np.max(np.abs(a[40:] - vr[40:])) < 1e-12           # everywhere else 1e-300 is no step at all
