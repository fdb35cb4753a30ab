"""The seeded generator: determinism, shapes, and the Plummer statistics the recipe promises."""
import math

import numpy as np
from scipy import stats

from paper_1206_5878_b200 import inputs


def test_deterministic_and_chunk_independent():
    a = inputs.plummer(50_000, 3)
    b = inputs.plummer(50_000, 3)
    for k in a:
        assert np.array_equal(a[k], b[k])
    c = inputs.plummer(50_000, 4)
    assert not np.array_equal(a["r"], c["r"])
    big = inputs.plummer(inputs.CHUNK + 1000, 3)            # first chunk identical for any n >= CHUNK
    big2 = inputs.plummer(inputs.CHUNK + 5, 3)
    assert np.array_equal(big["r"][:inputs.CHUNK], big2["r"][:inputs.CHUNK])


def test_plummer_statistics():
    n = 200_000
    c = inputs.plummer(n, 7)
    a = inputs.A_NBODY
    assert c["r"].dtype == np.float64 and c["id"].dtype == np.uint32
    assert np.all(c["r"] > 0) and c["r"].max() < inputs.R_CUT * a
    assert np.array_equal(c["id"], np.arange(n))
    assert abs(math.fsum(c["m"]) - 1) < 1e-12 and np.all(c["m"] == 1.0 / n)
    # cumulative mass of the Plummer sphere: M(<r) = (r/a)^3 / (1 + (r/a)^2)^(3/2), truncated at R_CUT
    norm = inputs.R_CUT ** 3 / (1 + inputs.R_CUT ** 2) ** 1.5
    cdf = lambda x: np.clip((x / a) ** 3 / (1 + (x / a) ** 2) ** 1.5 / norm, 0, 1)
    assert stats.kstest(c["r"], cdf).pvalue > 1e-3
    # speeds below the local escape speed; kinetic energy 1/4 of G M^2 / (virial radius = 1)
    v2 = c["v_r"] ** 2 + c["v_t"] ** 2
    assert np.all(v2 <= 2.0 / np.sqrt(c["r"] ** 2 + a * a) * (1 + 1e-12))
    assert abs(0.5 * np.sum(c["m"] * v2) - 0.25) < 0.003
    assert abs(np.mean(c["v_r"] ** 2) / (0.5 * np.mean(c["v_t"] ** 2)) - 1) < 0.02   # isotropy
    assert np.all(c["v_t"] >= 0)


def test_salpeter_masses():
    n = 200_000
    c = inputs.plummer(n, 8, "salpeter")
    m = c["m"]
    assert abs(math.fsum(m) - 1) < 1e-12
    assert 900 < m.max() / m.min() <= 1000.0001
    # dN/dm ~ m^-2.35 on [0.1, 100]: CDF in the unnormalised mass m * (sum of raw masses)
    raw = m / m.min() * 0.1                                   # smallest mass ~ 0.1 to within sampling
    lo, hi = 0.1 ** -1.35, 100.0 ** -1.35
    cdf = lambda x: np.clip((lo - x ** -1.35) / (lo - hi), 0, 1)
    assert stats.kstest(raw, cdf).pvalue > 1e-4
    # masses independent of position
    assert abs(stats.spearmanr(c["r"][:20000], m[:20000]).statistic) < 0.03


def test_config_table_matches_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cfgs = json.load(open(os.path.join(root, "BASELINE.json")))["configs"]
    assert len(cfgs) == len(inputs.CONFIGS) == 5
    for text, c in zip(cfgs, inputs.CONFIGS):
        assert "N=1e%d" % round(math.log10(c["n"])) in text
        assert "seed %d" % c["seed"] in text
        assert ("Salpeter" in text) == (c["masses"] == "salpeter")
