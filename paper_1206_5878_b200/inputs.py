"""Seeded synthetic inputs: Plummer-model star clusters (numpy only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic (no potential, no orbit, no Philox4x32 of the sampling stage):
it only draws initial conditions with numpy's own generator.

The paper's workloads are "clusters [with] N = 1e5, 1e6, 1e7 stars with positions and
velocities distributed according to a Plummer model", produced by
CMC's own initial-condition tool, which is not available.  The five configurations of
BASELINE.json stand in for them; recipe:

* radius, a = 1 units:  r~ = (X^(-2/3) - 1)^(-1/2),  X ~ U(0,1), redrawn until 0 < r~ < 300
* speed (Aarseth, Henon & Wielen 1974, von Neumann rejection):  q ~ U(0,1), y ~ 0.1 U(0,1)
  until y < q^2 (1 - q^2)^(7/2);  V = q sqrt(2) (1 + r~^2)^(-1/4)
* isotropic direction:  c = 1 - 2 U;  v_r = V c,  v_t = V sqrt(1 - c^2)
* N-body units (G = M = 1, E_tot = -1/4):  r = (3 pi / 16) r~,  v <- v / sqrt(3 pi / 16)
* masses: 1/N, or Salpeter dN/dm ~ m^-2.35 on [0.1, 100] drawn independently of position
  and rescaled to total mass 1
* id = i (persistent star id), stars are emitted UNSORTED (draw order)

Random numbers: numpy Generator over numpy's Philox bit generator, one independent
stream per chunk of 2^20 stars (key = (seed, chunk)), so the result depends only on
(n, seed, masses) and can be produced chunk by chunk.
"""
from __future__ import annotations

import math

import numpy as np

CHUNK = 1 << 20
R_CUT = 300.0                     # truncation radius in a = 1 units
A_NBODY = 3.0 * math.pi / 16.0    # Plummer scale length in N-body units

#: BASELINE.json "configs", in order.
CONFIGS = (
    dict(name="plummer_1e5", n=100_000, masses="equal", seed=1, steps=1),
    dict(name="plummer_1e6", n=1_000_000, masses="equal", seed=2, steps=11),
    dict(name="plummer_1e7", n=10_000_000, masses="equal", seed=3, steps=10),
    dict(name="plummer_1e7_salpeter", n=10_000_000, masses="salpeter", seed=4, steps=10),
    dict(name="plummer_1e8", n=100_000_000, masses="equal", seed=5, steps=5),
)


def _chunk(nc: int, seed: int, chunk: int, salpeter: bool):
    g = np.random.Generator(np.random.Philox(key=[seed, chunk]))
    # radii
    rt = np.empty(nc)
    todo = np.arange(nc)
    while todo.size:
        x = g.random(todo.size)
        with np.errstate(divide="ignore", invalid="ignore"):
            cand = (x ** (-2.0 / 3.0) - 1.0) ** -0.5
        ok = (x > 0.0) & (cand < R_CUT) & (cand > 0.0)
        rt[todo[ok]] = cand[ok]
        todo = todo[~ok]
    # speeds
    q = np.empty(nc)
    todo = np.arange(nc)
    while todo.size:
        qq = g.random(todo.size)
        y = 0.1 * g.random(todo.size)
        ok = y < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    v = q * math.sqrt(2.0) * (1.0 + rt * rt) ** -0.25
    c = 1.0 - 2.0 * g.random(nc)
    vr = v * c
    vt = v * np.sqrt(1.0 - c * c)
    if salpeter:
        lo, hi = 0.1 ** -1.35, 100.0 ** -1.35
        mt = (lo + g.random(nc) * (hi - lo)) ** (-1.0 / 1.35)
    else:
        mt = None
    return rt * A_NBODY, vr / math.sqrt(A_NBODY), vt / math.sqrt(A_NBODY), mt


def plummer(n: int, seed: int, masses: str = "equal"):
    """-> dict(r, v_r, v_t, m: float64[n]; id: uint32[n]), unsorted, N-body units."""
    if masses not in ("equal", "salpeter"):
        raise ValueError(masses)
    r = np.empty(n)
    vr = np.empty(n)
    vt = np.empty(n)
    m = np.empty(n)
    for ci, start in enumerate(range(0, n, CHUNK)):
        nc = min(CHUNK, n - start)
        a, b, c, mt = _chunk(nc, seed, ci, masses == "salpeter")
        r[start:start + nc] = a
        vr[start:start + nc] = b
        vt[start:start + nc] = c
        if mt is not None:
            m[start:start + nc] = mt
    if masses == "equal":
        m[:] = 1.0 / n
    else:
        m /= math.fsum(m)
    return dict(r=r, v_r=vr, v_t=vt, m=m, id=np.arange(n, dtype=np.uint32))


def config(index: int, n_override: int | None = None):
    """Inputs of BASELINE.json configs[index] (optionally at a reduced n, same recipe)."""
    c = dict(CONFIGS[index])
    if n_override is not None:
        c["n"] = int(n_override)
    c.update(plummer(c["n"], c["seed"], c["masses"]))
    return c
