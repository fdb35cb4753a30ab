"""CPU oracle for the Henon Monte Carlo orbit step (arXiv 1206.5878).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_1206_5878_b200/`` may import
this package; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs do.  The arithmetic lives in
``hmc_oracle.c`` (plain C, one translation unit, written from the paper); this
file only compiles it with gcc and marshals numpy arrays through ctypes.

Builds of the one source file (``use(name)`` selects which one the functions below call):
  serial  libhmc_oracle.so       the oracle as defined: single-threaded
  omp     libhmc_oracle_omp.so   -fopenmp over the per-star loops of S3 / S4 / energy correction and the
                                 gather; bit-identical results (tests check it)
  tmax3   libhmc_oracle_tmax3.so -DT_MAX=3u, test-only: reaches the exhaustion branch of S4 (the product's
                                 counterpart is libhmc_tmax3.so, built with -DHMC_T_MAX=3u)
"""
from __future__ import annotations

import contextlib
import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hmc_oracle.c")
# -ffp-contract=off: no FMA contraction; see the header of hmc_oracle.c.
CFLAGS = ["-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=gnu11", "-Wall", "-Wno-unknown-pragmas"]
VARIANTS = {
    "serial": ("libhmc_oracle.so", []),
    "omp": ("libhmc_oracle_omp.so", ["-fopenmp"]),
    "tmax3": ("libhmc_oracle_tmax3.so", ["-DT_MAX=3u"]),
    # AddressSanitizer + UndefinedBehaviorSanitizer build, selected for a whole test run with HMC_ORACLE_VARIANT=asan
    # and libasan preloaded into the interpreter (profiles/r2.md has the command and its result)
    "asan": ("libhmc_oracle_asan.so", ["-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-g"]),
}

ST_UNBOUND, ST_RADIAL, ST_DEGENERATE, ST_CIRCULAR, ST_MAXTRIES, ST_CLIPPED = 1, 2, 4, 8, 16, 32
T_MAX = 4096
C_F = 1.2

_libs = {}
_current = os.environ.get("HMC_ORACLE_VARIANT", "serial")


def build(force: bool = False, variant: str = "serial") -> str:
    """Compile hmc_oracle.c -> the variant's shared library (in-tree) if missing or stale."""
    name, extra = VARIANTS[variant]
    out = os.path.join(_HERE, name)
    stale = (not os.path.exists(out)) or os.path.getmtime(out) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = out + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", *CFLAGS, *extra, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, out)
    return out


def build_all(force: bool = False):
    return [build(force, v) for v in VARIANTS if v != "asan"]


def lib(variant: str | None = None) -> ctypes.CDLL:
    v = variant or _current
    if v not in _libs:
        L = ctypes.CDLL(build(variant=v))
        L.hmc_ref_t_max.restype = ctypes.c_uint32
        _libs[v] = L
    return _libs[v]


@contextlib.contextmanager
def use(variant: str):
    """``with oracle.use("omp"): ...`` -- the functions of this module call that build inside the block."""
    global _current
    prev, _current = _current, variant
    try:
        lib()
        yield
    finally:
        _current = prev


def t_max(variant: str | None = None) -> int:
    return int(lib(variant).hmc_ref_t_max())


def threads() -> int:
    """Threads the per-star loops of the current build use (1 for the builds without -fopenmp)."""
    if not lib().hmc_ref_openmp():
        return 1
    n = os.environ.get("OMP_NUM_THREADS")
    return int(n) if n else (len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count())


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().hmc_ref_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def sort_by_radius(r_in, cols=(), ids=None):
    """-> (r_sorted, perm, [cols_sorted...], ids_sorted or None)"""
    r_in = _f64(r_in)
    n = r_in.shape[0]
    r_sorted = np.empty(n, np.float64)
    perm = np.empty(n, np.uint32)
    cols = [_f64(c) for c in cols]
    outs = [np.empty(n, np.float64) for _ in cols]
    PtrArr = ctypes.c_void_p * max(len(cols), 1)
    cin = PtrArr(*[c.ctypes.data for c in cols]) if cols else PtrArr()
    cout = PtrArr(*[c.ctypes.data for c in outs]) if cols else PtrArr()
    id_out = None
    if ids is not None:
        ids = np.ascontiguousarray(ids, dtype=np.uint32)
        id_out = np.empty(n, np.uint32)
    rc = lib().hmc_ref_sort_by_radius(ctypes.c_uint64(n), _p(r_in), _p(r_sorted), _p(perm),
                                      ctypes.c_int(len(cols)), cin, cout, _p(ids), _p(id_out))
    assert rc == 0
    return r_sorted, perm, outs, id_out


def potential(r, m, G=1.0):
    """-> (phi, m_cum) on the radius-sorted arrays r, m."""
    r, m = _f64(r), _f64(m)
    n = r.shape[0]
    phi = np.empty(n, np.float64)
    mc = np.empty(n, np.float64)
    rc = lib().hmc_ref_potential(ctypes.c_uint64(n), ctypes.c_double(G), _p(r), _p(m), _p(phi), _p(mc))
    assert rc == 0
    return phi, mc


def orbit_turning_points(r, v_r, v_t, phi, m_cum, G=1.0, first=0, stride=1, count=None):
    """-> dict(E, J, r_min, r_max, k_min, k_max, status), compact over the selected stars."""
    r, v_r, v_t, phi, m_cum = map(_f64, (r, v_r, v_t, phi, m_cum))
    n = r.shape[0]
    if count is None:
        count = 0 if n <= first else (n - first + stride - 1) // stride
    o = dict(E=np.empty(count), J=np.empty(count), r_min=np.empty(count), r_max=np.empty(count),
             k_min=np.empty(count, np.uint32), k_max=np.empty(count, np.uint32),
             status=np.empty(count, np.uint8))
    rc = lib().hmc_ref_orbit_turning_points(
        ctypes.c_uint64(n), ctypes.c_double(G), _p(r), _p(v_r), _p(v_t), _p(phi), _p(m_cum),
        ctypes.c_uint64(first), ctypes.c_uint64(stride), ctypes.c_uint64(count),
        _p(o["E"]), _p(o["J"]), _p(o["r_min"]), _p(o["r_max"]), _p(o["k_min"]), _p(o["k_max"]),
        _p(o["status"]))
    assert rc == 0
    return o


def sample_new_radius(r, phi, m_cum, r_self, v_r_self, v_t_self, E, J, r_min, r_max, k_min, k_max,
                      ids, status, seed, step, G=1.0):
    """Tables r, phi, m_cum have length n; every other array is compact over the selected stars.
    -> dict(r_new, v_r_new, v_t_new, n_try, status, trials)"""
    r, phi, m_cum = map(_f64, (r, phi, m_cum))
    r_self, v_r_self, v_t_self, E, J, r_min, r_max = map(_f64, (r_self, v_r_self, v_t_self, E, J, r_min, r_max))
    k_min = np.ascontiguousarray(k_min, np.uint32)
    k_max = np.ascontiguousarray(k_max, np.uint32)
    ids = np.ascontiguousarray(ids, np.uint32)
    status = np.ascontiguousarray(status, np.uint8)
    n, count = r.shape[0], E.shape[0]
    o = dict(r_new=np.empty(count), v_r_new=np.empty(count), v_t_new=np.empty(count),
             n_try=np.empty(count, np.uint16), status=np.empty(count, np.uint8))
    counters = np.zeros(1, np.uint64)
    rc = lib().hmc_ref_sample_new_radius(
        ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_uint64(seed), ctypes.c_uint32(step),
        _p(r), _p(phi), _p(m_cum), ctypes.c_uint64(count),
        _p(r_self), _p(v_r_self), _p(v_t_self), _p(E), _p(J), _p(r_min), _p(r_max),
        _p(k_min), _p(k_max), _p(ids), _p(status),
        _p(o["r_new"]), _p(o["v_r_new"]), _p(o["v_t_new"]), _p(o["n_try"]), _p(o["status"]), _p(counters))
    assert rc == 0
    o["trials"] = int(counters[0])
    return o


DIAG_NAMES = ("M", "T", "W", "E_tot", "virial_ratio", "r_h", "t_rh")


def diagnostics(r, v_r, v_t, m, phi, m_cum, fractions=(), G=1.0):
    """Diagnostics on the radius-sorted arrays -> dict(M, T, W, E_tot, virial_ratio, r_h, t_rh, lagrange=[...])."""
    r, v_r, v_t, m, phi, m_cum = map(_f64, (r, v_r, v_t, m, phi, m_cum))
    fr = np.ascontiguousarray(np.asarray(fractions, dtype=np.float64))
    out = np.empty(7 + fr.shape[0], np.float64)
    rc = lib().hmc_ref_diagnostics(ctypes.c_uint64(r.shape[0]), ctypes.c_double(G), _p(r), _p(v_r), _p(v_t), _p(m),
                                   _p(phi), _p(m_cum), ctypes.c_int(fr.shape[0]), _p(fr), _p(out))
    assert rc == 0
    d = dict(zip(DIAG_NAMES, out[:7].tolist()))
    d["lagrange"] = out[7:].copy()
    return d


def energy_correction(r, phi, m_cum, E_old, r_old, p_old, v_r, v_t, G=1.0):
    """Energy correction for the time-varying potential, arrays in the NEW sorted order.
    -> (v_r', v_t', status)"""
    r, phi, m_cum, E_old, r_old, p_old, v_r, v_t = map(_f64, (r, phi, m_cum, E_old, r_old, p_old, v_r, v_t))
    n = r.shape[0]
    vro, vto, st = np.empty(n), np.empty(n), np.empty(n, np.uint8)
    rc = lib().hmc_ref_energy_correction(ctypes.c_uint64(n), ctypes.c_double(G), _p(r), _p(phi), _p(m_cum), _p(E_old),
                                         _p(r_old), _p(p_old), _p(v_r), _p(v_t), _p(vro), _p(vto), _p(st))
    assert rc == 0
    return vro, vto, st


BIN = 20


def n_bins(n):
    return (1 if n else 0) if n < BIN else n // BIN


def relaxation_timestep(r, v_r, v_t, m, gamma=0.1, theta_max=1.0, G=1.0, ln_gamma_n=None):
    """Eq. 7 per bin of 20 sorted stars and its minimum.  -> (t_rel_bin, t_rel_min)"""
    r, v_r, v_t, m = map(_f64, (r, v_r, v_t, m))
    n = r.shape[0]
    lg = math.log(gamma * n) if ln_gamma_n is None else float(ln_gamma_n)   # libm's log, as libhmc's host code
    tb = np.empty(n_bins(n), np.float64)
    tmin = np.empty(1, np.float64)
    rc = lib().hmc_ref_relaxation_timestep(ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_double(lg),
                                           ctypes.c_double(theta_max), _p(r), _p(v_r), _p(v_t), _p(m), _p(tb), _p(tmin))
    assert rc == 0
    return tb, float(tmin[0])


def two_body_relaxation(r, v_r, v_t, m, ids, dt, seed, step, gamma=0.1, G=1.0, ln_gamma_n=None):
    """Representative two-body encounter of every neighbour pair (R20).  -> (v_r', v_t')"""
    r, v_r, v_t, m = map(_f64, (r, v_r, v_t, m))
    ids = np.ascontiguousarray(ids, np.uint32)
    n = r.shape[0]
    lg = math.log(gamma * n) if ln_gamma_n is None else float(ln_gamma_n)   # libm's log, as libhmc's host code
    vro, vto = np.empty(n), np.empty(n)
    rc = lib().hmc_ref_two_body_relaxation(ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_double(lg), ctypes.c_double(dt),
                                           ctypes.c_uint64(seed), ctypes.c_uint32(step), _p(r), _p(v_r), _p(v_t), _p(m),
                                           _p(ids), _p(vro), _p(vto))
    assert rc == 0
    return vro, vto


def orbit_step(r, v_r, v_t, m, ids, seed, step, G=1.0, sample=None):
    """One pass of the whole path: sort -> potential -> turning points -> new radius.

    ``sample=(first, stride)`` restricts S3/S4 to every stride-th star of the sorted order
    (S1, S2 always run on all stars).  Returns a dict with every intermediate.
    """
    rs, perm, (vrs, vts, ms), ids_s = sort_by_radius(r, (v_r, v_t, m), ids)
    phi, mc = potential(rs, ms, G)
    first, stride = sample if sample is not None else (0, 1)
    tp = orbit_turning_points(rs, vrs, vts, phi, mc, G, first, stride)
    sl = slice(first, None, stride)
    sm = sample_new_radius(rs, phi, mc, rs[sl], vrs[sl], vts[sl], tp["E"], tp["J"], tp["r_min"], tp["r_max"],
                           tp["k_min"], tp["k_max"], ids_s[sl], tp["status"], seed, step, G)
    return dict(r=rs, perm=perm, v_r=vrs, v_t=vts, m=ms, id=ids_s, phi=phi, m_cum=mc, tp=tp, sample=sm)
