"""Thin binding over libhmc.so (C ABI declared in include/hmc.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of the library.
torch is used for device memory and the current stream, nothing else.  There is no CPU
fallback: if the library cannot be loaded, or a tensor is not a contiguous CUDA tensor of the
right dtype, the call raises.

The function names are those of the C ABI.  Outputs may be passed in (``out=...`` style keyword
arguments) to avoid allocation inside a timed loop; otherwise they are allocated with
``torch.empty`` on the inputs' device.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhmc.so")

ST_UNBOUND, ST_RADIAL, ST_DEGENERATE, ST_CIRCULAR, ST_MAXTRIES, ST_CLIPPED, ST_NOKINETIC = 1, 2, 4, 8, 16, 32, 64
COUNTER_NAMES = ("unbound", "radial", "degenerate", "circular", "maxtries", "clipped", "trials", "nokinetic")
NCOUNTERS = 8
MAX_N = 1 << 28
STATIC_MAX_N = 1 << 24          # HMC_STATIC_MAX_N: the most stars hmc_potential_static takes

_lib = None


class HmcError(RuntimeError):
    pass


def load(path: str) -> ctypes.CDLL:
    """Open a build of libhmc and declare its entry points.  Raises if absent (there is no CPU fallback)."""
    if not os.path.exists(path):
        raise HmcError("%s not found; run `python -m paper_1206_5878_b200.build` (there is no CPU fallback)" % path)
    L = ctypes.CDLL(path)
    L.hmc_workspace_bytes.restype = ctypes.c_size_t
    L.hmc_workspace_bytes.argtypes = [ctypes.c_uint64]
    L.hmc_step_host_arena_bytes.restype = ctypes.c_size_t
    L.hmc_step_host_arena_bytes.argtypes = [ctypes.c_uint64]
    L.hmc_status_string.restype = ctypes.c_char_p
    L.hmc_status_string.argtypes = [ctypes.c_int32]
    L.hmc_version.restype = ctypes.c_int32
    L.hmc_t_max.restype = ctypes.c_uint32
    L.hmc_launch_count.restype = ctypes.c_uint64
    for name in ("hmc_sort_by_radius", "hmc_potential", "hmc_orbit_turning_points", "hmc_sample_new_radius",
                 "hmc_orbit_step", "hmc_diagnostics", "hmc_energy_correction", "hmc_step_host", "hmc_potential_totals",
                 "hmc_potential_shard", "hmc_partition_points", "hmc_orbit_turning_points_range",
                 "hmc_sample_new_radius_range", "hmc_relaxation_timestep", "hmc_two_body_relaxation",
                 "hmc_sample_new_radius_dstep", "hmc_add_u32", "hmc_potential_shard_push", "hmc_orbit_build_tables",
                 "hmc_orbit_turning_points_prebuilt", "hmc_potential_static"):
        getattr(L, name).restype = ctypes.c_int32
    return L


def lib() -> ctypes.CDLL:
    """The library every binding call goes through: libhmc.so, loaded at first use."""
    global _lib
    if _lib is None:
        _lib = load(LIB_PATH)
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise HmcError("%s failed: %s" % (what, lib().hmc_status_string(rc).decode()))


def _dev(t: Optional[torch.Tensor], dtype, n: int, name: str):
    if t is None:
        return ctypes.c_void_p(0)
    if not t.is_cuda:
        raise HmcError("%s must be a CUDA tensor (no CPU path)" % name)
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != n:
        raise HmcError("%s must be contiguous %s[%d], got %s%s" % (name, dtype, n, t.dtype, tuple(t.shape)))
    return ctypes.c_void_p(t.data_ptr())


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def workspace_bytes(n: int) -> int:
    return int(lib().hmc_workspace_bytes(ctypes.c_uint64(n)))


def alloc_workspace(n: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(workspace_bytes(n), 256), dtype=torch.uint8, device=device)


def alloc_counters(device="cuda") -> torch.Tensor:
    return torch.zeros(NCOUNTERS, dtype=torch.int64, device=device)


def _ws(workspace, n, device):
    if workspace is None:
        workspace = alloc_workspace(n, device)
    return workspace, ctypes.c_void_p(workspace.data_ptr()), ctypes.c_size_t(workspace.numel())


def hmc_sort_by_radius(r_in: torch.Tensor, cols: Sequence[torch.Tensor] = (), ids: Optional[torch.Tensor] = None, *,
                       r_sorted=None, perm=None, cols_out=None, ids_out=None, workspace=None):
    """S1.  -> (r_sorted, perm, [cols_sorted...], ids_sorted or None)"""
    n = r_in.numel()
    dev = r_in.device
    r_sorted = torch.empty(n, dtype=torch.float64, device=dev) if r_sorted is None else r_sorted
    perm = torch.empty(n, dtype=torch.int32, device=dev) if perm is None else perm
    cols = list(cols)
    cols_out = [torch.empty(n, dtype=torch.float64, device=dev) for _ in cols] if cols_out is None else list(cols_out)
    if ids is not None and ids_out is None:
        ids_out = torch.empty(n, dtype=torch.int32, device=dev)
    nc = len(cols)
    Arr = ctypes.c_void_p * max(nc, 1)
    cin = Arr(*[_dev(c, torch.float64, n, "cols[%d]" % i).value or 0 for i, c in enumerate(cols)])
    cout = Arr(*[_dev(c, torch.float64, n, "cols_out[%d]" % i).value or 0 for i, c in enumerate(cols_out)])
    workspace, wp, wb = _ws(workspace, n, dev)
    rc = lib().hmc_sort_by_radius(ctypes.c_uint64(n), _dev(r_in, torch.float64, n, "r_in"),
                                  _dev(r_sorted, torch.float64, n, "r_sorted"), _dev(perm, torch.int32, n, "perm"),
                                  ctypes.c_int32(nc), cin, cout, _dev(ids, torch.int32, n, "ids"),
                                  _dev(ids_out, torch.int32, n, "ids_out"), wp, wb, _stream())
    _check(rc, "hmc_sort_by_radius")
    return r_sorted, perm, cols_out, ids_out


def hmc_potential(r_sorted: torch.Tensor, m_sorted: torch.Tensor, G: float = 1.0, *, phi=None, m_cum=None,
                  workspace=None):
    """S2.  -> (phi, m_cum)"""
    n = r_sorted.numel()
    dev = r_sorted.device
    phi = torch.empty(n, dtype=torch.float64, device=dev) if phi is None else phi
    m_cum = torch.empty(n, dtype=torch.float64, device=dev) if m_cum is None else m_cum
    workspace, wp, wb = _ws(workspace, n, dev)
    rc = lib().hmc_potential(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, torch.float64, n, "r_sorted"),
                             _dev(m_sorted, torch.float64, n, "m_sorted"), _dev(phi, torch.float64, n, "phi"),
                             _dev(m_cum, torch.float64, n, "m_cum"), wp, wb, _stream())
    _check(rc, "hmc_potential")
    return phi, m_cum


def hmc_potential_static(r_sorted: torch.Tensor, m_sorted: torch.Tensor, G: float = 1.0, *, phi=None, m_cum=None):
    """S2 without a workspace, for callers that cannot allocate device memory.  -> (phi, m_cum)

    Same result as hmc_potential, bit for bit.  The C call behind it allocates nothing: its scratch is a 544 KiB
    array built into libhmc.so, one per GPU.  Use it from code that must not call the CUDA allocator where it
    needs the potential: a plug-in inside a program that owns all device memory, a callback that runs under the
    allocator's lock, a loop that cannot take cudaMalloc's device synchronisation.  Pass ``phi`` and ``m_cum``
    (tensors you already own) if this Python layer must not allocate either; without them it makes them with
    torch.empty, which is a convenience of the binding, not of the library.

    Limits and rules (include/hmc.h): at most STATIC_MAX_N = 2**24 stars, more raises HmcError naming the limit;
    make the first call on each GPU outside stream capture (it looks up the array's address); all calls on a
    GPU share the one array, so calls that may run at the same time on different streams corrupt each other --
    keep them on one stream or order them with events."""
    n = r_sorted.numel()
    if n > STATIC_MAX_N:
        raise HmcError("hmc_potential_static takes at most %d stars (its scratch is a fixed array inside the library), "
                       "got %d; use hmc_potential with a workspace" % (STATIC_MAX_N, n))
    dev = r_sorted.device
    phi = torch.empty(n, dtype=torch.float64, device=dev) if phi is None else phi
    m_cum = torch.empty(n, dtype=torch.float64, device=dev) if m_cum is None else m_cum
    rc = lib().hmc_potential_static(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, torch.float64, n, "r_sorted"),
                                    _dev(m_sorted, torch.float64, n, "m_sorted"), _dev(phi, torch.float64, n, "phi"),
                                    _dev(m_cum, torch.float64, n, "m_cum"), _stream())
    _check(rc, "hmc_potential_static")
    return phi, m_cum


def hmc_orbit_build_tables(r_sorted, phi, m_cum, G: float = 1.0, *, workspace):
    """The search tables of S3 / S4 into the workspace (what hmc_orbit_turning_points starts with)."""
    n = r_sorted.numel()
    workspace, wp, wb = _ws(workspace, n, r_sorted.device)
    f = torch.float64
    _check(lib().hmc_orbit_build_tables(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"),
                                        _dev(phi, f, n, "phi"), _dev(m_cum, f, n, "m_cum"), wp, wb, _stream()),
           "hmc_orbit_build_tables")


def hmc_orbit_turning_points(r_sorted, v_r, v_t, phi, m_cum, G: float = 1.0, *, out=None, counters=None,
                             workspace=None, first: Optional[int] = None, prebuilt: bool = False):
    """S3.  -> dict(E, J, r_min, r_max, k_min, k_max, status)
    ``first`` given (sharded step): hmc_orbit_turning_points_range -- r_sorted, phi, m_cum are the table [n], v_r and
    v_t the stars at positions first .. first + len(v_r) - 1 of it; outputs have that length."""
    n = r_sorted.numel()
    c = n if first is None else v_r.numel()
    dev = r_sorted.device
    if out is None:
        out = alloc_turning_points(c, dev)
    workspace, wp, wb = _ws(workspace, n, dev)
    f = torch.float64
    head = (ctypes.c_uint64(n),) if first is None else (ctypes.c_uint64(n), ctypes.c_uint64(first), ctypes.c_uint64(c))
    fn = lib().hmc_orbit_turning_points if first is None else lib().hmc_orbit_turning_points_range
    if prebuilt:       # the workspace holds the tables of (r_sorted, phi, m_cum): hmc_orbit_build_tables was called
        head = (ctypes.c_uint64(n), ctypes.c_uint64(first or 0), ctypes.c_uint64(c))
        fn = lib().hmc_orbit_turning_points_prebuilt
    rc = fn(*head, ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"), _dev(v_r, f, c, "v_r"),
            _dev(v_t, f, c, "v_t"), _dev(phi, f, n, "phi"), _dev(m_cum, f, n, "m_cum"), _dev(out["E"], f, c, "E"),
            _dev(out["J"], f, c, "J"), _dev(out["r_min"], f, c, "r_min"), _dev(out["r_max"], f, c, "r_max"),
            _dev(out["k_min"], torch.int32, c, "k_min"), _dev(out["k_max"], torch.int32, c, "k_max"),
            _dev(out["status"], torch.uint8, c, "status"), _dev(counters, torch.int64, NCOUNTERS, "counters"), wp, wb,
            _stream())
    _check(rc, "hmc_orbit_turning_points")
    return out


def alloc_turning_points(n: int, device="cuda"):
    f = dict(dtype=torch.float64, device=device)
    i = dict(dtype=torch.int32, device=device)
    return dict(E=torch.empty(n, **f), J=torch.empty(n, **f), r_min=torch.empty(n, **f), r_max=torch.empty(n, **f),
                k_min=torch.empty(n, **i), k_max=torch.empty(n, **i),
                status=torch.empty(n, dtype=torch.uint8, device=device))


def alloc_sample(n: int, device="cuda", with_n_try: bool = True):
    f = dict(dtype=torch.float64, device=device)
    return dict(r_new=torch.empty(n, **f), v_r_new=torch.empty(n, **f), v_t_new=torch.empty(n, **f),
                n_try=torch.empty(n, dtype=torch.int16, device=device) if with_n_try else None,
                status=torch.empty(n, dtype=torch.uint8, device=device))


def hmc_sample_new_radius(r_sorted, phi, m_cum, v_r, v_t, tp, ids, seed: int, step: int, G: float = 1.0, *,
                          out=None, counters=None, workspace=None, reuse_tables: bool = False,
                          first: Optional[int] = None, step_dev: Optional[torch.Tensor] = None):
    """S4.  ``tp`` is the dict returned by hmc_orbit_turning_points.
    -> dict(r_new, v_r_new, v_t_new, n_try, status)
    ``first`` given (sharded step): hmc_sample_new_radius_range, per-star arrays of the range's length.
    ``step_dev`` given (int32[1] on the device): hmc_sample_new_radius_dstep, the step number is step + step_dev[0],
    read when the kernel runs (CUDA-graph replay)."""
    n = r_sorted.numel()
    c = n if first is None else v_r.numel()
    dev = r_sorted.device
    if out is None:
        out = alloc_sample(c, dev)
    workspace, wp, wb = _ws(workspace, n, dev)
    f = torch.float64
    head = (ctypes.c_uint64(n),) if first is None else (ctypes.c_uint64(n), ctypes.c_uint64(first), ctypes.c_uint64(c))
    fn = lib().hmc_sample_new_radius if first is None else lib().hmc_sample_new_radius_range
    stepargs = (ctypes.c_uint32(step),)
    if step_dev is not None:
        if first is not None:
            raise HmcError("step_dev and first cannot be combined")
        fn = lib().hmc_sample_new_radius_dstep
        stepargs = (ctypes.c_uint32(step), _dev(step_dev, torch.int32, 1, "step_dev"))
    rc = fn(*head, ctypes.c_double(G), ctypes.c_uint64(seed), *stepargs,
            _dev(r_sorted, f, n, "r_sorted"), _dev(phi, f, n, "phi"), _dev(m_cum, f, n, "m_cum"), _dev(v_r, f, c, "v_r"),
            _dev(v_t, f, c, "v_t"), _dev(tp["E"], f, c, "E"), _dev(tp["J"], f, c, "J"), _dev(tp["r_min"], f, c, "r_min"),
            _dev(tp["r_max"], f, c, "r_max"), _dev(tp["k_min"], torch.int32, c, "k_min"),
            _dev(tp["k_max"], torch.int32, c, "k_max"), _dev(ids, torch.int32, c, "ids"),
            _dev(tp["status"], torch.uint8, c, "status_in"), _dev(out["r_new"], f, c, "r_new"),
            _dev(out["v_r_new"], f, c, "v_r_new"), _dev(out["v_t_new"], f, c, "v_t_new"),
            _dev(out.get("n_try"), torch.int16, c, "n_try"), _dev(out["status"], torch.uint8, c, "status_out"),
            _dev(counters, torch.int64, NCOUNTERS, "counters"), ctypes.c_int32(1 if reuse_tables else 0), wp, wb,
            _stream())
    _check(rc, "hmc_sample_new_radius")
    return out


def hmc_add_u32(word: torch.Tensor, increment: int = 1):
    """word[0] += increment, enqueued on the current stream (the step counter of hmc_sample_new_radius_dstep)."""
    _check(lib().hmc_add_u32(_dev(word, torch.int32, 1, "word"), ctypes.c_uint32(increment), _stream()), "hmc_add_u32")


def hmc_potential_totals(r_sorted, m_sorted, *, totals=None, workspace=None):
    """Sharded step: a shard's (sum m, sum m/r) as two double-double pairs -> device float64[4]."""
    n = r_sorted.numel()
    dev = r_sorted.device
    totals = torch.empty(4, dtype=torch.float64, device=dev) if totals is None else totals
    workspace, wp, wb = _ws(workspace, n, dev)
    f = torch.float64
    rc = lib().hmc_potential_totals(ctypes.c_uint64(n), _dev(r_sorted, f, n, "r_sorted"), _dev(m_sorted, f, n, "m_sorted"),
                                    _dev(totals, f, 4, "totals"), wp, wb, _stream())
    _check(rc, "hmc_potential_totals")
    return totals


def hmc_potential_shard(r_sorted, m_sorted, rank: int, rank_totals, G: float = 1.0, *, phi=None, m_cum=None,
                        workspace=None, push=None):
    """Sharded step: S2 on shard ``rank``; rank_totals is the device float64[nranks, 4] of every shard's totals.
    ``push``: a list of (r, phi, m_cum) tensor triples of the shard's length -- views into the other ranks' copies of
    the replicated table at this shard's place; hmc_potential_shard_push stores the shard's slice there as it is
    produced (the table's all-gather fused into the scan)."""
    n = r_sorted.numel()
    dev = r_sorted.device
    nranks = rank_totals.numel() // 4
    f = torch.float64
    phi = torch.empty(n, dtype=f, device=dev) if phi is None else phi
    m_cum = torch.empty(n, dtype=f, device=dev) if m_cum is None else m_cum
    workspace, wp, wb = _ws(workspace, n, dev)
    if push:
        Arr = ctypes.c_void_p * len(push)
        pr = Arr(*[_dev(t[0], f, n, "push r").value or 0 for t in push])
        pp = Arr(*[_dev(t[1], f, n, "push phi").value or 0 for t in push])
        pc = Arr(*[_dev(t[2], f, n, "push m_cum").value or 0 for t in push])
        rc = lib().hmc_potential_shard_push(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"),
                                            _dev(m_sorted, f, n, "m_sorted"), ctypes.c_uint32(nranks), ctypes.c_uint32(rank),
                                            _dev(rank_totals, f, 4 * nranks, "rank_totals"), _dev(phi, f, n, "phi"),
                                            _dev(m_cum, f, n, "m_cum"), ctypes.c_int32(len(push)), pr, pp, pc, wp, wb, _stream())
        _check(rc, "hmc_potential_shard_push")
        return phi, m_cum
    rc = lib().hmc_potential_shard(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"),
                                   _dev(m_sorted, f, n, "m_sorted"), ctypes.c_uint32(nranks), ctypes.c_uint32(rank),
                                   _dev(rank_totals, f, 4 * nranks, "rank_totals"), _dev(phi, f, n, "phi"),
                                   _dev(m_cum, f, n, "m_cum"), wp, wb, _stream())
    _check(rc, "hmc_potential_shard")
    return phi, m_cum


def hmc_partition_points(r_sorted, splitters, *, counts=None):
    """Sample sort, phase 4: counts[j] = number of radii <= splitters[j] (device int64)."""
    n, k = r_sorted.numel(), splitters.numel()
    counts = torch.empty(k, dtype=torch.int64, device=r_sorted.device) if counts is None else counts
    f = torch.float64
    rc = lib().hmc_partition_points(ctypes.c_uint64(n), _dev(r_sorted, f, n, "r_sorted"), ctypes.c_uint32(k),
                                    _dev(splitters, f, k, "splitters"), _dev(counts, torch.int64, k, "counts"), _stream())
    _check(rc, "hmc_partition_points")
    return counts


def hmc_orbit_step(r_sorted, v_r, v_t, phi, m_cum, ids, seed: int, step: int, G: float = 1.0, *, tp=None, out=None,
                   counters=None, workspace=None):
    """S3 + S4 in one launch (same outputs as the two calls).  -> (tp dict, sample dict)"""
    n = r_sorted.numel()
    dev = r_sorted.device
    tp = alloc_turning_points(n, dev) if tp is None else tp
    out = alloc_sample(n, dev) if out is None else out
    workspace, wp, wb = _ws(workspace, n, dev)
    f = torch.float64
    rc = lib().hmc_orbit_step(
        ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_uint64(seed), ctypes.c_uint32(step),
        _dev(r_sorted, f, n, "r_sorted"), _dev(v_r, f, n, "v_r"), _dev(v_t, f, n, "v_t"), _dev(phi, f, n, "phi"),
        _dev(m_cum, f, n, "m_cum"), _dev(ids, torch.int32, n, "ids"), _dev(tp["E"], f, n, "E"), _dev(tp["J"], f, n, "J"),
        _dev(tp["r_min"], f, n, "r_min"), _dev(tp["r_max"], f, n, "r_max"), _dev(tp["k_min"], torch.int32, n, "k_min"),
        _dev(tp["k_max"], torch.int32, n, "k_max"), _dev(tp["status"], torch.uint8, n, "status"),
        _dev(out["r_new"], f, n, "r_new"), _dev(out["v_r_new"], f, n, "v_r_new"), _dev(out["v_t_new"], f, n, "v_t_new"),
        _dev(out.get("n_try"), torch.int16, n, "n_try"), _dev(out["status"], torch.uint8, n, "status_out"),
        _dev(counters, torch.int64, NCOUNTERS, "counters"), wp, wb, _stream())
    _check(rc, "hmc_orbit_step")
    return tp, out


def hmc_energy_correction(r_sorted, phi, m_cum, E_old, r_old, phi_old, v_r, v_t, G: float = 1.0, *, v_r_out=None,
                          v_t_out=None, status=None, counters=None, workspace=None):
    """Energy correction for the time-varying potential, arrays in the new sorted order.
    -> (v_r', v_t', status)"""
    n = r_sorted.numel()
    dev = r_sorted.device
    f = torch.float64
    v_r_out = torch.empty(n, dtype=f, device=dev) if v_r_out is None else v_r_out
    v_t_out = torch.empty(n, dtype=f, device=dev) if v_t_out is None else v_t_out
    status = torch.empty(n, dtype=torch.uint8, device=dev) if status is None else status
    workspace, wp, wb = _ws(workspace, n, dev)
    rc = lib().hmc_energy_correction(
        ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"), _dev(phi, f, n, "phi"),
        _dev(m_cum, f, n, "m_cum"), _dev(E_old, f, n, "E_old"), _dev(r_old, f, n, "r_old"), _dev(phi_old, f, n, "phi_old"),
        _dev(v_r, f, n, "v_r"), _dev(v_t, f, n, "v_t"), _dev(v_r_out, f, n, "v_r_out"), _dev(v_t_out, f, n, "v_t_out"),
        _dev(status, torch.uint8, n, "status"), _dev(counters, torch.int64, NCOUNTERS, "counters"), wp, wb, _stream())
    _check(rc, "hmc_energy_correction")
    return v_r_out, v_t_out, status


DIAG_NAMES = ("M", "T", "W", "E_tot", "virial_ratio", "r_h", "t_rh")
DIAG_MAX_FRACTIONS = 16


def hmc_diagnostics(r_sorted, v_r, v_t, m_sorted, phi, m_cum, fractions: Sequence[float] = (), G: float = 1.0, *,
                    out=None, workspace=None):
    """Diagnostics (Eq. 20).  -> device float64 tensor [7 + len(fractions)]:
    M, T, W, E_tot, virial ratio, r_h, t_rh, then the Lagrange radii of ``fractions`` (host floats)."""
    n = r_sorted.numel()
    dev = r_sorted.device
    nf = len(fractions)
    out = torch.empty(7 + nf, dtype=torch.float64, device=dev) if out is None else out
    fr = (ctypes.c_double * max(nf, 1))(*[float(x) for x in fractions])
    workspace, wp, wb = _ws(workspace, n, dev)
    f = torch.float64
    rc = lib().hmc_diagnostics(ctypes.c_uint64(n), ctypes.c_double(G), _dev(r_sorted, f, n, "r_sorted"),
                               _dev(v_r, f, n, "v_r"), _dev(v_t, f, n, "v_t"), _dev(m_sorted, f, n, "m_sorted"),
                               _dev(phi, f, n, "phi"), _dev(m_cum, f, n, "m_cum"), ctypes.c_int32(nf), fr,
                               _dev(out, f, 7 + nf, "out"), wp, wb, _stream())
    _check(rc, "hmc_diagnostics")
    return out


BIN = 20


def hmc_relaxation_timestep(r_sorted, v_r, v_t, m_sorted, gamma: float = 0.1, theta_max: float = 1.0, G: float = 1.0, *,
                            t_rel_bin=None, t_rel_min=None, workspace=None):
    """Eq. 7 per bin of 20 sorted stars and its minimum.
    -> (t_rel_bin: device float64[max(1, n // 20)], t_rel_min: device float64[1])"""
    n = r_sorted.numel()
    dev = r_sorted.device
    f = torch.float64
    nb = (1 if n else 0) if n < BIN else n // BIN
    t_rel_bin = torch.empty(nb, dtype=f, device=dev) if t_rel_bin is None else t_rel_bin
    t_rel_min = torch.empty(1, dtype=f, device=dev) if t_rel_min is None else t_rel_min
    workspace, wp, wb = _ws(workspace, n, dev)
    rc = lib().hmc_relaxation_timestep(ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_double(gamma),
                                       ctypes.c_double(theta_max), _dev(r_sorted, f, n, "r_sorted"), _dev(v_r, f, n, "v_r"),
                                       _dev(v_t, f, n, "v_t"), _dev(m_sorted, f, n, "m_sorted"),
                                       _dev(t_rel_bin, f, nb, "t_rel_bin"), _dev(t_rel_min, f, 1, "t_rel_min"), wp, wb, _stream())
    _check(rc, "hmc_relaxation_timestep")
    return t_rel_bin, t_rel_min


def hmc_two_body_relaxation(r_sorted, v_r, v_t, m_sorted, ids, dt: float, seed: int, step: int, gamma: float = 0.1,
                            G: float = 1.0, *, v_r_out=None, v_t_out=None, dt_device=None):
    """Representative two-body encounter of every neighbour pair.  -> (v_r', v_t')
    dt_device (device float64[1]) given: the step is dt * dt_device[0], read on the device."""
    n = r_sorted.numel()
    dev = r_sorted.device
    f = torch.float64
    v_r_out = torch.empty(n, dtype=f, device=dev) if v_r_out is None else v_r_out
    v_t_out = torch.empty(n, dtype=f, device=dev) if v_t_out is None else v_t_out
    rc = lib().hmc_two_body_relaxation(ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_double(gamma), ctypes.c_double(dt),
                                       _dev(dt_device, f, 1, "dt_device"), ctypes.c_uint64(seed), ctypes.c_uint32(step),
                                       _dev(r_sorted, f, n, "r_sorted"),
                                       _dev(v_r, f, n, "v_r"), _dev(v_t, f, n, "v_t"), _dev(m_sorted, f, n, "m_sorted"),
                                       _dev(ids, torch.int32, n, "ids"), _dev(v_r_out, f, n, "v_r_out"),
                                       _dev(v_t_out, f, n, "v_t_out"), _stream())
    _check(rc, "hmc_two_body_relaxation")
    return v_r_out, v_t_out


def launch_count() -> int:
    """Kernels this process has launched through libhmc so far (hmc_launch_count)."""
    return int(lib().hmc_launch_count())


class OrbitStepper:
    """Pre-allocated device state for repeated orbit steps (sort -> potential -> turning points ->
    new radius), the loop of BASELINE.json's multi-step configs.  Holds the carried state
    (r, v_r, v_t, m, id) and every intermediate; ``step()`` makes the four C-ABI calls on the
    current stream and swaps (r, v_r, v_t) <- (r_new, v_r', v_t'); m and id follow the sort."""

    def __init__(self, r, v_r, v_t, m, ids, seed: int, G: float = 1.0, with_n_try: bool = True,
                 energy_correction: bool = False, relaxation: bool = False, gamma: float = 0.1, theta_max: float = 1.0):
        """energy_correction=True: from the second step on, hmc_energy_correction adjusts the velocities
        between the potential and the turning points; three more columns (the star's energy,
        previous radius and the previous potential there) then travel through the sort."""
        self.n = n = r.numel()
        dev = r.device
        self.G, self.seed, self.step_index = G, seed, 0
        self.energy_correction = energy_correction
        # relaxation=True: between the potential and the turning points, the relaxation timestep of Eq. 7 and one
        # representative encounter per neighbour pair over that timestep, all on the device
        self.relaxation, self.gamma, self.theta_max = relaxation, gamma, theta_max
        if relaxation:
            self.t_rel_bin = torch.empty(max(1, n // BIN), dtype=torch.float64, device=r.device)
            self.t_rel_min = torch.empty(1, dtype=torch.float64, device=r.device)
            self.relaxed = dict(v_r=torch.empty(n, dtype=torch.float64, device=r.device),
                                v_t=torch.empty(n, dtype=torch.float64, device=r.device))
        self.state = dict(r=r.clone(), v_r=v_r.clone(), v_t=v_t.clone(), m=m.clone(), id=ids.clone())
        f = dict(dtype=torch.float64, device=dev)
        self.sorted = dict(r=torch.empty(n, **f), v_r=torch.empty(n, **f), v_t=torch.empty(n, **f),
                           m=torch.empty(n, **f), id=torch.empty(n, dtype=torch.int32, device=dev),
                           perm=torch.empty(n, dtype=torch.int32, device=dev))
        self.phi = torch.empty(n, **f)
        self.m_cum = torch.empty(n, **f)
        self.tp = alloc_turning_points(n, dev)
        self.sample = alloc_sample(n, dev, with_n_try)
        self.counters = alloc_counters(dev)
        self.workspace = alloc_workspace(n, dev)
        if energy_correction:
            for k in ("E", "r_old", "p_old"):
                self.state[k] = torch.zeros(n, **f)
                self.sorted[k] = torch.empty(n, **f)
            self.corrected = dict(v_r=torch.empty(n, **f), v_t=torch.empty(n, **f),
                                  status=torch.empty(n, dtype=torch.uint8, device=dev))
        self._graph = None
        self._step_dev = None

    def run_graph(self, steps: int):
        """``steps`` orbit steps (an even number), replayed from a CUDA graph of TWO steps captured at the first
        call (the carried arrays alternate between two sets of buffers with period two).  What changes from step to
        step, the Philox step number, is kept on the device: hmc_sample_new_radius_dstep reads it, hmc_add_u32
        advances it inside the graph.  For small N, where a step is bound by launching its 13 kernels one
        by one rather than by the GPU.  With or without the energy correction; not with the relaxation stage (its
        Philox step number is a host argument)."""
        if self.relaxation:
            raise HmcError("run_graph does not support the relaxation stage")
        if steps % 2:
            raise HmcError("run_graph takes an even number of steps (the buffers alternate with period two)")
        if self._graph is None:
            if self.step_index == 0:                 # first launches set function attributes: not inside a capture
                self.step()
                self.step()
                steps -= 2
            self._step_dev = torch.full((1,), self.step_index, dtype=torch.int32, device=self.state["r"].device)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                self._step_body(False, self._step_dev)
                self._step_body(False, self._step_dev)
            self._graph = g
            self._graph_parity = self.step_index % 2          # which of the two buffer arrangements the graph starts from
            self.step_index -= 2                     # the capture ran nothing
        else:
            if self.step_index % 2 != self._graph_parity:
                raise HmcError("run_graph: the graph starts from the buffer arrangement it was captured in; take an "
                               "even number of eager steps between replays")
            self._step_dev.fill_(self.step_index)    # eager steps may have been taken in between
        for _ in range(steps // 2):
            self._graph.replay()
            self.step_index += 2

    def step(self, fused: bool = False):
        """One orbit step.  fused=False: the four C-ABI calls; fused=True: S3 and S4 as the single
        call hmc_orbit_step (same results)."""
        self._step_body(fused, None)

    def _step_body(self, fused: bool, step_dev):
        s, so = self.state, self.sorted
        correct = self.energy_correction and self.step_index > 0
        if correct:
            # What the correction needs from the previous step -- each star's E in that potential (S3's output), its
            # radius then and the potential there -- becomes three record columns of this step's sort by exchanging
            # buffers, not by copying: the previous outputs are read as columns, and the previous columns' buffers
            # receive this step's E, sorted radii and potential.  (Until the next step begins, tp["E"], sorted["r"]
            # and phi still hold this step's values.)  The arrangement repeats with period two, like the state's.
            s["E"], self.tp["E"] = self.tp["E"], s["E"]
            s["r_old"], so["r"] = so["r"], s["r_old"]
            s["p_old"], self.phi = self.phi, s["p_old"]
        extra = ("E", "r_old", "p_old") if correct else ()
        hmc_sort_by_radius(s["r"], (s["v_r"], s["v_t"], s["m"]) + tuple(s[k] for k in extra), s["id"], r_sorted=so["r"],
                           perm=so["perm"], cols_out=(so["v_r"], so["v_t"], so["m"]) + tuple(so[k] for k in extra),
                           ids_out=so["id"], workspace=self.workspace)
        hmc_potential(so["r"], so["m"], self.G, phi=self.phi, m_cum=self.m_cum, workspace=self.workspace)
        if correct:
            co = self.corrected
            hmc_energy_correction(so["r"], self.phi, self.m_cum, so["E"], so["r_old"], so["p_old"], so["v_r"], so["v_t"],
                                  self.G, v_r_out=co["v_r"], v_t_out=co["v_t"], status=co["status"],
                                  counters=self.counters, workspace=self.workspace)
            so["v_r"], co["v_r"] = co["v_r"], so["v_r"]
            so["v_t"], co["v_t"] = co["v_t"], so["v_t"]
        if self.relaxation:
            rx = self.relaxed
            hmc_relaxation_timestep(so["r"], so["v_r"], so["v_t"], so["m"], self.gamma, self.theta_max, self.G,
                                    t_rel_bin=self.t_rel_bin[: (1 if self.n < BIN else self.n // BIN)], t_rel_min=self.t_rel_min,
                                    workspace=self.workspace)
            hmc_two_body_relaxation(so["r"], so["v_r"], so["v_t"], so["m"], so["id"], 1.0, self.seed, self.step_index,
                                    self.gamma, self.G, v_r_out=rx["v_r"], v_t_out=rx["v_t"], dt_device=self.t_rel_min)
            so["v_r"], rx["v_r"] = rx["v_r"], so["v_r"]
            so["v_t"], rx["v_t"] = rx["v_t"], so["v_t"]
        if fused:
            hmc_orbit_step(so["r"], so["v_r"], so["v_t"], self.phi, self.m_cum, so["id"], self.seed, self.step_index,
                           self.G, tp=self.tp, out=self.sample, counters=self.counters, workspace=self.workspace)
        else:
            hmc_orbit_turning_points(so["r"], so["v_r"], so["v_t"], self.phi, self.m_cum, self.G, out=self.tp,
                                     counters=self.counters, workspace=self.workspace)
            hmc_sample_new_radius(so["r"], self.phi, self.m_cum, so["v_r"], so["v_t"], self.tp, so["id"], self.seed,
                                  0 if step_dev is not None else self.step_index, self.G, out=self.sample,
                                  counters=self.counters, workspace=self.workspace, reuse_tables=True, step_dev=step_dev)
            if step_dev is not None:
                hmc_add_u32(step_dev, 1)
        # carried state for the next step: new phase-space coordinates, masses and ids in sorted order
        sm = self.sample
        s["r"], sm["r_new"] = sm["r_new"], s["r"]
        s["v_r"], sm["v_r_new"] = sm["v_r_new"], s["v_r"]
        s["v_t"], sm["v_t_new"] = sm["v_t_new"], s["v_t"]
        s["m"], so["m"] = so["m"], s["m"]
        s["id"], so["id"] = so["id"], s["id"]
        self.step_index += 1

    def diagnostics(self, fractions=()):
        """hmc_diagnostics of the cluster as the last step's S1/S2 saw it: the sorted radii and velocities the
        step started from, that step's potential (after step() the sorted masses are in state["m"])."""
        so = self.sorted
        return hmc_diagnostics(so["r"], so["v_r"], so["v_t"], self.state["m"], self.phi, self.m_cum, fractions,
                               self.G, workspace=self.workspace)


def step_host_arena_bytes(n: int) -> int:
    return int(lib().hmc_step_host_arena_bytes(ctypes.c_uint64(n)))


def hmc_step_host(r, v_r, v_t, m, ids, out, seed: int, step: int, G: float = 1.0, *, arena: torch.Tensor,
                  counters_host: Optional[torch.Tensor] = None):
    """Host-buffer variant of one whole step.  r, v_r, v_t, m (float64) and ids (int32) are HOST
    tensors (pinned for asynchronous copies); ``out`` is a dict of HOST tensors r_new, v_r_new,
    v_t_new, m, id; ``arena`` a CUDA uint8 tensor of step_host_arena_bytes(n).  Enqueues the copies
    and kernels on the current stream; synchronise before reading ``out``."""
    n = r.numel()

    def host(t, dtype, name):
        if t.is_cuda or t.dtype != dtype or not t.is_contiguous() or t.numel() != n:
            raise HmcError("%s must be a contiguous host %s[%d]" % (name, dtype, n))
        return ctypes.c_void_p(t.data_ptr())

    f = torch.float64
    cp = ctypes.c_void_p(0)
    if counters_host is not None:
        if counters_host.is_cuda or counters_host.dtype != torch.int64 or counters_host.numel() != NCOUNTERS:
            raise HmcError("counters_host must be a host int64[%d]" % NCOUNTERS)
        cp = ctypes.c_void_p(counters_host.data_ptr())
    if not arena.is_cuda or arena.dtype != torch.uint8:
        raise HmcError("arena must be a CUDA uint8 tensor")
    rc = lib().hmc_step_host(
        ctypes.c_uint64(n), ctypes.c_double(G), ctypes.c_uint64(seed), ctypes.c_uint32(step), host(r, f, "r"),
        host(v_r, f, "v_r"), host(v_t, f, "v_t"), host(m, f, "m"), host(ids, torch.int32, "ids"),
        host(out["r_new"], f, "r_new"), host(out["v_r_new"], f, "v_r_new"), host(out["v_t_new"], f, "v_t_new"),
        host(out["m"], f, "m_out"), host(out["id"], torch.int32, "id_out"), cp, ctypes.c_void_p(arena.data_ptr()),
        ctypes.c_size_t(arena.numel()), _stream())
    _check(rc, "hmc_step_host")
    return out
