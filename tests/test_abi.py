"""The C-ABI library loads on a CPU-only box and exports every symbol include/hmc.h declares.
No compute calls here (no GPU); only calls that are pure host arithmetic."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libhmc():
    from paper_1206_5878_b200 import build
    return ctypes.CDLL(build.build())


def declared_functions():
    text = open(os.path.join(ROOT, "include", "hmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hmc_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_four_stage_calls():
    names = declared_functions()
    for f in ("hmc_sort_by_radius", "hmc_potential", "hmc_orbit_turning_points", "hmc_sample_new_radius",
              "hmc_workspace_bytes", "hmc_status_string", "hmc_step_host", "hmc_step_host_arena_bytes", "hmc_version"):
        assert f in names


def test_every_declared_symbol_is_exported(libhmc):
    for f in declared_functions():
        assert hasattr(libhmc, f), f


def test_host_only_entry_points(libhmc):
    libhmc.hmc_workspace_bytes.restype = ctypes.c_size_t
    libhmc.hmc_workspace_bytes.argtypes = [ctypes.c_uint64]
    libhmc.hmc_step_host_arena_bytes.restype = ctypes.c_size_t
    libhmc.hmc_step_host_arena_bytes.argtypes = [ctypes.c_uint64]
    libhmc.hmc_status_string.restype = ctypes.c_char_p
    w5, w7 = libhmc.hmc_workspace_bytes(10 ** 5), libhmc.hmc_workspace_bytes(10 ** 7)
    assert 0 < w5 < w7 and w5 % 256 == 0
    assert w7 < 160 * 10 ** 7                     # scratch stays below 160 B/star (64 of them the sort's star records)
    assert libhmc.hmc_step_host_arena_bytes(10 ** 5) > w5
    assert libhmc.hmc_status_string(0) == b"HMC_OK"
    for code in (-1, -2, -3, -4, -5):
        assert libhmc.hmc_status_string(code).startswith(b"HMC_ERR")
    assert libhmc.hmc_version() >= 100


def test_build_variants_and_launch_counter(libhmc):
    """The product build caps the rejection loop at 4096 trials; the test-only build (GPU tests of the
    exhaustion path) at 3.  The launch counter starts at zero and nothing here launches a kernel."""
    from paper_1206_5878_b200 import build
    libhmc.hmc_t_max.restype = ctypes.c_uint32
    libhmc.hmc_launch_count.restype = ctypes.c_uint64
    assert libhmc.hmc_t_max() == 4096
    assert libhmc.hmc_launch_count() == 0
    t3 = ctypes.CDLL(build.build(variant="tmax3"))
    t3.hmc_t_max.restype = ctypes.c_uint32
    assert t3.hmc_t_max() == 3
    for f in declared_functions():
        assert hasattr(t3, f), f
    pairs = ctypes.CDLL(build.build(variant="pairs"))       # test-only: S3's pair search at every N
    pairs.hmc_t_max.restype = ctypes.c_uint32
    assert pairs.hmc_t_max() == 4096
    for f in declared_functions():
        assert hasattr(pairs, f), f


def test_argument_errors_do_not_need_a_gpu(libhmc):
    # call-level validation happens before any CUDA call
    null = ctypes.c_void_p(0)
    rc = libhmc.hmc_potential(ctypes.c_uint64(10), ctypes.c_double(1.0), null, null, null, null, null,
                              ctypes.c_size_t(0), null)
    assert rc == -1                                                   # HMC_ERR_NULL
    rc = libhmc.hmc_potential(ctypes.c_uint64((1 << 30) + 1), ctypes.c_double(1.0), null, null, null, null, null,
                              ctypes.c_size_t(0), null)
    assert rc == -2                                                   # HMC_ERR_SIZE
    rc = libhmc.hmc_potential(ctypes.c_uint64(0), ctypes.c_double(1.0), null, null, null, null, null,
                              ctypes.c_size_t(0), null)
    assert rc == 0                                                    # n == 0 is a no-op
    buf = (ctypes.c_double * 64)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    odd = ctypes.c_void_p(p.value + 4)
    rc = libhmc.hmc_potential(ctypes.c_uint64(8), ctypes.c_double(1.0), odd, p, p, p, null, ctypes.c_size_t(0), null)
    assert rc == -4                                                   # HMC_ERR_ALIGN
    rc = libhmc.hmc_potential(ctypes.c_uint64(8), ctypes.c_double(1.0), p, p, p, p, null, ctypes.c_size_t(0), null)
    assert rc == -3                                                   # HMC_ERR_WORKSPACE


def test_binding_has_no_cpu_fallback():
    import torch
    from paper_1206_5878_b200 import hmc
    r = torch.ones(4, dtype=torch.float64)
    with pytest.raises(hmc.HmcError):
        hmc.hmc_potential(r, r)                   # host tensors are refused, not computed on the CPU
    src = open(os.path.join(ROOT, "paper_1206_5878_b200", "hmc.py")).read()
    assert "oracle" not in src.replace("no CPU", "")
