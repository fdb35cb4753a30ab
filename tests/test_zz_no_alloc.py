"""hmc_potential_static: the potential for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is off limits at the moment they need Phi: a plug-in inside a
host program that hands out all device memory itself, a callback that runs while the allocator's lock is held,
a loop that cannot afford the device-wide synchronisation an allocation implies.  They own their star arrays but
have no workspace to give hmc_potential.  hmc_potential_static (include/hmc.h) takes none: its scratch is a
fixed 544 KiB array inside libhmc.so, good for up to 2**24 stars.

What is checked here:
  * on the GPU, two calls in a row (a large one, then a smaller one that finds the first call's partial sums
    still in the array) each give what hmc_potential gives on the same inputs -- within the 1e-12 the potential
    tests use, and in fact the same bits, because the same kernels run in the same configuration;
  * without a GPU, that a size beyond the limit is refused with the status that names the limit.

This file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide another test.
It does not depend on anything the other tests leave behind and passes alone in a fresh process as well.
"""
import ctypes

import numpy as np
import pytest

TOL_PHI = 1e-12                 # tests/test_gpu_parity.py's tolerance for Phi and M
STATIC_MAX_N = 1 << 24
HMC_ERR_STATIC_LIMIT = -6


def test_size_beyond_the_static_limit_is_refused():
    """n = limit + 1 comes back as HMC_ERR_STATIC_LIMIT before any pointer is looked at or any CUDA call is made
    (so this runs on a box without a GPU); the status string says what the limit is."""
    from paper_1206_5878_b200 import build
    L = ctypes.CDLL(build.build())
    L.hmc_status_string.restype = ctypes.c_char_p
    null = ctypes.c_void_p(0)
    rc = L.hmc_potential_static(ctypes.c_uint64(STATIC_MAX_N + 1), ctypes.c_double(1.0), null, null, null, null, null)
    assert rc == HMC_ERR_STATIC_LIMIT
    text = L.hmc_status_string(rc)
    assert text.startswith(b"HMC_ERR_STATIC_LIMIT") and b"2^24" in text
    assert L.hmc_potential_static(ctypes.c_uint64(0), ctypes.c_double(1.0), null, null, null, null, null) == 0
    assert L.hmc_potential_static(ctypes.c_uint64(10), ctypes.c_double(1.0), null, null, null, null, null) == -1


@pytest.mark.gpu
def test_static_scratch_potential_equals_workspace_potential_twice_in_a_row():
    import torch
    from paper_1206_5878_b200 import hmc, inputs

    def case(n, seed, masses, G):
        c = inputs.plummer(n, seed, masses)
        o = np.argsort(c["r"], kind="stable")
        r = torch.from_numpy(np.ascontiguousarray(c["r"][o])).cuda()
        m = torch.from_numpy(np.ascontiguousarray(c["m"][o])).cuda()
        want_phi, want_mc = hmc.hmc_potential(r, m, G)            # the existing path, caller's workspace
        # the caller of the no-allocation call owns its outputs; poison them so stale values cannot pass
        phi = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        mc = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        return r, m, G, want_phi.cpu().numpy(), want_mc.cpu().numpy(), phi, mc

    # a large call (several hundred slices in every CTA's chunk, ragged tail), then a small one that uses only the
    # front of the array and finds the large call's totals behind it
    cases = [case(1_000_003, 11, "salpeter", 1.0), case(100_000, 12, "equal", 2.5)]
    torch.cuda.synchronize()
    for r, m, G, want_phi, want_mc, phi, mc in cases:             # back to back on one stream
        hmc.hmc_potential_static(r, m, G, phi=phi, m_cum=mc)
    torch.cuda.synchronize()
    for r, m, G, want_phi, want_mc, phi, mc in cases:
        got_phi, got_mc = phi.cpu().numpy(), mc.cpu().numpy()
        assert np.isfinite(got_phi).all() and np.isfinite(got_mc).all()
        assert (np.abs(got_phi - want_phi) <= TOL_PHI * np.abs(want_phi)).all()
        assert (np.abs(got_mc - want_mc) <= TOL_PHI * np.abs(want_mc)).all()
        assert np.array_equal(got_phi, want_phi) and np.array_equal(got_mc, want_mc)

    with pytest.raises(hmc.HmcError, match="at most"):
        hmc.hmc_potential_static(torch.empty(STATIC_MAX_N + 1, dtype=torch.float64, device="cuda"),
                                 torch.empty(STATIC_MAX_N + 1, dtype=torch.float64, device="cuda"))
