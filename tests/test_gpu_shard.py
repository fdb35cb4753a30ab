"""The sharded step (paper_1206_5878_b200/shard.py) on one GPU: G shards held by one process
(shard.InProcessComm, device copies for collectives) must reproduce the single-GPU hmc.OrbitStepper BIT FOR BIT --
the sort is stable across the exchange, M_k and S_k are exact sums rounded once whatever the association, and the
random numbers are keyed by the persistent star id.  The single-GPU stepper is itself compared with the oracle in
tests/test_gpu_fullsize.py, and the pieces the sharded step adds are compared with the oracle here."""
import os
import warnings

import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import hmc, inputs, shard

pytestmark = pytest.mark.gpu


def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if t.dtype == torch.uint32:
        t = t.view(torch.int32)
    return t.cuda()


def device_cluster(n, seed, masses="equal"):
    c = inputs.plummer(n, seed, masses)
    return {k: dev(c[k]) for k in ("r", "v_r", "v_t", "m", "id")}, c


@pytest.mark.parametrize("push", [True, False])
@pytest.mark.parametrize("world", [2, 4, 8])
def test_sharded_step_equals_single_gpu_step(world, push):
    """N = 1e6, three chained steps: after every step the shards, put end to end, ARE the single-GPU state.
    push=True: every rank's potential scan stores its slice of (r, Phi, M) into every rank's copy of the replicated
    table (hmc_potential_shard_push); push=False: three all-gathers after the scans."""
    n, seed = 1_000_000, 2
    d, _ = device_cluster(n, seed)
    single = hmc.OrbitStepper(d["r"], d["v_r"], d["v_t"], d["m"], d["id"], seed)
    sharded = shard.ShardedStepper(shard.InProcessComm(world), shard.split_cluster(d, world), seed, push_tables=push)
    assert sharded.want == shard.partition_counts(n, world)
    for step in range(3):
        single.step()
        sharded.step()
        for key in ("r", "v_r", "v_t", "m", "id"):
            assert torch.equal(torch.cat([s[key] for s in sharded.state]), single.state[key]), (step, key)
        assert [s["r"].numel() for s in sharded.state] == sharded.want
        last = sharded.last
        assert torch.equal(torch.cat([x["r"] for x in last]), single.sorted["r"])
        assert torch.equal(torch.cat([x["phi"] for x in last]), single.phi)
        assert torch.equal(torch.cat([x["m_cum"] for x in last]), single.m_cum)
        assert sharded.pushed == push
        for key in ("E", "J", "r_min", "r_max", "k_min", "k_max", "status"):
            assert torch.equal(torch.cat([x["tp"][key] for x in last]), single.tp[key]), key
        assert torch.equal(torch.cat([x["sample"]["n_try"] for x in last]), single.sample["n_try"])
    assert int(sum(c for c in sharded.counters)[hmc.COUNTER_NAMES.index("trials")]) == int(single.counters[hmc.COUNTER_NAMES.index("trials")])


def test_sharded_step_salpeter_with_ties_and_uneven_ranks():
    """Salpeter masses, exact ties in radius across ranks, a star count that is no multiple of 20 or of G."""
    n, seed, world = 300_017, 4, 3
    d, c = device_cluster(n, seed, "salpeter")
    r = c["r"].copy()
    r[1::3] = r[0::3][: r[1::3].shape[0]]                          # a third of the stars share another star's radius
    d["r"] = dev(r)
    single = hmc.OrbitStepper(d["r"], d["v_r"], d["v_t"], d["m"], d["id"], seed)
    sharded = shard.ShardedStepper(shard.InProcessComm(world), shard.split_cluster(d, world), seed, sample_size=64)
    for step in range(2):
        single.step()
        sharded.step()
        for key in ("r", "v_r", "v_t", "m", "id"):
            assert torch.equal(torch.cat([s[key] for s in sharded.state]), single.state[key]), (step, key)


@pytest.mark.parametrize("n,world", [(100_000, 4), (2049, 3), (5, 2)])
def test_potential_shards_against_the_oracle(oracle, n, world):
    """hmc_potential_totals + hmc_potential_shard over consecutive shards == the oracle's potential of the whole."""
    c = inputs.plummer(n, 11, "salpeter")
    o = np.argsort(c["r"], kind="stable")
    r, m = c["r"][o], c["m"][o]
    o_phi, o_mc = oracle.potential(r, m, 1.5)
    counts = shard.partition_counts(n, world)
    offs = shard.exclusive_scan(counts)
    rs = [dev(r[a:a + k]) for a, k in zip(offs, counts)]
    ms = [dev(m[a:a + k]) for a, k in zip(offs, counts)]
    totals = torch.cat([hmc.hmc_potential_totals(x, y) for x, y in zip(rs, ms)])
    t = totals.cpu().numpy().reshape(world, 4)
    assert abs(t[:, 0].sum() - m.sum()) <= 1e-14 * m.sum()        # the hi parts are the shards' masses
    phi, mc = zip(*[hmc.hmc_potential_shard(x, y, rank, totals, 1.5) for rank, (x, y) in enumerate(zip(rs, ms))])
    assert np.array_equal(torch.cat(phi).cpu().numpy(), o_phi)
    assert np.array_equal(torch.cat(mc).cpu().numpy(), o_mc)


def test_range_calls_against_the_oracle(oracle):
    """S3 / S4 for a range of the table == the oracle's S3 / S4 of the same stars (first, stride 1, count)."""
    n, seed, first, count = 200_003, 13, 70_001, 50_000
    c = inputs.plummer(n, seed)
    o = oracle.orbit_step(c["r"], c["v_r"], c["v_t"], c["m"], c["id"], seed, 3)
    sl = slice(first, first + count)
    otp = oracle.orbit_turning_points(o["r"], o["v_r"], o["v_t"], o["phi"], o["m_cum"], 1.0, first, 1, count)
    osm = oracle.sample_new_radius(o["r"], o["phi"], o["m_cum"], o["r"][sl], o["v_r"][sl], o["v_t"][sl], otp["E"], otp["J"],
                                   otp["r_min"], otp["r_max"], otp["k_min"], otp["k_max"], o["id"][sl], otp["status"], seed, 3)
    tr, tphi, tm = dev(o["r"]), dev(o["phi"]), dev(o["m_cum"])
    vr, vt, ids = dev(o["v_r"][sl]), dev(o["v_t"][sl]), dev(o["id"][sl])
    ws = hmc.alloc_workspace(n)
    tp = hmc.hmc_orbit_turning_points(tr, vr, vt, tphi, tm, first=first, workspace=ws)
    sm = hmc.hmc_sample_new_radius(tr, tphi, tm, vr, vt, tp, ids, seed, 3, first=first, workspace=ws, reuse_tables=True)
    for k in ("E", "J", "r_min", "r_max", "status"):
        assert np.array_equal(tp[k].cpu().numpy(), otp[k]), k
    for k in ("k_min", "k_max"):
        assert np.array_equal(tp[k].cpu().numpy().view(np.uint32), otp[k]), k
    for k in ("r_new", "v_r_new", "v_t_new", "status"):
        assert np.array_equal(sm[k].cpu().numpy(), osm[k]), k
    assert np.array_equal(sm["n_try"].cpu().numpy().view(np.uint16), osm["n_try"])
    # without the tables of a preceding S3 call
    sm2 = hmc.hmc_sample_new_radius(tr, tphi, tm, vr, vt, tp, ids, seed, 3, first=first)
    assert torch.equal(sm2["r_new"], sm["r_new"])
    # argument errors
    with pytest.raises(hmc.HmcError):
        hmc.hmc_orbit_turning_points(tr, vr, vt, tphi, tm, first=n - count + 1)


def test_partition_points():
    g = np.random.default_rng(3)
    r = np.sort(np.round(np.exp(g.uniform(-3, 3, 100_000)), 2) + 0.01)
    spl = np.array([0.0, r[0], r[17], 1.0, r[-1], 1e9, r[50_000]])
    got = hmc.hmc_partition_points(dev(r), dev(spl)).cpu().numpy()
    assert np.array_equal(got, np.searchsorted(r, spl, side="right"))
    empty = torch.empty(0, dtype=torch.float64, device="cuda")
    assert hmc.hmc_partition_points(empty, dev(spl)).cpu().tolist() == [0] * len(spl)


def test_dist_comm_over_nccl_world_of_one():
    """The torch.distributed back-end with the NCCL backend on the one GPU there is: a world of one rank runs the
    same code path (size exchange, padded all-gather, point-to-point all-to-all) as a world of eight."""
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29631")
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        n, seed = 100_000, 6
        d, _ = device_cluster(n, seed)
        single = hmc.OrbitStepper(d["r"], d["v_r"], d["v_t"], d["m"], d["id"], seed)
        sharded = shard.ShardedStepper(shard.DistComm(), [d], seed)
        for _ in range(2):
            single.step()
            sharded.step()
        for key in ("r", "v_r", "v_t", "m", "id"):
            assert torch.equal(sharded.state[0][key], single.state[key]), key
        # the replicated table sits in torch's symmetric memory and is filled by the potential scan's own stores
        # (no peers in a world of one, but the allocation, the rendezvous and the barriers are the real ones)
        assert sharded.pushed
    finally:
        if created:
            dist.destroy_process_group()


def test_host_synchronisations_per_sharded_step():
    """A sharded step reads device memory back on the host once per rank (where the splitters fall in its sorted
    radii); the partition sizes are one more small exchange per rank between processes, none inside one process.
    Everything else -- samples, records, totals, the table -- moves with sizes every rank already knows.  Counted twice:
    by the communicator's own counter, and by PyTorch's synchronisation warnings during the step."""
    n, seed, world = 200_000, 8, 4
    d, _ = device_cluster(n, seed)
    comm = shard.InProcessComm(world)
    st = shard.ShardedStepper(comm, shard.split_cluster(d, world), seed)
    st.step()
    st.step()                     # (the first steps also build the cached index tensors of the sampling)
    torch.cuda.synchronize()
    before = comm.host_syncs
    torch.cuda.set_sync_debug_mode("warn")
    try:
        with warnings.catch_warnings(record=True) as caught:
            warnings.simplefilter("always")
            st.step()
    finally:
        torch.cuda.set_sync_debug_mode("default")
    torch.cuda.synchronize()
    seen = [str(w.message) for w in caught if "synchroniz" in str(w.message).lower()]
    print("host synchronisations in one step of %d shards: counter %d, torch warnings %d" % (world, comm.host_syncs - before, len(seen)))
    assert comm.host_syncs - before == world
    assert len(seen) <= world, seen


def test_record_packing_round_trip():
    g = torch.Generator().manual_seed(3)
    cols = [torch.rand(1000, generator=g, dtype=torch.float64).cuda(), torch.full((1000,), float("nan"), dtype=torch.float64).cuda(),
            torch.randint(-2 ** 31, 2 ** 31 - 1, (1000,), generator=g, dtype=torch.int64).to(torch.int32).cuda()]
    back = shard.unpack_records(shard.pack_records(cols), cols)
    for a, b in zip(cols, back):
        assert a.dtype == b.dtype and torch.equal(a.view(torch.int64) if a.dtype == torch.float64 else a,
                                                  b.view(torch.int64) if b.dtype == torch.float64 else b)
