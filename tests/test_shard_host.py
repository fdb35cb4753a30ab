"""Host logic of the sharded step (paper_1206_5878_b200/shard.py), CPU only.

Pins: the paper's worked redistribution example (tests/golden/redistribution_example.txt), Eq. 17
 against the decomposition rule of PAPER.md:194, and the Sample Sort + redistribution data movement
 against a global stable sort -- with CPU stand-ins (torch.sort, torch.searchsorted) for
the two libhmc kernels the product uses, over the in-process communicator and over two gloo ranks."""
import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest
import torch

from paper_1206_5878_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def golden_example():
    rec = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "redistribution_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        rec[key] = [int(v) for v in vals]
    return rec


def test_decomposition_of_the_worked_example():
    g = golden_example()
    n, p = sum(g["received"]), len(g["received"])
    assert n == 450 and p == 4
    want = shard.partition_counts(n, p)
    assert want == g["expected"]                                   # 120 120 100 110
    assert shard.exclusive_scan(want)[1:] == g["splitters"]        # global splitter points 120 240 340


def test_redistribution_plan_of_the_worked_example():
    g = golden_example()
    plan = shard.redistribution_plan(g["received"], g["expected"])
    # "processor 3 ... has stars with indices between 231 - 370 ... 231 - 240 and 341 - 370 need to be sent to
    # processors 2 and 4 respectively"
    assert plan[2] == [0, 10, 100, 30]
    assert plan[0] == [100, 0, 0, 0]                               # 1-100 stay
    assert plan[1] == [20, 110, 0, 0]                              # 101-120 go to processor 1, 121-230 stay
    assert plan[3] == [0, 0, 0, 80]
    for d in range(4):
        assert sum(plan[s][d] for s in range(4)) == g["expected"][d]
    for s in range(4):
        assert sum(plan[s]) == g["received"][s]


@pytest.mark.parametrize("n,p", [(450, 4), (100_000, 8), (1_000_000, 7), (19, 4), (20, 1), (10_000_019, 3), (59, 3)])
def test_eq17_global_index_matches_the_decomposition(n, p):
    counts = shard.partition_counts(n, p)
    assert sum(counts) == n
    assert all(c % shard.N_M == 0 for c in counts[:-1])            # multiples of 20 on the first p - 1 processors
    assert max(counts[:-1], default=0) - min(counts[:-1], default=0) <= shard.N_M
    offs = shard.exclusive_scan(counts)
    for rank in range(p):
        assert shard.global_index(0, rank, n, p) == offs[rank]
        if counts[rank]:
            assert shard.global_index(counts[rank] - 1, rank, n, p) == offs[rank] + counts[rank] - 1
    # every global index is produced exactly once
    if n <= 1000:
        seen = sorted(shard.global_index(i, r, n, p) for r in range(p) for i in range(counts[r]))
        assert seen == list(range(n))


def cpu_local_sort(columns):
    order = torch.sort(columns[0], stable=True).indices
    return [c[order] for c in columns]


def cpu_partition_points(keys, splitters):
    return torch.searchsorted(keys, splitters, right=True).tolist()


def make_columns(n, seed, ties):
    g = np.random.default_rng(seed)
    r = np.exp(g.uniform(-4, 4, n))
    if ties:
        r = np.round(r, 1) + 0.1                                   # many exactly equal radii, also across ranks
    return [torch.from_numpy(r), torch.from_numpy(g.random(n)), torch.arange(n, dtype=torch.int32)]


@pytest.mark.parametrize("world,n,ties", [(1, 1000, False), (2, 1000, True), (4, 5003, False), (8, 20_001, True),
                                          (8, 100, True), (3, 7, False)])
def test_sample_sort_in_process(world, n, ties):
    cols = make_columns(n, 5 + world, ties)
    counts = shard.partition_counts(n, world)
    offs = shard.exclusive_scan(counts)
    parts = [[c[o:o + k] for c in cols] for o, k in zip(offs, counts)]
    out = shard.sample_sort(shard.InProcessComm(world), parts, 16, counts, cpu_local_sort, cpu_partition_points)
    ref = cpu_local_sort(cols)                                     # the unique order by (r, input index)
    for rank in range(world):
        for k in range(3):
            assert torch.equal(out[rank][k], ref[k][offs[rank]:offs[rank] + counts[rank]]), (rank, k)


def test_sample_sort_with_all_stars_on_one_rank():
    """A rank may start empty (and another hold everything): the exchange and the redistribution still deliver."""
    n, world = 3000, 4
    cols = make_columns(n, 9, True)
    parts = [[c[:0] for c in cols], cols, [c[:0] for c in cols], [c[:0] for c in cols]]
    want = shard.partition_counts(n, world)
    out = shard.sample_sort(shard.InProcessComm(world), parts, 8, want, cpu_local_sort, cpu_partition_points)
    ref = cpu_local_sort(cols)
    offs = shard.exclusive_scan(want)
    for rank in range(world):
        assert torch.equal(out[rank][2], ref[2][offs[rank]:offs[rank] + want[rank]])


WORKER = textwrap.dedent("""
    import sys
    sys.path.insert(0, %r)
    sys.path.insert(0, %r)
    import torch, torch.distributed as dist
    from paper_1206_5878_b200 import shard
    from test_shard_host import make_columns, cpu_local_sort, cpu_partition_points
    dist.init_process_group("gloo")
    comm = shard.DistComm()
    assert comm.world == 2
    n = 4001
    cols = make_columns(n, 77, True)                       # both ranks build the same cluster and take their range
    counts = shard.partition_counts(n, comm.world)
    offs = shard.exclusive_scan(counts)
    o, k = offs[comm.rank], counts[comm.rank]
    # collectives on their own
    got = comm.all_gather([torch.arange(comm.rank + 2, dtype=torch.float64)])[0]
    assert [t.numel() for t in got] == [2, 3] and got[1][2] == 2.0
    dist.all_gather_object = None                           # nothing may be pickled between ranks any more
    sizes = comm.all_gather_ints([[3 + comm.rank, 4 + comm.rank]])[0]
    assert sizes == [[3, 4], [4, 5]]
    rows = torch.full((sum(sizes[comm.rank]), 2), comm.rank, dtype=torch.int64)
    back = comm.exchange([rows], sizes)[0]                  # rank d receives 3 + d rows of zeros, then 4 + d rows of ones
    assert back.shape == (7 + 2 * comm.rank, 2) and back[:3 + comm.rank].eq(0).all() and back[3 + comm.rank:].eq(1).all()
    before = comm.host_syncs
    # the sort
    out = shard.sample_sort(comm, [[c[o:o + k] for c in cols]], 32, counts, cpu_local_sort, cpu_partition_points)[0]
    ref = cpu_local_sort(cols)
    for j in range(3):
        assert torch.equal(out[j], ref[j][o:o + k]), j
    assert comm.host_syncs - before == 2                    # splitter positions, partition sizes: nothing else
    dist.barrier()
    if comm.rank == 0:
        print("SHARD_OK")
""") % (ROOT, os.path.join(ROOT, "tests"))


def test_sample_sort_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", CUDA_VISIBLE_DEVICES="")
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
         "127.0.0.1", "--master-port", "29617", str(script)],
        capture_output=True, text=True, env=env, timeout=240)
    assert out.returncode == 0, out.stderr[-3000:]
    assert "SHARD_OK" in out.stdout
