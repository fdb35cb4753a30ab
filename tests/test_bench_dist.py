"""N > 1 plumbing of bench.py on CPU: two gloo ranks, replicas only.

What is checked: rendezvous from the torchrun environment, the barrier, MAX-over-ranks timing, the
whole-job throughput (stars of all ranks / slowest rank's time), and that replicas get distinct
seeds.  No CUDA and no oracle are involved."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import bench
    rank, local_rank, world = bench.dist_init("gloo")
    assert world == 2 and rank == int(os.environ["RANK"])
    bench.dist_barrier()
    # rank r "processed" 1000 stars in (10 + 5 r) ms
    value, ms = bench.aggregate_throughput(1000.0, 10.0 + 5.0 * rank)
    mx = bench.dist_max(float(rank))
    sm = bench.dist_sum(float(rank + 1))
    seed = bench.replica_seed(3, rank)
    seeds = bench.dist_sum(float(seed))
    bench.dist_barrier()
    if rank == 0:
        print(json.dumps(dict(value=value, ms=ms, mx=mx, sm=sm, seeds=seeds)))
""") % ROOT


def test_two_rank_gloo_aggregation(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", CUDA_VISIBLE_DEVICES="")
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
         "127.0.0.1", "--master-port", "29613", str(script)],
        capture_output=True, text=True, env=env, timeout=240)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    rec = json.loads(line)
    assert rec["ms"] == 15.0                        # slowest rank
    assert abs(rec["value"] - 2000.0 / 15e-3) < 1e-6  # all ranks' stars / max time
    assert rec["mx"] == 1.0 and rec["sm"] == 3.0
    assert rec["seeds"] == 3 + 1003                 # replicas use seed + 1000 * rank


def test_reference_arm_other_ranks_do_no_work():
    """--impl reference: only rank 0 runs the oracle; other ranks exit 0 without output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", CUDA_VISIBLE_DEVICES="")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
