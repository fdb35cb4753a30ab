#!/usr/bin/env python
"""bench.py -- stars/s per orbit step (sort + potential + turning points + sampling), fp64.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference]

A "step" is one pass of the whole hot path over one synthetic Plummer cluster; steps are chained
(the output of a step is the input of the next, re-sorting each step), as in BASELINE.json's
multi-step configs.  The default workload is the configuration the metric is quoted on:
configs[2], N = 1e7 equal-mass stars, seed 3.

Timing: W untimed warm-up steps, then exactly K steps between barrier + torch.cuda.synchronize()
on both sides, CUDA events on the launching stream, MAX over ranks.  The star arrays (440 MB of
state and intermediates per step at N = 1e7) are several times the 126 MB L2, so no explicit L2
flush is needed between steps; `config.l2` says so.

N > 1 ranks run independent replicas (one cluster per GPU, seed + rank): the graded path is one GPU
(the sharded step of paper_1206_5878_b200/shard.py is covered by tests, not timed here),
there is no data-path collective, scaling is "weak".

After the headline's timed region the default run also times the other four BASELINE.json configs
(device-resident steps only, no CPU legs, no end-to-end leg) and reports them under `all_configs`
(--no-all-configs skips that; N = 1e8 takes about a minute to generate).

Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "stars/sec per orbit step (sort+potential+turning points+sampling), fp64, N=1e7"
UNIT = "stars/s"
STAGES = ("sort", "potential", "turning_points", "sampling")
GRAPH_AUTO_MAX_N = 20_000_000     # replaying the step from a graph saves 25 us of launch gaps per step (N = 1e5: 0.169 -> 0.126 ms, 1e7: 2.57 -> 2.54)


# --------------------------------------------------------------------------- roofline model
def algorithmic_bytes_per_star(n: int) -> dict:
    """bytes the method itself must move per star (each streamed array once,
    one table entry per probe of the paper's bisection: 16 B for an (r, Phi) probe, 8 B for an
    r-only probe)."""
    lg = math.log2(n)
    return dict(
        sort=8 + 8 * (12 + 12) + (4 + 28 + 28),
        potential=16 + 16,
        turning_points=40 + 41 + 16 * (2 * lg - 2.9) + 16,
        sampling=45 + 24 + 16 + 1.9 * (8 * (lg - 1.5) + 16),
    )


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def ncu_traffic_bytes(kernel: str, n: int):
    """(DRAM bytes per launch of `kernel`, what the capture was taken from) out of the committed ncu --set full
    capture, profiles/dram_traffic.csv: a constant of THAT build (the `# capture:` line names its commit), not
    something this run measured -- it goes stale when the kernel changes, which is why the line prints it."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    capture, found = None, None
    try:
        for line in open(p):
            if line.startswith("# capture:"):
                capture = line.split(":", 1)[1].strip()
            f = line.strip().split(",")
            if len(f) == 3 and f[0] == str(n) and f[1].split("<")[0] == kernel:
                found = int(f[2])
    except Exception:
        pass
    return found, capture


# --------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.sm_max = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            "hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else 0x8,
            "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4, "hw_power_brake": 0x80,
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        s = sorted(self.samples)
        return dict(sm_mhz=(s[len(s) // 2] if s else None), sm_max_mhz=self.sm_max, reasons=sorted(self.reasons),
                    samples=len(s))


# --------------------------------------------------------------------------- distributed plumbing
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    """Initialise torch.distributed from the torchrun environment (no-op for world size 1)."""
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max(x: float, device="cpu") -> float:
    """MAX over ranks of a host float (device-timed milliseconds)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(x: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def replica_seed(seed: int, rank: int) -> int:
    """Replicas only: rank r runs an independent cluster with seed + 1000 r."""
    return seed + 1000 * rank


def aggregate_throughput(stars_this_rank: float, ms_this_rank: float, device="cpu"):
    """Whole-job stars/s: stars processed by all ranks / max-over-ranks time."""
    ms = dist_max(ms_this_rank, device)
    stars = dist_sum(stars_this_rank, device)
    return stars / (ms * 1e-3), ms


# --------------------------------------------------------------------------- CPU oracle legs
def host_cpu():
    """(model string, logical cores visible to this process) of the box the oracle is timed on."""
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    return model, cores


def oracle_step_timed(cluster, seed, step, stride=1):
    """One step of the oracle (whichever build oracle.use() selected), timed per stage.  stride = 1: every
    star, everything measured.  stride > 1 (explicit opt-in): S3 / S4 on every stride-th star of the sorted
    order only; the caller scales the orbit stages and marks the figure as estimated.
    -> (per-stage seconds measured, result of the step)"""
    import oracle
    t0 = time.perf_counter()
    rs, perm, (vrs, vts, ms), ids = oracle.sort_by_radius(cluster["r"], (cluster["v_r"], cluster["v_t"], cluster["m"]),
                                                          cluster["id"])
    t1 = time.perf_counter()
    phi, mc = oracle.potential(rs, ms)
    t2 = time.perf_counter()
    tp = oracle.orbit_turning_points(rs, vrs, vts, phi, mc, 1.0, 0, stride)
    t3 = time.perf_counter()
    sl = slice(0, None, stride)
    sm = oracle.sample_new_radius(rs, phi, mc, rs[sl], vrs[sl], vts[sl], tp["E"], tp["J"], tp["r_min"], tp["r_max"],
                                  tp["k_min"], tp["k_max"], ids[sl], tp["status"], seed, step)
    t4 = time.perf_counter()
    meas = dict(sort=t1 - t0, potential=t2 - t1, turning_points=t3 - t2, sampling=t4 - t3)
    nxt = None
    if stride == 1:
        nxt = dict(r=sm["r_new"], v_r=sm["v_r_new"], v_t=sm["v_t_new"], m=ms, id=ids)
    return meas, nxt


def oracle_leg(cluster, seed, variant, stride=1):
    """One oracle step on `cluster` with the given build -> dict for the JSON line."""
    import oracle
    n = len(cluster["r"])
    with oracle.use(variant):
        threads = oracle.threads()
        meas, _ = oracle_step_timed(cluster, seed, 0, stride)
    secs = meas["sort"] + meas["potential"] + stride * (meas["turning_points"] + meas["sampling"])
    d = dict(value=n / secs, unit=UNIT, cores=threads, seconds_per_step=round(secs, 3),
             stage_seconds={k: round(v * (stride if k in ("turning_points", "sampling") else 1), 3) for k, v in meas.items()})
    if stride > 1:
        d["estimated"] = "turning points and sampling timed on every %d-th star and scaled x%d" % (stride, stride)
    return d


def cpu_baseline_leg(cluster, seed, stride=1):
    """the oracle as it stands on this box's host cores, same input bytes: (ii) the -fopenmp
    build of the same source on all cores (the top-level figure; `cores` = threads it used) and (i) the
    single-threaded build (`single_core`).  One whole step each at N <= 2e7: measured, nothing scaled."""
    n = len(cluster["r"])
    model, nproc = host_cpu()
    if stride == 1 and n > 20_000_000:
        stride = 16                      # about 10 min per step otherwise; marked as estimated
    allc = oracle_leg(cluster, seed, "omp", stride)
    one = oracle_leg(cluster, seed, "serial", stride)
    what = "every star" if stride == 1 else "S1/S2 on every star, S3/S4 on every %d-th star (scaled)" % stride
    out = dict(value=allc["value"], unit=UNIT, cores=allc["cores"], kind="oracle",
               sample="one whole orbit step at N=%d (%s): %.1f s with the -fopenmp build on %d threads, %.1f s "
                      "single-threaded" % (n, what, allc["seconds_per_step"], allc["cores"], one["seconds_per_step"]),
               cpu_model=model, nproc=nproc, flags="gcc -O2 -ffp-contract=off (-fopenmp: per-star loops of S3/S4 and the gather)",
               all_cores=allc, single_core=one)
    if stride > 1:
        out["estimated"] = allc["estimated"]
    return out


def run_reference(args, cfg):
    """The reference arm: the oracle, chained over warmup + steps whole steps on this arm's config.  Default build:
    -fopenmp on all host cores (a step at N = 1e7 takes seconds, so 25 steps end within a few minutes and every
    reported millisecond was measured); --ref-variant serial is the single-threaded oracle (about 30 s per step)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from paper_1206_5878_b200 import inputs
    import oracle
    oracle.build_all()
    c = inputs.config(args.config, args.n)
    cluster = {k: c[k] for k in ("r", "v_r", "v_t", "m", "id")}
    n = c["n"]
    stride = max(1, args.ref_stride)
    model, nproc = host_cpu()
    secs, stage = [], []
    with oracle.use(args.ref_variant):
        threads = oracle.threads()
        for i in range(args.warmup + args.steps):
            meas, nxt = oracle_step_timed(cluster, c["seed"], i, stride)
            if nxt is not None:
                cluster = nxt                     # chained, as the GPU arm
            if i >= args.warmup:
                secs.append(meas["sort"] + meas["potential"] + stride * (meas["turning_points"] + meas["sampling"]))
                stage.append(meas)
    ms = 1e3 * sum(secs) / len(secs)
    value = n / (ms * 1e-3)
    what = "every star of every step, steps chained" if stride == 1 else \
        "S1/S2 on every star, S3/S4 on every %d-th star and scaled x%d (ESTIMATED; steps not chained)" % (stride, stride)
    cpu = dict(value=value, unit=UNIT, cores=threads, kind="oracle", cpu_model=model, nproc=nproc,
               sample="%d whole orbit steps at N=%d with the %s build of oracle/hmc_oracle.c: %s"
                      % (args.steps, n, args.ref_variant, what),
               stage_seconds={k: round(sum(m[k] for m in stage) / len(stage), 3) for k in STAGES})
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=cfg, cpu_baseline=cpu,
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    if stride > 1:
        line["estimated"] = True
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- GPU arm
def staged_orbit_step(hmc, stepper, ev, stream, fused=False):
    """One step of `stepper` with an event after every stage (events are recorded on the launching stream).
    ev[0..4]: stage boundaries, ev[5]: after S3's table build."""
    s, so = stepper.state, stepper.sorted
    ev[0].record(stream)
    hmc.hmc_sort_by_radius(s["r"], (s["v_r"], s["v_t"], s["m"]), s["id"], r_sorted=so["r"], perm=so["perm"],
                           cols_out=(so["v_r"], so["v_t"], so["m"]), ids_out=so["id"], workspace=stepper.workspace)
    ev[1].record(stream)
    hmc.hmc_potential(so["r"], so["m"], stepper.G, phi=stepper.phi, m_cum=stepper.m_cum, workspace=stepper.workspace)
    ev[2].record(stream)
    if fused:
        ev[5].record(stream)
        ev[3].record(stream)      # "turning_points" reads 0; "sampling" is the fused S3 + S4 call
        hmc.hmc_orbit_step(so["r"], so["v_r"], so["v_t"], stepper.phi, stepper.m_cum, so["id"], stepper.seed,
                           stepper.step_index, stepper.G, tp=stepper.tp, out=stepper.sample,
                           counters=stepper.counters, workspace=stepper.workspace)
    else:
        # S3 as its two launches, with an event between them: hmc_orbit_build_tables + hmc_orbit_turning_points_prebuilt
        # are exactly what hmc_orbit_turning_points does; the event lets turning_points_kernel be timed by itself
        hmc.hmc_orbit_build_tables(so["r"], stepper.phi, stepper.m_cum, stepper.G, workspace=stepper.workspace)
        ev[5].record(stream)
        hmc.hmc_orbit_turning_points(so["r"], so["v_r"], so["v_t"], stepper.phi, stepper.m_cum, stepper.G,
                                     out=stepper.tp, counters=stepper.counters, workspace=stepper.workspace, prebuilt=True)
        ev[3].record(stream)
        hmc.hmc_sample_new_radius(so["r"], stepper.phi, stepper.m_cum, so["v_r"], so["v_t"], stepper.tp, so["id"],
                                  stepper.seed, stepper.step_index, stepper.G, out=stepper.sample,
                                  counters=stepper.counters, workspace=stepper.workspace, reuse_tables=True)
    ev[4].record(stream)
    sm = stepper.sample
    s["r"], sm["r_new"] = sm["r_new"], s["r"]
    s["v_r"], sm["v_r_new"] = sm["v_r_new"], s["v_r"]
    s["v_t"], sm["v_t_new"] = sm["v_t_new"], s["v_t"]
    s["m"], so["m"] = so["m"], s["m"]
    s["id"], so["id"] = so["id"], s["id"]
    stepper.step_index += 1


def time_config(index, steps, warmup, graph_mode, devs, local_rank, peak):
    """Device-resident timing of one BASELINE.json config, as the headline's: `warmup` eager steps, then `steps`
    chained steps between two CUDA events (replayed from a graph of two steps where the headline would be), clocks
    sampled during the timed region; per-stage times from eager steps afterwards.  -> dict for `all_configs`."""
    import numpy as np
    import torch
    from paper_1206_5878_b200 import hmc, inputs
    c = inputs.config(index)
    n = c["n"]
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devs)
    stepper = hmc.OrbitStepper(d(c["r"]), d(c["v_r"]), d(c["v_t"]), d(c["m"]), d(c["id"].view(np.int32)), c["seed"],
                               with_n_try=False)
    name, masses, seed = c["name"], c["masses"], c["seed"]
    del c
    stream = torch.cuda.current_stream()
    mk = lambda: [torch.cuda.Event(enable_timing=True) for _ in range(6)]
    for _ in range(max(warmup, 2)):
        staged_orbit_step(hmc, stepper, mk(), stream)
    if stepper.step_index % 2:
        staged_orbit_step(hmc, stepper, mk(), stream)
    use_graph = graph_mode == "on" or (graph_mode == "auto" and n <= GRAPH_AUTO_MAX_N and steps % 2 == 0)
    if use_graph:
        stepper.run_graph(2)
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    evs = [mk() for _ in range(steps)]
    if use_graph:
        t0.record(stream)
        stepper.run_graph(steps)
        t1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.stop()
        for e in evs:
            staged_orbit_step(hmc, stepper, e, stream)
    else:
        t0.record(stream)
        for e in evs:
            staged_orbit_step(hmc, stepper, e, stream)
        t1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.stop()
    torch.cuda.synchronize()
    ms = t0.elapsed_time(t1) / steps
    stage_ms = {nm: sum(e[i].elapsed_time(e[i + 1]) for e in evs) / steps for i, nm in enumerate(STAGES)}
    model = algorithmic_bytes_per_star(n)
    orbit_ms = stage_ms["potential"] + stage_ms["turning_points"] + stage_ms["sampling"]
    orbit_gbs = (model["potential"] + model["turning_points"] + model["sampling"]) * n / (orbit_ms * 1e-3) / 1e9
    step_gbs = sum(model.values()) * n / (ms * 1e-3) / 1e9
    del stepper
    torch.cuda.empty_cache()
    return dict(index=index, name=name, n=n, masses=masses, seed=seed, steps=steps, ms_per_step=ms,
                stars_per_s=n / (ms * 1e-3), launch="cuda graph of two steps, replayed" if use_graph else "eager",
                stage_ms=stage_ms,
                potential_plus_orbit=dict(ms=orbit_ms, frac_of_8TBs=orbit_gbs / 8000.0, frac_of_measured_peak=orbit_gbs / peak),
                step_frac_of_measured_peak=step_gbs / peak, clocks=clocks)


def run_gpu(args, cfg):
    import numpy as np
    import torch
    from paper_1206_5878_b200 import hmc, inputs

    rank, local_rank, world = dist_init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    devs = "cuda:%d" % local_rank
    hmc.lib()

    c = inputs.config(args.config, args.n)
    n = c["n"]
    if world > 1:   # independent replica per rank
        c.update(inputs.plummer(n, replica_seed(c["seed"], rank), c["masses"]))
    cluster = {k: c[k] for k in ("r", "v_r", "v_t", "m", "id")}
    seed = replica_seed(c["seed"], rank)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devs)
    stepper = hmc.OrbitStepper(d(cluster["r"]), d(cluster["v_r"]), d(cluster["v_t"]), d(cluster["m"]),
                               d(cluster["id"].view(np.int32)), seed, with_n_try=False)
    stream = torch.cuda.current_stream()

    def staged_step(ev):
        staged_orbit_step(hmc, stepper, ev, stream, args.fused)

    mk = lambda: [torch.cuda.Event(enable_timing=True) for _ in range(6)]      # 0-4: stage boundaries, 5: after the table build
    for _ in range(args.warmup):
        staged_step(mk())
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    dist_barrier()
    torch.cuda.synchronize()
    sampler.start()
    evs = [mk() for _ in range(args.steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launch = "eager: four C-ABI calls per step, launched one by one"
    use_graph = args.graph == "on" or (args.graph == "auto" and n <= GRAPH_AUTO_MAX_N and args.steps % 2 == 0 and not args.fused)
    if use_graph:
        # small N: a step is bound by launching its kernels one by one.  The timed steps are replays of a CUDA graph of
        # two steps (OrbitStepper.run_graph); the per-stage times below come from eager steps taken after the timed region.
        while stepper.step_index < 2:                                         # first launches are not captured
            staged_step(mk())
        before = int(hmc.lib().hmc_launch_count())
        stepper.run_graph(2)                                                  # captures two steps, replays them once
        per_two_steps = int(hmc.lib().hmc_launch_count()) - before            # the library counts a launch when it is captured
        torch.cuda.synchronize()
        dist_barrier()
        t_start.record(stream)
        stepper.run_graph(args.steps)
        t_end.record(stream)
        gpu_launches = per_two_steps * (args.steps // 2)                      # kernel nodes replayed in the timed region
        launch = "timed steps replayed from a CUDA graph of two steps (OrbitStepper.run_graph)"
        torch.cuda.synchronize()
        for i in range(args.steps):
            staged_step(evs[i])
        torch.cuda.synchronize()
    else:
        launches_before = int(hmc.lib().hmc_launch_count())
        t_start.record(stream)
        for i in range(args.steps):
            staged_step(evs[i])
        t_end.record(stream)
        gpu_launches = int(hmc.lib().hmc_launch_count()) - launches_before      # counted by the library at each launch
        torch.cuda.synchronize()
    dist_barrier()
    clocks = sampler.stop()
    ms_total = t_start.elapsed_time(t_end)
    value, ms_max = aggregate_throughput(float(n) * args.steps, ms_total, devs)
    stage_ms = {name: sum(e[i].elapsed_time(e[i + 1]) for e in evs) / args.steps for i, name in enumerate(STAGES)}
    s3_kernel_ms = sum(e[5].elapsed_time(e[3]) for e in evs) / args.steps      # turning_points_kernel alone
    counters = {k: int(v) for k, v in zip(hmc.COUNTER_NAMES, stepper.counters.cpu().tolist())}

    # ---- end to end through the host-buffer C-ABI call: pinned host inputs in, results out, every step
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hin = dict(r=pin(cluster["r"]), v_r=pin(cluster["v_r"]), v_t=pin(cluster["v_t"]), m=pin(cluster["m"]),
                   id=pin(cluster["id"].view(np.int32)))
        hout = dict(r_new=torch.empty(n, dtype=torch.float64).pin_memory(), v_r_new=torch.empty(n, dtype=torch.float64).pin_memory(),
                    v_t_new=torch.empty(n, dtype=torch.float64).pin_memory(), m=torch.empty(n, dtype=torch.float64).pin_memory(),
                    id=torch.empty(n, dtype=torch.int32).pin_memory())
        del stepper
        torch.cuda.empty_cache()
        arena = torch.empty(hmc.step_host_arena_bytes(n), dtype=torch.uint8, device=devs)

        def host_step(i):
            nonlocal hin, hout
            hmc.hmc_step_host(hin["r"], hin["v_r"], hin["v_t"], hin["m"], hin["id"], hout, seed, i, arena=arena)
            nxt = dict(r=hout["r_new"], v_r=hout["v_r_new"], v_t=hout["v_t_new"], m=hout["m"], id=hout["id"])
            hout = dict(r_new=hin["r"], v_r_new=hin["v_r"], v_t_new=hin["v_t"], m=hin["m"], id=hin["id"])
            hin = nxt

        e2e_steps = max(1, args.steps if args.e2e_steps is None else args.e2e_steps)
        for i in range(2):
            host_step(i)
        torch.cuda.synchronize()
        dist_barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for i in range(e2e_steps):
            host_step(2 + i)
        b.record(stream)
        torch.cuda.synchronize()
        dist_barrier()
        e2e_value, _ = aggregate_throughput(float(n) * e2e_steps, a.elapsed_time(b), devs)
        e2e = dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=n * (4 * 8 + 4), d2h_bytes_per_step=n * (4 * 8 + 4),
                   steps=e2e_steps, api="hmc_step_host (pinned host buffers; H2D, 4 stages, D2H per step)")

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel.  sample_new_radius_kernel is the longest single launch of a step
    # (profiles/: launch list) and the only kernel of its stage when S4 reuses S3's tables, so the CUDA events
    # around that call, recorded on the launching stream, time exactly that kernel, once per step.
    model = algorithmic_bytes_per_star(n)
    peak, peak_src = measured_peak_gbs()
    # The two long launches of a step, each timed exactly by the events around its call; the longer one is reported.
    cand = {"sampling": ("sample_new_radius_kernel", stage_ms["sampling"])}
    if not args.fused:
        cand["turning_points"] = ("turning_points_kernel", s3_kernel_ms)
    dom = max(cand, key=lambda k: cand[k][1])
    dom_kernel, dom_ms = cand[dom]
    achieved = model[dom] * n / (dom_ms * 1e-3) / 1e9
    traffic, capture = ncu_traffic_bytes(dom_kernel, n)
    # `bound`: what ncu shows the kernel is limited by (profiles/r2b_ncu_full_summary.txt); `metric_roofline`: the
    # roofline SURVEY.md 8(d) quotes the metric against, which `achieved`, `peak` and `frac` (= `model_frac`) refer to.
    roofline = dict(bound="issue", metric_roofline="hbm", kernel=dom_kernel, stage=dom, achieved=achieved, peak=peak, unit="GB/s",
                    frac=achieved / peak, traffic=traffic, peak_source=peak_src,
                    algorithmic_bytes_per_star=model[dom], stars_per_launch=n, launch_ms=dom_ms,
                    launches_timed=args.steps,
                    # `achieved` / `frac` are SURVEY.md 8(d)'s ALGORITHMIC bytes over the measured launch time: a model
                    # fraction (one table entry per probe of the paper's bisection; this kernel serves most probes from
                    # shared memory).  What the launch physically moved, by ncu, over the same measured time:
                    model_frac=achieved / peak,
                    physical=(dict(dram_bytes_per_launch=traffic, achieved=traffic / (dom_ms * 1e-3) / 1e9,
                                   frac=traffic / (dom_ms * 1e-3) / 1e9 / peak, capture=capture,
                                   measured_in_this_run=False,      # DRAM bytes: a constant of the committed ncu capture

                                   limiter="not streamed bytes: 8 warps per scheduler of dependent fp64 chains and loads "
                                           "(ncu: issue slots 54-56 % used), for turning_points_kernel together with the "
                                           "rate of random 128-byte DRAM lines (profiles/r2b.md, DESIGN.md 5 and 5a)")
                              if traffic else None),
                    # what ncu shows the kernel waits for, as opposed to the roofline the metric is quoted against
                    bound_observed="issue / dependent-instruction latency at 32 warps per SM",
                    other_long_launch={k: dict(kernel=v[0], launch_ms=v[1], model_frac=model[k] * n / (v[1] * 1e-3) / 1e9 / peak)
                                       for k, v in cand.items() if k != dom})
    orbit_ms = stage_ms["potential"] + stage_ms["turning_points"] + stage_ms["sampling"]
    orbit_bytes = model["potential"] + model["turning_points"] + model["sampling"]
    stages = {s: dict(ms=stage_ms[s], stars_per_s=n / (stage_ms[s] * 1e-3), algorithmic_bytes_per_star=model[s],
                      achieved_gbs=model[s] * n / (stage_ms[s] * 1e-3) / 1e9,
                      frac_of_peak=model[s] * n / (stage_ms[s] * 1e-3) / 1e9 / peak) for s in STAGES}
    potential_plus_orbit = dict(ms=orbit_ms, stars_per_s=n / (orbit_ms * 1e-3),
                                achieved_gbs=orbit_bytes * n / (orbit_ms * 1e-3) / 1e9,
                                frac_of_measured_peak=orbit_bytes * n / (orbit_ms * 1e-3) / 1e9 / peak,
                                frac_of_8TBs=orbit_bytes * n / (orbit_ms * 1e-3) / 1e9 / 8000.0)

    all_configs = None
    if world == 1 and not args.no_all_configs and args.n is None and not args.fused:
        if e2e is None:
            del stepper
        else:
            del arena, hin, hout
        torch.cuda.empty_cache()
        all_configs = [time_config(i, args.steps, args.warmup, args.graph, devs, local_rank, peak)
                       for i in range(len(inputs.CONFIGS)) if i != args.config]

    cpu = None
    if world == 1 or rank == 0:
        if not args.no_cpu_baseline:
            import oracle
            oracle.build_all()
            cpu = cpu_baseline_leg(cluster, c["seed"], max(1, args.ref_stride))

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_max / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=cfg, launch=launch, clocks=clocks, e2e=e2e, gpu_launches=gpu_launches,
                roofline=roofline, cpu_baseline=cpu, stages=stages, potential_plus_orbit=potential_plus_orbit,
                counters=counters, all_configs=all_configs)
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- sharded step (one cluster over the ranks)
def run_sharded(args, cfg):
    """--parallelism sharded: ONE cluster of the config's N stars cut over the ranks (paper_1206_5878_b200/shard.py:
    sample sort + redistribution, shard potentials, replicated table, range S3 / S4), so the scaling is "strong".
    Under torchrun every rank is a process with one shard (shard.DistComm over NCCL); a world of one goes through the
    same communicator.  --shards G (world of one only) instead holds G shards in this one process
    (shard.InProcessComm): the one-GPU proxy for what the sharded step costs beyond the single-GPU step -- extra sort
    passes, record packing and exchange copies, G table builds -- with a per-phase breakdown.  No multi-GPU hardware
    was available to run this with more than one rank."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1206_5878_b200 import hmc, inputs, shard

    rank, local_rank, world = dist_init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    devs = "cuda:%d" % local_rank
    hmc.lib()
    c = inputs.config(args.config, args.n)
    n, seed = c["n"], c["seed"]
    cluster = {k: (c[k].view(np.int32) if k == "id" else c[k]) for k in ("r", "v_r", "v_t", "m", "id")}
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devs)
    in_process = world == 1 and args.shards > 1
    if in_process:
        comm = shard.InProcessComm(args.shards)
        shards = [{k: d(v) for k, v in part.items()} for part in shard.split_cluster(cluster, args.shards)]
        how = "sharded x1 process, %d in-process shards on one GPU (proxy)" % args.shards
    else:
        if not dist.is_initialized():                       # a world of one still goes through DistComm / NCCL
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29633")
            dist.init_process_group("nccl", rank=0, world_size=1)
        comm = shard.DistComm()
        shards = [{k: d(v) for k, v in shard.split_cluster(cluster, world)[rank].items()}]
        how = "sharded x%d" % world
    stepper = shard.ShardedStepper(comm, shards, seed, n_total=n)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        stepper.step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    dist_barrier()
    torch.cuda.synchronize()
    sampler.start()
    launches, syncs = int(hmc.lib().hmc_launch_count()), comm.host_syncs
    stepper.marks = []
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for _ in range(args.steps):
        stepper.step()
    t1.record(stream)
    torch.cuda.synchronize()
    dist_barrier()
    clocks = sampler.stop()
    launches, syncs = int(hmc.lib().hmc_launch_count()) - launches, comm.host_syncs - syncs
    value, ms_max = aggregate_throughput(float(n) * args.steps / world, t0.elapsed_time(t1), devs)
    phases, marks = {}, stepper.marks
    for (_, a), (name, b) in zip(marks, marks[1:]):
        if name != "start":
            phases[name] = phases.get(name, 0.0) + a.elapsed_time(b) / args.steps
    stepper.marks = None
    # the single-GPU step on the same cluster in the same process (world of one only): what the sharded step is compared with
    single_ms = None
    if world == 1:
        del stepper, shards
        torch.cuda.empty_cache()
        one = hmc.OrbitStepper(d(cluster["r"]), d(cluster["v_r"]), d(cluster["v_t"]), d(cluster["m"]), d(cluster["id"]), seed,
                               with_n_try=False)
        for _ in range(max(args.warmup, 1)):
            one.step()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(args.steps):
            one.step()
        b.record(stream)
        torch.cuda.synchronize()
        single_ms = a.elapsed_time(b) / args.steps
    if rank != 0:
        return 0
    cfg = dict(cfg, parallelism=how)
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_max / args.steps, higher_is_better=True, scaling="strong", vs_baseline=None, dtype="f64",
                data="synthetic", config=cfg, launch="eager", clocks=clocks, e2e=None, gpu_launches=launches,
                roofline=None, cpu_baseline=None, phases_ms=phases,
                host_syncs_per_step=syncs / args.steps / (args.shards if in_process else 1),
                single_gpu_ms_per_step=single_ms,
                note="sharded step, device-resident; torch copies (record packing, concatenation) are not in gpu_launches")
    print(json.dumps(line))
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2: N=1e7, the metric's)")
    ap.add_argument("--n", type=int, default=None, help="override N (same recipe and seed); not a bench line")
    ap.add_argument("--ref-stride", type=int, default=1,
                    help="oracle legs, explicit opt-in: orbit stages on every k-th star, scaled (marks the figure ESTIMATED)")
    ap.add_argument("--ref-variant", default="omp", choices=["omp", "serial"],
                    help="--impl reference: which build of the oracle (omp = all host cores, serial = one core)")
    ap.add_argument("--e2e-steps", type=int, default=None, help="steps of the end-to-end leg (default: --steps)")
    ap.add_argument("--no-all-configs", action="store_true",
                    help="skip the device-resident timing of the other four BASELINE.json configs (`all_configs`)")
    ap.add_argument("--fused", action="store_true", help="S3 and S4 as the single call hmc_orbit_step")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="timed steps as replays of a CUDA graph of two steps (auto: N <= %d and an even --steps)" % GRAPH_AUTO_MAX_N)
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "sharded"],
                    help="replicas: one independent cluster per GPU (weak scaling, the graded path); sharded: one cluster "
                         "cut over the ranks (strong scaling, paper_1206_5878_b200/shard.py)")
    ap.add_argument("--shards", type=int, default=1,
                    help="--parallelism sharded with one process: hold this many shards in the process (one-GPU proxy)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args(argv)
    from paper_1206_5878_b200 import inputs
    base = inputs.CONFIGS[args.config]
    n = args.n or base["n"]
    cfg = dict(workload="BASELINE.json configs[%d]: %s, N=%d, %s masses, seed %d, chained orbit steps"
                        % (args.config, base["name"], n, base["masses"], base["seed"]),
               n_stars=n, masses=base["masses"], seed=base["seed"], parallelism="replicas x%d" % max(args.gpus, 1),
               l2="working set per step (>= 44 B/star state + 97 B/star intermediates) exceeds the 126 MB L2 at "
                  "N=1e7; no explicit flush")
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.parallelism == "sharded":
        return run_sharded(args, cfg)
    return run_gpu(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
