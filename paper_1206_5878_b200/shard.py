"""The orbit step sharded over G GPUs, in the paper's own shape:

* the stars are cut into G consecutive ranges of the radius-sorted order, every range but the last a multiple of
  n_m = 20 stars (Eq. 17);
* S1 is the paper's Sample Sort: sort the local stars, sample s keys per rank, gather the
  samples, pick the splitters, exchange partitions (all-to-all), sort what was received; then the redistribution
  phase (exclusive scan of the counts + all-to-all) restores the exact decomposition;
* S2 needs one all-gather of G x 4 doubles: every shard's (sum m, sum m/r) in double-double, from which each rank's
  launch adds up what lies before and after its range (the MPI_Exscan idea of PAPER.md:259 applied to the potential
  the paper calls "inherently sequential", :185);
* r, Phi and M are replicated by an all-gather ("we maintain a copy of it on all nodes"), after which S3
  and S4 of a rank's own stars need no communication.

This file holds HOST LOGIC ONLY: integer bookkeeping of the decomposition, which slices go where, and two
communication back-ends with the same five collectives.  Every sort, sum, search and draw is a libhmc kernel called
through ``hmc`` (there is no CPU path: the kernels need a GPU).  The random numbers are keyed by the persistent star id
(R9) and M_k, S_k are exact sums rounded once (R1p), so the sharded step reproduces the single-GPU step bit
for bit whatever G is (tests/test_gpu_shard.py).

Exchange format: the columns of a star travel as ONE record (a row of 64-bit words, one word per column), so each of
the two exchanges of the sort is one collective, and the only things the host reads back in a step are the splitter
positions (one read per rank) and the matrix of partition sizes (one small all-gather per rank): two host
synchronisations per rank and step, counted in ``comm.host_syncs``.  The redistribution needs no further exchange of
sizes: every rank holds the whole matrix, hence knows how many stars every rank holds after the first exchange.

Back-ends:
  InProcessComm(G)   G shards held by ONE process on one device; a collective is a hand-over of device tensors.
                     This is what one GPU can test, and what the tests use.
  DistComm()         one shard per process over torch.distributed (NCCL between GPUs; gloo on CPU tensors in the
                     world-size-2 host-logic tests); the replicated table in torch's symmetric memory, filled by
                     the ranks' own stores (see table_views below).  UNMEASURED ON HARDWARE: no multi-GPU node was
                     available.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence

import torch

N_M = 20   # "we choose a bin size of 20 ... the number of stars per processor is a multiple of 20"


# ------------------------------------------------------------------------------------------------ decomposition
def partition_counts(n_stars: int, p: int, n_m: int = N_M) -> List[int]:
    """Stars per processor: multiples of n_m for the first p - 1 processors, the rest to the last;
    the block counts are those Eq. 17 implies: with B = floor(N / n_m) blocks, processors id < B mod p hold
    floor(B / p) + 1 blocks, the others floor(B / p)."""
    blocks = n_stars // n_m
    q, rem = divmod(blocks, p)
    counts = [(q + 1) * n_m if rank < rem else q * n_m for rank in range(p)]
    counts[-1] += n_stars - blocks * n_m
    return counts


def global_index(i: int, rank: int, n_stars: int, p: int, n_m: int = N_M) -> int:
    """Eq. 17: global index of local star i on processor `rank`."""
    blocks = n_stars // n_m
    q, rem = divmod(blocks, p)
    if rank < rem:
        return i + rank * q * n_m + rank * n_m
    return i + rank * q * n_m + rem * n_m


def exclusive_scan(counts: Sequence[int]) -> List[int]:
    out, run = [], 0
    for c in counts:
        out.append(run)
        run += c
    return out


def redistribution_plan(have: Sequence[int], want: Sequence[int]) -> List[List[int]]:
    """PAPER.md:259-261.  After the sort processor s holds have[s] consecutive stars of the global order; the
    decomposition wants want[d] on processor d.  -> send[s][d] = how many of its stars s passes to d; a processor's
    stars go out in order, lowest destination first, and arrive in source order, which is the global order."""
    if sum(have) != sum(want):
        raise ValueError("redistribution_plan: %d stars held, %d wanted" % (sum(have), sum(want)))
    h0, w0 = exclusive_scan(have), exclusive_scan(want)      # the parallel prefix reduction (MPI_Exscan)
    p = len(have)
    send = [[0] * p for _ in range(p)]
    for s in range(p):
        for d in range(p):
            lo, hi = max(h0[s], w0[d]), min(h0[s] + have[s], w0[d] + want[d])
            send[s][d] = max(0, hi - lo)
    return send


def sample_positions(n_local: int, s: int) -> List[int]:
    """Phase 2: "uniformly sample s keys" of the locally sorted block."""
    return [min(n_local - 1, ((2 * k + 1) * n_local) // (2 * s)) for k in range(s)] if n_local > 0 else []


def splitter_positions(s: int, p: int) -> List[int]:
    """Phase 3: "keys at indices s, 2s, 3s, ..., (p-1)s" of the sorted combined sample."""
    return [j * s for j in range(1, p)]


# ------------------------------------------------------------------------------------------------ communication
# A communicator may offer ``table_views(n, device)``: for every local rank, (its own copy of the replicated table,
# the other ranks' copies) as dicts of (r, phi, m_cum) tensors [n] that this process can hand to a kernel -- its own
# memory, or peer GPUs' memory mapped into this process.  ShardedStepper then fuses the table's all-gather into the
# potential scan (hmc_potential_shard_push: each rank's launch stores its slice into every copy) and calls
# ``tables_complete()`` ("every rank's stores have landed") before S3.  ``table_views`` returns None when the
# communicator cannot offer that (CPU tensors, no peer mapping): the stepper then takes three all-gathers.
#   InProcessComm: all copies live on one device; stream order is the barrier.
#   DistComm:      torch's symmetric memory (one allocation per rank, every rank's mapped into every process over
#                  NVLink peer access; the handle's barrier orders the stores).  Exercised with a world of ONE on the
#                  one-GPU boxes this was built on; with more ranks it is correct by construction only.
class InProcessComm:
    """G ranks in one process.  Arguments and results are lists with one entry per rank."""

    def __init__(self, world: int):
        self.world = world
        self.local_ranks = list(range(world))
        self.host_syncs = 0          # times the host waited for the device or for other ranks (see sample_sort)

    def all_gather(self, xs: List[torch.Tensor], sizes: Optional[Sequence[int]] = None) -> List[List[torch.Tensor]]:
        """out[rank] = [x of rank 0, ..., x of rank G-1].  sizes: the ranks' element counts, if the caller knows them."""
        return [list(xs) for _ in self.local_ranks]

    def exchange(self, recs: List[torch.Tensor], counts: Sequence[Sequence[int]]) -> List[torch.Tensor]:
        """One all-to-all of records.  recs[src] = rows [n_src, W], the rows for destination 0 first, then 1, ...;
        counts[src][dst] = how many rows src sends to dst (the whole matrix, known to every rank).
        -> per destination, the rows it receives, in source order."""
        offs = [exclusive_scan(row) for row in counts]
        out = []
        for dst in range(self.world):
            parts = [recs[src][offs[src][dst]:offs[src][dst] + counts[src][dst]] for src in range(self.world) if counts[src][dst]]
            out.append(torch.cat(parts) if len(parts) > 1 else (parts[0] if parts else recs[dst][:0]))
        return out

    def all_gather_ints(self, xs: List[List[int]]) -> List[List[List[int]]]:
        return [list(xs) for _ in self.local_ranks]

    def table_views(self, n: int, device):
        """One copy of the replicated table per rank, every copy reachable by every rank (same device)."""
        if getattr(self, "_tables_n", None) != (n, str(device)):
            f = dict(dtype=torch.float64, device=device)
            self._tables = [dict(r=torch.empty(n, **f), phi=torch.empty(n, **f), m_cum=torch.empty(n, **f)) for _ in self.local_ranks]
            self._tables_n = (n, str(device))
        return [(t, [u for j, u in enumerate(self._tables) if j != i]) for i, t in enumerate(self._tables)]

    def tables_complete(self):
        """Every rank's pushes have landed in every copy: the shards share a device and a stream, so stream order says so."""


class DistComm:
    """One rank per process over torch.distributed.  Lists have ONE entry (this process's rank); the nested lists
    of the results run over all ranks.  Works with the tensors' own backend: NCCL for CUDA tensors, gloo for CPU."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        self.local_ranks = [self.rank]
        self.host_syncs = 0
        self.nccl = dist.get_backend(group) == "nccl"
        self.device = torch.device("cuda", torch.cuda.current_device()) if self.nccl else torch.device("cpu")

    def all_gather_ints(self, xs: List[List[int]]) -> List[List[List[int]]]:
        """Every rank's list of integers (all of one length) to every rank: ONE tensor all-gather and one read back to
        the host -- nothing is pickled."""
        mine = torch.tensor(list(xs[0]), dtype=torch.int64, device=self.device)
        out = torch.empty(self.world * mine.numel(), dtype=torch.int64, device=self.device)
        if self.nccl:
            self.dist.all_gather_into_tensor(out, mine, group=self.group)
        else:
            self.dist.all_gather(list(out.view(self.world, -1).unbind(0)), mine, group=self.group)
        self.host_syncs += 1
        return [out.view(self.world, -1).cpu().tolist()]

    def exchange(self, recs: List[torch.Tensor], counts: Sequence[Sequence[int]]) -> List[torch.Tensor]:
        """One all-to-all of records (see InProcessComm.exchange): all_to_all_single over NCCL; gloo, which has no
        all-to-all, gets the same transfers as one batch of point-to-point operations."""
        rec = recs[0].contiguous()
        send = [int(c) for c in counts[self.rank]]
        recv = [int(counts[src][self.rank]) for src in range(self.world)]
        out = torch.empty((sum(recv),) + tuple(rec.shape[1:]), dtype=rec.dtype, device=rec.device)
        if self.nccl:
            self.dist.all_to_all_single(out, rec, recv, send, group=self.group)
            return [out]
        so, ro = exclusive_scan(send), exclusive_scan(recv)
        out[ro[self.rank]:ro[self.rank] + recv[self.rank]] = rec[so[self.rank]:so[self.rank] + send[self.rank]]
        ops = []
        for other in range(self.world):
            if other == self.rank:
                continue
            if send[other]:
                ops.append(self.dist.P2POp(self.dist.isend, rec[so[other]:so[other] + send[other]], other, self.group))
            if recv[other]:
                ops.append(self.dist.P2POp(self.dist.irecv, out[ro[other]:ro[other] + recv[other]], other, self.group))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()
        return [out]

    def table_views(self, n: int, device):
        """This rank's copy of the replicated table in symmetric memory and the other ranks' copies mapped into this
        process; None when that is not available (CPU tensors, no symmetric-memory support)."""
        if torch.device(device).type != "cuda":
            return None
        if getattr(self, "_tables_n", None) != n:
            try:
                import torch.distributed._symmetric_memory as symm
                group = self.group if self.group is not None else self.dist.group.WORLD
                buf = symm.empty(3 * n, dtype=torch.float64, device=device)
                handle = symm.rendezvous(buf, group.group_name)
                views = [handle.get_buffer(p, (3 * n,), torch.float64) for p in range(self.world)]
            except Exception:
                self._tables, self._tables_n = None, n
                return None
            cut = lambda v: dict(r=v[:n], phi=v[n:2 * n], m_cum=v[2 * n:])
            self._symm, self._symm_buf = handle, buf
            self._tables = (cut(views[self.rank]), [cut(v) for p, v in enumerate(views) if p != self.rank])
            self._tables_n = n
        if self._tables is None:
            return None
        self._symm.barrier()          # nobody still reads the table of the step before while it is overwritten
        return [self._tables]

    def tables_complete(self):
        """Every rank's stores into every copy are done (device-side barrier across the ranks, on the current stream)."""
        self._symm.barrier()

    def all_gather(self, xs: List[torch.Tensor], sizes: Optional[Sequence[int]] = None) -> List[List[torch.Tensor]]:
        """sizes: the ranks' element counts when the caller knows them (samples, totals, the decomposition's ranges);
        otherwise they are exchanged first (one more host synchronisation)."""
        x = xs[0].contiguous()
        sizes = [v[0] for v in self.all_gather_ints([[x.numel()]])[0]] if sizes is None else [int(v) for v in sizes]
        biggest = max(sizes)
        pad = x if x.numel() == biggest else torch.cat([x.reshape(-1), x.new_zeros(biggest - x.numel())])
        bufs = [torch.empty(biggest, dtype=x.dtype, device=x.device) for _ in range(self.world)]
        self.dist.all_gather(bufs, pad.reshape(-1), group=self.group)
        return [[b[:k] for b, k in zip(bufs, sizes)]]


# ------------------------------------------------------------------------------------------------ sample sort
_INDEX_CACHE = {}


def _index_tensor(positions: Sequence[int], device) -> torch.Tensor:
    """The positions as an index tensor on `device`, made once per distinct list: building it is a blocking
    host-to-device copy, and the lists (sample positions of a rank's range, splitter positions) repeat every step."""
    key = (tuple(positions), str(device))
    t = _INDEX_CACHE.get(key)
    if t is None:
        if len(_INDEX_CACHE) > 256:
            _INDEX_CACHE.clear()
        t = _INDEX_CACHE[key] = torch.tensor(list(positions), dtype=torch.long, device=device)
    return t


def pack_records(columns: Sequence[torch.Tensor]) -> torch.Tensor:
    """The columns of a rank's stars (float64 or int32, equal lengths) as one row of 64-bit words per star."""
    words = [c.view(torch.int64) if c.dtype == torch.float64 else c.to(torch.int64) for c in columns]
    return torch.stack(words, dim=1)


def unpack_records(rec: torch.Tensor, like: Sequence[torch.Tensor]) -> List[torch.Tensor]:
    """Inverse of pack_records; `like` gives the dtype of each column."""
    return [rec[:, k].contiguous().view(torch.float64) if c.dtype == torch.float64 else rec[:, k].to(c.dtype)
            for k, c in enumerate(like)]


def sample_sort(comm, cols: List[List[torch.Tensor]], sample_size: int, want: Sequence[int],
                local_sort: Callable, partition_points: Callable, mark: Optional[Callable] = None) -> List[List[torch.Tensor]]:
    """The paper's Sample Sort + redistribution over the ranks of `comm`.

    cols[lr] = the columns of local rank lr, the KEY (radius) first; every column of a rank has the same length.
    local_sort(columns) -> columns sorted by the first one, stably; partition_points(sorted_keys, splitters) ->
    list of ints, the number of keys <= each splitter (this reads device memory back: one host synchronisation).
    Both are libhmc kernels in the product (ShardedStepper); the host-logic tests pass CPU stand-ins.
    mark(name), if given, is called after each phase (the stepper records CUDA events there).
    -> the columns of each local rank after the sort: rank d holds stars exclusive_scan(want)[d] ... of the global
    order, want[d] of them."""
    world, L = comm.world, len(comm.local_ranks)
    mark = mark or (lambda name: None)
    like = cols[0]
    # phase 1: sort local data
    cols = [local_sort(c) if c[0].numel() > 1 else c for c in cols]
    mark("local_sort")
    if world > 1:
        # phase 2: sampling (a rank without stars contributes +inf samples, which sort last)
        samples = []
        for c in cols:
            key = c[0]
            pos = sample_positions(key.numel(), sample_size)
            samples.append(key[_index_tensor(pos, key.device)] if pos
                           else torch.full((sample_size,), float("inf"), dtype=key.dtype, device=key.device))
        gathered = comm.all_gather(samples, sizes=[sample_size] * world)
        # phase 3: splitter selection (every rank does what the designated processor would broadcast)
        # phase 4: place the splitters: the local array falls into `world` consecutive partitions
        sizes = []
        for i, c in enumerate(cols):
            combined = local_sort([torch.cat(gathered[i])])[0]
            spl = combined[_index_tensor(splitter_positions(sample_size, world), combined.device)]
            cut = [0] + [int(x) for x in partition_points(c[0], spl)] + [c[0].numel()]
            comm.host_syncs += 1                                   # the splitter positions come back to the host
            sizes.append([cut[d + 1] - cut[d] for d in range(world)])
        counts = comm.all_gather_ints(sizes)[0]                    # counts[src][dst], the same on every rank
        received = comm.exchange([pack_records(c) for c in cols], counts)
        mark("exchange")
        # phase 5: merge = the partitions in source order, sorted again (stable: ties keep source order)
        cols = []
        for rec in received:
            c = unpack_records(rec, like)
            cols.append(local_sort(c) if c[0].numel() > 1 else c)
        mark("merge_sort")
        # redistribution: exclusive scan of the counts, all-to-all of the chunks that belong
        # elsewhere.  What every rank holds now is a column sum of the matrix every rank already has.
        have = [sum(counts[src][d] for src in range(world)) for d in range(world)]
        plan = redistribution_plan(have, want)
        received = comm.exchange([pack_records(c) for c in cols], plan)      # chunks arrive in source order = global order
        cols = [unpack_records(rec, like) for rec in received]
        mark("redistribute")
    return cols


# ------------------------------------------------------------------------------------------------ the stepper
class ShardedStepper:
    """hmc.OrbitStepper over the ranks of a communicator.  ``shards`` = one dict(r, v_r, v_t, m, id) of CUDA tensors
    per local rank: the rank's range of the (unsorted) cluster, the ranges in rank order making up the whole cluster
    in the order a single-GPU stepper would be given it.  After step() the state of rank d is the stars of its range
    of the sorted order with their new coordinates, exactly as hmc.OrbitStepper's state cut at the same places."""

    def __init__(self, comm, shards: List[dict], seed: int, G: float = 1.0, sample_size: int = 256,
                 n_total: Optional[int] = None, push_tables: Optional[bool] = None):
        """push_tables: fuse the replicated table's all-gather into the potential scan (needs a communicator with
        table_views; default: whenever it has one)."""
        from . import hmc
        self.push_tables = push_tables            # None: whenever the communicator can hand out the copies
        self.hmc = hmc
        self.comm, self.seed, self.G, self.sample_size, self.step_index = comm, seed, G, sample_size, 0
        self.state = [dict(s) for s in shards]
        if n_total is None:
            sizes = comm.all_gather_ints([[s["r"].numel()] for s in shards])[0]
            n_total = sum(v[0] for v in sizes)
        self.n = n_total
        self.want = partition_counts(self.n, comm.world)
        self.offsets = exclusive_scan(self.want)
        self.counters = [hmc.alloc_counters(s["r"].device) for s in shards]
        self.workspace = [hmc.alloc_workspace(self.n, s["r"].device) for s in shards]
        self.last = None
        self.marks = None            # set to [] to have step() append (phase name, CUDA event) pairs (bench.py)

    def _mark(self, name):
        if self.marks is not None:
            ev = torch.cuda.Event(enable_timing=True)
            ev.record()
            self.marks.append((name, ev))

    def _local_sort(self, ws):
        hmc = self.hmc

        def sort(columns):
            key, rest = columns[0], list(columns[1:])
            ids = next((c for c in rest if c.dtype == torch.int32), None)
            f64 = [c for c in rest if c.dtype == torch.float64]
            rs, _, cs, ids_s = hmc.hmc_sort_by_radius(key, f64, ids, workspace=ws)
            it = iter(cs)
            return [rs] + [ids_s if c.dtype == torch.int32 else next(it) for c in rest]
        return sort

    def step(self):
        hmc, comm = self.hmc, self.comm
        L = len(comm.local_ranks)
        cols = [[s["r"], s["v_r"], s["v_t"], s["m"], s["id"]] for s in self.state]
        # S1: sample sort + redistribution.  One workspace serves all local ranks' sorts (they run one after another).
        sort = self._local_sort(self.workspace[0])
        self._mark("start")
        cols = sample_sort(comm, cols, self.sample_size, self.want, sort,
                           lambda keys, spl: hmc.hmc_partition_points(keys, spl).cpu().tolist(), self._mark)
        # S2: shard totals -> all-gather -> local scan with what lies before and after
        totals = [hmc.hmc_potential_totals(c[0], c[3], workspace=self.workspace[i]) for i, c in enumerate(cols)]
        all_totals = [torch.cat(t) for t in comm.all_gather(totals, sizes=[4] * comm.world)]
        tabs = None
        if self.push_tables is not False and hasattr(comm, "table_views"):
            tabs = comm.table_views(self.n, cols[0][0].device)
        if self.push_tables and tabs is None:
            raise RuntimeError("push_tables=True, but the communicator cannot hand out the copies of the table")
        if tabs is not None:
            # the replicated table filled by the scans themselves: rank d's launch stores its slice of
            # (r, Phi, M) into every rank's copy as it produces it (hmc_potential_shard_push)
            pots = []
            for i, (c, rank) in enumerate(zip(cols, comm.local_ranks)):
                lo, hi = self.offsets[rank], self.offsets[rank] + self.want[rank]
                mine, peers = tabs[i]
                others = [(t["r"][lo:hi], t["phi"][lo:hi], t["m_cum"][lo:hi]) for t in peers]
                mine["r"][lo:hi].copy_(c[0])
                pots.append(hmc.hmc_potential_shard(c[0], c[3], rank, all_totals[i], self.G, phi=mine["phi"][lo:hi],
                                                    m_cum=mine["m_cum"][lo:hi], workspace=self.workspace[i], push=others))
            comm.tables_complete()
            table_r, table_phi, table_m = [t[0]["r"] for t in tabs], [t[0]["phi"] for t in tabs], [t[0]["m_cum"] for t in tabs]
            self.pushed = True
        else:
            self.pushed = False
            pots = [hmc.hmc_potential_shard(c[0], c[3], rank, all_totals[i], self.G, workspace=self.workspace[i])
                    for i, (c, rank) in enumerate(zip(cols, comm.local_ranks))]
            # the replicated table
            table_r = [torch.cat(t) for t in comm.all_gather([c[0] for c in cols], sizes=self.want)]
            table_phi = [torch.cat(t) for t in comm.all_gather([p[0] for p in pots], sizes=self.want)]
            table_m = [torch.cat(t) for t in comm.all_gather([p[1] for p in pots], sizes=self.want)]
        self._mark("potential_and_table")
        # S3 / S4 on the rank's own range: no communication
        new_state, last = [], []
        for i, rank in enumerate(comm.local_ranks):
            r, vr, vt, m, ids = cols[i]
            first = self.offsets[rank]
            if r.numel():
                tp = hmc.hmc_orbit_turning_points(table_r[i], vr, vt, table_phi[i], table_m[i], self.G, first=first,
                                                  counters=self.counters[i], workspace=self.workspace[i])
                sm = hmc.hmc_sample_new_radius(table_r[i], table_phi[i], table_m[i], vr, vt, tp, ids, self.seed,
                                               self.step_index, self.G, first=first, counters=self.counters[i],
                                               workspace=self.workspace[i], reuse_tables=True)
            else:
                tp, sm = hmc.alloc_turning_points(0, r.device), hmc.alloc_sample(0, r.device)
            new_state.append(dict(r=sm["r_new"], v_r=sm["v_r_new"], v_t=sm["v_t_new"], m=m, id=ids))
            last.append(dict(r=r, v_r=vr, v_t=vt, phi=pots[i][0], m_cum=pots[i][1], tp=tp, sample=sm))
        self._mark("orbit")
        self.state, self.last = new_state, last
        self.step_index += 1


def split_cluster(cluster: dict, world: int) -> List[dict]:
    """Cut the arrays of a cluster (any indexable columns of equal length) into the decomposition's ranges."""
    n = len(cluster["r"])
    counts = partition_counts(n, world)
    offs = exclusive_scan(counts)
    return [{k: v[o:o + c] for k, v in cluster.items()} for o, c in zip(offs, counts)]
