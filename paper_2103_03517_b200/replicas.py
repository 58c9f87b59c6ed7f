"""Replica scheduler: independent Monte Carlo points over several GPUs.

The paper's multi-device mode is the "embarrassingly parallel approach": BASELINE.json's c2 is 16 temperature
points and c4 is 33 (T, theta) points, each from its own start, and the domain decomposition the paper speculates about
 buys nothing at these sizes.  So the path shards over POINTS, with no data-path
collective: every point runs on one device through one library handle, and only the few numbers a point returns travel.

Two ways to run, same assignment and seeds (results do not depend on the number of devices):
  * several processes, one per GPU (torchrun / bench.py --gpus N): `torch.distributed` carries the gather of the per-point
    results to rank 0 and the max-over-ranks of a time -- nothing else;
  * one process, several devices: one handle + stream per device; the library's calls are asynchronous, so the points of a
    round are enqueued on all devices first and read back afterwards.
A third way packs SMALL points onto one device: a 64^3 colour pass fills a fraction of a B200 and a sweep is two ~5 us launches
whatever the size, so c2's 16 temperature points run concurrently, each on its own stream, their sweeps captured once as CUDA
graphs of `chunk` sweeps and replayed round robin (`run_points_concurrent`: 21.6 -> 105 G updates/s on c2, results bit-identical to
the serial loop -- the library's sweep calls allocate nothing and never synchronise, so they can be captured).
This module holds no Monte Carlo arithmetic and never touches the oracle.
"""
from __future__ import annotations

import os
from typing import Callable, Optional, Sequence


def assign(n_points: int, world_size: int, costs: Optional[Sequence[float]] = None) -> list:
    """Which rank runs which point: a list of `world_size` lists of point indices (each ascending).
    Without costs: round robin (point k -> rank k mod world_size).  With costs (e.g. sweeps x sites per point): longest
    processing time first onto the least loaded rank (ties: lower rank), deterministic."""
    if world_size < 1 or n_points < 0:
        raise ValueError("need world_size >= 1 and n_points >= 0")
    if costs is None:
        return [list(range(r, n_points, world_size)) for r in range(world_size)]
    if len(costs) != n_points:
        raise ValueError("one cost per point")
    load = [0.0] * world_size
    out = [[] for _ in range(world_size)]
    for k in sorted(range(n_points), key=lambda i: (-float(costs[i]), i)):
        r = min(range(world_size), key=lambda i: (load[i], i))
        out[r].append(k); load[r] += float(costs[k])
    return [sorted(v) for v in out]


def point_seed(base_seed: int, k: int) -> int:
    """Seed of point k: base_seed + k + 1 (BASELINE.json c2: "seed 42 + k", k = 1..16) -- a function of the point alone,
    never of the rank that happens to run it."""
    return int(base_seed) + int(k) + 1


def world():
    """(rank, local_rank, world_size) from the launcher's environment (torchrun); (0, 0, 1) without one."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init_distributed(backend: Optional[str] = None):
    """Joins the process group the launcher describes (MASTER_ADDR / MASTER_PORT / RANK / WORLD_SIZE).  backend: "nccl" on
    GPU boxes (default when CUDA is there), "gloo" on CPU (the tests).  Returns torch.distributed, or None if WORLD_SIZE = 1."""
    rank, local_rank, ws = world()
    if ws == 1:
        return None
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        kw = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank); kw["device_id"] = torch.device(f"cuda:{local_rank}")
        dist.init_process_group(backend, **kw)
    return dist


def max_over_ranks(value: float, dist=None) -> float:
    """The slowest rank's time: multi-GPU numbers are the max over ranks of a device-measured time, never a wall clock."""
    if dist is None:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_points(points: Sequence, fn: Callable, base_seed: int = 42, costs: Optional[Sequence[float]] = None, dist=None,
               device: Optional[str] = None):
    """Multi-process mode.  Every rank runs `fn(point, seed, device)` for its share of `points` (see `assign`), in ascending
    point order; the results (anything picklable: a dict of floats) are gathered on rank 0 and returned there as a list in
    POINT order; other ranks return None.  With dist = None this is the plain serial loop."""
    rank, local_rank, ws = world() if dist is not None else (0, 0, 1)
    if dist is not None:
        rank, ws = dist.get_rank(), dist.get_world_size()
    if device is None:
        device = f"cuda:{local_rank}"
    mine = assign(len(points), ws, costs)[rank]
    local = [(k, fn(points[k], point_seed(base_seed, k), device)) for k in mine]
    if dist is None:
        return [r for _, r in sorted(local, key=lambda kv: kv[0])]
    gathered = [None] * ws if rank == 0 else None
    dist.gather_object(local, gathered, dst=0)
    if rank != 0:
        return None
    flat = sorted((kv for part in gathered for kv in part), key=lambda kv: kv[0])
    if [k for k, _ in flat] != list(range(len(points))):
        raise RuntimeError("replica gather lost or duplicated a point")
    return [r for _, r in flat]


def run_points_multi_device(points: Sequence, enqueue: Callable, collect: Callable, devices: Sequence[str], base_seed: int = 42):
    """Single-process mode: one handle and stream per device.  `enqueue(point, seed, device)` creates the handle on
    `device` and enqueues all its (asynchronous) sweeps, returning whatever `collect(handle)` needs to read the result
    back (the only synchronising call).  The points of a round -- one per device -- are all enqueued before the first is
    collected, so the devices work concurrently.  Returns the results in point order."""
    if not devices:
        raise ValueError("need at least one device")
    out = [None] * len(points)
    for start in range(0, len(points), len(devices)):
        batch = list(range(start, min(start + len(devices), len(points))))
        handles = [enqueue(points[k], point_seed(base_seed, k), devices[i]) for i, k in enumerate(batch)]
        for k, h in zip(batch, handles):
            out[k] = collect(h)
    return out


def split_chunks(n: int, chunk: int):
    """n sweeps as (whole chunks, remainder): n = q * chunk + r, 0 <= r < chunk."""
    if n < 0 or chunk < 1:
        raise ValueError("need n >= 0 and chunk >= 1")
    return n // chunk, n % chunk


def run_points_concurrent(points: Sequence, create: Callable, phases: Callable, collect: Callable, device: str = "cuda:0",
                          base_seed: int = 42, chunk: int = 50, use_graphs: bool = True, max_concurrent: int = 32):
    """One device, many small points at once.  `create(point, seed, device, stream)` returns a library handle bound to `stream`;
    `phases(point)` lists what the point runs, in order, as tuples
        ("sweep", T, n) | ("constrained", T, theta, phi, n) | ("reset",)
    and `collect(handle, point)` reads its result (the only synchronising call).  All points of a batch (at most `max_concurrent`)
    advance together: a phase of n sweeps is cut into chunks of `chunk` sweeps that are enqueued round robin over the points, each on
    its own stream, so the device interleaves them.  With `use_graphs` a chunk is captured ONCE per point and phase as a CUDA graph
    (the sweep calls only launch kernels: no allocation, no synchronisation) and replayed, which takes the per-launch host cost off
    the critical path.  The remainder n mod chunk runs as a plain call.  Every point's phases must have the same structure (kinds
    and counts); T, theta, phi may differ.  Results in point order, identical bit for bit to running the points one after another.
    """
    import torch
    out = [None] * len(points)
    for start in range(0, len(points), max_concurrent):
        batch = list(range(start, min(start + max_concurrent, len(points))))
        streams = [torch.cuda.Stream(device=device) for _ in batch]
        handles = [create(points[k], point_seed(base_seed, k), device, st) for k, st in zip(batch, streams)]
        plans = [list(phases(points[k])) for k in batch]
        if any([(ph[0], ph[-1] if ph[0] != "reset" else 0) for ph in pl] != [(ph[0], ph[-1] if ph[0] != "reset" else 0) for ph in plans[0]] for pl in plans):
            raise ValueError("the points of a concurrent batch must share the structure of their phases")

        def call(h, ph, n):
            if ph[0] == "sweep":
                h.sweep(ph[1], n)
            elif ph[0] == "constrained":
                h.constrained_sweep(ph[1], ph[2], ph[3], n)
            else:
                raise ValueError(f"unknown phase {ph[0]!r}")

        for i in range(len(plans[0])):
            kind = plans[0][i][0]
            if kind == "reset":
                for h in handles:
                    h.reset_accumulators()
                continue
            n = int(plans[0][i][-1])
            if kind == "constrained" and n > 0:
                # the first constrained sweep of a state aligns M with e_C (one synchronising measurement): not capturable
                for h, pl in zip(handles, plans):
                    call(h, pl[i], 1)
                n -= 1
            q, r = split_chunks(n, chunk)
            if use_graphs and q > 1:
                graphs = []
                for h, pl, st in zip(handles, plans, streams):
                    st.synchronize()
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=st, capture_error_mode="thread_local"):
                        call(h, pl[i], chunk)
                    graphs.append(g)
                for _ in range(q):
                    for g, st in zip(graphs, streams):
                        with torch.cuda.stream(st):
                            g.replay()
                for st in streams:
                    st.synchronize()                       # the graphs must outlive their last replay
                del graphs
            else:
                for _ in range(q):
                    for h, pl in zip(handles, plans):
                        call(h, pl[i], chunk)
            if r:
                for h, pl in zip(handles, plans):
                    call(h, pl[i], r)
        for k, h in zip(batch, handles):
            out[k] = collect(h, points[k])
    return out
