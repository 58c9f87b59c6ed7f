#!/usr/bin/env python
"""bench.py -- headline benchmark: checkerboard Metropolis spin updates/s on BASELINE.json config c3.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (BASELINE.json configs[2], SURVEY section 8d "c3"): 224^3 = 11 239 424 unit Heisenberg spins, simple cubic,
periodic, J = 1, cubic anisotropy Kc = 0.01, B = 0, T cycling through {0.5, 1.2, 1.44}, spins start uniformly random
on the sphere (seeded, synthetic), adaptive cone.  One STEP = ``--sweeps-per-step`` full Monte Carlo iterations
(red pass + black pass + controller + fused reductions = every row of the hot-path table) through mc_sweep().

Printed JSON line (one, by rank 0): see the task contract; `value` = spin updates/s with the state resident in HBM,
`e2e` = the same through the C ABI with host buffers (mc_set_spins H2D + mc_sweep + mc_observables D2H every step),
`roofline` = algorithmic HBM bytes of one colour-pass launch / its CUDA-event duration against the measured copy peak,
`cpu_baseline` = the fp64 oracle timed on this box's host cores on a bounded sample.

--impl reference times the oracle itself (there is no reference implementation to install: /root/reference holds only
the paper's text), on the same config/metric/unit, each step a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "spin updates/sec (Metropolis attempts) at 11.2M spins; achieved HBM GB/s vs peak"
UNIT = "spin-updates/s"
SHAPE = (224, 224, 224)
HAM = dict(J=1.0, Kc=0.01)
TEMPS = (0.5, 1.2, 1.44)
BYTES_PER_UPDATE = 36          # read self 12 + read other colour once 12 + write self 12
DEV_STATE_BYTES = 504          # sizeof(DevState): what mc_observables copies back


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def recorded_traffic(key="pass_kernel_dram_bytes_per_launch_warm"):
    """dram bytes per colour-pass launch from the committed ncu captures, if any (profiles/traffic.txt): `warm` = back to back
    as the timed region runs it (ncu --cache-control none), `cold` = ncu's default flushed-cache replay."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(path):
            t = line.split()
            if t and t[0] == key:
                return float(t[1])
    except Exception:
        pass
    return None


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None
        self.t0 = self.t1 = None

    def start(self):
        """Launch nvidia-smi (it needs a few hundred ms to come up: start it before the warm-up).  Rows are stamped on arrival;
        only those that arrive between mark_begin() and mark_end() are used."""
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True); self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [t.strip() for t in line.split(",")]))

    def mark_begin(self): self.t0 = time.perf_counter()
    def mark_end(self): self.t1 = time.perf_counter()
    def samples_in_window(self):
        return sum(1 for t, _ in self.rows if self.t0 is not None and t >= self.t0 and (self.t1 is None or t <= self.t1))

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try: self.proc.wait(timeout=2)
        except Exception: self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, r in self.rows:
            if self.t0 is not None and (t < self.t0 or (self.t1 is not None and t > self.t1)): continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"): reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_cores_used():
    return 1   # the oracle is single-threaded by construction


def time_oracle(shape, T, n_warm, n_timed, seed=42):
    """Oracle (as it stands) on this box's host cores: returns (updates/s, seconds, description)."""
    import oracle
    from paper_2103_03517_b200 import inputs
    N = shape[0] * shape[1] * shape[2]
    o = oracle.Oracle(*shape, seed=seed, cone0=0.5, adaptive=True, **HAM)
    o.set_spins(inputs.random_unit_spins(N, seed=seed))
    if n_warm: o.sweep(T, n_warm)
    t0 = time.perf_counter(); o.sweep(T, n_timed); dt = time.perf_counter() - t0
    return N * n_timed / dt, dt, f"{shape[0]}x{shape[1]}x{shape[2]} lattice, c3 Hamiltonian, T={T}, {n_warm} warm-up + {n_timed} timed sweeps ({N * n_timed} updates), 1 thread"


def run_reference(args, rank, world):
    if rank != 0:
        return 0
    total_steps = args.steps + args.warmup
    # bounded sample: the largest cubic lattice (multiple of 8, <= 224) such that the run ends within ~2.5 minutes at ~2.5 M updates/s
    budget_updates = 150.0 * 2.5e6 / max(1, total_steps)
    L = 224
    while L > 16 and L ** 3 > budget_updates: L -= 8
    import oracle
    from paper_2103_03517_b200 import inputs
    N = L ** 3
    o = oracle.Oracle(L, L, L, seed=42, cone0=0.5, adaptive=True, **HAM)
    o.set_spins(inputs.random_unit_spins(N, seed=42))
    for i in range(args.warmup): o.sweep(TEMPS[i % 3], 1)
    t0 = time.perf_counter()
    for i in range(args.steps): o.sweep(TEMPS[i % 3], 1)
    dt = time.perf_counter() - t0
    value = N * args.steps / dt
    sample = f"each step = 1 full sweep (red+black+controller+observables) of a {L}^3 lattice with the c3 Hamiltonian ({N} updates), oracle fp64, 1 thread"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "c3: 224^3 simple cubic periodic, J=1, Kc=0.01, T in {0.5,1.2,1.44}, random-sphere start, adaptive cone", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_cores_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def time_other_paths(binding, torch, local_rank, sweeps=100):
    """The other rows of the hot-path table: CUDA events on the handle's stream, state resident; per row 200 warm-up sweeps (the legs are separated by host-side set-up during which the GPU
    idles and drops its clocks), then the best of three timed runs of `sweeps` sweeps (context numbers next to the headline, whose own protocol is the contract's)."""
    out = {}

    def best_ms(run, warm):
        warm(); torch.cuda.synchronize()
        best = None
        for _ in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); run(); b.record(); torch.cuda.synchronize()
            t = a.elapsed_time(b); best = t if best is None else min(best, t)
        return best
    g = binding.Lattice(*SHAPE, Ku=0.05, cone0=0.5, adaptive=True, seed=42, device=f"cuda:{local_rank}")
    ms = best_ms(lambda: g.constrained_sweep(0.8, 0.6, 0.0, sweeps), lambda: g.constrained_sweep(0.8, 0.6, 0.0, 200))
    N = SHAPE[0] * SHAPE[1] * SHAPE[2]
    ups = N * sweeps / (ms * 1e-3)
    out["constrained_224^3_Ku0.05_T0.8_theta0.6"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps,
                                                     "algorithmic_GBs": BYTES_PER_UPDATE * ups / 1e9, "kernel": "pair_kernel<4, uniaxial> (gather; compile-time in-group rotation, 4 x 128 threads per SM)"}
    g.close()
    # granular film c5 (BASELINE.json configs[4]): 2048 x 2048 x 4, Voronoi grains, J = 0 across grains, per-grain axes
    from paper_2103_03517_b200 import inputs
    nx, ny, nz = 2048, 2048, 4
    mask, region, axes = inputs.voronoi_film(nx, ny, nz, 40, seed=42)
    g = binding.Lattice(nx, ny, nz, periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes,
                        cone0=0.5, adaptive=True, seed=42, device=f"cuda:{local_rank}")
    ms = best_ms(lambda: g.sweep(0.5, sweeps), lambda: g.sweep(0.5, 200))
    N5 = nx * ny * nz
    ups = N5 * sweeps / (ms * 1e-3)
    out["c5_film_2048x2048x4_T0.5"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps, "algorithmic_GBs": 39 * ups / 1e9,
                                       "kernel": "pass_kernel<4, uniaxial, masked> (generic)"}
    g.close()
    # bcc lattice: 176^3 conventional cells = 10.9 M spins, 8 neighbours, the two sublattices as colours
    Lb = 176
    g = binding.Lattice(Lb, Lb, Lb, Ku=0.01, cone0=0.5, adaptive=True, seed=42, structure="bcc", device=f"cuda:{local_rank}")
    g.init_spins(2)
    ms = best_ms(lambda: g.sweep(1.8, sweeps), lambda: g.sweep(1.8, 200))
    ups = g.N * sweeps / (ms * 1e-3)
    out["bcc_176^3_cells_Ku0.01_T1.8"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps, "algorithmic_GBs": BYTES_PER_UPDATE * ups / 1e9,
                                        "kernel": "pass_kernel<4, uniaxial, bcc> (generic gather, 8 neighbours)"}
    # the constrained pair pass on the same bcc lattice (Table A2 with the 8-bond field)
    g.init_spins(0)
    ms = best_ms(lambda: g.constrained_sweep(0.8, 0.6, 0.0, sweeps), lambda: g.constrained_sweep(0.8, 0.6, 0.0, 200))
    ups = g.N * sweeps / (ms * 1e-3)
    out["bcc_constrained_176^3_cells_T0.8_theta0.6"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps, "algorithmic_GBs": BYTES_PER_UPDATE * ups / 1e9,
                                                      "kernel": "pair_kernel<4, uniaxial, bcc>"}
    g.close()
    # fcc lattice: 140^3 conventional cells = 11.0 M spins, 12 neighbours, FOUR colour passes per sweep
    Lf = 140
    g = binding.Lattice(Lf, Lf, Lf, Ku=0.01, cone0=0.5, adaptive=True, seed=42, structure="fcc", device=f"cuda:{local_rank}")
    g.init_spins(2)
    ms = best_ms(lambda: g.sweep(2.8, sweeps), lambda: g.sweep(2.8, 200))
    ups = g.N * sweeps / (ms * 1e-3)
    out["fcc_140^3_cells_Ku0.01_T2.8"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps, "algorithmic_GBs": 60 * ups / 1e9,
                                        "kernel": "pass_kernel<4, uniaxial, fcc, colour> (generic gather, colour as a compile-time constant, 12 neighbours, 4 passes per sweep; 60 B per update: each pass reads the three other sublattices)"}
    g.close()
    # eight-colour lattices (reading C-32): 176^3 cells of eight sites = 43.6 M spins (523 MB of state), EIGHT colour passes per sweep,
    # bonds from a table; a site is bonded into six of the seven other sublattices: 24 B own + 6 x 12 B = 96 B per update
    for name, kw, T in (("hcp", dict(), 2.8), ("sc_nnn", dict(J2=0.3), 2.0)):
        Lc = 176
        g = binding.Lattice(Lc, Lc, Lc, Ku=0.01, cone0=0.5, adaptive=True, seed=42, structure=name, device=f"cuda:{local_rank}", **kw)
        g.init_spins(2)
        ms = best_ms(lambda: g.sweep(T, sweeps), lambda: g.sweep(T, 200))
        ups = g.N * sweeps / (ms * 1e-3)
        out[f"{name}_176^3_cells_Ku0.01_T{T}"] = {"value": ups, "unit": UNIT, "us_per_sweep": 1e3 * ms / sweeps, "algorithmic_GBs": 96 * ups / 1e9,
                                              "kernel": "pass_kernel<4, uniaxial, structure, colour> (gather through the bond table of the sublattice as a compile-time constant: 12 / 18 bonds, 8 passes per sweep; 96 B per update)"}
        g.close()
    # TWO independent replicas of the headline lattice on two streams of one GPU (the paper's production pattern is many independent
    # points): the gaps one replica leaves -- the last-block finalize between its sweeps, the fill and drain of its plane ring
    # -- are filled by the other replica's passes.  Aggregate updates/s over both, wall clock around a synchronised region.
    hs = [binding.Lattice(*SHAPE, seed=42 + k, cone0=0.5, adaptive=True, device=f"cuda:{local_rank}", stream=torch.cuda.Stream(), **HAM) for k in range(2)]
    for h in hs: h.init_spins(2); h.sweep(1.2, 30)
    torch.cuda.synchronize()
    best = None
    for rep in range(3):
        t0 = time.perf_counter()
        for c in range(8):
            for h in hs: h.sweep(1.2, 25)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0; best = dt if best is None else min(best, dt)
    ups = 2 * SHAPE[0] * SHAPE[1] * SHAPE[2] * 200 / best
    out["c3_two_replicas_on_two_streams"] = {"value": ups, "unit": UNIT, "us_per_sweep_of_both": 1e6 * best / 200, "algorithmic_GBs": BYTES_PER_UPDATE * ups / 1e9,
                                             "kernel": "tile_pass_kernel<2, 0, 112> of two handles interleaved by the hardware scheduler; not the headline (that is ONE lattice)"}
    for h in hs: h.close()
    # c2 (BASELINE.json configs[1]): 16 temperature points of 64^3.  A 64^3 colour pass fills a fraction of the GPU and a sweep is two
    # ~5 us launches whatever the size: one after another the points run launch-bound; replicas.run_points_concurrent runs them all
    # at once, one stream each, their sweeps replayed as CUDA graphs (same results bit for bit: tests/test_gpu_replicas.py).
    # Wall-clock around a synchronised region (16 streams), 1000 sweeps per point.
    from paper_2103_03517_b200 import replicas
    pts = [(0.1 * k, 64, 500, 500) for k in range(1, 17)]
    mk = lambda p, seed, device, stream: binding.Lattice(p[1], p[1], p[1], Ku=0.01, cone0=0.5, adaptive=True, seed=seed, device=device, stream=stream)
    ph = lambda p: [("sweep", p[0], p[2]), ("reset",), ("sweep", p[0], p[3])]
    def fin(g, p):
        m = g.observables().m; g.close(); return m
    dev = f"cuda:{local_rank}"
    replicas.run_points_concurrent(pts[:2], mk, ph, fin, device=dev)                     # warm-up (module load, graph machinery)
    torch.cuda.synchronize(); t0 = time.perf_counter()
    replicas.run_points_concurrent(pts, mk, ph, fin, device=dev)
    torch.cuda.synchronize(); t_conc = time.perf_counter() - t0
    t0 = time.perf_counter()
    for k, p in enumerate(pts):
        g = mk(p, 43 + k, dev, None); g.sweep(p[0], p[2]); g.reset_accumulators(); g.sweep(p[0], p[3]); fin(g, p)
    torch.cuda.synchronize(); t_ser = time.perf_counter() - t0
    work = 16 * 64 ** 3 * 1000
    out["c2_16_points_64^3_concurrent"] = {"value": work / t_conc, "unit": UNIT, "seconds": t_conc, "one_after_another": work / t_ser,
                                           "kernel": "tile_pass_kernel<1, 0, 32> on 16 streams, 50-sweep CUDA graphs replayed round robin; wall clock incl. handle creation, capture and read-back"}
    out["note"] = ("these legs run back to back after the headline: by then the GPU sits at its software power cap (SM clock ~1780 instead of "
                   "1965 MHz after about a second of continuous load), so they are SUSTAINED figures; each kernel timed alone for ~0.2 s "
                   "(BASELINE.md section 4, profiles/) runs 5-10 % faster")
    return out


def scan_sizes(args):
    """--scan-sizes L1,L2,...: unconstrained sweeps (c3 Hamiltonian, random start) on L^3 lattices with the planner's kernel and
    with the generic gather; one JSON line per size (the table of BASELINE.md section 4)."""
    import torch
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    peak, _ = measured_peaks()
    names = {1: "generic", 2: "staged", 3: "march"}
    for L in [int(v) for v in args.scan_sizes.split(",")]:
        N = L ** 3
        row = {"L": L, "spins": N}
        spins = inputs.random_unit_spins(N, seed=42)
        for label, path in (("auto", None), ("generic", binding.MC_PATH_GENERIC)):
            g = binding.Lattice(L, L, L, seed=42, cone0=0.5, adaptive=True, **HAM)
            if path is not None: g.debug_set_path(path)
            g.set_spins(spins); g.sweep(1.2, 30); torch.cuda.synchronize()
            n = max(20, min(200, int(2e9 / N)))
            best = None
            for rep in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); g.sweep(1.2, n); e1.record(); torch.cuda.synchronize()
                us = e0.elapsed_time(e1) * 1e3 / n
                best = us if best is None else min(best, us)
            ups = N / (best * 1e-6)
            row[label] = {"kernel": names[g.debug_get_path()], "us_per_sweep": round(best, 2), "updates_per_s": ups,
                          "frac_of_measured_peak": BYTES_PER_UPDATE * ups / 1e9 / peak}
            g.close()
        print(json.dumps(row), flush=True)
    return 0


def run_ours(args, rank, local_rank, world):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    torch.cuda.set_device(local_rank)
    from paper_2103_03517_b200 import replicas
    dist = replicas.init_distributed("nccl") if world > 1 else None      # plumbing only: barrier + max over ranks

    N = SHAPE[0] * SHAPE[1] * SHAPE[2]
    spp = args.sweeps_per_step
    # replicas: every rank owns an independent lattice (own seed) -- no data-path collective ("replicas only")
    g = binding.Lattice(*SHAPE, seed=42 + rank, cone0=0.5, adaptive=True, device=f"cuda:{local_rank}", **HAM)
    host = torch.from_numpy(inputs.random_unit_spins(N, seed=42 + rank)).pin_memory()
    host_np = host.numpy()
    g.set_spins(host_np)

    def barrier():
        if dist is not None: dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput
    sampler = ClockSampler(local_rank)
    if rank == 0: sampler.start()
    for i in range(args.warmup): g.sweep(TEMPS[i % 3], spp)
    barrier()
    l0 = g.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.mark_begin()
    ev0.record()
    for i in range(args.steps): g.sweep(TEMPS[i % 3], spp)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - l0
    clock_window = "timed region"
    if rank == 0 and sampler.proc and sampler.samples_in_window() < 3:
        # a short timed region (few steps) sees fewer than 3 samples at 50 ms: keep the SAME load running, untimed, until there are
        # (at most 2 s); the clocks are then those of the timed region plus its immediate continuation
        t_ext = time.perf_counter(); i = 0
        while sampler.samples_in_window() < 3 and time.perf_counter() - t_ext < 2.0:
            g.sweep(TEMPS[i % 3], spp); torch.cuda.synchronize(); i += 1
        clock_window = f"timed region + {1e3 * (time.perf_counter() - t_ext):.0f} ms of the same load run on (untimed)"
    sampler.mark_end()
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None: clocks["window"] = clock_window
    ms = replicas.max_over_ranks(ms, dist)
    value = world * N * spp * args.steps / (ms * 1e-3)

    # ---- end to end through the C ABI with host buffers: H2D of the state + sweeps + D2H of the observables, every step
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    g.set_spins(host_np); g.sweep(TEMPS[0], spp); g.observables()
    e2e_s = None
    for region in range(2):                 # two timed regions of e2e_steps steps each, the faster one is reported
        barrier()                           # (a single host hiccup -- page faults, the clock sampler exiting -- otherwise dominates 80 ms)
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            g.set_spins(host_np)            # pinned host -> device, layout conversion on the device
            g.sweep(TEMPS[i % 3], spp)
            ob = g.observables()            # synchronises; device -> host
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        e2e_s = dt if e2e_s is None else min(e2e_s, dt)
    e2e_s = replicas.max_over_ranks(e2e_s, dist)
    e2e_value = world * N * spp * e2e_steps / e2e_s
    # the same protocol double-buffered over TWO handles (own workspace and stream each): the upload of step i + 1 runs while the
    # sweeps of step i do; every step still uploads its 134.9 MB and reads its observables back inside the timed region
    e2e_pipe = None
    if world == 1:
        g2 = binding.Lattice(*SHAPE, seed=43 + rank, cone0=0.5, adaptive=True, device=f"cuda:{local_rank}", stream=torch.cuda.Stream(), **HAM)
        hs = (g, g2)
        for h in hs: h.set_spins(host_np); h.sweep(TEMPS[0], spp); h.observables()
        best = None
        for region in range(2):
            torch.cuda.synchronize(); t0 = time.perf_counter()
            for i in range(e2e_steps):
                h = hs[i & 1]
                if i >= 2: h.observables()              # result of step i - 2 (synchronises this handle only)
                h.set_spins(host_np)
                h.sweep(TEMPS[i % 3], spp)
            for h in hs: h.observables()
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            best = dt if best is None else min(best, dt)
        e2e_pipe = {"value": N * spp * e2e_steps / best, "unit": UNIT, "handles": 2,
                    "note": "two handles alternate: the H2D upload of a step overlaps the sweeps of the step before on the other handle"}
        g2.close()

    if rank != 0:
        g.close(); return 0

    peak, peak_src = measured_peaks()
    t_launch = ms * 1e-3 / launches                       # average duration of one colour-pass launch over the timed region
    alg_bytes_per_launch = BYTES_PER_UPDATE * (N // 2)    # one launch updates one colour
    achieved = alg_bytes_per_launch / t_launch / 1e9
    roofline = {"bound": "hbm", "kernel": "tile_pass_kernel<ANISO=2, FIELD=0, RT=112> (one colour pass = one launch)", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": recorded_traffic(), "traffic_cold_cache": recorded_traffic("pass_kernel_dram_bytes_per_launch_cold"), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes_per_launch, "avg_launch_us": t_launch * 1e6,
                "frac_of_nominal_8TBs": achieved / 8000.0}

    # ---- the other rows of the hot-path table at the same lattice (context next to the headline; not part of `value`)
    other = None
    if world == 1 and not args.no_other_paths:
        g.close()
        other = time_other_paths(binding, torch, local_rank)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, dt, sample = time_oracle(SHAPE, 1.2, 1, 2)
        cpu = {"value": v, "unit": UNIT, "cores": cpu_cores_used(), "kind": "oracle", "sample": sample, "seconds": dt}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "c3: 224^3 simple cubic periodic, J=1, Kc=0.01, T in {0.5,1.2,1.44} cycling per step, random-sphere start, adaptive cone",
                       "sweeps_per_step": spp, "spins": N, "state_bytes": N * 12, "l2_policy": "inputs larger than L2 (134.9 MB state vs 126 MB L2)",
                       "parallelism": f"replicas x{world} (no collective)", "final_m": ob.m, "final_acceptance": ob.last_acceptance},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": N * 12, "d2h_bytes_per_step": DEV_STATE_BYTES, "steps": e2e_steps, "regions": "best of 2",
                    "sweeps_per_step": spp, "pipelined": e2e_pipe, "note": "one state upload (mc_set_spins, pinned host) and one mc_observables read-back per STEP of sweeps_per_step sweeps; a per-sweep upload would be PCIe-bound (134.9 MB at ~50 GB/s = 2.7 ms against ~90 us of compute)"},
            "gpu_launches": launches,
            "roofline": roofline,
            "cpu_baseline": cpu,
            "other_paths": other}
    print(json.dumps(line), flush=True)
    g.close()
    if dist is not None: dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sweeps-per-step", type=int, default=100)
    ap.add_argument("--e2e-steps", type=int, default=6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-paths", action="store_true")
    ap.add_argument("--scan-sizes", default="", help="comma-separated L: time L^3 lattices with the planner's kernel and the generic pass, then exit")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                   # timing rule: W >= 3
    rank = int(os.environ.get("RANK", "0")); local_rank = int(os.environ.get("LOCAL_RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under a launcher: spawn one rank per GPU ourselves (what the driver's torchrun line does) and relay their output
        import socket
        sock = socket.socket(); sock.bind(("127.0.0.1", 0)); port = sock.getsockname()[1]; sock.close()
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    if args.scan_sizes:
        return scan_sizes(args)
    if args.impl == "reference":
        return run_reference(args, rank, world)
    return run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    sys.exit(main())
