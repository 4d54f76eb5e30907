#!/usr/bin/env python
"""bench.py — throughput of the SPH hot path (libccake, C ABI) on B200, with the oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A "step" is one full RK step (ccake_step(ctx, 1)): every row a1-a8 of SURVEY.md §8(a) twice (RK2 midpoint) over
one batch of synthetic particles; row a9 (conserved totals) closes the run.  The default workload is BASELINE.json's
config 4 ("C4": (3+1)D viscous, DNMR shear + bulk + BSQ diffusion, 1,984,000 particles in 10 seeded event tiles,
100x32^3 EoS table with 11 columns) — the configuration `north_star` quotes its target on.  State (416 MB) and work
arrays are far larger than the 126 MB L2, so consecutive steps see cold data ("inputs larger than L2").

N > 1 (torchrun): the path shards by independent event tiles with no data-path collective — every rank runs its
own batch of tiles (different seeds), "scaling": "weak"; the only collectives are the barrier and the max-over-ranks
of the device time (NCCL).

One JSON line on stdout (rank 0).  DESIGN.md §"Measurement" defines every figure.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "SPH particle-updates/s (fp64)"
UNIT = "particle-updates/s"

# algorithmic work per unit (DESIGN.md §"Algorithmic work")
FLOP_SMOOTH_PER_PAIR = 35.0


def flop_grad_per_pair(D, visc, diff):
    terms = D + D * D + D          # FP, DU, div v
    if visc:
        terms += D * D             # FB
    if diff:
        terms += 6 * D             # grad alpha_q, FK_q
    return 34.0 + 3.0 * terms


FP64_NOMINAL_TFLOPS = 148 * 4 * 16 * 2 * 1.965e9 / 1e12   # 148 SMs x 4 sub-partitions x 16 DFMA lanes x 2 flop x 1.965 GHz


def ncu_traffic(config, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a pair kernel, read from the committed ncu --set full
    summary of this round (profiles/r2_traffic.txt: lines "config kernel bytes", written from the capture named in
    profiles/r2_README.md); None when the file has no entry for this workload — never a constant pasted into this script."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.txt")
    try:
        with open(p) as fh:
            for line in fh:
                t = line.split()
                if len(t) == 3 and t[0] == config and t[1] == kernel:
                    return float(t[2])
    except Exception:
        pass
    return None


_TABLES = {}


def shared_table():
    """C3, C4 and C4' read the same 100x32^3x11 table: build it once per process."""
    from paper_2511_22852_b200 import workloads as W
    if "t" not in _TABLES:
        _TABLES["t"] = W.make_eos_table(100, 32, with_wq=True)
    return _TABLES["t"]


def make_workload(name, rank=0, tiles=None, world=1):
    """Workload of one rank: rank r of `world` evolves the event tiles sharding.tile_range gives it (weak scaling: every rank
    the same number of tiles, seeds by global tile number)."""
    from paper_2511_22852_b200 import workloads as W
    from paper_2511_22852_b200 import sharding
    world = max(world, rank + 1)

    def first_tile(per_rank):
        return sharding.tile_range(per_rank * world, rank, world).start
    if name == "C1":
        return W.config_c1()
    if name == "C2":
        return W.config_c2()
    if name == "C3":
        return W.config_c3(tile0=first_tile(4), table=shared_table())
    if name == "C4":
        return W.config_c4(K=tiles or 10, tile0=first_tile(tiles or 10), table=shared_table())
    if name == "C5":
        return W.config_c5(tile0=first_tile(13))
    if name == "C4p":
        return W.config_c4p(table=shared_table())
    raise SystemExit(f"unknown config {name}")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.path = tempfile.mktemp(suffix=".csv")
        self.proc = None
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(device), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.fh,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            with open(self.path) as fh:
                for line in fh:
                    f = [x.strip() for x in line.split(",")]
                    if len(f) < 9:
                        continue
                    try:
                        sm.append(float(f[1])); smax.append(float(f[2]))
                    except ValueError:
                        continue
                    for nm, v in zip(names, f[5:9]):
                        if v.lower().startswith("active"):
                            reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


def oracle_sample(name):
    """Bounded sample of the workload for the CPU oracle: one event tile of the tiled configs (the tiles are
    independent events separated by gaps > 2h, so one tile is a faithful 1/K sample); whole workload for C1, C2."""
    from paper_2511_22852_b200 import workloads as W
    if name == "C3":
        return W.config_c3(K=1), "1 of 4 event tiles (54,289 particles), 1 RK2 step"
    if name == "C4":
        return W.config_c4(K=1), "1 of 10 event tiles (198,400 particles), 1 RK2 step"
    if name == "C5":
        return W.config_c5(K=1, n_eta=5), "1 of 13 event tiles cut to 5 rapidity slices (353,780 particles), 1 RK2 step"
    if name == "C4p":
        return W.config_c4p(n_side=60), "a 60^3 sub-lattice of the 126^3 probe (216,000 particles), 1 RK2 step"
    w = make_workload(name)
    return w, f"whole workload ({w.n} particles), 1 RK2 step"


def time_oracle(name, steps, warmup):
    """The oracle as it stands, on this host's cores; returns (updates/s, ms per step, cores, sample text)."""
    import oracle as O
    w, what = oracle_sample(name)
    o = O.Oracle(**w.params)
    if w.table is not None:
        o.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
    o.load_particles(w.fields)
    for _ in range(warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(1)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return w.n * steps / dt, 1e3 * dt / steps, cores, what, w


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(1, min(args.steps, 3))
    val, ms, cores, what, w = time_oracle(args.config, steps, 0 if args.config in ("C4", "C5") else min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_text(args.config), "sample": what},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_text(name):
    return {
        "C1": "BASELINE.json configs[0]: (2+1)D ideal Cartesian, 2,500 particles, closed-form EoS, RK2",
        "C2": "BASELINE.json configs[1]: (2+1)D ideal BSQ Gubser, hyperbolic, 40,000 particles, table 100x32^3x8, RK2",
        "C3": "BASELINE.json configs[2]: (2+1)D viscous hyperbolic, 217,156 particles (4 event tiles), IS shear+bulk+diffusion, table 100x32^3x11, RK2",
        "C4": "BASELINE.json configs[3]: (3+1)D viscous hyperbolic, 1,984,000 particles (10 event tiles of 80x80x31), DNMR shear+bulk+BSQ diffusion, table 100x32^3x11, h=0.3, RK2",
        "C5": "BASELINE.json configs[4]: (3+1)D viscous hyperbolic, 19,316,388 particles (13 event tiles of 266x266x21), IS shear+bulk+diffusion, table 200x48^3x11, RK2",
        "C4p": "SURVEY.md §8(d) C4' sparse probe: (3+1)D viscous hyperbolic, 2,000,376 particles on a simple cubic 126^3 lattice (spacing 0.2244, ~80 neighbours at h=0.3), C4 physics, table 100x32^3x11, RK2",
    }[name]


def algorithmic_bytes_per_particle(D, visc, bulk, diff, ncols):
    """HBM bytes each kernel group must move per particle per substep: 8 B x (fields read once + written once);
    a neighbour's data counts once (DESIGN.md §"Algorithmic work").  Returns dict per group."""
    n_pi = (6 if D == 3 else 4) if visc else 0
    n_J = 3 * D if diff else 0
    n_state = 2 * D + 4 + (1 if bulk else 0) + n_pi + n_J
    sort = 8 * D + 4 * 2 * 2 * 3            # read r; 3 radix passes each read+write (key, value) u32
    smooth = 8 * (D + 5 + 5)                # read r, S, N_q, m; write 5 sums
    n_pair_in = 1 + D + D + (D * D if visc else 0) + (n_J + 3 if diff else 0)      # P, u, v, B, K, alpha
    thermo = 8 * (5 + D + (1 if bulk else 0) + n_pi + n_J) + 8 * (8 + 3 + n_pair_in)
    gather = 16 * ncols * 8
    n_grad_out = 2 * D + D * D + 1 + (3 * D + 3 if diff else 0)
    grad = 8 * (D + n_pair_in + n_grad_out)
    eom = 8 * (n_grad_out + 14 + 2 * n_state + n_state)    # sums, thermo, y_cur, y_base; write y_out
    return {"sort": sort, "smooth": smooth, "thermo": thermo + gather, "grad": grad, "eom": eom}


def short_run(name, steps, device, hbm):
    """A short device-timed run of another config (3 warm-up steps, `steps` timed steps from the loaded state, CUDA events
    on the library's stream): ms per RK2 step, updates/s, neighbours, the substep's algorithmic HBM fraction."""
    import torch
    from paper_2511_22852_b200 import binding as B
    w = make_workload(name)
    p = w.params
    stream = torch.cuda.Stream()
    sim = B.Ccake(device=device, stream=stream.cuda_stream, **p)
    dev = torch.device("cuda", device)
    if w.table is not None:
        sim.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], torch.as_tensor(w.table["data"], device=dev))
    dfields = {k: torch.as_tensor(np.ascontiguousarray(v), device=dev) for k, v in w.fields.items()}
    sim.load_particles(dfields)
    npairs = float(sim.conserved_totals()[14])
    for _ in range(3):
        sim.step(1)
    sim.synchronize(strict=False)
    sim.load_particles(dfields)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record()
        for _ in range(steps):
            sim.step(1)
        e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    rc = sim.synchronize(strict=False)
    sim.close()
    D = p["dim"]
    on = p["eom"] != 0
    ncols = len(w.table["col_ids"]) if w.table is not None else 0
    bpp = algorithmic_bytes_per_particle(D, on and bool(p["flags"] & 1), on and bool(p["flags"] & 2), on and bool(p["flags"] & 4), ncols)
    nsub = 2 if p["integrator"] == 2 else 4
    del dfields
    torch.cuda.empty_cache()
    return {"particles": w.n, "steps": steps, "ms_per_step": ms, "updates_per_s": w.n / (ms * 1e-3),
            "neighbours_per_particle": npairs / w.n, "substep_hbm_frac": sum(bpp.values()) * w.n * nsub / (ms * 1e-3) / 1e9 / hbm,
            "rc": rc}


def slab_probe(device, steps=5):
    """One C4 event (198,400 particles, 80 x 80 x 31) as a single context and as 2 slabs cut in x on the SAME GPU (the slabs
    run one after the other, so this measures what the decomposition costs — ghost recomputation, packing, the hand-over of
    the messages — not a speed-up): ms per RK2 step each, ghosts per slab, message bytes per step."""
    import torch
    from paper_2511_22852_b200 import binding as B
    from paper_2511_22852_b200 import sharding as S
    w = make_workload("C4", tiles=1)
    p = w.params
    dev = torch.device("cuda", device)
    stream = torch.cuda.Stream()
    tab = torch.as_tensor(w.table["data"], device=dev)

    def ctx():
        g = B.Ccake(device=device, stream=stream.cuda_stream, **p)
        g.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], tab)
        return g

    def timed(fn):
        fn(2)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record()
            fn(steps)
            e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps

    one = ctx()
    one.load_particles(w.fields)
    ms_one = timed(one.step)
    one.close()
    axis, K = 0, 2
    planes = S.slab_planes(w.fields[B.R1 + axis], K)
    out = {"event_particles": w.n, "slabs": K, "axis": "x", "ms_per_step_one_context": ms_one,
           "note": "2 contexts on one GPU, run one after the other: the cost of the decomposition, not a scaling number"}
    for narrow in (False, True):
        width = S.slab_halo_width(p["h"], p["dx0"], narrow)
        slabs = {}
        for k in range(K):
            lo, hi = S.slab_bounds(planes, k)
            sel = np.nonzero((w.fields[B.R1 + axis] >= lo) & (w.fields[B.R1 + axis] < hi))[0]
            g = ctx()
            g.slab_load({f: np.ascontiguousarray(v[sel]) for f, v in w.fields.items()}, sel.astype(np.uint32), int(0.9 * w.n), axis, lo, hi, width)
            slabs[k] = g
        drv = S.SlabDriver(slabs, K, 2, int(0.5 * w.n), lambda r, c: torch.zeros((r, c), dtype=torch.float64, device=dev), narrow=narrow)
        with torch.cuda.stream(stream):
            ms_slabs = timed(drv.step)
            b0 = drv.bytes_moved
            drv.step(1)
            per_step = drv.bytes_moved - b0
            drv.refresh_ghosts()
        info = [g.slab_info() for g in slabs.values()]
        for g in slabs.values():
            g.close()
        out["narrow_halo" if narrow else "wide_halo"] = {
            "halo_width_fm": width, "exchanges_per_substep": 2 if narrow else 1, "ms_per_step_slabs_same_gpu": ms_slabs,
            "owned_per_slab": [i[0] for i in info], "ghosts_per_slab": [i[1] + i[2] for i in info], "message_bytes_per_step": per_step}
    return out


def run_slabs(args):
    """--decomp slabs: ONE event (C4, a single tile of 198,400 particles) cut into one slab per rank along x; halos and
    migrants travel by torch.distributed send / recv (NCCL).  value = particles of the event x steps / device time (max
    over ranks): strong scaling of one event."""
    import torch
    import torch.distributed as dist
    from paper_2511_22852_b200 import binding as B
    from paper_2511_22852_b200 import sharding as S
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    w = make_workload("C4", tiles=1)
    p = w.params
    K = max(world, 2) if world == 1 else world
    axis = 0
    planes = S.slab_planes(w.fields[B.R1 + axis], K)
    width = S.slab_halo_width(p["h"], p["dx0"], narrow=True)
    stream = torch.cuda.Stream()
    tab = torch.as_tensor(w.table["data"], device=dev)
    slabs = {}
    for k in S.tile_range(K, rank, world):
        lo, hi = S.slab_bounds(planes, k)
        sel = np.nonzero((w.fields[B.R1 + axis] >= lo) & (w.fields[B.R1 + axis] < hi))[0]
        g = B.Ccake(device=local, stream=stream.cuda_stream, **p)
        g.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], tab)
        g.slab_load({f: np.ascontiguousarray(v[sel]) for f, v in w.fields.items()}, sel.astype(np.uint32), w.n, axis, lo, hi, width)
        slabs[k] = g
    drv = S.SlabDriver(slabs, K, 2, w.n // 2, lambda r, c: torch.zeros((r, c), dtype=torch.float64, device=dev), rank=rank, world=world,
                       narrow=True)
    with torch.cuda.stream(stream):
        drv.step(max(args.warmup, 3))
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        drv.step(args.steps)
        e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = S.reduce_max(e0.elapsed_time(e1), dev)
    launches = sum(g.launch_count() for g in slabs.values())
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": w.n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": "one C4 event (80 x 80 x 31 = 198,400 particles) cut into %d slabs along x, halo %.2f fm, gradient records exchanged" % (K, width),
                                     "decomposition": "slabs", "slabs": K}, "gpu_launches": launches}), flush=True)
    for g in slabs.values():
        g.close()
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_22852_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()   # fails loudly when libccake.so is missing

    w = make_workload(args.config, rank=rank, tiles=args.tiles, world=world)
    p = w.params
    D = p["dim"]
    visc, bulk, diff = bool(p["flags"] & 1) and p["eom"] != 0, bool(p["flags"] & 2) and p["eom"] != 0, bool(p["flags"] & 4) and p["eom"] != 0
    stream = torch.cuda.Stream()
    sim = B.Ccake(device=local, stream=stream.cuda_stream, **p)
    dev = torch.device("cuda", local)
    if w.table is not None:
        sim.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"],
                           torch.as_tensor(w.table["data"], device=dev))
    ids = list(w.fields.keys())
    dfields = {k: torch.as_tensor(np.ascontiguousarray(w.fields[k]), device=dev) for k in ids}
    sim.load_particles(dfields)
    npairs0 = float(sim.conserved_totals()[14])         # ordered neighbour pairs (excluding self) at the loaded state
    fp64_peak = B.measure_fp64_peak(local) if rank == 0 else None     # DFMA chains on every SM, before the timed region

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -----------------------------------------------------------------------------
    for _ in range(args.warmup):
        sim.step(1)
    sim.synchronize(strict=False)
    sim.load_particles(dfields)       # timed steps start from the loaded state, inputs resident in HBM
    sim.launch_count()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record()
        for _ in range(args.steps):
            sim.step(1)               # the library replays its captured RK step (one CUDA graph per step)
        e1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if sampler else None
    ms_total = e0.elapsed_time(e1)
    launches = sim.launch_count()
    rc = sim.synchronize(strict=False)
    # the same K steps once more from the loaded state with the library's per-kernel CUDA events (which need the kernels
    # launched one by one): the per-kernel durations behind `kernels` and `roofline`
    sim.load_particles(dfields)
    sim.enable_timing(True)
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            sim.step(1)
    kt = sim.kernel_times()           # per-substep averages of each kernel group, CUDA events on the same stream
    sim.enable_timing(False)
    sim.synchronize(strict=False)
    from paper_2511_22852_b200 import sharding
    ms_total = sharding.reduce_max(ms_total, dev)                 # max over ranks of the device time
    tot_n = torch.tensor([float(w.n)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tot_n, op=dist.ReduceOp.SUM)
    n_all = float(tot_n.item())
    value = n_all * args.steps / (ms_total * 1e-3)
    totals = sim.conserved_totals()
    npairs1 = float(totals[14])                         # ... and at the end of the timed region (the event expands)
    npairs = 0.5 * (npairs0 + npairs1)

    # ---- end to end through the C ABI with HOST buffers -----------------------------------------------------
    host_in = {k: torch.empty(w.n, dtype=torch.float64).pin_memory() for k in ids}
    for k in ids:
        host_in[k].numpy()[:] = w.fields[k]
    out_ids = B.state_field_ids(p)
    host_out = [torch.empty(w.n, dtype=torch.float64).pin_memory() for _ in out_ids]
    # every e2e step restarts from the loaded state, the densest one of the expanding event: its device time, for comparison
    sim.load_particles({k: host_in[k] for k in ids})
    sim.step(1)                                                 # first step after a load (unsorted store): warm-up
    sim.load_particles({k: host_in[k] for k in ids})
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        g0.record()
        sim.step(1)
        g1.record()
    sim.synchronize(strict=False)
    first_step_ms = g0.elapsed_time(g1)
    e2e_steps = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.load_particles({k: host_in[k] for k in ids})       # H2D inside the timed region
        sim.step(1)
        sim.read_fields(out_ids, out=host_out)                  # D2H inside the timed region (synchronises)
    torch.cuda.synchronize()
    dt_blocking = time.perf_counter() - t0
    e2e_blocking = n_all * e2e_steps / sharding.reduce_max(dt_blocking, dev)
    # the same loop as a user would pipeline it over independent events: ccake_stage_particles copies step n + 1's inputs in
    # on one copy stream and ccake_read_fields_async copies step n's result out on another while step n's / n + 1's kernels
    # run; two sets of pinned output buffers; every copy of every step starts and lands before the clock stops
    host_out2 = [torch.empty(w.n, dtype=torch.float64).pin_memory() for _ in out_ids]
    e2e_steps = max(2, min(args.steps, 10))
    barrier()
    t0 = time.perf_counter()
    staged = {k: host_in[k] for k in ids}
    sim.stage_particles(staged)                                 # H2D of the first step's inputs: inside the timed region
    for it in range(e2e_steps):
        sim.load_staged()
        if it + 1 < e2e_steps:
            sim.stage_particles(staged)                         # H2D of the next step's inputs, under this step's kernels
        sim.step(1)
        sim.read_fields_async(out_ids, host_out if it % 2 == 0 else host_out2)   # D2H inside the timed region, overlapped
    sim.read_fields_wait()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    e2e_value = n_all * e2e_steps / sharding.reduce_max(dt, dev)
    h2d = 8 * w.n * len(ids)
    d2h = 8 * w.n * len(out_ids)

    # ---- NEXT-1: offline EoS inversion on the device, beside the oracle's on a bounded sample ----
    eos_inv = None
    if rank == 0 and w.table is not None and not args.no_cpu:
        import oracle as O
        tb = w.table
        nodes = int(np.prod([len(a) for a in tb["axes"]]))
        sim.invert_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"])        # warm-up (allocations)
        t0 = time.perf_counter()
        sim.invert_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"])        # synchronous: returns with the table installed
        t_gpu = time.perf_counter() - t0
        P = O.make_params(**p)
        rng = np.random.default_rng(7)
        nsample = 20000
        ii = [rng.integers(0, len(a), nsample) for a in tb["axes"]]
        t0 = time.perf_counter()
        for k in range(nsample):
            sv = tb["axes"][0][ii[0][k]]
            O.eos_closed_form(P, sv, [tb["axes"][q + 1][ii[q + 1][k]] * sv for q in range(3)])
        t_cpu = time.perf_counter() - t0
        eos_inv = {"nodes": nodes, "columns": len(tb["col_ids"]), "gpu_ms": 1e3 * t_gpu, "gpu_nodes_per_s": nodes / t_gpu,
                   "cpu_oracle_nodes_per_s": nsample / t_cpu, "cpu_sample": f"{nsample} seeded nodes, 1 thread, through ctypes"}
        # rest of NEXT-1: the same target grid from a TABULATED forward EoS (BASELINE.json configs[1]: 100 x 32^3 (T, mu) grid),
        # damped 4-D Newton per node on the device; the oracle's inverter on a seeded sample of nodes beside it
        from paper_2511_22852_b200 import workloads as W
        ft = W.make_forward_table(100, 32)
        sim.invert_forward_table(ft["axes"], ft["data"], tb["axes"], tb["axis_kind"], tb["col_ids"])      # warm-up
        t0 = time.perf_counter()
        _, _, n_backup = sim.invert_forward_table(ft["axes"], ft["data"], tb["axes"], tb["axis_kind"], tb["col_ids"])
        t_fwd = time.perf_counter() - t0
        sv = tb["axes"][0][ii[0]]
        nv = [tb["axes"][q + 1][ii[q + 1]] * sv for q in range(3)]
        t0 = time.perf_counter()
        O.invert_forward_table(P, ft["axes"], ft["data"], sv, nv)
        t_cpu_fwd = time.perf_counter() - t0
        eos_inv["forward_table"] = {"forward_grid": [len(a) for a in ft["axes"]], "gpu_ms": 1e3 * t_fwd,
                                    "gpu_nodes_per_s": nodes / t_fwd, "nodes_on_backup_eos": n_backup,
                                    "cpu_oracle_nodes_per_s": nsample / t_cpu_fwd,
                                    "cpu_sample": f"{nsample} seeded nodes, OpenMP over nodes, {os.cpu_count()} cores",
                                    "note": "gpu_ms includes the 131 MB host-to-device copy of the forward table"}
        sim.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], torch.as_tensor(tb["data"], device=dev))

    # ---- NEXT-2: freeze-out element pass (one more pair pass over the cached lists and masks), device buffers ----
    fo_ms = None
    if rank == 0:
        buf = torch.empty(w.n, dtype=torch.float64, device=dev)
        sim.read_fields([B.FO_DSIGMA], out=[buf])                         # warm-up (lazy kernel load, allocation)
        sim.load_particles(dfields)                                       # invalidates the derived fields
        sim.read_fields([B.T], out=[buf])                                 # refresh of the derived fields
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            f0.record()
            sim.read_fields([B.FO_DSIGMA], out=[buf])
            f1.record()
        torch.cuda.synchronize()
        fo_ms = f0.elapsed_time(f1)

    # ---- NEXT-3 (part): source smearing of Eq. 35, 2,000 seeded partons per step onto all particles (host API) ----
    src_ms = None
    if rank == 0:
        rng = np.random.default_rng(35)
        nsrc = 2000
        rs = np.zeros((3, nsrc))
        for k in range(D):
            rs[k] = rng.uniform(np.min(w.fields[B.R1 + k]), np.max(w.fields[B.R1 + k]), nsrc)
        ps = rng.normal(0.0, 1.0, (4, nsrc))
        x0_now = float(sim.conserved_totals()[0])
        ts = np.full(nsrc, x0_now)
        sim.smear_sources(ps, rs, ts, 1.4, 0.62)
        t0 = time.perf_counter()
        sim.smear_sources(ps, rs, ts, 1.4, 0.62)
        src_ms = 1e3 * (time.perf_counter() - t0)

    if rank == 0:
        hbm, which = peaks()
        nsub = 2 if p["integrator"] == 2 else 4
        ncols = len(w.table["col_ids"]) if w.table is not None else 0
        bytes_pp = algorithmic_bytes_per_particle(D, visc, bulk, diff, ncols)
        names = ["sort", "pack", "smooth", "thermo", "grad", "eom"]
        groups = {nm: float(kt[i]) for i, nm in enumerate(names)}
        fg = flop_grad_per_pair(D, visc, diff)
        dom = max(("smooth", "grad"), key=lambda k: groups[k])
        flop = npairs * (fg if dom == "grad" else FLOP_SMOOTH_PER_PAIR)
        ach = flop / (groups[dom] * 1e-3) / 1e12 if groups[dom] > 0 else 0.0
        kernels = {}
        for nm in names:
            if nm == "pack" or groups[nm] <= 0:
                continue
            b = bytes_pp[nm] * w.n
            if nm == "thermo" and w.table is not None:
                # the 16-node stencils of neighbouring particles overlap: the gather is served by L1/L2, and what HBM has
                # to deliver is at most the table itself, once — counted so (an upper bound of the unique bytes)
                gather = 16 * ncols * 8 * w.n
                table_b = float(np.prod([len(a) for a in w.table["axes"]])) * ncols * 8
                b = b - gather + min(gather, table_b)
            kernels[nm] = {"ms": groups[nm], "alg_GB": b / 1e9, "GBps": b / (groups[nm] * 1e-3) / 1e9,
                           "hbm_frac": b / (groups[nm] * 1e-3) / 1e9 / hbm}
            if nm == "thermo" and w.table is not None:
                kernels[nm]["gather_GB_l2_served"] = gather / 1e9
                kernels[nm]["note"] = "alg_GB = per-particle streams + the table once; the stencil gather (16 nodes x %d columns x 8 B per particle, read as 96-byte node records) is L1/L2-served" % ncols
        kernels["smooth"]["TFLOPs"] = npairs * FLOP_SMOOTH_PER_PAIR / (groups["smooth"] * 1e-3) / 1e12
        kernels["grad"]["TFLOPs"] = npairs * fg / (groups["grad"] * 1e-3) / 1e12
        total_bytes = sum(bytes_pp.values()) * w.n
        cpu_val, cpu_ms, cores, what, _ = time_oracle(args.config, 1, 0) if not args.no_cpu else (None, None, 0, "skipped", None)
        sim.close()
        others = None
        if not args.no_others and world == 1:
            others = {}
            for nm, st in (("C1", 20), ("C2", 20), ("C3", 10), ("C4p", 5), ("C5", 2)):
                if nm != args.config:
                    others[nm] = short_run(nm, st, local, hbm)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_text(args.config), "particles_per_gpu": w.n, "rk_substeps_per_step": nsub,
                       "ordered_pairs_per_pass": npairs, "l2": "inputs larger than L2 (state + work arrays > 1 GB per substep)"},
            "pair_interactions_per_s": npairs * 2 * nsub * args.steps * world / (ms_total * 1e-3),
            "pair_interactions_unit": "ordered neighbour pairs (a, b), a != b, r_ab < 2h, per pair pass; 2 passes (a4, a6) per substep",
            "substep_hbm_frac": total_bytes * nsub / (ms_total / args.steps * 1e-3) / 1e9 / hbm,
            "roofline": {"bound": "alu", "kernel": {"grad": "gradient pass a6", "smooth": "smoothing pass a4"}[dom],
                         "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach / fp64_peak,
                         "peak_source": "measured in this run (ccake_measure_fp64_peak: fma.rn.f64 chains on every SM)",
                         "peak_nominal": FP64_NOMINAL_TFLOPS,
                         "traffic": ncu_traffic(args.config, dom) if args.tiles is None else None,
                         "traffic_unit": "bytes per launch (ncu --set full, profiles/r2_README.md)",
                         "algorithmic_bytes": bytes_pp[dom] * w.n,
                         "flop_per_pair": fg if dom == "grad" else FLOP_SMOOTH_PER_PAIR,
                         "flop_convention": "algorithmic: 34 geometry + 3 per accumulated term (DESIGN.md §5); the kernel executes ~24 FP64 instructions + 6 DMMA per 32 pair evaluations",
                         "ordered_pairs_at_load": npairs0, "ordered_pairs_after_run": npairs1,
                         "hbm_peak_GBps": hbm, "hbm_peak_source": which},
            "kernels": kernels,
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what,
                             "ms_per_step": cpu_ms},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "blocking_value": e2e_blocking,
                    "device_ms_of_that_step": first_step_ms, "ms_per_step": 1e3 * n_all / e2e_value,
                    "note": "value: ccake_stage_particles / ccake_load_staged -> step -> ccake_read_fields_async per step (the "
                            "host-to-device copy of step n + 1 and the read-back of step n overlap the kernels; every copy starts and "
                            "completes inside the timed region); blocking_value: ccake_load_particles -> step -> the synchronous "
                            "ccake_read_fields; every step restarts from the loaded state (the densest one of the event)"},
            "gpu_launches": launches,
            "eos_inversion": eos_inv,
            "freezeout_element_ms": fo_ms,
            "source_smearing": {"partons": 2000, "h_source": 1.4, "ms": src_ms,
                                "note": "ccake_smear_sources through host buffers, incl. 63 MB device-to-host"},
            "other_configs": others,
            "slab_decomposition": slab_probe(local) if (not args.no_others and world == 1) else None,
            "clocks": clocks,
            "status": {"rc": rc, "n_out_of_table": totals[11], "n_bad": totals[13], "x0": totals[0]},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5", "C4p"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--tiles", type=int, default=None, help="C4 only: number of event tiles (profiling runs; default 10)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--decomp", default="events", choices=["events", "slabs"],
                    help="events: every rank evolves its own event tiles (default, weak scaling); slabs: ONE event cut into one slab per rank")
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other configs (other_configs)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp == "slabs":
        run_slabs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
