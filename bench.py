#!/usr/bin/env python
"""bench.py — throughput of the whole hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--impl ours|reference]

One bench "step" = one OUTPUT INTERVAL of the workload: `bin_every` model time steps (met time
weighting, Philox + Box-Muller, trilinear gathers, advection + random walk, reflection, decay,
dry/wet deposition and the deposit scatter, compaction in c5) followed by the concentration
binning and the read-out of the concentration grid (and, once at the end, the deposition map).
Default workload: BASELINE.json configs[3] ("Large ensemble", c4: 1e8 particles, two nuclides,
1000x1000x30 concentration grid) — BASELINE.json's metric names no single config, so the largest
single-GPU configuration is used; its particle store (2.0 GB) is far larger than L2 (126 MB), so
no L2 flush is needed between timed steps.  With the defaults (W = 3, K = 9) the run IS the whole
12 h config: 3 warm-up hours + 9 timed hours.

Printed JSON line (rank 0): metric particle-steps/s = born particles x model steps / device time
(CUDA events on the launching stream, max over ranks), plus
  e2e          the same run through the host-buffer C-ABI calls: every step uploads the next
               hourly met snapshot from pinned host memory and reads the concentration grid back
  roofline     the step kernel (dominant): algorithmic lane-operations per launch / its average
               launch duration (CUDA events recorded by the library around each launch)
  binning      the binning kernel in GB/s of particle bytes consumed
  cpu_baseline the fp64 oracle, as it stands, on the host cores, on a pid-strided subsample
  clocks       nvidia-smi SM clock / throttle reasons sampled during the timed region
`--impl reference` times the oracle (the reference arm of this tier) on the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle_steps_per_s"
UNIT = "particle-steps/s"
# SURVEY.md §8(d) / DESIGN.md §6: algorithmic lane-operations per particle-step (FMA = 1), frozen
# before any tuning: 250 with one met snapshot, 310 with time interpolation (the figure stays 310
# although the kernel now samples a time-blended buffer: the budget is implementation-independent).
LANE_OPS_STATIC, LANE_OPS_TIME = 250.0, 310.0
SMS, LANES_PER_SM = 148, 128          # 4 SMSP x 32 lanes: one warp instruction per clock per SMSP
LAUNCH_STEPS = 16                     # model steps fused per step-kernel launch (csrc kMaxFused)
# dram__bytes_read.sum + dram__bytes_write.sum of one captured step-kernel launch, bytes (profiles/r01c_c4_step_kernel_ncu.md)
NCU_TRAFFIC = {"c4": 4.069e9 + 1.985e9}   # launch 171 of `bench.py --steps 1 --warmup 3`: 16 steps x 3.16e7 particles, z-pair texels (profiles/r01c_c4_step_kernel_ncu.md, r01d)
ORACLE_STRIDE = {"c1": 1, "c2": 40, "c2_eq3": 40, "c3": 400, "c3_hdep80": 400, "c4": 4000, "c5": 1}
ORACLE_SCALE_C5 = 1.0e-3              # c5 cannot be pid-strided (capacity couples particles): 1/1000 scale


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# ------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is not None:
            time.sleep(0.15)
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------ workload helpers
def make_workload(name: str, scale: float, world: int, rank: int):
    """The BASELINE config `name`; with world > 1 the ensemble is `world` times larger and rank r
    simulates the global particle ids r, r + world, ... (weak scaling)."""
    from workloads import make
    w = make(name, scale=scale)
    if world > 1:
        r = w.release
        if r.n_particles > 0:
            cap = w.capacity
            r.n_particles *= world
            r.total_activity = [a * world for a in r.total_activity]
            r.pid_offset, r.pid_stride = rank, world
            w = w.replace(capacity=cap)
        else:                                  # rate mode (c5): independent replicas, different seeds
            w = w.replace(seed=w.seed + 1000 * rank)
    return w


def born_steps(w, s0: int, s1: int) -> float:
    """Born particle x model step pairs for model steps s0 <= n < s1 (R9 closed form, local ids)."""
    r = w.release
    start = int(math.ceil(r.t_start / w.dt))
    S = max(1, int(math.ceil((r.t_end - r.t_start) / w.dt)))
    tot = 0
    if r.n_particles > 0:
        N = r.n_particles
        for n in range(s0, s1):
            if n < start:
                continue
            B = N if n - start + 1 >= S else min(N, -(-(n - start + 1) * N // S))
            tot += 0 if B <= r.pid_offset else (B - r.pid_offset + r.pid_stride - 1) // r.pid_stride
    else:
        c = int(round(r.rate * w.dt))
        for n in range(s0, s1):
            if n >= start:
                tot += min(w.capacity, c * min(n - start + 1, S))
    return float(tot)


# ------------------------------------------------------------------ the oracle legs
def oracle_leg(name: str, scale: float, interval: int, warmup: int, steps: int, budget_s: float, threads: int = 0):
    """Run the fp64 oracle (as it stands) on a bounded sample of the workload: every
    ORACLE_STRIDE-th particle id (exact subset: particles are independent and Philox is keyed by
    the id), the same intervals as the CUDA arm.  Returns particle-steps/s over the timed part."""
    from oracle import oracle as orc
    from workloads import make
    all_threads = orc.num_threads()
    if threads:
        orc.set_num_threads(threads)
    if name == "c5":
        w = make(name, scale=scale * ORACLE_SCALE_C5)
        sample = f"c5 at 1/{int(1 / ORACLE_SCALE_C5)} scale (injection rate and capacity), same grids/met/cadence"
    else:
        w = make(name, scale=scale)
        stride = ORACLE_STRIDE[name]
        w.release.pid_stride = stride
        n_local = len(range(0, w.release.n_particles, stride))
        w = w.replace(capacity=max(n_local, 1))
        sample = f"every {stride}th particle id of {name} ({n_local} particles), full grids and met"
    o = orc.OracleSim(w)
    o.step(warmup * interval)
    t0 = time.perf_counter()
    done = 0
    live = 0.0
    for i in range(steps):
        n0 = o.n
        o.step(interval)
        o.concentration()
        live += 0.5 * (n0 + o.n) * interval      # c5: exits make the live count data-dependent
        done += 1
        if budget_s and time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    units = live if name == "c5" else born_steps(w, warmup * interval, (warmup + done) * interval)
    sample += f"; {done} interval(s) of {interval} model steps after {warmup} warm-up interval(s)"
    used = orc.num_threads()
    if threads:
        orc.set_num_threads(all_threads)
    return units / dt, dt, done, used, sample


# ------------------------------------------------------------------ the CUDA arm
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_0912_3223_b200.build import build
    build()
    import paper_0912_3223_b200 as lpm

    # measured denominators (lpm_probe micro-benchmarks, outside every timed region)
    probes = {}
    if rank == 0 and not args.no_probes:
        for key, kind, fp in (("ffma_lane_ops_per_s", "ffma", 0), ("imad_lop_lane_ops_per_s", "imad_lop", 0),
                              ("l1_gather_sectors_per_s", "gather", 64 << 10), ("l2_gather_sectors_per_s", "gather", 64 << 20),
                              ("red_f64_l2_resident_per_s", "red_f64", 16 << 20), ("red_f64_600MB_per_s", "red_f64", 600 << 20),
                              ("red_same_address_per_s", "red_same", 0), ("shared_atomic_per_s", "atoms", 0)):
            probes[key] = lpm.probe(kind, fp, scratch_bytes=1 << 30 if fp > (1 << 28) else 1 << 28)
        torch.cuda.empty_cache()

    w = make_workload(args.workload, args.scale, world, rank)
    interval = w.bin_every
    W, K = args.warmup, args.steps
    g = w.cgrid
    pk = peaks()

    fields_host = torch.from_numpy(np.ascontiguousarray(w.fields())).pin_memory()   # [nt][nz][ny][nx][4]
    conc_host = torch.empty((w.K, g.nz, g.ny, g.nx), dtype=torch.float32).pin_memory()
    dep_host = torch.empty((w.K, g.ny, g.nx), dtype=torch.float32).pin_memory()
    snap_bytes = fields_host[0].numel() * 4

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def allreduce(t):
        if world > 1:
            dist.all_reduce(t)

    def snapshot_for(step_index):
        # the snapshot that closes the hour simulated next (needed from the first step of it)
        t = step_index * w.dt
        return min(w.nt - 1, int(math.floor((t - w.t0) / w.dt_snap)) + 1) if w.nt > 1 else 0

    # ---------------- leg 1: inputs resident in HBM ----------------
    fields_dev = fields_host.to("cuda", non_blocking=True)
    sim = lpm.Simulation(w, fields_dev=fields_dev, dep_mode=args.dep_mode, texel_pairs=args.texel_pairs, gather_sort=args.gather_sort,
                         steps_per_launch=args.steps_per_launch)
    pairs = sim.texel_pairs
    conc_dev = torch.empty((w.K, g.nz, g.ny, g.nx), dtype=torch.float32, device="cuda")
    dep_dev = torch.empty((w.K, g.ny, g.nx), dtype=torch.float32, device="cuda")
    for _ in range(W):
        sim.step(interval)
        sim.concentration(conc_dev)
        allreduce(conc_dev)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = sim.launch_count
    sim.set_timing(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    binned_compact = 0.0
    for _ in range(K):
        sim.step(interval)
        sim.concentration(conc_dev)
        allreduce(conc_dev)
        if w.compact:
            binned_compact += sim.num_active      # device-side live count (syncs at the interval boundary)
    sim.deposition(dep_dev)
    allreduce(dep_dev)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    tim = sim.get_timing()
    launches = sim.launch_count - launches0
    clocks = sampler.stop() if rank == 0 else None
    units_local = born_steps(w, W * interval, (W + K) * interval)
    if w.compact:
        units_local = tim["particle_steps"]
        tim["binned_particles"] = binned_compact
    total_mass = float(conc_dev.sum().item())
    del sim
    torch.cuda.empty_cache()

    # ---------------- leg 2: end to end through the host-buffer C-ABI calls ----------------
    fields_dev.zero_()
    sim = lpm.Simulation(w, fields_dev=fields_dev, dep_mode=args.dep_mode, texel_pairs=args.texel_pairs, gather_sort=args.gather_sort,
                         steps_per_launch=args.steps_per_launch)
    sim.upload_meteo(0, fields_host[0:1])
    uploaded = 0
    h2d = d2h = 0

    def e2e_step():
        nonlocal uploaded, h2d, d2h
        need = snapshot_for(sim.step_index)
        while uploaded < need:
            uploaded += 1
            sim.upload_meteo(uploaded, fields_host[uploaded:uploaded + 1])
            h2d += snap_bytes
        sim.step(interval)
        if world > 1:
            sim.concentration(conc_dev)
            allreduce(conc_dev)
            conc_host.copy_(conc_dev, non_blocking=False)
        else:
            sim.concentration_host(conc_host)
        d2h += conc_host.numel() * 4

    for _ in range(W):
        e2e_step()
    barrier()
    h2d = d2h = 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(K):
        e2e_step()
    if world > 1:
        sim.deposition(dep_dev)
        allreduce(dep_dev)
        dep_host.copy_(dep_dev)
    else:
        sim.deposition_host(dep_host)
    d2h += dep_host.numel() * 4
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    e2e_mass = float(conc_host.sum().item())
    del sim

    # ---------------- reduce over ranks ----------------
    if world > 1:
        t = torch.tensor([ms, ms_e2e, tim["step_ms"], tim["bin_ms"]], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, ms_e2e, step_ms, bin_ms = t.tolist()
        u = torch.tensor([units_local, tim["particle_steps"], tim["binned_particles"], float(launches)], device="cuda", dtype=torch.float64)
        dist.all_reduce(u)
        units, k_units, b_units, launches = u.tolist()
        launches = int(launches)
    else:
        units, k_units, b_units, step_ms, bin_ms = units_local, tim["particle_steps"], tim["binned_particles"], tim["step_ms"], tim["bin_ms"]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---------------- roofline of the dominant kernel (step) ----------------
    lane_ops = LANE_OPS_TIME if w.nt > 1 else LANE_OPS_STATIC
    n_launch = max(tim["step_launches"], 1)
    avg_ms = step_ms / n_launch
    achieved = lane_ops * (k_units / world) / n_launch / (avg_ms * 1e-3) / 1e12 if avg_ms > 0 else 0.0
    peak = SMS * LANES_PER_SM * pk["sm_max_mhz"] * 1e6 / 1e12
    state_bytes = 16 + 4 * (w.K - 1) + (4 if w.compact else 0)
    k_rate = (k_units / world) / (step_ms * 1e-3) if step_ms > 0 else 0.0      # particle-steps/s inside the step kernel
    fused = 1 if w.compact else (min(args.steps_per_launch, LAUNCH_STEPS) if args.steps_per_launch > 0 else LAUNCH_STEPS)
    hbm_per_ps = 2.0 * (state_bytes + (0 if w.compact else 4)) / fused          # state read + written once per launch (+ list entry)
    roofline = {
        "kernel": "step_compact_kernel" if w.compact else "step_slots_kernel", "bound": "alu",
        "achieved": achieved, "peak": peak, "unit": "Tlane-op/s", "frac": achieved / peak if peak else None,
        # dram__bytes_read + dram__bytes_write of ONE captured launch (profiles/r01c_*): not per average launch
        "traffic": NCU_TRAFFIC.get(args.workload),
        "lane_ops_per_particle_step": lane_ops, "avg_launch_ms": avg_ms, "launches": tim["step_launches"],
        "kernel_particle_steps_per_s": k_rate,
        "share_of_step": step_ms / ms if ms else None,
        "peak_source": f"{SMS} SMs x {LANES_PER_SM} lanes x {pk['sm_max_mhz']:.0f} MHz (clocks.max.sm, {pk['source']}): one warp "
                       "instruction per clock per SM sub-partition (DESIGN.md 6)",
        "frac_of_measured_ffma": achieved * 1e12 / probes["ffma_lane_ops_per_s"] if probes.get("ffma_lane_ops_per_s") else None,
        "hbm_side": {"bytes_per_particle_step": hbm_per_ps, "fused_steps_per_launch": fused, "hbm_peak_gbs": pk["hbm_gbs"],
                     "peak_source": pk["source"], "frac": k_rate * hbm_per_ps / (pk["hbm_gbs"] * 1e9)},
        # what ncu shows to be the binding unit (profiles/r01c_*): the L1 data pipe, one 32-byte sector per gathered
        # texel; achieved = gathers issued per second against the probe's L1-resident gather rate
        # (z-pair texels, B8: 4 gathers of one 32-byte sector each instead of 8 of 16 bytes)
        "l1_gather_side": {"gathers_per_particle_step": 4 if pairs else 8, "achieved_per_s": (4.0 if pairs else 8.0) * k_rate,
                           "peak_per_s": probes.get("l1_gather_sectors_per_s"),
                           "frac": (4.0 if pairs else 8.0) * k_rate / probes["l1_gather_sectors_per_s"] if probes.get("l1_gather_sectors_per_s") else None,
                           "note": "upper bound of the sector count: lanes that share a texel share a sector"},
    }
    bpp = 12 + 4 * w.K
    n_bin = b_units / world
    bin_bytes = bpp * n_bin
    grid_bytes = (4 + 8 * w.K) * g.nx * g.ny * g.nz
    red_rate = probes.get("red_f64_l2_resident_per_s")
    t_hbm = (bin_bytes + tim["bin_launches"] * grid_bytes) / (pk["hbm_gbs"] * 1e9)      # particles read + grids zeroed
    t_atom = (1 + w.K) * n_bin / red_rate if red_rate else None                          # one count + K sums per particle
    t_roof = max(t_hbm, t_atom) if t_atom else t_hbm
    binning = {"kernel": "bin_kernel", "gbs": bin_bytes / (bin_ms * 1e-3) / 1e9 if bin_ms > 0 else None,
               "avg_ms": bin_ms / max(tim["bin_launches"], 1), "launches": tim["bin_launches"],
               "bytes_per_particle": bpp, "particles": n_bin,
               "roofline": {"bound": "atomic" if t_atom and t_atom >= t_hbm else "hbm", "roof_ms": t_roof * 1e3, "measured_ms": bin_ms,
                            "frac": t_roof * 1e3 / bin_ms if bin_ms > 0 else None,
                            "hbm_ms": t_hbm * 1e3, "atomic_ms": t_atom * 1e3 if t_atom else None,
                            "atomics_per_particle": 1 + w.K,
                            "atomic_peak_per_s": red_rate, "atomic_peak_source": "lpm_probe red.global.add.f64, random addresses, "
                            "L2-resident 16 MB footprint (the plume's cells are L2-resident; over the full grid footprint the "
                            "random-address rate is red_f64_600MB_per_s)"},
               "note": "span = memsets of the count and sum grids + bin kernel"}

    # ---------------- cpu baseline (oracle, bounded sample) ----------------
    cpu = None
    if not args.no_cpu_baseline:
        v, dt, done, cores, sample = oracle_leg(args.workload, args.scale, interval, 0 if args.workload != "c5" else 0, W + K, 20.0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": dt}
        # the paper's own baseline was ONE thread: the same sample on one thread, at most ~8 s
        v1, dt1, done1, _, _ = oracle_leg(args.workload, args.scale, interval, 0, W + K, 8.0, threads=1)
        cpu["value_1_thread"] = v1
        cpu["intervals_1_thread"] = done1

    sim_hours = K * interval * w.dt / 3600.0
    line = {
        "metric": METRIC, "value": units / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload} (BASELINE.json configs[{ {'c1': 0, 'c2': 1, 'c2_eq3': 1, 'c3': 2, 'c3_hdep80': 2, 'c4': 3, 'c5': 4}[args.workload] }])",
                   "particles_per_gpu": w.capacity, "nuclides": w.K, "model_steps_per_bench_step": interval, "dt_s": w.dt,
                   "conc_grid": [g.nx, g.ny, g.nz], "met_grid": [w.mgrid.nx, w.mgrid.ny, w.mgrid.nz], "met_snapshots": w.nt,
                   "scale": args.scale, "dep_mode": args.dep_mode, "met_texels": "z-pair, 32 B (DESIGN.md B8)" if pairs else "16 B", "gather_sort": args.gather_sort, "steps_per_launch": args.steps_per_launch, "l2": "particle store larger than L2, no flush" if w.capacity * state_bytes > 126e6 else "inputs fit L2 (small config)",
                   "parallelism": f"pid-strided ensemble x{world}, grids all-reduced per output" if world > 1 else "single GPU"},
        "sim_hours_per_s": sim_hours / (ms * 1e-3),
        "e2e": {"value": units / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
                "ms_per_step": ms_e2e / K, "sim_hours_per_s": sim_hours / (ms_e2e * 1e-3)},
        "gpu_launches": launches,
        "roofline": roofline, "binning": binning, "measured_peaks": probes, "cpu_baseline": cpu, "clocks": clocks,
        "check": {"conc_sum_resident": total_mass, "conc_sum_e2e": e2e_mass},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------ the reference arm (oracle)
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make
    w = make(args.workload, scale=args.scale)
    interval = w.bin_every
    v, dt, done, cores, sample = oracle_leg(args.workload, args.scale, interval, args.warmup, args.steps, 0.0)
    g = w.cgrid
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3 / max(done, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "model_steps_per_bench_step": interval, "conc_grid": [g.nx, g.ny, g.nz]},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=9)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--workload", default="c4", choices=("c1", "c2", "c2_eq3", "c3", "c3_hdep80", "c4", "c5"))
    ap.add_argument("--scale", type=float, default=1.0, help="particle-count scale of the workload (1.0 = BASELINE size)")
    ap.add_argument("--dep-mode", type=int, default=0, choices=(0, 1), help="0 expected-mass deposition (default), 1 Bernoulli deposition (S 8(f)1)")
    ap.add_argument("--texel-pairs", type=int, default=0, choices=(-1, 0, 1), help="lpm_params.texel_pairs: 0 auto (default), 1 z-pair texels, -1 16-byte texels")
    ap.add_argument("--gather-sort", type=int, default=0, help="lpm_params.gather_sort: 0 auto (every 32 steps), p > 0 every p steps, -1 never")
    ap.add_argument("--steps-per-launch", type=int, default=0, help="lpm_params.steps_per_launch: 0 auto (16), m fuses up to min(m, 16) steps per launch")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probes", action="store_true", help="skip the lpm_probe micro-benchmarks (measured peaks)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"note: --warmup {args.warmup} < 3; timing rules ask for at least 3", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
