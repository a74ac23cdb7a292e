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
12 h config: 3 warm-up hours + 9 timed hours.  Any other W, K walks the same config as a LOOP of its
output intervals (bench step i = interval i mod 12; every wrap restarts the run from step 0 inside the
timed region), so no bench step ever simulates an hour the config does not have.

Printed JSON line (rank 0): metric particle-steps/s = particle-steps the step kernels executed (born AND
active particles x model steps, counted on the device: a particle that has left the met box is inactive,
P:L108, and counts for nothing) / device time (CUDA events on the launching stream, max over ranks), plus
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
# before any tuning: 250.  (S§8(d) adds 60 for on-the-fly time interpolation "when a0 is not materialised"; here a0
# IS materialised - blend_kernel writes F(t_n) per met cell, < 1 lane-op per particle-step - so 250 applies throughout.)
LANE_OPS = 250.0
SMS, LANES_PER_SM = 148, 128          # 4 SMSP x 32 lanes: one warp instruction per clock per SMSP
LAUNCH_STEPS = 16                     # model steps fused per step-kernel launch (csrc kMaxFused)
# dram__bytes_read.sum + dram__bytes_write.sum of one captured step-kernel launch, bytes: NOT measured by this run, copied
# from the named ncu capture
NCU_TRAFFIC = {"c4": {"bytes": 2.605e9 + 1.173e9, "source": "profiles/r02_c4_step_kernel_ncu.md (r02b): launch 171 of `bench.py --steps 1 "
                      "--warmup 3`, 16 steps x 2.94e7 active particles, z-pair texels; 3.0 B algorithmic per particle-step = 1.4 GB"}}
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


# ------------------------------------------------------------------ the oracle legs
def oracle_leg(name: str, scale: float, interval: int, warmup: int, steps: int, budget_s: float, threads: int = 0):
    """Run the fp64 oracle (as it stands) on a bounded sample of the workload: every
    ORACLE_STRIDE-th particle id (exact subset: particles are independent and Philox is keyed by
    the id), the same looped intervals as the CUDA arm (a fresh run at every wrap of the config).
    Returns active particle-steps/s over the timed part (active = born and not yet inactive, as the CUDA arm counts)."""
    import numpy as np
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
    n_int = max(1, w.n_steps // interval)

    def active(o):
        return float((o.particles()["status"] == 0).sum()) if o.n else 0.0

    o = orc.OracleSim(w)
    for i in range(warmup):
        if i and i % n_int == 0:
            o = orc.OracleSim(w)
        o.step(interval)
    t0 = time.perf_counter()
    done = 0
    live = 0.0
    for i in range(warmup, warmup + steps):
        if i and i % n_int == 0:
            o = orc.OracleSim(w)
        a0 = active(o)
        o.step(interval)
        o.concentration()
        live += 0.5 * (a0 + active(o)) * interval      # trapezoid: births and exits make the active count vary inside an interval
        done += 1
        if budget_s and time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    sample += f"; {done} interval(s) of {interval} model steps after {warmup} warm-up interval(s) of the looped config"
    used = orc.num_threads()
    if threads:
        orc.set_num_threads(all_threads)
    return live / dt, dt, done, used, sample


# ------------------------------------------------------------------ the CUDA arm
class Looped:
    """The workload as a loop of its own output intervals: bench step i is interval (i mod n_int) of the config, and
    every wrap starts the run again from step 0 (lpm_restart on the same handle, inside the timed region), so that ANY --steps / --warmup stays on BASELINE.json's configuration: the run never simulates an hour
    the config does not have.  Per-handle timing totals are carried over the restarts."""

    KEYS = ("step_ms", "step_launches", "bin_ms", "bin_launches", "particle_steps", "binned_particles", "sort_ms", "sort_launches",
            "born_particle_steps", "bin_fused_launch_ms", "bin_fused_launches", "bin_fused_prev_launch_ms",
            "bin_fused_born_particle_steps", "bin_fused_prev_born_particle_steps")

    def __init__(self, sim, n_int, on_restart=None):
        self.sim, self.n_int, self.i, self.on_restart = sim, n_int, 0, on_restart
        self.tot = {k: 0.0 for k in self.KEYS}
        self.launches = 0
        self.timing = False
        self.l0 = sim.launch_count
        self.restarts = 0

    def begin_timing(self):
        self.timing = True
        self.tot = {k: 0.0 for k in self.KEYS}
        self.launches = 0
        self.l0 = self.sim.launch_count
        self.sim.set_timing(True)

    def _collect(self):
        if self.timing:
            t = self.sim.get_timing()
            for k in self.KEYS:
                self.tot[k] += t[k]
        self.launches += self.sim.launch_count - self.l0

    def next_interval(self):
        """Called before every bench step: wraps to a fresh run when the config is over."""
        if self.i and self.i % self.n_int == 0:
            self._collect()
            self.sim.restart()
            self.restarts += 1
            self.l0 = self.sim.launch_count
            if self.timing:
                self.sim.set_timing(True)
            if self.on_restart:
                self.on_restart()
        self.i += 1

    def end_timing(self):
        self._collect()
        self.l0 = self.sim.launch_count
        self.timing = False
        return dict(self.tot), self.launches


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
                              ("l1_gather32_sectors_per_s", "gather32", 64 << 10), ("smem_gather_1440B_lane_loads_per_s", "smem_gather", 1440),
                              ("smem_gather_16KB_lane_loads_per_s", "smem_gather", 16 << 10),
                              ("red_same_address_per_s", "red_same", 0), ("shared_atomic_per_s", "atoms", 0)):
            probes[key] = lpm.probe(kind, fp, scratch_bytes=1 << 28)
        torch.cuda.empty_cache()

    w = make_workload(args.workload, args.scale, world, rank)
    interval = w.bin_every
    n_int = max(1, w.n_steps // interval)        # output intervals of the config (c4: 12 hourly intervals)
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

    mk = dict(dep_mode=args.dep_mode, texel_pairs=args.texel_pairs, gather_sort=args.gather_sort, steps_per_launch=args.steps_per_launch)

    # ---------------- leg 1: inputs resident in HBM ----------------
    fields_dev = fields_host.to("cuda", non_blocking=True)
    sim = lpm.Simulation(w, fields_dev=fields_dev, **mk)
    pairs = sim.texel_pairs
    loop = Looped(sim, n_int)
    conc_dev = torch.empty((w.K, g.nz, g.ny, g.nx), dtype=torch.float32, device="cuda")
    dep_dev = torch.empty((w.K, g.ny, g.nx), dtype=torch.float32, device="cuda")

    def resident_step():
        loop.next_interval()
        sim.step(interval)
        sim.concentration(conc_dev)
        allreduce(conc_dev)

    for _ in range(W):
        resident_step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    loop.begin_timing()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(K):
        resident_step()
    sim.deposition(dep_dev)
    allreduce(dep_dev)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    tim, launches = loop.end_timing()
    clocks = sampler.stop() if rank == 0 else None
    total_mass = float(conc_dev.sum().item())
    touched = sim.touched_cells                       # cells that hold a particle in the last binning (untimed)
    # the stand-alone binning kernel (lpm_bin_now: what a caller gets outside the cadence), untimed region, on a FIXED state:
    # the end of the config (the run started again and taken through all its intervals), not wherever the timed loop stopped
    sim.restart()
    sim.step(n_int * interval)
    sim.set_timing(True)
    sb0, sb1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.bin_now()
    sb0.record()
    for _ in range(3):
        sim.bin_now()
    sb1.record()
    torch.cuda.synchronize()
    standalone_ms = sb0.elapsed_time(sb1) / 3.0
    standalone_n = sim.get_timing()["binned_particles"] / 4.0
    touched_sa = sim.touched_cells
    # fraction of the active particles that sit inside the met box: 1 by construction where leaving makes a particle inactive
    # (ABSORB: c3, c4, c5); measured on the final state of this leg where the boundary is OPEN (c1, c2)
    if w.boundary_mode == "absorb":
        in_domain, in_domain_how = 1.0, "by construction: a particle that leaves the met box is inactive (ABSORB) and is not stepped or counted"
    else:
        pp = sim.get_particles()
        xy, mg = pp["xyzq"], w.mgrid
        act = pp["status"] == 0
        ins = act & (xy[:, 0] >= mg.x0) & (xy[:, 0] < mg.x0 + mg.nx * mg.dx) & (xy[:, 1] >= mg.y0) & (xy[:, 1] < mg.y0 + mg.ny * mg.dy)
        in_domain = float(ins.sum().item()) / max(float(act.sum().item()), 1.0)
        in_domain_how = "OPEN boundary: active particles inside the met box / all active particles, on the final state of the resident leg"
        del pp, xy, act, ins
    restarts = loop.restarts
    del loop
    del sim
    torch.cuda.empty_cache()

    # ---------------- leg 2: end to end through the host-buffer C-ABI calls ----------------
    fields_dev.zero_()
    sim = lpm.Simulation(w, fields_dev=fields_dev, **mk)
    state = {"uploaded": 0, "h2d": 0, "d2h": 0}

    def first_snapshot():
        sim.upload_meteo(0, fields_host[0:1])
        state["uploaded"] = 0
        state["h2d"] += snap_bytes

    first_snapshot()
    loop = Looped(sim, n_int, on_restart=first_snapshot)

    def e2e_step():
        loop.next_interval()
        need = snapshot_for(sim.step_index)
        while state["uploaded"] < need:
            state["uploaded"] += 1
            u = state["uploaded"]
            sim.upload_meteo(u, fields_host[u:u + 1])
            state["h2d"] += snap_bytes
        sim.step(interval)
        if world > 1:
            sim.concentration(conc_dev)
            allreduce(conc_dev)
            conc_host.copy_(conc_dev, non_blocking=False)
        else:
            sim.concentration_host(conc_host)
        state["d2h"] += conc_host.numel() * 4

    for _ in range(W):
        e2e_step()
    barrier()
    state["h2d"] = state["d2h"] = 0
    loop.begin_timing()
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
    state["d2h"] += dep_host.numel() * 4
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    tim_e2e, _ = loop.end_timing()
    h2d, d2h = state["h2d"], state["d2h"]
    e2e_mass = float(conc_host.sum().item())
    del loop
    del sim
    torch.cuda.empty_cache()

    # the binning atomics' peak: random-address red.global.add.f64 over exactly the footprint the last binning touched
    if rank == 0 and not args.no_probes:
        fp = max(1 << 20, int(touched) * (4 + 8 * w.K))
        probes["red_f64_touched_footprint_per_s"] = lpm.probe("red_f64", fp, scratch_bytes=max(1 << 28, 1 << (fp - 1).bit_length()))
        probes["red_f64_touched_footprint_bytes"] = fp
        torch.cuda.empty_cache()

    # ---------------- reduce over ranks ----------------
    if world > 1:
        t = torch.tensor([ms, ms_e2e, tim["step_ms"], tim["bin_ms"]], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, ms_e2e, step_ms, bin_ms = t.tolist()
        u = torch.tensor([tim["particle_steps"], tim["binned_particles"], float(launches), tim["born_particle_steps"], tim_e2e["particle_steps"]],
                         device="cuda", dtype=torch.float64)
        dist.all_reduce(u)
        units, b_units, launches, born_units, units_e2e = u.tolist()
        launches = int(launches)
    else:
        units, b_units, step_ms, bin_ms = tim["particle_steps"], tim["binned_particles"], tim["step_ms"], tim["bin_ms"]
        born_units, units_e2e = tim["born_particle_steps"], tim_e2e["particle_steps"]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # the grid must hold something at the end of both legs: an empty grid means the run left the configuration
    if not (total_mass > 0.0 and e2e_mass > 0.0):
        raise SystemExit(f"bench.py: the concentration grid is empty at the end of the timed region "
                         f"(resident {total_mass}, e2e {e2e_mass}): not a valid measurement")

    # ---------------- roofline of the dominant kernel (step) ----------------
    lane_ops = LANE_OPS              # a0 is materialised (time-blended buffers), so every config is on the 250-op budget
    n_launch = max(tim["step_launches"], 1)
    avg_ms = step_ms / n_launch
    achieved = lane_ops * (units / world) / n_launch / (avg_ms * 1e-3) / 1e12 if avg_ms > 0 else 0.0
    peak = SMS * LANES_PER_SM * pk["sm_max_mhz"] * 1e6 / 1e12
    state_bytes = 16 + 4 * (w.K - 1) + (4 if w.compact else 0)
    k_rate = (units / world) / (step_ms * 1e-3) if step_ms > 0 else 0.0      # particle-steps/s inside the step kernel
    fused = 1 if w.compact else (min(args.steps_per_launch, LAUNCH_STEPS) if args.steps_per_launch > 0 else LAUNCH_STEPS)
    hbm_per_ps = 2.0 * (state_bytes + (0 if w.compact else 4)) / fused          # state read + written once per launch (+ list entry)
    roofline = {
        "kernel": "step_compact_kernel" if w.compact else "step_slots_kernel", "bound": "alu",
        "achieved": achieved, "peak": peak, "unit": "Tlane-op/s", "frac": achieved / peak if peak else None,
        # dram__bytes_read + dram__bytes_write of ONE captured launch (not measured in this run: from the named profile)
        "traffic": NCU_TRAFFIC.get(args.workload, {}).get("bytes"), "traffic_source": NCU_TRAFFIC.get(args.workload, {}).get("source"),
        "lane_ops_per_particle_step": lane_ops, "avg_launch_ms": avg_ms, "launches": tim["step_launches"],
        "kernel_particle_steps_per_s": k_rate,
        "share_of_step": step_ms / ms if ms else None,
        "peak_source": f"{SMS} SMs x {LANES_PER_SM} lanes x {pk['sm_max_mhz']:.0f} MHz (clocks.max.sm, {pk['source']}): one warp "
                       "instruction per clock per SM sub-partition (DESIGN.md 6)",
        "frac_of_measured_ffma": achieved * 1e12 / probes["ffma_lane_ops_per_s"] if probes.get("ffma_lane_ops_per_s") else None,
        "hbm_side": {"bytes_per_particle_step": hbm_per_ps, "fused_steps_per_launch": fused, "hbm_peak_gbs": pk["hbm_gbs"],
                     "peak_source": pk["source"], "frac": k_rate * hbm_per_ps / (pk["hbm_gbs"] * 1e9)},
        "l1_gather_side": {"gathers_per_particle_step": 4 if pairs else 8, "achieved_per_s": (4.0 if pairs else 8.0) * k_rate,
                           "peak_per_s": probes.get("l1_gather_sectors_per_s"),
                           "frac": (4.0 if pairs else 8.0) * k_rate / probes["l1_gather_sectors_per_s"] if probes.get("l1_gather_sectors_per_s") else None,
                           "note": "upper bound of the sector count: lanes that share a texel share a sector"},
    }
    # ---------------- binning (a8) ----------------
    # roofline of ANY binning design: the particle records at HBM peak (12 + 4 K bytes each) + the zeroing of the grids, or
    # one RED per touched cell and field at the measured random-address RED rate over exactly that footprint
    bpp = 12 + 4 * w.K
    grid_bytes = (4 + 8 * w.K) * g.nx * g.ny * g.nz
    red_rate = probes.get("red_f64_touched_footprint_per_s")

    def bin_roof(n_particles, n_launches, cells=None, memset=True):
        cells = touched if cells is None else cells
        t_hbm = (bpp * n_particles + (n_launches * grid_bytes if memset else 0)) / (pk["hbm_gbs"] * 1e9)
        t_atom = n_launches * cells * (1 + w.K) / red_rate if red_rate else None
        return t_hbm, t_atom, (max(t_hbm, t_atom) if t_atom else t_hbm)

    n_bin = b_units / world                                   # particles binned in the timed region (active, inside the grid)
    fused_n = tim["bin_fused_launches"]
    if fused_n:
        # slot-addressed store: the step launch that ends an output interval bins its particles from registers; what that
        # costs = (those launches) - (the launches right before them, per born particle-step), + the memset of the grids (the
        # timed "bin" span).  The last launch of an interval runs bin_every mod 16 steps (c2, c3: 8), its predecessor 16: the
        # predecessor's time is scaled by the ratio of the two launches' born particle-steps before it is subtracted (a
        # launch's fixed cost - state read and written once - does not scale, so a short last launch reads slightly HIGH)
        f_u, p_u = tim["bin_fused_born_particle_steps"], tim["bin_fused_prev_born_particle_steps"]
        unit_ratio = f_u / p_u if p_u > 0 else 1.0
        epi_ms = tim["bin_fused_launch_ms"] - tim["bin_fused_prev_launch_ms"] * unit_ratio
        measured_ms = max(epi_ms, 0.0) + bin_ms
        t_hbm, t_atom, t_roof = bin_roof(n_bin, fused_n)
        design = "fused into the step launch that ends each output interval (CTA-private table, one RED per touched cell, field and tile)"
    else:
        measured_ms = bin_ms
        t_hbm, t_atom, t_roof = bin_roof(n_bin, max(tim["bin_launches"], 1))
        design = "stand-alone bin_tile_kernel on the compact (physically sorted) store"
    sa_hbm, sa_atom, sa_roof = bin_roof(standalone_n, 1, cells=touched_sa)
    # the kernel work alone: particle records at HBM peak or one RED per touched cell and field, against the epilogue time -
    # no grid memset in the roof or in the measured time (where zeroing dominates the other fraction says nothing about the kernel)
    ko = None
    if fused_n and epi_ms > 0:
        k_hbm, k_atom, k_roof = bin_roof(n_bin, fused_n, memset=False)
        ko = {"roof_ms": k_roof * 1e3, "measured_ms": epi_ms, "frac": k_roof * 1e3 / epi_ms, "hbm_ms": k_hbm * 1e3,
              "atomic_ms": k_atom * 1e3 if k_atom else None, "per_binning_ms": epi_ms / fused_n}
    binning = {"kernel": "step_slots_kernel epilogue (bin_tile)" if fused_n else "bin_tile_kernel", "design": design,
               "gbs": bpp * n_bin / (measured_ms * 1e-3) / 1e9 if measured_ms > 0 else None,
               "measured_ms": measured_ms, "launches": fused_n or tim["bin_launches"], "memset_ms": bin_ms if fused_n else None,
               "epilogue_ms": epi_ms if fused_n else None, "epilogue_unit_ratio": unit_ratio if fused_n else None,
               "bytes_per_particle": bpp, "particles": n_bin, "touched_cells_last_binning": touched,
               "roofline": {"bound": "atomic" if t_atom and t_atom >= t_hbm else "hbm", "roof_ms": t_roof * 1e3, "measured_ms": measured_ms,
                            "frac": t_roof * 1e3 / measured_ms if measured_ms > 0 else None,
                            "hbm_ms": t_hbm * 1e3, "atomic_ms": t_atom * 1e3 if t_atom else None, "atomics_per_touched_cell": 1 + w.K,
                            "atomic_peak_per_s": red_rate, "atomic_peak_source": "lpm_probe red.global.add.f64, random addresses over "
                            "touched cells x (4 + 8 K) bytes (the footprint of the last binning, measured in this run)"},
               "kernel_only": ko,
               "standalone": {"kernel": "bin_tile_kernel (lpm_bin_now on the state at the END of the config, average of 3, outside the timed region)",
                              "touched_cells": touched_sa,
                              "ms": standalone_ms, "particles": standalone_n, "gbs": bpp * standalone_n / (standalone_ms * 1e-3) / 1e9,
                              "roof_ms": sa_roof * 1e3, "frac": sa_roof * 1e3 / standalone_ms if standalone_ms > 0 else None},
               "note": "fused: measured = sum over the intervals of (step launch with the epilogue - the step launch before it x epilogue_unit_ratio, "
                       "the ratio of the born particle-steps of the two launches) + the "
                       "memset of the grids; the two launches differ by 16 steps of births (< 0.1 % of the population).  Grids smaller than L2 (c2, c3) "
                       "are zeroed in L2, faster than the HBM copy peak the roofline uses: where the memset is the whole cost the fraction can read above 1"}

    # ---------------- cpu baseline (oracle, bounded sample) ----------------
    cpu = None
    if not args.no_cpu_baseline:
        ow = min(W + K, n_int)
        v, dt, done, cores, sample = oracle_leg(args.workload, args.scale, interval, 0, ow, 20.0)   # from step 0, at most ~20 s
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": dt}
        # the paper's own baseline was ONE thread: the same sample on one thread, at most ~8 s
        v1, dt1, done1, _, _ = oracle_leg(args.workload, args.scale, interval, 0, ow, 8.0, threads=1)
        cpu["value_1_thread"] = v1
        cpu["intervals_1_thread"] = done1

    sim_hours = K * interval * w.dt / 3600.0
    idx = {'c1': 0, 'c2': 1, 'c2_eq3': 1, 'c3': 2, 'c3_hdep80': 2, 'c4': 3, 'c5': 4}[args.workload]
    first = W % n_int
    line = {
        "metric": METRIC, "value": units / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload} (BASELINE.json configs[{idx}])",
                   "particles_per_gpu": w.capacity, "nuclides": w.K, "model_steps_per_bench_step": interval, "dt_s": w.dt,
                   "conc_grid": [g.nx, g.ny, g.nz], "met_grid": [w.mgrid.nx, w.mgrid.ny, w.mgrid.nz], "met_snapshots": w.nt,
                   "intervals_in_config": n_int, "timed_intervals": f"{K} consecutive output intervals of the looped config, starting at "
                   f"interval {first} of {n_int}; {restarts} restart(s) from step 0 inside the timed region",
                   "boundary": w.boundary_mode,
                   "scale": args.scale, "dep_mode": args.dep_mode, "met_texels": "z-pair, 32 B (DESIGN.md B8)" if pairs else "16 B", "gather_sort": args.gather_sort, "steps_per_launch": args.steps_per_launch, "l2": "particle store larger than L2, no flush" if w.capacity * state_bytes > 126e6 else "inputs fit L2 (small config)",
                   "parallelism": f"pid-strided ensemble x{world}, grids all-reduced per output" if world > 1 else "single GPU"},
        # unit of `value`: particle-steps the step kernels EXECUTED (born and still active: inside the met box, carrying
        # activity), counted on the device; particles that have left the domain are inactive and count for nothing
        "in_domain_fraction": in_domain, "in_domain_fraction_how": in_domain_how,
        "active_over_born": units / born_units if born_units else None,
        "born_particle_steps": born_units if born_units else None,
        # the same run in the units of round 1 (every BORN particle x step, whether or not it is still inside the domain): keeps the
        # rounds comparable across the OPEN -> ABSORB change of c3 / c4; not the headline
        "born_particle_steps_per_s": born_units / (ms * 1e-3) if born_units and ms > 0 else None,
        "sim_hours_per_s": sim_hours / (ms * 1e-3),
        "e2e": {"value": units_e2e / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
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


def spawn_ranks(n):
    """`python bench.py --gpus N` without torchrun: start the N ranks ourselves (the same launch the driver uses: one rank per
    GPU under torch.distributed.run, rendezvous on 127.0.0.1) and wait for them; rank 0 prints the JSON line."""
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count()
    if have < n:
        raise SystemExit(f"bench.py: --gpus {n} but only {have} CUDA device(s) are visible")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


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
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args.gpus)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
