"""Shared test helpers: small custom workloads (inputs only, no method arithmetic)."""
import os

import numpy as np

from workloads import Grid, Nuclide, RainBox, Release, Workload

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

T_I131 = 8.02 * 86400.0


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


def custom(met_fn, *, grid=None, mgrid=None, nt=1, t0=0.0, dt_snap=3600.0, Kh=0.0, H=1.0e9, kz_min=0.0,
           nuclides=None, dt=10.0, seed=1, n=100, boundary="open", compact=False, h_dep=None,
           bin_every=0, n_steps=10, src=(0.0, 0.0, 50.0), t_rel=(0.0, 0.0), activity=None,
           rate=0.0, capacity=None, rain=None, pid_offset=0, pid_stride=1, name="custom"):
    grid = grid or Grid(16, 16, 8, -800.0, -800.0, 0.0, 100.0, 100.0, 100.0)
    mgrid = mgrid or grid
    nuclides = nuclides or [Nuclide("X", 0.0)]
    activity = activity or [1.0] * len(nuclides)
    h_dep = H if h_dep is None else h_dep
    rel = None
    if n > 0 or rate > 0:
        rel = Release(src[0], src[1], src[2], t_rel[0], t_rel[1], list(activity),
                      n_particles=0 if rate > 0 else n, rate=rate, pid_offset=pid_offset, pid_stride=pid_stride)
    return Workload(name=name, cgrid=grid, mgrid=mgrid, nt=nt, t0=t0, dt_snap=dt_snap, Kh=Kh, H_mix=H,
                    kz_min=kz_min, nuclides=nuclides, dt=dt, seed=seed,
                    capacity=capacity if capacity is not None else max(n, 1),
                    boundary_mode=boundary, compact=compact, h_dep=h_dep, bin_every=bin_every,
                    n_steps=n_steps, release=rel, rain=rain, met_fn=met_fn)


def uniform_met(u=0.0, v=0.0, w=0.0, kz=0.0):
    return lambda t, Z, Y, X: (u, v, w, kz)


def gpu_state(sim):
    """The CUDA path's particle state in activity units: the binding returns the stored fp32 q and the fp64 scale
    G_k(t) (lpm_mass_scale, R8) separately; their product is formed here, on the test side."""
    p = sim.get_particles_host()
    p["m"] = p["q"] * p["scale"][:, None]
    return p
