"""The five BASELINE.json configs as seeded, synthetic, closed-form inputs.

Everything here is an INPUT RECIPE (restated in DESIGN.md §4):
grids, constants, sources and the closed-form meteorological fields, generated in
float64 and rounded ONCE to float32.  That float32 array is the input of both the
fp64 oracle and the CUDA path.  No method arithmetic lives here.

Lateral boundary (R7): c1 and c2 are OPEN (their plumes essentially stay inside the grid for the whole run).
c3 and c4 are ABSORB, the paper's own rule (a particle that "reaches the predefined boundaries" becomes
inactive): a 3-8 m/s wind whose direction swings +-45 degrees about a fixed mean carries a particle at least
3 cos(45 deg) x 12 h = 92 km, typically 250 km, so no source position keeps the particles inside the 100 km box of
BASELINE.json configs 3/4 for 12 or 24 h; what has left the box is inactive and is not counted as work.  The
particle store of c3/c4 stays slot-addressed (no compaction: BASELINE.json asks for it in config 5 only).

Paper scales used (citations are PAPER.md lines): dt ~ 10 s, Kx = Ky = 100 m^2/s
(P:L77), Kz profile of Eq.(3) with Phi = 1, low point source,
hours-long runs with 0.5 - several million particles.  The paper's own
ALADIN fields and Paks scenario are not available; these inputs stand in for them.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

NAMES = ("c1", "c2", "c2_eq3", "c3", "c3_hdep80", "c4", "c5")

HOUR = 3600.0
DAY = 86400.0
T_HALF_I131 = 8.02 * DAY                 # BASELINE config 1/3: "half-life 8.02 d"
T_HALF_CS137 = 30.17 * 365.25 * DAY      # BASELINE config 3: "30.17 y" (Julian years)


@dataclass
class Grid:
    nx: int
    ny: int
    nz: int
    x0: float
    y0: float
    z0: float
    dx: float
    dy: float
    dz: float

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)


@dataclass
class Nuclide:
    name: str
    half_life_s: float
    vd: float = 0.0            # dry deposition velocity, m/s
    lambda_wet: float = 0.0    # wet scavenging coefficient, 1/s


@dataclass
class RainBox:
    x0: float
    x1: float
    y0: float
    y1: float
    t_start: float
    t_end: float


@dataclass
class Release:
    x: float
    y: float
    z: float
    t_start: float
    t_end: float
    total_activity: List[float]          # Bq per nuclide over the whole release
    n_particles: int = 0                 # count mode (R9) when > 0
    rate: float = 0.0                    # particles per second, rate mode when n_particles == 0
    pid_offset: int = 0                  # take global particle ids offset, offset+stride, ...
    pid_stride: int = 1


@dataclass
class Workload:
    name: str
    cgrid: Grid                          # concentration grid; the 2-D deposition map uses its x/y
    mgrid: Grid                          # meteorology grid (cell-centred values)
    nt: int
    t0: float
    dt_snap: float
    Kh: float
    H_mix: float
    kz_min: float
    nuclides: List[Nuclide]
    dt: float
    seed: int
    capacity: int
    boundary_mode: str                   # "open" | "absorb"
    compact: bool
    h_dep: float
    bin_every: int
    n_steps: int
    release: Optional[Release]
    rain: Optional[RainBox] = None
    met_fn: object = field(default=None, repr=False)   # (t, Z, Y, X) -> u, v, w, kz  in float64
    kz_mode: int = 0                                   # 1: Kz from Eq.(3) per particle (R12) with the 2-D fields below
    surface_fn: object = field(default=None, repr=False)   # (t, Y, X) -> ustar, 1/L, Hz  in float64 (cell centres)
    z_levels: object = None                            # None: uniform levels; else mgrid.nz ascending level heights, m
    _fields: object = field(default=None, repr=False)

    @property
    def K(self) -> int:
        return len(self.nuclides)

    def fields(self) -> np.ndarray:
        """float32 array [nt][nz][ny][nx][4] = (u, v, w, Kz) at cell centres, x fastest."""
        if self._fields is None:
            g = self.mgrid
            xc = g.x0 + (np.arange(g.nx, dtype=np.float64) + 0.5) * g.dx
            yc = g.y0 + (np.arange(g.ny, dtype=np.float64) + 0.5) * g.dy
            zc = g.z0 + (np.arange(g.nz, dtype=np.float64) + 0.5) * g.dz
            if self.z_levels is not None:
                zc = np.asarray(self.z_levels, dtype=np.float64)
            Z, Y, X = np.meshgrid(zc, yc, xc, indexing="ij")
            out = np.empty((self.nt, g.nz, g.ny, g.nx, 4), dtype=np.float32)
            recipe = getattr(self.met_fn, "__name__", "") if self.met_fn in _RECIPES else None
            for s in range(self.nt):
                t = self.t0 + s * self.dt_snap
                key = (recipe, dataclasses.astuple(g), t, None if self.z_levels is None else tuple(np.asarray(self.z_levels).tolist()))
                if recipe is not None and key in _SNAP_CACHE:
                    out[s] = _SNAP_CACHE[key]
                    continue
                u, v, w, kz = self.met_fn(t, Z, Y, X)
                out[s, ..., 0] = np.broadcast_to(u, Z.shape)
                out[s, ..., 1] = np.broadcast_to(v, Z.shape)
                out[s, ..., 2] = np.broadcast_to(w, Z.shape)
                out[s, ..., 3] = np.broadcast_to(kz, Z.shape)
                if recipe is not None and len(_SNAP_CACHE) < 32:
                    _SNAP_CACHE[key] = out[s].copy()
            self._fields = out
        return self._fields

    def surface(self) -> np.ndarray:
        """float32 array [nt][ny][nx][4] = (u*, 1/L, Hz, 0) at the met grid's column centres, x fastest."""
        g = self.mgrid
        xc = g.x0 + (np.arange(g.nx, dtype=np.float64) + 0.5) * g.dx
        yc = g.y0 + (np.arange(g.ny, dtype=np.float64) + 0.5) * g.dy
        Y, X = np.meshgrid(yc, xc, indexing="ij")
        out = np.zeros((self.nt, g.ny, g.nx, 4), dtype=np.float32)
        for s in range(self.nt):
            us, il, hz = self.surface_fn(self.t0 + s * self.dt_snap, Y, X)
            out[s, ..., 0] = np.broadcast_to(us, Y.shape)
            out[s, ..., 1] = np.broadcast_to(il, Y.shape)
            out[s, ..., 2] = np.broadcast_to(hz, Y.shape)
        return out

    def replace(self, **kw) -> "Workload":
        w = dataclasses.replace(self, **kw)
        if "mgrid" in kw or "nt" in kw or "met_fn" in kw or "t0" in kw or "dt_snap" in kw or "z_levels" in kw:
            w._fields = None
        return w

    def born_particle_steps(self, n_steps: Optional[int] = None) -> int:
        """Number of (particle, step) pairs with birth step <= step < n_steps, ignoring
        exits/compaction (used only to label throughput; counting rule of R9)."""
        n_steps = self.n_steps if n_steps is None else n_steps
        r = self.release
        s0 = int(math.ceil(r.t_start / self.dt))
        S = max(1, int(math.ceil((r.t_end - r.t_start) / self.dt)))
        total = 0
        if r.n_particles > 0:
            N = r.n_particles
            for n in range(s0, n_steps):
                total += min(N, -(-(n - s0 + 1) * N // S))
        else:
            c = int(round(r.rate * self.dt))
            for n in range(s0, n_steps):
                total += min(self.capacity, c * min(n - s0 + 1, S))
        return total


# ----------------------------------------------------------------------------- met recipes
def _met_c1(t, Z, Y, X):
    return 5.0, 0.0, 0.0, 5.0


def _met_c2(t, Z, Y, X):
    ustar, k, z0, H = 0.4, 0.4, 0.1, 1000.0
    speed = (ustar / k) * np.log(Z / z0)
    theta = np.deg2rad(30.0 * Z / 1000.0 + 10.0 * (t / HOUR))
    kz = np.maximum(0.1, k * ustar * Z * (1.0 - Z / H) ** 2)
    return speed * np.cos(theta), speed * np.sin(theta), 0.0, kz


def _surface_c2(t, Y, X):
    """c2_eq3 (S§8(f)2): friction velocity, inverse Obukhov length and mixing height as smooth 2-D fields that
    change over the two hours: near-neutral with a stable (1/L > 0) half and an unstable half of the domain."""
    ustar = 0.4 * (1.0 + 0.2 * np.sin(2.0 * np.pi * X / 40.0e3)) * (1.0 + 0.1 * t / HOUR)
    inv_L = 0.004 * np.sin(2.0 * np.pi * Y / 60.0e3) - 0.002 * t / HOUR
    Hz = 1000.0 * (1.0 - 0.2 * np.cos(2.0 * np.pi * (X + Y) / 80.0e3)) - 50.0 * t / HOUR
    return ustar, inv_L, Hz


def _wind_c3(t, Z, Y, X):
    S = 5.5 + 2.5 * math.sin(2.0 * math.pi * t / (12.0 * HOUR))
    th = math.radians(45.0) * math.sin(2.0 * math.pi * t / (6.0 * HOUR))
    speed = S * (Z / 100.0) ** 0.15
    u = speed * math.cos(th) + np.sin(2.0 * np.pi * Y / 25.0e3)
    v = speed * math.sin(th) + np.sin(2.0 * np.pi * X / 25.0e3)
    return u, v


def _met_c3(t, Z, Y, X):
    H = 1000.0
    u, v = _wind_c3(t, Z, Y, X)
    zz = np.minimum(Z, H)
    kz = np.maximum(1.0, 0.16 * zz * (1.0 - zz / H) ** 2)
    return u, v, 0.0, kz


def _met_c5(t, Z, Y, X):
    H = 1250.0
    u, v = _wind_c3(t, Z, Y, X)
    zeta = np.minimum(Z, H) / H
    kz = 10.0 + 190.0 * (27.0 / 4.0) * zeta * (1.0 - zeta) ** 2
    return u, v, 0.0, kz


_RECIPES = (_met_c1, _met_c2, _met_c3, _met_c5)
_SNAP_CACHE = {}   # (recipe, grid, t) -> float32 snapshot; saves regenerating the big grids in tests


# ----------------------------------------------------------------------------- the configs
def _c1(scale):
    g = Grid(60, 60, 10, -500.0, -3000.0, 0.0, 100.0, 100.0, 50.0)
    n = max(1, int(round(10_000 * scale)))
    return Workload(
        name="c1", cgrid=g, mgrid=g, nt=1, t0=0.0, dt_snap=HOUR, Kh=50.0, H_mix=1000.0, kz_min=0.0,
        nuclides=[Nuclide("I-131", T_HALF_I131)], dt=10.0, seed=1, capacity=n,
        boundary_mode="open", compact=False, h_dep=1000.0, bin_every=50, n_steps=100,
        release=Release(0.0, 0.0, 50.0, 0.0, 0.0, [1.0e9], n_particles=n), met_fn=_met_c1)


def _c2(scale):
    g = Grid(200, 200, 20, -5.0e4, -5.0e4, 0.0, 500.0, 500.0, 50.0)
    n = max(1, int(round(1_000_000 * scale)))
    return Workload(
        name="c2", cgrid=g, mgrid=g, nt=3, t0=0.0, dt_snap=HOUR, Kh=100.0, H_mix=1000.0, kz_min=0.1,
        nuclides=[Nuclide("I-131", T_HALF_I131)], dt=5.0, seed=2, capacity=n,
        boundary_mode="open", compact=False, h_dep=1000.0, bin_every=120, n_steps=1440,
        release=Release(0.0, 0.0, 50.0, 0.0, HOUR, [6.0e9], n_particles=n), met_fn=_met_c2)


def _c3(scale, h_dep=1000.0, name="c3"):
    g = Grid(400, 400, 30, -5.0e4, -5.0e4, 0.0, 250.0, 250.0, 40.0)
    n = max(1, int(round(10_000_000 * scale)))
    return Workload(
        name=name, cgrid=g, mgrid=g, nt=25, t0=0.0, dt_snap=HOUR, Kh=100.0, H_mix=1000.0, kz_min=1.0,
        nuclides=[Nuclide("I-131", T_HALF_I131, 1.0e-3, 1.0e-4),
                  Nuclide("Cs-137", T_HALF_CS137, 2.0e-3, 1.0e-4)],
        dt=10.0, seed=3, capacity=n, boundary_mode="absorb", compact=False, h_dep=h_dep,
        bin_every=360, n_steps=8640,
        release=Release(-4.0e4, 0.0, 50.0, 0.0, 24 * HOUR, [1.0e15, 1.0e14], n_particles=n),
        rain=RainBox(-3.0e4, 1.0e4, -2.0e4, 2.0e4, 6 * HOUR, 9 * HOUR), met_fn=_met_c3)


def _c4(scale):
    cg = Grid(1000, 1000, 30, -5.0e4, -5.0e4, 0.0, 100.0, 100.0, 40.0)
    mg = Grid(400, 400, 30, -5.0e4, -5.0e4, 0.0, 250.0, 250.0, 40.0)
    n = max(1, int(round(100_000_000 * scale)))
    return Workload(
        name="c4", cgrid=cg, mgrid=mg, nt=13, t0=0.0, dt_snap=HOUR, Kh=100.0, H_mix=1000.0, kz_min=1.0,
        nuclides=[Nuclide("I-131", T_HALF_I131, 1.0e-3, 1.0e-4),
                  Nuclide("Cs-137", T_HALF_CS137, 2.0e-3, 1.0e-4)],
        dt=5.0, seed=4, capacity=n, boundary_mode="absorb", compact=False, h_dep=1000.0,
        bin_every=720, n_steps=8640,
        release=Release(-4.0e4, 0.0, 50.0, 0.0, 12 * HOUR, [1.0e15, 1.0e14], n_particles=n),
        rain=RainBox(-3.0e4, 1.0e4, -2.0e4, 2.0e4, 6 * HOUR, 9 * HOUR), met_fn=_met_c3)


def _c5(scale):
    g = Grid(500, 500, 25, -5.0e4, -5.0e4, 0.0, 200.0, 200.0, 50.0)
    rate = 2.0e4 * scale
    cap = max(1, int(round(50_000_000 * scale)))
    n_steps = 21600
    per_step = int(round(rate * 2.0))
    return Workload(
        name="c5", cgrid=g, mgrid=g, nt=13, t0=0.0, dt_snap=HOUR, Kh=100.0, H_mix=1250.0, kz_min=10.0,
        nuclides=[Nuclide("I-131", T_HALF_I131)], dt=2.0, seed=5, capacity=cap,
        boundary_mode="absorb", compact=True, h_dep=1250.0, bin_every=150, n_steps=n_steps,
        release=Release(-4.0e4, 0.0, 50.0, 0.0, n_steps * 2.0, [float(per_step * n_steps)], rate=rate),
        met_fn=_met_c5)


def make(name: str, scale: float = 1.0, n_steps: Optional[int] = None) -> Workload:
    """Build config `name`; `scale` multiplies the particle count (and, for c5, the injection
    rate and capacity) without touching grids, met or cadence; `n_steps` truncates the run."""
    if name == "c1":
        w = _c1(scale)
    elif name == "c2":
        w = _c2(scale)
    elif name == "c2_eq3":
        w = dataclasses.replace(_c2(scale), name="c2_eq3", kz_mode=1, surface_fn=_surface_c2)
    elif name == "c3":
        w = _c3(scale)
    elif name == "c3_hdep80":
        w = _c3(scale, h_dep=80.0, name="c3_hdep80")
    elif name == "c4":
        w = _c4(scale)
    elif name == "c5":
        w = _c5(scale)
    else:
        raise ValueError(f"unknown workload {name!r}; choose from {NAMES}")
    if n_steps is not None:
        w = w.replace(n_steps=int(n_steps))
    return w
