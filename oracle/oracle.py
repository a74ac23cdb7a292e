"""ctypes binding of the fp64 CPU oracle (oracle/lpm_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Imports nothing from paper_0912_3223_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lpm_oracle.c")
_LIB = os.path.join(_HERE, "liblpm_oracle.so")
MAXK = 2
NLEDGER = 7
LEDGER_NAMES = ("emitted", "airborne", "dry", "wet", "decayed", "exited", "dep_offgrid")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("pad_", C.c_int32),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class Config(C.Structure):
    _fields_ = [("cgrid", Grid), ("mgrid", Grid), ("nt", C.c_int32), ("K", C.c_int32),
                ("t0", C.c_double), ("dt_snap", C.c_double), ("fields", C.c_void_p),
                ("Kh", C.c_double), ("H_mix", C.c_double), ("kz_min", C.c_double),
                ("half_life", C.c_double * MAXK), ("vd", C.c_double * MAXK), ("lambda_wet", C.c_double * MAXK),
                ("dt", C.c_double), ("seed", C.c_uint64), ("capacity", C.c_uint64),
                ("boundary_mode", C.c_int32), ("compact", C.c_int32), ("h_dep", C.c_double),
                ("bin_every", C.c_int32), ("rain_on", C.c_int32),
                ("rx0", C.c_double), ("rx1", C.c_double), ("ry0", C.c_double), ("ry1", C.c_double),
                ("rt0", C.c_double), ("rt1", C.c_double),
                ("frag_delta", C.c_double), ("face_delta", C.c_double),
                ("dep_mode", C.c_int32), ("kz_mode", C.c_int32), ("surface", C.c_void_p), ("z_levels", C.c_void_p),
                ("drift", C.c_int32), ("pad3_", C.c_int32)]


class Source(C.Structure):
    _fields_ = [("x", C.c_double), ("y", C.c_double), ("z", C.c_double),
                ("t_start", C.c_double), ("t_end", C.c_double),
                ("total_activity", C.c_double * MAXK), ("n_particles", C.c_uint64), ("rate", C.c_double),
                ("pid_offset", C.c_uint64), ("pid_stride", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(Config)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_release.argtypes = [C.c_void_p, C.POINTER(Source)]
        L.orc_release.restype = C.c_int32
        L.orc_step.argtypes = [C.c_void_p, C.c_int32]
        L.orc_step.restype = C.c_int32
        L.orc_bin_now.argtypes = [C.c_void_p]
        for f in ("orc_num_particles", "orc_step_index", "orc_num_fragile"):
            getattr(L, f).argtypes = [C.c_void_p]
            getattr(L, f).restype = C.c_uint64
        L.orc_get_fragile.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_p_dry.argtypes = [C.c_void_p, C.c_int]
        L.orc_p_dry.restype = C.c_float
        L.orc_p_wet.argtypes = [C.c_void_p, C.c_int]
        L.orc_p_wet.restype = C.c_float
        L.orc_sigma_h.argtypes = [C.c_void_p]
        L.orc_sigma_h.restype = C.c_float
        L.orc_get_particles.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        L.orc_set_particles.argtypes = [C.c_void_p, C.c_uint64] + [C.c_void_p] * 7
        L.orc_set_step_index.argtypes = [C.c_void_p, C.c_uint64]
        L.orc_ledger.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_concentration.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_counts.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_enable_dose.argtypes = [C.c_void_p]
        L.orc_dose.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_enable_ground_decay.argtypes = [C.c_void_p]
        L.orc_deposition_ground.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_deposition.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_injected.argtypes = [C.c_void_p, C.c_uint64]
        L.orc_injected.restype = C.c_uint64
        L.orc_num_threads.restype = C.c_int32
        L.orc_set_num_threads.argtypes = [C.c_int32]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_philox_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, C.c_void_p]
        L.orc_uniforms.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_normals.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_time_weight.argtypes = [C.c_int32, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_sample_met.argtypes = [C.POINTER(Grid), C.c_int32, C.c_double, C.c_double, C.c_void_p,
                                     C.c_double, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_sample_met_levels.argtypes = [C.POINTER(Grid), C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_void_p,
                                            C.c_double, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_dkz_dz.argtypes = [C.POINTER(Grid), C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_void_p,
                                 C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_dkz_dz.restype = C.c_double
        L.orc_kz_eq3.argtypes = [C.c_double] * 4
        L.orc_kz_eq3.restype = C.c_double
        L.orc_sample_surface.argtypes = [C.POINTER(Grid), C.c_int32, C.c_double, C.c_double, C.c_void_p,
                                         C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_cell_index.argtypes = [C.c_float, C.c_double, C.c_double, C.c_int32]
        L.orc_cell_index.restype = C.c_int32
        _lib = L
    return _lib


def _grid(g) -> Grid:
    return Grid(g.nx, g.ny, g.nz, 0, g.x0, g.y0, g.z0, g.dx, g.dy, g.dz)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ---------------------------------------------------------------- stand-alone pieces (pins)
def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def philox_draw(seed, pid, step, stream=0):
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox_draw(seed, pid, step, stream, _p(out))
    return out


def uniforms(r):
    r = np.asarray(r, dtype=np.uint32).copy()
    u = np.zeros(4, dtype=np.float64)
    lib().orc_uniforms(_p(r), _p(u))
    return u


def normals(seed, pid, step):
    n = np.zeros(3, dtype=np.float64)
    lib().orc_normals(seed, pid, step, _p(n))
    return n


def time_weight(nt, t0, dt_snap, t):
    s = C.c_int32()
    a = C.c_float()
    lib().orc_time_weight(nt, t0, dt_snap, t, C.byref(s), C.byref(a))
    return s.value, a.value


def sample_met(grid, nt, t0, dt_snap, fields, t, x, y, z, z_levels=None):
    f = np.ascontiguousarray(fields, dtype=np.float32)
    out = np.zeros(4, dtype=np.float64)
    g = _grid(grid)
    lv = None if z_levels is None else np.ascontiguousarray(z_levels, dtype=np.float64)
    lib().orc_sample_met_levels(C.byref(g), None if lv is None else lv.ctypes.data, nt, t0, dt_snap, _p(f), t, x, y, z, _p(out))
    return out


def dkz_dz(grid, nt, t0, dt_snap, fields, t, x, y, z, z_levels=None):
    f = np.ascontiguousarray(fields, dtype=np.float32)
    lv = None if z_levels is None else np.ascontiguousarray(z_levels, dtype=np.float64)
    return lib().orc_dkz_dz(C.byref(_grid(grid)), None if lv is None else lv.ctypes.data, nt, t0, dt_snap, _p(f), t, x, y, z)


def kz_eq3(ustar, inv_L, Hz, z):
    return lib().orc_kz_eq3(ustar, inv_L, Hz, z)


def sample_surface(grid, nt, t0, dt_snap, surface, t, x, y):
    out = np.zeros(3)
    sf = np.ascontiguousarray(surface, dtype=np.float32)
    lib().orc_sample_surface(C.byref(_grid(grid)), nt, t0, dt_snap, sf.ctypes.data, t, x, y, _p(out))
    return out


def cell_index(p, p0, dp, n):
    return lib().orc_cell_index(float(np.float32(p)), p0, dp, n)


# ---------------------------------------------------------------- the simulation object
class OracleSim:
    """The fp64 oracle run of a `workloads.Workload`."""

    def __init__(self, w, frag_delta: float = 0.05, face_delta: float = 0.0, bin_every: Optional[int] = None,
                 dep_mode: int = 0, drift: bool = False):
        self.w = w
        self.K = w.K
        self._fields = np.ascontiguousarray(w.fields(), dtype=np.float32)
        cfg = Config()
        cfg.cgrid = _grid(w.cgrid)
        cfg.mgrid = _grid(w.mgrid)
        cfg.nt, cfg.K, cfg.t0, cfg.dt_snap = w.nt, w.K, w.t0, w.dt_snap
        cfg.fields = self._fields.ctypes.data
        cfg.Kh, cfg.H_mix, cfg.kz_min = w.Kh, w.H_mix, w.kz_min
        for k, nuc in enumerate(w.nuclides):
            cfg.half_life[k], cfg.vd[k], cfg.lambda_wet[k] = nuc.half_life_s, nuc.vd, nuc.lambda_wet
        cfg.dt, cfg.seed, cfg.capacity = w.dt, w.seed, w.capacity
        cfg.boundary_mode = 1 if w.boundary_mode == "absorb" else 0
        cfg.compact = 1 if w.compact else 0
        cfg.h_dep = w.h_dep
        cfg.bin_every = w.bin_every if bin_every is None else bin_every
        if w.rain is not None:
            cfg.rain_on = 1
            cfg.rx0, cfg.rx1, cfg.ry0, cfg.ry1 = w.rain.x0, w.rain.x1, w.rain.y0, w.rain.y1
            cfg.rt0, cfg.rt1 = w.rain.t_start, w.rain.t_end
        cfg.frag_delta, cfg.face_delta = frag_delta, face_delta
        cfg.dep_mode = dep_mode
        cfg.drift = 1 if drift else 0
        self._levels = None
        if getattr(w, "z_levels", None) is not None:
            self._levels = np.ascontiguousarray(w.z_levels, dtype=np.float64)
            assert self._levels.shape == (w.mgrid.nz,)
            cfg.z_levels = self._levels.ctypes.data
        self._surface = None
        if getattr(w, "kz_mode", 0) == 1:
            self._surface = np.ascontiguousarray(w.surface(), dtype=np.float32)
            cfg.kz_mode = 1
            cfg.surface = self._surface.ctypes.data
        self._cfg = cfg
        self._h = lib().orc_create(C.byref(cfg))
        if not self._h:
            raise RuntimeError("orc_create failed")
        if w.release is not None:
            self.release(w.release)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def release(self, r):
        s = Source()
        s.x, s.y, s.z, s.t_start, s.t_end = r.x, r.y, r.z, r.t_start, r.t_end
        for k in range(self.K):
            s.total_activity[k] = r.total_activity[k]
        s.n_particles, s.rate, s.pid_offset, s.pid_stride = r.n_particles, r.rate, r.pid_offset, r.pid_stride
        if lib().orc_release(self._h, C.byref(s)) != 0:
            raise RuntimeError("orc_release failed")

    def step(self, n=1):
        if lib().orc_step(self._h, n) != 0:
            raise RuntimeError("orc_step failed")

    def bin_now(self):
        lib().orc_bin_now(self._h)

    @property
    def n(self):
        return int(lib().orc_num_particles(self._h))

    @property
    def step_index(self):
        return int(lib().orc_step_index(self._h))

    def set_step_index(self, s):
        lib().orc_set_step_index(self._h, s)

    def p_dry(self, k):
        return float(lib().orc_p_dry(self._h, k))

    def p_wet(self, k):
        return float(lib().orc_p_wet(self._h, k))

    def sigma_h(self):
        return float(lib().orc_sigma_h(self._h))

    def particles(self):
        n = self.n
        x, y, z = (np.zeros(n) for _ in range(3))
        m = np.zeros((self.K, n))
        m1 = m[1] if self.K > 1 else None
        pid = np.zeros(n, dtype=np.uint64)
        st = np.zeros(n, dtype=np.uint8)
        lib().orc_get_particles(self._h, _p(x), _p(y), _p(z), _p(m[0]), _p(m1), _p(pid), _p(st))
        return dict(x=x, y=y, z=z, m=m, pid=pid, status=st)

    def set_particles(self, x, y, z, m, pid=None, status=None):
        x, y, z = (np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, z))
        m = np.ascontiguousarray(np.atleast_2d(m), dtype=np.float64)
        n = x.shape[0]
        assert m.shape == (self.K, n)
        m1 = m[1] if self.K > 1 else None
        pid = None if pid is None else np.ascontiguousarray(pid, dtype=np.uint64)
        status = None if status is None else np.ascontiguousarray(status, dtype=np.uint8)
        lib().orc_set_particles(self._h, n, _p(x), _p(y), _p(z), _p(m[0]), _p(m1), _p(pid), _p(status))

    def fragile_pids(self):
        n = int(lib().orc_num_fragile(self._h))
        out = np.zeros(n, dtype=np.uint64)
        if n:
            lib().orc_get_fragile(self._h, _p(out))
        return out

    def ledger(self):
        out = np.zeros((self.K, NLEDGER))
        lib().orc_ledger(self._h, _p(out))
        return out

    def concentration(self):
        g = self.w.cgrid
        out = np.zeros((self.K, g.nz, g.ny, g.nx))
        lib().orc_concentration(self._h, _p(out))
        return out

    def enable_dose(self):
        lib().orc_enable_dose(self._h)

    def dose(self):
        """time-integrated concentration [K][nz][ny][nx], Bq s m^-3 (S§8(f)3)"""
        g = self.w.cgrid
        out = np.zeros((self.K, g.nz, g.ny, g.nx), dtype=np.float64)
        lib().orc_dose(self._h, _p(out))
        return out

    def counts(self):
        g = self.w.cgrid
        out = np.zeros((g.nz, g.ny, g.nx), dtype=np.uint32)
        lib().orc_counts(self._h, _p(out))
        return out

    def deposition(self, with_slack=False):
        g = self.w.cgrid
        out = np.zeros((self.K, g.ny, g.nx))
        slack = np.zeros((self.K, g.ny, g.nx)) if with_slack else None
        lib().orc_deposition(self._h, _p(out), _p(slack))
        return (out, slack) if with_slack else out

    def enable_ground_decay(self):
        lib().orc_enable_ground_decay(self._h)

    def deposition_ground(self, with_slack=False):
        """deposition map whose content keeps decaying on the ground [K][ny][nx], Bq m^-2 at the current time (R13)"""
        g = self.w.cgrid
        out = np.zeros((self.K, g.ny, g.nx))
        slack = np.zeros((self.K, g.ny, g.nx)) if with_slack else None
        lib().orc_deposition_ground(self._h, _p(out), _p(slack))
        return (out, slack) if with_slack else out

    def injected(self, step):
        return int(lib().orc_injected(self._h, step))


def num_threads():
    return int(lib().orc_num_threads())


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))
