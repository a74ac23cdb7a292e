"""Thin Python binding of the C ABI in include/lpm.h (argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels
behind liblpm_b200.so.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblpm_b200.so")

MAX_NUCLIDES = 2
LEDGER_FIELDS = 7
LEDGER_NAMES = ("emitted", "airborne", "dry", "wet", "decayed", "exited", "dep_offgrid")

OK, ERR_INVALID_ARG, ERR_NO_DEVICE, ERR_WORKSPACE_TOO_SMALL, ERR_CAPACITY, ERR_STATE, ERR_CUDA = 0, -1, -2, -3, -4, -5, -6

# every symbol include/lpm.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "lpm_version", "lpm_status_string", "lpm_workspace_bytes", "lpm_schedule_born", "lpm_create", "lpm_destroy",
    "lpm_set_rain", "lpm_release", "lpm_step", "lpm_concentration", "lpm_counts", "lpm_deposition",
    "lpm_deposition_f64", "lpm_bin_now", "lpm_num_active", "lpm_step_index", "lpm_mass_scale", "lpm_get_particles",
    "lpm_set_particles", "lpm_ledger", "lpm_injected", "lpm_last_error", "lpm_launch_count", "lpm_test_philox",
    "lpm_test_normals", "lpm_test_sample", "lpm_upload_meteo", "lpm_concentration_host", "lpm_deposition_host",
    "lpm_set_timing", "lpm_get_timing", "lpm_probe", "lpm_test_box_muller", "lpm_dose", "lpm_test_curand_philox",
    "lpm_texel_pairs", "lpm_touched_cells", "lpm_restart", "lpm_sample_static",
)


class LpmError(RuntimeError):
    def __init__(self, status, where, detail=""):
        self.status = status
        super().__init__(f"{where}: status {status} ({status_string(status)}) {detail}".strip())


class lpm_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("reserved", C.c_int32),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class lpm_meteo(C.Structure):
    _fields_ = [("grid", lpm_grid), ("nt", C.c_int32), ("kz_mode", C.c_int32), ("t0", C.c_double),
                ("dt_snap", C.c_double), ("fields_dev", C.c_void_p), ("Kh", C.c_double), ("H_mix", C.c_double),
                ("kz_min", C.c_double), ("surface_dev", C.c_void_p), ("z_levels_host", C.c_void_p)]


class lpm_nuclide(C.Structure):
    _fields_ = [("half_life_s", C.c_double), ("vd", C.c_double), ("lambda_wet", C.c_double)]


class lpm_params(C.Structure):
    _fields_ = [("dt", C.c_double), ("seed", C.c_uint64), ("capacity", C.c_uint64), ("boundary_mode", C.c_int32),
                ("compact", C.c_int32), ("h_dep", C.c_double), ("bin_every", C.c_int32), ("steps_per_launch", C.c_int32),
                ("gather_sort", C.c_int32), ("dose", C.c_int32), ("dep_mode", C.c_int32), ("drift", C.c_int32), ("texel_pairs", C.c_int32), ("ground_decay", C.c_int32)]


class lpm_source(C.Structure):
    _fields_ = [("x", C.c_double), ("y", C.c_double), ("z", C.c_double), ("t_start", C.c_double), ("t_end", C.c_double)]


_lib = None


def load():
    """Load liblpm_b200.so (built by paper_0912_3223_b200.build); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_0912_3223_b200.build` (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, u64, i32, i64, dbl = C.c_void_p, C.c_uint64, C.c_int32, C.c_int64, C.c_double
    L.lpm_version.restype = i32
    L.lpm_status_string.restype = C.c_char_p
    L.lpm_status_string.argtypes = [i32]
    L.lpm_workspace_bytes.argtypes = [C.POINTER(lpm_grid), C.POINTER(lpm_meteo), C.POINTER(lpm_params), i32, C.POINTER(u64)]
    L.lpm_schedule_born.argtypes = [u64, u64, u64, i64, i64, i64, C.POINTER(u64)]
    L.lpm_create.argtypes = [C.POINTER(lpm_grid), C.POINTER(lpm_meteo), C.POINTER(lpm_nuclide), i32,
                             C.POINTER(lpm_params), vp, u64, vp, C.POINTER(vp)]
    L.lpm_destroy.argtypes = [vp]
    L.lpm_restart.argtypes = [vp]
    L.lpm_set_rain.argtypes = [vp, dbl, dbl, dbl, dbl, dbl, dbl]
    L.lpm_release.argtypes = [vp, C.POINTER(lpm_source), C.POINTER(dbl), u64, dbl, u64, u64]
    L.lpm_step.argtypes = [vp, i32]
    L.lpm_concentration.argtypes = [vp, vp]
    L.lpm_counts.argtypes = [vp, vp]
    L.lpm_dose.argtypes = [vp, vp]
    L.lpm_deposition.argtypes = [vp, vp]
    L.lpm_deposition_f64.argtypes = [vp, vp]
    L.lpm_bin_now.argtypes = [vp]
    L.lpm_num_active.argtypes = [vp, C.POINTER(u64)]
    L.lpm_step_index.argtypes = [vp, C.POINTER(u64)]
    L.lpm_mass_scale.argtypes = [vp, C.POINTER(dbl)]
    L.lpm_get_particles.argtypes = [vp, vp, vp, vp, vp, C.POINTER(u64)]
    L.lpm_set_particles.argtypes = [vp, vp, vp, vp, vp, u64, u64]
    L.lpm_ledger.argtypes = [vp, C.POINTER(dbl)]
    L.lpm_injected.argtypes = [vp, u64, C.POINTER(u64)]
    L.lpm_last_error.argtypes = [vp]
    L.lpm_last_error.restype = C.c_char_p
    L.lpm_launch_count.argtypes = [vp, C.POINTER(u64)]
    L.lpm_upload_meteo.argtypes = [vp, i32, i32, vp]
    L.lpm_concentration_host.argtypes = [vp, vp]
    L.lpm_deposition_host.argtypes = [vp, vp]
    L.lpm_set_timing.argtypes = [vp, i32]
    L.lpm_get_timing.argtypes = [vp, C.POINTER(dbl)]
    L.lpm_texel_pairs.argtypes = [vp, C.POINTER(i32)]
    L.lpm_touched_cells.argtypes = [vp, C.POINTER(u64)]
    L.lpm_probe.argtypes = [i32, u64, vp, u64, i32, C.POINTER(dbl), vp]
    L.lpm_test_box_muller.argtypes = [vp, u64, vp, vp]
    L.lpm_test_curand_philox.argtypes = [u64, u64, u64, u64, vp, vp]
    L.lpm_test_philox.argtypes = [u64, u64, C.c_uint32, u64, u64, vp, vp]
    L.lpm_test_normals.argtypes = [u64, u64, u64, u64, vp, vp]
    L.lpm_test_sample.argtypes = [C.POINTER(lpm_meteo), dbl, vp, u64, vp, vp]
    L.lpm_sample_static.argtypes = [C.POINTER(lpm_meteo), dbl, vp, u64, vp, vp]
    for s in SYMBOLS:
        if getattr(L, s).restype is C.c_int:
            getattr(L, s).restype = i32
    _lib = L
    return L


def status_string(status: int) -> str:
    return load().lpm_status_string(status).decode()


def version() -> int:
    return load().lpm_version()


def _grid(g) -> lpm_grid:
    return lpm_grid(g.nx, g.ny, g.nz, 0, g.x0, g.y0, g.z0, g.dx, g.dy, g.dz)


def workspace_bytes(cgrid, capacity: int, n_nuclides: int, compact: bool, mgrid=None, nt: int = 1, gather_sort: int = 0,
                    dose: bool = False, kz_mode: int = 0, dep_mode: int = 0, drift: bool = False, texel_pairs: int = 0,
                    z_levels=None) -> int:
    p = lpm_params(dt=1.0, capacity=capacity, compact=1 if compact else 0, h_dep=1.0, gather_sort=gather_sort, dose=1 if dose else 0,
                   dep_mode=dep_mode, drift=1 if drift else 0, texel_pairs=texel_pairs)
    out = C.c_uint64()
    g = _grid(cgrid)
    met = lpm_meteo(grid=_grid(mgrid if mgrid is not None else cgrid), nt=nt, kz_mode=kz_mode)
    if z_levels is not None:   # only its presence matters for the size
        lev = np.ascontiguousarray(z_levels, dtype=np.float64)
        met.z_levels_host = lev.ctypes.data
    rc = load().lpm_workspace_bytes(C.byref(g), C.byref(met), C.byref(p), n_nuclides, C.byref(out))
    if rc:
        raise LpmError(rc, "lpm_workspace_bytes")
    return out.value


def schedule_born(n_particles, pid_offset, pid_stride, s_start, S, step) -> int:
    out = C.c_uint64()
    rc = load().lpm_schedule_born(n_particles, pid_offset, pid_stride, s_start, S, step, C.byref(out))
    if rc:
        raise LpmError(rc, "lpm_schedule_born")
    return out.value


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_0912_3223_b200 needs a CUDA device (sm_100); there is no CPU fallback")
    return torch


class Simulation:
    """One lpm_handle on the current CUDA device, created from a `workloads.Workload`-like object.

    Methods mirror the C entry points: release, step, concentration, deposition, counts, ...
    Device buffers (workspace, met snapshots, outputs) are torch tensors owned by this object or
    by the caller; H2D/D2H copies happen only in the explicit `*_host` helpers.
    """

    def __init__(self, w, *, steps_per_launch: int = 0, bin_every: Optional[int] = None, fields_dev=None,
                 stream=None, auto_release: bool = True, gather_sort: int = 0, dose: bool = False, dep_mode: int = 0, drift: bool = False, texel_pairs: int = 0,
                 ground_decay: bool = False):
        torch = _require_cuda()
        L = load()
        self._L = L
        self.w = w
        self.K = w.K
        self.torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        if fields_dev is None:
            f = w.fields()
            fields_dev = torch.from_numpy(np.ascontiguousarray(f)).to(self.device)
        assert fields_dev.dtype == torch.float32 and fields_dev.is_contiguous()
        self.fields_dev = fields_dev
        kz_mode = int(getattr(w, "kz_mode", 0))
        self.surface_dev = None
        if kz_mode == 1:
            self.surface_dev = torch.from_numpy(np.ascontiguousarray(w.surface(), dtype=np.float32)).to(self.device)
        nbytes = workspace_bytes(w.cgrid, w.capacity, w.K, w.compact, w.mgrid, w.nt, gather_sort, dose, kz_mode, dep_mode, drift, texel_pairs,
                                 getattr(w, "z_levels", None))
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._levels = None
        if getattr(w, "z_levels", None) is not None:
            self._levels = np.ascontiguousarray(w.z_levels, dtype=np.float64)
        self._create_args = dict(kz_mode=kz_mode, bin_every=w.bin_every if bin_every is None else bin_every, steps_per_launch=steps_per_launch,
                                 gather_sort=gather_sort, dose=dose, dep_mode=dep_mode, drift=drift, texel_pairs=texel_pairs,
                                 ground_decay=ground_decay, auto_release=auto_release)
        self._h = None
        self._create()

    def _create(self):
        """lpm_create on this object's workspace (which the library zeroes), then the rain box and the release."""
        w, a, L, torch = self.w, self._create_args, self._L, self.torch
        cg = _grid(w.cgrid)
        met = lpm_meteo(grid=_grid(w.mgrid), nt=w.nt, t0=w.t0, dt_snap=w.dt_snap, fields_dev=self.fields_dev.data_ptr(),
                        Kh=w.Kh, H_mix=w.H_mix, kz_min=w.kz_min, kz_mode=a["kz_mode"],
                        surface_dev=self.surface_dev.data_ptr() if self.surface_dev is not None else None)
        if self._levels is not None:
            met.z_levels_host = self._levels.ctypes.data
        nucs = (lpm_nuclide * w.K)(*[lpm_nuclide(n.half_life_s, n.vd, n.lambda_wet) for n in w.nuclides])
        prm = lpm_params(dt=w.dt, seed=w.seed, capacity=w.capacity,
                         boundary_mode=1 if w.boundary_mode == "absorb" else 0, compact=1 if w.compact else 0,
                         h_dep=w.h_dep, bin_every=a["bin_every"], steps_per_launch=a["steps_per_launch"], gather_sort=a["gather_sort"],
                         dose=1 if a["dose"] else 0, dep_mode=a["dep_mode"], drift=1 if a["drift"] else 0,
                         texel_pairs=a["texel_pairs"], ground_decay=1 if a["ground_decay"] else 0)
        h = C.c_void_p()
        with torch.cuda.stream(self.stream):
            rc = L.lpm_create(C.byref(cg), C.byref(met), nucs, w.K, C.byref(prm), self.workspace.data_ptr(), self.workspace.numel(),
                              self.stream.cuda_stream, C.byref(h))
        if rc:
            raise LpmError(rc, "lpm_create")
        self._h = h
        if w.rain is not None:
            self._ck(L.lpm_set_rain(h, w.rain.x0, w.rain.x1, w.rain.y0, w.rain.y1, w.rain.t_start, w.rain.t_end), "lpm_set_rain")
        if a["auto_release"] and w.release is not None:
            self.release(w.release)

    def restart(self):
        """lpm_restart: the same run again from step 0 on the same handle."""
        self._ck(self._L.lpm_restart(self._h), "lpm_restart")

    # ------------------------------------------------------------------ plumbing
    def _ck(self, rc, where):
        if rc:
            raise LpmError(rc, where, self._L.lpm_last_error(self._h).decode() if self._h else "")

    def close(self):
        if getattr(self, "_h", None):
            self._L.lpm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ the boundary calls
    def release(self, r):
        src = lpm_source(r.x, r.y, r.z, r.t_start, r.t_end)
        act = (C.c_double * self.K)(*r.total_activity[: self.K])
        self._ck(self._L.lpm_release(self._h, C.byref(src), act, r.n_particles, r.rate, r.pid_offset, r.pid_stride), "lpm_release")

    def step(self, n: int = 1):
        self._ck(self._L.lpm_step(self._h, n), "lpm_step")

    def bin_now(self):
        self._ck(self._L.lpm_bin_now(self._h), "lpm_bin_now")

    def concentration(self, out=None):
        g = self.w.cgrid
        if out is None:
            out = self.torch.empty((self.K, g.nz, g.ny, g.nx), dtype=self.torch.float32, device=self.device)
        self._ck(self._L.lpm_concentration(self._h, out.data_ptr()), "lpm_concentration")
        return out

    def dose(self, out=None):
        g = self.w.cgrid
        if out is None:
            out = self.torch.empty((self.K, g.nz, g.ny, g.nx), dtype=self.torch.float32, device=self.device)
        self._ck(self._L.lpm_dose(self._h, out.data_ptr()), "lpm_dose")
        return out

    def counts(self, out=None):
        g = self.w.cgrid
        if out is None:
            out = self.torch.empty((g.nz, g.ny, g.nx), dtype=self.torch.int32, device=self.device)
        self._ck(self._L.lpm_counts(self._h, out.data_ptr()), "lpm_counts")
        return out

    def deposition(self, out=None, f64: bool = False):
        g = self.w.cgrid
        dt = self.torch.float64 if f64 else self.torch.float32
        if out is None:
            out = self.torch.empty((self.K, g.ny, g.nx), dtype=dt, device=self.device)
        fn = self._L.lpm_deposition_f64 if f64 else self._L.lpm_deposition
        self._ck(fn(self._h, out.data_ptr()), "lpm_deposition")
        return out

    # host-buffer entry points: pinned CPU tensors in / out
    def upload_meteo(self, first: int, fields_host):
        """fields_host: CPU float32 tensor [n][nz][ny][nx][4] (pinned for full PCIe speed)."""
        assert fields_host.device.type == "cpu" and fields_host.is_contiguous() and fields_host.dtype == self.torch.float32
        self._ck(self._L.lpm_upload_meteo(self._h, first, fields_host.shape[0], fields_host.data_ptr()), "lpm_upload_meteo")

    def concentration_host(self, out):
        assert out.device.type == "cpu" and out.is_contiguous() and out.dtype == self.torch.float32
        self._ck(self._L.lpm_concentration_host(self._h, out.data_ptr()), "lpm_concentration_host")
        return out

    def deposition_host(self, out):
        assert out.device.type == "cpu" and out.is_contiguous() and out.dtype == self.torch.float32
        self._ck(self._L.lpm_deposition_host(self._h, out.data_ptr()), "lpm_deposition_host")
        return out

    def set_timing(self, on: bool = True):
        self._ck(self._L.lpm_set_timing(self._h, 1 if on else 0), "lpm_set_timing")

    def get_timing(self):
        out = (C.c_double * 14)()
        self._ck(self._L.lpm_get_timing(self._h, out), "lpm_get_timing")
        return dict(step_ms=out[0], step_launches=int(out[1]), bin_ms=out[2], bin_launches=int(out[3]),
                    particle_steps=out[4], binned_particles=out[5], sort_ms=out[6], sort_launches=int(out[7]),
                    born_particle_steps=out[8], bin_fused_launch_ms=out[9], bin_fused_launches=int(out[10]), bin_fused_prev_launch_ms=out[11],
                    bin_fused_born_particle_steps=out[12], bin_fused_prev_born_particle_steps=out[13])

    @property
    def touched_cells(self) -> int:
        n = C.c_uint64()
        self._ck(self._L.lpm_touched_cells(self._h, C.byref(n)), "lpm_touched_cells")
        return n.value

    @property
    def texel_pairs(self) -> bool:
        on = C.c_int32()
        self._ck(self._L.lpm_texel_pairs(self._h, C.byref(on)), "lpm_texel_pairs")
        return bool(on.value)

    @property
    def num_active(self) -> int:
        n = C.c_uint64()
        self._ck(self._L.lpm_num_active(self._h, C.byref(n)), "lpm_num_active")
        return n.value

    @property
    def step_index(self) -> int:
        n = C.c_uint64()
        self._ck(self._L.lpm_step_index(self._h, C.byref(n)), "lpm_step_index")
        return n.value

    @property
    def launch_count(self) -> int:
        n = C.c_uint64()
        self._ck(self._L.lpm_launch_count(self._h, C.byref(n)), "lpm_launch_count")
        return n.value

    def mass_scale(self):
        s = (C.c_double * self.K)()
        self._ck(self._L.lpm_mass_scale(self._h, s), "lpm_mass_scale")
        return np.array(list(s))

    def ledger(self):
        out = (C.c_double * (self.K * LEDGER_FIELDS))()
        self._ck(self._L.lpm_ledger(self._h, out), "lpm_ledger")
        return np.array(list(out)).reshape(self.K, LEDGER_FIELDS)

    def injected(self, step: int) -> int:
        n = C.c_uint64()
        self._ck(self._L.lpm_injected(self._h, step, C.byref(n)), "lpm_injected")
        return n.value

    def get_particles(self):
        """Device tensors: xyzq [n,4] f32, q1 [n] f32 or None, pid [n] (int64 view of uint32), status [n] u8."""
        t = self.torch
        cap = self.w.capacity
        xyzq = t.empty((cap, 4), dtype=t.float32, device=self.device)
        q1 = t.empty(cap, dtype=t.float32, device=self.device) if self.K > 1 else None
        pid = t.empty(cap, dtype=t.int32, device=self.device)
        st = t.empty(cap, dtype=t.uint8, device=self.device)
        n = C.c_uint64()
        self._ck(self._L.lpm_get_particles(self._h, xyzq.data_ptr(), q1.data_ptr() if q1 is not None else None,
                                           pid.data_ptr(), st.data_ptr(), C.byref(n)), "lpm_get_particles")
        n = n.value
        pid64 = pid[:n].to(t.int64) & 0xFFFFFFFF
        return dict(xyzq=xyzq[:n], q1=None if q1 is None else q1[:n], pid=pid64, status=st[:n], n=n)

    def get_particles_host(self):
        """numpy copy of the state as stored: x, y, z (f32), q [K,n] (the stored fp32 values as f64), scale [K]
        (lpm_mass_scale: the activity of a particle is q * scale, R8 - the product is left to the caller), pid, status."""
        p = self.get_particles()
        xyzq = p["xyzq"].cpu().numpy()
        q = [xyzq[:, 3].astype(np.float64)]
        if self.K > 1:
            q.append(p["q1"].cpu().numpy().astype(np.float64))
        return dict(x=xyzq[:, 0].copy(), y=xyzq[:, 1].copy(), z=xyzq[:, 2].copy(), q=np.stack(q), scale=self.mass_scale(),
                    pid=p["pid"].cpu().numpy().astype(np.uint64), status=p["status"].cpu().numpy())

    def set_particles(self, xyzq, q1=None, pid=None, status=None, step_index: int = 0):
        t = self.torch
        with t.cuda.stream(self.stream):   # the staging copies and the library's copies run on the handle's stream
            xyzq = xyzq.to(device=self.device, dtype=t.float32).contiguous()
            n = xyzq.shape[0]
            q1 = None if q1 is None else q1.to(device=self.device, dtype=t.float32).contiguous()
            pid = None if pid is None else pid.to(device=self.device, dtype=t.int64).to(t.int32).contiguous()
            status = None if status is None else status.to(device=self.device, dtype=t.uint8).contiguous()
            self._ck(self._L.lpm_set_particles(self._h, xyzq.data_ptr(), None if q1 is None else q1.data_ptr(),
                                               None if pid is None else pid.data_ptr(),
                                               None if status is None else status.data_ptr(), n, step_index), "lpm_set_particles")
        self.stream.synchronize()


# ---------------------------------------------------------------- micro-benchmarks
PROBE_KINDS = {"ffma": 0, "imad_lop": 1, "red_f64": 2, "red_u32": 3, "red_same": 4, "atoms": 5, "gather": 6, "smem_gather": 7, "gather32": 8}


def probe(kind: str, footprint_bytes: int = 0, scratch_bytes: int = 1 << 28, reps: int = 5) -> float:
    """lpm_probe: operations per second of one micro-benchmark (see include/lpm.h)."""
    torch = _require_cuda()
    scratch = torch.zeros(scratch_bytes // 4, dtype=torch.float32, device="cuda")
    out = C.c_double()
    rc = load().lpm_probe(PROBE_KINDS[kind], footprint_bytes, scratch.data_ptr(), scratch_bytes, reps, C.byref(out),
                          torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_probe")
    return out.value


# ---------------------------------------------------------------- stand-alone parity kernels
def philox_kernel(seed, step, stream_id, pid0, n):
    torch = _require_cuda()
    out = torch.empty((n, 4), dtype=torch.int32, device="cuda")
    rc = load().lpm_test_philox(seed, step, stream_id, pid0, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_test_philox")
    return out.cpu().numpy().view(np.uint32)


def curand_philox_kernel(seed, step, pid0, n):
    torch = _require_cuda()
    out = torch.empty((n, 4), dtype=torch.int32, device="cuda")
    rc = load().lpm_test_curand_philox(seed, step, pid0, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_test_curand_philox")
    return out.cpu().numpy().view(np.uint32)


def box_muller_kernel(words):
    """normals of raw Philox words: words uint32 [n][4] (numpy) -> float32 [n][3]."""
    torch = _require_cuda()
    r = torch.from_numpy(np.ascontiguousarray(words, dtype=np.uint32).view(np.int32)).cuda()
    out = torch.empty((r.shape[0], 3), dtype=torch.float32, device="cuda")
    rc = load().lpm_test_box_muller(r.data_ptr(), r.shape[0], out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_test_box_muller")
    return out.cpu().numpy()


def normals_kernel(seed, step, pid0, n):
    torch = _require_cuda()
    out = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    rc = load().lpm_test_normals(seed, step, pid0, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_test_normals")
    return out.cpu().numpy()


def sample_kernel(w, t, xyz):
    """Met sampling R4 of workload `w` at time t for points xyz [n,3] (numpy) -> [n,4] numpy."""
    torch = _require_cuda()
    f = torch.from_numpy(np.ascontiguousarray(w.fields())).cuda()
    pts = np.zeros((xyz.shape[0], 4), dtype=np.float32)
    pts[:, :3] = xyz
    p = torch.from_numpy(pts).cuda()
    out = torch.empty_like(p)
    met = lpm_meteo(grid=_grid(w.mgrid), nt=w.nt, t0=w.t0, dt_snap=w.dt_snap, fields_dev=f.data_ptr(), Kh=w.Kh,
                    H_mix=w.H_mix, kz_min=w.kz_min)
    levels = None
    if getattr(w, "z_levels", None) is not None:
        levels = np.ascontiguousarray(w.z_levels, dtype=np.float64)
        met.z_levels_host = levels.ctypes.data
    rc = load().lpm_test_sample(C.byref(met), t, p.data_ptr(), p.shape[0], out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        raise LpmError(rc, "lpm_test_sample")
    torch.cuda.synchronize()
    return out.cpu().numpy()


SAMPLE_STATIC_MAX_CELLS = 262144   # LPM_SAMPLE_STATIC_MAX_CELLS of include/lpm.h


def sample_static(w, t, xyz):
    """lpm_sample_static: the met sampling of `sample_kernel`, for users who must not allocate on the device.

    Same arguments, same result bit for bit.  The difference is where the two temporary fields of the sampling path
    live: `sample_kernel` (lpm_test_sample) takes them from cudaMalloc on every call, this call keeps them in a 12 MiB
    array built into the library.  That is what a caller needs whose GPU memory belongs to someone else's pool, or who
    cannot have cudaMalloc / cudaFree stop every other stream of the device for a moment.  Limit: the met grid of `w`
    may have at most SAMPLE_STATIC_MAX_CELLS cells (LpmError with status ERR_WORKSPACE_TOO_SMALL beyond).  All calls
    share the one array: keep them on one stream, one after the other.  (The tensors created here are this wrapper's
    inputs and outputs, which a real caller already owns; the C call itself allocates nothing.)"""
    torch = _require_cuda()
    f = torch.from_numpy(np.ascontiguousarray(w.fields())).cuda()
    pts = np.zeros((xyz.shape[0], 4), dtype=np.float32)
    pts[:, :3] = xyz
    p = torch.from_numpy(pts).cuda()
    out = torch.empty_like(p)
    met = lpm_meteo(grid=_grid(w.mgrid), nt=w.nt, t0=w.t0, dt_snap=w.dt_snap, fields_dev=f.data_ptr(), Kh=w.Kh,
                    H_mix=w.H_mix, kz_min=w.kz_min)
    levels = None
    if getattr(w, "z_levels", None) is not None:
        levels = np.ascontiguousarray(w.z_levels, dtype=np.float64)
        met.z_levels_host = levels.ctypes.data
    rc = load().lpm_sample_static(C.byref(met), t, p.data_ptr(), p.shape[0], out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc:
        g = w.mgrid
        raise LpmError(rc, "lpm_sample_static", f"(met grid {g.nx} x {g.ny} x {g.nz} = {g.nx * g.ny * g.nz} cells; the built-in scratch "
                                                f"array holds at most {SAMPLE_STATIC_MAX_CELLS})" if rc == ERR_WORKSPACE_TOO_SMALL else "")
    torch.cuda.synchronize()   # the C call is asynchronous; `out` is read on the host next
    return out.cpu().numpy()
