"""CPU-side checks of the C-ABI library: it loads, exports every declared symbol, and its
host-only logic (workspace sizing, R9 schedule) agrees with the oracle's definition."""
import ctypes
import re
import os

import numpy as np
import pytest

import paper_0912_3223_b200 as lpm
from paper_0912_3223_b200 import binding
from paper_0912_3223_b200.build import build
from helpers import custom, uniform_met
from oracle import oracle as orc
from workloads import make

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "lpm.h")).read()
    declared = set(re.findall(r"\b(lpm_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"lpm_handle"}
    assert declared == set(binding.SYMBOLS)
    L = ctypes.CDLL(binding.LIB_PATH)
    for s in declared:
        assert hasattr(L, s), s


def test_version_and_status_strings():
    assert lpm.version() == 100
    assert lpm.status_string(0) == "ok"
    assert "fallback" in lpm.status_string(-2)


def test_workspace_bytes_monotone_and_errors():
    w = make("c2")
    a = lpm.workspace_bytes(w.cgrid, 1000, 1, False)
    b = lpm.workspace_bytes(w.cgrid, 2000, 1, False)
    c = lpm.workspace_bytes(w.cgrid, 2000, 2, True)
    assert a < b < c
    cells = w.cgrid.nx * w.cgrid.ny * w.cgrid.nz
    assert a >= 16 * 1000 + 12 * cells
    with pytest.raises(lpm.LpmError):
        lpm.workspace_bytes(w.cgrid, 0, 1, False)
    with pytest.raises(lpm.LpmError):
        lpm.workspace_bytes(w.cgrid, 10, 3, False)


def test_met_grid_beyond_the_32_bit_texel_index_is_refused():
    """The step kernel folds the blended-buffer number into one 32-bit texel index (16 buffers when nt > 1): a met grid of
    2^28 cells or more with several snapshots must be refused, not gathered from wrapped addresses.  With one snapshot
    there is one buffer, and the limit is grid_ok's 2^31."""
    from workloads import Grid
    cg = Grid(8, 8, 4, 0.0, 0.0, 0.0, 100.0, 100.0, 100.0)
    at = Grid(1024, 1024, 256, 0.0, 0.0, 0.0, 100.0, 100.0, 10.0)        # 2^28 cells
    below = Grid(1024, 1024, 255, 0.0, 0.0, 0.0, 100.0, 100.0, 10.0)
    with pytest.raises(lpm.LpmError):
        lpm.workspace_bytes(cg, 1000, 1, False, mgrid=at, nt=2)
    assert lpm.workspace_bytes(cg, 1000, 1, False, mgrid=below, nt=2) > 16 * 16 * 1024 * 1024 * 255
    assert lpm.workspace_bytes(cg, 1000, 1, False, mgrid=at, nt=1) > 16 * 1024 * 1024 * 256
    # straight through the C ABI: lpm_create refuses the same grid before it looks for a device
    L = binding.load()
    met = binding.lpm_meteo(grid=binding._grid(at), nt=2, t0=0.0, dt_snap=3600.0, fields_dev=256, Kh=1.0, H_mix=1000.0, kz_min=0.0)
    nuc = (binding.lpm_nuclide * 1)(binding.lpm_nuclide(1.0, 0.0, 0.0))
    prm = binding.lpm_params(dt=1.0, seed=1, capacity=16, h_dep=1000.0)
    h = ctypes.c_void_p()
    rc = L.lpm_create(ctypes.byref(binding._grid(cg)), ctypes.byref(met), nuc, 1, ctypes.byref(prm), 256, 1 << 40, None, ctypes.byref(h))
    assert rc == binding.ERR_INVALID_ARG and not h.value


def test_workspace_bytes_texel_pairs_rule():
    """lpm_params.texel_pairs (B8): 16 more bytes per met cell and fused step when on; auto from
    capacity >= 16 x met cells; never for the physics the pair kernels are not instantiated for."""
    w = make("c2")
    mc = w.mgrid.nx * w.mgrid.ny * w.mgrid.nz
    kw = dict(mgrid=w.mgrid, nt=3)
    off = lpm.workspace_bytes(w.cgrid, 1000, 1, False, texel_pairs=-1, **kw)
    on = lpm.workspace_bytes(w.cgrid, 1000, 1, False, texel_pairs=1, **kw)
    assert on - off == 16 * 16 * mc
    assert lpm.workspace_bytes(w.cgrid, 1000, 1, False, **kw) == off                                  # auto, small ensemble
    big, cap = lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, **kw), lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, texel_pairs=-1, **kw)
    assert big - cap == 16 * 16 * mc                                                                # auto, large ensemble
    assert lpm.workspace_bytes(w.cgrid, 16 * mc - 1, 1, False, **kw) == lpm.workspace_bytes(w.cgrid, 16 * mc - 1, 1, False, texel_pairs=-1, **kw)
    for no in (dict(dep_mode=1), dict(drift=True), dict(kz_mode=1), dict(z_levels=np.linspace(0.0, 1000.0, w.mgrid.nz))):
        a = lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, texel_pairs=1, **kw, **no)
        b = lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, texel_pairs=-1, **kw, **no)
        assert a == b, no
    assert lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, mgrid=w.mgrid, nt=1, texel_pairs=1) == \
        lpm.workspace_bytes(w.cgrid, 16 * mc, 1, False, mgrid=w.mgrid, nt=1, texel_pairs=-1)


def test_no_device_is_an_error_not_a_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        lpm.Simulation(make("c1", scale=0.01))
    # straight through the C ABI: lpm_create must refuse without a device
    L = binding.load()
    w = make("c1", scale=0.01)
    cg = binding._grid(w.cgrid)
    met = binding.lpm_meteo(grid=cg, nt=1, t0=0.0, dt_snap=3600.0, fields_dev=256, Kh=1.0, H_mix=1000.0, kz_min=0.0)
    nuc = (binding.lpm_nuclide * 1)(binding.lpm_nuclide(1.0, 0.0, 0.0))
    prm = binding.lpm_params(dt=1.0, seed=1, capacity=16, h_dep=1000.0)
    h = ctypes.c_void_p()
    rc = L.lpm_create(ctypes.byref(cg), ctypes.byref(met), nuc, 1, ctypes.byref(prm), 256, 1 << 30, None, ctypes.byref(h))
    assert rc == binding.ERR_NO_DEVICE and not h.value


@pytest.mark.parametrize("N,S,off,stride", [(1000, 7, 0, 1), (1_000_000, 720, 0, 1), (10, 3, 0, 1), (1000, 7, 3, 10),
                                            (12345, 100, 99, 100), (5, 1, 0, 1), (3, 10, 0, 1)])
def test_schedule_matches_oracle_injection_log(N, S, off, stride):
    """lpm_schedule_born (closed form) == the oracle's literal R9 loop, step by step."""
    w = custom(uniform_met(), n=N, dt=10.0, t_rel=(20.0, 20.0 + 10.0 * S), n_steps=S + 5, pid_offset=off, pid_stride=stride)
    sim = orc.OracleSim(w)
    cum = 0
    for s in range(S + 5):
        sim.step(1)
        cum += sim.injected(s)
        assert lpm.schedule_born(N, off, stride, 2, S, s) == cum
    assert cum == len(range(off, N, stride))
    assert lpm.schedule_born(N, off, stride, 2, S, 1) == 0
