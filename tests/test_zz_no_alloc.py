"""lpm_sample_static, the met sampler for callers that must not allocate device memory, against lpm_test_sample.

Who needs it: code that runs where a raw cudaMalloc is not an option - all of the GPU's memory already belongs to the host
application's own pool (so the call fails, or takes bytes somebody else has planned with), or other streams of the device
must keep running (cudaMalloc and cudaFree stop the whole device for a moment).  lpm_test_sample takes its two temporary
fields from cudaMalloc on every call; lpm_sample_static keeps them in one array built into the library, shared by all
calls and never cleared between them.  So the things to check are exactly the ones that sharing can break:

  - the result equals the allocating path's (same kernels: bit for bit, hence also within the 2e-5 x field scale + 1e-6
    the met-sampling parity tests allow against the oracle) on TWO CALLS IN A ROW that differ in grid, snapshot count and
    time, i.e. the second call finds the first call's field in the array;
  - a field of non-finite values left behind does not leak into a later, smaller call through the pad texel that the
    sampler reads with weight zero;
  - a grid of exactly the stated maximum works, one cell more is refused with a clear status before anything runs.

This file sorts after every other test file on purpose (pytest -x stops at the first failure): it must pass on its own in
a fresh process, where its first call is the one that looks up the array's device address, and at the end of the whole
suite.
"""
import ctypes

import numpy as np
import pytest

from helpers import custom, uniform_met
from workloads import Grid, make

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lpm():
    import torch
    assert torch.cuda.is_available()
    from paper_0912_3223_b200.build import build
    build()
    import paper_0912_3223_b200 as m
    return m


def _points(g, n, seed, H):
    """Seeded points inside, on the faces of and well outside the met grid (the sampler clamps at the edges)."""
    rng = np.random.default_rng(seed)
    lo = np.array([g.x0 - 2 * g.dx, g.y0 - 2 * g.dy, g.z0 - g.dz])
    hi = np.array([g.x0 + (g.nx + 2) * g.dx, g.y0 + (g.ny + 2) * g.dy, g.z0 + (g.nz + 1) * g.dz])
    xyz = rng.uniform(lo, hi, (n, 3)).astype(np.float32)
    xyz[:6] = [[g.x0, g.y0, g.z0], [g.x0 + g.nx * g.dx, g.y0, 0], [g.x0 + 0.5 * g.dx, g.y0 + 0.5 * g.dy, 0.5 * g.dz],
               [1e7, -1e7, 1e5], [0, 0, 0], [1, 1, H]]
    return xyz


def _same(got, want, w, what):
    scale = np.abs(w.fields()).reshape(-1, 4).max(axis=0)
    assert np.all(np.isfinite(got)), what
    err = np.abs(got.astype(np.float64) - want.astype(np.float64))
    assert np.all(err <= 2e-5 * scale + 1e-6), (what, err.max(axis=0))     # the tolerance of test_met_sampling
    assert np.array_equal(got, want), (what, err.max(axis=0))              # same kernels, same inputs: identical


def _smooth(t, Z, Y, X):
    return (3.0 * np.sin(X / 900.0) + t / 3600.0, 2.0 * np.cos(Y / 700.0), 0.02 * np.sin(Z / 300.0), 1.0 + Z / 150.0)


def test_two_calls_in_a_row_equal_the_allocating_path(lpm):
    """Call 1: a 100 x 100 x 20 window of c2's met grid, 3 snapshots, t inside the second interval (pair + blend path).
    Call 2, straight after it: c1's 60 x 60 x 10 grid with its single snapshot (transpose path) - a smaller field written
    over the remains of the first.  Call 3: the first one again at another time.  The references come from
    lpm_test_sample, which starts from fresh cudaMalloc'ed buffers every time."""
    a = make("c2", scale=1e-4)
    g = a.mgrid
    a = a.replace(mgrid=Grid(100, 100, g.nz, g.x0, g.y0, g.z0, g.dx, g.dy, g.dz))
    b = make("c1", scale=1e-4)
    assert a.nt > 1 and b.nt == 1
    assert b.mgrid.nx * b.mgrid.ny * b.mgrid.nz < a.mgrid.nx * a.mgrid.ny * a.mgrid.nz <= lpm.binding.SAMPLE_STATIC_MAX_CELLS
    pa, pb = _points(a.mgrid, 4000, 3, a.H_mix), _points(b.mgrid, 3001, 4, b.H_mix)
    got = [lpm.sample_static(a, 4321.0, pa), lpm.sample_static(b, 10.0, pb), lpm.sample_static(a, 100.0, pa)]
    want = [lpm.sample_kernel(a, 4321.0, pa), lpm.sample_kernel(b, 10.0, pb), lpm.sample_kernel(a, 100.0, pa)]
    for i, (x, y, w) in enumerate(zip(got, want, (a, b, a))):
        _same(x, y, w, f"call {i + 1}")
    assert not np.array_equal(got[0], got[2])    # the two times really give different fields


def test_non_finite_leftovers_do_not_reach_the_next_call(lpm):
    """The array keeps the last call's contents.  First a 4 x 4 x 3 field of +inf (48 texels), then a single-level
    4 x 4 x 1 grid: its pad texel, read with weight 0 behind the 16th texel, sits where the first call left an inf, and
    0 x inf would be a NaN.  lpm_sample_static clears that texel on every call."""
    inf = float("inf")
    g3 = Grid(4, 4, 3, -200.0, -200.0, 0.0, 100.0, 100.0, 100.0)
    g1 = Grid(4, 4, 1, -200.0, -200.0, 0.0, 100.0, 100.0, 100.0)
    poison = custom(uniform_met(inf, inf, inf, inf), grid=g3, n=0)
    flat = custom(_smooth, grid=g1, n=0)
    p3, p1 = _points(g3, 500, 5, 300.0), _points(g1, 777, 6, 100.0)
    assert not np.any(np.isfinite(lpm.sample_static(poison, 0.0, p3)[:, :3]))
    _same(lpm.sample_static(flat, 0.0, p1), lpm.sample_kernel(flat, 0.0, p1), flat, "single level after a field of inf")


def test_the_stated_maximum_works_and_one_cell_more_is_refused(lpm):
    """LPM_SAMPLE_STATIC_MAX_CELLS = 262144 = 64^3 met cells fill the built-in array to its last byte (two snapshots:
    both the pair buffer and the blended field are in use); 65 x 64 x 64 is refused with WORKSPACE_TOO_SMALL - the
    built-in array is this call's workspace - before any pointer is touched (the pointers passed here are not even valid)."""
    from paper_0912_3223_b200 import binding
    g = Grid(64, 64, 64, -3200.0, -3200.0, 0.0, 100.0, 100.0, 25.0)
    assert g.nx * g.ny * g.nz == binding.SAMPLE_STATIC_MAX_CELLS
    w = custom(_smooth, grid=g, nt=2, dt_snap=3600.0, n=0)
    p = _points(g, 5000, 7, 1600.0)
    _same(lpm.sample_static(w, 1234.5, p), lpm.sample_kernel(w, 1234.5, p), w, "grid of the maximum size")
    # non-uniform levels go through the same entry point (levels are copied on the host, no device allocation either)
    zl = np.cumsum(np.linspace(10.0, 60.0, 16))
    wl = custom(_smooth, grid=Grid(32, 32, 16, -1600.0, -1600.0, 0.0, 100.0, 100.0, 100.0), nt=2, n=0).replace(z_levels=zl)
    pl = _points(wl.mgrid, 2000, 8, 600.0)
    _same(lpm.sample_static(wl, 900.0, pl), lpm.sample_kernel(wl, 900.0, pl), wl, "non-uniform levels")

    L = binding.load()
    big = binding.lpm_meteo(grid=binding._grid(Grid(65, 64, 64, 0.0, 0.0, 0.0, 1.0, 1.0, 1.0)), nt=2, t0=0.0, dt_snap=1.0,
                            fields_dev=256, Kh=0.0, H_mix=1.0, kz_min=0.0)
    assert L.lpm_sample_static(ctypes.byref(big), 0.5, 256, 1, 256, None) == binding.ERR_WORKSPACE_TOO_SMALL
    with pytest.raises(lpm.LpmError, match="at most 262144"):
        lpm.sample_static(custom(uniform_met(1.0), grid=Grid(65, 64, 64, 0.0, 0.0, 0.0, 1.0, 1.0, 1.0), n=0), 0.0, p[:4])
    # and the array is still good afterwards
    _same(lpm.sample_static(wl, 900.0, pl), lpm.sample_kernel(wl, 900.0, pl), wl, "after a refused call")
