"""Pins of the oracle against things other than itself.

Each test names the plausible mistake it is there to catch."""
import math

import numpy as np
import pytest
from scipy import ndimage, stats

from helpers import T_I131, custom, read_golden, uniform_met
from oracle import oracle as orc
from workloads import Grid, Nuclide, RainBox, make


# ------------------------------------------------------------------ P1 Philox
def test_philox_known_answers():
    """wrong multiplier / round count / operand order in the Philox round."""
    rows = read_golden("philox_kat.txt")
    assert len(rows) == 5
    for r in rows:
        v = [int(h, 16) for h in r]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(o) for o in out] == v[6:10]


def test_philox_counter_layout():
    """ctr = (step, stream, pid_lo, pid_hi), key = (seed_lo, seed_hi) (R1)."""
    rows = read_golden("philox_kat.txt")
    assert [int(o) for o in orc.philox_draw(1, 0, 0)] == [int(h, 16) for h in rows[3][6:10]]
    assert [int(o) for o in orc.philox_draw(1, 7, 3)] == [int(h, 16) for h in rows[4][6:10]]
    a = orc.philox_draw((5 << 32) | 9, (3 << 32) | 2, 11, 4)
    b = orc.philox4x32_10([11, 4, 2, 3], [9, 5])
    assert list(a) == list(b)


# ------------------------------------------------------------------ P2 uniforms / normals
def test_worked_uniforms_normals():
    rows = {r[0]: [float(x) for x in r[1:]] for r in read_golden("worked_step.txt")}
    u = orc.uniforms(orc.philox_draw(1, 7, 3))
    np.testing.assert_allclose(u, rows["u"], atol=5e-10)
    n = orc.normals(1, 7, 3)
    np.testing.assert_allclose(n, rows["n"], atol=5e-9)


def test_uniform_ranges_exact():
    """u1,u3 in (0,1] (log never sees 0), u2,u4 in [0,1); exact multiples of 2^-24."""
    u = orc.uniforms([0, 0, 0xFFFFFFFF, 0xFFFFFFFF])
    assert u[0] == 2.0 ** -24 and u[1] == 0.0 and u[2] == 1.0 and u[3] == 1.0 - 2.0 ** -24
    u = orc.uniforms([0x12345678, 0x9ABCDEF0, 0x0F0F0F0F, 0xDEADBEEF])
    assert all(float(x) * 2 ** 24 == int(float(x) * 2 ** 24) for x in u)


def test_normals_distribution():
    """N(0,1): mean, variance, KS, independence of the three components, |n| bound (R3)."""
    N = 200_000
    z = np.array([orc.normals(12345, p, s) for p in range(N // 20) for s in range(20)])
    assert z.shape == (N, 3)
    for c in range(3):
        assert abs(z[:, c].mean()) < 4.0 / math.sqrt(N)
        assert abs(z[:, c].var() - 1.0) < 4.0 * math.sqrt(2.0 / N)
        assert stats.kstest(z[:, c], "norm").pvalue > 1e-3
    cc = np.corrcoef(z.T)
    assert np.all(np.abs(cc - np.eye(3)) < 4.0 / math.sqrt(N))
    assert np.abs(z).max() <= math.sqrt(48.0 * math.log(2.0)) + 1e-12
    # n0, n1 share a radius: n0^2 + n1^2 = -2 ln u1 is chi^2 with 2 dof (catches sin/cos of different angles)
    assert stats.kstest(z[:, 0] ** 2 + z[:, 1] ** 2, "chi2", args=(2,)).pvalue > 1e-3


# ------------------------------------------------------------------ P3 one full step
def test_worked_full_step():
    rows = {r[0]: [float(x) for x in r[1:]] for r in read_golden("worked_step.txt")}
    w = make("c1").replace(release=None)
    sim = orc.OracleSim(w)
    x0 = rows["x_old"]
    sim.set_particles([x0[0]], [x0[1]], [x0[2]], [[1.0]], pid=[7])
    sim.set_step_index(3)
    sim.step(1)
    p = sim.particles()
    np.testing.assert_allclose([p["x"][0], p["y"][0], p["z"][0]], rows["x_new"], atol=2e-6)
    assert abs(sim.sigma_h() - 31.6227766) < 1e-6


# ------------------------------------------------------------------ P4 Gaussian puff
def test_gaussian_puff_no_boundaries():
    """sum of iid normals: x ~ N(x0 + u t, 2 K t) exactly at every step (north_star check 1).
    Catches: dropped advection term, sigma without the factor 2, wrong axis pairing."""
    N, steps, dt = 40_000, 40, 10.0
    w = custom(uniform_met(u=5.0, v=-2.0, w=0.5, kz=5.0), Kh=50.0, H=1.0e9, dt=dt, n=N, n_steps=steps,
               src=(10.0, 20.0, 5.0e5), seed=7)
    sim = orc.OracleSim(w)
    sim.step(steps)
    p = sim.particles()
    t = steps * dt
    for arr, mean, var in ((p["x"], 10.0 + 5.0 * t, 2 * 50.0 * t), (p["y"], 20.0 - 2.0 * t, 2 * 50.0 * t),
                           (p["z"], 5.0e5 + 0.5 * t, 2 * 5.0 * t)):
        assert abs(arr.mean() - mean) < 4.0 * math.sqrt(var / N)
        assert abs(arr.var() / var - 1.0) < 4.0 * math.sqrt(2.0 / N)
        assert stats.kstest((arr - mean) / math.sqrt(var), "norm").pvalue > 1e-3
    assert abs(np.corrcoef(p["x"], p["y"])[0, 1]) < 4.0 / math.sqrt(N)


def test_c1_puff_with_ground_reflection():
    """C1 at t = 1000 s: x,y Gaussian, z folded normal (SURVEY P4 values, re-derived via scipy)."""
    rows = {r[0]: float(r[1]) for r in read_golden("closed_forms.txt")}
    w = make("c1")
    sim = orc.OracleSim(w)
    sim.step(100)
    p = sim.particles()
    N = w.release.n_particles
    assert sim.n == N
    assert abs(p["x"].mean() - 5000.0) < 4.0 * math.sqrt(1.0e5 / N)
    assert abs(p["x"].var() / 1.0e5 - 1.0) < 4.0 * math.sqrt(2.0 / N)
    assert abs(p["y"].var() / 1.0e5 - 1.0) < 4.0 * math.sqrt(2.0 / N)
    fold = stats.foldnorm(c=50.0 / 100.0, scale=100.0)
    assert abs(fold.mean() - rows["Ez"]) < 1e-3 and abs(fold.var() - rows["Varz"]) < 1e-1
    assert abs(p["z"].mean() - rows["Ez"]) < 4.0 * math.sqrt(rows["Varz"] / N)
    assert stats.kstest(p["z"], fold.cdf).pvalue > 1e-3
    assert p["z"].min() >= 0.0 and p["z"].max() <= 1000.0


# ------------------------------------------------------------------ P5 decay
def test_decay_exact():
    rows = {r[0]: float(r[1]) for r in read_golden("closed_forms.txt")}
    w = make("c1", scale=0.001)
    sim = orc.OracleSim(w)
    m0 = sim_m0 = w.release.total_activity[0] / w.release.n_particles
    sim.step(100)
    p = sim.particles()
    ratio = p["m"][0] / m0
    assert np.all(np.abs(ratio - 2.0 ** (-1000.0 / T_I131)) < 1e-12)
    assert abs(ratio[0] - rows["decay_I131_1000s"]) < 5e-10
    assert abs(math.log(2) / T_I131 / rows["lambda_I131"] - 1) < 1e-6
    assert abs(math.log(2) / (30.17 * 365.25 * 86400) / rows["lambda_Cs137"] - 1) < 1e-4
    assert sim_m0 == m0


# ------------------------------------------------------------------ P7 interpolation
def _field_from(fn, g, nt=1, t0=0.0, dts=3600.0):
    xc = g.x0 + (np.arange(g.nx) + 0.5) * g.dx
    yc = g.y0 + (np.arange(g.ny) + 0.5) * g.dy
    zc = g.z0 + (np.arange(g.nz) + 0.5) * g.dz
    Z, Y, X = np.meshgrid(zc, yc, xc, indexing="ij")
    out = np.zeros((nt, g.nz, g.ny, g.nx, 4), dtype=np.float32)
    for s in range(nt):
        for c in range(4):
            out[s, ..., c] = fn(c, t0 + s * dts, X, Y, Z)
    return out


def test_interpolation_affine_and_layout():
    """reproduces affine fields exactly inside the cell-centre hull; distinct coefficients per
    axis and per component catch transposed strides and swapped components; affine in t."""
    g = Grid(7, 5, 4, -10.0, 3.0, 0.0, 2.0, 3.0, 5.0)
    coef = [(1.0, 0.5, -0.25, 0.125, 2.0), (-2.0, 0.75, 0.5, -0.5, -1.0), (0.5, -1.0, 2.0, 0.25, 0.5), (3.0, 0.125, 0.25, 1.0, 0.25)]

    def fn(c, t, X, Y, Z):
        a, bx, by, bz, bt = coef[c]
        return a + bx * X + by * Y + bz * Z + bt * (t / 3600.0)
    f = _field_from(fn, g, nt=3)
    rng = np.random.default_rng(0)
    for _ in range(200):
        x = rng.uniform(g.x0 + 0.5 * g.dx, g.x0 + (g.nx - 0.5) * g.dx)
        y = rng.uniform(g.y0 + 0.5 * g.dy, g.y0 + (g.ny - 0.5) * g.dy)
        z = rng.uniform(g.z0 + 0.5 * g.dz, g.z0 + (g.nz - 0.5) * g.dz)
        t = rng.uniform(0.0, 7200.0)
        out = orc.sample_met(g, 3, 0.0, 3600.0, f, t, x, y, z)
        ref = [fn(c, t, x, y, z) for c in range(4)]
        np.testing.assert_allclose(out, ref, rtol=0, atol=2e-5)   # fp32 field values, fp32 time weight


def test_interpolation_vs_scipy_map_coordinates():
    """random field: trilinear + edge clamp == scipy.ndimage.map_coordinates(order=1, mode='nearest')."""
    g = Grid(9, 6, 5, 100.0, -50.0, 0.0, 10.0, 20.0, 30.0)
    rng = np.random.default_rng(1)
    f = rng.normal(size=(1, g.nz, g.ny, g.nx, 4)).astype(np.float32)
    pts = np.stack([rng.uniform(g.x0 - 30, g.x0 + g.nx * g.dx + 30, 300),
                    rng.uniform(g.y0 - 30, g.y0 + g.ny * g.dy + 30, 300),
                    rng.uniform(-20, g.nz * g.dz + 20, 300)], axis=1)
    for c in range(4):
        cz = (pts[:, 2] - g.z0) / g.dz - 0.5
        cy = (pts[:, 1] - g.y0) / g.dy - 0.5
        cx = (pts[:, 0] - g.x0) / g.dx - 0.5
        ref = ndimage.map_coordinates(f[0, ..., c].astype(np.float64), [cz, cy, cx], order=1, mode="nearest")
        got = np.array([orc.sample_met(g, 1, 0.0, 3600.0, f, 0.0, *p)[c] for p in pts])
        np.testing.assert_allclose(got, ref, atol=1e-12)


def test_time_weight_clamps():
    assert orc.time_weight(1, 0.0, 3600.0, 5000.0) == (0, 0.0)
    assert orc.time_weight(3, 0.0, 3600.0, -10.0) == (0, 0.0)
    assert orc.time_weight(3, 0.0, 3600.0, 1800.0) == (0, 0.5)
    assert orc.time_weight(3, 0.0, 3600.0, 3600.0) == (1, 0.0)
    assert orc.time_weight(3, 0.0, 3600.0, 7200.0) == (1, 1.0)
    assert orc.time_weight(3, 0.0, 3600.0, 9000.0) == (1, 1.0)


def test_deterministic_euler_in_affine_wind():
    """K = 0: forward Euler with the wind at the OLD position (Eq.(1)) in u = a + b*y, v = c has the
    closed form x_n = x0 + n dt a + b dt (n y0 + c dt n(n-1)/2).  Catches sampling at the new position,
    x/y transposition of the field, wrong component order."""
    a, b, c, dt, n = 2.0, 0.01, 1.5, 10.0, 25
    g = Grid(40, 40, 4, -2000.0, -2000.0, 0.0, 100.0, 100.0, 100.0)
    w = custom(lambda t, Z, Y, X: (a + b * Y, c, 0.0, 0.0), grid=g, Kh=0.0, H=1.0e9, dt=dt, n=3, n_steps=n,
               src=(-300.0, -400.0, 150.0))
    sim = orc.OracleSim(w)
    sim.step(n)
    p = sim.particles()
    x0, y0 = -300.0, -400.0
    xn = x0 + n * dt * a + b * dt * (n * y0 + c * dt * n * (n - 1) / 2.0)
    np.testing.assert_allclose(p["y"], y0 + n * c * dt, atol=1e-9)
    np.testing.assert_allclose(p["x"], xn, atol=2e-4)   # fp32 field values
    np.testing.assert_allclose(p["z"], 150.0, atol=0)
