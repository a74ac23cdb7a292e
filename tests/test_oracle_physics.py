"""More pins of the oracle: reflection, deposition closed forms, ledger, binning, schedule,
compaction, boundaries."""
import math

import numpy as np
import pytest
from scipy import stats

from helpers import T_I131, custom, uniform_met
from oracle import oracle as orc
from dataclasses import replace as dataclasses_replace

from workloads import Grid, Nuclide, RainBox, Release, make


# ------------------------------------------------------------------ P8 reflection
def test_well_mixed_under_reflection():
    """constant Kz, reflecting walls: a z-uniform cloud stays uniform; z in [0, H] always.
    Catches a wrong fold (e.g. z = H - (z - H) written as z = H + ...)."""
    H, N = 400.0, 20_000
    w = custom(uniform_met(kz=50.0), H=H, dt=10.0, n=0, n_steps=30, seed=3)
    sim = orc.OracleSim(w)
    rng = np.random.default_rng(5)
    z0 = rng.uniform(0, H, N)
    sim.set_particles(np.zeros(N), np.zeros(N), z0, [np.ones(N)], pid=np.arange(N))
    sim.step(30)
    z = sim.particles()["z"]
    assert z.min() >= 0.0 and z.max() <= H
    hist, _ = np.histogram(z, bins=20, range=(0, H))
    assert stats.chisquare(hist).pvalue > 1e-3


def test_reflection_single_cases():
    """z' = -z' below ground; z' = 2H - z' above H (R6): hand-computed from the worked normal n2."""
    n2 = orc.normals(1, 7, 3)[2]           # 1.119952999 (pinned in test_worked_uniforms_normals)
    for z_old, H in ((2.0, 1000.0), (995.0, 1000.0)):
        w = custom(uniform_met(kz=5.0), H=H, dt=10.0, n=0, seed=1)
        for sign_pid in (7,):
            sim = orc.OracleSim(w)
            sim.set_particles([0.0], [0.0], [z_old], [[1.0]], pid=[sign_pid])
            sim.set_step_index(3)
            sim.step(1)
            z_free = z_old + 10.0 * n2
            want = 2 * H - z_free if z_free > H else abs(z_free)
            assert abs(sim.particles()["z"][0] - want) < 1e-9
    # downward case: find a (pid, step) with a strongly negative n2
    for pid in range(200):
        n2 = orc.normals(1, pid, 0)[2]
        if n2 < -1.0:
            break
    w = custom(uniform_met(kz=5.0), H=1000.0, dt=10.0, n=0, seed=1)
    sim = orc.OracleSim(w)
    sim.set_particles([0.0], [0.0], [3.0], [[1.0]], pid=[pid])
    sim.step(1)
    assert abs(sim.particles()["z"][0] - (-(3.0 + 10.0 * n2))) < 1e-9


def test_kz_floor():
    """Kz <- max(Kz, kz_min) (R4): with field Kz = 0 the vertical spread is set by kz_min."""
    N = 20_000
    w = custom(uniform_met(kz=0.0), kz_min=2.0, H=1.0e9, dt=5.0, n=N, n_steps=1, src=(0, 0, 1.0e6))
    sim = orc.OracleSim(w)
    sim.step(1)
    z = sim.particles()["z"] - 1.0e6
    assert abs(z.var() / (2 * 2.0 * 5.0) - 1.0) < 4.0 * math.sqrt(2.0 / N)


# ------------------------------------------------------------------ P10 / P11 deposition closed forms
def test_dry_deposition_closed_form():
    """uniform dry deposition (h_dep >= H): airborne = m0 (f_d f_l)^n, deposited = m0 p_d (1-(f_d f_l)^n)/(1-f_d f_l)."""
    H, dt, n, vd = 500.0, 10.0, 60, 2.0e-2
    g = Grid(8, 8, 4, -4000.0, -4000.0, 0.0, 1000.0, 1000.0, 125.0)
    w = custom(uniform_met(kz=1.0), grid=g, H=H, Kh=1.0, dt=dt, n=50, n_steps=n,
               nuclides=[Nuclide("I", T_I131, vd=vd)], activity=[50.0])
    sim = orc.OracleSim(w)
    sim.step(n)
    p_d = float(np.float32(-math.expm1(-vd * dt / H)))
    assert sim.p_dry(0) == p_d
    f = (1.0 - p_d) * math.exp(-math.log(2) * dt / T_I131)
    led = sim.ledger()[0]
    assert abs(led[1] / (50.0 * f ** n) - 1) < 1e-12
    dep_total = 50.0 * p_d * (1 - f ** n) / (1 - f)
    assert abs(led[2] / dep_total - 1) < 1e-12
    dep = sim.deposition()
    assert abs(dep.sum() * g.dx * g.dy / dep_total - 1) < 1e-12
    assert abs(led[0] - (led[1] + led[2] + led[3] + led[4] + led[5])) < 1e-12 * led[0]


def test_dry_deposition_layer_threshold():
    """h_dep < H: only particles with z' < h_dep deposit (PAPER.md L84-86 eligibility)."""
    H, dt, vd, hd = 1000.0, 10.0, 1.0e-2, 80.0
    w = custom(uniform_met(), H=H, dt=dt, n=0, n_steps=1, h_dep=hd, nuclides=[Nuclide("I", 0.0, vd=vd)])
    sim = orc.OracleSim(w)
    sim.set_particles([0.0, 0.0], [0.0, 0.0], [79.0, 81.0], [[1.0, 1.0]], pid=[0, 1])
    sim.step(1)
    m = sim.particles()["m"][0]
    p_d = float(np.float32(-math.expm1(-vd * dt / hd)))
    assert m[0] == 1.0 - p_d and m[1] == 1.0


def test_wet_deposition_box_and_time():
    """rain covering the domain for n_r steps adds a factor (1-p_w)^n_r (P11); outside the box or
    outside the time window nothing is scavenged; dry is applied before wet (R8)."""
    dt, lam, vd, H = 10.0, 1.0e-3, 1.0e-2, 500.0
    rain = RainBox(-100.0, 100.0, -100.0, 100.0, 20.0, 50.0)     # steps 2, 3, 4
    w = custom(uniform_met(), H=H, dt=dt, n=0, n_steps=8, rain=rain,
               nuclides=[Nuclide("I", 0.0, vd=vd, lambda_wet=lam)])
    sim = orc.OracleSim(w)
    sim.set_particles([0.0, 500.0], [0.0, 0.0], [10.0, 10.0], [[1.0, 1.0]], pid=[0, 1])
    sim.step(8)
    m = sim.particles()["m"][0]
    p_w = float(np.float32(-math.expm1(-lam * dt)))
    p_d = float(np.float32(-math.expm1(-vd * dt / H)))
    assert abs(m[0] / ((1 - p_d) ** 8 * (1 - p_w) ** 3) - 1) < 1e-13
    assert abs(m[1] / ((1 - p_d) ** 8) - 1) < 1e-13
    led = sim.ledger()[0]
    # wet removes from what is left after dry in the same step
    wet_expected = sum(((1 - p_d) * (1 - p_w)) ** j * (1 - p_d) ** 2 * (1 - p_d) * p_w for j in range(3))
    assert abs(led[3] / wet_expected - 1) < 1e-12
    assert abs(2.0 - (led[1] + led[2] + led[3] + led[4] + led[5])) < 1e-13


# ------------------------------------------------------------------ P6 ledger on a full config
def test_ledger_conservation_c3_small():
    w = make("c3", scale=2e-4, n_steps=2400)      # 2000 particles, through the start of the rain
    sim = orc.OracleSim(w)
    sim.step(2400)
    led = sim.ledger()
    for k in range(2):
        tot = led[k][1] + led[k][2] + led[k][3] + led[k][4] + led[k][5]
        assert abs(tot / led[k][0] - 1) < 1e-12
    assert led[0][3] > 0 and led[1][2] > led[0][2] * 0.1    # wet happened; Cs (vd 2e-3, 1e14) vs I
    dep = sim.deposition()
    g = w.cgrid
    for k in range(2):
        on_grid = dep[k].sum() * g.dx * g.dy
        assert abs((on_grid + led[k][6]) / (led[k][2] + led[k][3]) - 1) < 1e-12


# ------------------------------------------------------------------ P9 binning
def test_binning_brute_force_and_faces():
    g = Grid(5, 4, 3, -10.0, 0.0, 0.0, 4.0, 5.0, 10.0)
    w = custom(uniform_met(), grid=g, n=0)
    sim = orc.OracleSim(w)
    rng = np.random.default_rng(2)
    N = 1000
    x = rng.uniform(-14, 14, N).astype(np.float32).astype(np.float64)
    y = rng.uniform(-3, 23, N).astype(np.float32).astype(np.float64)
    z = rng.uniform(-2, 33, N).astype(np.float32).astype(np.float64)
    # exact face / edge cases: on a face -> upper cell; x = x0 + nx dx is outside; x = x0 is inside
    x[:4] = [-10.0, 10.0, -6.0, 9.999999]
    y[:4] = [2.5, 2.5, 5.0, 19.999998]
    z[:4] = [0.0, 5.0, 10.0, 29.999998]
    m = rng.uniform(0.5, 1.5, N)
    st = (rng.uniform(size=N) < 0.1).astype(np.uint8)
    st[:4] = 0
    sim.set_particles(x, y, z, [m], pid=np.arange(N), status=st)
    sim.bin_now()
    cnt = np.zeros(g.shape, dtype=np.int64)
    s = np.zeros(g.shape)
    for i in range(N):
        if st[i]:
            continue
        # R10: the cell is DEFINED by the fp32 expression floorf((x - x0) * (float)(1/dx))
        f32 = np.float32
        ci = math.floor((f32(x[i]) - f32(-10.0)) * f32(1.0 / 4.0))
        cj = math.floor((f32(y[i]) - f32(0.0)) * f32(1.0 / 5.0))
        ck = math.floor((f32(z[i]) - f32(0.0)) * f32(1.0 / 10.0))
        if 0 <= ci < 5 and 0 <= cj < 4 and 0 <= ck < 3:
            cnt[ck, cj, ci] += 1
            s[ck, cj, ci] += m[i]
    np.testing.assert_array_equal(sim.counts(), cnt)
    np.testing.assert_allclose(sim.concentration()[0], s / (4.0 * 5.0 * 10.0), rtol=1e-13)
    assert cnt[0, 0, 0] >= 1 and sim.counts()[1, 1, 1] >= 1      # (-10,2.5,0) and (-6,5,10)
    assert orc.cell_index(10.0, -10.0, 4.0, 5) == -1 and orc.cell_index(-10.0, -10.0, 4.0, 5) == 0
    assert orc.cell_index(-6.0, -10.0, 4.0, 5) == 1 and orc.cell_index(-10.000001, -10.0, 4.0, 5) == -1
    # permutation invariance of the counts
    perm = rng.permutation(N)
    sim.set_particles(x[perm], y[perm], z[perm], [m[perm]], pid=np.arange(N), status=st[perm])
    sim.bin_now()
    np.testing.assert_array_equal(sim.counts(), cnt)


# ------------------------------------------------------------------ P13 schedule
def test_release_schedule_count_mode():
    """b_j = s_start + floor(j S / N): monotone, sums to N, births per step differ by at most 1."""
    N, S = 1000, 7
    w = custom(uniform_met(), n=N, dt=10.0, t_rel=(20.0, 20.0 + S * 10.0), n_steps=12)
    sim = orc.OracleSim(w)
    counts = []
    for s in range(12):
        sim.step(1)
        counts.append(sim.injected(s))
    assert counts[:2] == [0, 0] and sum(counts) == N and counts[9:] == [0, 0, 0]
    want = [sum(1 for j in range(N) if 2 + (j * S) // N == s) for s in range(12)]
    assert counts == want
    assert list(sim.particles()["pid"]) == list(range(N))
    led = sim.ledger()[0]
    assert abs(led[0] - 1.0) < 1e-12          # activity scaled to the particle count


def test_release_strided_subsample_is_exact_subset():
    """pid_stride / pid_offset pick a subset whose trajectories equal those of the full run."""
    kw = dict(Kh=10.0, H=500.0, dt=10.0, n=300, t_rel=(0.0, 100.0), n_steps=15, seed=9)
    full = orc.OracleSim(custom(uniform_met(u=1.0, kz=3.0), **kw))
    sub = orc.OracleSim(custom(uniform_met(u=1.0, kz=3.0), pid_offset=3, pid_stride=10, **kw))
    full.step(15)
    sub.step(15)
    pf, ps = full.particles(), sub.particles()
    assert list(ps["pid"]) == list(range(3, 300, 10))
    idx = ps["pid"].astype(int)
    for key in ("x", "y", "z"):
        np.testing.assert_array_equal(ps[key], pf[key][idx])
    np.testing.assert_array_equal(ps["m"][0], pf["m"][0][idx])


def test_rate_mode_capacity_and_compaction():
    """rate mode: c slots per step, pid = step*c + j; short capacity skips the highest j (R9);
    ABSORB + compaction keeps pids strictly increasing and equals a brute-force filter (P12)."""
    g = Grid(10, 10, 4, -500.0, -500.0, 0.0, 100.0, 100.0, 100.0)
    kw = dict(grid=g, Kh=400.0, H=400.0, dt=10.0, rate=2.0, t_rel=(0.0, 400.0), n_steps=40, seed=4,
              boundary="absorb", src=(300.0, 0.0, 50.0))
    a = orc.OracleSim(custom(uniform_met(u=8.0, kz=2.0), compact=True, capacity=150, **kw))
    b = orc.OracleSim(custom(uniform_met(u=8.0, kz=2.0), compact=False, capacity=10_000, **kw))
    throttled = False
    for s in range(40):
        a.step(1)
        b.step(1)
        throttled |= a.injected(s) < 20
        pa, pb = a.particles(), b.particles()
        assert np.all(np.diff(pa["pid"].astype(np.int64)) > 0)
        assert np.all(pa["status"] == 0) and a.n <= 150
        if not throttled:
            alive = pb["status"] == 0
            np.testing.assert_array_equal(pa["pid"], pb["pid"][alive])
            np.testing.assert_array_equal(pa["x"], pb["x"][alive])
    assert (b.particles()["status"] == 1).sum() > 50       # exits really happened
    led = a.ledger()[0]
    assert abs((led[1] + led[2] + led[3] + led[4] + led[5]) / led[0] - 1) < 1e-12 and led[5] > 0
    # throttle: tiny capacity
    c = orc.OracleSim(custom(uniform_met(), compact=True, capacity=35, grid=g, rate=2.0, dt=10.0,
                             t_rel=(0.0, 400.0), n_steps=3, boundary="absorb"))
    c.step(3)
    assert [c.injected(s) for s in range(3)] == [20, 15, 0]
    assert list(c.particles()["pid"]) == list(range(20)) + list(range(20, 35))


def test_absorb_boundary_is_met_box():
    g = Grid(10, 10, 4, -500.0, -500.0, 0.0, 100.0, 100.0, 100.0)
    w = custom(uniform_met(u=10.0), grid=g, dt=10.0, n=0, boundary="absorb")
    sim = orc.OracleSim(w)
    sim.set_particles([250.0, 399.0, 400.0], [0.0, 0.0, 0.0], [50.0] * 3, [[1.0, 2.0, 4.0]], pid=[0, 1, 2])
    sim.step(1)
    st = sim.particles()["status"]
    assert list(st) == [0, 0, 1]          # 350, 499 inside; 500 = x0 + nx dx is outside
    assert sim.ledger()[0][5] == 4.0
    sim.step(1)
    assert list(sim.particles()["status"]) == [0, 1, 1] and sim.particles()["x"][2] == 500.0   # exited: never moved again


# ------------------------------------------------------------------ P14 independent numpy trace
def _philox_np(ctr, key):
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c, k = [int(v) for v in ctr], [int(v) for v in key]
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF, ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
        k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
    return c


def test_brute_force_trace_c2_tiny():
    """independent scalar python loop (scipy map_coordinates for the sampling, python Philox) over a
    few particles and steps of config 2 (time-varying, z-dependent field, reflection, decay)."""
    from scipy import ndimage
    w = make("c2", scale=2e-5, n_steps=40)          # 20 particles
    sim = orc.OracleSim(w)
    sim.step(40)
    p = sim.particles()
    f = w.fields().astype(np.float64)
    g = w.mgrid
    N = w.release.n_particles
    S = 720
    sig_h = float(np.float32(math.sqrt(2 * w.Kh * w.dt)))
    for j in range(N):
        b = (j * S) // N
        if b >= 40:
            assert j >= sim.n
            continue
        x, y, z, m = 0.0, 0.0, 50.0, 6.0e9 / N
        for n in range(b, 40):
            t = n * w.dt
            s = min(max(int(math.floor(t / 3600.0)), 0), w.nt - 2)
            a = float(np.float32(min(max((t - s * 3600.0) / 3600.0, 0.0), 1.0)))
            r = _philox_np([n, 0, j, 0], [w.seed, 0])
            u1, u2, u3, u4 = ((r[0] >> 8) + 1) / 2 ** 24, (r[1] >> 8) / 2 ** 24, ((r[2] >> 8) + 1) / 2 ** 24, (r[3] >> 8) / 2 ** 24
            R1, R2 = math.sqrt(-2 * math.log(u1)), math.sqrt(-2 * math.log(u3))
            n0, n1, n2 = R1 * math.cos(2 * math.pi * u2), R1 * math.sin(2 * math.pi * u2), R2 * math.cos(2 * math.pi * u4)
            co = [[(z - g.z0) / g.dz - 0.5], [(y - g.y0) / g.dy - 0.5], [(x - g.x0) / g.dx - 0.5]]
            met = [(1 - a) * ndimage.map_coordinates(f[s, ..., c], co, order=1, mode="nearest")[0]
                   + a * ndimage.map_coordinates(f[s + 1, ..., c], co, order=1, mode="nearest")[0] for c in range(4)]
            kz = max(met[3], w.kz_min)
            x += met[0] * w.dt + sig_h * n0
            y += met[1] * w.dt + sig_h * n1
            z += met[2] * w.dt + math.sqrt(2 * kz * w.dt) * n2
            if z < 0:
                z = -z
            if z > w.H_mix:
                z = 2 * w.H_mix - z
            m *= math.exp(-math.log(2) * w.dt / T_I131)
        assert abs(p["x"][j] - x) < 1e-8 and abs(p["y"][j] - y) < 1e-8 and abs(p["z"][j] - z) < 1e-8
        assert abs(p["m"][0][j] / m - 1) < 1e-13


def test_oracle_deterministic_across_thread_counts():
    w = make("c3", scale=1e-4, n_steps=200)
    res = []
    for nt in (1, 4):
        orc.set_num_threads(nt)
        sim = orc.OracleSim(w)
        sim.step(200)
        res.append((sim.particles(), sim.deposition(), sim.ledger()))
    orc.set_num_threads(orc.num_threads())
    for key in ("x", "y", "z", "m"):
        np.testing.assert_array_equal(res[0][0][key], res[1][0][key])
    np.testing.assert_array_equal(res[0][1], res[1][1])
    np.testing.assert_array_equal(res[0][2], res[1][2])


# ------------------------------------------------------------------ P15: time-integrated concentration (S§8(f)3)
def test_dose_of_a_resting_decaying_cloud_is_a_geometric_series():
    """No wind, no diffusion: the particles rest, the cell concentration decays as 2^(-t/T), and the dose
    after n binnings is the rectangle-rule sum  C0 T_bin sum_{b=1..n} 2^(-b T_bin / T)  (closed form)."""
    T_half = 3600.0
    n, be, dt, nb = 50, 20, 10.0, 7
    w = custom(uniform_met(), n=n, nuclides=[Nuclide("X", T_half)], dt=dt, bin_every=be, src=(30.0, -20.0, 150.0),
               activity=[2.0e6], H=1000.0, n_steps=be * nb)
    o = orc.OracleSim(w)
    o.enable_dose()
    o.step(be * nb)
    g = w.cgrid
    V = g.dx * g.dy * g.dz
    Tb = be * dt
    r = 2.0 ** (-Tb / T_half)
    want = 2.0e6 / V * Tb * r * (1 - r ** nb) / (1 - r)
    d = o.dose()
    i, j, k = int((30.0 - g.x0) // g.dx), int((-20.0 - g.y0) // g.dy), int(150.0 // g.dz)
    assert abs(d[0, k, j, i] / want - 1) < 1e-12
    assert d.sum() == pytest.approx(d[0, k, j, i], rel=1e-15)
    # dose = sum over binnings of the concentration field times the interval (definition, re-run step by step)
    o2 = orc.OracleSim(w)
    acc = np.zeros_like(d)
    for _ in range(nb):
        o2.step(be)
        acc += o2.concentration() * Tb
    np.testing.assert_allclose(d, acc, rtol=1e-13, atol=0)


# ------------------------------------------------------------------ P16: Bernoulli deposition (S§8(f)1, R11)
def test_bernoulli_deposition_survival_law_and_ledger():
    """Uniform dry deposition as a per-step Bernoulli trial: survivors ~ Binomial(N, (1-p)^n); a deposited
    particle drops its whole (decayed) activity once; emitted = airborne + dry + decayed exactly."""
    N, n, dt, H = 20000, 12, 10.0, 100.0
    w = custom(uniform_met(u=1.0, kz=1.0), n=N, nuclides=[Nuclide("X", 5000.0, vd=1.0)], dt=dt, Kh=10.0, H=H, h_dep=H,
               activity=[float(N)], n_steps=n, src=(0.0, 0.0, 50.0))
    o = orc.OracleSim(w, dep_mode=1)
    o.step(n)
    p = float(o.p_dry(0))
    assert abs(p - (1 - math.exp(-1.0 * dt / H))) < 1e-7
    st = o.particles()["status"]
    surv = int((st == 0).sum())
    q = (1 - p) ** n
    assert abs(surv - N * q) < 4 * math.sqrt(N * q * (1 - q))
    assert set(np.unique(st)) <= {0, 2}
    led = o.ledger()[0]
    assert abs((led[1] + led[2] + led[4]) / led[0] - 1) < 1e-12 and led[3] == 0 and led[5] == 0
    # every deposit is one whole particle: dry ledger = sum over deposited particles of 2^(-t_dep/T)
    assert led[2] < (N - surv) * 1.0 and led[2] > (N - surv) * 2.0 ** (-n * dt / 5000.0)
    dep = o.deposition()
    g = w.cgrid
    assert abs(dep.sum() * g.dx * g.dy + led[6] - led[2]) < 1e-9 * led[2]


def test_bernoulli_deposition_replays_from_the_draws():
    """Independent replay: the step at which nuclide k of particle j deposits follows from Philox stream 1
    alone when every particle is eligible (uniform dry, rain everywhere): first step with u_dry < p_dry, else
    u_wet < p_wet."""
    n, steps = 60, 30
    nuc = [Nuclide("A", 0.0, vd=0.5, lambda_wet=2.0e-3), Nuclide("B", 0.0, vd=0.2, lambda_wet=8.0e-3)]
    w = custom(uniform_met(), n=n, nuclides=nuc, dt=10.0, H=100.0, h_dep=100.0, activity=[float(n), 2.0 * n], n_steps=steps,
               rain=RainBox(-1e9, 1e9, -1e9, 1e9, 0.0, 1e9), seed=77)
    o = orc.OracleSim(w, dep_mode=1)
    o.step(steps)
    m = o.particles()["m"]
    pd = [float(o.p_dry(k)) for k in range(2)]
    pw = [float(o.p_wet(k)) for k in range(2)]
    dry = np.zeros(2)
    wet = np.zeros(2)
    for j in range(n):
        for k in range(2):
            gone = None
            for s in range(steps):
                r = orc.philox_draw(77, j, s, 1)
                ud, uw = (int(r[k]) >> 8) / 2.0 ** 24, (int(r[2 + k]) >> 8) / 2.0 ** 24
                if ud < pd[k]:
                    gone = "d"
                    break
                if uw < pw[k]:
                    gone = "w"
                    break
            a = 1.0 if k == 0 else 2.0
            if gone is None:
                assert m[k][j] == a
            else:
                assert m[k][j] == 0.0
                (dry if gone == "d" else wet)[k] += a
    led = o.ledger()
    for k in range(2):
        assert led[k][2] == pytest.approx(dry[k], rel=1e-14) and led[k][3] == pytest.approx(wet[k], rel=1e-14)
    assert dry.sum() > 0 and wet.sum() > 0


# ------------------------------------------------------------------ P17: Eq.(3) per particle (S§8(f)2, R12)
def test_eq3_profile_values():
    """Kz = k u* z / Phi(z/L) (1 - z/Hz)^2 with Businger-Dyer Phi: hand-computed values and the neutral closed form."""
    for z in (0.5, 25.0, 333.3, 975.0):
        assert orc.kz_eq3(0.4, 0.0, 1000.0, z) == pytest.approx(0.16 * z * (1 - z / 1000.0) ** 2, rel=1e-15)
    assert orc.kz_eq3(0.5, 0.002, 1000.0, 100.0) == pytest.approx(8.1, rel=1e-14)                       # zeta = 0.2: Phi = 2
    assert orc.kz_eq3(0.5, -0.01, 1000.0, 100.0) == pytest.approx(16.2 * math.sqrt(17.0), rel=1e-14)    # zeta = -1: Phi = 17^-1/2
    assert orc.kz_eq3(0.5, 0.0, 1000.0, 1000.0) == 0.0 and orc.kz_eq3(0.5, 0.0, 1000.0, 1200.0) == 0.0
    assert orc.kz_eq3(0.5, 0.0, 1000.0, 0.0) == 0.0


def test_surface_sampling_reproduces_affine_fields():
    g = Grid(12, 9, 4, -600.0, 100.0, 0.0, 100.0, 50.0, 25.0)
    xc = g.x0 + (np.arange(g.nx) + 0.5) * g.dx
    yc = g.y0 + (np.arange(g.ny) + 0.5) * g.dy
    Y, X = np.meshgrid(yc, xc, indexing="ij")
    sf = np.zeros((2, g.ny, g.nx, 4), dtype=np.float32)
    for s, t in enumerate((0.0, 3600.0)):
        sf[s, ..., 0] = 0.25 + X / 4096.0 + t / 8192.0
        sf[s, ..., 1] = Y / 65536.0 - 1.0 / 1024.0          # exactly representable in fp32
        sf[s, ..., 2] = 1000.0 + 0.5 * X - 0.25 * Y
    rng = np.random.default_rng(4)
    for _ in range(200):
        x, y, t = rng.uniform(xc[0], xc[-1]), rng.uniform(yc[0], yc[-1]), rng.uniform(0, 3600.0)
        got = orc.sample_surface(g, 2, 0.0, 3600.0, sf, t, x, y)
        a = float(np.float32(t / 3600.0))                  # the time weight is an fp32 parameter (R4)
        assert got[0] == pytest.approx(0.25 + x / 4096.0 + a * 3600.0 / 8192.0, rel=1e-12)
        assert got[1] == pytest.approx(y / 65536.0 - 1.0 / 1024.0, rel=1e-9, abs=1e-15)
        assert got[2] == pytest.approx(1000.0 + 0.5 * x - 0.25 * y, rel=1e-12)
    lo = orc.sample_surface(g, 2, 0.0, 3600.0, sf, 0.0, -1e9, -1e9)       # edge-clamped
    assert lo[2] == pytest.approx(float(sf[0, 0, 0, 2]))


def test_eq3_mode_equals_gridded_mode_at_cell_centre_heights():
    """With uniform neutral surface fields Eq.(3) IS c2's Kz recipe, and the gridded field interpolates it exactly at
    the cell-centre heights: one step from there gives the same positions in both modes."""
    w0 = make("c2", scale=1e-3).replace(nt=2)
    w1 = dataclasses_replace(w0, kz_mode=1, surface_fn=lambda t, Y, X: (0.4, 0.0, 1000.0))
    g = w0.mgrid
    rng = np.random.default_rng(9)
    n = 500
    x = rng.uniform(-2e4, 2e4, n)
    y = rng.uniform(-2e4, 2e4, n)
    z = g.z0 + (rng.integers(1, g.nz - 1, n) + 0.5) * g.dz
    res = []
    for w in (w0, w1):
        o = orc.OracleSim(w.replace(release=None, capacity=n), bin_every=0)
        o.set_particles(x, y, z, np.ones((1, n)), pid=np.arange(n))
        o.set_step_index(100)
        o.step(1)
        res.append(o.particles())
    for k in ("x", "y", "z"):
        np.testing.assert_allclose(res[0][k], res[1][k], rtol=0, atol=2e-5)   # fp32 field values vs fp64 formula
    assert np.abs(res[0]["z"] - z).max() > 1.0


# ------------------------------------------------------------------ P18: non-uniform vertical levels
def test_nonuniform_levels_reproduce_piecewise_linear_profiles():
    """Values given on non-uniform levels: the sample is the linear interpolant between the bracketing levels
    (numpy.interp is the textbook definition), clamped outside; uniform levels given explicitly change nothing."""
    g = Grid(6, 5, 7, 0.0, 0.0, 0.0, 100.0, 100.0, 40.0)
    zl = np.array([5.0, 20.0, 50.0, 110.0, 230.0, 470.0, 950.0])
    prof = np.array([1.0, 2.5, 3.0, 4.75, 4.0, 6.5, 7.0])
    f = np.zeros((1, g.nz, g.ny, g.nx, 4), dtype=np.float32)
    f[0, :, :, :, 0] = prof[:, None, None]
    f[0, :, :, :, 3] = (2.0 * prof)[:, None, None]
    rng = np.random.default_rng(2)
    for z in list(rng.uniform(-20.0, 1100.0, 300)) + list(zl) + [0.0, 5.0, 950.0, 2000.0]:
        got = orc.sample_met(g, 1, 0.0, 3600.0, f, 0.0, 250.0, 250.0, float(z), z_levels=zl)
        want = np.interp(z, zl, prof)
        assert got[0] == pytest.approx(want, rel=1e-12) and got[3] == pytest.approx(2 * want, rel=1e-12)
    zu = g.z0 + (np.arange(g.nz) + 0.5) * g.dz
    for z in rng.uniform(-20.0, 320.0, 100):
        a = orc.sample_met(g, 1, 0.0, 3600.0, f, 0.0, 130.0, 310.0, float(z), z_levels=zu)
        b = orc.sample_met(g, 1, 0.0, 3600.0, f, 0.0, 130.0, 310.0, float(z))
        np.testing.assert_allclose(a, b, rtol=1e-13, atol=1e-15)


# ------------------------------------------------------------------ P19: drift-corrected walk (S§8(f)4, labelled departure)
def test_dkz_dz_is_the_slope_of_the_interpolant():
    g = Grid(5, 4, 6, 0.0, 0.0, 0.0, 100.0, 100.0, 50.0)
    zl = np.array([10.0, 40.0, 90.0, 170.0, 300.0, 520.0])
    for levels, zc in ((None, g.z0 + (np.arange(g.nz) + 0.5) * g.dz), (zl, zl)):
        prof = np.array([1.0, 4.0, 5.5, 5.0, 9.0, 2.0])
        f = np.zeros((2, g.nz, g.ny, g.nx, 4), dtype=np.float32)
        f[0, ..., 3] = prof[:, None, None]
        f[1, ..., 3] = 3.0 * prof[:, None, None]
        t, a = 900.0, 0.25
        for k in range(g.nz - 1):
            z = 0.3 * zc[k] + 0.7 * zc[k + 1]
            want = (1 + 2 * a) * (prof[k + 1] - prof[k]) / (zc[k + 1] - zc[k])
            got = orc.dkz_dz(g, 2, 0.0, 3600.0, f, t, 210.0, 170.0, float(z), z_levels=levels)
            assert got == pytest.approx(want, rel=1e-12)
            eps = 1e-3                                                    # and it IS the derivative of the sampled value
            hi = orc.sample_met(g, 2, 0.0, 3600.0, f, t, 210.0, 170.0, float(z + eps), z_levels=levels)[3]
            lo = orc.sample_met(g, 2, 0.0, 3600.0, f, t, 210.0, 170.0, float(z - eps), z_levels=levels)[3]
            assert got == pytest.approx((hi - lo) / (2 * eps), rel=1e-7)
        for z in (zc[0] - 1.0, zc[0], zc[-1], zc[-1] + 5.0):              # clamped: constant in z
            assert orc.dkz_dz(g, 2, 0.0, 3600.0, f, t, 210.0, 170.0, float(z), z_levels=levels) == 0.0


def test_drift_correction_keeps_a_uniform_cloud_well_mixed():
    """Kz growing linearly with height, reflection at 0 and H: the paper's walk (no drift term) piles particles up where
    Kz is small; with the + dKz/dz dt term a uniform cloud stays uniform (the well-mixed condition)."""
    H, nz, n = 500.0, 25, 40000
    g = Grid(4, 4, nz, -200.0, -200.0, 0.0, 100.0, 100.0, H / nz)
    met = lambda t, Z, Y, X: (0.0, 0.0, 0.0, 2.0 + 0.04 * Z)
    rng = np.random.default_rng(21)
    z0 = rng.uniform(0.0, H, n)
    hist = {}
    for drift in (False, True):
        w = custom(met, grid=g, n=n, dt=10.0, H=H, kz_min=0.0, n_steps=400)
        o = orc.OracleSim(w.replace(release=None), bin_every=0, drift=drift)
        o.set_particles(np.zeros(n), np.zeros(n), z0.copy(), np.ones((1, n)), pid=np.arange(n))
        o.step(400)
        hist[drift] = np.histogram(o.particles()["z"], bins=10, range=(0.0, H))[0]
    expect = n / 10
    chi2 = ((hist[True] - expect) ** 2 / expect).sum()
    assert chi2 < 40.0, (chi2, hist[True])                               # 9 degrees of freedom (+ O(dt) scheme error)
    assert hist[False][0] > 1.5 * expect and hist[False][-1] < 0.7 * expect, hist[False]


# ------------------------------------------------------------------ P20: ground decay of the deposition map (S§8(f)3, R13)
def test_ground_decay_total_activity_follows_the_decay_law():
    """A puff that moves, diffuses and deposits (dry everywhere + a rain box), everything on the map: with the ground
    activity decaying too, airborne + ground = emitted * 2^(-t/T) at every step, whatever the particles did; for a
    resting cloud the one cell holds m0 f^N (1 - (1-p)^N) (closed forms)."""
    T_half, dt, N = 2400.0, 10.0, 60
    nuc = [Nuclide("X", T_half, vd=0.5, lambda_wet=2.0e-3)]
    g = Grid(40, 40, 4, -2000.0, -2000.0, 0.0, 100.0, 100.0, 50.0)
    w = custom(uniform_met(u=1.5, v=-0.5, kz=2.0), grid=g, n=400, nuclides=nuc, dt=dt, Kh=20.0, H=200.0, activity=[7.0e5], n_steps=N,
               rain=RainBox(-500.0, 600.0, -400.0, 500.0, 100.0, 400.0))
    o = orc.OracleSim(w)
    o.enable_ground_decay()
    A = g.dx * g.dy
    for n in range(1, N + 1):
        o.step(1)
        if n % 12 == 0:
            air = o.particles()["m"].sum()
            tot = air + o.deposition_ground().sum() * A
            assert tot == pytest.approx(7.0e5 * 2.0 ** (-n * dt / T_half), rel=1e-12)
    led = np.array(o.ledger())
    assert led[0][6] == 0.0 and led[0][3] > 0.0                               # nothing fell off the map; it did rain
    assert o.deposition_ground().sum() < o.deposition().sum()
    # resting cloud
    w = custom(uniform_met(), grid=g, n=50, nuclides=[Nuclide("X", T_half, vd=0.5)], dt=dt, H=200.0, activity=[3.0e4], n_steps=N,
               src=(130.0, -270.0, 20.0))
    o = orc.OracleSim(w)
    o.enable_ground_decay()
    o.step(N)
    p, f = float(o.p_dry(0)), 2.0 ** (-dt / T_half)
    d = o.deposition_ground()
    i, j = int((130.0 - g.x0) // g.dx), int((-270.0 - g.y0) // g.dy)
    assert d[0, j, i] * A == pytest.approx(3.0e4 * f ** N * (1 - (1 - p) ** N), rel=1e-12)
    assert d.sum() == pytest.approx(d[0, j, i], rel=1e-15)


def test_ground_decay_is_the_sum_of_increments_each_decayed_from_its_own_step():
    """Definition, re-run step by step on a continuous release with layer deposition and rain, two nuclides: the increments
    of step n (differences of the undecayed map) decay from t_n: ground(t_N) = sum_n inc_n exp(-lambda (t_N - t_n))."""
    dt, N = 10.0, 90
    nuc = [Nuclide("A", 1800.0, vd=0.02, lambda_wet=1.0e-3), Nuclide("B", 5.0e4, vd=0.05, lambda_wet=3.0e-4)]
    g = Grid(30, 30, 6, -1500.0, -1500.0, 0.0, 100.0, 100.0, 50.0)
    w = custom(uniform_met(u=2.0, v=1.0, kz=3.0), grid=g, n=600, nuclides=nuc, dt=dt, Kh=30.0, H=300.0, h_dep=80.0, activity=[1.0e6, 4.0e5],
               t_rel=(0.0, 600.0), n_steps=N, rain=RainBox(-200.0, 900.0, -300.0, 800.0, 200.0, 700.0))
    o = orc.OracleSim(w)
    o.enable_ground_decay()
    prev = o.deposition()
    want = np.zeros_like(prev)
    lam = np.array([math.log(2.0) / n_.half_life_s for n_ in nuc])[:, None, None]
    for n in range(N):
        o.step(1)
        cur = o.deposition()
        want += (cur - prev) * np.exp(-lam * (N - n) * dt)
        prev = cur
    got = o.deposition_ground()
    assert got.sum() > 0
    np.testing.assert_allclose(got, want, rtol=1e-9, atol=1e-12 * got.max())
