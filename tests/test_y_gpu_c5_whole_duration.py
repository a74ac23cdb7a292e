"""BASELINE.json config 5 at 1/100 rate on its own domain over its WHOLE duration (12 h, dt = 2 s: 21600 steps), against the
oracle, with the within-tolerance fractions of T3 recorded at 1500 / 3000 / 6000 / 12000 / 21600 steps.

What is asserted is what holds without reference to a measured number: the decisions (status of every common non-fragile id,
the id sets up to the exits that fall one step apart, the throttled injection log), the ledger and counts bars of the 6000-step
test, and that the TYPICAL particle is inside T3's position tolerance at every checkpoint (median error on each axis below
1e-5 L).  The FRACTION of particles inside 1e-5 L falls below T3's 99.9 % on this config from about step 2500 on and is
printed, not asserted: DESIGN.md 5 carries the curve (measured on a B200: 100 % / 99.80 % / 98.65 % / 98.39 % / 97.36 %) and
says what it is - T3 is NOT met on c5 beyond 2500 steps; the tail grows with the run, the median does not leave the sub-mm range.

About two minutes (oracle: 1.1e10 particle-steps); runs the default compaction form of c5 (hole fill + physical record sort).
    python -m pytest tests/test_y_gpu_c5_whole_duration.py -m gpu -s
"""
import numpy as np
import pytest

from helpers import gpu_state
from workloads import make

pytestmark = pytest.mark.gpu

CHECKPOINTS = (1500, 3000, 6000, 12000, 21600)


def test_c5_own_domain_whole_duration():
    import torch
    assert torch.cuda.is_available()
    from paper_0912_3223_b200.build import build
    build()
    import paper_0912_3223_b200 as lpm
    from oracle import oracle as orc
    steps = CHECKPOINTS[-1]
    w = make("c5", scale=0.01, n_steps=steps)
    assert w.n_steps == 21600 and w.dt == 2.0 and w.nt == 13 and w.capacity == 500_000 and w.compact and w.boundary_mode == "absorb"
    o, sim = orc.OracleSim(w), lpm.Simulation(w)
    at, curve = 0, []
    for cp in CHECKPOINTS:
        o.step(cp - at)
        sim.step(cp - at)
        at = cp
        gp, p = gpu_state(sim), o.particles()
        frag = o.fragile_pids()
        assert sim.num_active == len(gp["pid"]) and len(np.unique(gp["pid"])) == len(gp["pid"])
        assert abs(len(gp["pid"]) - len(p["pid"])) <= 64 and (cp < 1250 or len(p["pid"]) > 450_000)     # both sides at the capacity plateau
        common, gi, pi = np.intersect1d(gp["pid"], p["pid"], return_indices=True)
        assert len(common) > 0.99 * len(p["pid"])
        ok = ~np.isin(common, frag)
        # (a particle may cross the boundary one step apart on the two sides - the 6000-step test's argument -, so at a
        # checkpoint a handful of ids can be active on one side and already out on the other)
        assert int((gp["status"][gi][ok] != p["status"][pi][ok]).sum()) <= 8
        rec = {"step": cp, "n": int(ok.sum())}
        tight = np.ones(ok.sum(), dtype=bool)
        wide = np.ones(ok.sum(), dtype=bool)
        for key, Li in (("x", 1.0e5), ("y", 1.0e5), ("z", 1250.0)):
            err = np.abs(gp[key][gi].astype(np.float64) - p[key][pi])[ok]
            tol = np.maximum(Li, np.abs(p[key][pi][ok]))
            assert np.median(err / tol) < 1e-5, (cp, key, np.median(err / tol))     # the typical particle is inside T3's band
            tight &= err <= 1e-5 * tol
            wide &= err <= 1e-4 * tol
            rec[key] = (float((err <= 1e-5 * tol).mean()), float(np.median(err)), float(np.quantile(err, 0.999)))
        act = (p["status"][pi] == 0)[ok]
        mrel = (np.abs(gp["m"][:, gi] - p["m"][:, pi]) / np.maximum(p["m"][:, pi], 1e-300))[:, ok][:, act]
        assert mrel.max() <= 1e-5, (cp, mrel.max())                                  # activities: every particle
        rec["within_1e-5_L"], rec["within_1e-4_L"] = float(tight.mean()), float(wide.mean())
        cg, co = sim.counts().cpu().numpy().astype(np.int64), o.counts().astype(np.int64)
        assert abs(int(cg.sum()) - int(co.sum())) <= 64
        rec["count_L1"] = float(np.abs(cg - co).sum() / co.sum())
        lg, lo = sim.ledger(), o.ledger()
        assert abs(lg[0][0] / lo[0][0] - 1) < 1e-4
        if lo[0][5] > 0:
            assert abs(lg[0][5] / lo[0][5] - 1) < 2e-3
        assert abs((lg[0][1] + lg[0][4] + lg[0][5]) / lg[0][0] - 1) < 1e-5
        curve.append(rec)
        print(f"[c5 whole duration] step {cp}: within 1e-5 L {rec['within_1e-5_L']:.4f}, within 1e-4 L {rec['within_1e-4_L']:.4f}; per axis "
              f"(fraction, median m, p99.9 m): x {rec['x']}, y {rec['y']}, z {rec['z']}; count L1 {rec['count_L1']:.2e}", flush=True)
    assert curve[0]["within_1e-5_L"] >= 0.999          # T3 as stated holds at 1500 steps
    assert [c["step"] for c in curve] == list(CHECKPOINTS)
