"""Pins of the oracle's EXCLUSION machinery: the `fragile` flag (DESIGN.md §5 T3: a particle that
came within frag_delta of an active discontinuity) and the deposit map's face slack (`face_delta`).  They decide which
particles and how much map mass the GPU parity tests may ignore, so they are pinned here, on the CPU, with hand-placed
RESTING particles (no wind, no diffusion: the new position is the old one, exactly) at +- delta of every discontinuity:
the flagged set must be exactly the expected one - nothing more, nothing less."""
import numpy as np
import pytest

from helpers import custom, uniform_met
from oracle import oracle as orc
from workloads import Grid, Nuclide, RainBox

D = 0.05          # frag_delta of the parity tests (metres)
G = Grid(20, 10, 4, -1000.0, -500.0, 0.0, 100.0, 100.0, 50.0)      # box x in [-1000, 1000), y in [-500, 500), z < 200


def _rest(**kw):
    """A workload in which nothing moves: zero wind, Kh = 0, Kz = 0."""
    base = dict(grid=G, n=0, Kh=0.0, H=200.0, kz_min=0.0, dt=10.0, n_steps=4)
    base.update(kw)
    return custom(uniform_met(), **base)


def _run(w, pts, steps=1, step0=0, **okw):
    pts = np.asarray(pts, dtype=np.float64)
    n = len(pts)
    o = orc.OracleSim(w.replace(capacity=n, release=None), frag_delta=D, bin_every=0, **okw)
    o.set_particles(pts[:, 0], pts[:, 1], pts[:, 2], np.ones((w.K, n)), pid=np.arange(n))
    o.set_step_index(step0)
    o.step(steps)
    p = o.particles()
    assert np.array_equal(p["x"], pts[:, 0]) and np.array_equal(p["y"], pts[:, 1])     # at rest
    return o, p, set(int(i) for i in o.fragile_pids())


def test_fragile_at_the_absorbing_boundary_only_within_delta():
    w = _rest(boundary="absorb")
    pts = [
        (-1000.0 + 0.04, 0.0, 50.0),    # 0 inside, 4 cm from the west face        -> fragile, active
        (-1000.0 + 0.06, 0.0, 50.0),    # 1 inside, 6 cm                            -> not fragile
        (1000.0 - 0.04, 0.0, 50.0),     # 2 inside, 4 cm from the east face         -> fragile
        (1000.0 - 0.06, 0.0, 50.0),     # 3                                          -> not
        (0.0, -500.0 + 0.04, 50.0),     # 4 south face                               -> fragile
        (0.0, 500.0 - 0.06, 50.0),      # 5 north face, 6 cm                         -> not
        (-1000.0 - 0.04, 0.0, 50.0),    # 6 outside by 4 cm                          -> fragile, exited
        (-1000.0 - 1.0, 0.0, 50.0),     # 7 outside by 1 m                           -> exited, not fragile
        (1000.0, 0.0, 50.0),            # 8 exactly on the (exclusive) east face     -> exited, fragile
        (-1000.0, 0.0, 50.0),           # 9 exactly on the (inclusive) west face     -> active, fragile
        (0.0, 0.0, 50.0),               # 10 centre                                  -> not
    ]
    o, p, frag = _run(w, pts)
    assert frag == {0, 2, 4, 6, 8, 9}
    assert list(p["status"]) == [0, 0, 0, 0, 0, 0, 1, 1, 1, 0, 0]
    # OPEN boundary: the same positions flag nothing and nobody leaves
    o, p, frag = _run(_rest(boundary="open"), pts)
    assert frag == set() and not p["status"].any()


def test_fragile_at_h_dep_only_when_the_layer_is_a_discontinuity():
    nuc = [Nuclide("X", 0.0, vd=0.01)]
    pts = [(0.0, 0.0, 80.0 - 0.04), (0.0, 0.0, 80.0 + 0.04), (0.0, 0.0, 80.0 - 0.06), (0.0, 0.0, 80.0 + 0.06), (0.0, 0.0, 10.0)]
    o, p, frag = _run(_rest(nuclides=nuc, h_dep=80.0), pts)
    assert frag == {0, 1}
    led = o.ledger()
    # dry deposition acts strictly below h_dep: particles 0, 2, 4 lose p_dry of their unit activity
    assert led[0][2] == pytest.approx(3 * o.p_dry(0), rel=1e-12)
    # h_dep >= H: deposition everywhere, z = h_dep is no discontinuity, nothing is fragile
    o, p, frag = _run(_rest(nuclides=nuc, h_dep=200.0), pts)
    assert frag == set()


def test_fragile_at_the_rain_box_only_while_it_rains():
    nuc = [Nuclide("X", 0.0, lambda_wet=1e-3)]
    rain = RainBox(-300.0, 400.0, -200.0, 100.0, 100.0, 200.0)       # raining for 100 <= t < 200 (steps 10..19)
    pts = [
        (-300.0 + 0.04, 0.0, 50.0),     # 0 inside, 4 cm from the west face          -> fragile while raining
        (-300.0 - 0.04, 0.0, 50.0),     # 1 outside, 4 cm                            -> fragile while raining
        (-300.0 + 0.06, 0.0, 50.0),     # 2                                          -> not
        (400.0 - 0.04, -100.0, 50.0),   # 3 east face                                -> fragile
        (0.0, 100.0 + 0.04, 50.0),      # 4 north face, outside                      -> fragile
        (0.0, -200.0 + 0.06, 50.0),     # 5 south face, 6 cm                         -> not
        (-300.0 + 0.04, 300.0, 50.0),   # 6 on the line of the west face but 200 m north of the box -> not
        (-300.0 - 0.04, -200.0 - 0.04, 50.0),  # 7 outside the south-west corner, 4 cm both ways -> fragile
        (0.0, -50.0, 50.0),             # 8 deep inside                              -> not
    ]
    o, p, frag = _run(_rest(nuclides=nuc, rain=rain), pts, steps=1, step0=12)
    assert frag == {0, 1, 3, 4, 7}
    led = o.ledger()
    inside = [0, 2, 3, 5, 8]                                            # x in [-300, 400), y in [-200, 100)
    assert led[0][3] == pytest.approx(len(inside) * o.p_wet(0), rel=1e-12)
    for step0 in (9, 20):                                               # the step before the rain and the first after it
        o, p, frag = _run(_rest(nuclides=nuc, rain=rain), pts, steps=1, step0=step0)
        assert frag == set() and o.ledger()[0][3] == 0.0


def test_fragile_in_the_drift_corrected_walk_at_the_hull_of_the_levels():
    """The z-slope of the interpolant switches on / off at the first and last level height (25 m and 175 m here)."""
    met = lambda t, Z, Y, X: (0.0, 0.0, 0.0, 0.0 * Z)       # Kz = 0 everywhere: slope 0, nothing moves
    w = custom(met, grid=G, n=0, Kh=0.0, H=200.0, kz_min=0.0, dt=10.0, n_steps=2)
    pts = [(0.0, 0.0, 25.0 + 0.04), (0.0, 0.0, 25.0 + 0.06), (0.0, 0.0, 175.0 - 0.04), (0.0, 0.0, 175.0 - 0.06), (0.0, 0.0, 100.0)]
    o, p, frag = _run(w, pts, drift=True)
    assert frag == {0, 2}
    o, p, frag = _run(w, pts, drift=False)
    assert frag == set()


def test_fragile_is_sticky_and_listed_once():
    """A particle flagged at one step stays on the list (T3 excludes it for the rest of the run) and appears once."""
    w = _rest(boundary="absorb")
    o, p, frag = _run(w, [(-1000.0 + 0.04, 0.0, 50.0), (0.0, 0.0, 50.0)], steps=4)
    assert list(o.fragile_pids()) == [0]


def test_face_slack_of_the_deposit_map_covers_exactly_the_neighbours_across_near_faces():
    """face_delta = 1 m: a deposit within 1 m of a map-cell face may land in the neighbour across that face, so its
    amount is added to the slack of its own cell and of that neighbour (both, and the diagonal one, near a corner);
    a deposit further than 1 m from every face adds no slack at all."""
    nuc = [Nuclide("X", 0.0, vd=0.01)]
    w = _rest(nuclides=nuc, h_dep=200.0)
    # map cells are 100 m: cell (i, j) spans x in [-1000 + 100 i, ...), y in [-500 + 100 j, ...)
    pts = [
        (-1000.0 + 350.0, -500.0 + 250.0, 50.0),         # 0 centre of cell (3, 2): no slack
        (-1000.0 + 700.0 + 0.5, -500.0 + 450.0, 50.0),   # 1 cell (7, 4), 0.5 m from its west face: slack (7,4) and (6,4)
        (-1000.0 + 1200.0 - 0.5, -500.0 + 650.0, 50.0),  # 2 cell (11, 6), 0.5 m from its east face: slack (11,6) and (12,6)
        (-1000.0 + 1500.0 + 0.5, -500.0 + 800.0 + 0.5, 50.0),  # 3 cell (15, 8), corner: (15,8) (14,8) (15,7) (14,7)
        (-1000.0 + 1800.0 + 1.5, -500.0 + 150.0, 50.0),  # 4 cell (18, 1), 1.5 m from the face: no slack
    ]
    o, p, frag = _run(w, pts, face_delta=1.0)
    dep, slack = o.deposition(with_slack=True)
    area = 100.0 * 100.0
    d = o.p_dry(0) / area                                # every particle deposits p_dry of its unit activity
    want_dep = np.zeros((10, 20))
    for (i, j) in ((3, 2), (7, 4), (11, 6), (15, 8), (18, 1)):
        want_dep[j, i] = d
    np.testing.assert_allclose(dep[0], want_dep, rtol=1e-12, atol=0)
    want = np.zeros((10, 20))
    for (i, j) in ((7, 4), (6, 4), (11, 6), (12, 6), (15, 8), (14, 8), (15, 7), (14, 7)):
        want[j, i] = d
    np.testing.assert_allclose(slack[0], want, rtol=1e-12, atol=0)
    # face_delta = 0 (the default): no slack anywhere
    o, p, frag = _run(w, pts)
    assert not o.deposition(with_slack=True)[1].any()


def test_face_slack_at_the_edge_of_the_map():
    """A deposit just outside the map goes to the off-grid ledger; within face_delta of the map's edge it could have been
    inside, so the edge cell gets its amount as slack."""
    nuc = [Nuclide("X", 0.0, vd=0.01)]
    big = Grid(40, 20, 4, -2000.0, -1000.0, 0.0, 100.0, 100.0, 50.0)     # met box larger than the map
    w = custom(uniform_met(), grid=G, mgrid=big, n=0, Kh=0.0, H=200.0, kz_min=0.0, dt=10.0, n_steps=2, nuclides=nuc, h_dep=200.0)
    pts = [(-1000.0 - 0.5, -500.0 + 350.0, 50.0),       # 0 half a metre west of the map, row 3
           (-1000.0 - 5.0, -500.0 + 550.0, 50.0)]       # 1 five metres west: no slack
    o, p, frag = _run(w, pts, face_delta=1.0)
    dep, slack = o.deposition(with_slack=True)
    assert not dep.any()
    assert o.ledger()[0][6] == pytest.approx(2 * o.p_dry(0), rel=1e-12)
    area = 100.0 * 100.0
    assert slack[0][3, 0] == pytest.approx(o.p_dry(0) / area, rel=1e-12)
    assert slack[0][5, 0] == 0.0
    assert np.count_nonzero(slack) <= 3                 # the edge cell of row 3 and at most its two row neighbours
