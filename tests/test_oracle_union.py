"""Pins for union-of-polygons footprints in the oracle ("polygon(s)", :129 "For a union of
polygons, the minimum distance over its components is used")."""
import numpy as np
import pytest

from harness import workloads as W


def rect(cx, cy, lx, ly):
    return (W.footprint_rect(lx, ly) + np.array([cx, cy], np.float32)).astype(np.float32)


def rect_distance(cx, cy, a, b, x, y):
    return float(np.hypot(max(abs(x - cx) - a, 0.0), max(abs(y - cy) - b, 0.0)))


@pytest.fixture()
def union(oracle_lib):
    return oracle_lib                                             # (components are an argument of every call: nothing to leak)


def test_l_shape_equals_its_two_rectangles(union):
    # the L of config 3 (0.8 x 0.6 box minus the 0.4 x 0.3 notch at +x +y) = two rectangles sharing an edge
    L = W.footprint_L()
    parts = np.concatenate([rect(0.0, -0.15, 0.8, 0.3), rect(-0.2, 0.15, 0.4, 0.3)])
    wl = W.make_workload(3, n_envs=8)
    pose = W.random_poses(wl, 3000, seed=5)
    f1, a1 = union.collision(wl.occ, wl.resolution, L, pose[0], pose[1], pose[2])
    f2, a2 = union.collision(wl.occ, wl.resolution, parts, pose[0], pose[1], pose[2], components=[4, 4])
    ok = (a1 == 0) & (a2 == 0)
    assert ok.mean() > 0.99 and np.array_equal(f1[ok], f2[ok]) and 0.2 < f1.mean() < 0.98
    rng = np.random.default_rng(0)
    for x, y in rng.uniform(-1.2, 1.2, (1500, 2)):
        d1 = union.footprint_distance(L, x, y)
        d2 = union.footprint_distance(parts, x, y, components=[4, 4])
        assert abs(d1 - d2) < 1e-6


def test_disjoint_and_overlapping_components(union):
    # a dumbbell (two disjoint squares) and a plus sign (two overlapping bars)
    bells = np.concatenate([rect(-0.5, 0.0, 0.3, 0.3), rect(0.5, 0.0, 0.3, 0.3)])
    C2 = [4, 4]
    rng = np.random.default_rng(1)
    for x, y in rng.uniform(-1.5, 1.5, (2000, 2)):
        expect = min(rect_distance(-0.5, 0, 0.15, 0.15, x, y), rect_distance(0.5, 0, 0.15, 0.15, x, y))
        assert abs(union.footprint_distance(bells, x, y, components=C2) - expect) < 1e-6
    assert union.footprint_distance(bells, 0.0, 0.0, components=C2) == pytest.approx(0.35, abs=1e-6)      # the gap is outside
    plus = np.concatenate([rect(0, 0, 0.8, 0.2), rect(0, 0, 0.2, 0.8)])
    # the overlap of the two bars is INSIDE the union (a single even-odd pass over both loops would call it outside)
    assert union.footprint_distance(plus, 0.0, 0.0, components=C2) == 0.0 and union.footprint_distance(plus, 0.05, -0.05, components=C2) == 0.0
    assert union.footprint_distance(plus, 0.3, 0.3, components=C2) == pytest.approx(0.2, abs=1e-6)
    # the same vertex lists read as ONE polygon give something else: the argument matters
    assert union.footprint_distance(plus, 0.0, 0.0) != 0.0 or union.footprint_distance(bells, 0.0, 0.0) != pytest.approx(0.35, abs=1e-6)
    # collision of the dumbbell on a single occupied cell: OR of the two squares' interval overlaps
    occ = np.zeros((60, 60), np.uint8)
    occ[30, 30] = 1
    res = np.float32(0.05)
    xs = rng.uniform(0.8, 2.2, 3000).astype(np.float32)
    ys = rng.uniform(1.2, 1.8, 3000).astype(np.float32)
    psi = np.zeros(3000, np.float32)
    flag, amb = union.collision(occ, res, bells, xs, ys, psi, components=C2)

    def hits(cx):                                                   # closed square [cx-0.15, cx+0.15]^2 vs cell [1.5, 1.55]^2
        lo_x, hi_x = xs.astype(np.float64) + cx - 0.15, xs.astype(np.float64) + cx + 0.15
        lo_y, hi_y = ys.astype(np.float64) - 0.15, ys.astype(np.float64) + 0.15
        return (hi_x >= 1.5) & (lo_x <= 1.55) & (hi_y >= 1.5) & (lo_y <= 1.55)
    expect = hits(-0.5) | hits(0.5)
    ok = amb == 0
    assert ok.mean() > 0.99 and np.array_equal(flag[ok] != 0, expect[ok]) and 0.05 < expect.mean() < 0.9


def test_reset_and_features_follow_the_union(union):
    bells = np.concatenate([rect(-0.5, 0.0, 0.3, 0.3), rect(0.5, 0.0, 0.3, 0.3)])
    wl = W.make_workload(1, n_envs=200)
    C2 = [4, 4]
    st = np.zeros((8, 200), np.float32); dp = np.zeros(200, np.float32); ep = np.zeros(200, np.int32)
    seeds = W.seed_tape(wl, 1, 3)
    union.reset(wl.occ, wl.resolution, bells, None, wl.goal_dist_min, wl.goal_dist_max, np.ones(200, np.uint8),
                seeds[0], st, dp, ep, components=C2)
    flag, _ = union.collision(wl.occ, wl.resolution, bells, st[0], st[1], st[2], components=C2)
    assert not flag.any()                                         # accepted start poses are collision-free for the union
    # ... while a single square at the body origin would accept poses the union rejects: the rule really uses both parts
    f_left, _ = union.collision(wl.occ, wl.resolution, bells, st[0] + np.float32(0.0), st[1], st[2], components=C2)
    assert not f_left.any()
    ang = W.beam_table(72, 360.0)
    r = np.full((1, 72), 1.0, np.float32)
    z = union.clearance_features(bells, ang, 5.0, 72, r, components=C2)
    expect = [min(rect_distance(-0.5, 0, 0.15, 0.15, np.cos(a), np.sin(a)), rect_distance(0.5, 0, 0.15, 0.15, np.cos(a), np.sin(a)))
              for a in ang.astype(np.float64)]
    assert np.allclose(z[0], expect, atol=2e-6)
