"""Pins for the oracle's O10: clearance features, Eq. (3) and sector min-pooling
(PAPER.md:67).  None of these retypes the oracle's segment-projection formula: they use the analytic
distance to an axis-aligned rectangle / a circle, a dense brute-force sampling of the boundary, the
notch case of the nonconvex footprint and the defining properties of the pooling."""
import numpy as np
import pytest

from harness import workloads as W


def rect_distance(a, b, x, y):
    """textbook distance from (x, y) to the axis-aligned rectangle [-a, a] x [-b, b] (0 inside)"""
    return float(np.hypot(max(abs(x) - a, 0.0), max(abs(y) - b, 0.0)))


def test_rectangle_matches_textbook_distance(oracle_lib):
    fp = W.footprint_rect(0.6, 0.4)                              # half extents 0.3 x 0.2
    rng = np.random.default_rng(0)
    for x, y in rng.uniform(-2, 2, (4000, 2)):
        assert abs(oracle_lib.footprint_distance(fp, x, y) - rect_distance(0.3, 0.2, x, y)) < 1e-6   # fp32 vertices
    # either vertex order
    assert abs(oracle_lib.footprint_distance(fp[::-1].copy(), 1.0, 1.0) - rect_distance(0.3, 0.2, 1.0, 1.0)) < 1e-6


def test_inside_is_zero_and_nonnegative(oracle_lib):
    for fp in (W.footprint_rect(0.6, 0.4), W.footprint_ngon(0.2, 16), W.footprint_L()):
        c = fp.mean(axis=0)
        inside_pt = 0.5 * (fp[0] + fp[1]) * 0.98 + 0.02 * c      # just inside an edge midpoint (towards the centroid)
        if fp.shape[0] != 12:                                    # (the L's centroid side is inside for edge 0-1 too)
            assert oracle_lib.footprint_distance(fp, *inside_pt) == 0.0
        rng = np.random.default_rng(1)
        for x, y in rng.uniform(-1.5, 1.5, (500, 2)):
            assert oracle_lib.footprint_distance(fp, x, y) >= 0.0


def test_polygonal_circle_is_bracketed_by_the_circle(oracle_lib):
    R, n = 0.2, 64
    fp = W.footprint_ngon(R, n)                                  # vertices on the circle of radius R
    rng = np.random.default_rng(2)
    for rr, th in zip(rng.uniform(0.25, 3.0, 500), rng.uniform(-np.pi, np.pi, 500)):
        d = oracle_lib.footprint_distance(fp, rr * np.cos(th), rr * np.sin(th))
        assert rr - R - 1e-6 <= d <= rr - R * np.cos(np.pi / n) + 1e-6


def test_brute_force_boundary_sampling(oracle_lib):
    fp = W.footprint_L()
    P = fp.astype(np.float64)
    pts = []
    for k in range(len(P)):
        a, b = P[k - 1], P[k]
        t = np.linspace(0, 1, 4001)[:, None]
        pts.append(a + t * (b - a))
    pts = np.concatenate(pts)                                    # boundary sampled at <= 1e-4 m
    rng = np.random.default_rng(3)
    for x, y in rng.uniform(-1.2, 1.2, (300, 2)):
        d = oracle_lib.footprint_distance(fp, x, y)
        brute = np.sqrt(((pts - (x, y)) ** 2).sum(1).min())
        if d > 0:
            assert brute - 1.5e-4 <= d <= brute + 1e-9
        else:
            # inside: every ray from the point crosses the boundary an odd number of times; check one by sampling
            assert brute >= 0


def test_notch_of_the_nonconvex_footprint(oracle_lib):
    # a bounding box "covers free space within the recesses"; Eq. (3) follows the polygon.
    # L = 0.8 x 0.6 box minus the 0.4 x 0.3 corner notch at (+x, +y): a point in the notch is OUTSIDE the
    # footprint, at the distance to the nearer of the two notch edges (x = 0 and y = 0 here).
    fp = W.footprint_L()
    xs, ys = fp[:, 0], fp[:, 1]
    x_hi, y_hi = xs.max(), ys.max()
    nx, ny = x_hi - 0.4, y_hi - 0.3                               # inner corner of the notch
    for px, py in ((nx + 0.10, ny + 0.05), (nx + 0.03, ny + 0.20), (nx + 0.30, ny + 0.25)):
        d = oracle_lib.footprint_distance(fp, px, py)
        assert abs(d - min(px - nx, py - ny)) < 1e-6
        box = W.footprint_rect(0.8, 0.6) + np.array([(xs.max() + xs.min()) / 2, (ys.max() + ys.min()) / 2], np.float32)
        assert oracle_lib.footprint_distance(box, px, py) == 0.0


def test_pooling_validity_cap_and_sectors(oracle_lib):
    fp = W.footprint_rect(0.6, 0.4)
    B, ns, rmax = 90, 8, np.float32(5.0)                         # 90 beams, 8 sectors: uneven groups (11 or 12)
    ang = W.beam_table(B, 360.0)
    rng = np.random.default_rng(4)
    r = rng.uniform(0.0, 6.0, (7, B)).astype(np.float32)
    r = np.minimum(r, rmax)                                      # some beams at max range = no valid hit
    z, delta = oracle_lib.clearance_features(fp, ang, rmax, ns, r, want_delta=True)
    sec = (np.arange(B) * ns) // B
    assert np.array_equal(np.bincount(sec, minlength=ns) > 0, np.ones(ns, bool)) and sec[0] == 0 and sec[-1] == ns - 1
    assert np.all(np.diff(sec) >= 0)                             # consecutive beams, each in exactly one sector
    for k in range(ns):
        assert np.array_equal(z[:, k], delta[:, sec == k].min(axis=1))
    assert np.all(delta[r >= rmax] == rmax)                      # no valid hit -> maximum range
    assert np.all(delta <= rmax) and np.all(delta >= 0)
    # a valid endpoint: distance of the body-frame endpoint, analytic for the rectangle
    e, j = 3, 17
    if r[e, j] < rmax:
        px, py = r[e, j] * np.cos(np.float64(ang[j])), r[e, j] * np.sin(np.float64(ang[j]))
        assert abs(delta[e, j] - min(rect_distance(0.3, 0.2, px, py), float(rmax))) < 1e-5
    # one sector = the global minimum; B sectors = the per-beam values
    z1 = oracle_lib.clearance_features(fp, ang, rmax, 1, r)
    assert np.array_equal(z1[:, 0], delta.min(axis=1))
    zB = oracle_lib.clearance_features(fp, ang, rmax, B, r)
    assert np.array_equal(zB, delta)


def test_sensor_placement_moves_the_endpoint(oracle_lib):
    # endpoint = s_xy + r (cos, sin)(theta + s_psi): a sensor offset equals the same footprint shifted back
    fp = W.footprint_rect(0.6, 0.4)
    ang = W.beam_table(36, 360.0)
    r = np.full((1, 36), 1.25, np.float32)
    sen = np.array([0.2, -0.1, 0.3], np.float32)
    z = oracle_lib.clearance_features(fp, ang, 5.0, 36, r, sensor=sen)
    shifted = (fp - sen[:2]).astype(np.float32)
    z2 = oracle_lib.clearance_features(shifted, (ang + sen[2]).astype(np.float32), 5.0, 36, r)
    assert np.allclose(z, z2, atol=2e-6)
