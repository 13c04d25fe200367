"""Pins for the oracle's O3 (footprint collision): PAPER.md:100-102, :118-123 (Eq. 2)."""
import numpy as np

from harness import workloads as W

RHO = np.float32(0.05)


def test_axis_aligned_rectangle_is_interval_overlap(oracle_lib):
    # at psi = 0 a rectangle [x-hl, x+hl] x [y-hw, y+hw] meets cell (i, j) iff the closed intervals overlap
    rng = np.random.default_rng(0)
    occ = np.zeros((40, 40), np.uint8)
    occ[17, 22] = 1
    fp = W.footprint_rect(0.6, 0.4)
    n = 4000
    x = (rng.uniform(14, 31, n) * 0.05).astype(np.float32)
    y = (rng.uniform(11, 24, n) * 0.05).astype(np.float32)
    flag, amb = oracle_lib.collision(occ, RHO, fp, x, y, np.zeros(n, np.float32))
    rho = np.float64(RHO)
    xc, yc = x / rho, y / rho
    hl, hw = np.float64(fp[1, 0]) / rho, np.float64(fp[2, 1]) / rho
    want = (xc - hl <= 23) & (xc + hl >= 22) & (yc - hw <= 18) & (yc + hw >= 17)
    ok = amb == 0
    assert ok.mean() > 0.99 and np.array_equal(flag[ok] != 0, want[ok])
    assert 0.1 < want.mean() < 0.9


def test_outside_map_is_collision(oracle_lib):
    occ = np.zeros((40, 40), np.uint8)
    fp = W.footprint_rect(0.6, 0.4)
    x = np.array([0.29, 0.31, 1.0, 1.0, 1.71, 1.69], np.float32)
    y = np.array([1.0, 1.0, 0.19, 0.21, 1.0, 1.0], np.float32)
    flag, amb = oracle_lib.collision(occ, RHO, fp, x, y, np.zeros(6, np.float32))
    assert list(flag) == [1, 0, 1, 0, 1, 0]


def test_ngon_vertex_direction_gap(oracle_lib):
    # a regular 16-gon of circumradius r with a vertex pointing at +x: touches the wall at x_w iff gap <= r
    occ = np.zeros((60, 60), np.uint8)
    occ[:, 40:] = 1
    fp = W.footprint_ngon(0.2, 16)
    r = np.float64(fp[0, 0])
    gaps = np.linspace(0.15, 0.25, 401)
    x = (40 * np.float64(RHO) - gaps).astype(np.float32)
    y = np.full_like(x, 1.5125)
    flag, amb = oracle_lib.collision(occ, RHO, fp, x, y, np.zeros_like(x))
    want = (40 * np.float64(RHO) - x.astype(np.float64)) <= r
    ok = amb == 0
    assert np.array_equal(flag[ok] != 0, want[ok]) and ok.sum() > 390
    # rotated by half a sector the nearest boundary point is an edge midpoint at r cos(pi/16)
    psi = np.full_like(x, np.pi / 16)
    flag, amb = oracle_lib.collision(occ, RHO, fp, x, y, psi)
    want = (40 * np.float64(RHO) - x.astype(np.float64)) <= r * np.cos(np.pi / 16) + 1e-9
    ok = amb == 0
    assert np.array_equal(flag[ok] != 0, want[ok])


def test_notch_is_free_space(oracle_lib):
    # "A single rectangular bounding box covers free space within the recesses" of a
    # nonconvex footprint.  An occupied cell inside the L's notch: no collision; bounding box: collision.
    occ = np.zeros((80, 80), np.uint8)
    fpL = W.footprint_L()
    bbox = W.footprint_rect(0.8, 0.6)
    x, y = np.float32(2.0), np.float32(2.0)
    # notch = body-frame x in [0, 0.4], y in [0, 0.3]; a cell well inside it, 0.2 m / 0.15 m from the corner
    i, j = int((2.0 + 0.15) / 0.05), int((2.0 + 0.2) / 0.05)
    occ[i, j] = 1
    f1, _ = oracle_lib.collision(occ, RHO, fpL, [x], [y], [0.0])
    f2, _ = oracle_lib.collision(occ, RHO, bbox, [x], [y], [0.0])
    assert f1[0] == 0 and f2[0] == 1
    # rotate the robot by pi: the notch moves to the opposite corner and the cell is now under the body
    f3, _ = oracle_lib.collision(occ, RHO, fpL, [x], [y], [np.float32(np.pi)])
    assert f3[0] == 1
    # an occupied cell swallowed entirely by the polygon interior (no edge touches it) still collides
    occ[:] = 0
    occ[int((2.0 - 0.15) / 0.05), int((2.0 - 0.2) / 0.05)] = 1
    f4, _ = oracle_lib.collision(occ, RHO, fpL, [x], [y], [0.0])
    assert f4[0] == 1


def _pip(vx, vy, px, py):
    """vectorised even-odd rule (numpy, independent of the oracle)."""
    inside = np.zeros(px.shape, bool)
    V = len(vx)
    for a in range(V):
        b = (a - 1) % V
        with np.errstate(divide="ignore", invalid="ignore"):
            cond = ((vy[a] > py) != (vy[b] > py)) & (px < (vx[b] - vx[a]) * (py - vy[a]) / (vy[b] - vy[a]) + vx[a])
        inside ^= cond
    return inside


def _supersample(occ, fp, x, y, psi, K=64):
    """brute force: K x K points in every occupied cell (and a one-cell ring outside the map); any in polygon?"""
    rho = np.float64(RHO)
    H, Wd = occ.shape
    c, s = np.cos(np.float64(psi)), np.sin(np.float64(psi))
    vx = (np.float64(x) + c * fp[:, 0].astype(np.float64) - s * fp[:, 1].astype(np.float64)) / rho
    vy = (np.float64(y) + s * fp[:, 0].astype(np.float64) + c * fp[:, 1].astype(np.float64)) / rho
    g = (np.arange(K) + 0.5) / K
    for i in range(int(np.floor(vy.min())), int(np.floor(vy.max())) + 1):
        for j in range(int(np.floor(vx.min())), int(np.floor(vx.max())) + 1):
            o = 1 if (i < 0 or j < 0 or i >= H or j >= Wd) else occ[i, j]
            if o:
                px, py = np.meshgrid(j + g, i + g)
                if _pip(vx, vy, px, py).any():
                    return 1
    return 0


def _scaled(fp, centre, s):
    c = np.asarray(centre, np.float32)
    return (c + s * (fp - c)).astype(np.float32)


def test_supersampling_and_eq2_sampling_bracket_exact(oracle_lib):
    # (a) brute force / Eq. (2) sampling says collision  =>  exact says collision   (always)
    # (b) exact collision of the footprint shrunk towards a kernel point by 10 %  =>  brute force and
    #     Eq. (2) sampling of the full footprint say collision (the overlap then contains a disc of
    #     radius >= 0.3 cell, which both samplings must hit)
    cases = [(W.footprint_rect(0.3, 0.2), (0.0, 0.0)), (W.footprint_ngon(0.2, 16), (0.0, 0.0)),
             (W.footprint_L(), (-0.2, -0.15))]
    for k, (fp, kern) in enumerate(cases):
        wl = W.tiny_workload(size=32, seed=10 + k, frac=0.15)
        poses = W.random_poses(wl, 300, k)
        flag, amb = oracle_lib.collision(wl.occ, RHO, fp, poses[0], poses[1], poses[2])
        shrunk, _ = oracle_lib.collision(wl.occ, RHO, _scaled(fp, kern, 0.9), poses[0], poses[1], poses[2])
        samp = oracle_lib.collision_sampled(wl.occ, RHO, fp, float(RHO) / 16, poses[0], poses[1], poses[2])
        sup = np.array([_supersample(wl.occ, fp, *poses[:, e]) for e in range(poses.shape[1])])
        assert np.all(flag[samp == 1] == 1) and np.all(flag[sup == 1] == 1)
        assert np.all(samp[shrunk == 1] == 1) and np.all(sup[shrunk == 1] == 1)
        assert np.all(flag[shrunk == 1] == 1)
        assert 0.15 < flag.mean() < 0.95, flag.mean()
        # the bracket is tight: exact and brute force disagree on only a sliver of poses
        assert (flag != sup).mean() < 0.05


def test_rotation_and_orientation_invariance(oracle_lib):
    wl = W.tiny_workload(size=32, seed=4, frac=0.15)
    poses = W.random_poses(wl, 400, 2)
    fp = W.footprint_L()
    f_ccw, a1 = oracle_lib.collision(wl.occ, RHO, fp, poses[0], poses[1], poses[2])
    f_cw, a2 = oracle_lib.collision(wl.occ, RHO, np.ascontiguousarray(fp[::-1]), poses[0], poses[1], poses[2])
    assert np.array_equal(f_ccw, f_cw)
    # transposed world: (x, y, psi) -> (y, x, pi/2 - psi) with the footprint mirrored in its own y axis
    fpm = fp.copy()
    fpm[:, 1] *= -1
    fT, a3 = oracle_lib.collision(np.ascontiguousarray(wl.occ.T), RHO, fpm, poses[1], poses[0],
                                  (np.float32(np.pi / 2) - poses[2]).astype(np.float32))
    ok = (a1 == 0) & (a3 == 0)
    assert ok.mean() > 0.98 and np.array_equal(f_ccw[ok], fT[ok])


def test_ambiguity_flag_marks_exact_touch(oracle_lib):
    occ = np.zeros((40, 40), np.uint8)
    occ[:, 30:] = 1
    fp = W.footprint_rect(0.5, 0.5)
    # right edge of the square exactly on the wall face x = 1.5 m (30 cells): touching, ambiguous
    flag, amb = oracle_lib.collision(occ, RHO, fp, [np.float32(1.25)], [np.float32(1.0)], [0.0])
    assert amb[0] == 1
    flag, amb = oracle_lib.collision(occ, RHO, fp, [np.float32(1.2), np.float32(1.3)], [1.0, 1.0], [0.0, 0.0])
    assert list(flag) == [0, 1] and list(amb) == [0, 0]
