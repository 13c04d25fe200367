"""Pins for the oracle's O4 (range sensing): what the mathematics fixes independently of the grid walk.
PAPER.md:86 (fixed-step samples), :133 (no hit => max range), :123 (outside the map is occupied)."""
import numpy as np

from harness import workloads as W

RHO = np.float32(0.05)


def _angles(n):
    return (-np.pi + np.arange(n) * 2 * np.pi / n).astype(np.float32)


def test_empty_map_gives_max_range(oracle_lib):
    occ = np.zeros((256, 256), np.uint8)
    ang = _angles(90)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 5.0, [6.4, 6.1], [6.4, 6.7], [0.3, -2.0])
    assert np.all(r == np.float32(5.0)) and np.all(hit == -1)


def test_axis_aligned_wall_analytic(oracle_lib):
    # wall occupying columns >= 150: r = (150 rho - o_x) / cos(phi) for beams that reach it
    occ = np.zeros((1200, 400), np.uint8)
    occ[:, 150:] = 1
    ang = np.linspace(-1.2, 1.2, 101).astype(np.float32)
    x, y, psi = np.float32(3.21), np.float32(30.0), np.float32(0.1)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 20.0, [x], [y], [psi])
    phi = np.float64(psi) + ang.astype(np.float64)
    want = (150 * np.float64(RHO) - np.float64(x)) / np.cos(phi)
    assert np.allclose(r[0], want, atol=1e-6)
    # hit cell is in column 150, row = floor of the crossing ordinate
    rows = np.floor((np.float64(y) + want * np.sin(phi)) / np.float64(RHO)).astype(int)
    assert np.array_equal(hit[0][amb[0] == 0], (rows * 400 + 150)[amb[0] == 0])


def test_wall_in_each_direction(oracle_lib):
    # same wall seen along +x, -x, +y, -y: catches a swapped axis or sign in the walk
    n = 201
    for k, (sl, phi0) in enumerate([((slice(None), slice(150, None)), 0.0),
                                    ((slice(None), slice(None, 51)), np.pi),
                                    ((slice(150, None), slice(None)), np.pi / 2),
                                    ((slice(None, 51), slice(None)), -np.pi / 2)]):
        occ = np.zeros((n, n), np.uint8)
        occ[sl] = 1
        ang = np.array([-0.4, 0.0, 0.3], np.float32)
        x = y = np.float32(100.5 * 0.05)
        r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 20.0, [x], [y], [np.float32(phi0)])
        gap = (150 * np.float64(RHO) - np.float64(x)) if k in (0, 2) else (np.float64(x) - 51 * np.float64(RHO))
        assert np.allclose(r[0], gap / np.cos(ang.astype(np.float64) + (np.float64(np.float32(phi0)) - phi0)), atol=2e-6), k


def _slab(ox, oy, dx, dy, xl, xh, yl, yh):
    """textbook ray/box slab intersection: entry parameter or inf (numpy, independent of the oracle)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        tx1, tx2 = (xl - ox) / dx, (xh - ox) / dx
        ty1, ty2 = (yl - oy) / dy, (yh - oy) / dy
    tmin = np.maximum(np.minimum(tx1, tx2), np.minimum(ty1, ty2))
    tmax = np.minimum(np.maximum(tx1, tx2), np.maximum(ty1, ty2))
    return np.where((tmax >= np.maximum(tmin, 0)), np.maximum(tmin, 0), np.inf)


def test_single_cell_slab_closed_form(oracle_lib):
    occ = np.zeros((256, 256), np.uint8)
    occ[140, 123] = 1
    ang = _angles(3600)
    x, y, psi = np.float32(5.013), np.float32(5.507), np.float32(0.0)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 3.0, [x], [y], [psi])
    rho = np.float64(RHO)
    phi = ang.astype(np.float64)
    t = _slab(x / rho, y / rho, np.cos(phi), np.sin(phi), 123.0, 124.0, 140.0, 141.0) * rho
    want = np.where(t < 3.0, t, 3.0)
    ok = amb[0] == 0
    assert ok.mean() > 0.99
    assert np.allclose(r[0][ok], want[ok], atol=1e-6)
    assert np.all(hit[0][ok & (t < 3.0)] == 140 * 256 + 123) and np.all(hit[0][ok & (t >= 3.0)] == -1)
    assert (t < 3.0).sum() > 20


def test_union_of_cells_is_min_over_slabs(oracle_lib):
    # r = min over occupied cells of the slab entry distance (plain definition, brute force)
    wl = W.tiny_workload(size=24, seed=3, frac=0.2)
    occ = wl.occ.copy()
    occ[0, :] = occ[-1, :] = 0
    occ[:, 0] = occ[:, -1] = 0                                  # no border: exercises the outside rule
    ang = _angles(97)
    poses = W.random_poses(wl, 40, 1)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 0.9, poses[0], poses[1], poses[2])
    rho = np.float64(RHO)
    ii, jj = np.nonzero(occ)
    H, Wd = occ.shape
    for e in range(poses.shape[1]):
        ox, oy = poses[0, e] / rho, poses[1, e] / rho
        phi = np.float64(poses[2, e]) + ang.astype(np.float64)
        dx, dy = np.cos(phi)[:, None], np.sin(phi)[:, None]
        t = _slab(ox, oy, dx, dy, jj[None, :], jj[None, :] + 1.0, ii[None, :], ii[None, :] + 1.0).min(1)
        # leaving the map counts as hitting an occupied cell: exit parameter of the map rectangle
        with np.errstate(divide="ignore"):
            tex = np.minimum(np.where(dx[:, 0] > 0, (Wd - ox) / dx[:, 0], np.where(dx[:, 0] < 0, -ox / dx[:, 0], np.inf)),
                             np.where(dy[:, 0] > 0, (H - oy) / dy[:, 0], np.where(dy[:, 0] < 0, -oy / dy[:, 0], np.inf)))
        t = np.minimum(t, tex)
        want = np.where(t * rho < 0.9, t * rho, 0.9)
        ok = amb[e] == 0
        assert np.allclose(r[e][ok], want[ok], atol=1e-6), e
        out = ok & (tex * rho < 0.9) & (tex <= t)
        assert np.all(hit[e][out & (tex < t - 1e-9)] == -2)


def test_fixed_step_march_brackets_exact(oracle_lib):
    # the paper's own definition with step D: r_exact <= r_march <= r_exact + D
    for seed, size in ((1, 32), (2, 20)):
        wl = W.tiny_workload(size=size, seed=seed, frac=0.15)
        ang = _angles(64)
        poses = W.random_poses(wl, 60, seed)
        r, hit, amb = oracle_lib.ranges(wl.occ, RHO, ang, 1.0, poses[0], poses[1], poses[2])
        D = float(RHO) / 256
        rm = oracle_lib.ranges_fixed_step(wl.occ, RHO, ang, 1.0, D, poses[0], poses[1], poses[2])
        assert np.all(r <= rm + 1e-6)
        ok = amb == 0
        assert ok.mean() > 0.98
        # the march can only overshoot by D unless it tunnels through a sliver thinner than D (corner graze)
        over = (rm - r)[ok]
        assert (over <= D + 1e-6).mean() > 0.995
        assert np.all(r[hit == -1] == np.float32(1.0))


def _rot90_pose(pose, H, Wd, rho):
    """np.rot90(occ, 1): new[i', j'] = old[j', Wd-1-i']  <=>  x' = y, y' = Wd*rho - x, psi' = psi - pi/2."""
    x, y, psi = pose.astype(np.float64)
    return np.stack([y, Wd * rho - x, psi - np.pi / 2]).astype(np.float32)


def test_symmetries(oracle_lib):
    wl = W.tiny_workload(size=32, seed=5, frac=0.15)
    occ = wl.occ
    H, Wd = occ.shape
    rho = np.float64(RHO)
    ang = _angles(72)
    # poses on a grid of exactly representable numbers so the transformed pose is the exact image
    rng = np.random.default_rng(0)
    x = (rng.integers(64, 32 * 64 - 64, 50) / 64.0 * 0.05).astype(np.float32)
    y = (rng.integers(64, 32 * 64 - 64, 50) / 64.0 * 0.05).astype(np.float32)
    psi = np.zeros(50, np.float32)
    r0, h0, a0 = oracle_lib.ranges(occ, RHO, ang, 1.0, x, y, psi)
    # transpose: swap x and y, mirror angles: beam at angle t maps to angle pi/2 - t
    rT, hT, aT = oracle_lib.ranges(np.ascontiguousarray(occ.T), RHO, (np.float32(np.pi / 2) - ang).astype(np.float32),
                                   1.0, y, x, psi)
    ok = (a0 == 0) & (aT == 0)
    assert ok.mean() > 0.95 and np.allclose(r0[ok], rT[ok], atol=2e-6)
    i0, j0 = np.divmod(h0, Wd)
    assert np.array_equal((j0 * H + i0)[ok & (h0 >= 0)], hT[ok & (h0 >= 0)])
    # left-right flip: x -> W rho - x, angle t -> pi - t
    rF, hF, aF = oracle_lib.ranges(np.ascontiguousarray(occ[:, ::-1]), RHO, (np.float32(np.pi) - ang).astype(np.float32),
                                   1.0, (Wd * rho - x.astype(np.float64)).astype(np.float32), y, psi)
    ok = (a0 == 0) & (aF == 0)
    assert ok.mean() > 0.95 and np.allclose(r0[ok], rF[ok], atol=2e-6)


def test_origin_inside_obstacle_and_outside_map(oracle_lib):
    occ = np.zeros((16, 16), np.uint8)
    occ[5, 7] = 1
    ang = _angles(8)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 1.0, [7.5 * 0.05], [5.5 * 0.05], [0.0])
    assert np.all(r == 0) and np.all(hit == 5 * 16 + 7)
    r, hit, amb = oracle_lib.ranges(occ, RHO, ang, 1.0, [-0.2], [0.3], [0.0])
    assert np.all(r == 0) and np.all(hit == -2)
    # a beam leaving the map hits "outside" at the map edge: 16 cells wide, origin at cell 14.5
    r, hit, amb = oracle_lib.ranges(occ, RHO, np.zeros(1, np.float32), 1.0, [14.5 * 0.05], [2.5 * 0.05], [0.0])
    assert abs(r[0, 0] - 1.5 * 0.05) < 1e-6 and hit[0, 0] == -2


def test_range_cap_and_hit_cell_consistency(oracle_lib):
    wl = W.make_workload(1)
    poses = W.random_poses(wl, 32, 3)
    r, hit, amb, vis = oracle_lib.ranges(wl.occ, wl.resolution, wl.beam_angles, wl.max_range,
                                         poses[0], poses[1], poses[2], eps=1e-3, want_visits=True)
    assert (amb == 0).mean() > 0.97
    assert r.max() <= wl.max_range and r.min() >= 0 and vis.min() >= 1
    H, Wd = wl.occ.shape
    rho = np.float64(wl.resolution)
    e, b = np.nonzero((hit >= 0) & (amb == 0) & (r > 0))
    phi = poses[2, e].astype(np.float64) + wl.beam_angles[b].astype(np.float64)
    # a point just beyond the reported range lies in the reported (occupied) cell ...
    t = r[e, b].astype(np.float64) + 2e-6
    px, py = (poses[0, e] + t * np.cos(phi)) / rho, (poses[1, e] + t * np.sin(phi)) / rho
    assert np.array_equal(np.floor(py).astype(int) * Wd + np.floor(px).astype(int), hit[e, b])
    assert np.all(wl.occ.reshape(-1)[hit[e, b]] == 1)
    # ... and a point just before it lies in a free cell
    t = r[e, b].astype(np.float64) - 2e-6
    px, py = (poses[0, e] + t * np.cos(phi)) / rho, (poses[1, e] + t * np.sin(phi)) / rho
    assert np.all(wl.occ[np.floor(py).astype(int), np.floor(px).astype(int)] == 0)


def test_sensor_offset(oracle_lib):
    # sensor mounted 0.1 m ahead, yawed by 0.5 rad == a robot 0.1 m further along its heading, yawed
    wl = W.tiny_workload(size=32, seed=9)
    ang = _angles(16)
    x, y, psi = np.float32(0.8), np.float32(0.8), np.float32(0.25)
    r1, h1, _ = oracle_lib.ranges(wl.occ, RHO, ang, 1.0, [x], [y], [psi], sensor=[0.1, 0.0, 0.5])
    x2 = np.float32(x + 0.1 * np.cos(np.float64(psi)))
    y2 = np.float32(y + 0.1 * np.sin(np.float64(psi)))
    r2, h2, _ = oracle_lib.ranges(wl.occ, RHO, ang, 1.0, [x2], [y2], [np.float32(psi + np.float32(0.5))])
    assert np.allclose(r1, r2, atol=1e-5)


def test_several_sensors(oracle_lib):
    # a robot with several range sensors, each with its own placement, beam
    # table and maximum range; the observation is the sensors' ranges one after the other.  Pins: (1) every sensor's
    # block equals a single-sensor robot with that sensor (the single-sensor function is pinned above: analytic
    # walls, slab formula, brute force); (2) a sensor with an offset is a moved, yawed robot (hand-computed pose);
    # (3) a wall straight ahead: front sensor at +0.2 m and rear-facing sensor at -0.2 m see analytic distances.
    wl = W.tiny_workload(size=32, seed=9)
    rng = np.random.default_rng(3)
    n = 40
    x = (0.3 + rng.random(n)).astype(np.float32); y = (0.3 + rng.random(n)).astype(np.float32)
    psi = (rng.random(n) * 6.28 - 3.14).astype(np.float32)
    sensors = [(_angles(16), 1.0, (0.1, 0.0, 0.5)), (_angles(7), 0.6, (-0.05, 0.08, -2.0)), (_angles(24), 1.4, (0.0, 0.0, 0.0))]
    r, h, a = oracle_lib.ranges_multi(wl.occ, RHO, sensors, x, y, psi)
    assert r.shape == (n, 47)
    off = 0
    for ang, rmax, plc in sensors:
        r1, h1, a1 = oracle_lib.ranges(wl.occ, RHO, ang, rmax, x, y, psi, sensor=list(plc))
        assert np.array_equal(r[:, off:off + len(ang)], r1) and np.array_equal(h[:, off:off + len(ang)], h1)
        assert np.array_equal(a[:, off:off + len(ang)], a1)
        assert r1.max() <= rmax + 1e-6
        off += len(ang)
    # (2) moved robot, for the second sensor
    ang, rmax, (sx, sy, sp) = sensors[1]
    c, s = np.cos(psi.astype(np.float64)), np.sin(psi.astype(np.float64))
    x2 = (x + c * sx - s * sy).astype(np.float32); y2 = (y + s * sx + c * sy).astype(np.float32)
    r2, _, a2 = oracle_lib.ranges(wl.occ, RHO, ang, rmax, x2, y2, (psi + np.float32(sp)).astype(np.float32))
    ok = (a[:, 16:23] == 0) & (a2 == 0)
    assert ok.mean() > 0.9 and np.allclose(r[:, 16:23][ok], r2[ok], atol=2e-5)
    # (3) analytic: empty 64 x 64 map with a wall at column 40 (x = 2.0 m) and its border at column 0
    occ = np.zeros((64, 64), np.uint8); occ[:, 40] = 1; occ[:, 0] = 1; occ[0, :] = 1; occ[-1, :] = 1
    front = (np.zeros(1, np.float32), 3.0, (0.2, 0.0, 0.0))
    rear = (np.zeros(1, np.float32), 3.0, (-0.2, 0.0, np.pi))
    rr, hh, _ = oracle_lib.ranges_multi(occ, RHO, [front, rear], np.float32([1.0]), np.float32([1.625]), np.float32([0.0]))
    assert abs(rr[0, 0] - (2.0 - 1.2)) < 1e-6 and abs(rr[0, 1] - (0.8 - 0.05)) < 1e-6
    assert hh[0, 0] == 32 * 64 + 40 and hh[0, 1] == 32 * 64 + 0
