"""Pins for the oracle's O1/O2 (clip + motion) and O5/O6 (goal obs, reward) -- closed forms and the
constants the paper prints."""
import os

import numpy as np

DIFF, OMNI = 0, 1
LIM_D = np.array([-5, 5, 0, 0, -5, 5], np.float32)
LIM_O = np.array([-5, 5, -5, 5, -5, 5], np.float32)


def _state(n, x=0.0, y=0.0, psi=0.0):
    s = np.zeros((8, n), np.float32)
    s[0], s[1], s[2] = x, y, psi
    return s


def test_diff_arc_closed_form(oracle_lib):
    # constant (v, w) from the origin: x = v/w sin(n w dt), y = v/w (1 - cos(n w dt)), psi = n w dt
    v, w, dt, n = 1.0, 2.0, 0.1, 12
    s = _state(1)
    a = np.array([[v, w]], np.float32)
    for k in range(1, n + 1):
        s = oracle_lib.motion(DIFF, LIM_D, dt, s, a)
        th = k * np.float64(np.float32(w)) * np.float64(np.float32(dt))
        assert abs(s[0, 0] - v / w * np.sin(th)) < 2e-6
        assert abs(s[1, 0] - v / w * (1 - np.cos(th))) < 2e-6
        assert abs(s[2, 0] - th) < 2e-6
    # a plain Euler step would be off by ~1e-2 m per step, midpoint by ~2e-4: both fail the bound above


def test_negative_turn_and_reverse(oracle_lib):
    v, w, dt = -0.5, -2.5, 0.1
    s = oracle_lib.motion(DIFF, LIM_D, dt, _state(1), np.array([[v, w]], np.float32))
    th = np.float64(np.float32(w)) * np.float64(np.float32(dt))
    assert abs(s[0, 0] - v / w * np.sin(th)) < 1e-6 and abs(s[1, 0] - v / w * (1 - np.cos(th))) < 1e-6
    assert s[1, 0] > 0 and s[0, 0] < 0      # reversing while turning clockwise: ends up behind, to the left


def test_straight_line_and_heading(oracle_lib):
    psi = 0.7
    s = oracle_lib.motion(DIFF, LIM_D, 0.1, _state(1, 1.0, 2.0, psi), np.array([[1.5, 0.0]], np.float32))
    assert abs(s[0, 0] - (1.0 + 0.15 * np.cos(np.float32(psi)))) < 1e-6
    assert abs(s[1, 0] - (2.0 + 0.15 * np.sin(np.float32(psi)))) < 1e-6
    assert s[2, 0] == np.float32(psi)
    # tiny but non-zero turn rate goes through the series branch and must agree with the limit
    s2 = oracle_lib.motion(DIFF, LIM_D, 0.1, _state(1, 1.0, 2.0, psi), np.array([[1.5, 1e-9]], np.float32))
    assert np.allclose(s[:2], s2[:2], atol=1e-7)


def test_omni_pure_translation_is_rotated(oracle_lib):
    # w = 0: displacement = R(psi) (vx, vy) dt ; at psi = pi/2 a lateral +vy moves along -x
    psi = np.float32(np.pi / 2)
    s = oracle_lib.motion(OMNI, LIM_O, 0.05, _state(1, 0, 0, psi), np.array([[0.0, 1.0, 0.0]], np.float32))
    assert abs(s[0, 0] + 0.05) < 1e-6 and abs(s[1, 0]) < 1e-6
    s = oracle_lib.motion(OMNI, LIM_O, 0.05, _state(1, 0, 0, 0), np.array([[0.3, 1.0, 0.0]], np.float32))
    assert abs(s[0, 0] - 0.015) < 1e-7 and abs(s[1, 0] - 0.05) < 1e-7


def test_omni_with_zero_lateral_equals_diff(oracle_lib):
    rng = np.random.default_rng(0)
    n = 64
    s = _state(n)
    s[:3] = rng.normal(size=(3, n)).astype(np.float32)
    vw = rng.uniform(-2, 2, size=(n, 2)).astype(np.float32)
    a3 = np.stack([vw[:, 0], np.zeros(n, np.float32), vw[:, 1]], 1)
    d = oracle_lib.motion(DIFF, LIM_D, 0.1, s, vw)
    o = oracle_lib.motion(OMNI, LIM_O, 0.1, s, a3)
    assert np.array_equal(d, o)


def test_omni_arc_matches_fine_integration(oracle_lib):
    # independent check of the (A, C) coefficients: integrate the body-frame twist with 20000 tiny
    # explicit steps in numpy fp64 and compare with one oracle step.
    vx, vy, w, dt = 0.8, -0.6, 1.9, 0.25
    x = y = 0.0
    psi = 0.3
    m = 20000
    h = dt / m
    for k in range(m):
        pm = psi + 0.5 * w * h
        x += h * (vx * np.cos(pm) - vy * np.sin(pm))
        y += h * (vx * np.sin(pm) + vy * np.cos(pm))
        psi += w * h
    s = oracle_lib.motion(OMNI, LIM_O, dt, _state(1, 0, 0, 0.3), np.array([[vx, vy, w]], np.float32))
    assert abs(s[0, 0] - x) < 1e-6 and abs(s[1, 0] - y) < 1e-6 and abs(s[2, 0] - psi) < 1e-6


def test_composition_two_half_steps(oracle_lib):
    a = np.array([[0.9, -1.3, 1.7]], np.float32)
    one = oracle_lib.motion(OMNI, LIM_O, 0.2, _state(1, 3, 4, 0.5), a)
    half = oracle_lib.motion(OMNI, LIM_O, 0.1, _state(1, 3, 4, 0.5), a)
    half[3:6] = 0
    two = oracle_lib.motion(OMNI, LIM_O, 0.1, half, a)
    assert np.allclose(one[:3], two[:3], atol=2e-6)


def test_clip_to_limits_and_diff_has_no_lateral(oracle_lib):
    lim = np.array([-0.5, 1.5, 0, 0, -2.5, 2.5], np.float32)
    s = oracle_lib.motion(DIFF, lim, 0.1, _state(2), np.array([[9.0, -9.0], [-9.0, 9.0]], np.float32))
    assert list(s[3]) == [1.5, -0.5] and list(s[4]) == [0, 0] and list(s[5]) == [-2.5, 2.5]
    lim = np.array([-1, 1, -0.25, 0.5, -2, 2], np.float32)
    s = oracle_lib.motion(OMNI, lim, 0.1, _state(1), np.array([[0.5, 7.0, 0.0]], np.float32))
    assert s[4, 0] == 0.5 and abs(s[1, 0] - 0.05) < 1e-7


def test_heading_wraps_to_minus_pi_pi(oracle_lib):
    s = oracle_lib.motion(DIFF, LIM_D, 0.1, _state(1, 0, 0, 3.1), np.array([[0.0, 2.0]], np.float32))
    assert -np.pi <= s[2, 0] < np.pi and abs(s[2, 0] - (3.1 + 0.2 - 2 * np.pi)) < 1e-6
    assert s[6, 0] == 0 and s[7, 0] == 0


def test_goal_obs(oracle_lib):
    g = oracle_lib.goal_obs([1.0], [1.0], [np.pi / 2], [1.0], [4.0])
    assert abs(g[0, 0] - 3.0) < 1e-6 and abs(g[1, 0]) < 1e-6          # goal dead ahead
    g = oracle_lib.goal_obs([0.0], [0.0], [0.0], [-3.0], [-4.0])
    assert abs(g[0, 0] - 5.0) < 1e-6 and abs(g[1, 0] - np.arctan2(-4, -3)) < 1e-6
    g = oracle_lib.goal_obs([0.0], [0.0], [3.0], [-1.0], [-0.5])        # wraps into [-pi, pi)
    assert -np.pi <= g[1, 0] < np.pi
    assert abs(g[1, 0] - (np.arctan2(-0.5, -1.0) - 3.0 + 2 * np.pi)) < 1e-6


def test_reward_eq1_golden(oracle_lib):
    path = os.path.join(os.path.dirname(__file__), "golden", "eq1_reward.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    for c, reached, d0, d1, want in rows:
        d_prev = np.array([float(d0)], np.float32)
        ep = np.zeros(1, np.int32)
        tol = 0.3 if int(reached) == 0 else 0.3
        r, done = oracle_lib.reward_done([float(d1)], [int(c)], None, d_prev, ep, goal_tol=tol)
        assert abs(r[0] - float(want)) < 1e-6, (c, reached, d0, d1)
        assert done[0] == (int(c) or int(reached))
        assert d_prev[0] == np.float32(float(d1)) and ep[0] == 1


def test_done_sources(oracle_lib):
    d_prev = np.full(4, 5.0, np.float32)
    ep = np.array([0, 8, 9, 0], np.int32)
    r, done = oracle_lib.reward_done(np.full(4, 4.0, np.float32), np.zeros(4, np.uint8),
                                     np.array([0, 0, 0, 1], np.uint8), d_prev, ep, max_episode_steps=10)
    assert list(done) == [0, 0, 1, 1] and np.allclose(r, 2.0)
    assert list(ep) == [1, 9, 10, 1]


def test_acceleration_limits_ramp_and_no_limit(oracle_lib):
    # reading G2 (U holds velocity AND acceleration limits): the clipped command is limited to the
    # previous applied velocity +- a_max dt.  From rest with a constant command the velocity is the ramp
    # min(k a dt, v*); deceleration is symmetric; +inf reproduces the unlimited update bit for bit.
    lim = np.array([-0.5, 1.5, -1, 1, -2.5, 2.5], np.float32)
    dt = np.float32(0.1)
    for drive, act in ((0, [1.2, -2.0]), (1, [1.2, -0.7, 2.0])):
        acc = np.array([2.0, 1.0, 4.0], np.float32)
        st = np.zeros((8, 1), np.float32)
        a = np.array([act], np.float32)
        for k in range(1, 12):
            st = oracle_lib.motion(drive, lim, dt, st, a, acc=acc)
            tgt = [act[0], 0.0 if drive == 0 else act[1], act[-1]]
            for p, (v_star, amax) in enumerate(zip(tgt, acc)):
                expect = np.sign(v_star) * min(k * amax * 0.1, abs(v_star))
                assert abs(st[3 + p, 0] - expect) < 2e-6, (drive, k, p)
        # brake: command zero, every component approaches 0 by at most a dt per step and never overshoots
        z = np.zeros_like(a)
        prev = st.copy()
        for k in range(20):
            st = oracle_lib.motion(drive, lim, dt, st, z, acc=acc)
            assert np.all(np.abs(st[3:6, 0]) <= np.abs(prev[3:6, 0]) + 1e-7)
            assert np.all(np.abs(st[3:6, 0] - prev[3:6, 0]) <= acc * 0.1 + 1e-6)
            prev = st.copy()
        assert np.all(st[3:6, 0] == 0.0)
        # +inf = no limit, bit for bit
        rng = np.random.default_rng(0)
        s0 = rng.uniform(-1, 1, (8, 50)).astype(np.float32)
        aa = rng.uniform(-3, 3, (50, len(act))).astype(np.float32)
        inf = np.full(3, np.inf, np.float32)
        assert np.array_equal(oracle_lib.motion(drive, lim, dt, s0, aa, acc=inf), oracle_lib.motion(drive, lim, dt, s0, aa))
