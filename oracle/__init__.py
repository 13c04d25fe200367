"""CPU oracle for the FlashNav simulator step -- TEST INFRASTRUCTURE, not the product.

Thin ctypes/NumPy binding over `fn_oracle.c` (plain fp64 C written from PAPER.md).  Only tests/,
bench.py's cpu_baseline / --impl reference legs and __graft_entry__.smoke() may import this package.
It imports nothing from `paper_2606_15846_b200` (the CUDA path) and that package never imports this.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "fn_oracle.c")
_LIB = os.path.join(_DIR, "libfnoracle.so")
_lib = None

EPS_CELL = 1e-5     # near-tie margin in cell units (BASELINE.json north_star)


def build(force: bool = False) -> str:
    """Compile fn_oracle.c with gcc (no FMA contraction: the fp32 reset arithmetic is single-rounded)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.fno_splitmix64.restype = C.c_uint64
        _lib.fno_splitmix64.argtypes = [C.c_uint64, C.c_uint64]
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f32(a):
    return np.ascontiguousarray(a, np.float32)


def _u8(a):
    return np.ascontiguousarray(a, np.uint8)


def splitmix64(sigma: int, c: int) -> int:
    return int(lib().fno_splitmix64(C.c_uint64(sigma), C.c_uint64(c)))


def motion(drive, lim, dt, states, actions, acc=None):
    """acc = None or [3] = maximum accelerations (a_x, a_y, a_w); inf = unlimited (reading G2)."""
    states, actions, lim = _f32(states), _f32(actions), _f32(lim)
    acc = None if acc is None else _f32(acc)
    n = states.shape[1]
    out = np.empty_like(states)
    lib().fno_motion_acc(C.c_int(drive), _p(lim, C.c_float), _p(acc, C.c_float), C.c_float(dt), C.c_int(n),
                         _p(states, C.c_float), _p(actions, C.c_float), _p(out, C.c_float))
    return out


def goal_obs(x, y, psi, gx, gy):
    x, y, psi, gx, gy = map(_f32, (x, y, psi, gx, gy))
    n = x.shape[0]
    out = np.empty((2, n), np.float32)
    lib().fno_goal_obs(C.c_int(n), *[_p(a, C.c_float) for a in (x, y, psi, gx, gy)],
                       _p(out[0], C.c_float), _p(out[1], C.c_float))
    return out


def reward_done(d_new, collision, forced, d_prev, ep_step, goal_tol=0.3, max_episode_steps=0,
                r_success=10.0, r_collision=-10.0, c_progress=2.0):
    """Updates d_prev (float32) and ep_step (int32) in place; returns reward, done."""
    d_new, collision = _f32(d_new), _u8(collision)
    forced = None if forced is None else _u8(forced)
    assert d_prev.dtype == np.float32 and ep_step.dtype == np.int32
    n = d_new.shape[0]
    reward = np.empty(n, np.float32)
    done = np.empty(n, np.uint8)
    lib().fno_reward_done(C.c_int(n), _p(d_new, C.c_float), _p(collision, C.c_uint8),
                          _p(forced, C.c_uint8), C.c_float(goal_tol), C.c_int(max_episode_steps),
                          C.c_float(r_success), C.c_float(r_collision), C.c_float(c_progress),
                          _p(d_prev, C.c_float), _p(ep_step, C.c_int32), _p(reward, C.c_float),
                          _p(done, C.c_uint8))
    return reward, done


def collision(occ, res, footprint, x, y, psi, eps=EPS_CELL, components=None):
    occ, fp = _u8(occ), _f32(footprint)
    x, y, psi = map(_f32, (x, y, psi))
    H, W = occ.shape
    n = x.shape[0]
    flag = np.empty(n, np.uint8)
    amb = np.empty(n, np.uint8)
    with _components(components):
        lib().fno_collision(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res),
                            C.c_int(fp.shape[0]), _p(fp, C.c_float), C.c_int(n), _p(x, C.c_float),
                            _p(y, C.c_float), _p(psi, C.c_float), C.c_double(eps),
                            _p(flag, C.c_uint8), _p(amb, C.c_uint8))
    return flag, amb


def collision_sampled(occ, res, footprint, h, x, y, psi):
    occ, fp = _u8(occ), _f32(footprint)
    x, y, psi = map(_f32, (x, y, psi))
    H, W = occ.shape
    n = x.shape[0]
    flag = np.empty(n, np.uint8)
    lib().fno_collision_sampled(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res),
                                C.c_int(fp.shape[0]), _p(fp, C.c_float), C.c_double(h), C.c_int(n),
                                _p(x, C.c_float), _p(y, C.c_float), _p(psi, C.c_float),
                                _p(flag, C.c_uint8))
    return flag


def ranges(occ, res, angles, max_range, x, y, psi, eps=EPS_CELL, sensor=None, want_visits=False):
    """Returns ranges [n,B] f32, hit [n,B] i32, amb [n,B] u8 (, visits [n,B] i32)."""
    occ, angles = _u8(occ), _f32(angles)
    x, y, psi = map(_f32, (x, y, psi))
    sensor = None if sensor is None else _f32(sensor)
    H, W = occ.shape
    n, B = x.shape[0], angles.shape[0]
    r = np.empty((n, B), np.float32)
    hit = np.empty((n, B), np.int32)
    amb = np.empty((n, B), np.uint8)
    vis = np.empty((n, B), np.int32) if want_visits else None
    lib().fno_ranges(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res), C.c_int(B),
                     _p(angles, C.c_float), C.c_float(max_range), _p(sensor, C.c_float), C.c_int(n),
                     _p(x, C.c_float), _p(y, C.c_float), _p(psi, C.c_float), C.c_double(eps),
                     _p(r, C.c_float), _p(hit, C.c_int32), _p(amb, C.c_uint8), _p(vis, C.c_int32))
    return (r, hit, amb, vis) if want_visits else (r, hit, amb)


def ranges_multi(occ, res, sensors, x, y, psi, eps=EPS_CELL):
    """A robot with several range sensors.  sensors = [(angles [B_k], max_range, (s_x, s_y, s_psi)), ...];
    returns ranges [n, sum B_k] f32, hit i32, amb u8, the sensors' beams one after the other."""
    occ = _u8(occ)
    x, y, psi = map(_f32, (x, y, psi))
    H, W = occ.shape
    n = x.shape[0]
    Bk = np.array([len(a) for a, _, _ in sensors], np.int32)
    ang = _f32(np.concatenate([np.asarray(a, np.float32) for a, _, _ in sensors]))
    rmax = _f32(np.array([m for _, m, _ in sensors], np.float32))
    plc = _f32(np.array([p for _, _, p in sensors], np.float32).reshape(-1, 3))
    B = int(Bk.sum())
    r = np.empty((n, B), np.float32)
    hit = np.empty((n, B), np.int32)
    amb = np.empty((n, B), np.uint8)
    lib().fno_ranges_multi(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res), C.c_int(len(sensors)), _p(Bk, C.c_int32),
                           _p(ang, C.c_float), _p(rmax, C.c_float), _p(plc, C.c_float), C.c_int(n), _p(x, C.c_float),
                           _p(y, C.c_float), _p(psi, C.c_float), C.c_double(eps), _p(r, C.c_float), _p(hit, C.c_int32),
                           _p(amb, C.c_uint8))
    return r, hit, amb


def ranges_fixed_step(occ, res, angles, max_range, delta, x, y, psi):
    occ, angles = _u8(occ), _f32(angles)
    x, y, psi = map(_f32, (x, y, psi))
    H, W = occ.shape
    n, B = x.shape[0], angles.shape[0]
    r = np.empty((n, B), np.float32)
    lib().fno_ranges_fixed_step(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res),
                                C.c_int(B), _p(angles, C.c_float), C.c_float(max_range),
                                C.c_double(delta), C.c_int(n), _p(x, C.c_float), _p(y, C.c_float),
                                _p(psi, C.c_float), _p(r, C.c_float))
    return r


def reset(occ, res, footprint, regions, goal_dist_min, goal_dist_max, mask, seeds, states, d_prev,
          ep_step, eps=EPS_CELL, components=None):
    """In place on states [8,n] f32, d_prev f32, ep_step i32 for masked envs. Returns amb, failed."""
    occ, fp, mask = _u8(occ), _f32(footprint), _u8(mask)
    seeds = np.ascontiguousarray(seeds, np.uint64)
    assert states.dtype == np.float32 and states.flags.c_contiguous
    assert d_prev.dtype == np.float32 and ep_step.dtype == np.int32
    H, W = occ.shape
    n = states.shape[1]
    nreg = 0 if regions is None else int(regions.shape[0])
    reg = None if regions is None else np.ascontiguousarray(regions, np.int32)
    amb = np.empty(n, np.uint8)
    failed = np.empty(n, np.uint8)
    with _components(components):
        lib().fno_reset(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(res), C.c_int(fp.shape[0]),
                        _p(fp, C.c_float), C.c_int(nreg), _p(reg, C.c_int32), C.c_float(goal_dist_min),
                        C.c_float(goal_dist_max), C.c_int(n), _p(mask, C.c_uint8), _p(seeds, C.c_uint64),
                        C.c_double(eps), _p(states, C.c_float), _p(d_prev, C.c_float),
                        _p(ep_step, C.c_int32), _p(amb, C.c_uint8), _p(failed, C.c_uint8))
    return amb, failed


def done_code(done, collision, d, goal_tol):
    """The ring row's done field (G18): 0 running, 1 terminated (collision or goal), 2 truncated (limit / forced)."""
    done, collision, d = _u8(done), _u8(collision), _f32(d)
    f = lib().fno_done_code
    f.restype = C.c_uint8
    f.argtypes = [C.c_uint8, C.c_uint8, C.c_float, C.c_float]
    return np.array([f(int(a), int(b), float(c), float(goal_tol)) for a, b, c in zip(done, collision, d)], np.uint8)


def ring_append(ring, capacity, head, obs_ranges, obs_goal, obs_vel, actions, reward, done):
    """done: the codes of done_code (stored as they are)."""
    obs_ranges, obs_goal, obs_vel, actions, reward = map(_f32, (obs_ranges, obs_goal, obs_vel,
                                                                actions, reward))
    done = _u8(done)
    n, B = obs_ranges.shape
    A = actions.shape[1]
    assert ring.dtype == np.float32 and ring.flags.c_contiguous
    lib().fno_ring_append(_p(ring, C.c_float), C.c_uint64(capacity), C.c_uint64(head), C.c_int(n),
                          C.c_int(B), C.c_int(A), _p(obs_ranges, C.c_float), _p(obs_goal, C.c_float),
                          _p(obs_vel, C.c_float), _p(actions, C.c_float), _p(reward, C.c_float),
                          _p(done, C.c_uint8))


def eval_update(collision, d_new, goal_tol, ep_step_after, step_limit, reward, outcome, steps, ret):
    """Evaluation completion masks; outcome u8 / steps i32 / ret f32 are updated in place."""
    collision, d_new, reward = _u8(collision), _f32(d_new), _f32(reward)
    ep = np.ascontiguousarray(ep_step_after, np.int32)
    assert outcome.dtype == np.uint8 and steps.dtype == np.int32 and ret.dtype == np.float32
    lib().fno_eval_update(C.c_int(outcome.shape[0]), _p(collision, C.c_uint8), _p(d_new, C.c_float), C.c_float(goal_tol),
                          _p(ep, C.c_int32), C.c_int(step_limit), _p(reward, C.c_float), _p(outcome, C.c_uint8),
                          _p(steps, C.c_int32), _p(ret, C.c_float))


class _components:
    """A union of polygons: the vertex lists are concatenated in `footprint`, `sizes` gives the
    vertex count of each polygon (None = one polygon).  The C side keeps the sizes in a file-scope variable; every
    wrapper sets it for exactly one call through this context and puts it back to "one polygon" afterwards, so that
    no call can inherit an earlier footprint's components."""

    def __init__(self, sizes):
        self.sizes = None if sizes is None else np.ascontiguousarray(sizes, np.int32)

    def __enter__(self):
        if self.sizes is not None and len(self.sizes) > 1:
            lib().fno_set_footprint_components(C.c_int(len(self.sizes)), _p(self.sizes, C.c_int32))
        else:
            lib().fno_set_footprint_components(C.c_int(0), None)

    def __exit__(self, *exc):
        lib().fno_set_footprint_components(C.c_int(0), None)
        return False


def sample_slot(seed: int, i: int, filled: int) -> int:
    f = lib().fno_sample_slot
    f.restype = C.c_uint64
    f.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
    return int(f(seed, i, filled))


def ring_valid(capacity: int, total: int, n_envs: int) -> int:
    """Completed transitions still in the ring and outside the pending window (reading G22)."""
    lib().fno_ring_valid.restype = C.c_uint64
    return int(lib().fno_ring_valid(C.c_uint64(capacity), C.c_uint64(total), C.c_int(n_envs)))


class TerminalStore:
    """The terminal-observation ring of fno_terminal_save: entries [t_cap, B+5] f32, the index of each
    ring row's entry, the global row id of each entry, the number of entries ever written."""

    def __init__(self, capacity, t_cap, B):
        self.t_cap = int(t_cap)
        self.term = np.zeros((self.t_cap, B + 5), np.float32)
        self.idx = np.full(int(capacity), -1, np.int32)
        self.id = np.full(self.t_cap, np.iinfo(np.uint64).max, np.uint64)
        self.start = np.zeros(self.t_cap, np.uint64)
        self.head = C.c_uint64(0)
        self.batch_start = 0

    def step_ended(self):
        """Call after every step that appended rows: the resets that follow form one batch."""
        self.batch_start = int(self.head.value)


def terminal_save(ring, capacity, total, n_envs, B, A, env_list, store: TerminalStore):
    """Before the listed envs are reset: keep the observation the last step left in their pending rows, for every one
    whose last completed row has a done code != 0 (and is not kept yet)."""
    assert ring.dtype == np.float32 and ring.flags.c_contiguous
    lst = np.ascontiguousarray(env_list, np.int32)
    lib().fno_terminal_save(_p(ring, C.c_float), C.c_uint64(capacity), C.c_uint64(total), C.c_int(n_envs), C.c_int(B),
                            C.c_int(A), _p(lst, C.c_int32), C.c_int(lst.size), _p(store.term, C.c_float),
                            C.c_uint64(store.t_cap), _p(store.idx, C.c_int32), _p(store.id, C.c_uint64),
                            _p(store.start, C.c_uint64), C.byref(store.head), C.c_uint64(store.batch_start))


def ring_sample(ring, capacity, total, n_envs, B, A, seed, n_samples, want_next=True, store: TerminalStore | None = None):
    """Uniform replay sampling after `total` appended rows.  ring [capacity, B+5+A+2] f32 -> rows
    [n,row], next_obs [n,B+5], slots [n].  store: terminal observations (next observation of done rows; the sampled
    rows' done field becomes 3 for truncated rows whose observation is gone)."""
    assert ring.dtype == np.float32 and ring.flags.c_contiguous
    row = B + 5 + A + 2
    rows = np.empty((n_samples, row), np.float32)
    nxt = np.empty((n_samples, B + 5), np.float32) if want_next else None
    slots = np.empty(n_samples, np.int64)
    lib().fno_ring_sample(_p(ring, C.c_float), C.c_uint64(capacity), C.c_uint64(total), C.c_int(n_envs), C.c_int(B),
                          C.c_int(A), C.c_uint64(seed), C.c_int(n_samples), _p(rows, C.c_float),
                          _p(nxt, C.c_float), _p(slots, C.c_int64),
                          None if store is None else _p(store.term, C.c_float),
                          C.c_uint64(0 if store is None else store.t_cap),
                          None if store is None else _p(store.idx, C.c_int32),
                          None if store is None else _p(store.id, C.c_uint64),
                          None if store is None else _p(store.start, C.c_uint64),
                          C.c_uint64(0 if store is None else store.head.value))
    return rows, nxt, slots


def footprint_distance(footprint, px, py, components=None) -> float:
    """Eq. (3) for one body-frame point: distance to the polygon, 0 inside."""
    fp = _f32(footprint)
    f = lib().fno_footprint_distance
    f.restype = C.c_double
    f.argtypes = [C.c_int, C.POINTER(C.c_float), C.c_double, C.c_double]
    with _components(components):
        return float(f(fp.shape[0], _p(fp, C.c_float), float(px), float(py)))


def clearance_features(footprint, angles, max_range, n_sectors, ranges_, sensor=None, want_delta=False, components=None):
    """Eq. (3) + sector min-pooling.  ranges_ [n,B] f32 -> z [n,n_sectors] f32
    (, delta [n,B] f32)."""
    fp, ang, rg = _f32(footprint), _f32(angles), _f32(ranges_)
    n, B = rg.shape
    z = np.empty((n, n_sectors), np.float32)
    delta = np.empty((n, B), np.float32) if want_delta else None
    sen = None if sensor is None else _f32(sensor)
    with _components(components):
        lib().fno_clearance_features(C.c_int(fp.shape[0]), _p(fp, C.c_float), C.c_int(B), _p(ang, C.c_float),
                                     _p(sen, C.c_float), C.c_float(max_range), C.c_int(n_sectors), C.c_int(n),
                                     _p(rg, C.c_float), _p(delta, C.c_float), _p(z, C.c_float))
    return (z, delta) if want_delta else z


def step(wl, states, actions, forced, d_prev, ep_step, want_hit=True):
    """One whole vector step on a harness Workload-like object (fields only; no harness import).
    states [8,n] f32 updated in place.  Returns dict(ranges, hit, collision, goal_obs, reward, done)."""
    occ, fp, ang, lim = _u8(wl.occ), _f32(wl.footprint), _f32(wl.beam_angles), _f32(wl.vel_limits)
    actions = _f32(actions)
    forced = None if forced is None else _u8(forced)
    assert states.dtype == np.float32 and states.flags.c_contiguous
    H, W = occ.shape
    n, B = states.shape[1], ang.shape[0]
    r = np.empty((n, B), np.float32)
    hit = np.empty((n, B), np.int32) if want_hit else None
    col = np.empty(n, np.uint8)
    gobs = np.empty((2, n), np.float32)
    rew = np.empty(n, np.float32)
    done = np.empty(n, np.uint8)
    with _components(getattr(wl, "components", None)):
      lib().fno_step(_p(occ, C.c_uint8), C.c_int(H), C.c_int(W), C.c_float(wl.resolution),
                   C.c_int(fp.shape[0]), _p(fp, C.c_float), C.c_int(B), _p(ang, C.c_float),
                   C.c_float(wl.max_range), C.c_int(wl.drive), _p(lim, C.c_float), C.c_float(wl.dt),
                   C.c_float(wl.goal_tol), C.c_int(wl.max_episode_steps), C.c_float(wl.r_success),
                   C.c_float(wl.r_collision), C.c_float(wl.c_progress), C.c_int(n),
                   _p(states, C.c_float), _p(actions, C.c_float), _p(forced, C.c_uint8),
                   _p(d_prev, C.c_float), _p(ep_step, C.c_int32), _p(r, C.c_float),
                   _p(hit, C.c_int32), _p(col, C.c_uint8), _p(gobs, C.c_float), _p(rew, C.c_float),
                   _p(done, C.c_uint8))
    return dict(ranges=r, hit=hit, collision=col, goal_obs=gobs, reward=rew, done=done)
