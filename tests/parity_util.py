"""Teacher-forced parity of the CUDA path (through the C ABI) against the CPU oracle.

Per step, the oracle is given the GPU's fp32 input state, action, forced mask and seeds; motion output
is compared at 1e-5; sensing, collision, goal obs and reward are evaluated by the oracle AT THE GPU's
fp32 post-motion pose (SURVEY.md 8(c) "Teacher forcing").  Tolerances are BASELINE.json north_star's:
collision flags / hit cells / done flags / reset states bit-exact outside counted near-ties (oracle
margin 1e-5 cell), ranges abs 1e-4 m, states 1e-5 relative (floor 1), psi modulo 2 pi.
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_2606_15846_b200 as fn
from harness import workloads as W

TOL_RANGE = 1e-4
TOL_STATE = 1e-5


def make_sim(wl, n=None):
    n = wl.n_envs if n is None else n
    m = fn.Map(wl.occ, float(wl.resolution))
    if wl.regions is not None:
        m.set_regions(wl.regions)
    r = fn.Robot(wl.footprint, wl.beam_angles, float(wl.max_range), wl.drive, wl.vel_limits,
                 components=getattr(wl, "components", None))
    if getattr(wl, "acc_limits", None) is not None:
        r.set_acc_limits(wl.acc_limits)
    if getattr(wl, "sensor", None) is not None:                     # sensor placement S (reading G8)
        r.set_sensor(*[float(v) for v in wl.sensor])
    s = fn.Sim(m, r, n, goal_tol=float(wl.goal_tol), max_episode_steps=wl.max_episode_steps,
               goal_dist_min=float(wl.goal_dist_min), goal_dist_max=float(wl.goal_dist_max),
               r_success=float(wl.r_success), r_collision=float(wl.r_collision), c_progress=float(wl.c_progress))
    return m, r, s


class Buffers:
    def __init__(self, n, B, A, dev="cuda"):
        self.states = torch.zeros(8, n, dtype=torch.float32, device=dev)
        self.mask = torch.zeros(n, dtype=torch.uint8, device=dev)
        self.ranges = torch.zeros(n, B, dtype=torch.float32, device=dev)
        self.col = torch.zeros(n, dtype=torch.uint8, device=dev)
        self.gobs = torch.zeros(2, n, dtype=torch.float32, device=dev)
        self.hit = torch.zeros(n, B, dtype=torch.int32, device=dev)
        self.reward = torch.zeros(n, dtype=torch.float32, device=dev)


def ang_diff(a, b):
    d = (a.astype(np.float64) - b.astype(np.float64) + np.pi) % (2 * np.pi) - np.pi
    return np.abs(d)


def close_state(got, ref):
    return np.abs(got.astype(np.float64) - ref.astype(np.float64)) <= TOL_STATE * np.maximum(1.0, np.abs(ref.astype(np.float64)))


class Report:
    def __init__(self):
        self.c = {}

    def add(self, k, v=1):
        self.c[k] = self.c.get(k, 0) + int(v)

    def __repr__(self):
        return "parity " + " ".join(f"{k}={v}" for k, v in sorted(self.c.items()))


def check_observation(wl, rep, x, y, psi, g_ranges, g_hit, env_idx=None, tag="obs"):
    """ranges / hit cells of the listed envs at fp32 poses (x, y, psi) vs the oracle."""
    r, hit, amb = oracle.ranges(wl.occ, wl.resolution, wl.beam_angles, wl.max_range, x, y, psi,
                                sensor=getattr(wl, "sensor", None))
    ok = amb == 0
    rep.add("beams", ok.size)
    rep.add("beams_ambiguous", (~ok).sum())
    bad_hit = ok & (g_hit != hit) if g_hit is not None else np.zeros_like(ok)    # (the production kernel gives no hit cells)
    bad_r = ok & (np.abs(g_ranges.astype(np.float64) - r.astype(np.float64)) > TOL_RANGE)
    if bad_hit.any() or bad_r.any():
        e, b = np.nonzero(bad_hit | bad_r)
        k = 0
        raise AssertionError(
            f"{tag}: {bad_hit.sum()} hit-cell and {bad_r.sum()} range mismatches outside near-ties; first: env "
            f"{(env_idx[e[k]] if env_idx is not None else e[k])} beam {b[k]} pose=({x[e[k]]!r},{y[e[k]]!r},{psi[e[k]]!r}) "
            f"gpu r={g_ranges[e[k], b[k]]!r} hit={g_hit[e[k], b[k]] if g_hit is not None else None} oracle r={r[e[k], b[k]]!r} hit={hit[e[k], b[k]]}")
    # ambiguous beams must still be sane
    assert np.all(np.isfinite(g_ranges)) and g_ranges.min() >= 0 and g_ranges.max() <= float(wl.max_range) + 1e-6


def run_parity(wl, steps, n=None, subset=None, seed=0, forced=None, check_every=1, full_every=None):
    """Free-running GPU trajectory, teacher-forced oracle check each `check_every` steps.
    subset: number of envs (a fixed random sample) whose beams are checked; None = all.
    full_every: the beams of ALL envs are checked on steps 0, 1, 2 and every full_every-th one."""
    n = wl.n_envs if n is None else n
    wl.n_envs = n
    B, A = wl.n_beams, wl.action_dim
    comp = getattr(wl, "components", None)                              # a union of polygons, or None
    m, r, s = make_sim(wl, n)
    buf = Buffers(n, B, A)
    s.bind_aux(buf.hit, buf.reward)
    actions = torch.from_numpy(W.action_tape(wl, steps, seed)).cuda()
    seeds_np = W.seed_tape(wl, steps + 1, seed)
    forced_np = W.forced_reset_tape(wl, steps, seed) if forced is None else forced
    rng = np.random.default_rng(seed + 99)
    sel = np.arange(n) if subset is None or subset >= n else np.sort(rng.choice(n, subset, replace=False))
    rep = Report()

    def do_reset(mask_np, seeds_row, tag):
        pre = buf.states.cpu().numpy()
        d_prev0, ep0 = s.episode_state()
        seeds_t = torch.from_numpy(seeds_row.view(np.int64)).cuda()
        mask_t = torch.from_numpy(mask_np).cuda()
        keep_r = buf.ranges.clone()
        s.reset(buf.states, mask_t, seeds_t, buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        post = buf.states.cpu().numpy()
        ref = pre.copy()
        d_prev, ep = d_prev0.copy(), ep0.copy()
        amb, failed = oracle.reset(wl.occ, wl.resolution, wl.footprint, wl.regions, wl.goal_dist_min,
                                   wl.goal_dist_max, mask_np, seeds_row, ref, d_prev, ep, components=comp)
        okm = (mask_np != 0) & (amb == 0)
        rep.add("resets", (mask_np != 0).sum())
        rep.add("resets_ambiguous", ((mask_np != 0) & (amb != 0)).sum())
        rep.add("reset_failures", failed.sum())
        assert np.array_equal(post[:, mask_np == 0], pre[:, mask_np == 0]), f"{tag}: reset touched unmasked envs"
        if not np.array_equal(post[:, okm], ref[:, okm]):
            e = np.nonzero(okm & np.any(post != ref, axis=0))[0][0]
            raise AssertionError(f"{tag}: reset state differs for env {e}: gpu {post[:, e]} oracle {ref[:, e]} seed {seeds_row[e]}")
        gd, ge = s.episode_state()
        assert np.array_equal(ge[okm], ep[okm]) and np.all(ge[mask_np == 0] == ep0[mask_np == 0])
        assert np.allclose(gd[okm], d_prev[okm], atol=1e-5) and np.array_equal(gd[mask_np == 0], d_prev0[mask_np == 0])
        # selective recompute: unmasked rows untouched, masked rows = observation at the new state
        rg = buf.ranges.cpu().numpy()
        assert np.array_equal(rg[mask_np == 0], keep_r.cpu().numpy()[mask_np == 0]), f"{tag}: recompute touched other rows"
        idx = np.nonzero(okm)[0]
        if subset is not None and idx.size > subset:
            idx = idx[:subset]
        if idx.size:
            check_observation(wl, rep, post[0, idx], post[1, idx], post[2, idx], rg[idx], buf.hit.cpu().numpy()[idx],
                              idx, tag + "/recompute")
            g = buf.gobs.cpu().numpy()
            og = oracle.goal_obs(post[0, idx], post[1, idx], post[2, idx], post[6, idx], post[7, idx])
            assert np.all(close_state(g[0, idx], og[0])) and np.all(ang_diff(g[1, idx], og[1]) <= 1e-5)

    do_reset(np.ones(n, np.uint8), seeds_np[0], "initial reset")

    n_done = 0
    for t in range(steps):
        check = (t % check_every == 0) or t < 3
        pre = buf.states.cpu().numpy() if check else None
        d_prev0, ep0 = s.episode_state() if check else (None, None)
        buf.mask.copy_(torch.from_numpy(forced_np[t]))
        s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        torch.cuda.synchronize()
        done = buf.mask.cpu().numpy()
        n_done += int(done.sum())
        if check:
            post = buf.states.cpu().numpy()
            ref = oracle.motion(wl.drive, wl.vel_limits, wl.dt, pre, actions[t].cpu().numpy(),
                                acc=getattr(wl, "acc_limits", None))
            if getattr(wl, "acc_limits", None) is not None:      # the slewed command is fp32 arithmetic: bit-exact
                assert np.array_equal(post[3:6], ref[3:6]), f"step {t}: applied velocities under acceleration limits"
            for p in (0, 1, 3, 4, 5, 6, 7):
                assert np.all(close_state(post[p], ref[p])), f"step {t}: state plane {p} off by {np.abs(post[p] - ref[p]).max()}"
            assert np.all(ang_diff(post[2], ref[2]) <= TOL_STATE * np.maximum(1, np.abs(ref[2]))), f"step {t}: psi"
            x, y, psi = post[0], post[1], post[2]
            flag, camb = oracle.collision(wl.occ, wl.resolution, wl.footprint, x, y, psi, components=comp)
            gcol = buf.col.cpu().numpy()
            okc = camb == 0
            rep.add("collision_checks", n)
            rep.add("collision_ambiguous", (~okc).sum())
            rep.add("collisions", int(flag.sum()))
            if not np.array_equal(gcol[okc], flag[okc]):
                e = np.nonzero(okc & (gcol != flag))[0][0]
                raise AssertionError(f"step {t}: collision flag differs for env {e}: gpu {gcol[e]} oracle {flag[e]} pose {x[e]!r},{y[e]!r},{psi[e]!r}")
            og = oracle.goal_obs(x, y, psi, post[6], post[7])
            g = buf.gobs.cpu().numpy()
            assert np.all(close_state(g[0], og[0])), f"step {t}: goal distance"
            far = og[0] > 1e-3
            assert np.all(ang_diff(g[1], og[1])[far] <= 1e-5), f"step {t}: goal direction"
            # reward / done from the ORACLE's own d and collision flag.  Near-tie class of the goal threshold: the
            # decision d < goal_tol is taken on an fp32 d that may differ from the oracle's by 1e-5 (tolerance above),
            # so envs with |d - goal_tol| < 1e-5 (and ambiguous collision flags) are excluded and counted.
            d_prev, ep = d_prev0.copy(), ep0.copy()
            tie = (np.abs(og[0].astype(np.float64) - float(wl.goal_tol)) < 1e-5) | ~okc
            rep.add("done_checks", n)
            rep.add("done_ambiguous", tie.sum())
            rew, odone = oracle.reward_done(og[0], flag, forced_np[t], d_prev, ep, float(wl.goal_tol), wl.max_episode_steps,
                                            float(wl.r_success), float(wl.r_collision), float(wl.c_progress))
            assert np.array_equal(done[~tie], odone[~tie]), f"step {t}: done flags"
            assert np.allclose(buf.reward.cpu().numpy()[~tie], rew[~tie], atol=1e-4), f"step {t}: reward"
            gd, ge = s.episode_state()
            assert np.array_equal(ge[~tie], ep[~tie]) and np.allclose(gd[~tie], d_prev[~tie], atol=1e-5)
            # (and, on the GPU's own bits, everything is exact: same d, same flags => same decisions)
            d_prev2, ep2 = d_prev0.copy(), ep0.copy()
            rew2, odone2 = oracle.reward_done(g[0], gcol, forced_np[t], d_prev2, ep2, float(wl.goal_tol), wl.max_episode_steps,
                                              float(wl.r_success), float(wl.r_collision), float(wl.c_progress))
            assert np.array_equal(done, odone2) and np.array_equal(ge, ep2) and np.array_equal(gd, d_prev2), f"step {t}: done / episode state"
            selt = np.arange(n) if full_every is not None and (t < 3 or t % full_every == 0) else sel
            check_observation(wl, rep, x[selt], y[selt], psi[selt], buf.ranges.cpu().numpy()[selt], buf.hit.cpu().numpy()[selt],
                              selt, f"step {t}")
            # The production (non-instrumented) beam kernel must give bit-identical ranges -- on the same sensing
            # poses.  fn_observe_all builds the poses from the state planes (a fresh sincos of the fp32 heading),
            # fn_step keeps cos / sin of the heading across steps (rotation by the step's angle, exact sincos every
            # 32nd episode step: ~2e-16 per step), so the two pose sets differ in the last bits and, about once in
            # 10^9 beams, so does the last bit of a range (found by the 1000-step run).  Hence: instrumented and
            # production kernel both through fn_observe_all = bit-equal; maintained rows against them = equal up to
            # one fp32 ulp on at most 1e-5 of the beams (counted).
            hit2 = torch.empty_like(buf.hit)
            s.bind_aux(hit2, buf.reward)
            inst = torch.empty_like(buf.ranges)
            s.observe_all(buf.states, inst)
            s.bind_aux(None, buf.reward)
            fast = torch.empty_like(buf.ranges)
            s.observe_all(buf.states, fast)
            torch.cuda.synchronize()
            if not torch.equal(fast, inst):
                bad = (fast != inst).nonzero()[0].tolist()
                raise AssertionError(f"step {t}: fast beam kernel differs from instrumented one at env {bad[0]} beam {bad[1]}: "
                                     f"{fast[bad[0], bad[1]].item()!r} vs {inst[bad[0], bad[1]].item()!r}")
            rep.add("fast_path_checks", n * B)
            assert_rows_equal_up_to_pose_rounding(rep, inst, buf.ranges, f"step {t}: maintained rows vs fn_observe_all")
            # ... and so must the production kernel with the coarse level (where the copies fit one CTA)
            if s.beam_config()["coarse_available"]:
                was = s.beam_config()["coarse"]
                s.set_coarse(not was)
                other = torch.empty_like(buf.ranges)
                s.observe_all(buf.states, other)
                torch.cuda.synchronize()
                s.set_coarse(was)
                if not torch.equal(other, fast):
                    bad = (other != fast).nonzero()[0].tolist()
                    raise AssertionError(f"step {t}: coarse level {'off' if was else 'on'}: beam kernel differs at env {bad[0]} beam {bad[1]}: "
                                         f"{other[bad[0], bad[1]].item()!r} vs {fast[bad[0], bad[1]].item()!r}")
                rep.add("coarse_level_checks", n * B)
            s.bind_aux(buf.hit, buf.reward)
        if done.any():
            if check:
                do_reset(done, seeds_np[t + 1], f"step {t} reset")
            else:
                s.reset(buf.states, buf.mask, torch.from_numpy(seeds_np[t + 1].view(np.int64)).cuda(), buf.ranges, buf.gobs)

    # observation is a pure function of state: the incrementally maintained rows equal a full recompute
    full_r = torch.empty_like(buf.ranges)
    full_g = torch.empty_like(buf.gobs)
    s.observe_all(buf.states, full_r, full_g)
    torch.cuda.synchronize()
    assert_rows_equal_up_to_pose_rounding(rep, full_r, buf.ranges, "observe_all vs incrementally maintained ranges")
    assert torch.equal(full_g, buf.gobs), "observe_all differs from incrementally maintained goal obs"
    rep.add("steps", steps)
    rep.add("done_events", n_done)
    cnt = s.counters()
    rep.add("rays_cast", cnt["rays_cast"])
    assert cnt["oob_window_loads"] == 0, "the instrumented beam kernel read a window outside the packed map"
    assert cnt["reset_failures"] == rep.c.get("reset_failures", 0) or check_every > 1
    s.close(); r.close(); m.close()
    assert_ambiguity_bounds(rep)
    return rep


def run_production_parity(wl, steps, n=None, subset=None, seed=0, full_steps=(0, 1, 2), ring=False):
    """The launch sequence bench.py TIMES, held against the oracle directly: no hit cells bound (so fn_step runs the
    production step kernel, not the instrumented one), the reset seeds announced before every step
    (fn_sim_prepare_reset), fn_reset(mask = NULL) of the step's done list.  Everything the production kernels return
    is compared with the oracle at the usual tolerances -- state planes, collision flags, goal obs, done, reward,
    reset states, and the RANGES (of `subset` envs per step, of all envs on `full_steps`); hit cells are the one thing
    these kernels cannot give.  Asserts that the prepared path served resets where the sim has it."""
    n = wl.n_envs if n is None else n
    wl.n_envs = n
    B, A = wl.n_beams, wl.action_dim
    comp = getattr(wl, "components", None)
    m, r, s = make_sim(wl, n)
    buf = Buffers(n, B, A)
    s.bind_aux(None, buf.reward)                                        # the reward is an output, not an instrument
    ring_t = None
    if ring:
        cap = 3 * n + 5
        ring_t = torch.zeros(cap * s.ring_row_floats(), device="cuda")
        s.ring_attach(ring_t, cap)
    actions = torch.from_numpy(W.action_tape(wl, steps, seed)).cuda()
    seeds_np = W.seed_tape(wl, steps + 1, seed)
    seeds_t = torch.from_numpy(seeds_np.view(np.int64)).cuda()
    forced_np = W.forced_reset_tape(wl, steps, seed)
    rng = np.random.default_rng(seed + 99)
    sel = np.arange(n) if subset is None or subset >= n else np.sort(rng.choice(n, subset, replace=False))
    rep = Report()
    sensor = getattr(wl, "sensor", None)

    def check_reset(mask_np, seeds_row, pre, d_prev0, ep0, keep_r, tag):
        post = buf.states.cpu().numpy()
        ref = pre.copy()
        d_prev, ep = d_prev0.copy(), ep0.copy()
        amb, failed = oracle.reset(wl.occ, wl.resolution, wl.footprint, wl.regions, wl.goal_dist_min,
                                   wl.goal_dist_max, mask_np, seeds_row, ref, d_prev, ep, components=comp)
        okm = (mask_np != 0) & (amb == 0)
        rep.add("resets", (mask_np != 0).sum())
        rep.add("resets_ambiguous", ((mask_np != 0) & (amb != 0)).sum())
        assert np.array_equal(post[:, mask_np == 0], pre[:, mask_np == 0]), f"{tag}: reset touched other envs"
        if not np.array_equal(post[:, okm], ref[:, okm]):
            e = np.nonzero(okm & np.any(post != ref, axis=0))[0][0]
            raise AssertionError(f"{tag}: reset state differs for env {e}: gpu {post[:, e]} oracle {ref[:, e]}")
        gd, ge = s.episode_state()
        assert np.array_equal(ge[okm], ep[okm]) and np.allclose(gd[okm], d_prev[okm], atol=1e-5)
        rg = buf.ranges.cpu().numpy()
        assert np.array_equal(rg[mask_np == 0], keep_r[mask_np == 0]), f"{tag}: recompute touched other rows"
        idx = np.nonzero(okm)[0]
        if subset is not None and idx.size > subset:
            idx = idx[:subset]
        if idx.size:
            check_observation(wl, rep, post[0, idx], post[1, idx], post[2, idx], rg[idx], None, idx, tag + "/recompute")
            g = buf.gobs.cpu().numpy()
            og = oracle.goal_obs(post[0, idx], post[1, idx], post[2, idx], post[6, idx], post[7, idx])
            assert np.all(close_state(g[0, idx], og[0])) and np.all(ang_diff(g[1, idx], og[1]) <= 1e-5)

    pre = buf.states.cpu().numpy()
    d0, e0 = s.episode_state()
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds_t[0], buf.ranges, buf.gobs)
    torch.cuda.synchronize()
    check_reset(np.ones(n, np.uint8), seeds_np[0], pre, d0, e0, buf.ranges.cpu().numpy(), "initial reset")

    for t in range(steps):
        pre = buf.states.cpu().numpy()
        d_prev0, ep0 = s.episode_state()
        buf.mask.copy_(torch.from_numpy(forced_np[t]))
        s.prepare_reset(seeds_t[t + 1])                                 # what bench.py does
        s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        torch.cuda.synchronize()
        done = buf.mask.cpu().numpy()
        post = buf.states.cpu().numpy()
        ref = oracle.motion(wl.drive, wl.vel_limits, wl.dt, pre, actions[t].cpu().numpy(), acc=getattr(wl, "acc_limits", None))
        for p in (0, 1, 3, 4, 5, 6, 7):
            assert np.all(close_state(post[p], ref[p])), f"step {t}: state plane {p}"
        assert np.all(ang_diff(post[2], ref[2]) <= TOL_STATE * np.maximum(1, np.abs(ref[2]))), f"step {t}: psi"
        x, y, psi = post[0], post[1], post[2]
        flag, camb = oracle.collision(wl.occ, wl.resolution, wl.footprint, x, y, psi, components=comp)
        gcol = buf.col.cpu().numpy()
        okc = camb == 0
        rep.add("collision_checks", n)
        rep.add("collision_ambiguous", (~okc).sum())
        assert np.array_equal(gcol[okc], flag[okc]), f"step {t}: collision flags"
        og = oracle.goal_obs(x, y, psi, post[6], post[7])
        g = buf.gobs.cpu().numpy()
        assert np.all(close_state(g[0], og[0])), f"step {t}: goal distance"
        assert np.all(ang_diff(g[1], og[1])[og[0] > 1e-3] <= 1e-5), f"step {t}: goal direction"
        d_prev, ep = d_prev0.copy(), ep0.copy()
        tie = (np.abs(og[0].astype(np.float64) - float(wl.goal_tol)) < 1e-5) | ~okc
        rep.add("done_checks", n)
        rep.add("done_ambiguous", tie.sum())
        rew, odone = oracle.reward_done(og[0], flag, forced_np[t], d_prev, ep, float(wl.goal_tol), wl.max_episode_steps,
                                        float(wl.r_success), float(wl.r_collision), float(wl.c_progress))
        assert np.array_equal(done[~tie], odone[~tie]), f"step {t}: done flags"
        assert np.allclose(buf.reward.cpu().numpy()[~tie], rew[~tie], atol=1e-4), f"step {t}: reward"
        selt = np.arange(n) if t in full_steps else sel
        rg = buf.ranges.cpu().numpy()
        check_observation(wl, rep, x[selt], y[selt], psi[selt], rg[selt], None, selt, f"step {t} (production kernel)")
        # the reset of the step's done list, prepared by the step where the sim has that path
        d1, e1 = s.episode_state()
        s.reset(buf.states, None, seeds_t[t + 1], buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        check_reset(done, seeds_np[t + 1], post, d1, e1, rg, f"step {t} reset")
    rep.add("steps", steps)
    cnt = s.counters()
    rep.add("resets_prepared", cnt["resets_prepared"])
    rep.add("rays_cast", cnt["rays_cast"])
    s.close(); r.close(); m.close()
    assert_ambiguity_bounds(rep)
    return rep


def assert_rows_equal_up_to_pose_rounding(rep, a, b, tag):
    """Ranges cast from two pose sets that differ by the rounding of cos / sin of the heading (see run_parity):
    equal, except for one fp32 ulp on at most 1e-5 of the beams."""
    diff = a != b
    k = int(diff.sum().item())
    rep.add("pose_rounding_checks", a.numel())
    rep.add("pose_rounding_ulp_diffs", k)
    if k:
        worst = (a[diff].double() - b[diff].double()).abs().max().item()
        assert k <= max(1, 1e-5 * a.numel()) and worst <= 1e-6 * max(1.0, float(a.max().item())), \
            f"{tag}: {k} ranges differ, worst by {worst!r}"


def assert_ambiguity_bounds(rep):
    """The excluded near-tie classes must stay small: an exclusion class that grows would hide mismatches."""
    c = rep.c
    assert c.get("beams_ambiguous", 0) <= max(2, 1e-3 * c.get("beams", 0)), f"too many ambiguous beams: {rep}"
    assert c.get("collision_ambiguous", 0) <= max(2, 1e-3 * c.get("collision_checks", 0)), f"too many ambiguous collision flags: {rep}"
    assert c.get("resets_ambiguous", 0) <= max(2, 1e-2 * c.get("resets", 0)), f"too many ambiguous resets: {rep}"
    assert c.get("done_ambiguous", 0) <= max(2, 1e-3 * c.get("done_checks", 0)), f"too many ambiguous done flags: {rep}"
