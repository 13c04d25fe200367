"""GPU parity tests proper: the CUDA path through the C ABI vs the CPU oracle (pytest -m gpu)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import oracle
    oracle.build()
    import parity_util
    return parity_util


def test_c1_tiny_full(pu):
    from harness import workloads as W
    wl = W.make_workload(1)
    rep = pu.run_parity(wl, steps=100)
    print(rep)
    assert rep.c["beams_ambiguous"] < 1e-3 * rep.c["beams"]


def test_c1_ragged_env_counts(pu):
    # env counts that are not multiples of a warp/CTA; 1 env; beams not a multiple of 32
    from harness import workloads as W
    for n in (1, 7, 33):
        wl = W.make_workload(1, n_envs=n)
        wl.beam_angles = W.beam_table(45 + n, 270.0)
        print(n, pu.run_parity(wl, steps=12, seed=n))


def test_degenerate_beam_tables(pu):
    # one beam per robot (B = 1: every "idx / B" of the kernels degenerates), 33 beams (one full round and one beam),
    # with and without clearance features; a shared-memory map and an L2 map; instrumented and production kernels
    import torch
    from harness import workloads as W
    for cfg, nb, n in ((1, 1, 70), (1, 33, 5), (4, 1, 300)):
        wl = W.make_workload(cfg, n_envs=n)
        wl.beam_angles = W.beam_table(nb, 200.0) if nb > 1 else np.array([0.3], np.float32)
        rep = pu.run_parity(wl, steps=8, seed=nb)
        print(cfg, nb, rep)
        assert rep.c["beams"] >= 8 * n * nb
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, nb, wl.action_dim)
        z = torch.zeros(n, 1, device="cuda")
        s.bind_features(1, z)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, torch.from_numpy(W.seed_tape(wl, 1, 2)[0].view(np.int64)).cuda(), buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        import oracle
        ze = oracle.clearance_features(wl.footprint, wl.beam_angles, wl.max_range, 1, buf.ranges.cpu().numpy())
        assert np.abs(z.cpu().numpy() - ze).max() <= 1e-4
        s.close(); r.close(); m.close()


def test_c2_rect_subset(pu):
    from harness import workloads as W
    wl = W.make_workload(2)
    rep = pu.run_parity(wl, steps=30, subset=256, check_every=10)
    print(rep)


def test_c3_nonconvex_omni(pu):
    from harness import workloads as W
    wl = W.make_workload(3, n_envs=1024)
    rep = pu.run_parity(wl, steps=30, subset=256, check_every=5)
    print(rep)
    assert rep.c["collisions"] > 0


def test_c4_large_map_l2_path_forced_resets(pu):
    from harness import workloads as W
    wl = W.make_workload(4, n_envs=2048)
    rep = pu.run_parity(wl, steps=20, subset=512, check_every=5)
    print(rep)
    assert rep.c["resets"] > 2048


def test_c5_tiles_regions(pu):
    from harness import workloads as W
    wl = W.make_workload(5, n_envs=1024)
    rep = pu.run_parity(wl, steps=20, subset=128, check_every=5)
    print(rep)


def test_tiny_maps_odd_sizes_and_no_border(pu):
    # map sizes that are not multiples of 32, no border walls (beams and robots leave the map)
    from harness import workloads as W
    for size, seed in ((19, 1), (33, 2), (70, 3)):
        wl = W.tiny_workload(size=size, n_envs=64, n_beams=41, seed=seed, max_range=2.0)
        wl.occ[0, :] = wl.occ[-1, :] = 0
        wl.occ[:, 0] = wl.occ[:, -1] = 0
        wl.goal_dist_min, wl.goal_dist_max = np.float32(0.2), np.float32(0.6)
        print(size, pu.run_parity(wl, steps=15, seed=seed))


def test_axis_aligned_and_degenerate_beams(pu):
    # beams exactly along the axes and diagonals from exactly representable poses (ties, long spans)
    import torch
    import oracle
    import paper_2606_15846_b200 as fn
    from harness import workloads as W
    occ = np.zeros((200, 300), np.uint8)
    occ[:, 280:] = 1
    occ[150:, :] = 1
    occ[:, :3] = 1
    occ[:2, :] = 1
    ang = np.array([0, np.pi / 2, np.pi, -np.pi / 2, np.pi / 4, -3 * np.pi / 4, 1e-7, np.pi / 2 + 1e-7], np.float32)
    m = fn.Map(occ, 0.05)
    r = fn.Robot(W.footprint_rect(0.2, 0.2), ang, 20.0, 0, [0, 1, 0, 0, -1, 1])
    n = 8
    s = fn.Sim(m, r, n)
    st = torch.zeros(8, n, device="cuda")
    # rows 1 and 3 sit exactly on lattice lines (legitimately ambiguous); the others do not
    xs = np.array([5.025, 5.0, 7.5125, 1.0, 12.3, 5.0125, 9.9875, 3.3375], np.float32)
    ys = np.array([5.025, 5.0, 2.5125, 6.0, 0.7, 3.7625, 6.2625, 1.1125], np.float32)
    st[0] = torch.from_numpy(xs).cuda(); st[1] = torch.from_numpy(ys).cuda()
    out = torch.zeros(n, len(ang), device="cuda")
    hit = torch.zeros(n, len(ang), dtype=torch.int32, device="cuda")
    s.bind_aux(hit, None)
    s.observe_all(st, out)
    torch.cuda.synchronize()
    ro, ho, amb = oracle.ranges(occ, np.float32(0.05), ang, 20.0, xs, ys, np.zeros(n, np.float32))
    ok = amb == 0
    assert ok.sum() >= 32
    assert np.allclose(out.cpu().numpy()[ok], ro[ok], atol=1e-4)
    assert np.array_equal(hit.cpu().numpy()[ok], ho[ok])


def test_argument_errors(pu):
    import paper_2606_15846_b200 as fn
    from harness import workloads as W
    occ = np.zeros((8, 8), np.uint8)
    with pytest.raises(fn.FlashNavError):
        fn.Map(occ, 0.0)
    with pytest.raises(fn.FlashNavError):
        fn.Robot(W.footprint_rect(0.2, 0.2)[:2], [0.0], 1.0, 0, [0, 1, 0, 0, -1, 1])
    with pytest.raises(fn.FlashNavError):
        fn.Robot(W.footprint_rect(0.2, 0.2), [0.0], 1.0, 0, [1, 0, 0, 0, -1, 1])
    with pytest.raises(fn.FlashNavError):
        fn.Robot(W.footprint_rect(0.2, 0.2), [0.0], 1.0, 5, [0, 1, 0, 0, -1, 1])
    m = fn.Map(occ, 0.05)
    with pytest.raises(fn.FlashNavError):
        m.set_regions([[0, 0, 9, 9]])
    r = fn.Robot(W.footprint_rect(0.2, 0.2), [0.0], 1.0, 0, [0, 1, 0, 0, -1, 1])
    with pytest.raises(fn.FlashNavError):
        fn.Sim(m, r, 0)


def test_ring_rows_and_wraparound_gpu(pu):
    # S7 (BASELINE.json config 5): every completed ring row equals the tuple (obs the action
    # was chosen from, action, reward, done) logged by the harness, including slots that wrap around a
    # capacity that is not a multiple of the batch.  The expected ring is written by the oracle's append.
    import torch
    import oracle
    from harness import workloads as W
    for drive_cfg in (5, 3):                                   # differential (A = 2) and omnidirectional (A = 3)
        wl = W.make_workload(drive_cfg, n_envs=96)
        wl.forced_reset_frac = 0.05                            # forced resets: done code 2 (truncated)
        codes = set()
        n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, A)
        s.bind_aux(None, buf.reward)
        cap = 3 * n + 37
        row = B + 5 + A + 2
        ring = torch.zeros(cap * row, device="cuda")
        s.ring_attach(ring, cap)
        steps = 9
        actions = torch.from_numpy(W.action_tape(wl, steps, 3)).cuda()
        seeds = W.seed_tape(wl, steps + 1, 3)
        forced = W.forced_reset_tape(wl, steps, 3)
        expect = np.zeros((cap, row), np.float32)
        written = np.zeros(cap, bool)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, torch.from_numpy(seeds[0].view(np.int64)).cuda(), buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        head = 0
        for t in range(steps):
            obs_r = buf.ranges.cpu().numpy().copy()
            obs_g = buf.gobs.cpu().numpy().copy()              # [2, n] = d, alpha
            obs_v = buf.states.cpu().numpy()[3:6].copy()       # [3, n] = vx, vy, w
            buf.mask.copy_(torch.from_numpy(forced[t]))
            s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            torch.cuda.synchronize()
            done = oracle.done_code(buf.mask.cpu().numpy(), buf.col.cpu().numpy(), buf.gobs[0].cpu().numpy(), wl.goal_tol)
            codes |= set(done.tolist())
            oracle.ring_append(expect, cap, head, obs_r, obs_g, obs_v, actions[t].cpu().numpy(),
                               buf.reward.cpu().numpy(), done)
            written[(head + np.arange(n)) % cap] = True
            head = (head + n) % cap
            s.reset(buf.states, buf.mask, torch.from_numpy(seeds[t + 1].view(np.int64)).cuda(), buf.ranges, buf.gobs)
            torch.cuda.synchronize()
        got = ring.cpu().numpy().reshape(cap, row)
        pending = (head + np.arange(n)) % cap                  # rows started for the next step: obs part only
        check = written.copy()
        check[pending] = False
        assert check.sum() >= cap - n - 1
        assert np.array_equal(got[check], expect[check])
        assert {0, 2} <= codes                                 # (1 = terminated: the full-scale C5 test sees collisions)
        # pending rows already hold the observation the next action will be chosen from
        assert np.array_equal(got[pending, :B], buf.ranges.cpu().numpy())
        assert np.array_equal(got[pending, B:B + 2], buf.gobs.cpu().numpy().T)
        assert np.array_equal(got[pending, B + 2:B + 5], buf.states.cpu().numpy()[3:6].T)
        s.close(); r.close(); m.close()


def test_ring_at_full_scale_c5(pu):
    # S7 at BASELINE.json config 5's own size: 65 536 envs, ring of 2^22 transitions (12.2 GB), 66 steps, so that the
    # head wraps (2^22 = 64 x 65 536).  The rows of a fixed sample of 64 envs are checked after every step (4224 rows):
    # content against the oracle's append of the same envs, slot (head + e) mod capacity in Python integers.
    import torch
    import oracle
    from harness import workloads as W
    wl = W.make_workload(5)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    cap = 1 << 22
    row = B + 5 + A + 2
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    s.bind_aux(None, buf.reward)
    ring = torch.zeros(cap * row, device="cuda")
    s.ring_attach(ring, cap)
    ring2 = ring.view(cap, row)
    steps = 66
    rng = np.random.default_rng(11)
    sub = np.sort(rng.choice(n, 64, replace=False))
    sub_t = torch.from_numpy(sub).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 4).view(np.int64)).cuda()
    act_rng = np.random.default_rng(12)
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
    head = 0
    rows_checked = 0
    codes_seen = set()
    for t in range(steps):
        obs_r = buf.ranges[sub_t].cpu().numpy()
        obs_g = buf.gobs[:, sub_t].cpu().numpy()
        obs_v = buf.states[3:6, sub_t].cpu().numpy()
        a_np = (act_rng.random((n, A), dtype=np.float32) * np.array([1.0, 4.0], np.float32) - np.array([0.0, 2.0], np.float32))
        actions = torch.from_numpy(a_np).cuda()
        buf.mask.zero_()
        s.step(buf.states, actions, float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        torch.cuda.synchronize()
        expect = np.zeros((sub.size, row), np.float32)
        code = oracle.done_code(buf.mask[sub_t].cpu().numpy(), buf.col[sub_t].cpu().numpy(),
                                buf.gobs[0, sub_t].cpu().numpy(), wl.goal_tol)
        codes_seen |= set(code.tolist())
        oracle.ring_append(expect, sub.size, 0, obs_r, obs_g, obs_v, a_np[sub], buf.reward[sub_t].cpu().numpy(), code)
        slots = torch.tensor([(head + int(e)) % cap for e in sub], device="cuda")
        got = ring2[slots].cpu().numpy()
        assert np.array_equal(got, expect), f"step {t}: ring rows of the sampled envs"
        rows_checked += sub.size
        head = (head + n) % cap
        s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
    assert head == (steps * n) % cap == 2 * n and rows_checked == 4224
    # rows the wrap has overwritten hold steps 64 and 65; the pending rows hold the current observation
    pend = torch.tensor([(head + int(e)) % cap for e in sub], device="cuda")
    assert torch.equal(ring2[pend][:, :B], buf.ranges[sub_t])
    assert {0, 1} <= codes_seen                                # running and terminated rows (collisions within 66 steps)
    s.close(); r.close(); m.close()
    del ring, ring2
    torch.cuda.empty_cache()


def test_several_sensors_against_the_oracle(pu):
    # SURVEY 8(f) NEXT-3 (PAPER.md:65 "S defines sensor placement and range-sensing parameters", :125): a robot with
    # three range sensors (different beam tables, ranges and placements).  Rows = the sensors' ranges one after the
    # other; ranges and hit cells against oracle.ranges_multi (tolerances of run_parity) through steps, resets of the
    # done list and of a mask, fn_observe_all; production kernel == instrumented kernel; ring rows carry the full row.
    import torch
    import oracle
    import paper_2606_15846_b200 as fn
    from harness import workloads as W
    for cfg in (2, 4):                                            # map in shared memory / read through L2
        wl = W.make_workload(cfg, n_envs=400)
        n, A = wl.n_envs, wl.action_dim
        sensors = [(wl.beam_angles, float(wl.max_range), (0.1, -0.05, 0.2)),
                   (W.beam_table(90, 120.0), 4.0, (-0.2, 0.1, 3.0)),
                   (W.beam_table(33, 360.0), 2.5, (0.0, 0.15, -1.0))]
        m = fn.Map(wl.occ, float(wl.resolution))
        r = fn.Robot(wl.footprint, wl.beam_angles, float(wl.max_range), wl.drive, wl.vel_limits)
        r.set_sensor(*sensors[0][2])
        for ang, rmax, plc in sensors[1:]:
            r.add_sensor(ang, rmax, *plc)
        B = r.B
        assert B == wl.n_beams + 90 + 33
        s = fn.Sim(m, r, n, goal_tol=float(wl.goal_tol), goal_dist_min=float(wl.goal_dist_min), goal_dist_max=float(wl.goal_dist_max))
        assert not s.beam_config()["split_step"] and not s.beam_config()["fused_reset"]
        buf = pu.Buffers(n, B, A)
        s.bind_aux(buf.hit, buf.reward)
        cap = 4 * n + 5
        row = B + 5 + A + 2
        ring = torch.zeros(cap * row, device="cuda")
        s.ring_attach(ring, cap)
        steps = 6
        actions = torch.from_numpy(W.action_tape(wl, steps, 8)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 8).view(np.int64)).cuda()

        def check(tag, idx=None):
            torch.cuda.synchronize()
            st = buf.states.cpu().numpy()
            idx = np.arange(n) if idx is None else idx
            ro, ho, ao = oracle.ranges_multi(wl.occ, wl.resolution, sensors, st[0, idx], st[1, idx], st[2, idx])
            g, gh = buf.ranges.cpu().numpy()[idx], buf.hit.cpu().numpy()[idx]
            ok = ao == 0
            assert (~ok).sum() <= max(2, 1e-3 * ok.size)
            assert np.array_equal(gh[ok], ho[ok]), f"{tag}: hit cells"
            assert np.all(np.abs(g.astype(np.float64) - ro)[ok] <= pu.TOL_RANGE), f"{tag}: ranges"
            off = 0
            for ang, rmax, _ in sensors:                          # every block is capped at its own sensor's range
                assert g[:, off:off + len(ang)].max() <= rmax + 1e-6
                off += len(ang)

        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
        check("initial reset")
        head = 0
        for t in range(steps):
            obs = buf.ranges.clone()
            buf.mask.zero_()
            s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            check(f"step {t}")
            torch.cuda.synchronize()
            slots = (head + torch.arange(n, device="cuda")) % cap
            assert torch.equal(ring.view(cap, row)[slots][:, :B], obs), "ring rows carry the observation of all sensors"
            head = (head + n) % cap
            done = np.nonzero(buf.mask.cpu().numpy())[0]
            keep = buf.ranges.clone()
            if t % 2 == 0:
                s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
            else:
                s.reset(buf.states, buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
            if done.size:
                check(f"reset {t}", done)
            other = np.setdiff1d(np.arange(n), done)
            assert torch.equal(buf.ranges[other], keep[other]), "recompute touched other rows"
        # instrumented and production kernels, all envs
        inst = torch.empty_like(buf.ranges)
        s.observe_all(buf.states, inst)
        s.bind_aux(None, buf.reward)
        fast = torch.empty_like(buf.ranges)
        s.observe_all(buf.states, fast)
        torch.cuda.synchronize()
        assert torch.equal(inst, fast)
        z = torch.zeros(n, 8, device="cuda")
        with pytest.raises(fn.FlashNavError):
            s.bind_features(8, z)                                 # clearance features: single-sensor robots only
        # a sensor added after fn_sim_create: the sim's poses and rows were sized without it, every call refuses
        if cfg == 2:
            r.add_sensor(W.beam_table(8, 90.0), 1.0, 0.0, 0.0, 0.0)
            before = buf.states.clone()
            big = torch.zeros(n, r.B, device="cuda")              # (sized for the new row, so that the library decides)
            for call in (lambda: s.step(buf.states, actions[0], float(wl.dt), buf.mask, big, buf.col, buf.gobs),
                         lambda: s.reset(buf.states, buf.mask, seeds[0], big, buf.gobs),
                         lambda: s.observe_all(buf.states, big),
                         lambda: s.ranges_fixed_step(buf.states, 0.025, True, big),
                         lambda: s.bind_features(4, torch.zeros(n, 4, device="cuda"))):
                with pytest.raises(fn.FlashNavError, match="sensors changed"):
                    call()
            torch.cuda.synchronize()
            assert torch.equal(buf.states, before)
        s.close(); r.close(); m.close()


def test_sensor_offset_in_the_beam_kernel(pu):
    # Sensor placement S (PAPER.md:65 "S defines sensor placement", :125; reading G8): beams start at the sensor, not
    # at the body origin.  The oracle casts from the offset pose (pinned by "sensor offset == moved robot",
    # tests/test_oracle_ranges.py); here the kernels' ranges and hit cells are compared with it on C2 and C3,
    # through steps and resets (pose from the motion kernel and from the reset kernels).
    from harness import workloads as W
    for cfg in (2, 3):
        wl = W.make_workload(cfg, n_envs=600)
        wl.sensor = (0.1, -0.05, 0.2)
        rep = pu.run_parity(wl, steps=8, subset=160, check_every=2)
        print(cfg, rep)
        assert rep.c["beams"] > 100000


def test_long_trajectories_c2_and_c5(pu):
    # the configs run 1000 / 500 steps; full batch on steps 0, 1, 2 and every 100th, a fixed subset of
    # envs on every step (C5: every 50th step).  Reaches what short runs do not: many episodes per env, the
    # cached-heading path of the motion kernel (exact sincos only every 32nd episode step), ring wrap-around.
    from harness import workloads as W
    wl = W.make_workload(2)
    rep = pu.run_parity(wl, steps=1000, subset=128, check_every=1, full_every=250)
    print(rep)
    assert rep.c["steps"] == 1000 and rep.c["done_events"] > 50 * wl.n_envs // 4
    wl = W.make_workload(5, n_envs=16384)
    rep = pu.run_parity(wl, steps=500, subset=96, check_every=50)
    print(rep)
    assert rep.c["steps"] == 500


def test_production_launch_sequence_against_the_oracle(pu):
    # What bench.py times, held against the oracle with no GPU kernel in between: no hit cells bound (fn_step runs the
    # production step kernel step_beam_kernel<1,0,0,1>, not the instrumented one), reset seeds announced before every
    # step, fn_reset(mask = NULL) served by prepared_reset_kernel.  States, collision, goal obs, done, reward, reset
    # states and RANGES against the oracle at the usual tolerances: C2's full batch over 50 steps (all beams on steps
    # 0-2, 192 envs' beams on every step), C3's full batch (union-free nonconvex footprint, omni drive), and C5 at
    # 16 384 envs with the ring attached (map read through L2: production beam kernel, no prepared resets).
    from harness import workloads as W
    wl = W.make_workload(2)
    wl.forced_reset_frac = 0.02
    rep = pu.run_production_parity(wl, steps=50, subset=192)
    print(rep)
    assert rep.c["resets_prepared"] > 0.5 * (rep.c["resets"] - wl.n_envs) > 0, rep
    assert rep.c["beams"] >= 3 * wl.n_envs * wl.n_beams
    wl = W.make_workload(3)
    rep = pu.run_production_parity(wl, steps=8, subset=128, full_steps=(0,))
    print(rep)
    assert rep.c["resets_prepared"] > 0, rep
    wl = W.make_workload(5, n_envs=16384)
    rep = pu.run_production_parity(wl, steps=6, subset=96, full_steps=(), ring=True)
    print(rep)
    assert rep.c["resets_prepared"] == 0 and rep.c["resets"] > wl.n_envs


def test_prepared_reset_without_its_head_start(pu, monkeypatch):
    # prepared_reset_kernel works under the step kernel's tail once the step's outcome warps have reported in; if they
    # have not within its patience (a debugger, a time-sliced context) it waits for the whole step instead and does
    # the same work afterwards -- no guard that could kill the context.  FLASHNAV_PREP_SPIN=0 (read at fn_sim_create)
    # forces that branch: the production sequence must still agree with the oracle, resets prepared.
    from harness import workloads as W
    monkeypatch.setenv("FLASHNAV_PREP_SPIN", "0")
    wl = W.make_workload(2)
    wl.forced_reset_frac = 0.03
    rep = pu.run_production_parity(wl, steps=6, subset=96, full_steps=(0,))
    print(rep)
    assert rep.c["resets_prepared"] > 0.5 * (rep.c["resets"] - wl.n_envs) > 0, rep


def test_full_size_sampled_c3_c4(pu):
    # BASELINE.json's full batch sizes in the launch configuration bench.py times; beams of a fixed random
    # subset of envs against the oracle, everything per-env (motion, collision, goal obs, reward/done) in full.
    from harness import workloads as W
    for cfg in (3, 4):
        wl = W.make_workload(cfg)
        rep = pu.run_parity(wl, steps=6, subset=192, check_every=3)
        print(cfg, rep)
        assert rep.c["collision_checks"] >= 2 * wl.n_envs


def test_full_size_sampled_c5_with_regions(pu):
    from harness import workloads as W
    wl = W.make_workload(5)
    rep = pu.run_parity(wl, steps=4, subset=96, check_every=2)
    print(rep)
    assert rep.c["resets"] > wl.n_envs


def test_cuda_graph_replay_equals_direct_launches(pu):
    # fn_step / fn_reset only enqueue kernels and keep per-step state on the device: a captured sequence
    # replayed as a CUDA graph must reproduce the directly launched trajectory bit for bit.
    import torch
    from harness import workloads as W
    wl = W.make_workload(1, n_envs=128)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    steps = 12
    actions = torch.from_numpy(W.action_tape(wl, steps, 5)).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 5).view(np.int64)).cuda()
    results = []
    for use_graph in (False, True):
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, A)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
        torch.cuda.synchronize()

        def run():
            for t in range(steps):
                buf.mask.zero_()
                s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
                s.reset(buf.states, buf.mask, seeds[t + 1], buf.ranges, buf.gobs)

        if use_graph:
            cs = torch.cuda.Stream()
            cs.wait_stream(torch.cuda.current_stream())
            g = torch.cuda.CUDAGraph()
            s.set_stream(cs)
            with torch.cuda.graph(g, stream=cs):
                run()
            s.set_stream(torch.cuda.current_stream())
            g.replay()
        else:
            run()
        torch.cuda.synchronize()
        results.append((buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), buf.col.clone(), s.counters()["envs_reset"]))
        s.close(); r.close(); m.close()
    for a, b in zip(results[0][:4], results[1][:4]):
        assert torch.equal(a, b)
    assert results[0][4] == results[1][4] > n


def test_reset_of_the_steps_done_list_equals_masked_reset(pu):
    # fn_reset(mask = NULL) resets exactly the envs the preceding fn_step reported done, from the list the
    # step kernel keeps on the device (any order): same states, observations and counters as the mask path.
    import torch
    import paper_2606_15846_b200 as fn
    from harness import workloads as W
    wl = W.make_workload(4, n_envs=1500)                       # forced resets + collisions; not a multiple of 32
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    steps = 7
    actions = torch.from_numpy(W.action_tape(wl, steps, 11)).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 11).view(np.int64)).cuda()
    forced = torch.from_numpy(W.forced_reset_tape(wl, steps, 11)).cuda()
    out = []
    for use_list in (False, True):
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, A)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
        for t in range(steps):
            buf.mask.copy_(forced[t])
            s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            s.reset(buf.states, None if use_list else buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        c = s.counters()
        out.append((buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), c["envs_reset"], c["rays_cast"]))
        if use_list:
            with pytest.raises(fn.FlashNavError):              # the step's list is consumed
                s.reset(buf.states, None, seeds[0], buf.ranges, buf.gobs)
        s.close(); r.close(); m.close()
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1]) and torch.equal(out[0][2], out[1][2])
    assert out[0][3] == out[1][3] > n and out[0][4] == out[1][4]


def test_fused_reset_kernel_equals_the_two_kernel_path(pu):
    # fn_reset runs ONE kernel when the map is staged in shared memory (each CTA resets its share of the list
    # from its shared copy of the map, then recomputes those envs' beams) and two kernels otherwise: same
    # states, goal observations, ranges, ring rows and counters, bit for bit -- for the step's done list, for
    # a mask, for an all-env reset (several envs per CTA), an empty list, and with the instrumented kernels.
    import torch
    from harness import workloads as W
    for cfg, n, ring_cap, aux in ((2, 1500, 0, False), (3, 777, 0, False), (1, 64, 0, True), (2, 9000, 0, False), (1, 300, 1024, False)):
        wl = W.make_workload(cfg, n_envs=n)
        B, A = wl.n_beams, wl.action_dim
        steps = 6
        actions = torch.from_numpy(W.action_tape(wl, steps, 5)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 2, 5).view(np.int64)).cuda()
        forced = torch.from_numpy((np.random.default_rng(5).random((steps, n)) < 0.03).astype(np.uint8)).cuda()
        out = []
        for fused in (True, False):
            m, r, s = pu.make_sim(wl, n)
            assert s.beam_config()["smem"]
            assert s.set_fused_reset(2 if fused else 0) == fused            # 2: the fused kernel for masks too
            buf = pu.Buffers(n, B, A)
            hit = torch.full((n, B), -9, dtype=torch.int32, device="cuda")
            rew = torch.zeros(n, device="cuda")
            if aux:
                s.bind_aux(hit, rew)
            ring = None
            if ring_cap:
                row = B + 5 + A + 2
                ring = torch.zeros(ring_cap * row, device="cuda")
                s.ring_attach(ring, ring_cap)
            buf.mask.fill_(1)
            s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)          # all envs: several per CTA
            snap = [buf.states.clone(), buf.ranges.clone()]
            buf.mask.zero_()
            s.reset(buf.states, buf.mask, seeds[1], buf.ranges, buf.gobs)          # empty list: nothing changes
            assert torch.equal(snap[0], buf.states) and torch.equal(snap[1], buf.ranges)
            for t in range(steps):
                buf.mask.copy_(forced[t])
                s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
                s.reset(buf.states, None if t % 2 == 0 else buf.mask, seeds[t + 2], buf.ranges, buf.gobs)
            torch.cuda.synchronize()
            c = s.counters()
            assert c["oob_window_loads"] == 0
            out.append((buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), hit.clone(),
                        None if ring is None else ring.clone(), c["envs_reset"], c["rays_cast"], c["reset_failures"]))
            s.close(); r.close(); m.close()
        for a, b in zip(out[0][:4], out[1][:4]):
            assert torch.equal(a, b)
        if ring_cap:
            assert torch.equal(out[0][4], out[1][4])
        assert out[0][5:] == out[1][5:] and out[0][5] > n


def test_step_host_equals_the_device_calls(pu):
    # fn_step_host = H2D + fn_step + fn_reset(done list) + D2H in one call.  With PINNED host buffers the beam
    # kernels store the ranges straight into the caller's memory (zero-copy), with pageable ones they go
    # through a device staging buffer and a copy: both must equal the device-side calls bit for bit.
    import torch
    from harness import workloads as W
    wl = W.make_workload(2, n_envs=700)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    steps = 5
    act = W.action_tape(wl, steps, 9)
    seeds = W.seed_tape(wl, steps + 1, 9).view(np.int64)
    # device path
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, torch.from_numpy(seeds[0]).cuda(), buf.ranges, buf.gobs)
    torch.cuda.synchronize()
    st0 = buf.states.cpu().numpy().copy()
    ref = []
    for t in range(steps):
        buf.mask.zero_()
        s.step(buf.states, torch.from_numpy(act[t]).cuda(), float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        done = buf.mask.clone(); col = buf.col.clone()
        s.reset(buf.states, None, torch.from_numpy(seeds[t + 1]).cuda(), buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        ref.append([x.cpu().numpy().copy() for x in (buf.states, buf.ranges, buf.gobs, done, col)])
    s.close(); r.close(); m.close()
    for pinned in (True, False):
        m, r, s = pu.make_sim(wl, n)
        dev = pu.Buffers(n, B, A)
        dev.mask.fill_(1)
        s.reset(dev.states, dev.mask, torch.from_numpy(seeds[0]).cuda(), dev.ranges, dev.gobs)   # same episode state
        torch.cuda.synchronize()
        def host(shape, dtype):
            t = torch.zeros(shape, dtype=dtype)
            return t.pin_memory() if pinned else t.numpy()
        hs, hr, hg = host((8, n), torch.float32), host((n, B), torch.float32), host((2, n), torch.float32)
        hm, hc = host((n,), torch.uint8), host((n,), torch.uint8)
        (hs.numpy() if pinned else hs)[...] = st0
        for t in range(steps):
            (hm.numpy() if pinned else hm)[...] = 0
            ha = torch.from_numpy(act[t]).pin_memory() if pinned else act[t]
            hq = torch.from_numpy(seeds[t + 1]).pin_memory() if pinned else seeds[t + 1]
            s.step_host(hs, ha, float(wl.dt), hm, hq, hr, hc, hg)
            got = [np.asarray(x.numpy() if pinned else x) for x in (hs, hr, hg, hm, hc)]
            for a, b in zip(got, ref[t]):
                assert np.array_equal(a, b)
        s.close(); r.close(); m.close()
    # pipelined form: two slots, step t + 1 is enqueued before step t's outputs are awaited
    m, r, s = pu.make_sim(wl, n)
    dev = pu.Buffers(n, B, A)
    dev.mask.fill_(1)
    s.reset(dev.states, dev.mask, torch.from_numpy(seeds[0]).cuda(), dev.ranges, dev.gobs)
    torch.cuda.synchronize()
    slots = []
    for k in range(2):
        slots.append({"s": torch.zeros(8, n).pin_memory(), "r": torch.zeros(n, B).pin_memory(), "g": torch.zeros(2, n).pin_memory(),
                      "m": torch.zeros(n, dtype=torch.uint8).pin_memory(), "c": torch.zeros(n, dtype=torch.uint8).pin_memory()})
    h0 = torch.from_numpy(st0).pin_memory()
    has = [torch.from_numpy(act[t]).pin_memory() for t in range(steps)]
    hqs = [torch.from_numpy(seeds[t + 1]).pin_memory() for t in range(steps)]
    with pytest.raises(Exception):
        s.step_host_end(0)                                       # nothing in flight
    for t in range(steps + 1):
        if t < steps:
            b = slots[t & 1]
            b["m"].zero_()
            s.step_host_begin(t & 1, h0 if t == 0 else None, has[t], float(wl.dt), b["m"], hqs[t], b["s"], b["r"], b["c"], b["g"])
            if t == 0:
                with pytest.raises(Exception):
                    s.step_host_begin(0, None, has[0], float(wl.dt), b["m"], hqs[0], b["s"], b["r"], b["c"], b["g"])   # slot in flight
        if t >= 1:
            b = slots[(t - 1) & 1]
            s.step_host_end((t - 1) & 1)
            for a, e in zip((b["s"], b["r"], b["g"], b["m"], b["c"]), ref[t - 1]):
                assert np.array_equal(a.numpy(), e), f"pipelined step {t - 1}"
    s.close(); r.close(); m.close()


def test_step_host_after_the_pipelined_form_on_one_sim(pu):
    # The two host entry points share one staging buffer (the states) and each has others of its own: a sim that has
    # served fn_step_host_begin / _end must still serve fn_step_host (it answered FN_ERR_CUDA: copies to buffers it
    # had skipped allocating), and the other way round.  Sim A: pipelined step 0, fn_step_host step 1, pipelined
    # step 2; sim B: fn_step_host for all three.  Outputs must agree bit for bit.
    import torch
    from harness import workloads as W
    wl = W.make_workload(1, n_envs=96)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    act = W.action_tape(wl, 3, 4)
    seeds = W.seed_tape(wl, 4, 4).view(np.int64)
    outs = {}
    for name in ("A", "B"):
        m, r, s = pu.make_sim(wl, n)
        dev = pu.Buffers(n, B, A)
        dev.mask.fill_(1)
        s.reset(dev.states, dev.mask, torch.from_numpy(seeds[0]).cuda(), dev.ranges, dev.gobs)
        torch.cuda.synchronize()
        hs = dev.states.cpu().pin_memory()
        hr, hg = torch.zeros(n, B).pin_memory(), torch.zeros(2, n).pin_memory()
        hm, hc = torch.zeros(n, dtype=torch.uint8).pin_memory(), torch.zeros(n, dtype=torch.uint8).pin_memory()
        got = []
        for t in range(3):
            ha, hq = torch.from_numpy(act[t]).pin_memory(), torch.from_numpy(seeds[t + 1]).pin_memory()
            hm.zero_()
            if name == "A" and t != 1:
                s.step_host_begin(0, hs, ha, float(wl.dt), hm, hq, hs, hr, hc, hg)
                s.step_host_end(0)
            else:
                s.step_host(hs, ha, float(wl.dt), hm, hq, hr, hc, hg)
            got.append([x.numpy().copy() for x in (hs, hr, hg, hm, hc)])
        outs[name] = got
        s.close(); r.close(); m.close()
    for t in range(3):
        for a, b in zip(outs["A"][t], outs["B"][t]):
            assert np.array_equal(a, b), f"step {t}"


def test_split_step_equals_the_single_env_step_kernel(pu):
    # fn_step either runs one env-step kernel, the ring-advance kernel and the beam kernel, or (default) a
    # motion kernel and a beam kernel whose last warps compute collision / goal / reward / done for the envs
    # their CTAs own and whose last CTA advances the ring head and the done-list parity: same states, flags,
    # observations, rewards, hit cells, ring rows, done lists and counters, bit for bit.  Shared-memory and
    # L2 maps, one and many envs per CTA (more than a warp's 32), a ring, the instrumented kernels.
    import torch
    from harness import workloads as W
    for cfg, n, ring_cap, aux in ((1, 64, 0, True), (2, 1500, 0, False), (3, 2000, 0, False), (4, 1100, 0, False),
                                  (1, 20000, 0, False), (5, 300, 1024, False), (5, 700, 0, True)):
        wl = W.make_workload(cfg, n_envs=n)
        B, A = wl.n_beams, wl.action_dim
        steps = 6
        actions = torch.from_numpy(W.action_tape(wl, steps, 6)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 6).view(np.int64)).cuda()
        forced = torch.from_numpy((np.random.default_rng(6).random((steps, n)) < 0.03).astype(np.uint8)).cuda()
        out = []
        for split in (True, False):
            m, r, s = pu.make_sim(wl, n)
            assert s.set_split_step(split) == split
            buf = pu.Buffers(n, B, A)
            hit = torch.full((n, B), -9, dtype=torch.int32, device="cuda")
            rew = torch.zeros(n, device="cuda")
            s.bind_aux(hit if aux else None, rew)
            ring = None
            if ring_cap:
                ring = torch.zeros(ring_cap * (B + 5 + A + 2), device="cuda")
                s.ring_attach(ring, ring_cap)
            buf.mask.fill_(1)
            s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
            trace = []
            for t in range(steps):
                buf.mask.copy_(forced[t])
                s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
                trace += [buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), buf.mask.clone(), buf.col.clone(), rew.clone(), hit.clone()]
                s.reset(buf.states, None if t % 2 == 0 else buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
                trace += [buf.states.clone(), buf.ranges.clone()]
            torch.cuda.synchronize()
            c = s.counters()
            assert c["oob_window_loads"] == 0
            if ring is not None:
                trace.append(ring.clone())
            d_prev, ep = s.episode_state()
            trace += [torch.from_numpy(d_prev), torch.from_numpy(ep)]
            out.append((trace, c))
            s.close(); r.close(); m.close()
        for a, b in zip(out[0][0], out[1][0]):
            assert torch.equal(a, b)
        assert out[0][1] == out[1][1] and out[0][1]["envs_reset"] > n


def test_coarse_level_on_and_off_give_identical_results(pu):
    # BASELINE.json north_star "coarse block-occupancy level for empty-space skipping"; SURVEY.md 8(c) pin
    # "coarse-level on/off => identical".  The production beam kernels either walk the fine copies line by line
    # or the coarse copies (one window per pair of lines, fine lines only behind a non-empty window): same
    # states, flags, ranges, goal observations and counters, bit for bit, over steps with resets, for maps staged
    # in shared memory (C1, C2, C3, ragged sizes, a map without border walls, a sensor offset).
    import torch
    from harness import workloads as W
    cases = [(1, 64), (2, 1500), (3, 2000), (1, 7)]
    for ci, (cfg, n) in enumerate(cases):
        wl = W.make_workload(cfg, n_envs=n)
        if ci == 3:
            wl.beam_angles = W.beam_table(77, 270.0)
            wl.occ = wl.occ.copy(); wl.occ[0, :] = 0; wl.occ[-1, :] = 0; wl.occ[:, 0] = 0; wl.occ[:, -1] = 0
        B, A = wl.n_beams, wl.action_dim
        steps = 8
        actions = torch.from_numpy(W.action_tape(wl, steps, 9)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 9).view(np.int64)).cuda()
        out = []
        for coarse in (True, False):
            m, r, s = pu.make_sim(wl, n)
            if ci == 2:
                r.set_sensor(0.1, -0.05, 0.2)
            assert s.beam_config()["coarse_available"], "the coarse copies of a 512 x 512 map fit one CTA"
            assert s.set_coarse(coarse) == coarse and s.beam_config()["coarse"] == coarse
            buf = pu.Buffers(n, B, A)
            buf.mask.fill_(1)
            s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
            trace = [buf.ranges.clone()]
            for t in range(steps):
                buf.mask.zero_()
                s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
                trace += [buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), buf.mask.clone(), buf.col.clone()]
                s.reset(buf.states, None if t % 2 == 0 else buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
                trace += [buf.states.clone(), buf.ranges.clone()]
                full = torch.empty_like(buf.ranges)
                s.observe_all(buf.states, full)
                trace.append(full)
            torch.cuda.synchronize()
            out.append((trace, s.counters()))
            s.close(); r.close(); m.close()
        for k, (a, b) in enumerate(zip(out[0][0], out[1][0])):
            assert torch.equal(a, b), f"config {cfg}: item {k} differs with the coarse level on"
        assert out[0][1] == out[1][1]


def test_prepared_reset_equals_the_plain_reset(pu):
    # fn_sim_prepare_reset: with the seeds announced, the step's outcome warps run the reset of the envs
    # they report done and fn_reset(mask = NULL) only copies and recomputes the observations.  The plain path is the
    # one the parity tests hold against the oracle; here both paths give the same states, flags, ranges, goal
    # observations, episode counters, ring and counters, bit for bit, step by step -- at C2's full batch (several done
    # envs per CTA), with forced resets, a union footprint with a sensor offset (C3), a ring, with announcements that
    # must NOT be used (other seeds, a setter in between), and for sims whose announcements are dropped altogether.
    import torch
    from harness import workloads as W
    cases = ((2, 4096, 40, False, True), (3, 4096, 12, True, True), (1, 4000, 12, True, True),
             (2, 4097, 9, True, True),                            # with a step limit of 3: every env ends at once, twice
             (1, 64, 40, True, False),                            # too few beams to hide a reset under: dropped
             (5, 512, 6, False, False))                           # map read through L2: no such kernel
    for cfg, n, steps, with_ring, expect_used in cases:
        wl = W.make_workload(cfg, n_envs=n)
        wl.forced_reset_frac = 0.03
        if n == 4097:
            wl.max_episode_steps = 3
        B, A = wl.n_beams, wl.action_dim
        actions = torch.from_numpy(W.action_tape(wl, steps, 5)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 2, 5).view(np.int64)).cuda()
        forced = torch.from_numpy(W.forced_reset_tape(wl, steps, 5)).cuda()
        out = []
        for prepare in (True, False):
            m, r, s = pu.make_sim(wl, n)
            if cfg == 3:
                r.set_sensor(0.1, -0.05, 0.2)
            buf = pu.Buffers(n, B, A)
            s.bind_aux(None, buf.reward)
            ring = None
            if with_ring:
                cap = 3 * n + 11
                ring = torch.zeros(cap * s.ring_row_floats(), device="cuda")
                s.ring_attach(ring, cap)
            buf.mask.fill_(1)
            s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
            trace = []
            for t in range(steps):
                buf.mask.copy_(forced[t])
                odd = t % 7 == 3                                  # an announcement that fn_reset must not use
                if prepare:
                    s.prepare_reset(seeds[steps + 1] if odd and t % 14 == 3 else seeds[t + 1])
                s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
                trace += [buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), buf.mask.clone(), buf.col.clone(), buf.reward.clone()]
                if odd and t % 14 == 10:
                    r.set_sensor(*((0.1, -0.05, 0.2) if cfg == 3 else (0.0, 0.0, 0.0)))     # same values, new version
                s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
                dp, ep = s.episode_state()
                trace += [buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), torch.from_numpy(dp), torch.from_numpy(ep)]
                if t % 5 == 4:                                    # the poses the reset left behind serve later launches
                    full = torch.empty_like(buf.ranges)
                    s.observe_all(buf.states, full)
                    trace.append(full)
            torch.cuda.synchronize()
            if ring is not None:
                trace.append(ring.clone())
            out.append((trace, s.counters()))
            s.close(); r.close(); m.close()
        for k, (a, b) in enumerate(zip(out[0][0], out[1][0])):
            assert torch.equal(a, b), f"config {cfg}: item {k} differs with the reset prepared by the step"
        c1, c0 = dict(out[0][1]), dict(out[1][1])
        used = c1.pop("resets_prepared")
        assert c0.pop("resets_prepared") == 0
        assert c1 == c0, (c1, c0)
        assert c1["envs_reset"] > n + steps // 2
        if not expect_used:
            assert used == 0
        else:
            assert 0.5 * (c1["envs_reset"] - n) <= used < c1["envs_reset"] - n, (used, c1)
            if n == 4097:
                assert c1["envs_reset"] > 3 * n                   # the list was the whole batch at least twice


def test_prepared_reset_takes_the_seed_values_of_the_step(pu):
    # The contract of fn_sim_prepare_reset, pinned from its sharp side: the announced buffer is READ DURING fn_step,
    # and the library recognises the announcement at fn_reset by the buffer's address.  A caller that keeps one seeds
    # tensor and rewrites it in place between fn_step and fn_reset therefore gets the resets drawn from the values the
    # buffer held during the step -- not from the new ones, and unlike the un-announced path.  (Header, binding
    # docstring and README say so: announce a buffer that stays untouched until fn_reset, e.g. two alternating ones.)
    import torch
    from harness import workloads as W
    n = 4096
    wl = W.make_workload(2, n_envs=n)
    wl.forced_reset_frac = 0.05
    B, A = wl.n_beams, wl.action_dim
    actions = torch.from_numpy(W.action_tape(wl, 1, 3)).cuda()
    tape = torch.from_numpy(W.seed_tape(wl, 3, 3).view(np.int64)).cuda()
    forced = torch.from_numpy(W.forced_reset_tape(wl, 1, 3)).cuda()
    res = {}
    for name in ("announced, refilled in place", "plain, old seeds", "plain, new seeds"):
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, A)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, tape[0], buf.ranges, buf.gobs)
        buf.mask.copy_(forced[0])
        live = tape[1].clone()                                    # the caller's one persistent seeds tensor
        if name.startswith("announced"):
            s.prepare_reset(live)
        s.step(buf.states, actions[0], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        if name != "plain, old seeds":
            live.copy_(tape[2])                                   # rewritten between fn_step and fn_reset
        s.reset(buf.states, None, live, buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        res[name] = (buf.states.clone(), buf.ranges.clone(), buf.gobs.clone(), s.counters())
        s.close(); r.close(); m.close()
    a, old, new = res["announced, refilled in place"], res["plain, old seeds"], res["plain, new seeds"]
    assert a[3]["resets_prepared"] > 0.03 * n and old[3]["resets_prepared"] == 0
    for k in range(3):
        assert torch.equal(a[k], old[k]), "a prepared reset uses the seed values the buffer held during fn_step"
    assert not torch.equal(a[0], new[0])


def test_clearance_features_against_the_oracle(pu):
    # NEXT-1 (Eq. (3)): sector-pooled footprint clearances.  Teacher-forced:
    # the oracle computes them in fp64 from the GPU's own fp32 ranges; tolerance 1e-4 m like the ranges
    # (the clearance is continuous across the polygon boundary, so there is no near-tie class).
    import torch
    import oracle
    from harness import workloads as W
    cases = ((2, 300, 36, None), (3, 257, 24, (0.1, -0.05, 0.2)), (1, 64, 360, None), (5, 200, 7, None))
    for cfg, n, ns, sensor in cases:
        wl = W.make_workload(cfg, n_envs=n)
        B, A = wl.n_beams, wl.action_dim
        m, r, s = pu.make_sim(wl, n)
        if sensor is not None:
            r.set_sensor(*sensor)
        buf = pu.Buffers(n, B, A)
        z = torch.full((n, ns), -1.0, device="cuda")
        s.bind_features(ns, z)
        steps = 6
        actions = torch.from_numpy(W.action_tape(wl, steps, 2)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 2).view(np.int64)).cuda()
        forced = torch.from_numpy(W.forced_reset_tape(wl, steps, 2)).cuda()

        def expect():
            return oracle.clearance_features(wl.footprint, wl.beam_angles, wl.max_range, ns, buf.ranges.cpu().numpy(),
                                             sensor=None if sensor is None else np.array(sensor, np.float32))

        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        assert np.abs(z.cpu().numpy() - expect()).max() <= 1e-4
        n_reset = 0
        for t in range(steps):
            buf.mask.copy_(forced[t])
            s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            torch.cuda.synchronize()
            zs = z.cpu().numpy().copy()
            assert np.abs(zs - expect()).max() <= 1e-4, f"cfg {cfg} step {t}"
            done = buf.mask.cpu().numpy() != 0
            s.reset(buf.states, None if t % 2 else buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
            torch.cuda.synchronize()
            zr = z.cpu().numpy()
            assert np.array_equal(zr[~done], zs[~done])            # only the reset envs' rows are rewritten
            assert np.abs(zr - expect()).max() <= 1e-4, f"cfg {cfg} step {t} after reset"
            n_reset += int(done.sum())
        assert n_reset > 0
        # features are a pure function of the ranges: a full recompute reproduces the maintained rows
        z2 = torch.empty_like(z)
        s.bind_features(ns, z2)
        full_r = torch.empty_like(buf.ranges)
        s.observe_all(buf.states, full_r)
        torch.cuda.synchronize()
        assert torch.equal(z2, z)
        s.bind_features(ns, None)
        s.close(); r.close(); m.close()


def test_replay_sampling_against_the_oracle(pu):
    # NEXT-2: U x B transitions sampled uniformly from the device ring.  A gather: bit-exact
    # against the oracle's fno_ring_sample on the GPU's own ring, before and after the ring has wrapped,
    # with and without the next-observation output; an empty ring writes nothing.
    import torch
    import oracle
    from harness import workloads as W
    wl = W.make_workload(5, n_envs=64)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    cap = 5 * n + 13
    row = B + 5 + A + 2
    ring = torch.zeros(cap * row, device="cuda")
    s.ring_attach(ring, cap)
    ns = 777
    rows = torch.full((ns, row), -7.0, device="cuda")
    nxt = torch.full((ns, B + 5), -7.0, device="cuda")
    s.ring_sample(5, rows, nxt)
    torch.cuda.synchronize()
    assert float(rows.min()) == -7.0 and float(nxt.max()) == -7.0        # empty ring: nothing written
    steps = 8
    actions = torch.from_numpy(W.action_tape(wl, steps, 4)).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, steps + 1, 4).view(np.int64)).cuda()
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
    for t in range(steps):
        buf.mask.zero_()
        s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
        total = (t + 1) * n
        for seed, with_next in ((1000 + t, True), (2**63 + 12345 + t, False)):
            s.ring_sample(seed, rows, nxt if with_next else None)
            torch.cuda.synchronize()
            ring_np = ring.cpu().numpy().reshape(cap, row)
            er, en, slots = oracle.ring_sample(ring_np, cap, total, n, B, A, seed, ns)
            assert not set(((total % cap + np.arange(n)) % cap).tolist()) & set(slots.tolist())   # no pending row
            assert np.array_equal(rows.cpu().numpy(), er)
            if with_next:
                assert np.array_equal(nxt.cpu().numpy(), en)
    assert steps * n > cap                                                 # the ring has wrapped
    s.close(); r.close(); m.close()


def test_terminal_observations_in_replay(pu):
    # PAPER.md:86 "Observations before reset are retained as next observations in replay, while reset observations are
    # returned to the collector."  fn_ring_attach_terminal keeps the observation a step leaves behind for the envs that
    # are then reset; fn_ring_sample hands it out as the next observation of their done rows and marks truncated rows
    # whose observation is gone with code 3.  Against the oracle (fno_terminal_save / fno_ring_sample, pinned by a
    # dictionary model) fed with the GPU's own ring before every reset: sampled rows and next observations bit for
    # bit -- done list and explicit mask, prepared resets (C2-size batch) and plain ones, a reset called twice, envs
    # reset without a finished episode, a terminal ring that wraps, and no terminal ring at all.
    import torch
    import oracle
    from harness import workloads as W
    for cfg, n, steps, t_rows, announce in ((5, 64, 14, 70, False), (2, 4096, 6, 4096 + 100, True)):
        wl = W.make_workload(cfg, n_envs=n)
        wl.forced_reset_frac = 0.06                              # truncated rows (done code 2)
        wl.max_episode_steps = 5                                 # ... and time-outs
        B, A = wl.n_beams, wl.action_dim
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, A)
        cap = 5 * n + 13
        row = B + 5 + A + 2
        ring = torch.zeros(cap * row, device="cuda")
        term = torch.zeros(t_rows * (B + 5), device="cuda")
        s.ring_attach(ring, cap)
        s.ring_attach_terminal(term, t_rows)
        store = oracle.TerminalStore(cap, t_rows, B)
        ns = 999
        rows = torch.empty(ns, row, device="cuda")
        nxt = torch.empty(ns, B + 5, device="cuda")
        actions = torch.from_numpy(W.action_tape(wl, steps, 4)).cuda()
        seeds = torch.from_numpy(W.seed_tape(wl, steps + 2, 4).view(np.int64)).cuda()
        forced = torch.from_numpy(W.forced_reset_tape(wl, steps, 4)).cuda()
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)      # (no row completed yet: nothing to keep)
        codes = set()
        for t in range(steps):
            buf.mask.copy_(forced[t])
            if announce:
                s.prepare_reset(seeds[t + 1])
            s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            torch.cuda.synchronize()
            total = (t + 1) * n
            store.step_ended()
            done = buf.mask.cpu().numpy().copy()
            lst = np.nonzero(done)[0]
            use_mask = t % 3 == 1
            if use_mask and t % 2 == 1:
                done[(t * 7) % n] = 1                            # an env reset although its episode may go on
                lst = np.nonzero(done)[0]
            ring_np = ring.cpu().numpy().reshape(cap, row)
            oracle.terminal_save(ring_np, cap, total, n, B, A, lst, store)
            if use_mask:
                buf.mask.copy_(torch.from_numpy(done))
                s.reset(buf.states, buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
                if t % 2 == 1:                                   # the same reset again: nothing is kept twice
                    ring_np = ring.cpu().numpy().reshape(cap, row)
                    oracle.terminal_save(ring_np, cap, total, n, B, A, lst, store)
                    s.reset(buf.states, buf.mask, seeds[t + 1], buf.ranges, buf.gobs)
            else:
                s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
            torch.cuda.synchronize()
            ring_np = ring.cpu().numpy().reshape(cap, row)
            s.ring_sample(50 + t, rows, nxt)
            torch.cuda.synchronize()
            er, en, slots = oracle.ring_sample(ring_np, cap, total, n, B, A, 50 + t, ns, store=store)
            assert np.array_equal(rows.cpu().numpy(), er), f"config {cfg} step {t}: sampled rows"
            assert np.array_equal(nxt.cpu().numpy(), en), f"config {cfg} step {t}: next observations"
            codes |= set(er[:, -1].astype(int).tolist())
            # the kept observation differs from the post-reset one the ring holds (so the test can tell them apart)
            kept = (er[:, -1] == 1) | (er[:, -1] == 2)
            if kept.any():
                assert (en[kept] != ring_np[(slots[kept] + n) % cap, :B + 5]).any(axis=1).mean() > 0.5
        assert {0, 1, 2} <= codes and (3 in codes or t_rows > 4000), codes
        # no terminal ring: every truncated row is marked 3, next observations are the next rows'
        s.ring_attach_terminal(None, 0)
        s.ring_sample(7, rows, nxt)
        torch.cuda.synchronize()
        er, en, slots = oracle.ring_sample(ring_np, cap, total, n, B, A, 7, ns)
        assert np.array_equal(rows.cpu().numpy(), er) and np.array_equal(nxt.cpu().numpy(), en)
        assert not (er[:, -1] == 2).any()
        with pytest.raises(fn_error()):
            s.ring_attach_terminal(term, n - 1)
        s.close(); r.close(); m.close()


def fn_error():
    import paper_2606_15846_b200 as fn
    return fn.FlashNavError


def test_acceleration_limits(pu):
    # NEXT-3 (reading G2): command limited to the previous applied velocity +- a_max dt.
    from harness import workloads as W
    for cfg, acc in ((2, (1.0, np.inf, 3.0)), (3, (2.0, 1.5, 4.0))):
        wl = W.make_workload(cfg, n_envs=512)
        wl.acc_limits = np.array(acc, np.float32)
        rep = pu.run_parity(wl, steps=12, subset=64, check_every=1)
        print(cfg, rep)


def test_paper_fixed_step_query_as_comparison(pu):
    # NEXT-4: the paper's own range query as a comparison kernel.  "Blockwise" and "All samples"
    # give the same ranges ("All variants used the same ... ray resolution"); a fixed-step march
    # can only hit at or after the exact first hit and, away from corner grazes, within one step of it; and
    # it agrees with the oracle's fp64 march (fno_ranges_fixed_step) except where fp32 sample positions
    # fall on the other side of a cell boundary.
    import torch
    import oracle
    from harness import workloads as W
    wl = W.make_workload(2, n_envs=256)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    seeds = torch.from_numpy(W.seed_tape(wl, 1, 9).view(np.int64)).cuda()
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
    delta = 0.025                                                 # half a cell
    rb = torch.empty_like(buf.ranges)
    ra = torch.empty_like(buf.ranges)
    s.ranges_fixed_step(buf.states, delta, True, rb)
    s.ranges_fixed_step(buf.states, delta, False, ra)
    torch.cuda.synchronize()
    assert torch.equal(rb, ra)
    exact = buf.ranges.cpu().numpy()
    fixed = rb.cpu().numpy()
    assert np.all(fixed >= exact - 1e-3)
    assert np.mean(fixed <= exact + delta + 1e-3) > 0.97          # the rest cut a corner shorter than one step
    st = buf.states.cpu().numpy()
    ref = oracle.ranges_fixed_step(wl.occ, wl.resolution, wl.beam_angles, wl.max_range, delta, st[0], st[1], st[2])
    assert np.mean(np.abs(fixed - ref) <= 1e-5) > 0.98 and np.mean(np.abs(fixed - ref) <= delta + 1e-5) > 0.995
    s.close(); r.close(); m.close()


def test_ring_untouched_by_evaluation_and_capacity_rule(pu):
    # Evaluation steps are not training transitions: ring rows and head stay as they were across
    # fn_eval_begin, evaluation steps and fn_eval_end; training then resumes where it stopped.  And a ring must hold
    # two batches (the completed rows and the pending ones): smaller capacities are refused.
    import torch
    import paper_2606_15846_b200 as fn
    from harness import workloads as W
    wl = W.make_workload(1, n_envs=48)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    row = B + 5 + A + 2
    cap = 5 * n + 3
    ring = torch.zeros(cap * row, device="cuda")
    with pytest.raises(fn.FlashNavError):
        s.ring_attach(ring, 2 * n - 1)
    s.ring_attach(ring, cap)
    actions = torch.from_numpy(W.action_tape(wl, 12, 5)).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, 13, 5).view(np.int64)).cuda()
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
    for t in range(3):
        buf.mask.zero_()
        s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        s.reset(buf.states, None, seeds[t + 1], buf.ranges, buf.gobs)
    torch.cuda.synchronize()
    before = ring.clone()
    rows = torch.zeros(64, row, device="cuda")
    s.ring_sample(3, rows, None)
    keep_states, keep_r, keep_g = buf.states.clone(), buf.ranges.clone(), buf.gobs.clone()
    est, er, eg = buf.states.clone(), torch.empty_like(buf.ranges), torch.empty_like(buf.gobs)
    s.eval_begin(est, n, 6, er, eg)
    for t in range(6):
        buf.mask.zero_()
        s.step(est, actions[3 + t], float(wl.dt), buf.mask, er, buf.col, eg)
        if t == 2:                                                # resets and full recomputes in between are evaluation too
            buf.mask.fill_(1)
            s.reset(est.clone(), buf.mask, seeds[9], torch.empty_like(er), torch.empty_like(eg))
            s.observe_all(est, torch.empty_like(er))
    s.eval_end()
    torch.cuda.synchronize()
    assert torch.equal(ring, before), "evaluation wrote into the replay ring"
    rows2 = torch.zeros(64, row, device="cuda")
    s.ring_sample(3, rows2, None)                                 # same head, same completed rows => same batch
    torch.cuda.synchronize()
    assert torch.equal(rows, rows2)
    s.close(); r.close(); m.close()


def test_two_sims_with_different_maps_side_by_side(pu):
    # the paper's own workflow: a training sim on one map and an evaluation sim on another in one process.
    # The kernels' shared-memory limit is a property of the function, not of a sim: creating the second, smaller sim
    # must not break the launches of the first (and vice versa).
    import torch
    from harness import workloads as W
    wl_a, wl_b = W.make_workload(2, n_envs=300), W.make_workload(1, n_envs=64)
    sims = []
    for wl in (wl_a, wl_b):
        m, r, s = pu.make_sim(wl, wl.n_envs)
        sims.append((wl, m, r, s, pu.Buffers(wl.n_envs, wl.n_beams, wl.action_dim)))
    for rnd in range(3):
        for wl, m, r, s, buf in sims:
            seeds = torch.from_numpy(W.seed_tape(wl, 2, rnd).view(np.int64)).cuda()
            actions = torch.from_numpy(W.action_tape(wl, 1, rnd)).cuda()
            if rnd == 0:
                buf.mask.fill_(1)
                s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
            buf.mask.zero_()
            s.step(buf.states, actions[0], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
            s.reset(buf.states, None, seeds[1], buf.ranges, buf.gobs)
            full = torch.empty_like(buf.ranges)
            s.observe_all(buf.states, full)
            torch.cuda.synchronize()
            assert torch.equal(full, buf.ranges)
    for wl, m, r, s, buf in sims:
        s.close(); r.close(); m.close()


def test_evaluation_mode_completion_masks(pu):
    # NEXT-3: fixed start-goal cases, completion masks that record each case once and freeze it,
    # evaluation step limit.  The bookkeeping is checked against the oracle's fno_eval_update, fed per step
    # with flags recomputed by the oracle at the GPU's poses (teacher forcing, near-ties excluded).
    import torch
    import oracle
    from harness import workloads as W
    wl = W.make_workload(2, n_envs=384)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    n_cases, limit = 300, 25
    m, r, s = pu.make_sim(wl, n)
    buf = pu.Buffers(n, B, A)
    s.bind_aux(None, buf.reward)
    # cases: collision-free starts and goals from the (pinned) reset rule, then fixed
    seeds = torch.from_numpy(W.seed_tape(wl, 1, 21).view(np.int64)).cuda()
    buf.mask.fill_(1)
    s.reset(buf.states, buf.mask, seeds[0], buf.ranges, buf.gobs)
    buf.states[3:6] = 0.37                                        # eval_begin must zero the velocities
    s.eval_begin(buf.states, n_cases, limit, buf.ranges, buf.gobs)
    torch.cuda.synchronize()
    st0 = buf.states.cpu().numpy()
    assert np.all(st0[3:6] == 0)
    o, steps, ret, running = s.eval_result()
    assert running == n_cases and np.all(o[:n_cases] == 0) and np.all(o[n_cases:] == 4) and np.all(steps == 0)
    og = oracle.goal_obs(st0[0], st0[1], st0[2], st0[6], st0[7])
    assert np.allclose(buf.gobs.cpu().numpy()[0], og[0], atol=1e-5)
    actions = torch.from_numpy(W.action_tape(wl, limit + 3, 8)).cuda()
    e_out = o.copy(); e_steps = np.zeros(n, np.int32); e_ret = np.zeros(n, np.float32)
    amb_any = np.zeros(n, bool)
    for t in range(limit + 3):
        pre = buf.states.cpu().numpy()
        pre_r = buf.ranges.clone()
        o_before = s.eval_result()[0]
        buf.mask.zero_()
        s.step(buf.states, actions[t], float(wl.dt), buf.mask, buf.ranges, buf.col, buf.gobs)
        torch.cuda.synchronize()
        post = buf.states.cpu().numpy()
        done = buf.mask.cpu().numpy()
        rew = buf.reward.cpu().numpy()
        frozen = o_before != 0
        # completed cases (and inactive slots) are frozen: nothing moves, no reward, not done again
        assert np.array_equal(post[:, frozen], pre[:, frozen]) and np.all(done[frozen] == 0) and np.all(rew[frozen] == 0)
        assert torch.equal(buf.ranges[torch.from_numpy(frozen).cuda()], pre_r[torch.from_numpy(frozen).cuda()])
        # oracle flags at the GPU's poses for the running cases
        flag, camb = oracle.collision(wl.occ, wl.resolution, wl.footprint, post[0], post[1], post[2])
        amb_any |= (camb != 0) & ~frozen
        gcol = buf.col.cpu().numpy()
        okc = (camb == 0) & ~frozen
        assert np.array_equal(gcol[okc], flag[okc])
        d_new = buf.gobs.cpu().numpy()[0]
        _, ep_after = s.episode_state()
        oracle.eval_update(gcol, d_new, float(wl.goal_tol), ep_after, limit, rew, e_out, e_steps, e_ret)
        o_now, steps_now, ret_now, running = s.eval_result()
        assert np.array_equal(o_now, e_out) and np.array_equal(steps_now[e_out != 0], e_steps[e_out != 0])
        assert np.allclose(ret_now, e_ret, atol=1e-4)
        assert np.array_equal(done != 0, (o_now != 0) & (o_before == 0))      # done exactly on the completing step
        if running == 0:
            break
    assert running == 0 and t + 1 <= limit                       # the batch ends at the step limit at the latest
    assert set(np.unique(e_out[:n_cases])) <= {1, 2, 3} and (e_out[:n_cases] == 3).any() and (e_out[:n_cases] == 2).any()
    assert amb_any.sum() <= 2
    s.eval_end()
    s.close(); r.close(); m.close()


def test_union_of_polygons_footprints(pu):
    # NEXT-3: footprints that are unions of polygons -- the L of config 3 as two
    # rectangles, a dumbbell of two disjoint squares, a plus sign of two overlapping bars -- through the
    # whole step (collision, reset with its sample pre-test, goal obs, beams) and the clearance features.
    import torch
    import oracle
    from harness import workloads as W

    def rect(cx, cy, lx, ly):
        return (W.footprint_rect(lx, ly) + np.array([cx, cy], np.float32)).astype(np.float32)
    shapes = {
        "L": (np.concatenate([rect(0.0, -0.15, 0.8, 0.3), rect(-0.2, 0.15, 0.4, 0.3)]), [4, 4], 3),
        "dumbbell": (np.concatenate([rect(-0.3, 0.0, 0.2, 0.2), rect(0.3, 0.0, 0.2, 0.2)]), [4, 4], 2),
        "plus": (np.concatenate([rect(0, 0, 0.6, 0.16), rect(0, 0, 0.16, 0.6), W.footprint_ngon(0.12, 8)]), [4, 4, 8], 1),
    }
    for name, (fp, comp, cfg) in shapes.items():
        wl = W.make_workload(cfg, n_envs=384)
        wl.footprint, wl.components = fp, comp
        rep = pu.run_parity(wl, steps=10, subset=48, check_every=2)
        print(name, rep)
        assert rep.c["collisions"] > 0 and rep.c["resets"] > 384
        # clearance features of the union
        n, B = 64, wl.n_beams
        wl.n_envs = n
        m, r, s = pu.make_sim(wl, n)
        buf = pu.Buffers(n, B, wl.action_dim)
        z = torch.zeros(n, 18, device="cuda")
        s.bind_features(18, z)
        buf.mask.fill_(1)
        s.reset(buf.states, buf.mask, torch.from_numpy(W.seed_tape(wl, 1, 1)[0].view(np.int64)).cuda(), buf.ranges, buf.gobs)
        torch.cuda.synchronize()
        ze = oracle.clearance_features(fp, wl.beam_angles, wl.max_range, 18, buf.ranges.cpu().numpy(), components=comp)
        assert np.abs(z.cpu().numpy() - ze).max() <= 1e-4, name
        s.close(); r.close(); m.close()
