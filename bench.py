#!/usr/bin/env python
"""bench.py -- env-steps/s and rays/s of the FlashNav simulator step on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch: fn_step (clip + motion, footprint collision,
goal obs / reward / done, beam casting for all envs) followed by fn_reset of the done envs (compaction,
reset, observation recompute for those envs only).  Default workload: BASELINE.json configs[1]
(C2: 512x512 map, 4096 envs, 720 beams over 270 deg, 10 m range, differential drive).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

N > 1 (torchrun): environments are independent, so every rank runs its own batch on its own GPU with no
data-path collective ("scaling": "weak"); value = total env-steps of all ranks / max-over-ranks time.
--impl reference times the CPU oracle (oracle/) on the host cores on a bounded sample of the same
workload; it is a deliberately slow program (parity and the roofline fraction are the headline).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from harness import workloads as W  # noqa: E402

import glob
import re


def read_ncu_capture(cfg, kernel_pat):
    """Per-launch counters of the dominant kernel from the NEWEST committed ncu --set full summary of this config
    (profiles/r*_beam_kernels_full_c<cfg>.txt), read at run time: never a pasted constant.  Returns None when no
    summary exists or the kernel is not in it.  The file names the command and the commit it was taken at."""
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_beam_kernels_full_c{cfg}.txt")))
    if not files:
        return None
    path = files[-1]
    txt = open(path).read()
    commit = re.search(r"^# commit[: ]+(\S+)", txt, re.M)
    out = None
    for sec in txt.split("\n== ")[1:]:
        if not re.search(kernel_pat, sec.split("\n", 1)[0]):
            continue
        def val(name, scale_units=False):
            mm = re.search(rf"^{re.escape(name)}\s+([0-9.eE+-]+)\s*(\S*)", sec, re.M)
            if not mm:
                return None
            v = float(mm.group(1))
            if scale_units:
                v *= {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(mm.group(2), 1)
            return v
        rd, wr = val("dram__bytes_read.sum", True), val("dram__bytes_write.sum", True)
        out = {"dram_bytes": None if rd is None or wr is None else rd + wr,
               "warp_inst": val("smsp__inst_executed.sum"),
               "lanes": val("smsp__thread_inst_executed_per_inst_executed.ratio"),
               "source": os.path.relpath(path, ROOT) + " (dram__bytes_read.sum + dram__bytes_write.sum, per launch)",
               "commit": commit.group(1) if commit else None, "kernel": sec.split("\n", 1)[0].strip()}
        break
    return out


METRIC = "env_steps_per_s"
UNIT = "env-steps/s"


def workload_name(cfg):
    return f"BASELINE.json configs[{cfg - 1}]" if cfg <= 5 else "extra: C1's robot on C2's map (N sweep, PAPER.md:175 Fig. 5)"


def config_dict(cfg, wl):
    """The workload, in the same words in both arms (launch choices of our arm go under "launch")."""
    return {"workload": workload_name(cfg), "name": wl.name, "n_envs_per_gpu": int(wl.n_envs), "beams": int(wl.n_beams),
            "map": list(wl.occ.shape), "max_range_m": float(wl.max_range), "dt": float(wl.dt),
            "ring": bool(wl.ring_capacity), "config_steps": int(wl.steps)}


# --------------------------------------------------------------------------- reference arm = the oracle
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    wl = W.make_workload(args.config, n_envs=args.envs or None)
    cfg_d = config_dict(args.config, wl)
    n = min(wl.n_envs, args.ref_envs)
    wl.n_envs = n
    st = np.zeros((8, n), np.float32)
    dp = np.zeros(n, np.float32)
    ep = np.zeros(n, np.int32)
    seeds = W.seed_tape(wl, args.steps + args.warmup + 1)
    act = W.action_tape(wl, args.steps + args.warmup)
    oracle.reset(wl.occ, wl.resolution, wl.footprint, wl.regions, wl.goal_dist_min, wl.goal_dist_max,
                 np.ones(n, np.uint8), seeds[0], st, dp, ep)

    def one(t):
        out = oracle.step(wl, st, act[t], None, dp, ep, want_hit=False)
        done = out["done"]
        if done.any():
            oracle.reset(wl.occ, wl.resolution, wl.footprint, wl.regions, wl.goal_dist_min, wl.goal_dist_max,
                         done, seeds[t + 1], st, dp, ep)
            idx = np.nonzero(done)[0]
            oracle.ranges(wl.occ, wl.resolution, wl.beam_angles, wl.max_range, st[0, idx], st[1, idx], st[2, idx], eps=0.0)
        return int(done.sum())

    for t in range(args.warmup):
        one(t)
    t0 = time.perf_counter()
    resets = 0
    for t in range(args.warmup, args.warmup + args.steps):
        resets += one(t)
    dt = time.perf_counter() - t0
    v = n * args.steps / dt
    sample = f"{n} of {W.make_workload(args.config, n_envs=args.envs or None).n_envs} envs x {args.steps} steps, single thread"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg_d,
            "rays_per_s": (n * args.steps + resets) * wl.n_beams / dt,
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- clocks sampling
class ClockSampler:
    """Polls NVML from a thread during the timed region: SM clock, max SM clock, clock-event reasons."""
    BITS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, gpu_index, period_s=0.002):
        self.idx, self.period = gpu_index, period_s
        self.sm, self.reasons, self.smax = [], set(), None
        self._stop = threading.Event()
        self.th = None
        self.err = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.idx]) if vis and vis.split(",")[0].isdigit() else self.idx
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.th = threading.Thread(target=self._run, daemon=True)
            self.th.start()
        except Exception as e:          # noqa: BLE001
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:       # noqa: BLE001
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.BITS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception as e:      # noqa: BLE001
                self.err = repr(e)
                return
            time.sleep(self.period)

    def stop(self):
        self._stop.set()
        if self.th is not None:
            self.th.join(timeout=2)
        out = {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.smax,
               "reasons": sorted(self.reasons), "samples": len(self.sm)}
        if self.err:
            out["error"] = self.err
        return out


# --------------------------------------------------------------------------- algorithmic bytes per beam
def algorithmic_bytes_per_beam(wl, states_np, n_sample=128, seed=0):
    """A_ray from the ORACLE's exact path, for the word shape the kernel uses:
    one 32-bit word for the origin-cell test + one 64-bit window per line the beam visits along its minor
    axis up to and including the hit line (+1 window per further 32 cells of a span longer than 32 cells)."""
    import oracle
    n = states_np.shape[1]
    idx = np.random.default_rng(seed).choice(n, min(n, n_sample), replace=False)
    x, y, psi = states_np[0, idx], states_np[1, idx], states_np[2, idx]
    r, hit, amb = oracle.ranges(wl.occ, wl.resolution, wl.beam_angles, wl.max_range, x, y, psi, eps=0.0)
    rho = np.float64(wl.resolution)
    phi = psi[:, None].astype(np.float64) + wl.beam_angles[None, :].astype(np.float64)
    dx, dy = np.cos(phi), np.sin(phi)
    t = r.astype(np.float64) / rho
    ox, oy = x[:, None] / rho, y[:, None] / rho
    ex, ey = ox + t * dx, oy + t * dy
    # entry point of the hit cell lies on its boundary: nudge inside along the beam to name the cell
    ex, ey = ex + 1e-9 * dx, ey + 1e-9 * dy
    major_x = np.abs(dx) >= np.abs(dy)
    lines = np.where(major_x, np.abs(np.floor(ey) - np.floor(oy)), np.abs(np.floor(ex) - np.floor(ox))) + 1
    slope = np.maximum(np.abs(dx), np.abs(dy)) / np.maximum(np.minimum(np.abs(dx), np.abs(dy)), 1e-12)
    extra = np.where(slope > 32, np.floor(np.where(major_x, np.abs(ex - ox), np.abs(ey - oy)) / 32), 0)
    windows = lines + extra
    return float(4.0 + 8.0 * windows.mean()), float(windows.mean())


# --------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_15846_b200 as fn

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fn.load_library()

    wl = W.make_workload(args.config, n_envs=args.envs or None)
    n, B, A = wl.n_envs, wl.n_beams, wl.action_dim
    # protocol of PAPER.md:175: precomputed actions, 100 warm-up steps, the config's own step count timed with a
    # sync at both ends, 5 repetitions, median and IQR (flags override the counts)
    K = args.steps if args.steps > 0 else int(wl.steps)
    Wm = args.warmup if args.warmup >= 0 else 100
    Wm = max(Wm, 3)
    R = max(1, args.reps)
    tape_len = min(K + Wm, 256)
    actions = torch.from_numpy(W.action_tape(wl, tape_len, seed=wl.seed + 17 * rank)).cuda()
    seeds = torch.from_numpy(W.seed_tape(wl, tape_len + 1, seed=wl.seed + 17 * rank).view(np.int64)).cuda()
    forced = torch.from_numpy(W.forced_reset_tape(wl, tape_len, seed=wl.seed + 17 * rank)).cuda()

    m = fn.Map(wl.occ, float(wl.resolution))
    if wl.regions is not None:
        m.set_regions(wl.regions)
    rb = fn.Robot(wl.footprint, wl.beam_angles, float(wl.max_range), wl.drive, wl.vel_limits)
    sim = fn.Sim(m, rb, n, goal_tol=float(wl.goal_tol), max_episode_steps=wl.max_episode_steps,
                 goal_dist_min=float(wl.goal_dist_min), goal_dist_max=float(wl.goal_dist_max))
    if args.fused_reset >= 0:
        sim.set_fused_reset(args.fused_reset)
    if args.split_step >= 0:
        sim.set_split_step(bool(args.split_step))
    if args.coarse >= 0:
        sim.set_coarse(bool(args.coarse))
    fused_active, split_step = sim.beam_config()["fused_reset"], sim.beam_config()["split_step"]
    coarse_active = sim.beam_config()["coarse"]
    states = torch.zeros(8, n, device="cuda")
    mask = torch.ones(n, dtype=torch.uint8, device="cuda")
    ranges = torch.zeros(n, B, device="cuda")
    col = torch.zeros(n, dtype=torch.uint8, device="cuda")
    gobs = torch.zeros(2, n, device="cuda")
    ring = None
    if wl.ring_capacity and args.ring:
        ring = torch.zeros(wl.ring_capacity * sim.ring_row_floats(), device="cuda")
        sim.ring_attach(ring, wl.ring_capacity)
        if args.terminal:
            # pre-reset observations kept as next observations; an eighth of the ring's rows as entries
            # (C5: 12 % of the envs end per step)
            term_rows = max(n, wl.ring_capacity // 8)
            term = torch.zeros(term_rows * (B + 5), device="cuda")
            sim.ring_attach_terminal(term, term_rows)
    sim.reset(states, mask, seeds[tape_len], ranges, gobs)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def step(t):
        k = t % tape_len
        mask.copy_(forced[k])
        if args.prepare:                                      # the seeds of the reset below, announced before the step
            sim.prepare_reset(seeds[k])
        sim.step(states, actions[k], float(wl.dt), mask, ranges, col, gobs)
        sim.reset(states, None, seeds[k], ranges, gobs)       # mask = None: the envs this step reported done

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for t in range(Wm):
        step(t)
    barrier()
    c0 = sim.counters()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    # ---- timed region: R repetitions of K steps, L2 flushed between steps (outside the per-step events)
    rep_ms, per_step_all = [], []
    for rep in range(R):
        ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        barrier()
        for k in range(K):
            flush.fill_(k & 0xff)
            ev0[k].record()
            step(Wm + rep * K + k)
            ev1[k].record()
        barrier()
        ps = np.array([ev0[k].elapsed_time(ev1[k]) for k in range(K)])
        per_step_all.append(ps)
        rep_ms.append(float(ps.sum()))
    clocks = sampler.stop() if rank == 0 else None
    per_step_ms = np.concatenate(per_step_all)
    c1 = sim.counters()
    # ---- per-kernel durations: the same K steps again with the library's events around each kernel
    # (a separate pass: an event between two kernels keeps the second from starting under the first)
    sim.profile(True)
    for k in range(K):
        flush.fill_(k & 0xff)
        step(Wm + k)
    barrier()
    prof = sim.profile_read()
    sim.profile(False)

    # steady state (no L2 flush, back to back): information only
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record()
    for k in range(K):
        step(Wm + K + k)
    s1.record()
    barrier()
    steady_ms = s0.elapsed_time(s1)

    # the same K steps replayed as ONE CUDA graph (no L2 flush): information only.  fn_step / fn_reset only
    # enqueue kernels and keep their per-step state on the device, so a captured sequence replays.
    graph_ms = None
    if args.graph:
        try:
            cs = torch.cuda.Stream()
            cs.wait_stream(torch.cuda.current_stream())
            g = torch.cuda.CUDAGraph()
            sim.set_stream(cs)
            with torch.cuda.graph(g, stream=cs):
                for k in range(min(K, tape_len)):
                    step(k)
            sim.set_stream(torch.cuda.current_stream())
            reps = max(1, K // min(K, tape_len))
            g.replay()
            barrier()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record()
            for _ in range(reps):
                g.replay()
            g1.record()
            barrier()
            graph_ms = g0.elapsed_time(g1) / (reps * min(K, tape_len))
        except Exception as ex:         # noqa: BLE001
            graph_ms = None
            sys.stderr.write(f"bench.py: graph replay leg skipped: {ex!r}\n")
            sim.set_stream(torch.cuda.current_stream())

    # clearance features (Eq. (3)): the extra kernel when they are bound
    feat = None
    if args.features > 0:
        zbuf = torch.zeros(n, args.features, device="cuda")
        sim.bind_features(args.features, zbuf)
        for k in range(3):
            step(k)
        barrier()
        sim.profile(True)
        for k in range(K):
            flush.fill_(k & 0xff)
            step(Wm + k)
        barrier()
        pf = sim.profile_read()
        sim.profile(False)
        sim.bind_features(args.features, None)
        f_s = pf["features"][0] * 1e-3 / max(1, pf["features"][1])
        feat = {"n_sectors": args.features, "kernel_ms": f_s * 1e3, "kernel_ms_reset_list": pf["features_reset"][0] / max(1, pf["features_reset"][1]),
                "beams_per_s": n * B / f_s, "read_GBps": n * B * 4 / f_s / 1e9,
                "note": "fn::features_kernel over all envs after the beam kernel (ranges read from L2); not in the timed step"}

    # the paper's own fixed-step range query on the same poses (Table III-b):
    # comparison only, information
    paper_query = None
    if args.paper_query:
        delta = float(wl.resolution) * 0.5
        rq = torch.empty_like(ranges)
        ex = torch.empty_like(ranges)
        res = {}
        for name, fnq in (("blockwise", lambda: sim.ranges_fixed_step(states, delta, True, rq)),
                          ("all_samples", lambda: sim.ranges_fixed_step(states, delta, False, rq)),
                          ("exact_traversal", lambda: sim.observe_all(states, ex))):
            fnq()
            barrier()
            tot = 0.0
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for k in range(5):
                flush.fill_(k & 0xff)
                q0.record()
                fnq()
                q1.record()
                torch.cuda.synchronize()
                tot += q0.elapsed_time(q1)
            res[name] = tot / 5
        err = (rq - ex)
        paper_query = {"delta_m": delta, "ms": res, "speedup_exact_vs_blockwise": res["blockwise"] / res["exact_traversal"],
                       "range_error_m": {"mean": float(err.mean()), "max": float(err.max()), "min": float(err.min())},
                       "note": "fn_ranges_fixed_step (the paper's query, fp32 samples every delta) vs fn_observe_all (pose kernel + "
                               "exact traversal) on the same states; all three include the pose kernel"}

    # replay sampling: U x B transitions gathered from the ring (HBM-bound)
    sample = None
    if ring is not None and args.sample_batch > 0:
        ns = args.sample_batch
        rowf = sim.ring_row_floats()
        bufs = [(torch.empty(ns, rowf, device="cuda"), torch.empty(ns, B + 5, device="cuda")) for _ in range(2)]
        for k in range(3):
            sim.ring_sample(k, *bufs[k & 1])
        barrier()
        reps = 20
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tot = 0.0
        for k in range(reps):
            flush.fill_(k & 0xff)
            q0.record()
            sim.ring_sample(100 + k, *bufs[k & 1])               # the paper's two batch buffers, alternating
            q1.record()
            torch.cuda.synchronize()
            tot += q0.elapsed_time(q1)
        s_s = tot * 1e-3 / reps
        nbytes = ns * (rowf + B + 5) * 4 * 2                     # rows + next obs, read + write
        hbm = None
        try:
            hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        except Exception:                                        # noqa: BLE001
            pass
        peak = hbm if hbm else 6650.0
        sample = {"n_samples": ns, "kernel_ms": s_s * 1e3, "transitions_per_s": ns / s_s,
                  "roofline": {"bound": "hbm", "achieved": nbytes / s_s / 1e9, "peak": peak, "unit": "GB/s",
                               "frac": nbytes / s_s / 1e9 / peak,
                               "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if hbm else "guide fallback 6.65 TB/s (of fallback)"},
                  "note": "fn::ring_sample_kernel: rows + next observations, L2 flushed before each call; not in the timed step"}

    tmax = torch.tensor(rep_ms + [steady_ms], device="cuda", dtype=torch.float64)
    rays = torch.tensor([float(c1["rays_cast"] - c0["rays_cast"]), float(c1["envs_reset"] - c0["envs_reset"])],
                        device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)             # a repetition takes as long as its slowest rank
        dist.all_reduce(rays, op=dist.ReduceOp.SUM)
    rep_ms, steady_ms = [float(v) for v in tmax[:R]], float(tmax[R])
    rep_values = np.array([world * n * K / (ms * 1e-3) for ms in rep_ms])
    total_ms = float(np.median(rep_ms))                          # the median repetition
    value = float(np.median(rep_values))
    rays = rays / R                                              # per repetition of K steps

    out = None
    if rank == 0:
        # ---- roofline of the dominant kernel (full-batch beam kernel of fn_step), live CUDA events
        beam_ms, beam_launches = prof["beam_step"]
        env_ms, _ = prof["env_step"]
        reset_ms, _ = prof["reset_path"]
        st_np = states.cpu().numpy()
        a_ray, windows = algorithmic_bytes_per_beam(wl, st_np)
        smem_peak = fn.measure_peak(0)
        l2_peak = fn.measure_peak(2)
        use_smem = sim.beam_config()["smem"]
        peak = smem_peak if use_smem else l2_peak
        beam_s = beam_ms * 1e-3 / max(1, beam_launches)
        achieved = a_ray * n * B / beam_s
        ncu = read_ncu_capture(args.config, r"step_beam_kernel" if split_step else r"(?<!step_)(?<!reset_)beam_kernel")
        if ncu and (ncu["warp_inst"] is None or ncu["lanes"] is None):
            ncu = None
        sm_hz = (clocks or {}).get("sm_mhz") or 1965.0
        issue_peak = 148 * 4 * sm_hz * 1e6                      # warp instructions / s: 1 per scheduler per clock
        roofline = {"bound": "smem" if use_smem else "l2", "kernel": ("fn::step_beam_kernel (fn_step, all envs: beams + collision / goal / reward / done of the split step)"
                               if split_step else "fn::beam_kernel (fn_step, all envs)"),
                    "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "GB/s", "frac": achieved / peak,
                    "peak_source": "fn_measure_peak in this run (conflict-free ld.shared / L2-resident ld.global.nc)",
                    "algorithmic_bytes_per_beam": a_ray, "windows_per_beam": windows,
                    "kernel_ms": beam_s * 1e3, "share_of_step": beam_ms / (env_ms + beam_ms + reset_ms),
                    "traffic": ncu["dram_bytes"] if ncu else None,
                    "traffic_source": ncu["source"] if ncu else None,
                    "traffic_commit": ncu["commit"] if ncu else None,
                    "smem_peak_GBps": smem_peak / 1e9, "l2_peak_GBps": l2_peak / 1e9,
                    "beams_per_s": n * B / beam_s,
                    "issue": None if not ncu else {
                        "note": "the kernel is issue/latency bound (DESIGN.md 6.1): warp instructions per launch from the "
                                "ncu capture, duration live", "warp_inst_per_launch": ncu["warp_inst"],
                        "achieved_Ginst_per_s": ncu["warp_inst"] / beam_s / 1e9, "peak_Ginst_per_s": issue_peak / 1e9,
                        "frac": ncu["warp_inst"] / beam_s / issue_peak, "lanes_active_of_32": ncu["lanes"]}}
        # ---- oracle on the host cores, bounded sample of the same workload
        cpu = None
        if not args.no_cpu:
            import oracle
            oracle.build()
            ns = min(n, args.ref_envs)
            st = np.ascontiguousarray(st_np[:, :ns])
            dp = np.zeros(ns, np.float32)
            ep = np.zeros(ns, np.int32)
            wl_s = W.make_workload(args.config, n_envs=ns)
            act = W.action_tape(wl_s, args.cpu_steps)
            t0 = time.perf_counter()
            for t in range(args.cpu_steps):
                oracle.step(wl_s, st, act[t], None, dp, ep, want_hit=False)
            dtc = time.perf_counter() - t0
            cpu = {"value": ns * args.cpu_steps / dtc, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": f"{ns} of {n} envs x {args.cpu_steps} steps (fn_step part only, no resets), single thread",
                   "rays_per_s": ns * args.cpu_steps * B / dtc, "host_cores_available": os.cpu_count()}
            # the same unmodified oracle, env-sharded over all host cores: one thread per
            # contiguous env range, each thread calls the single-threaded C oracle (ctypes drops the GIL)
            from concurrent.futures import ThreadPoolExecutor
            nc = max(1, min(os.cpu_count() or 1, ns))
            cuts = [ns * i // nc for i in range(nc + 1)]
            shards = [(np.ascontiguousarray(st_np[:, a:b]), np.zeros(b - a, np.float32), np.zeros(b - a, np.int32),
                       np.ascontiguousarray(act[:, a:b])) for a, b in zip(cuts[:-1], cuts[1:])]

            def run_shard(sh):
                for t in range(args.cpu_steps):
                    oracle.step(wl_s, sh[0], sh[3][t], None, sh[1], sh[2], want_hit=False)
            with ThreadPoolExecutor(nc) as ex:
                t0 = time.perf_counter()
                list(ex.map(run_shard, shards))
                dta = time.perf_counter() - t0
            cpu["all_cores"] = {"value": ns * args.cpu_steps / dta, "unit": UNIT, "cores": nc,
                                "note": "same sample, contiguous env ranges over threads, oracle unmodified"}
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
               "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f64", "data": "synthetic",
               "config": config_dict(args.config, wl),
               "launch": {"l2": "flushed between timed steps", "ring_attached": bool(ring is not None),
                          "terminal_observations_kept": bool(ring is not None and args.terminal),
                          "fused_reset": bool(fused_active), "split_step": bool(split_step), "coarse_level": bool(coarse_active),
                          "prepared_resets": float(c1["resets_prepared"] - c0["resets_prepared"]) / max(1, c1["envs_reset"] - c0["envs_reset"])},
               "protocol": {"repetitions": R, "value": "median over repetitions", "value_iqr": [float(np.percentile(rep_values, 25)), float(np.percentile(rep_values, 75))],
                            "values": [float(v) for v in rep_values], "ms_per_step_iqr": [float(np.percentile(rep_ms, 25)) / K, float(np.percentile(rep_ms, 75)) / K],
                            "note": "PAPER.md:175: warm-up, then K timed steps between syncs, repeated; median and IQR"},
               "rays_per_s": float(rays[0]) / (total_ms * 1e-3),
               "useful_rays_per_s": world * n * B * K / (total_ms * 1e-3),
               "reset_rate_per_step": float(rays[1]) / (world * n * K),
               "steady_state": {"value": world * n * K / (steady_ms * 1e-3), "unit": UNIT, "ms_per_step": steady_ms / K,
                                "note": "no L2 flush, K steps back to back"},
               "graph_replay": None if graph_ms is None else {
                   "value": world * n / (graph_ms * 1e-3), "unit": UNIT, "ms_per_step": graph_ms,
                   "note": "the same steps captured once and replayed as a CUDA graph, no L2 flush (rank 0)"},
               "kernel_ms_per_step": {"env_step": env_ms / K, "beam_step": beam_ms / K, "reset_path": reset_ms / K,
                                      "compact": prof["compact"][0] / K, "reset": prof["reset"][0] / K,
                                      "beam_reset": prof["beam_reset"][0] / K},
               "ms_per_step_p50": float(np.median(per_step_ms)), "ms_per_step_p90": float(np.percentile(per_step_ms, 90)),
               "features": feat, "replay_sample": sample, "paper_fixed_step_query": paper_query, "roofline": roofline, "cpu_baseline": cpu, "clocks": clocks,
               # per step: env step (or its motion half), beam kernel, [ring_advance unless split], [terminal_save with a
               # terminal ring], then fn_reset = ONE kernel when the step prepared the resets (prepared_reset_kernel; read
               # off the resets_prepared counter of the timed region, not assumed) or when the fused reset serves the done
               # list, else reset kernel + beam kernel
               "gpu_launches": (2 + (1 if ring is not None and not split_step else 0)
                                + (1 if (c1["resets_prepared"] > c0["resets_prepared"] or fused_active) else 2)
                                + (1 if ring is not None and args.terminal else 0)) * K * R}

    if rank == 0:
        # HBM view of the whole step ("report HBM GB/s separately for C5"): state planes in / out,
        # actions, flags and goal obs, one range row per env, and with a ring its row (obs + action + reward + done)
        per_env = 32 + 24 + 4 * A + 10 + 4 * B + (4 * (B + 5 + A + 2) if ring is not None else 0)
        hbm_peak = None
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        except Exception:                                        # noqa: BLE001
            pass
        pk = hbm_peak if hbm_peak else 6650.0
        ach = per_env * n * world / (total_ms / K * 1e-3) / 1e9
        out["hbm"] = {"bytes_per_env_step": per_env, "achieved": ach, "peak": pk * world, "unit": "GB/s", "frac": ach / (pk * world),
                      "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if hbm_peak else "guide fallback 6.65 TB/s (of fallback)",
                      "note": "algorithmic state / observation / ring bytes of one step over the step time; the reset envs' rows add reset_rate x that"}

    # ---- end to end through the public API with HOST buffers (copies inside the timed region)
    hs = torch.empty(8, n, dtype=torch.float32).pin_memory()
    ha = W.action_tape(wl, 8, seed=3)
    ha_p = [torch.from_numpy(ha[k]).pin_memory() for k in range(8)]
    hseed = [torch.from_numpy(W.seed_tape(wl, 8, seed=3)[k].view(np.int64)).pin_memory() for k in range(8)]
    hm = torch.zeros(n, dtype=torch.uint8).pin_memory()
    hr = torch.empty(n, B, dtype=torch.float32).pin_memory()
    hc = torch.empty(n, dtype=torch.uint8).pin_memory()
    hg = torch.empty(2, n, dtype=torch.float32).pin_memory()
    hs.copy_(states)
    Ke = max(3, min(K, args.e2e_steps)) if args.e2e_steps > 0 else 3
    for k in range(3):
        hm.zero_()
        sim.step_host(hs, ha_p[k % 8], float(wl.dt), hm, hseed[k % 8], hr, hc, hg)
    barrier()
    t0 = time.perf_counter()
    for k in range(Ke):
        hm.zero_()
        sim.step_host(hs, ha_p[k % 8], float(wl.dt), hm, hseed[k % 8], hr, hc, hg)
    barrier()
    e2e_s = time.perf_counter() - t0
    # the same through the pipelined calls (two slots: the copies of step t overlap the kernels of step t + 1; every
    # copy is still inside the timed region, and every step's result is awaited)
    sl = [{"s": torch.empty(8, n).pin_memory(), "r": torch.empty(n, B).pin_memory(), "g": torch.empty(2, n).pin_memory(),
           "m": torch.zeros(n, dtype=torch.uint8).pin_memory(), "c": torch.empty(n, dtype=torch.uint8).pin_memory()} for _ in range(2)]
    def pipe(nsteps, first):
        for k in range(nsteps + 1):
            if k < nsteps:
                b = sl[k & 1]
                b["m"].zero_()
                sim.step_host_begin(k & 1, hs if (k == 0 and first) else None, ha_p[k % 8], float(wl.dt), b["m"], hseed[k % 8],
                                    b["s"], b["r"], b["c"], b["g"])
            if k >= 1:
                sim.step_host_end((k - 1) & 1)
    pipe(3, True)
    barrier()
    t0 = time.perf_counter()
    pipe(Ke, False)
    barrier()
    pipe_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s, pipe_s], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    if rank == 0:
        h2d = 8 * n * 4 + n * A * 4 + n + n * 8
        d2h = 8 * n * 4 + n * B * 4 + 2 * n * 4 + n + n
        d2h_pipe = d2h
        h2d_pipe = n * A * 4 + n + n * 8                         # the states stay on the device between steps
        # e2e.value: since round 2 the PIPELINED public calls (round 1 reported the serial fn_step_host here, which has
        # been e2e.serial since; BASELINE.md and DESIGN.md 10 state the change) -- compare round 1's e2e.value with e2e.serial
        out["e2e"] = {"value": world * n * Ke / float(te[1]), "unit": UNIT, "h2d_bytes_per_step": h2d_pipe, "d2h_bytes_per_step": d2h_pipe,
                      "definition": "pipelined (fn_step_host_begin / _end); round 1's e2e.value is e2e.serial here",
                      "steps": Ke, "note": "fn_step_host_begin / _end over two slots: pinned host buffers; per step H2D of actions, mask "
                                           "and seeds, fn_step + fn_reset, D2H of states, ranges, flags and goal obs on a copy stream "
                                           "that overlaps the next step's kernels; every step's outputs are awaited",
                      "serial": {"value": world * n * Ke / float(te[0]), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                                 "note": "fn_step_host: H2D + fn_step + fn_reset + D2H + sync per step"}}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="timed steps per repetition (0 = the config's own count, PAPER.md:175)")
    ap.add_argument("--warmup", type=int, default=-1, help="warm-up steps (-1 = 100, PAPER.md:175)")
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the timed block (median and IQR are reported)")
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--envs", type=int, default=0, help="override the config's env count per GPU (0 = the config's own)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-envs", type=int, default=4096, help="oracle sample size (envs)")
    ap.add_argument("--cpu-steps", type=int, default=8, help="oracle steps in the cpu_baseline leg")
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--sample-batch", type=int, default=65536, help="U x B of the replay-sampling leg (configs with a ring; 0 = skip)")
    ap.add_argument("--paper-query", type=int, default=1, help="also time the paper's fixed-step range query (information only)")
    ap.add_argument("--features", type=int, default=36, help="sectors of the clearance-feature leg (0 = skip; information only)")
    ap.add_argument("--prepare", type=int, default=1, help="announce each step's reset seeds before the step (fn_sim_prepare_reset)")
    ap.add_argument("--graph", type=int, default=1, help="also time a CUDA-graph replay of the steps (information only)")
    ap.add_argument("--fused-reset", type=int, default=-1, choices=[-1, 0, 1],
                    help="fn_reset(done list) as one fused kernel (1) or two kernels (0); -1 = the library's default")
    ap.add_argument("--split-step", type=int, default=-1, choices=[-1, 0, 1],
                    help="fn_step with the env step split around the beam kernel (1) or one env-step kernel (0); -1 = the library's default")
    ap.add_argument("--coarse", type=int, default=-1, choices=[-1, 0, 1],
                    help="coarse level in the production beam kernels: -1 = the library's choice")
    ap.add_argument("--ring", type=int, default=1, help="attach the replay ring when the config has one (C5)")
    ap.add_argument("--terminal", type=int, default=1, help="with the ring: keep pre-reset observations (fn_ring_attach_terminal)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started by hand without torchrun: launch the ranks ourselves (one process per GPU, replicas only -- there is
        # no per-step collective; NCCL serves the barrier and the max over ranks of the timing)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.impl == "reference":
        # the counts the caller gave are honoured (same accounting as our arm); without flags a bounded sample:
        # a C2 step takes ~0.9 s on one core
        if args.steps <= 0:
            args.steps = 8
        if args.warmup < 0:
            args.warmup = 1
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
