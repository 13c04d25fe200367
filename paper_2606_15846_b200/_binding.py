"""ctypes binding of libflashnav.so -- same names as include/flashnav.h, marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_DIR, "libflashnav.so")
_lib = None

DRIVE_DIFF, DRIVE_OMNI = 0, 1
N_COUNTERS = 8
COUNTER_NAMES = ("rays_cast", "map_words_loaded", "envs_reset", "reset_failures", "nonfinite_actions",
                 "env_steps", "oob_window_loads", "resets_prepared")

EXPORTED_SYMBOLS = (
    "fn_map_create", "fn_map_set_regions", "fn_map_destroy", "fn_robot_create", "fn_robot_create_union", "fn_robot_set_sensor", "fn_robot_add_sensor", "fn_robot_set_acc_limits",
    "fn_robot_destroy", "fn_task_default", "fn_sim_create", "fn_sim_destroy", "fn_sim_set_stream", "fn_step", "fn_reset",
    "fn_sim_bind_aux", "fn_sim_bind_features", "fn_ring_attach", "fn_ring_attach_terminal", "fn_ring_sample", "fn_ranges_fixed_step", "fn_eval_begin", "fn_eval_result", "fn_eval_end", "fn_observe_all", "fn_observe_noalloc", "fn_get_counters", "fn_sim_count_words",
    "fn_sim_episode_state", "fn_sim_beam_config", "fn_sim_set_fused_reset", "fn_sim_set_split_step", "fn_sim_set_coarse", "fn_sim_prepare_reset", "fn_sim_profile", "fn_sim_profile_read", "fn_step_host", "fn_step_host_begin", "fn_step_host_end", "fn_measure_peak", "fn_last_error", "fn_version")


class FlashNavError(RuntimeError):
    pass


class _Task(C.Structure):
    _fields_ = [("goal_tol_m", C.c_float), ("max_episode_steps", C.c_int), ("goal_dist_min_m", C.c_float),
                ("goal_dist_max_m", C.c_float), ("r_success", C.c_float), ("r_collision", C.c_float),
                ("c_progress", C.c_float)]


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """Loads libflashnav.so (built in-tree by paper_2606_15846_b200/build.py). Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise FlashNavError(f"{_LIB_PATH} is missing: run `python -m paper_2606_15846_b200.build` "
                            "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, f32, u64 = C.c_void_p, C.c_int, C.c_float, C.c_uint64
    sig = {
        "fn_map_create": [vp, i32, i32, f32, C.POINTER(vp)],
        "fn_map_set_regions": [vp, i32, vp],
        "fn_map_destroy": [vp],
        "fn_robot_create": [vp, i32, vp, i32, f32, i32, vp, C.POINTER(vp)],
        "fn_robot_create_union": [vp, vp, i32, vp, i32, f32, i32, vp, C.POINTER(vp)],
        "fn_robot_set_sensor": [vp, f32, f32, f32],
        "fn_robot_add_sensor": [vp, vp, i32, f32, f32, f32, f32],
        "fn_robot_set_acc_limits": [vp, vp],
        "fn_robot_destroy": [vp],
        "fn_sim_create": [vp, vp, i32, C.POINTER(_Task), vp, C.POINTER(vp)],
        "fn_sim_destroy": [vp],
        "fn_sim_set_stream": [vp, vp],
        "fn_step": [vp, vp, vp, f32, vp, vp, vp, vp],
        "fn_reset": [vp, vp, vp, vp, vp, vp],
        "fn_sim_bind_aux": [vp, vp, vp],
        "fn_sim_bind_features": [vp, i32, vp],
        "fn_ring_attach": [vp, vp, u64],
        "fn_ring_attach_terminal": [vp, vp, u64],
        "fn_ring_sample": [vp, u64, i32, vp, vp],
        "fn_observe_all": [vp, vp, vp, vp],
        "fn_observe_noalloc": [vp, vp, i32, vp, vp, vp, vp],
        "fn_eval_begin": [vp, vp, i32, i32, vp, vp],
        "fn_eval_result": [vp, vp, vp, vp, vp],
        "fn_eval_end": [vp],
        "fn_ranges_fixed_step": [vp, vp, f32, i32, vp],
        "fn_get_counters": [vp, vp],
        "fn_sim_count_words": [vp, i32],
        "fn_sim_episode_state": [vp, vp, vp],
        "fn_sim_beam_config": [vp, vp],
        "fn_sim_set_fused_reset": [vp, i32, vp],
        "fn_sim_set_split_step": [vp, i32, vp],
        "fn_sim_set_coarse": [vp, i32, vp],
        "fn_sim_prepare_reset": [vp, vp],
        "fn_sim_profile": [vp, i32],
        "fn_sim_profile_read": [vp, vp, vp],
        "fn_step_host": [vp, vp, vp, f32, vp, vp, vp, vp, vp],
        "fn_step_host_begin": [vp, i32, vp, vp, f32, vp, vp, vp, vp, vp, vp],
        "fn_step_host_end": [vp, i32],
        "fn_measure_peak": [i32, vp, C.POINTER(C.c_double)],
    }
    for name, argtypes in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = argtypes
        fn.restype = i32
    lib.fn_task_default.argtypes = [C.POINTER(_Task)]
    lib.fn_task_default.restype = None
    lib.fn_last_error.restype = C.c_char_p
    lib.fn_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load_library().fn_last_error().decode("utf-8", "replace")
        raise FlashNavError(f"{what} failed ({rc}): {msg}")


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dev_ptr(t, dtype, numel, name):
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise FlashNavError(f"{name}: expected a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise FlashNavError(f"{name}: expected contiguous {dtype} with {numel} elements, got {t.dtype} "
                            f"{tuple(t.shape)} contiguous={t.is_contiguous()}")
    return C.c_void_p(t.data_ptr())


class Map:
    """fn_map: a shared occupancy bitmap (uint8 [H, W], != 0 occupied)."""

    def __init__(self, bitmap: np.ndarray, resolution: float):
        lib = load_library()
        bm = np.ascontiguousarray(bitmap, np.uint8)
        if bm.ndim != 2:
            raise FlashNavError("bitmap must be [H, W]")
        self.H, self.W = int(bm.shape[0]), int(bm.shape[1])
        self.resolution = float(np.float32(resolution))
        h = C.c_void_p()
        _check(lib.fn_map_create(_np_ptr(bm), self.H, self.W, C.c_float(resolution), C.byref(h)), "fn_map_create")
        self._h = h

    def set_regions(self, rects):
        n = 0 if rects is None else int(len(rects))
        arr = None if n == 0 else np.ascontiguousarray(rects, np.int32).reshape(n, 4)
        _check(load_library().fn_map_set_regions(self._h, n, None if arr is None else _np_ptr(arr)), "fn_map_set_regions")

    def close(self):
        if getattr(self, "_h", None):
            load_library().fn_map_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Robot:
    """fn_robot: footprint polygon [V,2], beam angles [B], max range, drive type, velocity limits [6]."""

    def __init__(self, footprint, beam_angles, max_range, drive, vel_limits, components=None):
        """components: vertex counts of the polygons whose vertex lists are concatenated in `footprint`
        (a union of polygons); None = one polygon."""
        lib = load_library()
        fp = np.ascontiguousarray(footprint, np.float32).reshape(-1, 2)
        ang = np.ascontiguousarray(beam_angles, np.float32).reshape(-1)
        lim = np.ascontiguousarray(vel_limits, np.float32).reshape(-1)
        if lim.shape[0] != 6:
            raise FlashNavError("vel_limits must have 6 entries")
        self.V, self.B, self.drive = int(fp.shape[0]), int(ang.shape[0]), int(drive)
        self.A = 2 if self.drive == DRIVE_DIFF else 3
        h = C.c_void_p()
        if components is None:
            _check(lib.fn_robot_create(_np_ptr(fp), self.V, _np_ptr(ang), self.B, C.c_float(max_range), self.drive,
                                       _np_ptr(lim), C.byref(h)), "fn_robot_create")
        else:
            comp = np.ascontiguousarray(components, np.int32).reshape(-1)
            if int(comp.sum()) != self.V:
                raise FlashNavError("components must add up to the number of footprint vertices")
            _check(lib.fn_robot_create_union(_np_ptr(fp), _np_ptr(comp), int(comp.shape[0]), _np_ptr(ang), self.B,
                                             C.c_float(max_range), self.drive, _np_ptr(lim), C.byref(h)),
                   "fn_robot_create_union")
        self._h = h

    def set_sensor(self, sx, sy, spsi):
        _check(load_library().fn_robot_set_sensor(self._h, C.c_float(sx), C.c_float(sy), C.c_float(spsi)), "fn_robot_set_sensor")

    def add_sensor(self, beam_angles, max_range, sx, sy, spsi):
        """A further range sensor: own beam table, range and placement; rows grow by its beam count."""
        ang = np.ascontiguousarray(beam_angles, np.float32).reshape(-1)
        _check(load_library().fn_robot_add_sensor(self._h, _np_ptr(ang), int(ang.shape[0]), C.c_float(max_range), C.c_float(sx),
                                                  C.c_float(sy), C.c_float(spsi)), "fn_robot_add_sensor")
        self.B += int(ang.shape[0])

    def set_acc_limits(self, acc):
        a = np.ascontiguousarray(acc, np.float32).reshape(3)
        _check(load_library().fn_robot_set_acc_limits(self._h, _np_ptr(a)), "fn_robot_set_acc_limits")

    def close(self):
        if getattr(self, "_h", None):
            load_library().fn_robot_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Sim:
    """fn_sim: n_envs environments on one Map with one Robot; work goes to torch's current stream at creation."""

    def __init__(self, map_: Map, robot: Robot, n_envs: int, goal_tol=0.3, max_episode_steps=0, goal_dist_min=3.0,
                 goal_dist_max=8.0, r_success=10.0, r_collision=-10.0, c_progress=2.0, stream=None):
        import torch
        lib = load_library()
        if not torch.cuda.is_available():
            raise FlashNavError("no CUDA device: libflashnav has no CPU fallback")
        self.map, self.robot, self.n = map_, robot, int(n_envs)
        t = _Task(goal_tol, int(max_episode_steps), goal_dist_min, goal_dist_max, r_success, r_collision, c_progress)
        self._stream = torch.cuda.current_stream() if stream is None else stream
        h = C.c_void_p()
        _check(lib.fn_sim_create(map_._h, robot._h, self.n, C.byref(t), C.c_void_p(self._stream.cuda_stream), C.byref(h)),
               "fn_sim_create")
        self._h = h
        self._keep = []

    def set_stream(self, stream=None):
        """Later work goes to `stream` (a torch.cuda.Stream; default: torch's current stream)."""
        import torch
        self._stream = torch.cuda.current_stream() if stream is None else stream
        _check(load_library().fn_sim_set_stream(self._h, C.c_void_p(self._stream.cuda_stream)), "fn_sim_set_stream")

    # --- the four calls of the north star ------------------------------------------------------
    def step(self, states, actions, dt, reset_mask, out_ranges, out_collision, out_goal_obs):
        import torch
        n, B, A = self.n, self.robot.B, self.robot.A
        _check(load_library().fn_step(
            self._h, _dev_ptr(states, torch.float32, 8 * n, "states"), _dev_ptr(actions, torch.float32, n * A, "actions"),
            C.c_float(dt), _dev_ptr(reset_mask, torch.uint8, n, "reset_mask"),
            _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges"), _dev_ptr(out_collision, torch.uint8, n, "out_collision"),
            _dev_ptr(out_goal_obs, torch.float32, 2 * n, "out_goal_obs")), "fn_step")

    def reset(self, states, mask, seeds, out_ranges, out_goal_obs):
        """mask = None: the envs the preceding step() reported done (no mask scan)."""
        import torch
        n, B = self.n, self.robot.B
        if seeds.dtype not in (torch.int64, torch.uint64):
            raise FlashNavError("seeds must be a 64-bit integer tensor")
        _check(load_library().fn_reset(
            self._h, _dev_ptr(states, torch.float32, 8 * n, "states"),
            None if mask is None else _dev_ptr(mask, torch.uint8, n, "mask"),
            _dev_ptr(seeds, seeds.dtype, n, "seeds"), _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges"),
            _dev_ptr(out_goal_obs, torch.float32, 2 * n, "out_goal_obs")), "fn_reset")

    # --- hooks ----------------------------------------------------------------------------------------
    def bind_aux(self, out_hit_cell=None, out_reward=None):
        import torch
        n, B = self.n, self.robot.B
        self._keep = [out_hit_cell, out_reward]
        _check(load_library().fn_sim_bind_aux(self._h, _dev_ptr(out_hit_cell, torch.int32, n * B, "out_hit_cell"),
                                              _dev_ptr(out_reward, torch.float32, n, "out_reward")), "fn_sim_bind_aux")

    def bind_features(self, n_sectors, out_z=None):
        """Clearance features z [N, n_sectors] (Eq. (3)); out_z = None unbinds."""
        import torch
        self._feat = out_z
        _check(load_library().fn_sim_bind_features(
            self._h, int(n_sectors), _dev_ptr(out_z, torch.float32, self.n * int(n_sectors), "out_z")
            if out_z is not None else None), "fn_sim_bind_features")

    def ring_row_floats(self):
        return self.robot.B + 5 + self.robot.A + 2

    def ring_attach(self, ring, capacity):
        import torch
        self._ring = ring
        _check(load_library().fn_ring_attach(self._h, _dev_ptr(ring, torch.float32, capacity * self.ring_row_floats(), "ring")
                                             if ring is not None else None, C.c_uint64(capacity)), "fn_ring_attach")

    def ring_attach_terminal(self, term, rows):
        """Terminal observations: term [rows, B + 5] f32 keeps the pre-reset observation of done rows;
        ring_sample returns it as their next observation.  After ring_attach; None detaches."""
        import torch
        self._term = term
        _check(load_library().fn_ring_attach_terminal(
            self._h, _dev_ptr(term, torch.float32, rows * (self.robot.B + 5), "term") if term is not None else None,
            C.c_uint64(rows)), "fn_ring_attach_terminal")

    def ring_sample(self, seed, out_rows, out_next_obs=None):
        """Uniform replay batch: out_rows [n, row] (, out_next_obs [n, B + 5]) gathered from the ring."""
        import torch
        n = int(out_rows.shape[0])
        _check(load_library().fn_ring_sample(
            self._h, C.c_uint64(int(seed) & ((1 << 64) - 1)), n,
            _dev_ptr(out_rows, torch.float32, n * self.ring_row_floats(), "out_rows"),
            _dev_ptr(out_next_obs, torch.float32, n * (self.robot.B + 5), "out_next_obs")
            if out_next_obs is not None else None), "fn_ring_sample")

    def observe_all(self, states, out_ranges, out_goal_obs=None):
        import torch
        n, B = self.n, self.robot.B
        _check(load_library().fn_observe_all(
            self._h, _dev_ptr(states, torch.float32, 8 * n, "states"), _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges"),
            _dev_ptr(out_goal_obs, torch.float32, 2 * n, "out_goal_obs")), "fn_observe_all")

    def ranges_fixed_step(self, states, delta_m, blockwise, out_ranges):
        """Comparison only: the paper's fixed-step range query, blockwise or all samples."""
        import torch
        n, B = self.n, self.robot.B
        _check(load_library().fn_ranges_fixed_step(
            self._h, _dev_ptr(states, torch.float32, 8 * n, "states"), C.c_float(delta_m), int(bool(blockwise)),
            _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges")), "fn_ranges_fixed_step")

    def eval_begin(self, states, n_cases, step_limit, out_ranges, out_goal_obs):
        """Evaluation mode: fixed start-goal cases in `states`, completion masks, step limit."""
        import torch
        n, B = self.n, self.robot.B
        _check(load_library().fn_eval_begin(
            self._h, _dev_ptr(states, torch.float32, 8 * n, "states"), int(n_cases), int(step_limit),
            _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges"),
            _dev_ptr(out_goal_obs, torch.float32, 2 * n, "out_goal_obs")), "fn_eval_begin")

    def eval_result(self):
        """(outcome u8 [N], steps i32 [N], return f32 [N], n_running); synchronises."""
        o = np.empty(self.n, np.uint8); st = np.empty(self.n, np.int32); rt = np.empty(self.n, np.float32)
        nr = C.c_int()
        _check(load_library().fn_eval_result(self._h, _np_ptr(o), _np_ptr(st), _np_ptr(rt), C.byref(nr)), "fn_eval_result")
        return o, st, rt, int(nr.value)

    def eval_end(self):
        _check(load_library().fn_eval_end(self._h), "fn_eval_end")

    def counters(self) -> dict:
        out = np.zeros(N_COUNTERS, np.uint64)
        _check(load_library().fn_get_counters(self._h, _np_ptr(out)), "fn_get_counters")
        return {k: int(v) for k, v in zip(COUNTER_NAMES, out)}

    def count_words(self, enable: bool):
        _check(load_library().fn_sim_count_words(self._h, int(bool(enable))), "fn_sim_count_words")

    def profile(self, enable: bool):
        _check(load_library().fn_sim_profile(self._h, int(bool(enable))), "fn_sim_profile")

    def profile_read(self):
        """dict kernel -> (total ms, launches) since the last read; synchronises."""
        ms = np.zeros(8, np.float64)
        ln = np.zeros(8, np.uint64)
        _check(load_library().fn_sim_profile_read(self._h, _np_ptr(ms), _np_ptr(ln)), "fn_sim_profile_read")
        return {"env_step": (float(ms[0]), int(ln[0])), "beam_step": (float(ms[1]), int(ln[1])),
                "compact": (float(ms[2]), int(ln[2])), "reset": (float(ms[3]), int(ln[3])),
                "beam_reset": (float(ms[4]), int(ln[4])),
                "features": (float(ms[5]), int(ln[5])), "features_reset": (float(ms[6]), int(ln[6])),
                "reset_path": (float(ms[2] + ms[3] + ms[4]), int(ln[2] + ln[3] + ln[4]))}

    def episode_state(self):
        """Host copies of the sim's d_prev [N] f32 and ep_step [N] i32 (synchronises)."""
        d = np.empty(self.n, np.float32)
        e = np.empty(self.n, np.int32)
        _check(load_library().fn_sim_episode_state(self._h, _np_ptr(d), _np_ptr(e)), "fn_sim_episode_state")
        return d, e

    def beam_config(self) -> dict:
        cfg = np.zeros(8, np.int32)
        _check(load_library().fn_sim_beam_config(self._h, _np_ptr(cfg)), "fn_sim_beam_config")
        return {"smem": bool(cfg[0]), "grid": int(cfg[1]), "block": int(cfg[2]), "smem_bytes": int(cfg[3]),
                "split_step": bool(cfg[4]), "fused_reset": bool(cfg[5]), "coarse": bool(cfg[6]), "coarse_available": bool(cfg[7])}

    def set_fused_reset(self, enable) -> bool:
        """fn_reset(mask=None) as one fused kernel (1 / True, default where possible), never (0 / False), or for
        masks too (2); returns whether the fused kernel is available and enabled."""
        act = C.c_int(0)
        _check(load_library().fn_sim_set_fused_reset(self._h, int(enable), C.byref(act)), "fn_sim_set_fused_reset")
        return bool(act.value)

    def set_split_step(self, enable: bool) -> bool:
        """fn_step with the env step split around the beam kernel (default where possible) or as one env-step kernel;
        returns whether the split step is used."""
        act = C.c_int(0)
        _check(load_library().fn_sim_set_split_step(self._h, 1 if enable else 0, C.byref(act)), "fn_sim_set_split_step")
        return bool(act.value)

    def set_coarse(self, enable: bool) -> bool:
        """Coarse level for empty-space skipping in the production beam kernels; returns whether it is in use."""
        act = C.c_int(0)
        _check(load_library().fn_sim_set_coarse(self._h, 1 if enable else 0, C.byref(act)), "fn_sim_set_coarse")
        return bool(act.value)

    def prepare_reset(self, seeds):
        """Announce the seeds of the reset(mask=None) that follows the NEXT step(): that step then also prepares the
        reset of the envs it reports done (same results, the reset's latency leaves the critical path).  None withdraws.

        CONTRACT: the values in `seeds` are read DURING the next step(), and reset() recognises the announcement by the
        tensor's ADDRESS.  Do not write into this tensor between that step() and its reset(): a tensor refilled in place
        in between yields resets drawn from the old values, silently (the library cannot see the write; this binding
        only keeps the tensor alive).  With one persistent seeds tensor per loop, refill it BEFORE prepare_reset(), or
        alternate between two tensors."""
        import torch
        if seeds is not None and seeds.dtype not in (torch.int64, torch.uint64):
            raise FlashNavError("seeds must be a 64-bit integer tensor")
        self._prep_keep = seeds
        _check(load_library().fn_sim_prepare_reset(
            self._h, None if seeds is None else _dev_ptr(seeds, seeds.dtype, self.n, "seeds")), "fn_sim_prepare_reset")

    @staticmethod
    def _host_ptr(a, name):
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            if not a.flags.c_contiguous:
                raise FlashNavError(f"{name}: not contiguous")
            return C.c_void_p(a.ctypes.data)
        if a.is_cuda or not a.is_contiguous():
            raise FlashNavError(f"{name}: expected a contiguous CPU tensor")
        return C.c_void_p(a.data_ptr())

    def step_host_begin(self, slot, states_in, actions, dt, reset_mask, seeds, out_states, out_ranges, out_collision, out_goal_obs):
        """Pipelined end-to-end step (two slots): enqueues copies in, fn_step, fn_reset and the copies out; returns at once."""
        hp = self._host_ptr
        _check(load_library().fn_step_host_begin(self._h, int(slot), hp(states_in, "states_in"), hp(actions, "actions"), C.c_float(dt),
                                                 hp(reset_mask, "reset_mask"), hp(seeds, "seeds"), hp(out_states, "out_states"),
                                                 hp(out_ranges, "out_ranges"), hp(out_collision, "out_collision"),
                                                 hp(out_goal_obs, "out_goal_obs")), "fn_step_host_begin")

    def step_host_end(self, slot):
        """Blocks until the outputs of the slot's step have arrived in its host buffers."""
        _check(load_library().fn_step_host_end(self._h, int(slot)), "fn_step_host_end")

    def step_host(self, states, actions, dt, reset_mask, seeds, out_ranges, out_collision, out_goal_obs):
        """End to end with HOST buffers (numpy arrays or pinned CPU tensors); copies inside the call."""
        hp = self._host_ptr
        _check(load_library().fn_step_host(self._h, hp(states, "states"), hp(actions, "actions"), C.c_float(dt),
                                           hp(reset_mask, "reset_mask"), hp(seeds, "seeds"), hp(out_ranges, "out_ranges"),
                                           hp(out_collision, "out_collision"), hp(out_goal_obs, "out_goal_obs")), "fn_step_host")

    def close(self):
        if getattr(self, "_h", None):
            load_library().fn_sim_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


NOALLOC_MAX_ENVS = 8192   # FN_NOALLOC_MAX_ENVS of include/flashnav.h


def observe_noalloc(map_: Map, robot: Robot, n_envs: int, states, out_ranges, out_goal_obs=None, stream=None):
    """fn_observe_noalloc: what Sim.observe_all computes (ranges [N, B] and, optionally, goal obs [2, N] of the poses
    in `states` [8, N]), for callers that may not allocate device memory at the point of the call -- all of it already
    belongs to a framework's memory pool, or a latency bound forbids the device-wide stall of cudaMalloc.  Needs no Sim:
    the poses between its two kernels live in a fixed ~0.75 MiB array inside the library, so n_envs x sensors is limited
    to NOALLOC_MAX_ENVS (beyond it the call raises and names Sim.observe_all).  Every call on a device shares that
    array: calls that could overlap on the GPU (two streams, two threads) must be ordered by the caller.  The first call
    on a device does a one-time address lookup; make it at start-up, before any stream capture.  Enqueues on `stream`
    (default: torch's current stream) and does not synchronise."""
    import torch
    n, B = int(n_envs), robot.B
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().fn_observe_noalloc(
        map_._h, robot._h, n, _dev_ptr(states, torch.float32, 8 * n, "states"),
        _dev_ptr(out_ranges, torch.float32, n * B, "out_ranges"), _dev_ptr(out_goal_obs, torch.float32, 2 * n, "out_goal_obs"),
        C.c_void_p(st.cuda_stream)), "fn_observe_noalloc")


def measure_peak(kind: int) -> float:
    """bytes/s of kind 0 (smem conflict-free), 1 (smem random), 2 (L2-resident global)."""
    import torch
    out = C.c_double()
    _check(load_library().fn_measure_peak(int(kind), C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out)),
           "fn_measure_peak")
    return float(out.value)
