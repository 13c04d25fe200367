"""The C-ABI library loads without a GPU and exports every symbol include/flashnav.h declares."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fn():
    from paper_2606_15846_b200 import build
    build.build()
    import paper_2606_15846_b200 as fn
    return fn


def _declared():
    src = open(os.path.join(ROOT, "include", "flashnav.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fn_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(fn):
    lib = fn.load_library()
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(fn.EXPORTED_SYMBOLS), set(names) ^ set(fn.EXPORTED_SYMBOLS)


def test_version_and_task_defaults(fn):
    lib = fn.load_library()
    assert b"sm_100a" in lib.fn_version()
    from paper_2606_15846_b200._binding import _Task
    t = _Task()
    lib.fn_task_default(ctypes.byref(t))
    # Eq. (1) constants of the paper
    assert (t.r_success, t.r_collision, t.c_progress) == (10.0, -10.0, 2.0)
    assert t.max_episode_steps == 0 and abs(t.goal_tol_m - 0.3) < 1e-7


def test_host_side_argument_errors_need_no_gpu(fn):
    lib = fn.load_library()
    out = ctypes.c_void_p()
    bm = np.zeros((4, 4), np.uint8)
    assert lib.fn_map_create(None, 4, 4, ctypes.c_float(0.05), ctypes.byref(out)) == -1
    assert lib.fn_map_create(bm.ctypes.data_as(ctypes.c_void_p), 0, 4, ctypes.c_float(0.05), ctypes.byref(out)) == -1
    assert lib.fn_map_create(bm.ctypes.data_as(ctypes.c_void_p), 4, 4, ctypes.c_float(float("nan")), ctypes.byref(out)) == -1
    assert b"resolution" in lib.fn_last_error()
    fp = np.array([[0, 0], [1, 0], [1, 1]], np.float32)
    ang = np.zeros(1, np.float32)
    lim = np.array([0, 1, 0, 0, -1, 1], np.float32)
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    assert lib.fn_robot_create(p(fp), 2, p(ang), 1, ctypes.c_float(1.0), 0, p(lim), ctypes.byref(out)) == -1
    assert lib.fn_robot_create(p(fp), 65, p(ang), 1, ctypes.c_float(1.0), 0, p(lim), ctypes.byref(out)) == -2
    assert lib.fn_robot_create(p(fp), 3, p(ang), 0, ctypes.c_float(1.0), 0, p(lim), ctypes.byref(out)) == -1
    assert lib.fn_step(None, None, None, ctypes.c_float(0.1), None, None, None, None) == -1
    # the entry points of the widened rows validate on the host as well
    comp = np.array([3, 2], np.int32)
    fp5 = np.zeros((5, 2), np.float32)
    assert lib.fn_robot_create_union(p(fp5), p(comp), 2, p(ang), 1, ctypes.c_float(1.0), 0, p(lim), ctypes.byref(out)) == -1
    assert lib.fn_robot_create_union(p(fp5), p(comp), 0, p(ang), 1, ctypes.c_float(1.0), 0, p(lim), ctypes.byref(out)) == -1
    assert lib.fn_robot_set_acc_limits(None, p(lim)) == -1
    assert lib.fn_sim_bind_features(None, 8, None) == -1
    assert lib.fn_ring_sample(None, ctypes.c_uint64(1), 4, None, None) == -1
    assert lib.fn_eval_begin(None, None, 1, 1, None, None) == -1
    assert lib.fn_eval_result(None, None, None, None, None) == -1 and lib.fn_eval_end(None) == -1
    assert lib.fn_ranges_fixed_step(None, None, ctypes.c_float(0.1), 1, None) == -1
    assert lib.fn_sim_set_stream(None, None) == -1 and lib.fn_reset(None, None, None, None, None, None) == -1
    # the switches between equivalent launch sequences
    assert lib.fn_sim_set_fused_reset(None, 1, None) == -1 and lib.fn_sim_set_split_step(None, 1, None) == -1
    assert lib.fn_step_host(None, None, None, ctypes.c_float(0.1), None, None, None, None, None) == -1
    # round 2: coarse level, pipelined host step, further sensors
    assert lib.fn_sim_set_coarse(None, 1, None) == -1
    assert lib.fn_step_host_begin(None, 0, None, None, ctypes.c_float(0.1), None, None, None, None, None, None) == -1
    assert lib.fn_step_host_end(None, 0) == -1
    assert lib.fn_robot_add_sensor(None, p(ang), 1, ctypes.c_float(1.0), ctypes.c_float(0), ctypes.c_float(0), ctypes.c_float(0)) == -1
    assert lib.fn_sim_beam_config(None, None) == -1


def test_no_cpu_fallback(fn):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(fn.FlashNavError):
        fn.Map(np.zeros((8, 8), np.uint8), 0.05)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_15846_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("an oracle", ""), f
    for f in ("fn_oracle.c", "__init__.py"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_2606_15846_b200" not in txt and "from paper_2606_15846_b200" not in txt and "libflashnav" not in txt
