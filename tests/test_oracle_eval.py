"""Pins for the oracle's O12: evaluation completion masks -- hand cases."""
import numpy as np


def test_cases_are_recorded_once_and_excluded_afterwards(oracle_lib):
    n = 6
    outcome = np.array([0, 0, 0, 0, 4, 0], np.uint8)              # slot 4 inactive
    steps = np.zeros(n, np.int32)
    ret = np.zeros(n, np.float32)
    tol, limit = 0.3, 3
    # step 1: env 0 collides AND is within the goal tolerance (collision wins, Eq. (1)); env 1 reaches the goal
    oracle_lib.eval_update([1, 0, 0, 0, 1, 0], [0.1, 0.2, 5, 5, 0.0, 5], tol, [1] * n, limit,
                           [-10, 10, 0.5, 0.25, 99, -0.5], outcome, steps, ret)
    assert outcome.tolist() == [2, 1, 0, 0, 4, 0] and steps.tolist() == [1, 1, 0, 0, 0, 0]
    assert ret.tolist() == [-10, 10, 0.5, 0.25, 0, -0.5]
    # step 2: completed cases ignore whatever the flags say; env 2 collides
    oracle_lib.eval_update([0, 1, 1, 0, 0, 0], [5, 5, 5, 5, 5, 5], tol, [2] * n, limit,
                           [7, 7, -10, 0.25, 7, 1.0], outcome, steps, ret)
    assert outcome.tolist() == [2, 1, 2, 0, 4, 0] and steps.tolist() == [1, 1, 2, 0, 0, 0]
    assert ret.tolist() == [-10, 10, -9.5, 0.5, 0, 0.5]
    # step 3 = the step limit: the remaining cases time out (env 5 reaches the goal on that very step: success)
    oracle_lib.eval_update([0, 0, 0, 0, 0, 0], [5, 5, 5, 5, 5, 0.29], tol, [3] * n, limit,
                           [1, 1, 1, 1, 1, 10], outcome, steps, ret)
    assert outcome.tolist() == [2, 1, 2, 3, 4, 1] and steps.tolist() == [1, 1, 2, 3, 0, 3]
    assert ret.tolist() == [-10, 10, -9.5, 1.5, 0, 10.5]
    assert not np.any(outcome == 0)                               # the batch has ended
