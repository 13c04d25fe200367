"""Pins for the oracle's O11: uniform replay sampling.  The generator
is SplitMix64 (pinned against its published stream in test_oracle_reset.py); here: the slot mapping
against Python big integers, uniformity (chi-square), the gather identity and the next-observation rule."""
import numpy as np


def splitmix64_py(sigma, c):
    M = (1 << 64) - 1
    z = (sigma + (c + 1) * 0x9E3779B97F4A7C15) & M
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
    return z ^ (z >> 31)


def test_slot_mapping_against_big_integers(oracle_lib):
    for seed in (0, 1, 0xDEADBEEF, (1 << 64) - 1):
        for filled in (1, 2, 7, 4096, (1 << 22), (1 << 22) - 3):
            for i in (0, 1, 2, 1000, 123456789):
                w = splitmix64_py(seed, i)
                assert oracle_lib.sample_slot(seed, i, filled) == (w * filled) >> 64 < filled


def test_uniform_over_the_filled_rows(oracle_lib):
    filled, n = 97, 200000
    slots = np.array([oracle_lib.sample_slot(12345, i, filled) for i in range(0, n, 1)][:n])
    cnt = np.bincount(slots, minlength=filled)
    assert cnt.min() > 0 and len(cnt) == filled
    chi2 = ((cnt - n / filled) ** 2 / (n / filled)).sum()
    assert chi2 < 160.0                                          # 96 dof: mean 96, p(chi2 > 160) ~ 5e-5


def test_gather_identity_and_next_observation(oracle_lib):
    B, A, n_envs, cap = 11, 2, 6, 40
    row = B + 5 + A + 2
    ring = np.arange(cap * row, dtype=np.float32).reshape(cap, row)
    # total rows appended: before the pending window reaches the end, when it does, after one and several wraps
    for total in (12, 30, 34, 36, 40, 42, 78, 5 * 40 + 18):
        head = total % cap
        valid = min(total, cap - n_envs)                         # restated: completed rows outside the pending window
        assert oracle_lib.ring_valid(cap, total, n_envs) == valid
        rows, nxt, slots = oracle_lib.ring_sample(ring, cap, total, n_envs, B, A, seed=77, n_samples=500)
        expect = [(head - valid + oracle_lib.sample_slot(77, i, valid)) % cap for i in range(500)]   # Python integers
        assert np.array_equal(slots, expect)
        pending = {(head + e) % cap for e in range(n_envs)}
        assert not pending & set(slots.tolist()), "a pending row (stale action / reward / done) was sampled"
        if total <= cap - n_envs:
            assert slots.max() < total                           # not yet full: the rows appended so far, from slot 0
        else:
            assert len(set(slots.tolist())) == cap - n_envs      # every other row is reachable (500 draws of 34)
        assert np.array_equal(rows, ring[slots])
        assert np.array_equal(nxt, ring[(slots + n_envs) % cap, :B + 5])
    # different seeds give different batches, the same seed the same batch
    a = oracle_lib.ring_sample(ring, cap, cap, n_envs, B, A, 1, 64)[2]
    b = oracle_lib.ring_sample(ring, cap, cap, n_envs, B, A, 2, 64)[2]
    c = oracle_lib.ring_sample(ring, cap, cap, n_envs, B, A, 1, 64)[2]
    assert not np.array_equal(a, b) and np.array_equal(a, c)
    # nothing to sample: no row appended yet
    rows = oracle_lib.ring_sample(np.zeros((cap, row), np.float32), cap, 0, n_envs, B, A, 3, 8)[0]
    assert rows.shape == (8, row)
