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


def test_terminal_observations_against_a_dictionary_model(oracle_lib):
    # PAPER.md:86 "Observations before reset are retained as next observations in replay, while reset observations are
    # returned to the collector."  The oracle keeps them in a small second ring (fno_terminal_save) and the sampler
    # hands them out as the next observation of done rows.  Pinned against plain Python bookkeeping: a dictionary
    # from the global row id to the observation the step left behind, and per kept id the index of the first entry
    # written after the step it belongs to (a batch of entries is given up as soon as a later write reuses one of them).
    # Every value written anywhere is unique, so a wrong row, a wrong entry or a stale entry shows.  Covers: ring wrap,
    # terminal-ring wrap (entries lost), envs reset without a finished episode, a reset called twice, codes 1 / 2 / 3.
    n, B, A, cap, t_cap = 5, 3, 2, 23, 7
    row, obs = B + 5 + A + 2, B + 5
    rng = np.random.default_rng(3)
    ring = np.zeros((cap, row), np.float32)
    store = oracle_lib.TerminalStore(cap, t_cap, B)
    uniq = iter(range(1, 10 ** 6))
    new_obs = lambda: np.array([next(uniq) for _ in range(obs)], np.float32)
    left_behind = {}                                              # row id -> the observation the step left (pre-reset)
    kept_at = {}                                                  # row id -> entries written when its step ended
    written = 0                                                   # entries written so far
    alive = lambda g: g in kept_at and written <= kept_at[g] + t_cap
    was_reset = set()                                             # row ids whose env was reset right after the row
    total = 0
    for e in range(n):                                            # the first observation (a reset of all envs): pending rows
        ring[e, :obs] = new_obs()
    seen_codes = set()
    for t in range(60):
        head = total % cap
        code = rng.choice([0, 0, 0, 1, 2], n)
        for e in range(n):                                        # the step completes rows [head, head + n) ...
            r = ring[(head + e) % cap]
            r[obs:obs + A] = [next(uniq) for _ in range(A)]
            r[obs + A] = next(uniq)
            r[obs + A + 1] = code[e]
            o = new_obs()                                         # ... and leaves the next observation in the pending rows
            ring[(head + n + e) % cap, :obs] = o
            left_behind[total + e] = o
        total += n
        head = total % cap
        store.step_ended()
        batch = written
        lst = [e for e in range(n) if code[e] != 0]
        if t % 4 == 1:
            lst.append(int(rng.integers(0, n)))                   # an env reset although its episode goes on (or twice)
        rng.shuffle(lst)
        for rep in range(2 if t % 5 == 2 else 1):                 # sometimes the reset is called twice
            oracle_lib.terminal_save(ring, cap, total, n, B, A, lst, store)
            for e in lst:                                         # the model, in list order
                g = total - n + e
                if code[e] != 0 and not alive(g):
                    kept_at[g] = batch
                    written += 1
            for e in lst:                                         # the reset writes the reset observation
                ring[(head + e) % cap, :obs] = new_obs()
                was_reset.add(total - n + e)
        rows, nxt, slots = oracle_lib.ring_sample(ring, cap, total, n, B, A, 100 + t, 64, store=store)
        valid = min(total, cap - n)
        for i in range(64):
            si = oracle_lib.sample_slot(100 + t, i, valid)
            g = total - valid + si
            slot = (head - valid + si) % cap
            assert slot == slots[i]
            want_row = ring[slot].copy()
            want_next = ring[(slot + n) % cap, :obs]
            c = want_row[-1]
            if c != 0:
                if alive(g):
                    want_next = left_behind[g]
                elif c == 2:
                    want_row[-1] = 3
            elif g not in was_reset:
                assert np.array_equal(want_next, left_behind[g])  # a running row's next row IS what the step left
            seen_codes.add(int(want_row[-1]))
            assert np.array_equal(rows[i], want_row), (t, i)
            assert np.array_equal(nxt[i], want_next), (t, i)
        # without a terminal ring every truncated row is marked 3 and the next observation is the next row's
        rows0, nxt0, _ = oracle_lib.ring_sample(ring, cap, total, n, B, A, 100 + t, 64)
        assert np.array_equal(nxt0, ring[(slots + n) % cap, :obs])
        assert not (rows0[:, -1] == 2).any() and np.array_equal(rows0[:, -1] == 3, ring[slots, -1] == 2)
    assert seen_codes == {0, 1, 2, 3} and store.head.value == written > 3 * t_cap
