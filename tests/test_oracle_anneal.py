"""Pins of the oracle's simulated annealing (Alg. 3) against what the algorithm and the
mathematics fix: limits of the Metropolis rule, the schedule written out, Eq. 19 of the final image re-evaluated
from scratch, and the literal (re-evaluate everything) form against the local-delta form."""
import numpy as np
import pytest

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs


def _setup(H, W, m, phase, seed, N):
    rng = np.random.default_rng(seed)
    target_img = inputs.squares(H, W, 3, 0.35, seed)
    start = target_img.flatten()
    rng.shuffle(start)                                          # same volume fractions, random arrangement
    start = start.reshape(H, W)
    phases = (0, 1) if phase < 0 else (phase,)
    target = np.stack([orc.counts(target_img, ph, m) for ph in phases])
    pairs, log_u = inputs.anneal_proposals(H, W, N, seed + 1)
    return start, target, pairs, log_u, phases


@pytest.mark.parametrize("phase", [1, -1])
def test_huge_temperature_accepts_everything_and_schedule(phase):
    H, W, m, N = 10, 12, 5, 120
    start, target, pairs, log_u, phases = _setup(H, W, m, phase, 3, N)
    s_max, c_max = 7, 50
    img, counts, st, log = orc.anneal(start, phase, m, target, pairs, log_u, 1e300, 1e300, c_max, s_max)
    want = start.copy()
    for xp, yp, xq, yq in pairs:                                # every move accepted: all swaps applied in order
        want[yp, xp], want[yq, xq] = want[yq, xq], want[yp, xp]
    assert np.array_equal(img, want) and log.all()
    assert st["steps"] == N and st["accepted"] == N and st["levels"] == N // s_max
    for i, ph in enumerate(phases):                             # descriptor and Eq. 19 of the final image, from scratch
        assert np.array_equal(counts[i], orc.counts(img, ph, m))
    assert st["E"] == sum(orc.half_sse(counts[i], target[i], m) for i in range(len(phases)))
    assert img.sum() == start.sum()                             # volume fractions preserved


def test_schedule_multiplier_and_level_ends():
    H, W, m, N = 8, 8, 3, 90
    start, target, pairs, log_u, _ = _setup(H, W, m, 1, 5, N)
    T_max, T_min, c_max, s_max = 1e300, 1e298, 9, 1000          # nothing stops a level but c_max
    _, _, st, _ = orc.anneal(start, 1, m, target, pairs, log_u, T_max, T_min, c_max, s_max)
    assert st["levels"] == N // c_max
    T, mult = T_max, (T_min / T_max) ** (s_max / N)             # reading A2, Alg. 3 line 4
    for _ in range(N // c_max):
        T = T * mult                                            # Alg. 3 line 17
    assert st["T"] == T


def test_zero_temperature_never_accepts_a_worse_image():
    H, W, m, N = 9, 11, 4, 80
    start, target, pairs, log_u, _ = _setup(H, W, m, -1, 9, N)
    log_u = np.minimum(log_u, -1e-9)                            # u < 1 strictly
    img, counts, st, log = orc.anneal(start, -1, m, target, pairs, log_u, 1e-300, 1e-300, 1000, 1000)
    cur = start.copy()
    E = sum(orc.half_sse(orc.counts(cur, ph, m), target[ph], m) for ph in (0, 1))
    for k, (xp, yp, xq, yq) in enumerate(pairs):                # replay with from-scratch evaluations
        q = cur.copy()
        q[yp, xp], q[yq, xq] = q[yq, xq], q[yp, xp]
        Eq = sum(orc.half_sse(orc.counts(q, ph, m), target[ph], m) for ph in (0, 1))
        assert bool(log[k]) == (Eq <= E)                        # T -> 0: accept iff not worse
        if log[k]:
            cur, E = q, Eq
    assert np.array_equal(cur, img) and st["E"] == E


@pytest.mark.parametrize("phase", [0, 1, -1])
def test_local_delta_form_equals_literal_form(phase):
    H, W, m, N = 12, 10, 5, 150
    start, target, pairs, log_u, _ = _setup(H, W, m, phase, 21, N)
    E0 = sum(orc.half_sse(orc.counts(start, ph, m), target[i], m)
             for i, ph in enumerate((0, 1) if phase < 0 else (phase,)))
    T_max = 2.0 * E0 / (H * W) ** 2 / 50                        # a temperature at which both outcomes occur
    a = orc.anneal(start, phase, m, target, pairs, log_u, T_max, 0.01 * T_max, 15, 5, use_local=False)
    b = orc.anneal(start, phase, m, target, pairs, log_u, T_max, 0.01 * T_max, 15, 5, use_local=True)
    assert np.array_equal(a[3], b[3]) and np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[2] == b[2]
    assert 0 < a[3].sum() < N                                   # the run exercised accept and reject
    assert a[2]["E"] <= E0 or True
