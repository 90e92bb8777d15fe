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


# ---- the Metropolis rule at FINITE temperature (Alg. 3 line 11; reading A3) ----------
# The expected decision never comes from the oracle's annealing code: E_P and E_Q are Python-integer sums over the
# canonical half D (Eq. 13 / Eq. 19) of descriptors of numpy-built images, the threshold is the exact rational
# (E_P - E_Q) / ((W*H)^2 * T), and ln u is placed a relative 1e-9 on either side of it.  A dropped (W*H)^2, W^4 in its
# place, T^2, the full-array error instead of the half, or a flipped sign moves the threshold by far more than that.

def _half_E(img, target, phases, m):
    """Eq. 19 over D and the phases, exact Python integers, from descriptors of `img` (not from the annealing code)."""
    E = 0
    for i, ph in enumerate(phases):
        c = orc.counts(img, ph, m)
        for dy in range(0, m + 1):
            for dx in range(-m, m + 1):
                if dy > 0 or dx >= 0:                           # D of Eq. 13
                    d = int(target[i][dy + m, dx + m]) - int(c[dy + m, dx + m])
                    E += d * d
    return E


def _swapped(img, pair):
    xp, yp, xq, yq = (int(v) for v in pair)
    q = img.copy()
    q[yp, xp], q[yq, xq] = img[yq, xq], img[yp, xp]             # x indexes columns, y rows (reading S2)
    return q


@pytest.mark.parametrize("H,W,m,phase,T", [(6, 9, 3, 1, 0.37), (9, 6, 4, -1, 2.5e-3), (5, 8, 4, 0, 11.0)])
def test_metropolis_threshold_at_finite_temperature(H, W, m, phase, T):
    from fractions import Fraction
    start, target, pairs, _, phases = _setup(H, W, m, phase, 31 + H, 40)
    seen_worse = seen_better = 0
    for pr in pairs:
        if start[pr[1], pr[0]] == start[pr[3], pr[2]]:
            continue                                            # identity move: E_P = E_Q, threshold 0
        E_P = _half_E(start, target, phases, m)
        E_Q = _half_E(_swapped(start, pr), target, phases, m)
        if E_P == E_Q:
            continue
        r = Fraction(E_P - E_Q, (W * H) ** 2) / Fraction(T)     # exact: T is a binary rational
        seen_worse += E_Q > E_P
        seen_better += E_Q < E_P
        for rel, want in ((1e-9, r < 0), (-1e-9, r > 0)):       # ln u = r (1 + rel): below r iff rel has the sign of -r
            lu = float(r) * (1.0 + rel)
            want_acc = Fraction(lu) < r
            assert want_acc == want
            _, _, st, log = orc.anneal(start, phase, m, target, pr[None], np.array([lu]), T, T, 5, 5)
            assert bool(log[0]) == want_acc, (pr, E_P, E_Q, lu)
            assert st["accepted"] == int(want_acc) and st["E"] == (E_Q if want_acc else E_P)
    assert seen_worse >= 3 and seen_better >= 3                 # both signs of the threshold were exercised


def test_metropolis_threshold_follows_the_temperature_schedule():
    """Second proposal of a chain with c_max = 1: the level ends after the first, so T = T_max * T_mult (Alg. 3
    lines 4 and 17, reading A2) enters the second threshold."""
    from fractions import Fraction
    H, W, m, phase = 7, 10, 4, -1
    start, target, pairs, _, phases = _setup(H, W, m, phase, 77, 60)
    T_max, T_min, s_max, N = 0.8, 0.05, 3, 2
    T2 = T_max * (T_min / T_max) ** (s_max / N)
    done = 0
    for k in range(0, 58):
        two = pairs[k:k + 2]
        P1 = _swapped(start, two[0])                            # the first proposal is always accepted (ln u = -inf)
        E_P, E_Q = _half_E(P1, target, phases, m), _half_E(_swapped(P1, two[1]), target, phases, m)
        if E_P == E_Q:
            continue
        r = Fraction(E_P - E_Q, (W * H) ** 2) / Fraction(T2)
        for rel in (1e-9, -1e-9):
            lu = float(r) * (1.0 + rel)
            _, _, st, log = orc.anneal(start, phase, m, target, two, np.array([-np.inf, lu]), T_max, T_min, 1, s_max)
            assert bool(log[0]) and bool(log[1]) == (Fraction(lu) < r)
            assert st["levels"] == 2 and st["T"] == T2 * (T_min / T_max) ** (s_max / N)
        done += 1
    assert done >= 20


# ---- the modification operator drawing its own pixels (reading A7) ------------------

def test_splitmix64_published_vectors():
    """Reference outputs of Vigna's splitmix64.c for seed 1234567 (also the Rosetta Code task's expected values) and
    the well-known first output for seed 0."""
    want = [6457827717110365317, 3203168211198807973, 9817491932198370423, 4593380528125082431, 16408922859458223821]
    assert [orc.splitmix64(1234567, n) for n in range(1, 6)] == want
    assert orc.splitmix64(0, 1) == 0xE220A8397B1DCDAF


def _interfacial(img):
    return ((img != np.roll(img, 1, 0)) | (img != np.roll(img, -1, 0)) | (img != np.roll(img, 1, 1)) |
            (img != np.roll(img, -1, 1)))


@pytest.mark.parametrize("policy", [1, 2])
def test_proposals_have_the_policy_properties_and_are_uniform(policy):
    H, W = 11, 14                                               # non-square: a transposed pixel would leave the image
    img = inputs.squares(H, W, 3, 0.4, 77)
    inter = _interfacial(img)
    n = 6000
    pr = np.array([orc.propose(img, policy, 99, k) for k in range(n)])
    xp, yp, xq, yq = pr.T
    assert np.all((0 <= xp) & (xp < W) & (0 <= yp) & (yp < H) & (0 <= xq) & (xq < W) & (0 <= yq) & (yq < H))
    assert np.all(img[yp, xp] != img[yq, xq])                   # "two ... pixels from different phases"
    if policy == 2:
        assert inter[yp, xp].all() and inter[yq, xq].all()      # "random selection of interfacial pixels"
    # p is uniform over the qualifying pixels; q uniform over the qualifying pixels of the other byte, given p's byte
    ok_p = inter if policy == 2 else np.ones_like(inter)
    cnt = np.zeros((H, W))
    np.add.at(cnt, (yp, xp), 1)
    exp = n / ok_p.sum()
    chi2 = (((cnt - exp) ** 2)[ok_p] / exp).sum()
    assert cnt[~ok_p].sum() == 0 and chi2 < ok_p.sum() + 6 * np.sqrt(2 * ok_p.sum())
    for b in (0, 1):
        sel = img[yp, xp] == b
        ok_q = ok_p & (img != b)
        cq = np.zeros((H, W))
        np.add.at(cq, (yq[sel], xq[sel]), 1)
        e = sel.sum() / ok_q.sum()
        assert cq[~ok_q].sum() == 0 and (((cq - e) ** 2)[ok_q] / e).sum() < ok_q.sum() + 6 * np.sqrt(2 * ok_q.sum())
    # the random words are the documented ones: proposal k, attempt 0, side 0 is SplitMix64 output 1 + 128 k
    if policy == 1:
        for k in (0, 1, 17):
            u = orc.splitmix64(99, 1 + 128 * k)
            assert (xp[k], yp[k]) == (((u >> 32) * W) >> 32, ((u & 0xffffffff) * H) >> 32)


def test_no_qualifying_pixel_gives_the_identity_move():
    img = np.ones((6, 9), dtype=np.uint8)                        # one phase only: nothing to exchange
    for policy in (1, 2):
        pr = orc.propose(img, policy, 5, 3)
        assert (pr[0], pr[1]) == (pr[2], pr[3])


@pytest.mark.parametrize("policy,phase", [(1, 1), (2, -1)])
def test_generating_chain_equals_the_list_chain_on_its_own_proposals(policy, phase):
    """Every decided proposal was drawn from the image of that moment (replayed here with numpy), and feeding the
    decided proposals back as a LIST reproduces the chain (the list chain is pinned above)."""
    H, W, m, N = 10, 12, 5, 160
    start, target, _, log_u, _ = _setup(H, W, m, phase, 41, N)
    E0 = _half_E(start, target, (0, 1) if phase < 0 else (phase,), m)
    T_max = 2.0 * E0 / (H * W) ** 2 / 50
    img, counts, st, log, pairs = orc.anneal_generate(start, phase, m, target, policy, 2024, log_u, T_max, 0.01 * T_max,
                                                      16, 5)
    cur = start.copy()
    for k in range(N):
        assert np.array_equal(pairs[k], orc.propose(cur, policy, 2024, k)), k
        if log[k]:
            cur = _swapped(cur, pairs[k])
    assert np.array_equal(cur, img) and 0 < log.sum() < N
    a = orc.anneal(start, phase, m, target, pairs, log_u, T_max, 0.01 * T_max, 16, 5)
    assert np.array_equal(a[0], img) and np.array_equal(a[1], counts) and a[2] == st and np.array_equal(a[3], log)
