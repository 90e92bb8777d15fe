"""Pins for the oracle's objective (Eq. 14/19) and two-pixel-swap delta."""
import numpy as np
import pytest

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs


def half_mask(m):
    S = 2 * m + 1
    dy, dx = np.mgrid[-m:m + 1, -m:m + 1]
    return (dy > 0) | ((dy == 0) & (dx >= 0))


def test_sse_exact_integer():
    rng = np.random.default_rng(1)
    c = rng.integers(0, 2 ** 18, size=(7, 7)).astype(np.int64)
    t = rng.integers(0, 2 ** 18, size=(7, 7)).astype(np.int64)
    want = sum((int(a) - int(b)) ** 2 for a, b in zip(c.ravel(), t.ravel()))   # python big ints
    assert orc.sse(c, t) == want
    assert orc.sse(c, c) == 0
    t2 = c.copy(); t2[3, 5] += 1
    assert orc.sse(c, t2) == 1
    # large magnitudes stay exact: (2^26)^2 * 100 < 2^64
    big = np.full(100, 2 ** 26, dtype=np.int64)
    assert orc.sse(big, np.zeros(100, dtype=np.int64)) == 100 * 2 ** 52


def test_objective_full_vs_half_domain_identity():
    """Eq. 14/19 sum over D (half); the library sums the whole [2m+1]^2 array.  For point
    symmetric arrays E_full = 2*E_D - (c0 - t0)^2 (reading S9)."""
    m = 6
    a = orc.counts(inputs.bernoulli(16, 16, 0.6, 3), 1, m)
    b = orc.counts(inputs.bernoulli(16, 16, 0.5, 4), 1, m)
    hm = half_mask(m)
    e_half = int(((a[hm] - b[hm]) ** 2).sum())
    assert orc.sse(a, b) == 2 * e_half - int(a[m, m] - b[m, m]) ** 2


@pytest.mark.parametrize("H,W,m,seed", [(9, 9, 4, 0), (8, 12, 7, 1), (12, 8, 5, 2), (6, 6, 5, 3)])
def test_swap_delta_local_equals_full_reevaluation(H, W, m, seed):
    img = inputs.bernoulli(H, W, 0.55, 100 + seed)
    pairs = inputs.swap_pairs(img, 12, 200 + seed)
    for phase in (0, 1):
        for pr in pairs:
            full = orc.swap_delta_full(img, phase, m, pr, threads=2)
            loc = orc.swap_delta_local(img, phase, m, pr)
            assert np.array_equal(full, loc)
            assert full[m, m] == 0                      # volume fraction preserved
            assert np.array_equal(full, full[::-1, ::-1])
            n = np.maximum(*np.abs(np.mgrid[-m:m + 1, -m:m + 1])) + 1
            assert np.all(np.abs(full) <= 2 * n)        # at most 2(n_v+1) segments can change


def test_swap_delta_adjacent_and_same_segment_pixels():
    # p and q on one segment: the de-duplicated candidate set matters
    img = np.ones((7, 7), dtype=np.uint8)
    img[3, 2] = 0
    pr = (2, 3, 3, 3)                                    # p=(2,3) is 0, q=(3,3) is 1, neighbours
    for phase in (0, 1):
        assert np.array_equal(orc.swap_delta_full(img, phase, 5, pr),
                              orc.swap_delta_local(img, phase, 5, pr))
    # swapping moves the single hole: every count is unchanged by translation invariance
    assert not orc.swap_delta_full(img, 1, 5, pr).any()


def test_swap_pairs_generator_contract():
    img = inputs.disks(32, 32, 4.0, 0.3, 5)
    pr = inputs.swap_pairs(img, 500, 6)
    assert pr.shape == (500, 4) and pr.dtype == np.int32
    assert np.all(img[pr[:, 1], pr[:, 0]] == 0) and np.all(img[pr[:, 3], pr[:, 2]] == 1)


def test_swap_delta_full_pixel_convention_against_numpy_built_image():
    """(x_p, y_p) addresses column x_p of row y_p (reading S2; Eq. 6 `x%W, y%H`): the oracle's delta equals
    counts(I') - counts(I) with I' built here with numpy indexing, on a NON-square image and a pair whose transposed
    reading (x <-> y) is in range too and gives a different answer."""
    H, W, m = 7, 11, 5
    img = inputs.bernoulli(H, W, 0.6, 4242)
    zeros = [(x, y) for y in range(H) for x in range(W) if img[y, x] == 0 and x < H and y < W and x != y]
    ones = [(x, y) for y in range(H) for x in range(W) if img[y, x] == 1 and x < H and y < W and x != y]
    checked = 0
    for (xp, yp), (xq, yq) in zip(zeros[:6], ones[:6]):
        q = img.copy()
        q[yp, xp], q[yq, xq] = img[yq, xq], img[yp, xp]
        tr = img.copy()                                          # the transposed (wrong) reading of the same pair
        tr[xp, yp], tr[xq, yq] = img[xq, yq], img[xp, yp]
        for phase in (0, 1):
            want = orc.counts(q, phase, m, full_template=True) - orc.counts(img, phase, m, full_template=True)
            wrong = orc.counts(tr, phase, m, full_template=True) - orc.counts(img, phase, m, full_template=True)
            got = orc.swap_delta_full(img, phase, m, (xp, yp, xq, yq))
            assert np.array_equal(got, want)
            assert np.array_equal(orc.swap_delta_local(img, phase, m, (xp, yp, xq, yq)), want)
            checked += not np.array_equal(want, wrong)
    assert checked >= 6                                          # the cases do tell the two readings apart
