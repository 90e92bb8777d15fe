"""Pins of the oracle's S2 (Eq. 6) and masked L2~ functions against what the
paper and the mathematics fix: the FFT form Eq. 7, closed forms, additivity, the definition on one-pixel masks."""
import numpy as np
import pytest

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs


@pytest.mark.parametrize("H,W,m,phase", [(12, 20, 9, 1), (16, 16, 15, 0), (9, 31, 8, 1)])
def test_s2_equals_fft_autocorrelation_eq7(H, W, m, phase):
    rng = np.random.default_rng(H * 100 + W)
    img = (rng.random((H, W)) < 0.45).astype(np.uint8)
    img[rng.random((H, W)) < 0.05] = 3                      # a byte that belongs to neither phase
    chi = (img == phase).astype(np.float64)
    F = np.fft.fft2(chi)
    corr = np.rint(np.fft.ifft2(F * np.conj(F)).real).astype(np.int64)   # Eq. 7 without 1/(WH); [y, x] lag
    got = orc.s2_counts(img, phase, m)
    for dy in range(-m, m + 1):
        for dx in range(-m, m + 1):
            # Eq. 6 pairs (x1, x1 + d): IDFT{F conj(F)}[d] = sum chi(x1) chi(x1 - d) = the count at lag -d = at lag d
            assert got[dy + m, dx + m] == corr[(-dy) % H, (-dx) % W]
    assert got[m, m] == int(chi.sum())                      # S2(0) = phi * WH
    assert np.array_equal(got, got[::-1, ::-1])             # S2(v) = S2(-v)


def test_s2_stripes_closed_form_and_neighbours_match_l2():
    H, W, m = 24, 40, 7
    img = inputs.stripes(H, W, 8, 3, horizontal=True)       # rows y % 8 < 3 are phase 1
    got = orc.s2_counts(img, 1, m)
    for dy in range(-m, m + 1):
        both = sum(1 for y in range(H) if y % 8 < 3 and (y + dy) % 8 < 3)
        assert (got[dy + m] == both * W).all()              # independent of dx
    rng = np.random.default_rng(4)
    img = (rng.random((H, W)) < 0.6).astype(np.uint8)
    s2 = orc.s2_counts(img, 1, 1)
    l2 = orc.counts(img, 1, 1, full_template=True)          # |P_v| = 2 for the 8 neighbours: L2 = S2 there
    assert np.array_equal(s2, l2)


def test_masked_counts_pins():
    rng = np.random.default_rng(11)
    H, W, m = 14, 19, 9
    img = (rng.random((H, W)) < 0.7).astype(np.uint8)
    vecs = np.array([(dx, dy) for dy in range(-m, m + 1, 2) for dx in range(-m, m + 1, 3)], dtype=np.int32)
    full, _ = orc.counts_list(img, 1, vecs)
    ones = np.ones((H, W), dtype=np.uint8)
    assert np.array_equal(orc.counts_masked(img, ones, 1, vecs), full)          # N = all positions: exact L2
    a = (rng.random((H, W)) < 0.3).astype(np.uint8)
    b = ((rng.random((H, W)) < 0.5) & (a == 0)).astype(np.uint8) * 9            # any non-zero byte selects
    rest = ((a == 0) & (b == 0)).astype(np.uint8)
    ca, cb, cr = (orc.counts_masked(img, k, 1, vecs) for k in (a, b, rest))
    assert np.array_equal(ca + cb + cr, full)                                   # additive over a partition
    assert not orc.counts_masked(img, np.zeros((H, W), np.uint8), 1, vecs).any()
    # one selected position: the definition for that start pixel, written out with numpy indexing
    y0, x0 = 5, 17
    one = np.zeros((H, W), np.uint8)
    one[y0, x0] = 1
    got = orc.counts_masked(img, one, 1, vecs)
    for i, (dx, dy) in enumerate(vecs):
        pth = orc.path(int(dx), int(dy))
        want = int(all(img[(y0 + int(py)) % H, (x0 + int(px)) % W] == 1 for px, py in pth))
        assert got[i] == want


# ---- ensemble sum over an image stack ("averaged over 100 slices") -------------------------------

def test_counts_sum_pins():
    rows = ["110111", "111101", "011111", "111011"]            # tests/golden/worked_image.txt (hand-derived counts)
    img = np.array([[int(c) for c in r] for r in rows], dtype=np.uint8)
    gold1 = np.array([[13, 13, 12, 14, 15], [14, 16, 16, 17, 13], [12, 16, 20, 16, 12], [13, 17, 16, 16, 14],
                      [15, 14, 12, 13, 13]])
    assert np.array_equal(orc.counts_sum(np.stack([img] * 3), 1, 2), 3 * gold1)    # k copies = k x the golden counts
    # the worked image and its complement: phase 1 of the pair = golden phase 1 + golden phase 0
    gold0 = np.zeros((5, 5), dtype=np.int64)
    gold0[2, 2], gold0[1, 3], gold0[3, 1] = 4, 1, 1
    assert np.array_equal(orc.counts_sum(np.stack([img, 1 - img]), 1, 2), gold1 + gold0)
    rng = np.random.default_rng(8)
    stack = (rng.random((7, 9, 13)) < 0.7).astype(np.uint8)
    m = 6
    one = orc.counts_sum(stack[:1], 1, m)
    assert np.array_equal(one, orc.counts(stack[0], 1, m, full_template=True))     # B = 1: the single-image function
    whole = orc.counts_sum(stack, 1, m)
    assert np.array_equal(whole, orc.counts_sum(stack[:3], 1, m) + orc.counts_sum(stack[3:], 1, m))   # additive
    assert whole[m, m] == int(stack.sum())                                          # Eq. 10 summed over the stack
    assert np.array_equal(whole, whole[::-1, ::-1])                                 # Eq. 12
    assert np.array_equal(orc.counts_sum(stack, 0, m)[m, m], (stack == 0).sum())
