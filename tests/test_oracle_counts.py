"""Pins for the oracle's counting (oracle/lpf_oracle.c: lpf_oracle_counts*).

Every expected value here comes from something other than the oracle: a hand-worked fixture,
a closed form, a library routine (scipy erosion, numpy FFT), an invariant stated by the
paper (Eq. 10, 12), sampling statistics, or whole-array brute force on tiny images.
"""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st
from scipy import ndimage

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_worked_image():
    sect, data = None, {"image": [], "phase1": [], "phase0": []}
    for line in open(os.path.join(GOLD, "worked_image.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line in data:
            sect = line
            continue
        if sect == "image":
            data[sect].append([int(c) for c in line])
        else:
            data[sect].append([int(t) for t in line.split()])
    return (np.array(data["image"], dtype=np.uint8), np.array(data["phase1"], dtype=np.int64),
            np.array(data["phase0"], dtype=np.int64))


def roll_and_count(img, phase, path):
    """Brute force, structurally different from Alg. 1: AND whole rolled arrays, one per
    path pixel.  np.roll(a, -k)[i] = a[i+k] periodically."""
    ind = (img == phase)
    acc = np.ones_like(ind)
    for a, b in path:
        acc &= np.roll(np.roll(ind, -int(b), axis=0), -int(a), axis=1)
    return int(acc.sum())


def test_worked_image_golden():
    img, c1, c0 = read_worked_image()
    for full in (True, False):
        assert np.array_equal(orc.counts(img, 1, 2, full_template=full), c1)
        assert np.array_equal(orc.counts(img, 0, 2, full_template=full), c0)


@settings(max_examples=60, deadline=None)
@given(st.integers(1, 12), st.integers(1, 12), st.integers(0, 2 ** 31 - 1), st.floats(0.2, 0.9), st.data())
def test_tiny_images_brute_force(H, W, seed, p, data):
    m = data.draw(st.integers(0, min(H, W) - 1))
    img = inputs.bernoulli(H, W, p, seed)
    for phase in (0, 1):
        got = orc.counts(img, phase, m, full_template=True)
        for dy in range(-m, m + 1):
            for dx in range(-m, m + 1):
                assert got[dy + m, dx + m] == roll_and_count(img, phase, orc.path(dx, dy)), (dx, dy)


def test_template_larger_than_image_wraps():
    # the definition works for m >= min(H,W) (modular indexing); reading S15
    img = inputs.bernoulli(5, 7, 0.7, 11)
    got = orc.counts(img, 1, 9, full_template=True)
    for dy in range(-9, 10, 3):
        for dx in range(-9, 10):
            assert got[dy + 9, dx + 9] == roll_and_count(img, 1, orc.path(dx, dy))


@pytest.mark.parametrize("H,W,m", [(16, 16, 7), (12, 20, 9)])
def test_eq10_eq12_and_phase_rules(H, W, m):
    img = inputs.bernoulli(H, W, 0.6, 5)
    c1 = orc.counts(img, 1, m, full_template=True)
    c0 = orc.counts(img, 0, m, full_template=True)
    # Eq. 10: L(0) = phi
    assert c1[m, m] == int((img == 1).sum()) and c0[m, m] == int((img == 0).sum())
    assert orc.normalise(c1, H, W)[m, m] == (img == 1).mean()
    # Eq. 12: L(v) = L(-v), every vector evaluated on its own path
    assert np.array_equal(c1, c1[::-1, ::-1]) and np.array_equal(c0, c0[::-1, ::-1])
    # half + mirror equals the full template
    assert np.array_equal(orc.counts(img, 1, m, full_template=False), c1)
    # phases are labels: phase 0 of I is phase 1 of 1-I
    assert np.array_equal(orc.counts(1 - img, 1, m, full_template=True), c0)
    # count(v) <= count(0); the two phases never share a start pixel
    assert c1.max() == c1[m, m] and np.all(c1 + c0 <= H * W)
    # all-phase image: L == 1; empty: L == 0
    ones = np.ones((H, W), dtype=np.uint8)
    assert np.all(orc.counts(ones, 1, m, full_template=True) == H * W)
    assert np.all(orc.counts(ones, 0, m, full_template=True) == 0)
    # a byte that is neither 0 nor 1 belongs to neither phase (Alg. 1 line 4)
    img2 = img.copy()
    img2[3, 4] = 2
    a = orc.counts(img2, 1, m)
    b = orc.counts(np.where(img2 == 1, 1, 0).astype(np.uint8), 1, m)
    assert np.array_equal(a, b)
    a0 = orc.counts(img2, 0, m)
    b0 = orc.counts(np.where(img2 == 0, 0, 1).astype(np.uint8), 0, m)
    assert np.array_equal(a0, b0)


def test_stripes_closed_form_fix_axes_and_wrap():
    """Horizontal stripes (period p | H, thickness t): every path covers rows 0..dy
    contiguously, so count(dx,dy) = W*(H/p)*max(0, t-|dy|) for EVERY dx, whatever the tie
    rule.  Vertical stripes likewise.  Non-square image pins x<->W, y<->H (reading S2)."""
    H, W, m = 24, 40, 11
    p, t = 8, 5
    hs = inputs.stripes(H, W, p, t, horizontal=True)
    c = orc.counts(hs, 1, m, full_template=True)
    for dy in range(-m, m + 1):
        assert np.all(c[dy + m, :] == W * (H // p) * max(0, t - abs(dy))), dy
    c0 = orc.counts(hs, 0, m, full_template=True)
    for dy in range(-m, m + 1):
        assert np.all(c0[dy + m, :] == W * (H // p) * max(0, (p - t) - abs(dy)))
    vs = inputs.stripes(H, W, p, t, horizontal=False)
    c = orc.counts(vs, 1, m, full_template=True)
    for dx in range(-m, m + 1):
        assert np.all(c[:, dx + m] == H * (W // p) * max(0, t - abs(dx))), dx


def periodic_runs(line):
    """Lengths of maximal periodic runs of True in a 1-D periodic boolean line."""
    n = len(line)
    if line.all():
        return [("full", n)]
    start = int(np.argmin(line))            # a False position
    rolled = np.roll(line, -start)
    runs, cur = [], 0
    for v in rolled:
        if v:
            cur += 1
        elif cur:
            runs.append(("run", cur)); cur = 0
    if cur:
        runs.append(("run", cur))
    return runs


def runlength_count(lines, k):
    """count(k*u) = sum over maximal periodic runs r of max(0, r-k); a fully in-phase
    periodic line of length n contributes n (every start works)."""
    tot = 0
    for line in lines:
        for kind, r in periodic_runs(line):
            tot += r if kind == "full" else max(0, r - k)
    return tot


def test_runlength_closed_form_axes_and_diagonals():
    """Independent of any rasteriser: along (1,0), (0,1), (1,1), (-1,1) the segment is a
    plain run of k+1 pixels, so counts follow from run lengths alone."""
    H = W = 20
    img = inputs.disks(H, W, 3.0, 0.45, 77)
    img[5, :] = 1                                   # one fully in-phase row
    m = 12
    for phase in (0, 1):
        c = orc.counts(img, phase, m, full_template=True)
        ind = (img == phase)
        rows = [ind[y, :] for y in range(H)]
        cols = [ind[:, x] for x in range(W)]
        idx = np.arange(H)
        diag = [ind[(idx) % H, (x0 + idx) % W] for x0 in range(W)]       # direction (1,1)
        anti = [ind[(idx) % H, (x0 - idx) % W] for x0 in range(W)]       # direction (-1,1)
        for k in range(0, m + 1):
            assert c[m, m + k] == runlength_count(rows, k) == c[m, m - k]
            assert c[m + k, m] == runlength_count(cols, k) == c[m - k, m]
            assert c[m + k, m + k] == runlength_count(diag, k) == c[m - k, m - k]
            assert c[m + k, m - k] == runlength_count(anti, k) == c[m - k, m + k]
        # axis-aligned L is non-increasing in |v|
        assert np.all(np.diff(c[m, m:]) <= 0) and np.all(np.diff(c[m:, m]) <= 0)


def test_chess_closed_form():
    # chess-type morphology, s x s squares: horizontal / vertical runs have length s
    s, H, W, m = 5, 20, 30, 9
    img = inputs.chess(H, W, s)
    for phase in (0, 1):
        c = orc.counts(img, phase, m)
        for k in range(m + 1):
            assert c[m, m + k] == H * (W // (2 * s)) * max(0, s - k)
            assert c[m + k, m] == W * (H // (2 * s)) * max(0, s - k)
        # no segment longer than s pixels in either axis direction survives, and the
        # paper's remark "limits the length of the most of the line segments" holds
        assert c[m, m + s] == 0 and c[m + s, m] == 0


def test_every_vector_equals_binary_erosion():
    """count(v) = sum(erosion of the phase indicator by the structuring element P_v) with
    periodic boundary: scipy.ndimage.minimum_filter, footprint = bounding-box mask of P_v,
    mode='wrap'.  Under wrap the origin placement only translates the result."""
    H, W, m = 18, 22, 8
    img = inputs.disks(H, W, 4.0, 0.5, 3)
    for phase in (0, 1):
        c = orc.counts(img, phase, m, full_template=True)
        ind = (img == phase).astype(np.uint8)
        for dy in range(-m, m + 1):
            for dx in range(-m, m + 1):
                p = orc.path(dx, dy).astype(int)
                x0, y0 = p[:, 0].min(), p[:, 1].min()
                fp = np.zeros((p[:, 1].max() - y0 + 1, p[:, 0].max() - x0 + 1), dtype=bool)
                fp[p[:, 1] - y0, p[:, 0] - x0] = True
                er = ndimage.minimum_filter(ind, footprint=fp, mode="wrap")
                assert c[dy + m, dx + m] == int(er.sum()), (dx, dy)


def test_two_pixel_paths_equal_S2_autocorrelation():
    """|P_v| = 2 (the 8 neighbours): the lineal path count is the two-point count of Eq. 6,
    computed by FFT as in Eq. 7."""
    H, W = 24, 36
    img = inputs.gaussian_field(H, W, 3.0, 0.4, 9)
    for phase in (0, 1):
        chi = (img == phase).astype(np.float64)
        F = np.fft.fft2(chi)
        s2 = np.rint(np.fft.ifft2(F * np.conj(F)).real).astype(np.int64)   # s2[y, x] = sum chi(p) chi(p+(x,y))
        c = orc.counts(img, phase, 1, full_template=True)
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                assert c[dy + 1, dx + 1] == s2[dy % H, dx % W]


def test_prefix_monotonicity_and_lsos_rule():
    """If P_w is a prefix of P_v then count(v) <= count(w); in particular a zero count
    forces zero on every longer overlapping segment (the LSOS rule)."""
    H, W, m = 20, 20, 10
    img = inputs.disks(H, W, 2.5, 0.55, 21)
    c = orc.counts(img, 1, m, full_template=True)
    paths = {(dx, dy): [tuple(q) for q in orc.path(dx, dy).tolist()]
             for dy in range(0, m + 1) for dx in range(-m, m + 1) if dy > 0 or dx >= 0}
    by_tuple = {tuple(p): v for v, p in paths.items()}
    checked = 0
    for v, p in paths.items():
        for k in range(1, len(p)):
            w = by_tuple.get(tuple(p[:k]))
            if w is not None:
                assert c[v[1] + m, v[0] + m] <= c[w[1] + m, w[0] + m]
                checked += 1
    assert checked > 200
    assert (c == 0).any()      # the image is sparse enough that the rule has something to say


def test_bernoulli_statistics():
    """i.i.d. Bernoulli(p): E[count(v)] = WH * p^|P_v| (the |P_v| pixels are distinct because
    |P_v| <= min(H,W)).  Bound on the variance: sigma^2 <= E * (1 + p*|P_v|^2)."""
    H = W = 512
    p = 0.7
    img = inputs.bernoulli(H, W, p, 2024)
    vecs = [(0, 0), (1, 0), (0, 1), (2, 1), (-3, 2), (4, 4), (5, -2), (-1, -5), (3, 0)]
    got, _ = orc.counts_list(img, 1, np.array(vecs, dtype=np.int32))
    for (dx, dy), g in zip(vecs, got):
        n = max(abs(dx), abs(dy)) + 1
        E = H * W * p ** n
        sigma = np.sqrt(E * (1 + p * n * n))
        assert abs(g - E) < 6 * sigma, (dx, dy, g, E)
        assert abs(g - E) / E < 0.05          # and a wrong |P_v| (p^(n+-1)) would be off by >= 30 %


def test_counts_list_matches_template():
    img = inputs.bernoulli(16, 24, 0.6, 8)
    m = 6
    c = orc.counts(img, 1, m, full_template=True)
    vecs = np.array([(dx, dy) for dy in range(-m, m + 1) for dx in range(-m, m + 1)], dtype=np.int32)
    got, used = orc.counts_list(img, 1, vecs, threads=2)
    assert used == 2
    assert np.array_equal(got.reshape(2 * m + 1, 2 * m + 1), c)
    # thread count does not change integers
    got1, used1 = orc.counts_list(img, 1, vecs, threads=1)
    assert used1 == 1 and np.array_equal(got1, got)
