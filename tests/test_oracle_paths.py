"""Pins for the oracle's rasteriser (oracle/lpf_oracle.c: lpf_oracle_path).

Nothing here re-types the oracle's incremental-error loop: the pins are the paper's closed
forms (Eq. 13, 15-17, the 6.716e9 operation count), hand-worked literals (tests/golden/),
and the mathematical definition of a Bresenham line (closest pixel to the ideal line).
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import lpf_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def half_vectors(m):
    return [(dx, dy) for dy in range(-m, m + 1) for dx in range(-m, m + 1)
            if dy > 0 or (dy == 0 and dx >= 0)]


def test_worked_paths_golden():
    # tests/golden/worked_paths.txt -- D1, D2 (tie rule), D3 (point symmetry)
    n = 0
    for line in open(os.path.join(GOLD, "worked_paths.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, tail = line.split(":")
        dx, dy = (int(t) for t in head.split())
        want = [tuple(int(c) for c in p.split(",")) for p in tail.split()]
        got = [tuple(p) for p in orc.path(dx, dy).tolist()]
        assert got == want, (dx, dy)
        n += 1
    assert n == 16


def test_canonical_half_is_eq13():
    # Eq. 13: D = [-W+1;-1]x[1;H-1] + [0;W-1]x[0;H-1]; |D| = 2HW-H-W+1
    for (W, H) in [(1, 1), (3, 5), (6, 4), (9, 9)]:
        D = {(dx, dy) for dx in range(-W + 1, 0) for dy in range(1, H)} | \
            {(dx, dy) for dx in range(0, W) for dy in range(0, H)}
        assert len(D) == 2 * H * W - H - W + 1
        for dy in range(-H + 1, H):
            for dx in range(-W + 1, W):
                assert orc.in_half(dx, dy) == ((dx, dy) in D)
    # exactly one of v, -v is canonical (v != 0)
    for dy in range(-4, 5):
        for dx in range(-4, 5):
            if (dx, dy) != (0, 0):
                assert orc.in_half(dx, dy) != orc.in_half(-dx, -dy)


@pytest.mark.parametrize("W,H", [(1, 1), (2, 2), (5, 5), (17, 17), (4, 7), (6, 11), (40, 40)])
def test_table_size_eq15_16_17(W, H):
    # Eq. 15: M = sum_{i=1..W} sum_{j=1..H} max(i,j) + sum_{i=2..W} sum_{j=2..H} max(i,j)
    eq15 = sum(max(i, j) for i in range(1, W + 1) for j in range(1, H + 1)) + \
        sum(max(i, j) for i in range(2, W + 1) for j in range(2, H + 1))
    D = [(dx, dy) for dx in range(-W + 1, 0) for dy in range(1, H)] + \
        [(dx, dy) for dx in range(0, W) for dy in range(0, H)]
    got = sum(orc.path(dx, dy).shape[0] for dx, dy in D)
    assert got == eq15
    if W <= H:
        # Eq. 16
        eq16 = Fraction(W * (3 * H * H + 3 * H + W * W - 1), 3) - Fraction(W * (W + 1), 2) \
            - Fraction(H * (H + 1), 2) + 1
        assert eq16 == eq15
    if W == H:
        # Eq. 17
        assert Fraction(4 * W ** 3 - 4 * W + 3, 3) == eq15


def test_template_table_size_closed_form():
    # square template |dx|,|dy| <= m is Eq. 17 with W = m+1 (reading S7)
    for m in [0, 1, 2, 7, 16, 33]:
        W = m + 1
        hv = half_vectors(m)
        assert len(hv) == 2 * m * m + 2 * m + 1 == 2 * W * W - 2 * W + 1
        assert 3 * sum(orc.path(dx, dy).shape[0] for dx, dy in hv) == 4 * W ** 3 - 4 * W + 3


def test_operation_count_6_716e9():
    # "the overall number of operations for single standard calculation of the
    # L2^i-function is 6.716e9" at 100x100 = W*H * sum_{i,j=1..100} max(i,j) (first term of Eq. 15)
    lens = sum(orc.path(dx, dy).shape[0] for dx in range(100) for dy in range(100))
    assert 100 * 100 * lens == 6716500000
    assert round(100 * 100 * lens / 1e9, 3) == 6.716


@pytest.mark.parametrize("m", [1, 2, 3, 8, 21])
def test_path_is_closest_pixel_line(m):
    """Bresenham [20] = for every major-axis step the pixel closest to the ideal line;
    an exact tie (distance 1/2) goes to the larger |minor| (reading D2)."""
    for dx, dy in half_vectors(m):
        p = orc.path(dx, dy).astype(int)
        n = max(abs(dx), abs(dy))
        assert p.shape == (n + 1, 2)
        assert tuple(p[0]) == (0, 0) and tuple(p[-1]) == (dx, dy)
        xmajor = abs(dx) >= abs(dy)
        maj, mnr = (0, 1) if xmajor else (1, 0)
        dmaj, dmnr = (dx, dy) if xmajor else (dy, dx)
        for k in range(n + 1):
            assert abs(p[k, maj]) == k and (p[k, maj] == 0 or np.sign(p[k, maj]) == np.sign(dmaj))
            if n == 0:
                continue
            ideal = Fraction(k * abs(dmnr), n)           # |minor| of the ideal line at step k
            got = abs(p[k, mnr])
            assert p[k, mnr] == 0 or np.sign(p[k, mnr]) == np.sign(dmnr)
            err = Fraction(got) - ideal
            assert -Fraction(1, 2) < err <= Fraction(1, 2), (dx, dy, k)
        steps = np.diff(p, axis=0)
        assert np.all(np.abs(steps) <= 1)                  # 8-connected, monotone
        assert np.all(np.abs(steps[:, maj]) == 1) if n else True


@pytest.mark.parametrize("m", [1, 2, 5, 12])
def test_point_symmetry_D3_and_mirror_transpose(m):
    for dy in range(-m, m + 1):
        for dx in range(-m, m + 1):
            p = orc.path(dx, dy).astype(int)
            q = orc.path(-dx, -dy).astype(int)
            # same pixel set as the reversed segment
            assert np.array_equal(p, q[::-1] + np.array([dx, dy]))
            assert tuple(p[0]) == (0, 0) and tuple(p[-1]) == (dx, dy)
    # inside D the rule is mirror-symmetric in dx and transposition-symmetric (used by the
    # CUDA library to reduce all orientations to one octant; stated here as a property of D2)
    for dy in range(1, m + 1):
        for dx in range(0, m + 1):
            p = orc.path(dx, dy).astype(int)
            assert np.array_equal(orc.path(-dx, dy).astype(int), p * np.array([-1, 1]))
            assert np.array_equal(orc.path(dy, dx).astype(int), p[:, ::-1])


def test_tie_rule_is_not_point_symmetric_by_itself():
    """applying D2 independently to -v would give a different pixel set on
    tie vectors, so D3 is a real choice.  (2,1): D2 on (-2,-1) with ties up in magnitude would
    give (0,0),(-1,-1),(-2,-1); D3 gives (0,0),(-1,0),(-2,-1)."""
    assert orc.path(-2, -1).tolist() == [[0, 0], [-1, 0], [-2, -1]]
    assert orc.path(-2, -1).tolist() != (-orc.path(2, 1)).tolist()
