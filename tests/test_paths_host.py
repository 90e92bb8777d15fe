"""Host side of liblpf.so (no GPU): C-ABI exports, lpf_build_paths table vs the paper's closed
forms (Eq. 13, 15-17), vs the worked paths in tests/golden/, and vs the
oracle's independently written rasteriser; structure of the linearised node program."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import build as lpf_build
from paper_1601_04359_b200 import lpf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    lpf_build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "lpf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(lpf_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(lpf.EXPORTS)
    lib = ctypes.CDLL(lpf.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_error_codes_on_host():
    lib = lpf.load()
    h = ctypes.c_void_p()
    assert lib.lpf_build_paths(-1, -1, ctypes.byref(h)) == lpf.LPF_E_INVAL
    assert lib.lpf_build_paths(512, -1, ctypes.byref(h)) == lpf.LPF_E_UNSUPPORTED
    assert lib.lpf_build_paths(3, -1, None) == lpf.LPF_E_INVAL
    p = lpf.lpf_build_paths(3, -1)
    with pytest.raises(lpf.LpfError):
        lpf.lpf_paths_get(p, 4, 0)
    # a host-only table refuses the device entry points (no CPU fallback)
    buf = (ctypes.c_uint8 * 64)()
    out = (ctypes.c_int64 * 49)()
    assert lib.lpf_eval(p.handle, buf, 1, 8, 8, 1, out, 0, None) == lpf.LPF_E_INVAL
    assert lib.lpf_swap_delta(p.handle, buf, 8, 8, 1, buf, 1, out, None) == lpf.LPF_E_INVAL
    assert lib.lpf_swap_delta_static(p.handle, buf, 8, 8, 1, buf, 1, out, None) == lpf.LPF_E_INVAL
    assert lib.lpf_strerror(lpf.LPF_E_UNSUPPORTED) == b"unsupported shape"
    assert b"LPF_STATIC_SCRATCH_BYTES" in lib.lpf_strerror(lpf.LPF_E_TOO_LARGE)
    # the tuning hooks check their arguments
    for fn, bad in ((lib.lpf_set_tmem_stack, (2, -1)), (lib.lpf_set_level, (7, -2)), (lib.lpf_set_teams, (33, -1)),
                    (lib.lpf_set_shared_memory, (1000, -1))):
        for v in bad:
            assert fn(p.handle, v) == lpf.LPF_E_INVAL, (fn, v)
        assert fn(None, 0) == lpf.LPF_E_INVAL
    assert lib.lpf_set_tmem_stack(p.handle, 0) == lpf.LPF_OK and lib.lpf_set_tmem_stack(p.handle, 1) == lpf.LPF_OK
    lpf.lpf_free_paths(p)


@pytest.mark.parametrize("m", [0, 1, 2, 5, 16, 64])
def test_table_sizes_closed_forms(m):
    p = lpf.lpf_build_paths(m, -1)
    info = lpf.lpf_paths_info(p)
    # |D| = 2HW - H - W + 1 at H = W = m + 1
    assert info["n_half_vectors"] == 2 * (m + 1) ** 2 - 2 * (m + 1) + 1
    # Eq. 17 with W = m + 1: (4 W^3 - 4 W + 3) / 3
    Wd = m + 1
    assert info["sum_path_len"] * 3 == 4 * Wd ** 3 - 4 * Wd + 3
    assert info["max_depth"] == m
    assert info["n_trie_nodes"] <= info["sum_path_len"]


def test_trie_node_counts_of_the_five_configs():
    # distinct prefixes for m = 16 / 64 / 128
    for m, n in ((16, 1552), (64, 82072), (128, 635544)):
        p = lpf.lpf_build_paths(m, -1)
        assert lpf.lpf_paths_info(p)["n_trie_nodes"] == n


def test_worked_paths_golden():
    p = lpf.lpf_build_paths(8, -1)
    for line in open(os.path.join(ROOT, "tests", "golden", "worked_paths.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        head, tail = line.split(":")
        dx, dy = (int(t) for t in head.split())
        want = [tuple(int(t) for t in pt.split(",")) for pt in tail.split()]
        got = [tuple(int(t) for t in r) for r in lpf.lpf_paths_get(p, dx, dy)]
        assert got == want, (dx, dy)


@pytest.mark.parametrize("m", [1, 4, 13, 40])
def test_closed_form_rasteriser_equals_oracle_incremental_form(m):
    # two formulations, no shared code: library closed form vs oracle error accumulation
    p = lpf.lpf_build_paths(m, -1)
    for dy in range(-m, m + 1):
        for dx in range(-m, m + 1):
            assert np.array_equal(lpf.lpf_paths_get(p, dx, dy), orc.path(dx, dy)), (dx, dy)


def _decode(entries):
    x = (entries & np.uint64(0xffffffff)).astype(np.int64)
    y = (entries >> np.uint64(32)).astype(np.int64)
    return dict(sh=x & 31, reload=(x >> 5) & 1, terminal=(x >> 6) & 1, save=(x >> 7) & 1, restore=(x >> 8) & 1,
                init=(x >> 9) & 1, pair=(x >> 10) & 1, eroded=(x >> 11) & 1, off=x >> 12, cidx=y & ((1 << 20) - 1),
                rslot=(y >> 20) & 7, sslot=(y >> 23) & 7, q=(y >> 26) & 63)


def _from_view(o, a, b):
    # inverse of the octant view transforms documented in include/lpf.h (lpf_paths_program)
    return [(a, b), (b, a), (-b, a), (-a, b)][o]


def _balanced(q, K):
    """Any two factors of equal length of the K-step pattern differ by at most one in their number of down steps."""
    bits = [(q >> j) & 1 for j in range(K)]
    for L in range(1, K + 1):
        sums = [sum(bits[s:s + L]) for s in range(K - L + 1)]
        if max(sums) - min(sums) > 1:
            return False
    return True


@pytest.mark.parametrize("m,H,W,piece,flags,level", [
    (5, 8, 8, 0, 0, -1), (12, 40, 100, 16, 0, -1), (33, 64, 64, 256, 0, -1), (70, 300, 128, 512, 0, -1),
    (12, 40, 100, 16, 0, 1), (33, 64, 64, 256, 0, 2), (33, 64, 64, 64, 0, 3), (70, 300, 128, 512, 0, 1),
    (33, 64, 64, 64, 0, 4), (60, 64, 64, 256, 0, 5), (60, 64, 64, 256, 0, 6), (100, 512, 512, 512, 0, 6),
    (100, 128, 128, 512, 0, 6),
    (2, 8, 9, 0, 0, 3), (3, 8, 9, 4, 0, 3), (1, 5, 5, 0, 0, -1), (7, 9, 8, 0, 0, 6),
    (12, 13, 13, 0, lpf.LPF_NO_TRIE, -1), (12, 64, 32, 64, lpf.LPF_NO_TRIE, -1), (33, 64, 64, 256, lpf.LPF_NO_E2, -1),
    (40, 41, 97, 64, lpf.LPF_NO_E2, -1), (33, 64, 64, 256, 0, 0),
    # little shared memory: the classes of steep slopes run at lower levels than the program's (negative level = that
    # many KiB for a CTA, automatic level)
    (40, 64, 64, 64, 0, -24), (40, 64, 64, 0, 0, -32), (24, 33, 40, 16, 0, -16), (33, 64, 96, 64, 0, -20)])
def test_program_walk_reproduces_every_canonical_path_once(m, H, W, piece, flags, level):
    """Interpret the node program on the host with a stack of pixel lists instead of masks:
    every terminal must be reached exactly once with exactly the pixel list P_v, and the row-strip
    reload flag must be set whenever the row, word column or plane differs from the previous entry.
    At level K >= 1 a window covers K + 1 pixels of which the first `back` must already be the tail of the
    running list; the vectors shorter than K have no entry (a separate kernel counts them)."""
    p = lpf.lpf_build_paths(m, -1)
    smem_kib = 0
    if level < -1:
        smem_kib, level = -level, -1
        lpf.lpf_set_shared_memory(p, smem_kib * 1024)
    lpf.lpf_set_level(p, level)
    entries, items, n_slots, strides = lpf.lpf_paths_program(p, H, W, piece, flags)
    d = _decode(entries)
    K = strides[8]
    if flags & (lpf.LPF_NO_E2 | lpf.LPF_NO_TRIE) or level == 0:
        assert K == 0
    elif level > 0:
        assert 1 <= K <= min(level, m)                       # lpf_set_level is a cap
        if m >= 12:
            assert K == level                                # these shapes are small: every level fits
    else:
        assert 1 <= K <= min(6, m)                           # the default program is an eroded one
    # pattern classes: slope sectors of one octant; the patterns of a class are balanced words, one plane slot each
    n_classes = strides[9]
    classes = []
    for c in range(n_classes):
        rec = strides[10 + 41 * c: 10 + 41 * (c + 1)]
        octant, n, bw, rows, Kc = rec[0], rec[1], rec[2], rec[3], rec[4]
        pats = rec[5:5 + n]
        assert 0 <= octant < 4 and 1 <= n <= 36 and len(set(pats)) == n and 1 <= Kc <= K
        assert all(0 <= q < (1 << Kc) and _balanced(q, Kc) for q in pats)
        assert all(q == -1 for q in rec[5 + n:])
        # the class's band: only the rows its paths reach, never more than the full-height band, and its n planes and
        # the plain band fit where the geometry reserved full-height bands
        assert rows * strides[octant] <= bw <= strides[4 + octant] and bw % 4 == 0
        classes.append((octant, pats, bw, rows, Kc))
    assert (n_classes > 0) == (K > 0)
    if smem_kib:                                             # mixed levels: a steep class below a shallow one
        assert len({c[4] for c in classes}) > 1 or max(c[4] for c in classes) < K
    if (m, H, W, level) == (100, 512, 512, 6):
        assert n_classes > 4                                 # a band of this shape has room for few planes: several classes
    S = 2 * m + 1
    seen = {}
    covered = np.zeros(len(entries), dtype=bool)
    assert n_slots <= 8
    for first, cnt, o, cls in items:
        cur, stack, held = None, {}, None
        assert strides[o] % 2 == 1
        if K:
            assert classes[cls][0] == o
        for e in range(first, first + cnt):
            assert not covered[e]
            covered[e] = True
            assert bool(d["init"][e]) == (e == first)        # the kernel initialises the mask once, at the item's start
            if d["init"][e]:
                cur = []
            elif d["restore"][e]:
                cur = list(stack[int(d["rslot"][e])])
            assert cur is not None
            assert bool(d["eroded"][e]) == (K > 0)
            q = int(d["q"][e])
            slot, rem = divmod(int(d["off"][e]), classes[cls][2]) if K else (0, int(d["off"][e]))
            if K:
                assert classes[cls][1][slot] == q            # the plane slot holds the entry's pattern
            bv, col = divmod(rem, strides[o])
            av = col * 32 + int(d["sh"][e])
            plane = slot if K else -1
            if d["reload"][e]:
                held = (bv, col, plane)
            assert held == (bv, col, plane), "stale row strip"
            Kc = classes[cls][4] if K else 0                 # the level of the item's class
            window = [(av, bv)]                              # the Kc + 1 pixels of the plane of pattern q at (av, bv)
            for j in range(1, Kc + 1):
                window.append((window[-1][0] + 1, window[-1][1] + ((q >> (j - 1)) & 1)))
            for a, b in window:
                assert 0 <= b <= a <= m
                assert not K or b < classes[cls][3]          # inside the class's band (start row 0)
            window = [_from_view(o, a, b) for a, b in window]
            # the first pixels of a window may be nodes that are already in the mask: as many as the list is longer than
            # the window's first column
            back = len(cur) - av
            assert 0 <= back <= Kc
            if d["init"][e]:
                assert back == 0 and window[0] == (0, 0)     # every item starts at the root with a full window
            assert back == 0 or cur[-back:] == window[:back]
            cur = cur + window[back:]
            if d["terminal"][e]:
                cidx = int(d["cidx"][e])
                dy, dx = cidx // S - m, cidx % S - m
                assert (dx, dy) == cur[-1]
                assert (dx, dy) not in seen
                seen[(dx, dy)] = cur
            if d["save"][e]:
                assert int(d["sslot"][e]) < max(n_slots, 1)
                stack[int(d["sslot"][e])] = list(cur)
            # PAIR: this entry's own mask is never needed and the next entry of the item continues from it
            want_pair = (not d["terminal"][e] and not d["save"][e] and e + 1 < first + cnt
                         and not d["init"][e + 1] and not d["restore"][e + 1])
            assert bool(d["pair"][e]) == bool(want_pair)
    assert covered.all()
    # vectors whose path has fewer than K + 1 pixels have no entry
    short = [(dx, dy) for dy in range(0, m + 1) for dx in range(-m, m + 1)
             if orc.in_half(dx, dy) and max(abs(dx), abs(dy)) < K]
    assert len(short) == (2 * (K - 1) * (K - 1) + 2 * (K - 1) + 1 if K else 0)
    assert not (set(short) & set(seen))
    assert len(seen) + len(short) == 2 * m * m + 2 * m + 1
    for (dx, dy), pix in seen.items():
        assert orc.in_half(dx, dy)
        assert pix == [tuple(int(t) for t in r) for r in orc.path(dx, dy)], (dx, dy)


def test_balanced_pattern_counts_and_classes_of_config3():
    """The K-step patterns of digital straight segments are the balanced words: 2, 4, 8, 14, 24, 36 of them for K = 1..6
    (1 + sum over i <= K of (K - i + 1) phi(i), the number of factors of length K of Sturmian words).  The program of
    config 3 (512 x 512, m = 256) is of level 6; a class has as many planes as fit in shared memory beside its plain band
    (7 at full band height, more for the shallow slopes whose bands are lower), and the classes together cover every pattern."""
    from math import gcd
    for K, want in zip(range(1, 7), (2, 4, 8, 14, 24, 36)):
        phi = lambda n: sum(1 for k in range(1, n + 1) if gcd(k, n) == 1)
        assert want == 1 + sum((K - i + 1) * phi(i) for i in range(1, K + 1))
        assert want == sum(1 for q in range(1 << K) if _balanced(q, K))
    p = lpf.lpf_build_paths(256, -1)
    entries, items, n_slots, layout = lpf.lpf_paths_program(p, 512, 512, 1024, 0)
    assert layout[8] == 6 and n_slots <= 8
    n_classes = layout[9]
    per_octant = {}
    for c in range(n_classes):
        rec = layout[10 + 41 * c: 10 + 41 * (c + 1)]
        assert 1 <= rec[1] <= 36 and (rec[1] + 1) * rec[2] <= 8 * layout[4 + rec[0]]    # planes + plain band fit
        if rec[4] == 6:
            per_octant.setdefault(rec[0], set()).update(rec[5:5 + rec[1]])
        else:
            assert rec[4] == 5 and rec[1] <= 7                   # the steepest classes: room for 7 planes only
    assert 20 <= n_classes <= 48 and sorted(per_octant) == [0, 1, 2, 3]
    assert all(30 <= len(v) <= 36 for v in per_octant.values())
    assert len(entries) < 900000                                 # 5.0 M trie nodes: more than 5.5 nodes per entry
