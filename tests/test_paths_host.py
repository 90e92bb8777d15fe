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
    assert lib.lpf_strerror(lpf.LPF_E_UNSUPPORTED) == b"unsupported shape"
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
                init=(x >> 9) & 1, pair=(x >> 10) & 1, e2=(x >> 11) & 1, off=x >> 12, cidx=y & ((1 << 20) - 1), rslot=(y >> 20) & 15, sslot=(y >> 24) & 15, back=(y >> 28) & 1,
                d2=(y >> 29) & 1, rootcount=(y >> 30) & 1)


def _from_view(o, a, b):
    # inverse of the octant view transforms documented in include/lpf.h (lpf_paths_program)
    return [(a, b), (b, a), (-b, a), (-a, b)][o]


@pytest.mark.parametrize("m,H,W,piece,flags", [(5, 8, 8, 0, 0), (12, 40, 100, 16, 0), (33, 64, 64, 256, 0),
                                               (70, 300, 128, 512, 0), (12, 13, 13, 0, lpf.LPF_NO_TRIE),
                                               (12, 64, 32, 64, lpf.LPF_NO_TRIE), (33, 64, 64, 256, lpf.LPF_NO_E2),
                                               (40, 41, 97, 64, lpf.LPF_NO_E2)])
def test_program_walk_reproduces_every_canonical_path_once(m, H, W, piece, flags):
    """Interpret the node program on the host with a stack of pixel lists instead of masks:
    every terminal must be reached exactly once with exactly the pixel list P_v, and the row-strip
    reload flag must be set whenever the row or word column differs from the previous entry."""
    p = lpf.lpf_build_paths(m, -1)
    entries, items, n_slots, strides = lpf.lpf_paths_program(p, H, W, piece, flags)
    d = _decode(entries)
    S = 2 * m + 1
    seen = {}
    covered = np.zeros(len(entries), dtype=bool)
    assert n_slots <= 8
    for first, cnt, o, _ in items:
        cur, stack, held = None, {}, None
        assert strides[o] % 2 == 1
        eroded = strides[4 + o] > 0                          # shared memory holds E2 and D2 instead of the plain plane
        if eroded:
            assert not (flags & (lpf.LPF_NO_E2 | lpf.LPF_NO_TRIE))
        for e in range(first, first + cnt):
            assert not covered[e]
            covered[e] = True
            assert bool(d["init"][e]) == (e == first)        # the kernel initialises the mask once, at the item's start
            if d["init"][e]:
                cur = [(0, 0)] if eroded else []             # eroded mode: INIT loads the root pixel from the plain view
                if d["rootcount"][e]:
                    assert eroded and o == 0 and (0, 0) not in seen
                    seen[(0, 0)] = [(0, 0)]
            elif d["restore"][e]:
                cur = list(stack[int(d["rslot"][e])])
            assert cur is not None and not (d["rootcount"][e] and not d["init"][e])
            plane = (2 if d["d2"][e] else 1) if d["e2"][e] else 0
            assert (plane > 0) == eroded
            bv, col = divmod(int(d["off"][e]) - (strides[4 + o] if plane == 2 else 0), strides[o])
            av = col * 32 + int(d["sh"][e])
            assert 0 <= bv <= av <= m
            if d["reload"][e]:
                held = (bv, col, plane)
            assert held == (bv, col, plane), "stale row strip"
            if plane == 0:
                assert not d["back"][e]
                cur = cur + [_from_view(o, av, bv)]
            else:
                second = (av + 1, bv) if plane == 1 else (av + 1, bv + 1)    # E2: right neighbour, D2: lower right
                assert second[1] <= second[0] <= m
                if d["back"][e]:                             # one node, read at its parent: the first pixel is old
                    assert cur[-1] == _from_view(o, av, bv)
                else:                                        # a node whose mask is never needed and its only child
                    cur = cur + [_from_view(o, av, bv)]
                cur = cur + [_from_view(o, *second)]
            if d["terminal"][e]:
                cidx = int(d["cidx"][e])
                dy, dx = cidx // S - m, cidx % S - m
                assert (dx, dy) == cur[-1]
                assert (dx, dy) not in seen
                seen[(dx, dy)] = cur
            if d["save"][e]:
                assert int(d["sslot"][e]) < max(n_slots, 1)
                stack[int(d["sslot"][e])] = list(cur)
            # PAIR: this node's own mask is never needed and the next entry of the item continues from it
            want_pair = (not d["terminal"][e] and not d["save"][e] and e + 1 < first + cnt
                         and not d["init"][e + 1] and not d["restore"][e + 1])
            assert bool(d["pair"][e]) == bool(want_pair)
    assert covered.all()
    assert len(seen) == 2 * m * m + 2 * m + 1
    if not (flags & (lpf.LPF_NO_E2 | lpf.LPF_NO_TRIE)) and m >= 1:
        assert d["e2"].all() and d["d2"].any() and (~d["d2"].astype(bool)).any()   # the default program is the eroded one
    for (dx, dy), pix in seen.items():
        assert orc.in_half(dx, dy)
        assert pix == [tuple(int(t) for t in r) for r in orc.path(dx, dy)], (dx, dy)
