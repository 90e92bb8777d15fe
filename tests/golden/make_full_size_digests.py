"""Writes the full-size expected values of configs 3, 4 and 5 (BASELINE.json) as small text digests.

    python tests/golden/make_full_size_digests.py [3] [4] [5]

Every number comes from `oracle/` on the seeded inputs of `paper_1601_04359_b200/inputs.py` (which holds no method
arithmetic); nothing here imports, loads or calls the CUDA library.  The whole-config oracle runs take minutes on a few
cores (config 3: 131 585 canonical vectors x 512 x 512 start pixels x 2 phases, Alg. 1 as printed),
too long for every test run, so the tests compare the CUDA result with these digests instead:

  config3_counts.digest.txt   sha256 of the int64 [2][513][513] counts (little endian, C order) + crc32 of every row
  config4_counts.digest.txt   sha256 of the int64 [1024][129][129] counts + per image: crc32 of its counts and the exact
                              Eq. 14/19 squared error against the target image's counts
  config5_deltas.digest.txt   crc32 of the int32 [129][129] swap delta (definition-level local form, pinned to the
                              full re-evaluation in tests/test_oracle_swap.py) of the first 1000 proposals for phase 1
                              and the first 200 for phase 0 (reading S10)
"""
from __future__ import annotations

import hashlib
import os
import sys
import time
import zlib
from multiprocessing import Pool

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import lpf_oracle as orc  # noqa: E402
from paper_1601_04359_b200 import inputs  # noqa: E402


def crc(a: np.ndarray) -> str:
    return "%08x" % (zlib.crc32(np.ascontiguousarray(a).tobytes()) & 0xFFFFFFFF)


def sha(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def config3():
    img = inputs.config_image(3)
    m = 256
    t0 = time.time()
    c = np.stack([orc.counts(img, ph, m) for ph in (0, 1)]).astype("<i8")
    with open(os.path.join(HERE, "config3_counts.digest.txt"), "w") as f:
        f.write("# config 3 (BASELINE.json): 512x512 thresholded Gaussian field, both phases, m = 256\n")
        f.write("# counts[phase][dy+m][dx+m] by oracle/lpf_oracle.c lpf_oracle_counts (Alg. 1, PAPER.md:216-250; canonical\n")
        f.write("# half evaluated, the rest by Eq. 12, PAPER.md:142-148), written by tests/golden/make_full_size_digests.py\n")
        f.write("sha256 %s\n" % sha(c))
        for ph in (0, 1):
            for r in range(2 * m + 1):
                f.write("row %d %d %s\n" % (ph, r, crc(c[ph, r])))
    print("config 3 done in %.0f s" % (time.time() - t0), flush=True)


def config4():
    B, m = 1024, 64
    imgs, target_img = inputs.config4_batch(B)
    t0 = time.time()
    target = orc.counts(target_img, 1, m)
    c = np.stack([orc.counts(imgs[b], 1, m) for b in range(B)]).astype("<i8")
    with open(os.path.join(HERE, "config4_counts.digest.txt"), "w") as f:
        f.write("# config 4 (BASELINE.json): 1024 disk images 128x128 (+ target = image index 1024), phase 1, m = 64\n")
        f.write("# oracle counts (lpf_oracle_counts) and exact squared error vs the target (lpf_oracle_sse, Eq. 14/19,\n")
        f.write("# PAPER.md:162, 400), written by tests/golden/make_full_size_digests.py\n")
        f.write("sha256 %s\n" % sha(c))
        f.write("target %s\n" % crc(target.astype("<i8")))
        for b in range(B):
            f.write("img %d %s %d\n" % (b, crc(c[b]), orc.sse(c[b], target)))
    print("config 4 done in %.0f s" % (time.time() - t0), flush=True)


_IMG5 = None


def _delta5(job):
    global _IMG5
    if _IMG5 is None:
        _IMG5 = inputs.config_image(5)
    phase, pair = job
    return crc(orc.swap_delta_local(_IMG5, phase, 64, pair).astype("<i4"))


def config5():
    img = inputs.config_image(5)
    pairs = inputs.config5_pairs(img, 100000)
    t0 = time.time()
    jobs = [(1, tuple(int(v) for v in pairs[i])) for i in range(1000)] + \
           [(0, tuple(int(v) for v in pairs[i])) for i in range(200)]
    with Pool(os.cpu_count() or 1) as pool:
        out = pool.map(_delta5, jobs, chunksize=8)
    with open(os.path.join(HERE, "config5_deltas.digest.txt"), "w") as f:
        f.write("# config 5 (BASELINE.json): 256x256 disk image, m = 64, proposals inputs.config5_pairs(img, 100000)\n")
        f.write("# crc32 of the int32 [129][129] delta of proposal i by oracle lpf_oracle_swap_delta_local\n")
        f.write("# (PAPER.md:357-359), written by tests/golden/make_full_size_digests.py\n")
        for (phase, _), (i, h) in zip(jobs, [(k if k < 1000 else k - 1000, h) for k, h in enumerate(out)]):
            f.write("swap %d %d %s\n" % (phase, i, h))
    print("config 5 done in %.0f s" % (time.time() - t0), flush=True)


if __name__ == "__main__":
    which = [int(a) for a in sys.argv[1:]] or [5, 4, 3]
    for c in which:
        {3: config3, 4: config4, 5: config5}[c]()
