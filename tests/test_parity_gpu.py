"""GPU parity: the CUDA path behind the C ABI (liblpf.so) against the CPU oracle, bit-exact
(integer counts: SURVEY.md 8(c) S14), on the same seeded inputs (paper_1601_04359_b200.inputs).

Small/medium cases compare element by element with the oracle called in the test.  The full-size configs
3, 4 and 5 are compared IN FULL with digests of the oracle's result (tests/golden/*.digest.txt, written by
tests/golden/make_full_size_digests.py, which calls only oracle/): sha256 of the whole array plus a crc32 per
row / image / proposal so that a mismatch is located; on top of that sampled vectors / images are compared with
the oracle called here, and properties that hold at any size are checked (Eq. 10 and Eq. 12 of the paper,
PAPER.md:131-148; prefix monotonicity)."""
import hashlib
import os
import zlib

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs, lpf

pytestmark = pytest.mark.gpu

_PATHS = {}


def paths(m):
    if m not in _PATHS:
        _PATHS[m] = lpf.lpf_build_paths(m, 0)
    return _PATHS[m]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def digest_lines(name):
    out = []
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            out.append(line.split())
    return out


def crc(a):
    return "%08x" % (zlib.crc32(np.ascontiguousarray(a).tobytes()) & 0xFFFFFFFF)


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def gpu_counts(img, phase, m, flags=0):
    a = img if img.ndim == 3 else img[None]
    out = lpf.lpf_eval(paths(m), dev(a), phase, flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_extension_is_loaded_and_device_is_b200_class():
    lib = lpf.load()
    assert lib is not None and torch.cuda.is_available()
    assert torch.cuda.get_device_capability(0)[0] >= 10


def test_worked_image_golden_on_gpu():
    rows = ["110111", "111101", "011111", "111011"]      # tests/golden/worked_image.txt
    img = np.array([[int(c) for c in r] for r in rows], dtype=np.uint8)
    c1 = gpu_counts(img, 1, 2)[0]
    c0 = gpu_counts(img, 0, 2)[0]
    assert np.array_equal(c1, orc.counts(img, 1, 2, full_template=True))
    assert np.array_equal(c0, orc.counts(img, 0, 2, full_template=True))
    assert c1[2, 2] == 20 and c1[2, 3] == 16 and c1[3, 2] == 16 and c0[1, 3] == 1


@pytest.mark.parametrize("flags", [0, lpf.LPF_PRUNE, lpf.LPF_NO_TRIE, lpf.LPF_PRUNE | lpf.LPF_NO_TRIE])
def test_config1_full_template_bit_exact(flags):
    img = inputs.config_image(1)
    want = orc.counts(img, 1, 16, full_template=True)      # every vector on its own path, no mirroring
    got = gpu_counts(img, 1, 16, flags)[0]
    assert got.dtype == np.int64 and np.array_equal(got, want)


SHAPES = [(1, 1, 0), (1, 7, 0), (2, 2, 1), (3, 5, 2), (8, 8, 7), (12, 9, 8), (33, 31, 30), (31, 33, 12),
          (40, 70, 39), (64, 96, 20), (100, 100, 50), (65, 129, 64), (50, 200, 17), (200, 50, 49)]


@pytest.mark.parametrize("H,W,m", SHAPES)
def test_ragged_shapes_both_phases_all_flags(H, W, m):
    rng = np.random.default_rng(H * 1000 + W)
    img = (rng.random((H, W)) < 0.8).astype(np.uint8)
    img[rng.random((H, W)) < 0.02] = 7                     # bytes other than 0/1 belong to neither phase
    for phase in (0, 1):
        want = orc.counts(img, phase, m, full_template=(H * W <= 4096))
        for flags in (0, lpf.LPF_PRUNE, lpf.LPF_NO_TRIE):
            got = gpu_counts(img, phase, m, flags)[0]
            assert np.array_equal(got, want), (phase, flags)


@pytest.mark.parametrize("size", [50, 200, 500])
def test_tab1_morphologies_entire_domain(size):
    """The paper's Tab. 1 workloads: chess with 10x10 px fields and 4x4 px squares, ALL segments up to
    (W-1, H-1) (m = size - 1, widths that are not multiples of 32), standard and enhanced, sampled vectors.  At 500 a
    plane is 563 rows and two of them fit in shared memory beside the plain band: the pattern classes run at mixed
    levels (6 for the shallow slopes down to 1 for the steepest)."""
    m = size - 1
    rng = np.random.default_rng(size)
    vecs = rng.integers(-m, m + 1, size=(150, 2))
    for img in (inputs.chess(size, size, 10), inputs.squares(size, size, 4, 0.20, inputs.seed_for(6, size))):
        for flags in (0, lpf.LPF_PRUNE):
            both = lpf.lpf_eval_both(paths(m), dev(img[None]), flags)
            torch.cuda.synchronize()
            c = both.cpu().numpy()[0]
            for phase in (0, 1):
                want, _ = orc.counts_list(img, phase, vecs)
                assert np.array_equal(c[phase][vecs[:, 1] + m, vecs[:, 0] + m], want)
                assert c[phase][m, m] == int((img == phase).sum())
                assert np.array_equal(c[phase], c[phase][::-1, ::-1])


def test_degenerate_images():
    H, W, m = 48, 80, 20
    S = 2 * m + 1
    full = np.ones((H, W), dtype=np.uint8)
    assert np.array_equal(gpu_counts(full, 1, m)[0], np.full((S, S), H * W))
    assert np.array_equal(gpu_counts(full, 0, m)[0], np.zeros((S, S)))
    assert np.array_equal(gpu_counts(1 - full, 1, m, lpf.LPF_PRUNE)[0], np.zeros((S, S)))
    stripes = inputs.stripes(H, W, 8, 3, horizontal=True)
    got = gpu_counts(stripes, 1, m)[0]
    dy = np.abs(np.arange(-m, m + 1))[:, None]
    want = np.broadcast_to(W * (H // 8) * np.maximum(0, 3 - dy), (S, S))
    assert np.array_equal(got, want)


def test_eval_both_and_batch_match_single_calls():
    rng = np.random.default_rng(5)
    imgs = (rng.random((5, 40, 64)) < 0.7).astype(np.uint8)
    m = 24
    both = lpf.lpf_eval_both(paths(m), dev(imgs)).cpu().numpy()
    for b in range(5):
        for phase in (0, 1):
            assert np.array_equal(both[b, phase], orc.counts(imgs[b], phase, m))
    one = gpu_counts(imgs, 1, m)
    assert np.array_equal(one, both[:, 1])


def test_error_codes_on_device():
    p = paths(16)
    img = dev(np.zeros((1, 16, 64), dtype=np.uint8))
    with pytest.raises(lpf.LpfError) as e:
        lpf.lpf_eval(p, img, 1)                            # m > min(H, W) - 1
    assert e.value.code == lpf.LPF_E_INVAL
    with pytest.raises(lpf.LpfError) as e:
        lpf.lpf_eval(p, dev(np.zeros((1, 64, 64), dtype=np.uint8)), 2)
    assert e.value.code == lpf.LPF_E_INVAL


def test_config2_both_phases_bit_exact():
    img = inputs.config_image(2)
    got = lpf.lpf_eval_both(paths(128), dev(img[None])).cpu().numpy()[0]
    for phase in (0, 1):
        assert np.array_equal(got[phase], orc.counts(img, phase, 128)), phase


def _properties(counts, img, phase, m):
    S = 2 * m + 1
    assert counts[m, m] == int((img == phase).sum())                 # Eq. 10
    assert np.array_equal(counts, counts[::-1, ::-1])                 # Eq. 12
    assert counts.max() == counts[m, m] and counts.min() >= 0
    ax = counts[m, m:]
    assert np.all(ax[1:] <= ax[:-1])                                  # axis-aligned: non-increasing
    ay = counts[m:, m]
    assert np.all(ay[1:] <= ay[:-1])
    assert counts.shape == (S, S)


def test_config3_sampled_vectors_and_properties():
    img = inputs.config_image(3)
    m = 256
    got = lpf.lpf_eval_both(paths(m), dev(img[None])).cpu().numpy()[0]
    rng = np.random.default_rng(3)
    vecs = np.concatenate([rng.integers(-m, m + 1, size=(1500, 2)),
                           np.array([[0, 0], [m, m], [-m, m], [m, 0], [0, m], [m, -m], [-m, -m], [1, 0], [255, 256],
                                     [256, 255], [-256, 1], [31, 1], [32, 1], [33, 1], [-31, 2], [-32, 2], [-33, 2]])])
    for phase in (0, 1):
        want, _ = orc.counts_list(img, phase, vecs)
        assert np.array_equal(got[phase][vecs[:, 1] + m, vecs[:, 0] + m], want), phase
        _properties(got[phase], img, phase, m)
    pruned = lpf.lpf_eval_both(paths(m), dev(img[None]), lpf.LPF_PRUNE).cpu().numpy()[0]
    assert np.array_equal(pruned, got)


def test_config3_whole_template_against_the_oracle_digest():
    """ALL 2 x 513 x 513 counts of config 3 against the oracle's (tests/golden/config3_counts.digest.txt): crc32 of
    every row, then sha256 of the whole array; default flags, LPF_PRUNE and LPF_NO_E2."""
    img = inputs.config_image(3)
    m = 256
    lines = digest_lines("config3_counts.digest.txt")
    want_sha = [t[1] for t in lines if t[0] == "sha256"][0]
    rows = {(int(t[1]), int(t[2])): t[3] for t in lines if t[0] == "row"}
    assert len(rows) == 2 * (2 * m + 1)
    for flags in (0, lpf.LPF_PRUNE, lpf.LPF_NO_E2):
        got = lpf.lpf_eval_both(paths(m), dev(img[None]), flags).cpu().numpy()[0].astype("<i8")
        bad = [(ph, r) for ph in (0, 1) for r in range(2 * m + 1) if crc(got[ph, r]) != rows[(ph, r)]]
        assert not bad, (flags, bad[:10])
        assert sha(got) == want_sha, flags
        assert lpf.lpf_last_launch_info(paths(m))["level"] == (0 if flags & lpf.LPF_NO_E2 else 6)


def test_config4_sampled_images_properties_and_objective():
    B = 1024
    imgs, target_img = inputs.config4_batch(B)
    m = 64
    p = paths(m)
    d_counts = lpf.lpf_eval(p, dev(imgs), 1)
    d_target = lpf.lpf_eval(p, dev(target_img[None]), 1)
    sse = lpf.lpf_objective(d_counts, d_target[0]).cpu().numpy()
    counts = d_counts.cpu().numpy()
    target = d_target.cpu().numpy()[0]
    assert np.array_equal(target, orc.counts(target_img, 1, m))
    # ALL 1024 images against the oracle's digest: crc32 of every image's counts, its exact squared error, sha256 of all
    lines = digest_lines("config4_counts.digest.txt")
    per_img = {int(t[1]): (t[2], int(t[3])) for t in lines if t[0] == "img"}
    assert len(per_img) == B
    assert crc(target.astype("<i8")) == [t[1] for t in lines if t[0] == "target"][0]
    bad = [b for b in range(B) if crc(counts[b].astype("<i8")) != per_img[b][0] or int(sse[b]) != per_img[b][1]]
    assert not bad, bad[:10]
    assert sha(counts.astype("<i8")) == [t[1] for t in lines if t[0] == "sha256"][0]
    # 64 images element by element against the oracle called here (every 16th, the last group included)
    for b in list(range(0, B, 16))[:62] + [1022, 1023]:
        want = orc.counts(imgs[b], 1, m)
        assert np.array_equal(counts[b], want), b
        assert int(sse[b]) == orc.sse(want, target)
    # every image: Eq. 10, Eq. 12, and the objective recomputed from the GPU counts by the oracle's sse
    assert np.array_equal(counts[:, m, m], imgs.reshape(B, -1).sum(axis=1))
    assert np.array_equal(counts, counts[:, ::-1, ::-1])
    for b in range(0, B, 37):
        assert int(sse[b]) == orc.sse(counts[b], target)
    # the same image twice gives sse 0
    assert int(lpf.lpf_objective(d_target, d_target[0]).cpu().numpy()[0]) == 0


def test_objective_exact_large_values():
    rng = np.random.default_rng(11)
    c = rng.integers(0, 2 ** 26, size=(7, 4099), dtype=np.int64)
    t = rng.integers(0, 2 ** 26, size=(4099,), dtype=np.int64)
    got = lpf.lpf_objective(dev(c), dev(t)).cpu().numpy()
    for b in range(7):
        assert int(got[b]) == orc.sse(c[b], t)


def _swapped_images(d_img, d_pairs):
    """[n, H, W] copies of the base image with the two pixels of each proposal exchanged (built on the device)."""
    n = d_pairs.shape[0]
    mod = d_img.expand(n, -1, -1).contiguous()
    idx = torch.arange(n, device=d_img.device)
    xp, yp, xq, yq = (d_pairs[:, k].long() for k in range(4))
    bp, bq = d_img[0, yp, xp], d_img[0, yq, xq]
    mod[idx, yp, xp] = bq
    mod[idx, yq, xq] = bp
    return mod


def test_config5_swap_delta_all_proposals():
    """Config 5: 100 000 proposals on the 256 x 256 disk image, m = 64.  (i) EVERY delta against a full re-evaluation
    of I' by lpf_eval (itself verified against the oracle) minus the base counts; (ii) the first 1000 (phase 1) and 200
    (phase 0) against the oracle's definition-level delta through its digest; (iii) 24 + 3 against the oracle called
    here (local form / full re-evaluation); invariants on all."""
    img = inputs.config_image(5)
    m = 64
    p = paths(m)
    n = 100000
    pairs = inputs.config5_pairs(img, n)
    d_img = dev(img[None])
    d_pairs = dev(pairs)
    S = 2 * m + 1
    dig = {(int(t[1]), int(t[2])): t[3] for t in digest_lines("config5_deltas.digest.txt") if t[0] == "swap"}
    assert sum(1 for k in dig if k[0] == 1) == 1000 and sum(1 for k in dig if k[0] == 0) == 200
    for phase, count in ((1, n), (0, 4000)):
        base = lpf.lpf_eval(p, d_img, phase)[0]
        assert np.array_equal(base.cpu().numpy(), orc.counts(img, phase, m))
        chunk = 2000
        for s0 in range(0, count, chunk):
            d = lpf.lpf_swap_delta(p, d_img, phase, d_pairs[s0:s0 + chunk])
            assert d.shape == (chunk, S, S)
            assert bool((d[:, m, m] == 0).all())                          # volume fraction preserved
            assert bool((d == d.flip(1, 2)).all())                        # delta(v) = delta(-v)
            re = lpf.lpf_eval(p, _swapped_images(d_img, d_pairs[s0:s0 + chunk]), phase) - base[None]
            same = (re == d.to(torch.int64)).flatten(1).all(dim=1)
            assert bool(same.all()), (phase, s0, torch.nonzero(~same).flatten()[:10].tolist())
            if s0 == 0:
                dn = d.cpu().numpy().astype("<i4")
                lim = 1000 if phase == 1 else 200
                bad = [i for i in range(lim) if crc(dn[i]) != dig[(phase, i)]]
                assert not bad, (phase, bad[:10])
                for i in range(24 if phase == 1 else 6):
                    assert np.array_equal(dn[i], orc.swap_delta_local(img, phase, m, pairs[i])), i
                for i in range(3 if phase == 1 else 1):
                    assert np.array_equal(dn[i], orc.swap_delta_full(img, phase, m, pairs[i])), i
            del d, re


def test_swap_delta_dense_image_overflows_the_warp_stacks():
    """An image that is >= 95 % in phase: almost every prefix survives, the per-warp stacks of swap_delta_kernel_v3
    fill up and the serial fall-back walk runs.  Every delta against full re-evaluation on the GPU, a few against the
    oracle; both phases."""
    H = W = 160
    m = 64
    rng = np.random.default_rng(95)
    img = (rng.random((H, W)) < 0.97).astype(np.uint8)
    p = paths(m)
    pairs = inputs.swap_pairs(img, 96, 96)
    d_img, d_pairs = dev(img[None]), dev(pairs)
    for phase in (1, 0):
        base = lpf.lpf_eval(p, d_img, phase)[0]
        d = lpf.lpf_swap_delta(p, d_img, phase, d_pairs)
        re = lpf.lpf_eval(p, _swapped_images(d_img, d_pairs), phase) - base[None]
        assert bool((re == d.to(torch.int64)).all()), phase
        dn = d.cpu().numpy()
        for i in range(3):
            assert np.array_equal(dn[i], orc.swap_delta_local(img, phase, m, pairs[i])), (phase, i)
    assert int(d_img.sum()) > 0.95 * H * W


def test_swap_delta_sparse_phase_with_large_live_regions_on_the_reversed_trie():
    """Broad stripes that fill 47 % of the image: the phase counts as sparse (below one half), so the backward walks run
    on the reversed trie, but inside a stripe almost every walk survives: the CTA's stack overflows and the serial
    fall-back over the reversed trie runs.  The complementary phase (53 %, per-node walks) rides along.  Every delta
    against full re-evaluation on the GPU, a few against the oracle."""
    H, W, m = 192, 256, 64
    img = np.zeros((H, W), dtype=np.uint8)
    img[:, 10:70] = 1
    img[:, 130:190] = 1
    rng = np.random.default_rng(47)
    img[rng.random((H, W)) < 0.002] ^= 1                      # a few defects so that not everything is one run
    assert 0.44 < img.mean() < 0.5
    p = paths(m)
    pairs = inputs.swap_pairs(img, 48, 47)
    d_img, d_pairs = dev(img[None]), dev(pairs)
    for phase in (1, 0):
        base = lpf.lpf_eval(p, d_img, phase)[0]
        d = lpf.lpf_swap_delta(p, d_img, phase, d_pairs)
        re = lpf.lpf_eval(p, _swapped_images(d_img, d_pairs), phase) - base[None]
        assert bool((re == d.to(torch.int64)).all()), phase
        dn = d.cpu().numpy()
        for i in range(2):
            assert np.array_equal(dn[i], orc.swap_delta_local(img, phase, m, pairs[i])), (phase, i)


def test_swap_delta_small_and_degenerate_pairs():
    rng = np.random.default_rng(9)
    H, W, m = 20, 45, 11
    img = (rng.random((H, W)) < 0.6).astype(np.uint8)
    p = paths(m)
    pairs = inputs.swap_pairs(img, 40, 123)
    pairs[0] = (3, 4, 3, 4)                                            # same pixel: nothing changes
    zy, zx = np.nonzero(img == 0)
    pairs[1] = (zx[0], zy[0], zx[1], zy[1])                            # same phase: nothing changes
    pairs[2] = (-1, 0, 5, 5)                                           # out of range: all-zero delta
    got = lpf.lpf_swap_delta(p, dev(img[None]), 1, dev(pairs)).cpu().numpy()
    assert not got[0].any() and not got[1].any() and not got[2].any()
    for i in range(3, 40):
        assert np.array_equal(got[i], orc.swap_delta_full(img, 1, m, pairs[i])), i


def test_eval_host_end_to_end_entry():
    img = inputs.config_image(1)
    got = lpf.lpf_eval_host(paths(16), img, 1)
    assert np.array_equal(got[0], orc.counts(img, 1, 16))
    both = lpf.lpf_eval_host(paths(16), img, -1)
    assert np.array_equal(both[0, 0], orc.counts(img, 0, 16))


# ---- S2 (LPF_S2, Eq. 6) and masked L2~ (lpf_eval_masked) -------------------------------------

@pytest.mark.parametrize("H,W,m", [(1, 1, 0), (3, 5, 2), (12, 9, 8), (33, 31, 30), (40, 70, 39), (96, 128, 63)])
def test_s2_counts_bit_exact(H, W, m):
    rng = np.random.default_rng(7 * H + W)
    img = (rng.random((H, W)) < 0.55).astype(np.uint8)
    img[rng.random((H, W)) < 0.03] = 5
    for phase in (0, 1):
        want = orc.s2_counts(img, phase, m)
        for flags in (lpf.LPF_S2, lpf.LPF_S2 | lpf.LPF_PRUNE):
            got = gpu_counts(img, phase, m, flags)[0]
            assert np.array_equal(got, want), (phase, flags)
    both = lpf.lpf_eval_both(paths(m), dev(img[None]), lpf.LPF_S2).cpu().numpy()[0]
    assert np.array_equal(both[0], orc.s2_counts(img, 0, m)) and np.array_equal(both[1], orc.s2_counts(img, 1, m))


def test_s2_config2_size_against_fft_form():
    """Full config-2 size: the exact integer S2 counts equal the rounded FFT autocorrelation of Eq. 7."""
    img = inputs.config_image(2)
    m = 128
    got = gpu_counts(img, 1, m, lpf.LPF_S2)[0]
    chi = (img == 1).astype(np.float64)
    F = np.fft.fft2(chi)
    corr = np.rint(np.fft.ifft2(F * np.conj(F)).real).astype(np.int64)
    idx = (np.arange(-m, m + 1)) % 256
    assert np.array_equal(got, corr[np.ix_((-np.arange(-m, m + 1)) % 256, (-np.arange(-m, m + 1)) % 256)])
    assert idx.size == 2 * m + 1


@pytest.mark.parametrize("H,W,m", [(2, 2, 1), (12, 9, 8), (31, 33, 12), (64, 96, 20), (65, 129, 64)])
def test_masked_eval_matches_oracle_on_canonical_half(H, W, m):
    rng = np.random.default_rng(H + 31 * W)
    img = (rng.random((H, W)) < 0.8).astype(np.uint8)
    mask = (rng.random((H, W)) < 0.3).astype(np.uint8) * rng.integers(1, 255, size=(H, W)).astype(np.uint8)
    p = paths(m)
    vecs = np.array([(dx, dy) for dy in range(0, m + 1) for dx in range(-m, m + 1)
                     if orc.in_half(dx, dy)], dtype=np.int32)
    if len(vecs) > 400:
        vecs = vecs[rng.choice(len(vecs), 400, replace=False)]
    for phase in (0, 1):
        want = orc.counts_masked(img, mask, phase, vecs)
        for flags in (0, lpf.LPF_PRUNE, lpf.LPF_NO_TRIE):
            got = lpf.lpf_eval_masked(p, dev(img[None]), phase, dev(mask), flags).cpu().numpy()[0]
            assert np.array_equal(got[vecs[:, 1] + m, vecs[:, 0] + m], want), (phase, flags)
            assert np.array_equal(got, got[::-1, ::-1])       # the half outside D repeats D (reading S16)
            assert got[m, m] == int(((img == phase) & (mask != 0)).sum())
    # all positions selected: exactly lpf_eval; both phases in one call
    ones = np.full((H, W), 200, dtype=np.uint8)
    full = lpf.lpf_eval_both(p, dev(img[None])).cpu().numpy()
    got = lpf.lpf_eval_masked(p, dev(img[None]), -1, dev(ones)).cpu().numpy()
    assert np.array_equal(got, full)
    # no position selected
    assert not lpf.lpf_eval_masked(p, dev(img[None]), 1, dev(np.zeros((H, W), np.uint8))).cpu().numpy().any()


def test_masked_batch_and_s2_combination():
    rng = np.random.default_rng(5)
    H, W, m = 48, 64, 17
    imgs = (rng.random((5, H, W)) < 0.7).astype(np.uint8)
    mask = (rng.random((H, W)) < 0.5).astype(np.uint8)
    p = paths(m)
    got = lpf.lpf_eval_masked(p, dev(imgs), 1, dev(mask)).cpu().numpy()
    vecs = np.array([(3, 0), (0, 5), (-4, 9), (17, 17), (-17, 1), (7, 2)], dtype=np.int32)
    for b in range(5):
        assert np.array_equal(got[b][vecs[:, 1] + m, vecs[:, 0] + m], orc.counts_masked(imgs[b], mask, 1, vecs))
    # masked two-point counts: start pixel selected and in phase, end pixel in phase
    s2m = lpf.lpf_eval_masked(p, dev(imgs[:1]), 1, dev(mask), lpf.LPF_S2).cpu().numpy()[0]
    chi = imgs[0] == 1
    for dx, dy in vecs:
        want = int((chi & (mask != 0) & np.roll(chi, (-dy, -dx), axis=(0, 1))).sum())
        assert s2m[dy + m, dx + m] == want


# ---- simulated annealing (lpf_anneal, Alg. 3) ---------------------------------------------------------------

def _anneal_case(H, W, m, phase, seed, N):
    rng = np.random.default_rng(seed)
    target_img = inputs.squares(H, W, 3, 0.35, seed)
    start = target_img.flatten()
    rng.shuffle(start)
    start = start.reshape(H, W)
    phases = (0, 1) if phase < 0 else (phase,)
    target = np.stack([orc.counts(target_img, ph, m) for ph in phases])
    pairs, log_u = inputs.anneal_proposals(H, W, N, seed + 1)
    E0 = sum(orc.half_sse(orc.counts(start, ph, m), target[i], m) for i, ph in enumerate(phases))
    return start, target, pairs, log_u, E0


@pytest.mark.parametrize("H,W,m,phase,N,c_max,s_max,use_local", [
    (12, 10, 5, 1, 150, 15, 5, False),          # literal oracle (re-evaluates everything per proposal)
    (12, 10, 5, -1, 150, 15, 5, False),
    (24, 40, 11, 0, 600, 60, 12, True),
    (33, 31, 16, -1, 400, 40, 9, True),
])
def test_anneal_chain_is_decision_for_decision_the_oracles(H, W, m, phase, N, c_max, s_max, use_local):
    start, target, pairs, log_u, E0 = _anneal_case(H, W, m, phase, 100 + H, N)
    T_max = 2.0 * E0 / (H * W) ** 2 / 50
    w_img, w_counts, w_st, w_log = orc.anneal(start, phase, m, target, pairs, log_u, T_max, 0.01 * T_max, c_max, s_max,
                                              use_local=use_local)
    d_img = dev(start)
    d_log = torch.zeros(N, dtype=torch.uint8, device="cuda")
    counts, st = lpf.lpf_anneal(paths(m), d_img, phase, dev(target), dev(pairs), dev(log_u), T_max, 0.01 * T_max,
                                c_max, s_max, accept_log=d_log)
    assert np.array_equal(d_log.cpu().numpy(), w_log)                  # every Metropolis decision
    assert np.array_equal(d_img.cpu().numpy(), w_img)
    assert np.array_equal(counts.cpu().numpy(), w_counts)
    assert st == w_st                                                  # steps, accepted, levels, final T (bitwise), E
    assert 0 < w_log.sum() < N


@pytest.mark.parametrize("H,W,m,phase,policy,N", [(24, 40, 11, 1, 1, 500), (33, 31, 16, -1, 2, 400),
                                                   (20, 26, 9, 0, 2, 600), (100, 100, 20, -1, 2, 300)])
def test_anneal_with_generated_proposals_is_the_oracles_chain(H, W, m, phase, policy, N):
    """lpf_anneal_generate: the modification operator draws its own pixels from the current image on the device
    (opposite phases / interfacial, reading A7): proposals, decisions, final image, descriptor and statistics are the
    oracle's."""
    start, target, _, log_u, E0 = _anneal_case(H, W, m, phase, 300 + H, N)
    T_max = 2.0 * E0 / (H * W) ** 2 / 50
    c_max, s_max = max(1, N // 10), max(1, N // 40)
    w_img, w_counts, w_st, w_log, w_pairs = orc.anneal_generate(start, phase, m, target, policy, 777, log_u, T_max,
                                                               0.01 * T_max, c_max, s_max, use_local=True)
    d_img = dev(start)
    d_log = torch.zeros(N, dtype=torch.uint8, device="cuda")
    counts, st, pairs = lpf.lpf_anneal_generate(paths(m), d_img, phase, dev(target), policy, 777, dev(log_u), T_max,
                                                0.01 * T_max, c_max, s_max, accept_log=d_log)
    assert np.array_equal(pairs.cpu().numpy(), w_pairs)
    assert np.array_equal(d_log.cpu().numpy(), w_log)
    assert np.array_equal(d_img.cpu().numpy(), w_img)
    assert np.array_equal(counts.cpu().numpy(), w_counts)
    assert st == w_st and 0 < w_log.sum() < N


def test_anneal_limits_and_identity_moves():
    H, W, m, N = 16, 16, 7, 200
    start, target, pairs, log_u, _ = _anneal_case(H, W, m, 1, 77, N)
    pairs[5] = (3, 3, 3, 3)                                            # same pixel: identity move, accepted
    # huge temperature: every proposal accepted, final image = all swaps applied
    d_img = dev(start)
    counts, st = lpf.lpf_anneal(paths(m), d_img, 1, dev(target), dev(pairs), dev(log_u), 1e300, 1e300, 50, 7)
    want = start.copy()
    for xp, yp, xq, yq in pairs:
        want[yp, xp], want[yq, xq] = want[yq, xq], want[yp, xp]
    assert np.array_equal(d_img.cpu().numpy(), want)
    assert st["steps"] == N and st["accepted"] == N and st["levels"] == N // 7
    assert np.array_equal(counts.cpu().numpy()[0], orc.counts(want, 1, m))
    assert st["E"] == orc.half_sse(orc.counts(want, 1, m), target[0], m)
    # N = 0: nothing happens, the descriptor of the start image comes back
    d_img = dev(start)
    counts, st = lpf.lpf_anneal(paths(m), d_img, 1, dev(target), dev(pairs[:0]), dev(log_u[:0]), 1.0, 0.01, 5, 5)
    assert st["steps"] == 0 and np.array_equal(counts.cpu().numpy()[0], orc.counts(start, 1, m))


@pytest.mark.parametrize("H,W,m", [(64, 4640, 20), (4640, 40, 33), (1024, 1024, 40)])
def test_large_and_very_elongated_images(H, W, m):
    """More than 8 strips of 16 words per row (several strip bands per work item) in the direct and in the
    transposed views, and a megapixel image; sampled vectors, both phases, all flags."""
    rng = np.random.default_rng(H + W)
    img = (rng.random((H, W)) < 0.93).astype(np.uint8)
    vecs = rng.integers(-m, m + 1, size=(120, 2))
    vecs[:4] = [(0, 0), (m, m), (-m, m), (m, 0)]
    for flags in (0, lpf.LPF_PRUNE, lpf.LPF_NO_TRIE, lpf.LPF_S2):
        both = lpf.lpf_eval_both(paths(m), dev(img[None]), flags).cpu().numpy()[0]
        for phase in (0, 1):
            if flags & lpf.LPF_S2:
                chi = img == phase
                want = np.array([int((chi & np.roll(chi, (-dy, -dx), axis=(0, 1))).sum()) for dx, dy in vecs])
            else:
                want, _ = orc.counts_list(img, phase, vecs)
            assert np.array_equal(both[phase][vecs[:, 1] + m, vecs[:, 0] + m], want), (flags, phase)
            assert np.array_equal(both[phase], both[phase][::-1, ::-1])


def test_maximum_template_m511():
    """The largest template the library takes (m = 511 = MAX_M, 1023 x 1023 vectors, 4e7 program entries) on a
    512 x 512 image: sampled vectors against the oracle, Eq. 10 and Eq. 12; m = 512 is refused."""
    m, H, W = 511, 512, 512
    img = inputs.gaussian_field(H, W, 12.0, 0.40, inputs.seed_for(3, 7))
    p = lpf.lpf_build_paths(m, 0)
    try:
        got = lpf.lpf_eval(p, dev(img[None]), 1).cpu().numpy()[0]
    finally:
        lpf.lpf_free_paths(p)
    rng = np.random.default_rng(511)
    vecs = rng.integers(-m, m + 1, size=(200, 2))
    vecs[:6] = [(0, 0), (m, m), (-m, m), (m, 0), (0, m), (-m, 1)]
    want, _ = orc.counts_list(img, 1, vecs)
    assert np.array_equal(got[vecs[:, 1] + m, vecs[:, 0] + m], want)
    assert got[m, m] == int(img.sum()) and np.array_equal(got, got[::-1, ::-1])
    with pytest.raises(lpf.LpfError) as ei:
        lpf.lpf_build_paths(512, 0)
    assert ei.value.code == lpf.LPF_E_UNSUPPORTED


def test_hypothesis_generated_small_cases():
    """Random small shapes, template sizes, fill fractions, batch sizes and flags (hypothesis, derandomised):
    full-template bit-exact parity of lpf_eval / lpf_eval_both with the oracle."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=250, deadline=None, derandomize=True)
    @given(st.integers(1, 48), st.integers(1, 70), st.floats(0.05, 0.98), st.integers(0, 2 ** 31 - 1),
           st.sampled_from([0, lpf.LPF_PRUNE, lpf.LPF_NO_TRIE, lpf.LPF_NO_E2, lpf.LPF_PRUNE | lpf.LPF_NO_E2]),
           st.integers(1, 3), st.data())
    def check(H, W, fill, seed, flags, B, data):
        m = data.draw(st.integers(0, min(H, W) - 1))
        rng = np.random.default_rng(seed)
        imgs = (rng.random((B, H, W)) < fill).astype(np.uint8)
        both = lpf.lpf_eval_both(paths(m), dev(imgs), flags).cpu().numpy()
        one = lpf.lpf_eval(paths(m), dev(imgs), 1, flags).cpu().numpy()
        for b in range(B):
            for phase in (0, 1):
                want = orc.counts(imgs[b], phase, m, full_template=(H * W <= 600))
                assert np.array_equal(both[b, phase], want), (H, W, m, flags, b, phase)
            assert np.array_equal(one[b], both[b, 1])

    check()


def test_hypothesis_generated_levels_teams_and_tiles():
    """Random shapes up to 96 x 160 with a capped erosion level (1..6: pattern classes, derived planes, the short-vector
    kernel), a fixed team count and thread tile (hypothesis, derandomised): full-template bit-exact parity."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=120, deadline=None, derandomize=True)
    @given(st.integers(2, 96), st.integers(2, 160), st.floats(0.2, 0.97), st.integers(0, 2 ** 31 - 1),
           st.integers(1, 6), st.integers(0, 3), st.sampled_from([(0, 0), (4, 2), (8, 1), (4, 4), (8, 2), (16, 1)]),
           st.integers(0, 8), st.integers(1, 2), st.data())
    def check(H, W, fill, seed, level, teams, tile, cta_warps, B, data):
        m = data.draw(st.integers(1, min(H, W) - 1))
        rng = np.random.default_rng(seed)
        imgs = (rng.random((B, H, W)) < fill).astype(np.uint8)
        p = paths(m)
        lpf.lpf_set_level(p, level)
        lpf.lpf_set_tile(p, tile[0], tile[1], cta_warps)
        try:
            try:
                lpf.lpf_set_teams(p, teams)
                both = lpf.lpf_eval_both(p, dev(imgs)).cpu().numpy()
            except lpf.LpfError as e:                # a fixed team count that the shape cannot take is refused
                assert e.code == lpf.LPF_E_UNSUPPORTED and teams > 0
                lpf.lpf_set_teams(p, 0)
                both = lpf.lpf_eval_both(p, dev(imgs)).cpu().numpy()
            assert lpf.lpf_last_launch_info(p)["level"] <= level
        finally:
            lpf.lpf_set_level(p, -1)
            lpf.lpf_set_teams(p, 0)
            lpf.lpf_set_tile(p, 0, 0, 0)
        for b in range(B):
            for phase in (0, 1):
                want = orc.counts(imgs[b], phase, m, full_template=(H * W <= 600))
                assert np.array_equal(both[b, phase], want), (H, W, m, level, teams, tile, cta_warps, b, phase)

    check()


def test_hypothesis_generated_mixed_class_levels_with_little_shared_memory():
    """Random shapes up to 96 x 160 with 16 .. 40 KiB of shared memory for a CTA (lpf_set_shared_memory): fewer planes
    fit beside a band than one path has patterns at the program's level, so the pattern classes of steep slopes run at
    lower levels than those of shallow slopes (what happens to templates that are large against the image at the full
    227 KiB).  Hypothesis, derandomised: full-template bit-exact parity, both phases."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=60, deadline=None, derandomize=True)
    @given(st.integers(24, 96), st.integers(24, 160), st.floats(0.3, 0.97), st.integers(0, 2 ** 31 - 1),
           st.integers(16, 40), st.integers(0, 3), st.sampled_from([(0, 0), (4, 2), (8, 1), (4, 4)]), st.data())
    def check(H, W, fill, seed, kib, teams, tile, data):
        m = data.draw(st.integers(min(H, W) // 2, min(H, W) - 1))
        rng = np.random.default_rng(seed)
        img = (rng.random((1, H, W)) < fill).astype(np.uint8)
        p = paths(m)
        lpf.lpf_set_shared_memory(p, kib * 1024)
        lpf.lpf_set_tile(p, tile[0], tile[1], 0)
        try:
            try:
                lpf.lpf_set_teams(p, teams)
                both = lpf.lpf_eval_both(p, dev(img)).cpu().numpy()
            except lpf.LpfError as e:
                assert e.code == lpf.LPF_E_UNSUPPORTED and teams > 0
                lpf.lpf_set_teams(p, 0)
                both = lpf.lpf_eval_both(p, dev(img)).cpu().numpy()
            assert lpf.lpf_last_launch_info(p)["smem_bytes"] <= kib * 1024
        finally:
            lpf.lpf_set_shared_memory(p, 0)
            lpf.lpf_set_teams(p, 0)
            lpf.lpf_set_tile(p, 0, 0, 0)
        for phase in (0, 1):
            want = orc.counts(img[0], phase, m, full_template=(H * W <= 600))
            assert np.array_equal(both[0, phase], want), (H, W, m, kib, teams, tile, phase)

    check()


def test_random_mid_size_shapes_flags_teams_and_shared_memory_limits():
    """36 seeded random cases between the hypothesis shapes and the configs: 40..640 pixels a side, templates up to the
    whole domain (m = min(H, W) - 1, at most 511), disks / Bernoulli / Gaussian-field images, every flag, fixed team
    counts and shared-memory limits (so: every level, mixed class levels, the plain fall-back).  Sampled vectors (the
    template's corners, 40 random ones, 20 short ones) against the oracle, both phases, plus point symmetry."""
    rng = np.random.default_rng(20260601)
    for case in range(36):
        H, W = int(rng.integers(40, 640)), int(rng.integers(40, 640))
        mode = int(rng.integers(0, 4))
        m = min(H, W) - 1 if mode == 0 else int(rng.integers(1, min(H, W) if mode == 1 else min(H, W, 200)))
        m = min(m, 511)
        flags = int(rng.choice([0, 0, 0, lpf.LPF_PRUNE, lpf.LPF_NO_E2, lpf.LPF_S2, lpf.LPF_NO_TRIE if m <= 64 else 0]))
        if flags & lpf.LPF_S2:                       # the oracle's S2 is the O(WH S^2) definition: a smaller case
            H, W = min(H, 200), min(W, 200)
            m = min(m, 40, H - 1, W - 1)
        kind = int(rng.integers(0, 3))
        seed = int(rng.integers(1 << 30))
        if kind == 0:
            img = inputs.disks(H, W, float(rng.uniform(2, 12)), float(rng.uniform(0.1, 0.8)), seed)
        elif kind == 1:
            img = inputs.bernoulli(H, W, float(rng.uniform(0.5, 0.99)), seed)
        else:
            img = inputs.gaussian_field(H, W, float(rng.uniform(3, 20)), float(rng.uniform(0.2, 0.8)), seed)
        smem = int(rng.choice([0, 0, 0, 64, 100, 160])) * 1024
        teams = int(rng.choice([0, 0, 0, 1, 2, 5]))
        p = lpf.lpf_build_paths(m, 0)
        try:
            lpf.lpf_set_shared_memory(p, smem)
            try:
                lpf.lpf_set_teams(p, teams)
                got = lpf.lpf_eval_both(p, dev(img[None]), flags).cpu().numpy()[0]
            except lpf.LpfError as e:
                assert e.code == lpf.LPF_E_UNSUPPORTED and teams > 0
                lpf.lpf_set_teams(p, 0)
                got = lpf.lpf_eval_both(p, dev(img[None]), flags).cpu().numpy()[0]
        finally:
            lpf.lpf_free_paths(p)
        vecs = rng.integers(-m, m + 1, size=(40, 2))
        vecs[:4] = [(0, 0), (m, m), (-m, m), (m, 0)]
        k = min(m, 7)
        vecs = np.concatenate([vecs, rng.integers(-k, k + 1, size=(20, 2))])
        for phase in (0, 1):
            if flags & lpf.LPF_S2:
                want = orc.s2_counts(img, phase, m)[vecs[:, 1] + m, vecs[:, 0] + m]
            else:
                want, _ = orc.counts_list(img, phase, vecs)
            assert np.array_equal(got[phase][vecs[:, 1] + m, vecs[:, 0] + m], want), (case, H, W, m, flags, smem, teams)
            assert np.array_equal(got[phase], got[phase][::-1, ::-1]), (case, H, W, m, flags)


def test_mask_stack_in_tensor_memory_equals_the_one_in_local_memory():
    """The walker saves its mask at the branching nodes of the trie: in tensor memory (tcgen05.st / tcgen05.ld) when the
    launch runs one CTA per SM, in local memory otherwise or after lpf_set_tmem_stack(p, 0).  Whole results must be
    identical on shapes that take the tensor-memory path (which one ran is read from lpf_last_launch_info): thread tiles
    of 16 and of 8 words, with and without pruning, a batch, the masked evaluation; sampled vectors against the oracle."""
    cases = [(384, 512, 150, 0, (0, 0), 1), (200, 260, 120, lpf.LPF_PRUNE, (0, 0), 1), (256, 256, 100, 0, (8, 1), 1),
             (160, 192, 90, 0, (4, 2), 2), (300, 300, 149, lpf.LPF_NO_E2, (0, 0), 1)]
    took = 0
    for H, W, m, flags, tile, B in cases:
        imgs = np.stack([inputs.disks(H, W, 6.0, 0.4, inputs.seed_for(9, H + b)) for b in range(B)])
        p = lpf.lpf_build_paths(m, 0)
        try:
            lpf.lpf_set_tile(p, tile[0], tile[1], 0)
            res = {}
            for on in (True, False):
                lpf.lpf_set_tmem_stack(p, on)
                res[on] = lpf.lpf_eval_both(p, dev(imgs), flags).cpu().numpy()
                info = lpf.lpf_last_launch_info(p)
                assert info["tmem_stack"] in ((0, 1) if on else (0,)), info
                took += info["tmem_stack"]
                if on and info["ctas_per_sm"] == 1 and info["tile"] % 10 > 0:
                    assert info["tmem_stack"] == 1, info
            assert np.array_equal(res[True], res[False]), (H, W, m, flags, tile)
            if flags == 0 and B == 1:
                mask = (np.random.default_rng(m).random((H, W)) < 0.3).astype(np.uint8)
                lpf.lpf_set_tmem_stack(p, True)
                a = lpf.lpf_eval_masked(p, dev(imgs), 1, dev(mask)).cpu().numpy()
                lpf.lpf_set_tmem_stack(p, False)
                assert np.array_equal(a, lpf.lpf_eval_masked(p, dev(imgs), 1, dev(mask)).cpu().numpy())
        finally:
            lpf.lpf_free_paths(p)
        rng = np.random.default_rng(H)
        vecs = rng.integers(-m, m + 1, size=(60, 2))
        for phase in (0, 1):
            if flags & lpf.LPF_S2:
                continue
            want, _ = orc.counts_list(imgs[0], phase, vecs)
            assert np.array_equal(res[True][0, phase][vecs[:, 1] + m, vecs[:, 0] + m], want), (H, W, m, flags, phase)
    assert took >= 4                                     # the tensor-memory path did run


# ---- the plain-plane program at full size, the automatic fall-back, the boundary contract --------------------

def test_every_erosion_level_and_team_count_at_full_size():
    """The plain program (LPF_NO_E2 and level 0) and the eroded programs of level 1, 2, 3 on a 256 x 384 image, a shape
    where only the lower levels fit in shared memory (300 x 300, m = 299), and fixed team counts; which program ran
    is read from lpf_last_launch_info.  Sampled vectors (all the short ones among them: at level K the vectors shorter
    than K are counted by their own kernel) against the oracle, both phases, plus Eq. 10 / Eq. 12."""
    cases = [(256, 384, 120, lpf.LPF_NO_E2, -1, 0, 0), (256, 384, 120, 0, 0, 0, 0), (256, 384, 120, 0, 1, 0, 1),
             (256, 384, 120, 0, 2, 0, 2), (256, 384, 120, 0, 3, 0, 3), (256, 384, 120, 0, -1, 1, None),
             (256, 384, 120, 0, 4, 0, 4), (256, 384, 120, 0, 5, 0, 5), (256, 384, 120, 0, 6, 0, 6),
             (256, 384, 120, 0, 2, 3, 2), (300, 300, 299, 0, -1, 0, None), (300, 300, 299, 0, 0, 0, 0)]
    for H, W, m, flags, level, teams, want_level in cases:
        img = inputs.disks(H, W, 7.0, 0.45, inputs.seed_for(8, H + m))
        rng = np.random.default_rng(m)
        vecs = rng.integers(-m, m + 1, size=(300, 2))
        vecs[:6] = [(0, 0), (m, m), (-m, m), (m, 0), (0, m), (-m, 1)]
        short = np.array([(dx, dy) for dy in range(-6, 7) for dx in range(-6, 7)])
        vecs = np.concatenate([vecs, short])
        p = lpf.lpf_build_paths(m, 0)
        try:
            lpf.lpf_set_level(p, level)
            lpf.lpf_set_teams(p, teams)
            got = lpf.lpf_eval_both(p, dev(img[None]), flags).cpu().numpy()[0]
            info = lpf.lpf_last_launch_info(p)
        finally:
            lpf.lpf_free_paths(p)
        if want_level is not None:
            assert info["level"] == want_level, (H, W, m, flags, level, info)
        else:
            assert 1 <= info["level"] <= 6, info
        if teams:
            assert info["teams"] == teams
        assert info["shallow_vectors"] == [0, 1, 5, 13, 25, 41, 61][info["level"]]
        for phase in (0, 1):
            want, _ = orc.counts_list(img, phase, vecs)
            assert np.array_equal(got[phase][vecs[:, 1] + m, vecs[:, 0] + m], want), (H, W, m, flags, level, phase)
            _properties(got[phase], img, phase, m)


def test_reserved_calls_only_enqueue_cuda_graph_capture():
    """After lpf_reserve the hot calls neither allocate, copy synchronously nor synchronise: they can
    be captured into a CUDA graph (a cudaMalloc / cudaMemcpy / stream sync inside would abort the capture), and the
    replayed graph gives the oracle's counts for NEW image contents."""
    H, W, m, B = 96, 128, 40, 6
    p = lpf.lpf_build_paths(m, 0)
    try:
        lpf.lpf_reserve(p, B, H, W, 0, lpf.LPF_FOR_EVAL | lpf.LPF_FOR_EVAL_BOTH | lpf.LPF_FOR_SWAP_DELTA)
        lpf.lpf_reserve(p, B, H, W, 0, lpf.LPF_FOR_EVAL | lpf.LPF_FOR_MASKED)
        rng = np.random.default_rng(17)
        imgs = (rng.random((B, H, W)) < 0.75).astype(np.uint8)
        d_imgs = dev(np.zeros_like(imgs))
        d_mask = dev((rng.random((H, W)) < 0.5).astype(np.uint8))
        S = 2 * m + 1
        out1 = torch.zeros((B, S, S), dtype=torch.int64, device="cuda")
        out2 = torch.zeros((B, 2, S, S), dtype=torch.int64, device="cuda")
        outm = torch.zeros((B, S, S), dtype=torch.int64, device="cuda")
        outs = torch.zeros((S, S), dtype=torch.int64, device="cuda")
        sse = torch.zeros((B,), dtype=torch.int64, device="cuda")
        pairs = inputs.swap_pairs(imgs[0], 16, 3)
        d_pairs = dev(pairs)
        delta = torch.zeros((16, S, S), dtype=torch.int32, device="cuda")
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.graph(graph, stream=side):
            st = torch.cuda.current_stream()
            lpf.lpf_eval(p, d_imgs, 1, out=out1, stream=st)
            lpf.lpf_eval_both(p, d_imgs, out=out2, stream=st)
            lpf.lpf_eval_masked(p, d_imgs, 1, d_mask, out=outm, stream=st)
            lpf.lpf_eval_sum(p, d_imgs, 1, out=outs, stream=st)
            lpf.lpf_objective(out1, out1[0], out=sse, stream=st)
            lpf.lpf_swap_delta(p, d_imgs[:1], 1, d_pairs, out=delta, stream=st)
        d_imgs.copy_(dev(imgs))                                   # new contents: the graph must recompute
        graph.replay()
        torch.cuda.synchronize()
        c1, c2 = out1.cpu().numpy(), out2.cpu().numpy()
        for b in range(B):
            want1 = orc.counts(imgs[b], 1, m)
            assert np.array_equal(c1[b], want1) and np.array_equal(c2[b, 1], want1)
            assert np.array_equal(c2[b, 0], orc.counts(imgs[b], 0, m))
            assert int(sse[b]) == orc.sse(want1, c1[0])
        assert np.array_equal(outs.cpu().numpy(), orc.counts_sum(imgs, 1, m))
        mv = np.array([(0, 0), (1, 0), (-3, 2), (m, m), (-m, 1), (7, 40)])
        assert np.array_equal(outm.cpu().numpy()[2][mv[:, 1] + m, mv[:, 0] + m],
                              orc.counts_masked(imgs[2], d_mask.cpu().numpy(), 1, mv))
        dn = delta.cpu().numpy()
        for i in range(4):
            assert np.array_equal(dn[i], orc.swap_delta_local(imgs[0], 1, m, pairs[i]))
    finally:
        lpf.lpf_free_paths(p)


def test_calls_return_before_the_device_has_finished():
    """Asynchrony seen from the host: right after lpf_eval_both of config 3 returns, an event recorded behind it is
    not yet complete (the evaluation takes milliseconds; the call only enqueued it)."""
    img = inputs.config_image(3)
    p = paths(256)
    d_img = dev(img[None])
    out = lpf.lpf_eval_both(p, d_img)                             # plans and workspace exist from here on
    torch.cuda.synchronize()
    ev = torch.cuda.Event()
    not_ready = 0
    for _ in range(5):
        lpf.lpf_eval_both(p, d_img, out=out)
        ev.record()
        not_ready += not ev.query()
        torch.cuda.synchronize()
    assert not_ready >= 4


def test_two_streams_share_one_table_safely():
    """Consecutive calls on DIFFERENT streams share the packed-image workspace: the library orders them on the device
    (event wait, no host sync), so both results are right."""
    rng = np.random.default_rng(23)
    H, W, m = 128, 160, 50
    a = (rng.random((3, H, W)) < 0.7).astype(np.uint8)
    b = (rng.random((3, H, W)) < 0.4).astype(np.uint8)
    p = paths(m)
    d_a, d_b = dev(a), dev(b)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    outs = []
    for rep in range(6):
        st, src = (s1, d_a) if rep % 2 == 0 else (s2, d_b)
        with torch.cuda.stream(st):
            outs.append(lpf.lpf_eval(p, src, 1, stream=st))
    torch.cuda.synchronize()
    want_a = np.stack([orc.counts(a[i], 1, m) for i in range(3)])
    want_b = np.stack([orc.counts(b[i], 1, m) for i in range(3)])
    for rep, o in enumerate(outs):
        assert np.array_equal(o.cpu().numpy(), want_a if rep % 2 == 0 else want_b), rep
    # the host-buffer entry runs on a private stream and is ordered behind work in flight on the table too
    lpf.lpf_eval(p, d_a, 1, stream=s1)
    got = lpf.lpf_eval_host(p, b, 1)
    assert np.array_equal(got, want_b)


# ---- ensemble sum over an image stack (lpf_eval_sum) ----------------------------------------------

def test_eval_sum_hundred_slices():
    """100 slices of 100 x 100 (the paper's bone specimen is 100^3 voxels, its descriptor the average over 100 slices,
    PAPER.md:493-495): the device-side ensemble sum against the oracle's, one phase, both phases, pruned, and S2."""
    B, H, W, m = 100, 100, 100, 49
    stack = np.stack([inputs.disks(H, W, 5.0, 0.3, inputs.seed_for(9, i)) for i in range(B)])
    p = paths(m)
    d = dev(stack)
    want = [orc.counts_sum(stack, ph, m) for ph in (0, 1)]
    for flags in (0, lpf.LPF_PRUNE):
        assert np.array_equal(lpf.lpf_eval_sum(p, d, 1, flags).cpu().numpy(), want[1])
        both = lpf.lpf_eval_sum(p, d, -1, flags).cpu().numpy()
        assert np.array_equal(both[0], want[0]) and np.array_equal(both[1], want[1])
    # against the per-image call summed on the device
    per = lpf.lpf_eval(p, d, 1).sum(dim=0).cpu().numpy()
    assert np.array_equal(per, want[1])
    s2 = lpf.lpf_eval_sum(p, d[:7], 1, lpf.LPF_S2).cpu().numpy()
    assert np.array_equal(s2, sum(orc.s2_counts(stack[i], 1, m) for i in range(7)))
    # a ragged stack: B not a multiple of the images per CTA
    r = lpf.lpf_eval_sum(p, d[:13], 0).cpu().numpy()
    assert np.array_equal(r, orc.counts_sum(stack[:13], 0, m))
