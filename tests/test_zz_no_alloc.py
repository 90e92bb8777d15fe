"""lpf_swap_delta_static: the swap-delta evaluation with its scratch in the library's static device array (include/lpf.h),
for callers that cannot allocate device memory.  Collected last on purpose (the suite runs with pytest -x).

The result must be bit for bit that of lpf_swap_delta (integer work: no tolerance) on two calls in a row -- the second on
another image, shape, template and phase, so that anything the array kept from the first call would show -- and PyTorch's
allocator must not have been asked for anything, and the device's free memory must not have changed, across the calls."""
import numpy as np
import pytest
import torch

from oracle import lpf_oracle as orc
from paper_1601_04359_b200 import inputs, lpf

pytestmark = pytest.mark.gpu


def _case(H, W, m, phase, n, seed):
    img = inputs.disks(H, W, 5.0, 0.35, inputs.seed_for(5, seed))
    pairs = inputs.swap_pairs(img, n, inputs.seed_for(5, seed + 1))
    return img, pairs, m, phase


def test_static_scratch_swap_delta_equals_the_allocating_path_on_two_calls_in_a_row():
    cases = [_case(96, 160, 40, 1, 300, 11), _case(70, 64, 21, 0, 200, 13)]
    tables = {}
    want = []
    for img, pairs, m, phase in cases:               # the existing path first: it also uploads the trie records
        p = tables.setdefault(m, lpf.lpf_build_paths(m, 0))
        H, W = img.shape
        lpf.lpf_reserve(p, 1, H, W, 0, lpf.LPF_FOR_SWAP_DELTA)
        d_img, d_pairs = torch.from_numpy(img[None]).cuda(), torch.from_numpy(pairs).cuda()
        want.append((d_img, d_pairs, lpf.lpf_swap_delta(p, d_img, phase, d_pairs)))
    outs = [torch.full_like(w[2], 7) for w in want]  # the caller's outputs, allocated before the calls; never zeroed
    try:
        # the first call on a device looks up the array's address (the runtime may load the device image then)
        lpf.lpf_swap_delta_static(tables[cases[1][2]], want[1][0], cases[1][3], want[1][1][:1], outs[1][:1])
        torch.cuda.synchronize()
        n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]
        free_before = torch.cuda.mem_get_info()[0]
        for (img, pairs, m, phase), (d_img, d_pairs, _), out in zip(cases, want, outs):
            lpf.lpf_swap_delta_static(tables[m], d_img, phase, d_pairs, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc      # nothing through PyTorch
        assert torch.cuda.mem_get_info()[0] >= free_before                             # and no cudaMalloc beside it
        for (img, pairs, m, phase), (_, _, ref), out in zip(cases, want, outs):
            assert torch.equal(out, ref), (img.shape, m, phase)
            got = out.cpu().numpy()
            for i in range(3):                       # and the oracle's definition-level delta on a few proposals
                assert np.array_equal(got[i], orc.swap_delta_local(img, phase, m, pairs[i])), i
        # the same call again, on the first case after the second: the array now holds the second case's bits
        again = torch.full_like(outs[0], -3)
        lpf.lpf_swap_delta_static(tables[cases[0][2]], want[0][0], cases[0][3], want[0][1], again)
        assert torch.equal(again, want[0][2])
    finally:
        for p in tables.values():
            lpf.lpf_free_paths(p)


def test_static_scratch_limits_and_errors():
    m = 8
    p = lpf.lpf_build_paths(m, 0)
    try:
        img = torch.zeros((1, 64, 64), dtype=torch.uint8, device="cuda")
        pairs = torch.zeros((1, 4), dtype=torch.int32, device="cuda")
        out = torch.zeros((1, 2 * m + 1, 2 * m + 1), dtype=torch.int32, device="cuda")
        with pytest.raises(lpf.LpfError) as ei:      # the trie records were never uploaded: nothing is allocated here
            lpf.lpf_swap_delta_static(p, img, 1, pairs, out)
        assert ei.value.code == lpf.LPF_E_INVAL
        lpf.lpf_reserve(p, 1, 64, 64, 0, lpf.LPF_FOR_SWAP_DELTA)
        lpf.lpf_swap_delta_static(p, img, 1, pairs, out)
        assert int(out.abs().sum()) == 0             # equal bytes: the identity move
        # 1024 x 1024 with m = 8 needs 4 * (2 * 1024 * 32 + 1040 * 33) + 256 = 399 KB: beyond the 256 KiB array
        big = torch.zeros((1, 1024, 1024), dtype=torch.uint8, device="cuda")
        assert 4 * (2 * 1024 * 32 + 1040 * 33) + 256 > lpf.LPF_STATIC_SCRATCH_BYTES
        with pytest.raises(lpf.LpfError) as ei:
            lpf.lpf_swap_delta_static(p, big, 1, pairs, out)
        assert ei.value.code == lpf.LPF_E_TOO_LARGE and "LPF_STATIC_SCRATCH_BYTES" in str(ei.value)
        lpf.lpf_swap_delta(p, big, 1, pairs, out)    # the allocating path takes that shape
        # 720 x 720 with m = 8 needs 4 * (2 * 720 * 23 + 736 * 23) + 256 = 200 KB: fits
        mid = torch.zeros((1, 720, 720), dtype=torch.uint8, device="cuda")
        mid[0, 100, 100] = 1
        pr = torch.tensor([[100, 100, 400, 300]], dtype=torch.int32, device="cuda")
        got = lpf.lpf_swap_delta_static(p, mid, 1, pr, out)
        assert torch.equal(got, lpf.lpf_swap_delta(p, mid, 1, pr))
        with pytest.raises(lpf.LpfError) as ei:
            lpf.lpf_swap_delta_static(p, img, 2, pairs, out)
        assert ei.value.code == lpf.LPF_E_INVAL
    finally:
        lpf.lpf_free_paths(p)
