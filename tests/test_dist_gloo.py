"""world_size-2 gloo test of the multi-rank plumbing bench.py uses (shards, max-over-ranks timing,
whole-job unit count).  CPU only; rendezvous on 127.0.0.1."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1601_04359_b200 import dist as lpf_dist
from paper_1601_04359_b200 import inputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_units, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b, e = lpf_dist.shard_range(n_units, rank, world)
        # every rank draws its own images (weak scaling) and its slice of one shared batch
        img = inputs.bernoulli(8, 8, 0.5, inputs.seed_for(1) + lpf_dist.rank_seed_offset(rank))
        times = lpf_dist.max_over_ranks([10.0 + rank, 5.0 - rank])
        total = lpf_dist.sum_over_ranks(e - b)
        dist.barrier()
        np.save(os.path.join(out_dir, "r%d.npy" % rank), np.array([b, e, total, times[0], times[1], int(img.sum())]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_units", [1024, 7])
def test_two_ranks_partition_units_and_reduce_times(tmp_path, n_units):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_units, str(tmp_path)), nprocs=world, join=True)
    r = [np.load(tmp_path / ("r%d.npy" % k)) for k in range(world)]
    assert r[0][0] == 0 and r[0][1] == r[1][0] and r[1][1] == n_units          # partition, in order
    assert abs((r[0][1] - r[0][0]) - (r[1][1] - r[1][0])) <= 1
    for k in range(world):
        assert r[k][2] == n_units                                                 # whole-job unit count
        assert r[k][3] == 11.0 and r[k][4] == 5.0                                 # max over ranks
    assert r[0][5] != r[1][5]                                                     # independent images per rank


def _split_worker(rank, world, port, n_img, out_dir):
    """Strong-scaling split of ONE batch (bench.py --scaling strong): every rank holds the batch,
    evaluates only its shard (here with the CPU oracle standing in for lpf_eval) and all-gathers the count slices."""
    from oracle import lpf_oracle as orc
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = 4
        batch = np.stack([inputs.bernoulli(9, 11, 0.6, inputs.seed_for(1, i)) for i in range(n_img)])
        b, e = lpf_dist.shard_range(n_img, rank, world)
        local = torch.from_numpy(np.stack([orc.counts(batch[i], 1, m, threads=1) for i in range(b, e)])
                                 if e > b else np.zeros((0, 2 * m + 1, 2 * m + 1), dtype=np.int64))
        buf = lpf_dist.gather_buffer(local, n_img, world)
        whole = lpf_dist.gather_shards(local, buf, n_img, rank, world)
        np.save(os.path.join(out_dir, "g%d.npy" % rank), whole.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_img", [8, 7])
def test_two_ranks_split_one_batch_and_gather_the_whole_result(tmp_path, n_img):
    from oracle import lpf_oracle as orc
    world = 2
    mp.spawn(_split_worker, args=(world, _free_port(), n_img, str(tmp_path)), nprocs=world, join=True)
    batch = np.stack([inputs.bernoulli(9, 11, 0.6, inputs.seed_for(1, i)) for i in range(n_img)])
    want = np.stack([orc.counts(batch[i], 1, 4) for i in range(n_img)])            # the unsplit, one-rank result
    for k in range(world):
        got = np.load(tmp_path / ("g%d.npy" % k))
        assert got.shape == want.shape and np.array_equal(got, want), k


def test_gather_without_process_group_is_identity():
    local = torch.arange(12).reshape(3, 4)
    buf = lpf_dist.gather_buffer(local, 3, 1)
    assert lpf_dist.gather_shards(local, buf, 3, 0, 1) is local


def test_shard_range_properties():
    for n in (0, 1, 5, 1024, 100000):
        for world in (1, 2, 3, 8):
            cuts = [lpf_dist.shard_range(n, k, world) for k in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[k][1] == cuts[k + 1][0] for k in range(world - 1))
            sizes = [e - b for b, e in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        lpf_dist.shard_range(4, 2, 2)
    assert lpf_dist.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]      # no process group: identity
