"""World-size-2 gloo test of the only multi-rank exchange (sharding.combine_spectra) and of the shard bounds."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1312_4698_b200.sharding import combine_shards, combine_spectra, shard_bounds


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # per-trajectory "spectra" s_j[i]; every trajectory good except #3
    rng = np.random.default_rng(0)
    s = rng.uniform(0, 1, (11, 7))
    good = np.ones(11, bool)
    good[3] = False
    lo, hi = shard_bounds(11, rank, world)
    ng = int(good[lo:hi].sum())
    I_local = torch.from_numpy(s[lo:hi][good[lo:hi]].sum(0) / max(ng, 1))
    I, n_good = combine_spectra(I_local, ng)
    expect = s[good].sum(0) / good.sum()
    ret[rank] = (float(np.max(np.abs(I.numpy() - expect))), n_good)
    dist.destroy_process_group()


def test_combine_spectra_world2_gloo():
    port = _free_port()
    with mp.Manager() as m:
        ret = m.dict()
        mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
        for r in range(2):
            err, ng = ret[r]
            assert err < 1e-15 and ng == 10


def test_shard_bounds_partition():
    for n in (1, 7, 131072, 131073):
        for world in (1, 2, 3, 8):
            b = [shard_bounds(n, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1


def test_combine_single_process_no_group():
    I, ng = combine_spectra(torch.tensor([1.0, 2.0], dtype=torch.float64), 5)
    assert ng == 5 and torch.equal(I, torch.tensor([1.0, 2.0], dtype=torch.float64))
    I, ng = combine_spectra(torch.tensor([1.0, 2.0], dtype=torch.float64), 0)
    assert ng == 0 and not I.any()


def test_combine_shards_equals_the_collective_arithmetic():
    rng = np.random.default_rng(1)
    parts = [torch.from_numpy(rng.uniform(0, 1, 5)) for _ in range(3)]
    ngs = [4, 0, 9]
    I, ng = combine_shards(parts, ngs)
    want = (parts[0] * 4 + parts[2] * 9) / 13
    assert ng == 13 and float((I - want).abs().max()) < 1e-15
    I0, ng0 = combine_shards(parts, [0, 0, 0])
    assert ng0 == 0 and float(I0.abs().max()) == 0.0
