"""N > 1 path on CPU: two gloo ranks shard the walkers the way bench.py --gpus 2 does
(paper_1802_06922_b200/sharding.py).  Walkers are independent Markov chains
(PAPER.md L181), so the ranks' results, concatenated, must equal the single-process result bit for
bit, with no data-path collective; the only communication is the max / sum of a few scalars."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1802_06922_b200 import inputs, sharding


def test_walker_range_partitions():
    for world in (1, 2, 3, 8):
        for nw in (0, 1, 5, 8, 512, 513):
            spans = [sharding.walker_range(r, world, nw) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == nw
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.walker_range(2, 2, 8)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out_dir):
    import oracle                                   # tests may use the oracle; the product path never does
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = inputs.custom_config("shard", (10, 12, 9), 24, (5.0, 6.0, 4.5), nw=7, nsweeps=2, sigma=0.2)
        x = inputs.make_inputs(cfg)                 # every rank draws all walkers, keeps its own
        pos, delta, unif = sharding.shard_inputs(x.pos, x.delta, x.unif, rank, world)
        lo, hi = sharding.walker_range(rank, world, cfg.nw)
        assert pos.shape[0] == hi - lo and delta.shape[2] == hi - lo and unif.shape[2] == hi - lo
        coefs = x.coefs_numpy()
        B, ld, sg = oracle.init_walkers(coefs, x.lattice, pos, nthreads=1)
        res = oracle.sweep(coefs, x.lattice, pos, B, ld, sg, delta, unif, nthreads=1)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), pos=res["pos"], B=res["B"], accept=res["accept"],
                 ratios=res["ratios"], lo=lo, hi=hi)
        # the only communication of the path: max of the per-rank times, sum of the counters
        t = sharding.max_over_ranks(10.0 + rank)
        moves, acc = sharding.sum_over_ranks([res["accept"].size, float(res["accept"].sum())])
        np.savez(os.path.join(out_dir, f"stats{rank}.npz"), t=t, moves=moves, acc=acc)
    finally:
        dist.destroy_process_group()


def test_two_ranks_equal_one_process(tmp_path):
    import oracle
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = inputs.custom_config("shard", (10, 12, 9), 24, (5.0, 6.0, 4.5), nw=7, nsweeps=2, sigma=0.2)
    x = inputs.make_inputs(cfg)
    coefs = x.coefs_numpy()
    B, ld, sg = oracle.init_walkers(coefs, x.lattice, x.pos, nthreads=1)
    ref = oracle.sweep(coefs, x.lattice, x.pos, B, ld, sg, x.delta, x.unif, nthreads=1)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert [int(p["lo"]) for p in parts] == [0, 4] and [int(p["hi"]) for p in parts] == [4, 7]
    assert np.array_equal(np.concatenate([p["pos"] for p in parts]), ref["pos"])
    assert np.array_equal(np.concatenate([p["B"] for p in parts]), ref["B"])
    assert np.array_equal(np.concatenate([p["accept"] for p in parts], axis=2), ref["accept"])
    assert np.array_equal(np.concatenate([p["ratios"] for p in parts], axis=2), ref["ratios"])
    for r in range(world):
        st = np.load(tmp_path / f"stats{r}.npz")
        assert float(st["t"]) == 11.0                               # max over ranks, on every rank
        assert float(st["moves"]) == ref["accept"].size and float(st["acc"]) == float(ref["accept"].sum())


def test_single_process_reductions_are_identity():
    assert sharding.max_over_ranks(3.5) == 3.5
    assert sharding.sum_over_ranks([1, 2.5]) == [1.0, 2.5]
