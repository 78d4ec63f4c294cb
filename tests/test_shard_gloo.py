"""The N > 1 path on CPU: world_size-2 (and 3) `gloo` runs of the sharding logic.

The per-rank fitter is injected (the fp64 oracle) because the product's fitter is the CUDA library and this suite
runs without a GPU; what is tested is the host logic: block ranges, the block_index that keeps the Philox streams
of the full track, the padded all-gather, and that the gathered parameters give the same Doppler products as
the unsharded track.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1906_10598_b200 import shard, workloads as W


def test_block_range_partitions_every_block_once():
    for B in (0, 1, 2, 7, 60, 3600, 36001):
        for world in (1, 2, 3, 8):
            got = [b for r in range(world) for b in shard.block_range(B, r, world)]
            assert got == list(range(B))
            sizes = [len(shard.block_range(B, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.block_range(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _oracle_fitter(x, fs, lo, hi, cfg, block_index):
    r = oracle.fit_blocks(x.numpy(), fs, lo.numpy(), hi.numpy(), NP=cfg["NP"], generations=cfg["generations"], F=cfg["F"],
                          CR=cfg["CR"], seed=cfg["seed"], block_index=block_index.numpy().astype(np.uint32))
    return {"best": torch.from_numpy(r["best"]), "best_rss": torch.from_numpy(r["best_rss"].astype(np.float32)),
            "status": torch.from_numpy(r["status"].astype(np.int32))}


def _worker(rank, world, port, B, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.config1(blocks=range(B), NP=24, generations=6)
        mine = shard.block_range(B, rank, world)
        sl = slice(mine.start, mine.stop)
        cfg = dict(NP=24, generations=6, F=0.5, CR=0.9, seed=77)
        got = shard.fit_track_sharded(torch.from_numpy(wl.x[sl]), wl.fs, torch.from_numpy(wl.lo[sl]),
                                      torch.from_numpy(wl.hi[sl]), cfg, B, fit=_oracle_fitter)
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), **{k: v.numpy() for k, v in got.items()})
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,B", [(2, 7), (2, 4), (3, 2)])
def test_sharded_track_equals_the_unsharded_track(tmp_path, world, B):
    port = _free_port()
    mp.spawn(_worker, args=(world, port, B, str(tmp_path)), nprocs=world, join=True)
    wl = W.config1(blocks=range(B), NP=24, generations=6)
    ref = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=24, generations=6, F=0.5, CR=0.9, seed=77,
                            block_index=wl.block_index)
    pb_ref, tot_ref, iv_ref = oracle.doppler_products(ref["best"], wl.T, 0.0, [1, 2])
    for rank in range(world):
        got = np.load(os.path.join(str(tmp_path), "rank%d.npz" % rank))
        assert got["best"].shape == (B, 5) and got["best"].dtype == np.float64
        assert np.array_equal(got["best"], ref["best"])                    # same Philox streams, same fp64 arithmetic
        assert np.array_equal(got["best_rss"], ref["best_rss"].astype(np.float32))
        assert np.array_equal(got["status"], ref["status"].astype(np.int32))
        pb, tot, iv = oracle.doppler_products(got["best"], wl.T, 0.0, [1, 2])
        assert np.array_equal(tot, tot_ref) and np.array_equal(np.nan_to_num(pb), np.nan_to_num(pb_ref))
