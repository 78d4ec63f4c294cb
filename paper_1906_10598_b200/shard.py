"""One track over several GPUs: contiguous ranges of blocks per rank, one all-gather of the fitted parameters.

Blocks are independent (every block is fitted about its own centre), so the DE fit shards with no
data-path collective.  The only exchange step of the path is before the Doppler products, whose running
total-count phase (Eq. 16-17) needs every block's parameters: one all-gather of
``best[B_local][D]`` fp64 (1.7 MB for BASELINE config 3).  The Philox counter carries the block's index within
the full track (``block_index``), so a sharded track draws exactly the random numbers of the unsharded one.

Host logic only (torch.distributed: NCCL on the GPUs, gloo in the CPU tests).  ``fit`` defaults to the CUDA path
(``pt.pt_fit_blocks``); there is no CPU fallback -- the tests pass their own fitter to exercise the plumbing.
"""
from __future__ import annotations

from typing import Callable, Optional

import torch
import torch.distributed as dist


def block_range(B: int, rank: int, world: int) -> range:
    """Contiguous blocks of `rank`: sizes differ by at most one, earlier ranks take the larger shares."""
    if not (0 <= rank < world) or B < 0:
        raise ValueError("bad rank/world/B")
    q, r = divmod(B, world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


def all_gather_blocks(local: torch.Tensor, B: int, group=None) -> torch.Tensor:
    """[B_local][...] of every rank (block_range order) -> [B][...] on every rank.  Shares are padded to the
    largest one so that the collective is a plain all_gather on both NCCL and gloo."""
    world = dist.get_world_size(group)
    sizes = [len(block_range(B, r, world)) for r in range(world)]
    if local.shape[0] != sizes[dist.get_rank(group)]:
        raise ValueError("local has %d blocks, this rank owns %d" % (local.shape[0], sizes[dist.get_rank(group)]))
    pad = max(sizes)
    buf = local.new_zeros((pad,) + tuple(local.shape[1:]))
    buf[: local.shape[0]] = local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf, group=group)
    return torch.cat([o[:n] for o, n in zip(out, sizes)], dim=0)


def _cuda_fit(x, fs, lo, hi, cfg, block_index):
    from . import pt
    return pt.pt_fit_blocks(x, fs, lo, hi, cfg, block_index=block_index)


def fit_track_sharded(x_local: torch.Tensor, fs: float, lo_local: torch.Tensor, hi_local: torch.Tensor, cfg, B: int,
                      *, group=None, fit: Optional[Callable] = None) -> dict:
    """Fit this rank's blocks of a B-block track and gather the results of all ranks.

    x_local / lo_local / hi_local hold the blocks ``block_range(B, rank, world)``.  Returns, on every rank,
    ``best[B][D]`` fp64, ``best_rss[B]`` fp32, ``status[B]`` int32 -- the inputs of ``pt_doppler_products``.
    """
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    mine = block_range(B, rank, world)
    if x_local.shape[0] != len(mine):
        raise ValueError("x_local has %d blocks, this rank owns %d" % (x_local.shape[0], len(mine)))
    bidx = torch.arange(mine.start, mine.stop, dtype=torch.int32, device=x_local.device)
    if len(mine) == 0:     # more ranks than blocks: this rank only takes part in the exchange
        dev = x_local.device
        r = {"best": torch.empty((0, lo_local.shape[1]), dtype=torch.float64, device=dev),
             "best_rss": torch.empty(0, dtype=torch.float32, device=dev),
             "status": torch.empty(0, dtype=torch.int32, device=dev)}
    else:
        r = (fit or _cuda_fit)(x_local, fs, lo_local, hi_local, cfg, bidx)
    return {k: all_gather_blocks(r[k], B, group) for k in ("best", "best_rss", "status")}
