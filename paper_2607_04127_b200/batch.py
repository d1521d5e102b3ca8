"""Mapping batches over several GPUs (host logic only).

The keyframes of a mapping batch (BASELINE.json configs[4]) are independent given a replicated map: every rank
renders its own keyframes with `accumulate = 1` into its own map-sized gradient buffers, then ONE all-reduce(sum)
of the [N,3] / [N,4] / [N,2] / [N] buffers gives every rank the gradient of the whole batch (R18: the sum of the
per-frame losses) -- the only exchange step of the path; NCCL over NVLink on the GPUs.  Nothing here computes:
the frames run through the C-ABI calls of `binding.Rasterizer`, the reduction is torch.distributed's.
"""
from __future__ import annotations

from typing import Callable, Sequence


def frames_of_rank(n_frames: int, rank: int, world: int) -> range:
    """Contiguous, balanced share of the keyframes: the first n_frames % world ranks take one frame more."""
    if world < 1 or not (0 <= rank < world) or n_frames < 0:
        raise ValueError("bad (n_frames, rank, world) = (%d, %d, %d)" % (n_frames, rank, world))
    base, extra = divmod(n_frames, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def batch_gradients(run_frame: Callable[[int, bool], None], n_frames: int, grads: Sequence, rank: int = 0, world: int = 1,
                    group=None) -> None:
    """Gradient of a mapping batch in `grads` (tensors, summed over all keyframes, identical on every rank).

    run_frame(f, accumulate) must add (accumulate = True) or write (False) the gradient of keyframe f into `grads`
    -- on the GPU: set_pose / forward / loss stage / backward(accumulate=...) of a `Rasterizer` whose g_* buffers
    are `grads`.  A rank without frames contributes zeros."""
    mine = frames_of_rank(n_frames, rank, world)
    if len(mine) == 0:
        for g in grads:
            g.zero_()
    for j, f in enumerate(mine):
        run_frame(f, j > 0)
    if world > 1:
        import torch.distributed as dist
        for g in grads:
            dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)


def all_reduce_gradients(grads: Sequence, world: int = 1, group=None) -> None:
    """The exchange step alone: sum the gradient buffers over the ranks (after each rank rendered its share of the
    keyframes in ONE batched call, `binding.BatchRasterizer` over `frames_of_rank(...)`)."""
    if world > 1:
        import torch.distributed as dist
        for g in grads:
            dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)
