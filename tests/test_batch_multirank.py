"""Frame-sharded mapping batch (paper_2607_04127_b200/batch.py) on CPU: two gloo ranks, the per-frame gradients
come from the oracle (the GPU path cannot run here), the all-reduced sum must equal the serial sum over all frames."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_frames_of_rank_partitions_the_batch():
    from paper_2607_04127_b200 import frames_of_rank
    for n in (0, 1, 7, 8, 9):
        for world in (1, 2, 3, 8):
            parts = [list(frames_of_rank(n, r, world)) for r in range(world)]
            assert sum(parts, []) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        frames_of_rank(4, 2, 2)


def _frame_grads(w, f):
    import oracle
    from workloads import simulate_scan
    S = w.sensors[f]
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed + f)
    lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, w.keep_masks[f], **w.lambdas)
    return oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, lr.gD, None, lr.gN)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2607_04127_b200 import batch_gradients
    from workloads import make_mapping_batch
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_mapping_batch(n_surfels=400, H=8, W=64, n_frames=3)
    grads = [torch.full((w.N, k), float("nan"), dtype=torch.float64) for k in (3, 4, 2, 1)]   # garbage: must be overwritten

    def run_frame(f, accumulate):
        g = _frame_grads(w, f)
        for dst, src in zip(grads, (g[0], g[1], g[2], g[3][:, None])):
            t = torch.from_numpy(np.ascontiguousarray(src))
            if accumulate:
                dst += t
            else:
                dst.copy_(t)

    batch_gradients(run_frame, len(w.sensors), grads, rank, world)
    # the one-launch form (what bench.py --config batch --gpus N runs): the rank's share summed locally as ONE batched
    # call would leave it, then the exchange step alone
    from paper_2607_04127_b200 import all_reduce_gradients, frames_of_rank
    g2 = [torch.zeros((w.N, k), dtype=torch.float64) for k in (3, 4, 2, 1)]
    for f in frames_of_rank(len(w.sensors), rank, world):
        g = _frame_grads(w, f)
        for dst, src in zip(g2, (g[0], g[1], g[2], g[3][:, None])):
            dst += torch.from_numpy(np.ascontiguousarray(src))
    all_reduce_gradients(g2, world)
    for a, b in zip(g2, grads):
        assert torch.allclose(a, b, rtol=1e-12, atol=1e-15)
    dist.barrier()
    dist.destroy_process_group()
    out[rank] = [g.numpy().copy() for g in grads]


def test_two_ranks_allreduce_equals_serial_sum():
    world = 2
    port = 29700 + os.getpid() % 200
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    sys.path.insert(0, ROOT)
    from workloads import make_mapping_batch
    w = make_mapping_batch(n_surfels=400, H=8, W=64, n_frames=3)
    ref = [np.zeros((w.N, k)) for k in (3, 4, 2, 1)]
    for f in range(3):                                            # rank 0 takes frames 0-1, rank 1 frame 2
        g = _frame_grads(w, f)
        for a, b in zip(ref, (g[0], g[1], g[2], g[3][:, None])):
            a += b
    assert any(np.abs(a).max() > 0 for a in ref)
    for r in range(world):
        for a, b in zip(res[r], ref):
            assert np.allclose(a, b, rtol=1e-12, atol=1e-15)
