"""GPU parity of lgs_prune_compact (opacity prune + compaction) against oracle/map_prune.py:
a selection and a copy, so the bar is bit-exact (count, order, every row)."""
import numpy as np
import pytest

from oracle import map_prune as mp

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _lgs():
    import paper_2607_04127_b200 as lgs
    return lgs


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")


@pytest.mark.parametrize("N,alpha_min", [(0, 0.05), (1, 0.05), (255, 0.3), (256, 0.3), (257, 0.3), (300_001, 0.05),
                                         (300_001, 0.0), (300_001, 2.0), (2_000_003, 0.5)])
def test_prune_compact_parity(N, alpha_min):
    lgs = _lgs()
    rng = np.random.default_rng(N % 1000 + 1)
    f32 = np.float32
    arrs = [rng.normal(size=(N, 3)).astype(f32), rng.normal(size=(N, 4)).astype(f32), rng.normal(size=(N, 2)).astype(f32),
            rng.uniform(0, 1, N).astype(f32), rng.uniform(0.05, 2, (N, 2)).astype(f32),
            rng.normal(size=(N, 10)).astype(f32), rng.uniform(0, 1, (N, 10)).astype(f32)]
    if N > 10:
        arrs[3][3] = np.nan; arrs[3][5] = f32(alpha_min)            # NaN dropped, the threshold itself kept
    kept, ref = mp.prune_compact(alpha_min, arrs[3], arrs[0], arrs[1], arrs[2], arrs[4], arrs[5], arrs[6])
    n, outs = lgs.lgs_prune_compact(alpha_min, *[_dev(a) for a in arrs])
    assert n == len(kept)
    got = {k: o.cpu().numpy()[:n] for k, o in zip(("mean", "quat", "ls", "op", "scale", "m", "v"), outs)}
    for k, r in zip(("op", "mean", "quat", "ls", "scale", "m", "v"), ref):
        assert np.array_equal(got[k], r, equal_nan=True), k
    # optional arrays left out
    n2, outs2 = lgs.lgs_prune_compact(alpha_min, *[_dev(a) for a in arrs[:4]])
    assert n2 == n and len(outs2) == 4 and np.array_equal(outs2[0].cpu().numpy()[:n], ref[1])


def test_pruned_map_renders_like_the_masked_map():
    """Dropping surfels below alpha_min = 1/255 changes nothing: the renderer culls them anyway (R4)."""
    lgs = _lgs()
    from workloads import make_newer_college
    w = make_newer_college(n_surfels=20_000, H=32, W=256)
    S = w.sensors[0]
    op = w.opacity.copy()
    op[::3] = 0.001                                                  # a third of the map below the renderer's cut-off
    p = [_dev(w.mean), _dev(w.quat), _dev(np.log(w.scale)), _dev(op), _dev(w.scale)]
    n, (mean, quat, ls, opk, scale) = lgs.lgs_prune_compact(1.0 / 255.0, *p)
    assert n == int((op >= np.float32(1.0 / 255.0)).sum())
    R0 = lgs.Rasterizer(w.N, S, 400_000)
    R0.forward(p[0], p[1], p[4], p[3])
    R1 = lgs.Rasterizer(n, S, 400_000)
    R1.forward(mean[:n].contiguous(), quat[:n].contiguous(), scale[:n].contiguous(), opk[:n].contiguous())
    torch.cuda.synchronize()
    assert R0.query()[:3] == R1.query()[:3]                          # same visible surfels, keys and contributing pairs
    assert torch.equal(R0.range, R1.range) and torch.equal(R0.alpha, R1.alpha) and torch.equal(R0.normal, R1.normal)
