"""Pins of oracle/map_prune.py (opacity prune + compaction).  All CPU."""
import numpy as np

from oracle import map_prune as mp


def test_closed_cases():
    op = np.array([0.5, 0.01, 0.3, np.nan, 0.05, 0.049999], dtype=np.float32)
    rows = np.arange(12, dtype=np.float32).reshape(6, 2)
    kept, (o, r) = mp.prune_compact(0.05, op, rows)
    assert kept.tolist() == [0, 2, 4]                       # 0.05 itself is kept (>=), NaN and 0.049999 are dropped
    assert o.tolist() == [0.5, np.float32(0.3), np.float32(0.05)]
    assert r.tolist() == [[0, 1], [4, 5], [8, 9]]
    kept, (o,) = mp.prune_compact(0.0, op)
    assert kept.tolist() == [0, 1, 2, 4, 5]                 # everything but the NaN
    kept, (o,) = mp.prune_compact(2.0, op)
    assert len(kept) == 0 and o.shape == (0,)
    kept, (o,) = mp.prune_compact(0.5, np.zeros(0, dtype=np.float32))
    assert len(kept) == 0


def test_is_numpys_boolean_indexing_order_preserving_and_idempotent():
    rng = np.random.default_rng(0)
    N = 5000
    op = rng.uniform(0, 1, N).astype(np.float32)
    a, b = rng.normal(size=(N, 3)).astype(np.float32), rng.normal(size=(N, 10)).astype(np.float32)
    kept, (o, a2, b2) = mp.prune_compact(0.3, op, a, b)
    mask = op >= np.float32(0.3)
    assert np.array_equal(kept, np.nonzero(mask)[0]) and (np.diff(kept) > 0).all()
    assert np.array_equal(o, op[mask]) and np.array_equal(a2, a[mask]) and np.array_equal(b2, b[mask])
    kept2, (o2, a3, b3) = mp.prune_compact(0.3, o, a2, b2)          # nothing left to prune
    assert len(kept2) == len(kept) and np.array_equal(a3, a2) and np.array_equal(b3, b2)
