"""ORACLE -- test infrastructure only (see oracle/__init__.py).

Opacity pruning with compaction, the part of the paper's map management that is fully specified (SURVEY.md 8(f)
NEXT-3, first item): "Beyond opacity-based pruning/densification ..."; candidates elsewhere must
satisfy "sufficient opacity alpha_min <= alpha_i".  A surfel is KEPT iff alpha_i >= alpha_min
(fp32 comparison, the parameters are fp32); the survivors keep their relative order; every per-surfel row (mu, q, s~,
alpha, s and the optimiser moments m, v) moves with its surfel.  Reading R28: alpha_min is a caller input
(the paper prints no value); NaN opacities are dropped.

Pinned by tests/test_oracle_map_prune.py (closed cases, order preservation, idempotence, numpy's own boolean
indexing).  Nothing here is imported by the CUDA path.
"""
from __future__ import annotations

import numpy as np


def prune_compact(alpha_min, opacity, *rows):
    """Returns (kept indices, [opacity and every array of `rows` restricted to the kept surfels, order preserved])."""
    op = np.asarray(opacity, dtype=np.float32)
    thr = np.float32(alpha_min)
    kept = []
    for i in range(op.shape[0]):                 # plain loop: the definition
        if op[i] >= thr:                         # (False for NaN)
            kept.append(i)
    kept = np.asarray(kept, dtype=np.int64)
    out = [np.asarray(a)[kept] for a in (op,) + rows]
    return kept, out
