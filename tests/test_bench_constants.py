"""bench.py's step roofline is built from oracle-side work counts stored as constants per workload (SURVEY.md 8(d):
"all counts from the oracle-side definitions, never from the implementation"): k16 = (surfel, 16x16 tile) pairs of the
list reference, nfp = (frame, surfel) pairs with a non-empty footprint.  A change to a workload generator or to the
list rule would silently skew every roofline fraction: recount them here with the oracle (all five configs at full
size, about a minute and a half on the CPU)."""
import pytest

import bench
import oracle
import workloads


@pytest.mark.parametrize("cfg", sorted(bench.CONFIGS))
def test_stored_work_counts_match_the_oracle(cfg):
    c = bench.CONFIGS[cfg]
    w = getattr(workloads, c["maker"])()
    k16 = nfp = nrect = 0
    for S in w.sensors:
        tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, tile=16)
        fp = oracle.footprint_surfels(w.mean, w.quat, w.scale, w.opacity, S)
        rect = tl.rects[:, 1] > 0
        assert not (fp & ~rect).any()                # a footprint implies a non-empty rect (the rect rule is conservative)
        k16 += len(tl.keys); nfp += int(fp.sum()); nrect += int(rect.sum())
    assert k16 == c["k16"] and nfp == c["nfp"]
    assert nfp <= nrect


def test_both_arms_print_the_same_config_object():
    """The driver compares the `config` objects of the two arms: they come from one function and hold nothing that only
    one arm knows (those facts are under `run`)."""
    w = workloads.make_tiny()
    a = bench.config_dict("tiny", w)
    assert set(a) == {"workload", "frames_per_step", "l2"} and a == bench.config_dict("tiny", w)
    src = open(bench.__file__).read()
    assert src.count('"config": config_dict(cfg, w)') == 2
