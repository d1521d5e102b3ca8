"""Pins for the tile-list reference: the rect is a superset of the exact
footprint (checked against the oracle's per-pixel definition), lists are the stable sort of
the emission, ranges partition the list."""
import numpy as np
import pytest

import oracle
from helpers import make_sensor, _rot_zyx
from workloads import make_newer_college, make_random_shell, make_tiny

TILE = (8, 4)        # the CUDA path's list tiles; square 16 x 16 tiles are checked too


def _check_structure(tl, H, W, N, tile=TILE):
    TW, TH = tile
    ntc, ntr = -(-W // TW), -(-H // TH)
    K = len(tl.keys)
    # independent re-derivation of the emission from (rects, rkeys) and a lexsort
    tiles, ids = [], []
    for i in np.nonzero(tl.rects[:, 1] > 0)[0]:
        c0, nc, r0, r1 = tl.rects[i]
        cols = (c0 + np.arange(nc)) % W
        tcs = np.unique(cols // TW)
        trs = np.arange(r0 // TH, r1 // TH + 1)
        for tr in trs:
            for tc in tcs:
                tiles.append(tr * ntc + tc)
                ids.append(i)
    tiles = np.array(tiles, dtype=np.uint64)
    ids = np.array(ids, dtype=np.uint32)
    assert len(tiles) == K
    kb = tl.rkeys.view(np.uint32)[ids].astype(np.uint64)
    keys = (tiles << np.uint64(32)) | kb
    order = np.lexsort((ids, keys))          # by key, ties by surfel index == stable sort of index-ordered emission
    assert np.array_equal(tl.keys, keys[order])
    assert np.array_equal(tl.vals, ids[order])
    # ranges partition [0, K) in tile order
    tr = tl.tile_ranges.astype(np.int64)
    assert tr.shape[0] == ntc * ntr
    assert (tr[:, 1] >= tr[:, 0]).all() and tr[:, 1].max() == K
    t_of_key = (tl.keys >> np.uint64(32)).astype(np.int64)
    for t in range(ntc * ntr):
        s, e = tr[t]
        assert (t_of_key[s:e] == t).all() and (e - s) == int((t_of_key == t).sum())
    # positive floats order like their bit patterns
    r = tl.rkeys[tl.rects[:, 1] > 0]
    assert (r > 0).all()
    o = np.argsort(r, kind="stable")
    assert np.array_equal(np.argsort(r.view(np.uint32), kind="stable"), o)


def test_lists_structure_on_tiny():
    w = make_tiny()
    S = w.sensors[0]
    tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, TILE)
    _check_structure(tl, S.H, S.W, w.N)
    tl16 = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, 16)
    _check_structure(tl16, S.H, S.W, w.N, (16, 16))
    assert np.array_equal(tl16.rects, tl.rects) and np.array_equal(tl16.rkeys, tl.rkeys)   # independent of the tiling
    # the key is the fp32 rounding of the fp64 centre range
    c = w.mean.astype(np.float64)
    assert np.array_equal(tl.rkeys, np.linalg.norm(c, axis=1).astype(np.float32)) or \
        np.abs(tl.rkeys.astype(np.float64) - np.linalg.norm(c, axis=1)).max() < 2e-6


@pytest.mark.parametrize("case", ["tiny", "big_scales_seam", "poles", "scene", "ragged"])
def test_rect_is_a_superset_of_the_exact_footprint(case):
    if case == "tiny":
        w = make_tiny(); S = w.sensors[0]
    elif case == "big_scales_seam":
        T = np.concatenate([_rot_zyx(3.0, 0.1, -0.2), [[0.5], [0.2], [-0.1]]], 1)
        w = make_random_shell(21, 1500, 32, 128, s_lo=0.3, s_hi=1.5, r_lo=5.0, pose=T); S = w.sensors[0]
    elif case == "poles":
        w = make_random_shell(22, 3000, 64, 128, fov_deg=(-85, 85), s_lo=0.1, s_hi=1.0, r_lo=3.5); S = w.sensors[0]
    elif case == "scene":
        w = make_newer_college(n_surfels=30_000, H=64, W=512); S = w.sensors[0]
    else:
        w = make_random_shell(23, 1200, 40, 200, fov_deg=(-30, 10), s_lo=0.05, s_hi=0.8); S = w.sensors[0]
    tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S, TILE)
    _check_structure(tl, S.H, S.W, w.N)
    out = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED, check_rects=tl.rects)
    assert out.stats["I_c"] > 1000
    assert out.stats["rect_violations"] == 0
    # and it is not absurdly loose: rect pixels within a small multiple of the in-3-sigma pairs
    rect_px = int((tl.rects[:, 1] * (tl.rects[:, 3] - tl.rects[:, 2] + 1))[tl.rects[:, 1] > 0].sum())
    if case in ("tiny", "scene", "ragged"):
        assert rect_px < 6 * max(out.stats["I_3sigma"], 1)


def test_wrapped_rect_touches_each_tile_column_once():
    # one huge surfel behind the sensor: its column interval wraps and covers most of the image
    S = make_sensor(32, 128)
    mean = np.array([[-4.0, 0.3, 0.0]])
    quat = np.array([[0.0, 0.0, 0.7071, 0.7071]])
    tl = oracle.tile_lists(mean, quat, np.array([[1.2, 1.2]]), np.array([0.9]), S, TILE)
    _check_structure(tl, S.H, S.W, 1)
    c0, nc, r0, r1 = tl.rects[0]
    assert nc > 16 and (c0 + nc > S.W or nc == S.W)   # wraps across the seam
    assert len(np.unique(tl.keys)) == len(tl.keys)    # no tile listed twice


def test_footprint_census_against_one_surfel_renders():
    """oracle.footprint_surfels (the N_fp of SURVEY.md 8(d)) pinned by the forward it does not use: a surfel has a
    non-empty footprint iff, rendered ALONE with opacity 1 (alpha G >= exp(-4.5) > 1/255 wherever rho2 <= 9, no other
    surfel to stop the beam), it puts opacity into at least one pixel.  Also: what stands in front of a surfel does not
    change its flag, culled surfels (alpha < 1/255) have none, and the footprint implies a non-empty rect."""
    w = make_random_shell(21, 60, 32, 128, s_lo=0.02, s_hi=0.3)
    S = w.sensors[0]
    ones = np.ones(1, dtype=np.float32)
    alone = np.array([oracle.render_forward(w.mean[i:i + 1], w.quat[i:i + 1], w.scale[i:i + 1], ones, S,
                                            oracle.BRUTE).alpha.max() > 0 for i in range(w.N)])
    fp = oracle.footprint_surfels(w.mean, w.quat, w.scale, w.opacity, S)
    assert fp.dtype == bool and fp.shape == (w.N,)
    assert np.array_equal(fp, alone)
    assert 0 < fp.sum() < w.N                                   # the case has both kinds (some surfels miss every beam)
    tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S)
    assert not (fp & ~(tl.rects[:, 1] > 0)).any()
    # an opaque shell of large surfels in front of everything: the flags of the original surfels do not move
    front = make_random_shell(22, 400, 32, 128, r_lo=0.8, r_hi=1.0, s_lo=0.3, s_hi=0.5, a_lo=0.99, a_hi=0.99)
    both = [np.concatenate([a, b]) for a, b in ((front.mean, w.mean), (front.quat, w.quat), (front.scale, w.scale),
                                                (front.opacity, w.opacity))]
    assert np.array_equal(oracle.footprint_surfels(*both, S)[front.N:], fp)
    # a transparent surfel is culled before it has a footprint
    op = w.opacity.copy(); k = int(np.nonzero(fp)[0][0]); op[k] = 0.5 / 255.0
    fp2 = oracle.footprint_surfels(w.mean, w.quat, w.scale, op, S)
    assert not fp2[k] and np.array_equal(np.delete(fp2, k), np.delete(fp, k))
