"""Pin T6: C-B against numpy's stable sort and a difference-array count."""
import numpy as np

from oracle import oracle
from paper_2606_16566_b200 import scenes


def _check_binning(sc, ci=0):
    r = oracle.render(sc, ci, flags=oracle.NO_RENDER)
    vis = np.nonzero(r.tiles_touched)[0]
    # duplication in index order
    tiles, ids = [], []
    for i in vis:
        x0, y0, x1, y1 = r.rect[i]
        ty, tx = np.mgrid[y0:y1, x0:x1]
        tiles.append((ty * r.grid_x + tx).ravel()); ids.append(np.full(tiles[-1].size, i))
    tiles = np.concatenate(tiles) if tiles else np.zeros(0, int); ids = np.concatenate(ids) if ids else np.zeros(0, int)
    assert tiles.size == r.n_dup == r.tiles_touched.sum()
    key = (tiles.astype(np.uint64) << np.uint64(32)) | r.depth_bits[ids].astype(np.uint64)   # PAPER.md:53 64-bit key
    order = np.argsort(key, kind="stable")
    assert np.array_equal(ids[order].astype(np.uint32), r.sorted_ids)
    counts = np.bincount(tiles, minlength=r.n_tiles)
    assert np.array_equal(counts, r.tile_counts)
    assert np.array_equal(np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64), r.list_offsets)
    # depth bits are order preserving for positive floats
    d = r.depth_bits[vis].view(np.float32)
    assert (d > 0.2).all() and np.array_equal(np.argsort(d, kind="stable"), np.argsort(r.depth_bits[vis], kind="stable"))
    return r


def test_t6_binning_config1():
    _check_binning(scenes.make_scene(1))


def test_t6_binning_config3_small_with_ties():
    sc = scenes.make_scene(3, P=3000, W=200, H=120, f=150.0, poses=2)
    # force exact depth ties: duplicate means (different scales/colours keep them distinguishable)
    sc.means3D[1500:] = sc.means3D[:1500]
    r = _check_binning(sc, 1)
    assert len(np.unique(r.depth_bits[r.tiles_touched > 0])) < (r.tiles_touched > 0).sum()


def test_subset_mode_matches_full():
    sc = scenes.make_scene(2, P=2000, W=160, H=128, f=200.0, poses=1)
    full = oracle.render(sc)
    sub = [3, 17, 42, 79]
    part = oracle.render(sc, tile_subset=sub)
    assert np.array_equal(full.tile_counts, part.tile_counts) and full.n_dup == part.n_dup
    for l, t in enumerate(sub):
        a = full.sorted_ids[int(full.list_offsets[t]):int(full.list_offsets[t + 1])]
        b = part.sorted_ids[int(part.list_offsets[l]):int(part.list_offsets[l + 1])]
        assert np.array_equal(a, b)
        ty, tx = divmod(t, full.grid_x)
        sl = (slice(None), slice(16 * ty, 16 * ty + 16), slice(16 * tx, 16 * tx + 16))
        assert np.array_equal(full.image[sl], part.image[sl])
        assert np.array_equal(full.n_contrib[sl[1:]], part.n_contrib[sl[1:]])
    assert part.rendered.sum() == len(sub)
    thr = oracle.render(sc, n_threads=4)
    assert np.array_equal(thr.image, full.image) and thr.pairs_traversed == full.pairs_traversed


def test_culling_rules():
    """Reading S2/S7: only depth <= 0.2, degenerate covariance and empty rects cull; off-screen centres still render."""
    W = H = 64
    means = np.array([[0, 0, 0.19], [0, 0, 0.21], [0, 0, -3.0], [50.0, 0, 4.0], [0.95, 0, 4.0]], np.float32)
    sc = scenes.single_gaussian_scene(means, [0.05, 0.05, 0.05], [1, 0, 0, 0], 0.9, [0.5, 0.5, 0.5], [0, 0, 0], W, H, 64.0, 64.0)
    sc.scales[4] = 0.5   # centre off-screen (mu_x = 64*0.95/4*... ) but large
    sc.means3D[4] = [3.0, 0, 4.0]
    r = oracle.render(sc)
    assert list(r.tiles_touched > 0) == [False, True, False, False, True]
    assert r.mu[4, 0] > W - 1   # centre is outside the image, the splat is kept because its rect overlaps


def test_threaded_oracle_equals_single_threaded():
    """n_threads > 1 spreads the per-list sorts and the tiles of the blend over threads; nothing may change."""
    sc = scenes.make_scene(3, P=3000, W=200, H=120, f=150.0, poses=2)
    a = oracle.render(sc, 1, n_threads=1)
    b = oracle.render(sc, 1, n_threads=5)
    assert np.array_equal(a.sorted_ids, b.sorted_ids) and np.array_equal(a.list_offsets, b.list_offsets)
    assert np.array_equal(a.image, b.image) and np.array_equal(a.n_contrib, b.n_contrib) and np.array_equal(a.fragile, b.fragile)
