"""Pins of the oracle's exact ellipse-tile mode C-P8'' (oracle flag TILE_CULL_EXACT, off by default): a
(tile, Gaussian) pair of the C-P8' rect is counted and listed only if the (slightly widened) ellipse alpha >= 1/255 meets the
tile's box of pixel centres.

  * exactness, against an INDEPENDENT formulation: the minimum of the quadratic form q over the box (a box-constrained
    convex QP solved in float64: the unconstrained minimum if it lies inside, else the best of the four edges) compared
    with tau_e -- no kept pair with q_min > tau_e (1 + 1e-3), no dropped pair with q_min < tau_e (1 - 1e-3).  The oracle
    instead takes the x-extent of the ellipse over the row band (the paper's tight box, Eq. 13-18, transposed);
  * soundness by brute force: no pixel whose alpha reaches 1/255 lies in a dropped tile -- hence
  * image, final T and contributor counts bit-identical to the standard definition's;
  * rect, tiles_touched and n_dup stay those of C-P8'; the lists only lose entries, and keep their order.
"""
import numpy as np

from oracle import oracle
from paper_2606_16566_b200 import scenes
from test_oracle_tile_cull import _needle_scene


def _pairs(res):
    """{(tile, gaussian)} of a full oracle result."""
    out = set()
    for l, t in enumerate(res.list_tile):
        for g in res.sorted_ids[int(res.list_offsets[l]):int(res.list_offsets[l + 1])]:
            out.add((int(t), int(g)))
    return out


def _qmin_over_box(a, b, c, x0, x1, y0, y1):
    """min of a x^2 + 2 b x y + c y^2 over [x0, x1] x [y0, y1] (float64; positive definite form, minimum at the origin)."""
    if x0 <= 0.0 <= x1 and y0 <= 0.0 <= y1:
        return 0.0
    best = np.inf
    for y in (y0, y1):                       # horizontal edges: minimise over x at fixed y
        x = min(max(-b * y / a, x0), x1)
        best = min(best, a * x * x + 2 * b * x * y + c * y * y)
    for x in (x0, x1):                       # vertical edges
        y = min(max(-b * x / c, y0), y1)
        best = min(best, a * x * x + 2 * b * x * y + c * y * y)
    return best


def test_kept_pairs_are_exactly_the_tiles_the_ellipse_meets():
    n_kept = n_dropped = 0
    for seed in range(6):
        sc = _needle_scene(seed, P=300)
        cul = oracle.render(sc, flags=oracle.NO_RENDER | oracle.TILE_CULL)
        ex = oracle.render(sc, flags=oracle.NO_RENDER | oracle.TILE_CULL_EXACT)
        assert np.array_equal(cul.rect, ex.rect) and np.array_equal(cul.tiles_touched, ex.tiles_touched)
        assert cul.n_dup == ex.n_dup
        kept = _pairs(ex)
        assert kept <= _pairs(cul)
        gx = ex.grid_x
        for g in np.flatnonzero(ex.tiles_touched > 0):
            a, b, c = (float(v) for v in ex.conic[g])
            mx, my = (float(v) for v in ex.mu[g])
            # tau as C-P8' defines it, re-derived with the library logarithm: the oracle's value is an upper bound within 0.03
            tau = 2.0 * np.log(255.0 * float(np.float32(sc.opacities[g])))
            x0, y0, x1, y1 = ex.rect[g]
            for ty in range(y0, y1):
                for tx in range(x0, x1):
                    q = _qmin_over_box(a, b, c, 16 * tx - mx, 16 * tx + 15 - mx, 16 * ty - my, 16 * ty + 15 - my)
                    k = (ty * gx + tx, int(g)) in kept
                    if k:
                        n_kept += 1
                        assert q <= (tau + 0.05 + 0.03) * (1 + 1e-3), (seed, g, tx, ty, q, tau)
                    else:
                        n_dropped += 1
                        assert q >= (tau + 0.05) * (1 - 1e-3), (seed, g, tx, ty, q, tau)
    assert n_kept > 3000 and n_dropped > 1000, (n_kept, n_dropped)


def test_no_contributing_pixel_is_dropped_and_image_is_bit_identical():
    for seed in (1, 4, 9):
        sc = _needle_scene(seed)
        std = oracle.render(sc)
        ex = oracle.render(sc, flags=oracle.TILE_CULL_EXACT)
        assert np.array_equal(ex.image, std.image) and np.array_equal(ex.final_T, std.final_T)
        assert np.array_equal(ex.n_contrib, std.n_contrib)
        kept = _pairs(ex)
        W, H, gx = std.W, std.H, std.grid_x
        yy, xx = np.mgrid[0:H, 0:W].astype(np.float64)
        tile_of = ((yy // 16) * gx + (xx // 16)).astype(int)
        ln_amin = np.log(np.float64(np.float32(1.0) / np.float32(255.0)))
        for g in np.flatnonzero(std.tiles_touched > 0):
            a, b, c = std.conic[g].astype(np.float64)
            dx, dy = xx - float(std.mu[g, 0]), yy - float(std.mu[g, 1])
            power = -0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy
            contributes = (power <= 0) & (np.log(np.float64(sc.opacities[g])) + power >= ln_amin)
            x0, y0, x1, y1 = std.rect[g]
            tx, ty = (xx // 16).astype(int), (yy // 16).astype(int)
            contributes &= (tx >= x0) & (tx < x1) & (ty >= y0) & (ty < y1)
            for t in np.unique(tile_of[contributes]):
                assert (int(t), int(g)) in kept, (seed, g, t)


def test_paper_shaped_scenes_lists_shrink_and_keep_their_order():
    ratios = []
    for cfg, kw in ((2, dict(P=6000, W=256, H=192, f=300.0)), (3, dict(P=8000, W=320, H=208, f=250.0)),
                    (5, dict(P=20000, W=480, H=272, f=375.0)), (4, dict(P=3000, W=240, H=135, f=190.0))):
        sc = scenes.make_scene(cfg, poses=2, **kw)
        std = oracle.render(sc, 1, n_threads=4)
        cul = oracle.render(sc, 1, n_threads=4, flags=oracle.TILE_CULL)
        ex = oracle.render(sc, 1, n_threads=4, flags=oracle.TILE_CULL_EXACT)
        assert np.array_equal(ex.image, std.image) and np.array_equal(ex.n_contrib, std.n_contrib)
        assert (ex.tile_counts <= cul.tile_counts).all() and ex.tile_counts.sum() < cul.tile_counts.sum()
        assert int(ex.tile_counts.sum()) == len(ex.sorted_ids)
        for l in range(0, len(ex.list_tile), 7):          # a kept list is a sub-sequence of the C-P8' list of its tile
            e = ex.sorted_ids[int(ex.list_offsets[l]):int(ex.list_offsets[l + 1])]
            c = cul.sorted_ids[int(cul.list_offsets[l]):int(cul.list_offsets[l + 1])]
            assert np.array_equal(c[np.isin(c, e)], e)
        ratios.append((cfg, float(ex.tile_counts.sum()) / float(std.tile_counts.sum())))
    print(ratios)
    assert max(r for _, r in ratios) < 0.9
