"""Pins of the oracle's optional tile-cull mode C-P8' (oracle flag TILE_CULL, off by default): the tile
rect of a Gaussian is the 3-sigma square INTERSECTED with the axis-aligned bounding box of its alpha >= 1/255 ellipse.

What must hold, and is checked by brute force here:
  * soundness: no pixel whose alpha reaches 1/255 (evaluated directly in float64 from the oracle's own
    per-Gaussian outputs) and that the standard rect contains lies in a tile the tighter rect drops -- hence
  * the image, final T and the contributor counts are IDENTICAL to the standard definition's, bit for bit;
  * the rect only ever shrinks, and on the paper-shaped scenes it removes a third to a half of the list entries.
"""
import numpy as np

from oracle import oracle
from paper_2606_16566_b200 import scenes


def _needle_scene(seed, P=400, W=160, H=112, f=120.0):
    """Anisotropic, often needle-like splats at every orientation, opacities from below 1/255 to 0.999."""
    rng = np.random.default_rng(seed)
    z = rng.uniform(1.5, 5.0, P)
    means = np.stack([rng.uniform(-0.9, 0.9, P) * z * (0.5 * W / f), rng.uniform(-0.9, 0.9, P) * z * (0.5 * H / f), z], 1)
    s = np.exp(rng.normal(-2.5, 1.0, (P, 3)))
    s[:, 0] *= np.exp(rng.uniform(0.0, 3.0, P))                  # one long axis: aspect ratios up to ~20 and more
    q = rng.standard_normal((P, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    o = 1.0 / (1.0 + np.exp(-rng.normal(-1.0, 3.0, P)))
    o[: P // 10] = rng.uniform(0.001, 0.01, P // 10)             # around and below 1/255 = 0.0039
    o[P // 10: P // 5] = rng.uniform(0.97, 0.9999, P // 5 - P // 10)
    return scenes.single_gaussian_scene(means, s, q, o, rng.uniform(0, 1, (P, 3)), [0.1, 0.2, 0.3], W, H, f, f)


def test_no_contributing_pixel_is_ever_in_a_dropped_tile():
    n_pairs = 0
    for seed in range(12):
        sc = _needle_scene(seed)
        std = oracle.render(sc, flags=oracle.NO_LISTS)
        cul = oracle.render(sc, flags=oracle.NO_LISTS | oracle.TILE_CULL)
        W, H = std.W, std.H
        yy, xx = np.mgrid[0:H, 0:W].astype(np.float64)
        ln_amin = np.log(np.float64(np.float32(1.0) / np.float32(255.0)))
        for g in np.flatnonzero(std.tiles_touched > 0):
            a, b, c = std.conic[g].astype(np.float64)
            dx, dy = xx - float(std.mu[g, 0]), yy - float(std.mu[g, 1])
            power = -0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy
            contributes = (power <= 0) & (np.log(np.float64(sc.opacities[g])) + power >= ln_amin)
            x0, y0, x1, y1 = std.rect[g]
            tx, ty = (xx // 16).astype(int), (yy // 16).astype(int)
            contributes &= (tx >= x0) & (tx < x1) & (ty >= y0) & (ty < y1)      # the standard definition truncates at its rect
            if not contributes.any():
                continue
            X0, Y0, X1, Y1 = cul.rect[g]
            inside = (tx >= X0) & (tx < X1) & (ty >= Y0) & (ty < Y1)
            assert cul.tiles_touched[g] > 0 and not (contributes & ~inside).any(), (seed, g)
            n_pairs += int(contributes.sum())
    assert n_pairs >= 100_000, n_pairs


def test_rect_only_shrinks_and_image_is_bit_identical():
    ratios = []
    for cfg, kw in ((2, dict(P=6000, W=256, H=192, f=300.0)), (3, dict(P=8000, W=320, H=208, f=250.0)),
                    (5, dict(P=20000, W=480, H=272, f=375.0)), (4, dict(P=3000, W=240, H=135, f=190.0))):
        sc = scenes.make_scene(cfg, poses=2, **kw)
        for pose in (0, 1):
            std = oracle.render(sc, pose, n_threads=4)
            cul = oracle.render(sc, pose, n_threads=4, flags=oracle.TILE_CULL)
            assert (cul.rect[:, 0] >= std.rect[:, 0])[cul.tiles_touched > 0].all() and (cul.rect[:, 2] <= std.rect[:, 2]).all()
            assert (cul.rect[:, 1] >= std.rect[:, 1])[cul.tiles_touched > 0].all() and (cul.rect[:, 3] <= std.rect[:, 3]).all()
            assert (cul.tiles_touched <= std.tiles_touched).all()
            assert np.array_equal(cul.image, std.image) and np.array_equal(cul.final_T, std.final_T)
            assert np.array_equal(cul.n_contrib, std.n_contrib)
            assert np.array_equal(cul.depth_bits[cul.tiles_touched > 0], std.depth_bits[cul.tiles_touched > 0])
            assert cul.n_dup < std.n_dup, (cfg, pose, cul.n_dup, std.n_dup)
            ratios.append((cfg, cul.n_dup / std.n_dup))
    print(ratios)   # at these reduced image sizes most splats cover one or two tiles; full size: 0.70 / 0.50 / 0.46 / 0.57 (configs 2-5)
    assert min(r for _, r in ratios) < 0.8
    sc = _needle_scene(99)
    std, cul = oracle.render(sc), oracle.render(sc, flags=oracle.TILE_CULL)
    assert np.array_equal(cul.image, std.image) and np.array_equal(cul.n_contrib, std.n_contrib)


def test_gaussians_that_can_never_blend_are_dropped_and_opaque_ones_keep_the_standard_rect():
    # o <= 1/255: tau <= 0, never blended (reading S20 keeps it in the standard lists; the cull mode drops it)
    sc = scenes.single_gaussian_scene([0, 0, 4.0], [0.3] * 3, [1, 0, 0, 0], 0.0039, [1, 1, 1], [0, 0, 0], 65, 65, 60.0, 60.0)
    assert oracle.render(sc).tiles_touched[0] > 0 and oracle.render(sc, flags=oracle.TILE_CULL).tiles_touched[0] == 0
    # an opaque isotropic splat reaches alpha >= 1/255 beyond 3 sigma (tau = 2 ln(255 * 0.9) = 10.9 > 9): the rect stays the 3-sigma one
    sc = scenes.single_gaussian_scene([0, 0, 4.0], [0.3] * 3, [1, 0, 0, 0], 0.9, [1, 1, 1], [0, 0, 0], 65, 65, 60.0, 60.0)
    a, b = oracle.render(sc), oracle.render(sc, flags=oracle.TILE_CULL)
    assert np.array_equal(a.rect, b.rect) and np.array_equal(a.image, b.image)
    # a faint one shrinks: o = 0.02 -> tau = 3.26, half-extent sqrt(3.26) sigma = 1.8 sigma
    sc = scenes.single_gaussian_scene([0, 0, 4.0], [0.8] * 3, [1, 0, 0, 0], 0.02, [1, 1, 1], [0, 0, 0], 129, 129, 60.0, 60.0)
    a, b = oracle.render(sc), oracle.render(sc, flags=oracle.TILE_CULL)
    sig = np.sqrt((60.0 * 0.8 / 4.0) ** 2 + 0.3)
    want_r = int(np.ceil(np.sqrt(2 * np.log(255 * 0.02)) * sig)) + 1
    lo, hi = int(np.floor((64 - want_r) / 16)), int(np.floor((64 + want_r + 15) / 16))
    assert b.tiles_touched[0] < a.tiles_touched[0]
    assert list(b.rect[0]) in ([lo, lo, hi, hi], [lo, lo, hi + 1, hi + 1], [lo - 1, lo - 1, hi, hi], [lo - 1, lo - 1, hi + 1, hi + 1])
    assert np.array_equal(a.image, b.image)
