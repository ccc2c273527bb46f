"""Pins T1-T3: the oracle against closed forms (BASELINE.json north_star (a))."""
import math
import os

import numpy as np

from oracle import oracle
from paper_2606_16566_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_t1():
    params = derived = None
    pixels = []
    for line in open(os.path.join(GOLD, "t1_closed_form.txt")):
        tok = line.split()
        if not tok or tok[0].startswith("#"):
            continue
        if tok[0] == "params":
            params = [float(t) for t in tok[1:]]
        elif tok[0] == "derived":
            derived = [float(t) for t in tok[1:]]
        elif tok[0] == "pixel":
            pixels.append([float(t) for t in tok[1:]])
    return params, derived, pixels


def test_t1_golden_fixture():
    """One camera-facing isotropic Gaussian: bg*(1-a) + c*a with a = o*exp(-r^2/(2 sigma'^2)), within 1e-6."""
    p, d, pixels = _read_t1()
    W, H, f, z0, s, o = int(p[0]), int(p[1]), p[2], p[3], p[4], p[5]
    c, bg = p[6:9], p[9:12]
    # a non-trivial rotation must not matter for an isotropic Gaussian
    q = np.array([0.5, -0.5, 0.5, 0.5])
    sc = scenes.single_gaussian_scene([0.0, 0.0, z0], [s, s, s], q, o, c, bg, W, H, f, f)
    r = oracle.render(sc)
    assert r.radius[0] == int(d[1])
    assert abs(float(r.mu[0, 0]) - d[2]) < 1e-5 and abs(float(r.mu[0, 1]) - d[3]) < 1e-5
    assert list(r.rect[0]) == [0, 0, 2, 2] and r.tiles_touched[0] == 4 and r.n_dup == 4
    for x, y, a, cr, cg, cb, T in pixels:
        x, y = int(x), int(y)
        assert abs(r.image[0, y, x] - cr) < 1e-6 and abs(r.image[1, y, x] - cg) < 1e-6 and abs(r.image[2, y, x] - cb) < 1e-6
        assert abs(r.final_T[y, x] - T) < 1e-6
        assert r.n_contrib[y, x] == (1 if a > 0 else 0)


def test_t1_closed_form_all_pixels_random_cases():
    """Same closed form, every pixel inside the rect, several (s, z0, o, f); outside the rect the image is bg."""
    rng = np.random.default_rng(7)
    for _ in range(6):
        W, H = 49, 35
        f = float(rng.uniform(30, 90)); z0 = float(rng.uniform(1.5, 6)); s = float(rng.uniform(0.05, 0.4))
        o = float(rng.uniform(0.05, 0.999)); c = rng.uniform(0, 1, 3); bg = rng.uniform(0, 1, 3)
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        sc = scenes.single_gaussian_scene([0.0, 0.0, z0], [s, s, s], q, o, c, bg, W, H, f, f)
        r = oracle.render(sc)
        sig2 = (f * s / z0) ** 2 + 0.3
        mux, muy = (W - 1) / 2.0, (H - 1) / 2.0
        yy, xx = np.mgrid[0:H, 0:W]
        r2 = (xx - mux) ** 2 + (yy - muy) ** 2
        a = np.minimum(0.99, np.float32(o).astype(np.float64) * np.exp(-r2 / (2 * sig2)))
        a[a < 1 / 255.0] = 0.0
        x0, y0, x1, y1 = r.rect[0]
        inrect = (xx // 16 >= x0) & (xx // 16 < x1) & (yy // 16 >= y0) & (yy // 16 < y1)
        a[~inrect] = 0.0
        c32 = np.maximum(0.0, 0.5 + ((c - 0.5) * scenes.SH_C0_INV).astype(np.float32).astype(np.float64) / scenes.SH_C0_INV)
        for ch in range(3):
            want = np.float32(bg[ch]).astype(np.float64) * (1 - a) + c32[ch] * a
            assert np.abs(r.image[ch] - want).max() < 2e-6
        assert np.abs(r.final_T - (1 - a)).max() < 1e-6
        # the rect is the 3-sigma square of the larger eigenvalue (isotropic: sigma'^2 + sqrt(0.1))
        assert r.radius[0] == math.ceil(3 * math.sqrt(sig2 + math.sqrt(max(0.1, 0.0))))


def _two(z1, z2, o1, o2, order):
    W = H = 33
    c1, c2, bg = np.array([0.9, 0.2, 0.1]), np.array([0.1, 0.3, 0.8]), np.array([0.25, 0.5, 0.75])
    means = np.array([[0, 0, z1], [0, 0, z2]], dtype=np.float32)[order]
    sc = scenes.single_gaussian_scene(means, [0.2, 0.2, 0.2], [1, 0, 0, 0], np.array([o1, o2], np.float32)[order],
                                      np.stack([c1, c2])[order], bg, W, H, 40.0, 40.0)
    return sc, oracle.render(sc), (c1, c2, bg)


def test_t2_two_coaxial_gaussians_order_and_tie_break():
    """C = c1 a1 + c2 a2 (1-a1) + bg (1-a1)(1-a2); input order irrelevant unless depths are EQUAL (lower index in front)."""
    o1, o2 = 0.6, 0.8
    for order in ([0, 1], [1, 0]):
        sc, r, (c1, c2, bg) = _two(3.0, 5.0, o1, o2, order)
        a1 = np.float32(o1).astype(np.float64); a2 = np.float32(o2).astype(np.float64)  # centre pixel: exp(0) = 1
        want = c1 * a1 + c2 * a2 * (1 - a1) + bg * (1 - a1) * (1 - a2)
        assert np.abs(r.image[:, 16, 16] - want).max() < 1e-6
        assert r.n_contrib[16, 16] == 2
    # equal depth: index 0 is in front
    for order in ([0, 1], [1, 0]):
        sc, r, (c1, c2, bg) = _two(4.0, 4.0, o1, o2, order)
        cols = np.stack([c1, c2])[order]; ops = np.array([o1, o2], np.float32).astype(np.float64)[order]
        want = cols[0] * ops[0] + cols[1] * ops[1] * (1 - ops[0]) + bg * (1 - ops[0]) * (1 - ops[1])
        assert np.abs(r.image[:, 16, 16] - want).max() < 1e-6
        tile = (16 // 16) * r.grid_x + 16 // 16
        lo, hi = int(r.list_offsets[tile]), int(r.list_offsets[tile + 1])
        assert list(r.sorted_ids[lo:hi]) == [0, 1]


def test_t3_termination_rule_r1():
    """Stack of identical centred Gaussians, o = 0.8: T = .2,.04,.008,.0016,3.2e-4, then T' = 6.4e-5 < 1e-4 => stop.
    n_contrib = 5, final_T = 3.2e-4, C = c (1 - 3.2e-4): the Gaussian that would cross the threshold is NOT blended."""
    n = 9
    c = np.array([0.7, 0.4, 0.2]); bg = np.zeros(3)
    sc = scenes.single_gaussian_scene(np.tile([[0, 0, 4.0]], (n, 1)), [0.3, 0.3, 0.3], [1, 0, 0, 0], 0.8, np.tile(c, (n, 1)), bg,
                                      33, 33, 40.0, 40.0)
    r = oracle.render(sc)
    o = np.float32(0.8).astype(np.float64)
    T5 = (1 - o) ** 5
    assert r.n_contrib[16, 16] == 5 and r.last_k[16, 16] == 5
    assert abs(r.final_T[16, 16] - T5) < 1e-9 and abs(T5 - 3.2e-4) < 1e-9
    c32 = 0.5 + ((c - 0.5) * scenes.SH_C0_INV).astype(np.float32).astype(np.float64) / scenes.SH_C0_INV
    assert np.abs(r.image[:, 16, 16] - c32 * (1 - T5)).max() < 1e-6
    assert not (r.fragile[16, 16] & 2)   # 36 % away from the threshold
    assert r.final_T.min() >= 1e-4 * (1 - 1e-6)   # I4: under R1 final_T never drops below 1e-4


def test_alpha_clamp_099():
    """alpha is clamped to [0, 0.99]: an o = 0.999 splat leaves T = 0.01 at its centre."""
    sc = scenes.single_gaussian_scene([0, 0, 4.0], [0.3, 0.3, 0.3], [1, 0, 0, 0], 0.999, [1.0, 1.0, 1.0], [0, 0, 0], 33, 33, 40.0, 40.0)
    r = oracle.render(sc)
    assert abs(r.final_T[16, 16] - (1 - np.float32(0.99).astype(np.float64))) < 1e-7
    assert abs(r.image[0, 16, 16] - np.float32(0.99).astype(np.float64)) < 1e-6
