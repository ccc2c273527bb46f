"""Pins I1-I5: the paper's machinery proven on the CPU (BASELINE.json north_star (c))."""
import os

import numpy as np

from oracle import oracle
from paper_2606_16566_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _paper_constants():
    out = {}
    for line in open(os.path.join(GOLD, "paper_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def _random_conics(rng, n):
    """Positive-definite conics from random 2D covariances (sigma 0.6..60 px, any orientation)."""
    s1 = np.exp(rng.uniform(np.log(0.6), np.log(60), n)); s2 = np.exp(rng.uniform(np.log(0.6), np.log(60), n))
    th = rng.uniform(0, np.pi, n)
    c, s = np.cos(th), np.sin(th)
    cxx = c * c * s1 ** 2 + s * s * s2 ** 2; cyy = s * s * s1 ** 2 + c * c * s2 ** 2; cxy = c * s * (s1 ** 2 - s2 ** 2)
    det = cxx * cyy - cxy ** 2
    return cyy / det, -cxy / det, cxx / det


def test_i1_hoisted_form_equals_direct_conic_form():
    """Eq. 7-10: ln(alpha) = V . B_local must equal ln(o) - 0.5 x~^T Sigma^-1 x~ (Eq. 4-6).
    Pins the reconstruction of the garbled Eq. 8 (reading G2): any wrong row fails."""
    rng = np.random.default_rng(11)
    a, b, c = _random_conics(rng, 2000)
    o = rng.uniform(0.01, 0.999, 2000)
    for i in range(2000):
        Tx, Ty = 16 * rng.integers(0, 240), 16 * rng.integers(0, 135)
        mux, muy = Tx + rng.uniform(-300, 316), Ty + rng.uniform(-300, 316)
        V = oracle.hoist(a[i], b[i], c[i], o[i], mux - Tx, muy - Ty)          # Eq. 2: Delta = mu - T
        xs, ys = rng.integers(0, 16, 4), rng.integers(0, 16, 4)                # Eq. 1: x' = x - T
        for xp, yp in zip(xs, ys):
            B = np.array([xp * xp, xp * yp, yp * yp, xp, yp, 1.0])             # Eq. 9
            xt, yt = xp - (mux - Tx), yp - (muy - Ty)                          # Eq. 3
            direct = np.log(o[i]) - 0.5 * (a[i] * xt * xt + 2 * b[i] * xt * yt + c[i] * yt * yt)
            assert abs(V @ B - direct) <= 1e-9 * (1 + abs(V[5]))


def test_i2_warp_mask_is_conservative_and_tight():
    """Eq. 13-21: every pixel with alpha >= 1/255 lies in a 16x2 strip whose mask bit is set."""
    rng = np.random.default_rng(5)
    n = 6000
    a, b, c = _random_conics(rng, n)
    o = np.concatenate([rng.uniform(0.001, 0.999, n - 200), rng.uniform(0.0005, 1 / 255, 200)])
    yy, xx = np.mgrid[0:16, 0:16].astype(np.float64)
    set_bits = ideal_bits = 0
    for i in range(n):
        Tx, Ty = 16.0 * rng.integers(0, 50), 16.0 * rng.integers(0, 50)
        mux, muy = Tx + rng.uniform(-80, 96), Ty + rng.uniform(-80, 96)
        m, span = oracle.warp_mask(a[i], b[i], c[i], o[i], mux, muy, Tx, Ty)
        dx, dy = Tx + xx - mux, Ty + yy - muy
        alpha = o[i] * np.exp(-0.5 * (a[i] * dx * dx + c[i] * dy * dy) - b[i] * dx * dy)
        hit_rows = (alpha >= 1 / 255.0).any(axis=1)
        need = 0
        for w in range(8):
            if hit_rows[2 * w] or hit_rows[2 * w + 1]:
                need |= 1 << w
        assert (need & ~m) == 0, (i, bin(need), bin(m))
        assert m < 256
        set_bits += bin(m).count("1"); ideal_bits += bin(need).count("1")
    assert ideal_bits > 3000                     # the test actually exercised visible cases
    assert set_bits <= 1.25 * ideal_bits + 50    # and the box is tight (paper: "Tight Box")


def test_i2_tau_threshold_algebra():
    """o*exp(-q/2) >= 1/255  <=>  q <= tau = 2 ln(255 o)."""
    rng = np.random.default_rng(2)
    o = rng.uniform(0.01, 1, 1000); q = rng.uniform(0, 12, 1000)
    assert np.array_equal(o * np.exp(-q / 2) >= 1 / 255, q <= 2 * np.log(255 * o))


def test_i3_partition_of_unity_and_i4_monotone_T():
    """sum_g alpha_g T_g + final_T = 1  => with every colour = 1 and bg = 1 the image is 1 (I3); T in [1e-4, 1] (I4)."""
    sc = scenes.make_scene(1, P=600, W=96, H=64, f=96.0)
    sh = np.zeros_like(sc.sh); sh[:, 0, :] = 0.5 * scenes.SH_C0_INV
    sc1 = scenes.Scene(sc.name, 1, sc.means3D, sc.scales, sc.rotations, sc.opacities, sh, 0, np.ones(3, np.float32), sc.cameras)
    r = oracle.render(sc1)
    assert np.abs(r.image - 1.0).max() < 1e-6
    assert r.final_T.max() <= 1.0 and r.final_T.min() >= 1e-4 * (1 - 1e-6)
    # more Gaussians in front can only lower T: rendering a prefix of the depth order gives T >= full T
    keep = r.depth_bits <= np.median(r.depth_bits[r.tiles_touched > 0])
    sc2 = scenes.Scene(sc.name, 1, sc.means3D[keep], sc.scales[keep], sc.rotations[keep], sc.opacities[keep], sh[keep], 0,
                       np.ones(3, np.float32), sc.cameras)
    r2 = oracle.render(sc2)
    assert (r2.final_T >= r.final_T - 1e-7).all()


def test_i5_eq11_eq12_constants():
    """Eq. 11-12: 4*4000^2*2^-24 = 3.81 and 4*32^2*2^-24 = 2.44e-4, and empirically the fp32 hoisted
    polynomial in GLOBAL coordinates errs at that scale while the tile-local one does not."""
    k = _paper_constants()
    eps = 2.0 ** -24
    assert abs(eps - k["eps_mach"]) / eps < 1e-2
    assert abs(4 * 4000 ** 2 * eps - k["E_global"]) < 0.01
    assert abs(4 * 32 ** 2 * eps - k["E_local"]) / k["E_local"] < 0.01
    rng = np.random.default_rng(0)
    worst_g = worst_l = 0.0
    for _ in range(4000):
        sig = rng.uniform(0.6, 3.0)
        a = c = 1 / sig ** 2; b = 0.0; o = 0.9
        Tx, Ty = 3824.0, 2144.0                       # last tile of a 4K frame
        mux, muy = Tx + rng.uniform(0, 15), Ty + rng.uniform(0, 15)
        xp, yp = float(rng.integers(0, 16)), float(rng.integers(0, 16))
        exact = np.log(o) - 0.5 * (a * (Tx + xp - mux) ** 2 + c * (Ty + yp - muy) ** 2)
        def poly32(dx, dy, x, y):
            V = oracle.hoist(a, b, c, o, dx, dy).astype(np.float32)
            B = np.array([x * x, x * y, y * y, x, y, 1.0], dtype=np.float32)
            acc = np.float32(0)
            for v, bb in zip(V, B):
                acc = np.float32(acc + np.float32(v * bb))
            return float(acc)
        worst_l = max(worst_l, abs(poly32(mux - Tx, muy - Ty, xp, yp) - exact))
        worst_g = max(worst_g, abs(poly32(mux, muy, Tx + xp, Ty + yp) - exact))   # origin at (0,0): global coordinates
    assert worst_l < k["E_local"] * 3.0          # bound scaled by the conic (a <= 2.8)
    assert worst_g > 100 * worst_l               # four orders of magnitude in the bound, >= two observed
    assert worst_g < k["E_global"] * 3.0
