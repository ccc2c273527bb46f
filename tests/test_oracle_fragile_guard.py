"""Pins of the two parts of the oracle that had none:

  * the FRAGILE classifier of the parity protocol (m_alpha = min |ln o + power - ln(1/255)|,
    m_T = min |T'/1e-4 - 1|, fragile = (m_alpha < delta) | (m_T < delta) << 1).  It decides which mismatches the GPU
    parity test forgives, so it is checked against closed forms: one isotropic camera-facing Gaussian
    (ln alpha = ln o - r^2 / (2 sigma'^2), Eq. 4-5) with o chosen so that the margin at a known pixel is
    0.5e-3 / 2e-3 on either side of the threshold, and a stack of identical Gaussians (T' = (1 - o)^k) with o chosen
    so that T'/1e-4 - 1 = +-0.5e-3 / +-2e-3.
  * the guard-band clamp of C-P4 (reading S3: x/z, y/z clamped to +-1.3 (W/2)/fx before the Jacobian is formed), checked
    against a float64 numpy restatement with np.clip / np.linalg.inv / eigvalsh on a scene whose Gaussians sit at
    |x/z| in [1, 3] tan(fov/2), so that the clamp is active for a known subset.
"""
import math

import numpy as np
from scipy.spatial.transform import Rotation

from oracle import oracle
from paper_2606_16566_b200 import scenes

LN_AMIN = math.log(float(np.float32(1.0) / np.float32(255.0)))   # the fp32 constant 1.0f/255.0f, promoted
T_MIN = float(np.float32(0.0001))
DELTA = 1e-3


def _one(o, W=33, H=33, f=40.0, s=0.125, z=4.0):
    return scenes.single_gaussian_scene([0.0, 0.0, z], [s, s, s], [1.0, 0.0, 0.0, 0.0], o, [0.9, 0.5, 0.1], [0.2, 0.3, 0.4], W, H, f, f)


def _sigma2(f=40.0, s=0.125, z=4.0):
    # (f s / z)^2 is exact in binary32 for these values; the only rounding is the "+ 0.3f" of the dilation (reading S4)
    return float(np.float32((f * s / z) ** 2) + np.float32(0.3))


def test_m_alpha_is_the_closed_form_margin_on_every_pixel():
    o = 0.7
    r = oracle.render(_one(o), fragile_delta=DELTA)
    sig2 = _sigma2()
    yy, xx = np.mgrid[0:33, 0:33]
    r2 = (xx - 16.0) ** 2 + (yy - 16.0) ** 2
    want = np.abs(math.log(float(np.float32(o))) - r2 / (2 * sig2) - LN_AMIN)
    inrect = (xx < 32) & (yy < 32)                       # rect = tiles [0,2) x [0,2) (golden fixture T1)
    # m_alpha is returned as fp32: 2e-6 absolute near the threshold, 2 ulp of the value far from it
    assert (np.abs(r.m_alpha[inrect] - want[inrect]) < 2e-6 + 2.4e-7 * want[inrect]).all()
    assert np.isinf(r.m_alpha[~inrect]).all()            # no Gaussian reached: nothing can be fragile there
    assert np.isinf(r.m_T[r.n_contrib == 0]).all()       # m_T only counts Gaussians that passed the alpha test
    assert not r.fragile[~inrect].any()
    assert np.array_equal((r.fragile & 1) != 0, r.m_alpha < DELTA)


def test_fragile_alpha_bit_on_both_sides_of_the_threshold():
    """o chosen so that ln(alpha) - ln(1/255) = margin at the pixels with r^2 = 9 (e.g. (19,16), (16,13))."""
    sig2 = _sigma2()
    for margin, fragile in ((+0.5e-3, True), (-0.5e-3, True), (+2e-3, False), (-2e-3, False)):
        o = math.exp(LN_AMIN + 9.0 / (2 * sig2) + margin)
        assert 0.0 < o < 0.99
        r = oracle.render(_one(o), fragile_delta=DELTA)
        for (x, y) in ((19, 16), (13, 16), (16, 19), (16, 13)):
            assert abs(float(r.m_alpha[y, x]) - abs(margin)) < 2e-6, (margin, r.m_alpha[y, x])
            assert bool(r.fragile[y, x] & 1) == fragile
            assert r.n_contrib[y, x] == (1 if margin > 0 else 0)   # above the floor it blends, below it does not
        # the neighbouring radii are far from the threshold: never flagged
        assert not (r.fragile[16, 16] & 1) and not (r.fragile[16, 18] & 1) and not (r.fragile[16, 20] & 1)


def _stack(o, n=7):
    return scenes.single_gaussian_scene(np.tile([[0.0, 0.0, 4.0]], (n, 1)), [0.3, 0.3, 0.3], [1, 0, 0, 0], o,
                                        np.tile([0.7, 0.4, 0.2], (n, 1)), [0.0, 0.0, 0.0], 33, 33, 40.0, 40.0)


def test_fragile_T_bit_on_both_sides_of_the_threshold():
    """Identical centred Gaussians: at the centre pixel alpha = o, T' after k of them = (1 - o)^k.  With
    (1 - o)^4 = 1e-4 (1 + eps): eps > 0 -> the 4th is blended (n = 4, then the 5th stops); eps < 0 -> the 4th stops
    (n = 3, rule R1: the crossing Gaussian is not blended).  m_T = |eps| either way; bit 1 iff |eps| < delta."""
    for eps, fragile in ((+0.5e-3, True), (-0.5e-3, True), (+2e-3, False), (-2e-3, False)):
        q = (T_MIN * (1.0 + eps)) ** 0.25
        o32 = float(np.float32(1.0 - q))
        r = oracle.render(_stack(o32), fragile_delta=DELTA)
        steps = [(1.0 - o32) ** k for k in range(1, 8)]
        n_want = 4 if eps > 0 else 3
        m_want = min(abs(t / T_MIN - 1.0) for t in steps[: n_want + 1])   # every T' formed, the stopping one included
        assert abs(m_want - abs(eps)) < 1e-5
        assert r.n_contrib[16, 16] == n_want and r.last_k[16, 16] == n_want
        assert abs(float(r.m_T[16, 16]) - m_want) < 2e-6, (eps, r.m_T[16, 16], m_want)
        assert bool(r.fragile[16, 16] & 2) == fragile
        assert abs(float(r.final_T[16, 16]) - steps[n_want - 1]) < 1e-9
        assert not (r.fragile[16, 16] & 1)               # alpha = o ~ 0.9: far from 1/255


def test_fragile_delta_argument_is_the_threshold():
    sig2 = _sigma2()
    o = math.exp(LN_AMIN + 9.0 / (2 * sig2) + 2e-3)
    assert not (oracle.render(_one(o), fragile_delta=1e-3).fragile[16, 19] & 1)
    assert oracle.render(_one(o), fragile_delta=3e-3).fragile[16, 19] & 1


def test_fragile_share_of_a_dense_scene_is_a_few_percent():
    """SURVEY.md 8(c) parity protocol: about 20 delta of the pixels have an alpha within delta of 1/255 and about
    12 delta a T' within delta of 1e-4, i.e. ~3 % at delta = 1e-3.  An over-flagging classifier would loosen parity."""
    sc = scenes.make_scene(2, P=20_000, W=256, H=192, f=300.0, poses=2)
    r = oracle.render(sc, 1, n_threads=4, fragile_delta=DELTA)
    share = float((r.fragile != 0).mean())
    assert 1e-4 < share < 0.05, share
    assert np.array_equal(r.fragile != 0, (r.m_alpha < DELTA) | (r.m_T < DELTA))


# ---------------------------------------------------------------------------------------------------------------------
# guard band (C-P4, reading S3)
# ---------------------------------------------------------------------------------------------------------------------
def _numpy_cov(sc, clamp):
    """float64 library restatement of C-P0..C-P7 with (clamp=True) or without the guard band of reading S3."""
    cam = sc.cameras[0]
    V = cam.viewmatrix.astype(np.float64); W, H, fx, fy = cam.W, cam.H, cam.fx, cam.fy
    pc = sc.means3D.astype(np.float64) @ V[:3, :3].T + V[:3, 3]
    q = sc.rotations.astype(np.float64)
    R = Rotation.from_quat(q[:, [1, 2, 3, 0]]).as_matrix()
    S = sc.scales.astype(np.float64)
    Sig = np.einsum("nij,nj,nkj->nik", R, S * S, R)
    limx, limy = 1.3 * (0.5 * W) / fx, 1.3 * (0.5 * H) / fy
    xz, yz = pc[:, 0] / pc[:, 2], pc[:, 1] / pc[:, 2]
    if clamp:
        xz, yz = np.clip(xz, -limx, limx), np.clip(yz, -limy, limy)
    tx, ty, tz = xz * pc[:, 2], yz * pc[:, 2], pc[:, 2]
    conic = np.zeros((sc.P, 3)); radius = np.zeros(sc.P, int)
    for i in range(sc.P):
        J = np.array([[fx / tz[i], 0, -fx * tx[i] / tz[i] ** 2], [0, fy / tz[i], -fy * ty[i] / tz[i] ** 2]])
        cov = J @ V[:3, :3] @ Sig[i] @ V[:3, :3].T @ J.T + 0.3 * np.eye(2)
        ci = np.linalg.inv(cov)
        conic[i] = (ci[0, 0], ci[0, 1], ci[1, 1])
        lam = max(np.linalg.eigvalsh(cov)[-1], 0.5 * np.trace(cov) + math.sqrt(0.1))
        radius[i] = int(math.ceil(3 * math.sqrt(lam)))
    active = (np.abs(pc[:, 0] / pc[:, 2]) > limx) | (np.abs(pc[:, 1] / pc[:, 2]) > limy)
    return conic, radius, active


def test_guard_band_clamp_matches_numpy_clip_restatement():
    rng = np.random.default_rng(11)
    P, W, H, f = 600, 96, 80, 96.0
    tanx, tany = 0.5 * W / f, 0.5 * H / f
    z = rng.uniform(2.0, 4.0, P)
    # |x/z| in [1, 3] tan(fov/2) on one axis, anything inside the frustum on the other; both signs
    side = rng.random(P) < 0.5
    u = rng.uniform(1.0, 3.0, P) * rng.choice([-1.0, 1.0], P)
    v = rng.uniform(-0.9, 0.9, P)
    xz = np.where(side, u * tanx, v * tanx)
    yz = np.where(side, v * tany, u * tany)
    means = np.stack([xz * z, yz * z, z], 1)
    scales = np.exp(rng.normal(-0.3, 0.35, (P, 3)))          # large splats: off-screen centres still reach the image
    q = rng.standard_normal((P, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    sc = scenes.single_gaussian_scene(means, scales, q, np.full(P, 0.5), np.full((P, 3), 0.5), [0, 0, 0], W, H, f, f)
    r = oracle.render(sc, flags=oracle.NO_LISTS)
    conic, radius, active = _numpy_cov(sc, clamp=True)
    conic_raw, radius_raw, _ = _numpy_cov(sc, clamp=False)
    vis = r.tiles_touched > 0
    sub = vis & active
    assert sub.sum() >= 100 and (vis & ~active).sum() >= 50, (sub.sum(), (vis & ~active).sum())
    rel = np.abs(r.conic - conic) / (np.abs(conic) + 1e-4)
    assert rel[vis].max() < 2e-3, rel[vis].max()
    assert np.abs(r.radius[vis] - radius[vis]).max() <= 1
    assert (r.radius[vis] == radius[vis]).mean() > 0.98
    # the pin is sensitive: WITHOUT the clamp the same restatement misses the oracle on the clamped subset
    rel_raw = np.abs(r.conic - conic_raw) / (np.abs(conic_raw) + 1e-4)
    assert np.median(rel_raw[sub].max(axis=1)) > 2e-2
    assert (np.abs(r.radius[sub] - radius_raw[sub]) > 1).mean() > 0.3
    # and the limit is 1.3, not 1.0 or something larger: Gaussians between 1.0 and 1.3 tan(fov/2) are NOT clamped
    between = vis & ~active & ((np.abs(means[:, 0] / z) > tanx) | (np.abs(means[:, 1] / z) > tany))
    assert between.sum() >= 10
    assert rel_raw[between].max() < 2e-3
