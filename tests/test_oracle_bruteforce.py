"""Pins T4, T8: tiled oracle == untiled brute force; permutation invariance; an independent numpy
float64 restatement built from LIBRARY routines (np.linalg.inv / eigvalsh, scipy Rotation) within tolerance."""
import numpy as np
from scipy.spatial.transform import Rotation

from oracle import oracle
from paper_2606_16566_b200 import scenes


def test_t4_tiled_equals_untiled_bitwise_config1_small():
    sc = scenes.make_scene(1, P=300, W=70, H=45, f=70.0)   # ragged tail in both directions
    r = oracle.render(sc)
    img, fT, nc = oracle.render_untiled(sc, use_rect=True)
    assert np.array_equal(img, r.image) and np.array_equal(fT, r.final_T) and np.array_equal(nc, r.n_contrib)


def test_t4_random_scenes_and_rect_truncation_is_small():
    for P, cfg in ((150, 2), (200, 3)):
        sc = scenes.make_scene(cfg, P=P, W=64, H=48, f=60.0, poses=2)
        for ci in range(2):
            r = oracle.render(sc, ci)
            img, fT, nc = oracle.render_untiled(sc, ci, use_rect=True)
            assert np.array_equal(img, r.image) and np.array_equal(nc, r.n_contrib)
            img2, _, _ = oracle.render_untiled(sc, ci, use_rect=False)
            # the 3-sigma rect truncates opaque splats slightly (alpha can exceed 1/255 beyond 3 sigma when o > 0.353)
            assert np.abs(img2 - r.image).max() < 0.05


def _numpy_reference(sc, ci=0):
    """float64, untiled, library linear algebra; only valid when no Gaussian hits the guard band / culls."""
    cam = sc.cameras[ci]
    V = cam.viewmatrix.astype(np.float64); W, H, fx, fy = cam.W, cam.H, cam.fx, cam.fy
    P = sc.P
    p = sc.means3D.astype(np.float64)
    pc = p @ V[:3, :3].T + V[:3, 3]
    mu = np.stack([fx * pc[:, 0] / pc[:, 2] + (W - 1) / 2, fy * pc[:, 1] / pc[:, 2] + (H - 1) / 2], 1)
    q = sc.rotations.astype(np.float64)
    R = Rotation.from_quat(q[:, [1, 2, 3, 0]]).as_matrix()      # scipy wants (x,y,z,w)
    S = sc.scales.astype(np.float64)
    Sig = np.einsum("nij,nj,nkj->nik", R, S * S, R)
    conic = np.zeros((P, 2, 2)); radius = np.zeros(P, int)
    for i in range(P):
        x, y, z = pc[i]
        J = np.array([[fx / z, 0, -fx * x / z ** 2], [0, fy / z, -fy * y / z ** 2]])
        cov = J @ V[:3, :3] @ Sig[i] @ V[:3, :3].T @ J.T + 0.3 * np.eye(2)
        conic[i] = np.linalg.inv(cov)
        lam = max(np.linalg.eigvalsh(cov)[-1], 0.5 * np.trace(cov) + np.sqrt(0.1))   # reading S5: discriminant floor 0.1
        radius[i] = int(np.ceil(3 * np.sqrt(lam)))
    campos = -V[:3, :3].T @ V[:3, 3]
    d = p - campos; d /= np.linalg.norm(d, axis=1, keepdims=True)
    rgb = np.zeros((P, 3))
    for i in range(P):
        rgb[i] = np.maximum(0, 0.5 + oracle.sh_basis(sc.sh_degree, d[i])[: sc.sh.shape[1]] @ sc.sh[i].astype(np.float64))
    order = np.lexsort((np.arange(P), pc[:, 2].astype(np.float32).view(np.uint32)))
    yy, xx = np.mgrid[0:H, 0:W].astype(np.float64)
    T = np.ones((H, W)); C = np.zeros((3, H, W)); done = np.zeros((H, W), bool)
    gx0 = np.floor((mu[:, 0] - radius) / 16); gx1 = np.floor((mu[:, 0] + radius + 15) / 16)
    gy0 = np.floor((mu[:, 1] - radius) / 16); gy1 = np.floor((mu[:, 1] + radius + 15) / 16)
    for g in order:
        if pc[g, 2] <= 0.2:
            continue
        dx, dy = xx - mu[g, 0], yy - mu[g, 1]
        power = -0.5 * (conic[g, 0, 0] * dx * dx + conic[g, 1, 1] * dy * dy) - conic[g, 0, 1] * dx * dy
        a = np.minimum(0.99, float(sc.opacities[g]) * np.exp(power))
        inrect = (xx // 16 >= gx0[g]) & (xx // 16 < gx1[g]) & (yy // 16 >= gy0[g]) & (yy // 16 < gy1[g])
        ok = (a >= 1 / 255) & inrect & ~done
        Tn = T * (1 - a)
        stop = ok & (Tn < 1e-4)
        done |= stop
        ok &= ~stop
        C += np.where(ok, a * T, 0)[None] * rgb[g][:, None, None]
        T = np.where(ok, Tn, T)
    return C + T[None] * sc.bg.astype(np.float64)[:, None, None], T, mu, conic, radius, rgb


def test_numpy_float64_library_restatement_config1():
    sc = scenes.make_scene(1, P=256, W=96, H=80, f=96.0)
    r = oracle.render(sc)
    img, T, mu, conic, radius, rgb = _numpy_reference(sc)
    vis = r.tiles_touched > 0
    assert np.abs(r.mu[vis] - mu[vis]).max() < 2e-3
    ca = np.stack([conic[:, 0, 0], conic[:, 0, 1], conic[:, 1, 1]], 1)
    assert (np.abs(r.conic[vis] - ca[vis]) / (np.abs(ca[vis]) + 1e-3)).max() < 2e-3
    assert (r.radius[vis] == radius[vis]).mean() > 0.99 and np.abs(r.radius[vis] - radius[vis]).max() <= 1
    assert np.abs(r.rgb[vis] - rgb[vis]).max() < 1e-5
    bad = np.abs(r.image - img).max(0) > 1e-4
    assert bad.mean() < 5e-3      # threshold crossings / off-by-one radii only
    assert np.abs(r.image - img).max() < 0.02


def test_numpy_float64_library_restatement_config2_view_dependent():
    sc = scenes.make_scene(2, P=400, W=80, H=64, f=90.0, poses=4)
    for ci in (0, 1, 3):
        r = oracle.render(sc, ci)
        img, T, mu, conic, radius, rgb = _numpy_reference(sc, ci)
        vis = r.tiles_touched > 0
        assert np.abs(r.mu[vis] - mu[vis]).max() < 2e-3
        assert np.abs(r.rgb[vis] - rgb[vis]).max() < 1e-5
        bad = np.abs(r.image - img).max(0) > 1e-4
        assert bad.mean() < 5e-3 and np.abs(r.image - img).max() < 0.02


def test_t8_permutation_invariance():
    """Shuffling the input order permutes ids but leaves the image unchanged (no exact depth ties in this scene)."""
    sc = scenes.make_scene(2, P=500, W=64, H=64, f=70.0, poses=1)
    r = oracle.render(sc)
    assert len(np.unique(r.depth_bits[r.tiles_touched > 0])) == (r.tiles_touched > 0).sum()
    perm = np.random.default_rng(3).permutation(sc.P)
    sc2 = scenes.Scene(sc.name, sc.config, sc.means3D[perm], sc.scales[perm], sc.rotations[perm], sc.opacities[perm], sc.sh[perm],
                       sc.sh_degree, sc.bg, sc.cameras)
    r2 = oracle.render(sc2)
    assert np.array_equal(r.image, r2.image) and np.array_equal(r.n_contrib, r2.n_contrib)
    assert np.array_equal(perm[r2.sorted_ids], r.sorted_ids)
