"""Input generators: determinism, shapes, the statistics BASELINE.json configs state."""
import numpy as np

from paper_2606_16566_b200 import scenes


def test_deterministic_and_shapes():
    a, b = scenes.make_scene(2, P=5000), scenes.make_scene(2, P=5000)
    for x, y in ((a.means3D, b.means3D), (a.scales, b.scales), (a.rotations, b.rotations), (a.opacities, b.opacities), (a.sh, b.sh)):
        assert x.dtype == np.float32 and np.array_equal(x, y)
    assert a.sh.shape == (5000, 16, 3) and len(a.cameras) == 8 and a.cameras[0].W == 800
    assert np.abs(np.linalg.norm(a.rotations, axis=1) - 1).max() < 1e-6
    assert (a.scales > 0).all() and (a.opacities > 0).all() and (a.opacities < 1).all()
    assert abs(np.log(a.scales).mean() + 4.5) < 0.05 and abs(np.log(a.scales).std() - 0.7) < 0.05


def test_camera_conventions():
    cam = scenes.make_scene(2, P=10).cameras[3]
    V, PM = cam.viewmatrix.astype(np.float64), cam.projmatrix.astype(np.float64)
    R = V[:3, :3]
    assert np.abs(R @ R.T - np.eye(3)).max() < 1e-6 and abs(np.linalg.det(R) - 1) < 1e-6
    eye = -R.T @ V[:3, 3]
    assert abs(np.linalg.norm(eye) - 4.0) < 1e-5
    p = np.array([0.1, -0.2, 0.3, 1.0])
    pc, h = V @ p, PM @ p
    assert abs(h[3] - pc[2]) < 1e-5
    mux = ((h[0] / h[3] + 1) * cam.W - 1) / 2
    assert abs(mux - (cam.fx * pc[0] / pc[2] + (cam.W - 1) / 2)) < 1e-3
    # the camera looks at the origin: the origin projects to the image centre
    h0 = PM @ np.array([0, 0, 0, 1.0])
    assert abs(h0[0] / h0[3]) < 1e-5 and abs(h0[1] / h0[3]) < 1e-5


def test_all_configs_build_small():
    for c in range(1, 6):
        s = scenes.make_scene(c, P=2000)
        assert s.P == 2000 and s.means3D.shape == (2000, 3) and np.isfinite(s.means3D).all() and np.isfinite(s.scales).all()
        d = scenes.config_defaults(c)
        assert len(s.cameras) == d["poses"] and s.cameras[0].W == d["W"] and s.cameras[0].H == d["H"]
