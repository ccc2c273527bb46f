"""Seeded synthetic 3DGS scenes and cameras (input generators only).

This module serves BOTH the CUDA path and the CPU oracle with identical bytes.  It holds
none of the method's arithmetic: no projection of Gaussians, no conics, no SH evaluation,
no blending -- only random draws, activations of raw parameters (exp / sigmoid) and the
camera matrices that are *inputs* of ``gs_render``.

The five configurations follow BASELINE.json ``configs`` as completed in SURVEY.md §8(d)
(DESIGN.md "Input recipe").  They stand in for the trained Mip-NeRF 360 / Tanks & Temples /
Deep Blending models the paper measures on, which are not available here.

Conventions (readings S1, S18, S19):
  * camera frame: x right, y down, z forward; matrices row-major, column-vector convention
    ``p_cam = V @ [p, 1]``; ``PM = Proj @ V`` is the full transform handed to ``gs_render``;
  * quaternions are (w, x, y, z), unit; scales and opacities are ACTIVATED;
  * SH coefficients ``[P, K, 3]``, K = (deg+1)^2, RGB innermost; the DC coefficient is
    ``(rgb - 0.5) * 2*sqrt(pi)``.
Generator: ``numpy.random.Generator(PCG64(seed))``, float64 draws cast to float32 once.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np

TILE = 16
SH_C0_INV = 2.0 * math.sqrt(math.pi)  # 1 / Y_00


@dataclasses.dataclass
class Camera:
    viewmatrix: np.ndarray  # [4,4] float32 row-major, p_cam = V @ [p;1]
    projmatrix: np.ndarray  # [4,4] float32 row-major, FULL transform Proj @ V
    fx: float
    fy: float
    W: int
    H: int


@dataclasses.dataclass
class Scene:
    name: str
    config: int
    means3D: np.ndarray    # [P,3] f32
    scales: np.ndarray     # [P,3] f32, activated (positive)
    rotations: np.ndarray  # [P,4] f32, unit quaternion (w,x,y,z)
    opacities: np.ndarray  # [P]   f32, activated, in (0,1)
    sh: np.ndarray         # [P,K,3] f32
    sh_degree: int
    bg: np.ndarray         # [3] f32
    cameras: List[Camera]

    @property
    def P(self) -> int:
        return int(self.means3D.shape[0])

    def input_bytes(self) -> int:
        return sum(a.nbytes for a in (self.means3D, self.scales, self.rotations, self.opacities, self.sh))


# --------------------------------------------------------------------------------------
# cameras
# --------------------------------------------------------------------------------------
def _normalize(v):
    return v / np.linalg.norm(v)


def lookat(eye, target) -> np.ndarray:
    """World->camera matrix, float64 [4,4]; y is DOWN in the camera frame."""
    eye = np.asarray(eye, dtype=np.float64)
    target = np.asarray(target, dtype=np.float64)
    z_c = _normalize(target - eye)
    x_c = _normalize(np.cross(np.array([0.0, 1.0, 0.0]), z_c))
    y_c = np.cross(z_c, x_c)
    V = np.eye(4)
    V[0, :3], V[0, 3] = x_c, -x_c @ eye
    V[1, :3], V[1, 3] = y_c, -y_c @ eye
    V[2, :3], V[2, 3] = z_c, -z_c @ eye
    return V


def projection(fx, fy, W, H, zn=0.01, zf=100.0) -> np.ndarray:
    """Reading S18: ndc_x = (2 fx / W) x / z, so that mu_x = fx x/z + (W-1)/2."""
    Pm = np.zeros((4, 4))
    Pm[0, 0] = 2.0 * fx / W
    Pm[1, 1] = 2.0 * fy / H
    Pm[2, 2] = zf / (zf - zn)
    Pm[2, 3] = -zf * zn / (zf - zn)
    Pm[3, 2] = 1.0
    return Pm


def make_camera(V64: np.ndarray, fx: float, fy: float, W: int, H: int) -> Camera:
    PM = projection(fx, fy, W, H) @ V64
    return Camera(np.ascontiguousarray(V64, dtype=np.float32), np.ascontiguousarray(PM, dtype=np.float32),
                  float(fx), float(fy), int(W), int(H))


# --------------------------------------------------------------------------------------
# draws
# --------------------------------------------------------------------------------------
_CHUNK = 1 << 22


def _normal(rng, shape, mean=0.0, std=1.0) -> np.ndarray:
    """float64 standard-normal stream, drawn in chunks (same stream as one big draw), cast to f32 once."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)
    for s in range(0, n, _CHUNK):
        e = min(n, s + _CHUNK)
        out[s:e] = (mean + std * rng.standard_normal(e - s)).astype(np.float32)
    return out.reshape(shape)


def _uniform(rng, shape, lo=0.0, hi=1.0) -> np.ndarray:
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float64)
    for s in range(0, n, _CHUNK):
        e = min(n, s + _CHUNK)
        out[s:e] = lo + (hi - lo) * rng.random(e - s)
    return out.reshape(shape)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x.astype(np.float64)))


def _common_attributes(rng, P, ls_mean, ls_std, op_mean, op_std, sh_degree, ls_extra=None):
    """log-scales -> quaternions -> opacity logits -> DC colour -> higher SH bands (SURVEY §8(d) draw order)."""
    log_s = _normal(rng, (P, 3), ls_mean, ls_std).astype(np.float64)
    if ls_extra is not None:
        log_s = log_s + ls_extra[:, None]
    scales = np.exp(log_s).astype(np.float32)
    q = _normal(rng, (P, 4)).astype(np.float64)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    rotations = q.astype(np.float32)
    opac = _sigmoid(_normal(rng, (P,), op_mean, op_std)).astype(np.float32)
    K = (sh_degree + 1) ** 2
    sh = np.empty((P, K, 3), dtype=np.float32)
    rgb = _uniform(rng, (P, 3))
    sh[:, 0, :] = ((rgb - 0.5) * SH_C0_INV).astype(np.float32)
    if K > 1:
        sh[:, 1:, :] = _normal(rng, (P, K - 1, 3), 0.0, 0.05)
    return scales, rotations, opac, sh


def _random_rotations(rng, n) -> np.ndarray:
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - w * z); R[:, 0, 2] = 2 * (x * z + w * y)
    R[:, 1, 0] = 2 * (x * y + w * z); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - w * x)
    R[:, 2, 0] = 2 * (x * z - w * y); R[:, 2, 1] = 2 * (y * z + w * x); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


# --------------------------------------------------------------------------------------
# the five configurations
# --------------------------------------------------------------------------------------
_DEFAULTS = {
    1: dict(P=1024, W=128, H=128, f=128.0, deg=0, poses=1, name="tiny"),
    2: dict(P=100_000, W=800, H=800, f=1111.0, deg=3, poses=8, name="object-centric"),
    3: dict(P=1_500_000, W=1264, H=832, f=1000.0, deg=3, poses=16, name="indoor-dense"),
    4: dict(P=3_500_000, W=1920, H=1080, f=1500.0, deg=3, poses=16, name="outdoor-unbounded"),
    5: dict(P=10_000_000, W=3840, H=2160, f=3000.0, deg=3, poses=8, name="city-overlap-stress"),
}


def config_defaults(config: int) -> dict:
    return dict(_DEFAULTS[config])


def make_scene(config: int, P: Optional[int] = None, W: Optional[int] = None, H: Optional[int] = None,
               f: Optional[float] = None, poses: Optional[int] = None, sh_degree: Optional[int] = None) -> Scene:
    """Build configuration ``config`` (1..5).  Overrides shrink a config for oracle-sized parity cases;
    with no overrides the result is the BASELINE.json configuration (seed = config - 1)."""
    d = config_defaults(config)
    P = d["P"] if P is None else int(P)
    W = d["W"] if W is None else int(W)
    H = d["H"] if H is None else int(H)
    f = d["f"] if f is None else float(f)
    n_pose = d["poses"] if poses is None else int(poses)
    deg = d["deg"] if sh_degree is None else int(sh_degree)
    rng = np.random.Generator(np.random.PCG64(config - 1))
    ls_extra = None
    if config == 1:
        xy = _uniform(rng, (P, 2), -1.0, 1.0)
        z = _uniform(rng, (P, 1), 2.0, 4.0)
        means = np.concatenate([xy, z], axis=1)
        attrs = (-3.0, 0.5, 0.0, 1.5)
        bg = np.zeros(3, np.float32)
        views = [np.eye(4)]
    elif config == 2:
        means = _normal(rng, (P, 3), 0.0, 0.6).astype(np.float64)
        attrs = (-4.5, 0.7, 0.5, 2.0)
        bg = np.ones(3, np.float32)
        el = math.radians(20.0)
        views = []
        for k in range(n_pose):
            az = 2.0 * math.pi * k / n_pose
            eye = 4.0 * np.array([math.cos(el) * math.sin(az), -math.sin(el), -math.cos(el) * math.cos(az)])
            views.append(lookat(eye, np.zeros(3)))
    elif config == 3:
        half = np.array([5.0, 2.0, 5.0])
        centres = _uniform(rng, (64, 3), -1.0, 1.0) * half
        sig = np.exp(_uniform(rng, (64, 3), math.log(0.15), math.log(1.5)))
        R = _random_rotations(rng, 64)
        cid = np.arange(P) % 64
        local = _normal(rng, (P, 3)).astype(np.float64) * sig[cid]
        means = centres[cid] + np.einsum("nij,nj->ni", R[cid], local)
        means = np.clip(means, -half, half)
        attrs = (-4.0, 1.0, 0.0, 2.0)
        bg = np.zeros(3, np.float32)
        views = []
        for k in range(n_pose):
            th = 2.0 * math.pi * k / n_pose
            eye = np.array([2.5 * math.cos(th), 0.3 * math.sin(2 * th), 2.5 * math.sin(th)])
            views.append(lookat(eye, np.zeros(3)))
    elif config == 4:
        n_fg = int(round(0.8 * P))
        n_bg = P - n_fg
        fg = _normal(rng, (n_fg, 3), 0.0, 2.0).astype(np.float64)
        d3 = _normal(rng, (n_bg, 3)).astype(np.float64)
        d3 /= np.linalg.norm(d3, axis=1, keepdims=True)
        r = np.exp(_uniform(rng, (n_bg,), math.log(10.0), math.log(200.0)))
        means = np.concatenate([fg, d3 * r[:, None]], axis=0)
        ls_extra = np.concatenate([np.zeros(n_fg), np.log(r)])
        attrs = (-3.5, 1.2, 0.0, 2.0)
        bg = np.zeros(3, np.float32)
        views = []
        for k in range(n_pose):
            th = 2.0 * math.pi * k / n_pose
            views.append(lookat(np.array([3.0 * math.cos(th), 0.0, 3.0 * math.sin(th)]), np.zeros(3)))
    elif config == 5:
        nb = 400
        bc = np.stack([_uniform(rng, (nb,), -100.0, 100.0), _uniform(rng, (nb,), -100.0, 100.0)], axis=1)
        wd = _uniform(rng, (nb, 2), 4.0, 12.0)
        hh = _uniform(rng, (nb,), 5.0, 20.0)
        vol_b = wd[:, 0] * wd[:, 1] * hh
        v_slab = 200.0 * 20.0 * 200.0
        p_b = 10.0 * vol_b.sum() / (v_slab + 10.0 * vol_b.sum())
        u_sel = _uniform(rng, (P,))
        in_b = u_sel < p_b
        cdf = np.cumsum(vol_b) / vol_b.sum()
        which = np.minimum(np.searchsorted(cdf, _uniform(rng, (P,))), nb - 1)
        u3 = _uniform(rng, (P, 3))
        slab = np.stack([-100.0 + 200.0 * u3[:, 0], -20.0 + 20.0 * u3[:, 1], -100.0 + 200.0 * u3[:, 2]], axis=1)
        bx = bc[which, 0] + (u3[:, 0] - 0.5) * wd[which, 0]
        bz = bc[which, 1] + (u3[:, 2] - 0.5) * wd[which, 1]
        by = -u3[:, 1] * hh[which]            # ground at y = 0, up is -y
        bld = np.stack([bx, by, bz], axis=1)
        means = np.where(in_b[:, None], bld, slab)
        attrs = (-2.5, 1.0, 1.0, 1.5)
        bg = np.zeros(3, np.float32)
        views = []
        for k in range(n_pose):
            th = 2.0 * math.pi * k / n_pose
            views.append(lookat(np.array([60.0 * math.cos(th), -30.0, 60.0 * math.sin(th)]), np.array([0.0, -5.0, 0.0])))
    else:
        raise ValueError("config must be 1..5")
    scales, rotations, opac, sh = _common_attributes(rng, P, *attrs, sh_degree=deg, ls_extra=ls_extra)
    cams = [make_camera(V, f, f, W, H) for V in views]
    return Scene(d["name"], config, np.ascontiguousarray(means, dtype=np.float32), scales, rotations, opac, sh, deg, bg, cams)


def single_gaussian_scene(mean, scale, quat, opacity, rgb, bg, W, H, fx, fy, V=None) -> Scene:
    """One degree-0 Gaussian (or several, row-wise) -- the closed-form fixtures of DESIGN.md T1-T3."""
    mean = np.atleast_2d(np.asarray(mean, dtype=np.float32))
    n = mean.shape[0]
    scale = np.broadcast_to(np.asarray(scale, dtype=np.float32), (n, 3)) if np.ndim(scale) < 2 else np.asarray(scale, np.float32)
    quat = np.broadcast_to(np.asarray(quat, dtype=np.float32), (n, 4)) if np.ndim(quat) < 2 else np.asarray(quat, np.float32)
    opacity = np.broadcast_to(np.asarray(opacity, dtype=np.float32), (n,)) if np.ndim(opacity) < 1 else np.asarray(opacity, np.float32)
    rgb = np.broadcast_to(np.asarray(rgb, dtype=np.float64), (n, 3)) if np.ndim(rgb) < 2 else np.asarray(rgb, np.float64)
    sh = ((rgb - 0.5) * SH_C0_INV).astype(np.float32).reshape(n, 1, 3)
    V64 = np.eye(4) if V is None else np.asarray(V, dtype=np.float64)
    return Scene("fixture", 0, np.ascontiguousarray(mean), np.ascontiguousarray(scale), np.ascontiguousarray(quat),
                 np.ascontiguousarray(opacity), np.ascontiguousarray(sh), 0, np.asarray(bg, dtype=np.float32),
                 [make_camera(V64, fx, fy, W, H)])
