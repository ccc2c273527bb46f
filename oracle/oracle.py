"""ctypes binding of libgs_oracle.so (see gs_oracle.h).  Test infrastructure only."""
from __future__ import annotations

import ctypes as C
import os
from types import SimpleNamespace

import numpy as np

from . import build_oracle

NO_RENDER = 1
NO_LISTS = 2
TILE_CULL = 4
TILE_CULL_EXACT = 8   # C-P8'': TILE_CULL's rect + exact ellipse-tile test per (tile, Gaussian)

_u32p, _i32p, _f32p, _u64p, _u8p = (C.POINTER(t) for t in (C.c_uint32, C.c_int32, C.c_float, C.c_uint64, C.c_uint8))


class _View(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("P", "W", "H", "grid_x", "grid_y", "n_tiles", "n_lists", "full")] + [
        ("n_dup", C.c_uint64), ("n_list_entries", C.c_uint64), ("pairs_traversed", C.c_uint64), ("pairs_blended", C.c_uint64),
        ("depth_bits", _u32p), ("radius", _i32p), ("rect", _i32p), ("tiles_touched", _u32p),
        ("mu", _f32p), ("conic", _f32p), ("rgb", _f32p),
        ("tile_counts", _u32p), ("list_tile", _i32p), ("list_offsets", _u64p), ("sorted_ids", _u32p),
        ("image", _f32p), ("final_T", _f32p), ("n_contrib", _u32p), ("last_k", _u32p), ("fragile", _u8p),
        ("m_alpha", _f32p), ("m_T", _f32p), ("rendered", _u8p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = build_oracle.build()
        L = C.CDLL(path)
        fp, ip = C.c_void_p, C.c_void_p
        L.gs_oracle_render.restype = C.c_void_p
        L.gs_oracle_render.argtypes = [C.c_int, fp, fp, fp, fp, fp, C.c_int, fp, fp, C.c_float, C.c_float, C.c_int, C.c_int,
                                       fp, ip, C.c_int, C.c_int, C.c_int, C.c_double]
        L.gs_oracle_get_view.argtypes = [C.c_void_p, C.POINTER(_View)]
        L.gs_oracle_get_view.restype = None
        L.gs_oracle_free.argtypes = [C.c_void_p]
        L.gs_oracle_free.restype = None
        L.gs_oracle_render_untiled.restype = C.c_int
        L.gs_oracle_render_untiled.argtypes = [C.c_int, fp, fp, fp, fp, fp, C.c_int, fp, fp, C.c_float, C.c_float, C.c_int,
                                               C.c_int, fp, C.c_int, fp, fp, fp]
        L.gs_oracle_hoist.argtypes = [C.c_double] * 6 + [C.POINTER(C.c_double)]
        L.gs_oracle_hoist.restype = None
        L.gs_oracle_warp_mask.argtypes = [C.c_double] * 8 + [C.POINTER(C.c_double)]
        L.gs_oracle_warp_mask.restype = C.c_uint32
        L.gs_oracle_sh_basis.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.gs_oracle_sh_basis.restype = None
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.c_void_p)


def _arr(ptr, shape, dtype):
    n = int(np.prod(shape))
    if n == 0:
        return np.zeros(shape, dtype=dtype)
    return np.ctypeslib.as_array(ptr, shape=(n,)).view(dtype).reshape(shape).copy()


def render(scene, cam_index=0, tile_subset=None, n_threads=1, flags=0, fragile_delta=1e-3):
    """Runs the oracle on ``scene`` (a paper_2606_16566_b200.scenes.Scene-like object) and returns numpy copies."""
    cam = scene.cameras[cam_index]
    keep = [_f32(x) for x in (scene.means3D, scene.scales, scene.rotations, scene.opacities, scene.sh,
                              cam.viewmatrix, cam.projmatrix, scene.bg)]
    sub_ptr, n_sub = None, 0
    if tile_subset is not None:
        sub = np.ascontiguousarray(tile_subset, dtype=np.int32)
        sub_ptr, n_sub = sub.ctypes.data_as(C.c_void_p), int(sub.size)
    L = lib()
    h = L.gs_oracle_render(scene.means3D.shape[0], keep[0][1], keep[1][1], keep[2][1], keep[3][1], keep[4][1],
                           int(scene.sh_degree), keep[5][1], keep[6][1], float(cam.fx), float(cam.fy), int(cam.W), int(cam.H),
                           keep[7][1], sub_ptr, n_sub, int(n_threads), int(flags), float(fragile_delta))
    if not h:
        raise ValueError("gs_oracle_render rejected its arguments")
    try:
        v = _View()
        L.gs_oracle_get_view(h, C.byref(v))
        P, W, H, T, nl = v.P, v.W, v.H, v.n_tiles, v.n_lists
        out = SimpleNamespace(
            P=P, W=W, H=H, grid_x=v.grid_x, grid_y=v.grid_y, n_tiles=T, n_lists=nl, full=bool(v.full),
            n_dup=int(v.n_dup), pairs_traversed=int(v.pairs_traversed), pairs_blended=int(v.pairs_blended),
            depth_bits=_arr(v.depth_bits, (P,), np.uint32), radius=_arr(v.radius, (P,), np.int32),
            rect=_arr(v.rect, (P, 4), np.int32), tiles_touched=_arr(v.tiles_touched, (P,), np.uint32),
            mu=_arr(v.mu, (P, 2), np.float32), conic=_arr(v.conic, (P, 3), np.float32), rgb=_arr(v.rgb, (P, 3), np.float32),
            tile_counts=_arr(v.tile_counts, (T,), np.uint32), list_tile=_arr(v.list_tile, (nl,), np.int32),
            list_offsets=_arr(v.list_offsets, (nl + 1,), np.uint64),
            sorted_ids=_arr(v.sorted_ids, (int(v.n_list_entries),), np.uint32),
            image=_arr(v.image, (3, H, W), np.float32), final_T=_arr(v.final_T, (H, W), np.float32),
            n_contrib=_arr(v.n_contrib, (H, W), np.uint32), last_k=_arr(v.last_k, (H, W), np.uint32),
            fragile=_arr(v.fragile, (H, W), np.uint8), m_alpha=_arr(v.m_alpha, (H, W), np.float32),
            m_T=_arr(v.m_T, (H, W), np.float32), rendered=_arr(v.rendered, (T,), np.uint8))
    finally:
        L.gs_oracle_free(h)
    return out


def render_untiled(scene, cam_index=0, use_rect=True):
    cam = scene.cameras[cam_index]
    keep = [_f32(x) for x in (scene.means3D, scene.scales, scene.rotations, scene.opacities, scene.sh,
                              cam.viewmatrix, cam.projmatrix, scene.bg)]
    H, W = cam.H, cam.W
    img = np.zeros((3, H, W), np.float32)
    fT = np.zeros((H, W), np.float32)
    nc = np.zeros((H, W), np.uint32)
    rc = lib().gs_oracle_render_untiled(scene.means3D.shape[0], keep[0][1], keep[1][1], keep[2][1], keep[3][1], keep[4][1],
                                        int(scene.sh_degree), keep[5][1], keep[6][1], float(cam.fx), float(cam.fy), W, H,
                                        keep[7][1], int(bool(use_rect)), img.ctypes.data_as(C.c_void_p),
                                        fT.ctypes.data_as(C.c_void_p), nc.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise ValueError("gs_oracle_render_untiled rejected its arguments")
    return img, fT, nc


def hoist(a, b, c, o, dx, dy):
    V = (C.c_double * 6)()
    lib().gs_oracle_hoist(a, b, c, o, dx, dy, V)
    return np.array(V[:], dtype=np.float64)


def warp_mask(a, b, c, o, mux, muy, Tx, Ty):
    span = (C.c_double * 2)()
    m = lib().gs_oracle_warp_mask(a, b, c, o, mux, muy, Tx, Ty, span)
    return int(m), (span[0], span[1])


def sh_basis(deg, d):
    dd = (C.c_double * 3)(*[float(x) for x in d])
    out = (C.c_double * 16)()
    lib().gs_oracle_sh_basis(int(deg), dd, out)
    return np.array(out[:], dtype=np.float64)
