"""Thin ctypes binding of libgs.so (include/gs.h): argument marshalling only -- every step of the path runs in the
library's CUDA kernels.  PyTorch supplies device memory and the stream.  There is NO CPU fallback: if the library
cannot be built or loaded, importing this module's functions raises.

Functions mirror the C ABI one to one: gs_workspace_bytes, gs_render, gs_get_intermediates, gs_set_timing,
gs_get_timings, gs_set_render_variant, gs_get_render_variant, gs_last_launch_count, gs_error_string.
"""
from __future__ import annotations

import ctypes as C
import os
from types import SimpleNamespace

import numpy as np
import torch

from . import build as _build

GS_OK, GS_ERR_BAD_ARG, GS_ERR_WORKSPACE, GS_ERR_OVERFLOW, GS_ERR_CUDA, GS_ERR_LIMIT = 0, -1, -2, -3, -4, -5
GS_NOALLOC_MAX_KEYS = 262144   # include/gs.h: key capacity of gs_depth_sort_noalloc's fixed scratch
GS_TILE = 16
GS_DEFAULT_RENDER_VARIANT = 4   # include/gs.h: the B200 render kernel
GS_N_TIMINGS = 8
TIMING_NAMES = ("preprocess", "depth_sort", "tile_grid", "offset_scan", "duplicate", "tile_sort", "render", "frame")

EXPORTS = ("gs_workspace_bytes", "gs_render", "gs_get_intermediates", "gs_set_timing", "gs_get_timings",
           "gs_set_render_variant", "gs_get_render_variant", "gs_last_launch_count", "gs_error_string",
           "gs_last_cuda_error", "gs_copy_to_host", "gs_set_stats", "gs_get_stats", "gs_selftest_atomic_order",
           "gs_set_render_stream", "gs_selftest_issue_peak", "gs_set_tile_cull", "gs_get_tile_cull",
           "gs_set_workspace_option", "gs_release", "gs_set_rank_mode", "gs_get_rank_mode", "gs_set_graph",
           "gs_noalloc_max_keys", "gs_depth_sort_noalloc")
GS_OPT_RENDER_VARIANT, GS_OPT_TILE_CULL, GS_OPT_TIMING, GS_OPT_STATS, GS_OPT_RENDER_STREAM, GS_OPT_GRAPH = range(6)
GS_N_STATS = 4
STATS_NAMES = ("warp_slots_walked", "pairs_blended", "entries_staged", "pairs_evaluated")


class _Intermediates(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("P", "W", "H", "grid_x", "grid_y", "n_tiles")] + [
        ("n_visible", C.c_uint32), ("n_dup", C.c_uint64), ("max_dup", C.c_uint64),
        ("per_gaussian", C.c_void_p), ("record", C.c_void_p), ("depth_sorted", C.c_void_p),
        ("dup_offsets", C.c_void_p), ("tile_ranges", C.c_void_p), ("sorted_ids", C.c_void_p), ("n_coarse", C.c_uint64)]


class GsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().gs_error_string(code).decode()
        if code == GS_ERR_CUDA:
            msg += " (cudaError %d)" % lib().gs_last_cuda_error()
        super().__init__("%s: %s" % (where, msg))


_lib = None


def lib():
    """Loads (building if needed) libgs.so.  Raises if the CUDA extension is unavailable."""
    global _lib
    if _lib is None:
        if os.environ.get("GS_DEBUG_BOUNDS") == "1":   # the bounds-checked build of the same sources (tests only)
            path = _build.build(debug_bounds=True)
        else:
            path = _build.LIB
            if not os.path.exists(path) or os.environ.get("GS_REBUILD"):
                path = _build.build()
        L = C.CDLL(path)
        vp = C.c_void_p
        L.gs_workspace_bytes.restype = C.c_size_t
        L.gs_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_uint64]
        L.gs_render.restype = C.c_int
        L.gs_render.argtypes = [C.c_int, vp, vp, vp, vp, vp, C.c_int, vp, vp, C.c_float, C.c_float, C.c_int, C.c_int, vp,
                                vp, vp, vp, vp, vp, C.c_size_t, vp]
        L.gs_get_intermediates.restype = C.c_int
        L.gs_get_intermediates.argtypes = [vp, C.POINTER(_Intermediates)]
        L.gs_set_timing.restype = C.c_int
        L.gs_set_timing.argtypes = [C.c_int]
        L.gs_get_timings.restype = C.c_int
        L.gs_get_timings.argtypes = [vp, C.POINTER(C.c_float)]
        L.gs_set_render_variant.restype = C.c_int
        L.gs_set_render_variant.argtypes = [C.c_int]
        L.gs_get_render_variant.restype = C.c_int
        L.gs_set_render_stream.restype = C.c_int
        L.gs_set_render_stream.argtypes = [C.c_int]
        L.gs_last_launch_count.restype = C.c_int
        L.gs_error_string.restype = C.c_char_p
        L.gs_error_string.argtypes = [C.c_int]
        L.gs_last_cuda_error.restype = C.c_int
        L.gs_set_stats.restype = C.c_int
        L.gs_set_stats.argtypes = [C.c_int]
        L.gs_get_stats.restype = C.c_int
        L.gs_get_stats.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.gs_copy_to_host.restype = C.c_int
        L.gs_copy_to_host.argtypes = [vp, vp, C.c_size_t]
        L.gs_set_workspace_option.restype = C.c_int
        L.gs_set_workspace_option.argtypes = [vp, C.c_int, C.c_int]
        L.gs_set_graph.restype = C.c_int
        L.gs_set_graph.argtypes = [C.c_int]
        L.gs_release.restype = C.c_int
        L.gs_release.argtypes = [vp]
        L.gs_set_rank_mode.restype = C.c_int
        L.gs_set_rank_mode.argtypes = [C.c_int]
        L.gs_get_rank_mode.restype = C.c_int
        L.gs_set_tile_cull.restype = C.c_int
        L.gs_set_tile_cull.argtypes = [C.c_int]
        L.gs_get_tile_cull.restype = C.c_int
        L.gs_noalloc_max_keys.restype = C.c_uint32
        L.gs_noalloc_max_keys.argtypes = []
        L.gs_depth_sort_noalloc.restype = C.c_int
        L.gs_depth_sort_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        L.gs_selftest_issue_peak.restype = C.c_int
        L.gs_selftest_issue_peak.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.gs_selftest_atomic_order.restype = C.c_int
        L.gs_selftest_atomic_order.argtypes = [C.c_int, C.POINTER(C.c_uint64)]
        _lib = L
    return _lib


def gs_workspace_bytes(P: int, W: int, H: int, max_dup: int) -> int:
    n = lib().gs_workspace_bytes(int(P), int(W), int(H), int(max_dup))
    if n == 0:
        raise GsError(GS_ERR_BAD_ARG, "gs_workspace_bytes")
    return int(n)


def _dev(t: torch.Tensor, dtype, name):
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise ValueError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return C.c_void_p(t.data_ptr())


def _host16(a, n, name):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32).reshape(-1))
    if a.size != n:
        raise ValueError("%s must hold %d floats" % (name, n))
    return a


def gs_render(means3D, scales, rotations, opacities, sh_coeffs, sh_degree, viewmatrix, projmatrix, fx, fy, W, H, bg,
              out_rgb, out_final_T, out_tile_counts, out_n_contrib, workspace, stream=None) -> None:
    """gs_render of include/gs.h.  Per-Gaussian inputs, outputs and `workspace` are CUDA tensors (outputs are
    overwritten in place); viewmatrix/projmatrix/bg are host arrays.  Enqueues on `stream` (default: torch's current
    stream) and returns without synchronising."""
    P = int(means3D.shape[0])
    V = _host16(viewmatrix, 16, "viewmatrix")
    PM = _host16(projmatrix, 16, "projmatrix")
    BG = _host16(bg, 3, "bg")
    if stream is None:
        stream = torch.cuda.current_stream(workspace.device)
    f32, u32 = torch.float32, torch.int32  # torch has no uint32 arithmetic; int32 storage is bit-compatible
    if not (workspace.is_cuda and workspace.is_contiguous() and workspace.dtype == torch.uint8):
        raise ValueError("workspace must be a contiguous CUDA uint8 tensor")
    rc = lib().gs_render(P, _dev(means3D, f32, "means3D"), _dev(scales, f32, "scales"), _dev(rotations, f32, "rotations"),
                         _dev(opacities, f32, "opacities"), _dev(sh_coeffs, f32, "sh_coeffs"), int(sh_degree),
                         V.ctypes.data_as(C.c_void_p), PM.ctypes.data_as(C.c_void_p), float(fx), float(fy), int(W), int(H),
                         BG.ctypes.data_as(C.c_void_p), _dev(out_rgb, f32, "out_rgb"), _dev(out_final_T, f32, "out_final_T"),
                         _dev(out_tile_counts, u32, "out_tile_counts"), _dev(out_n_contrib, u32, "out_n_contrib"),
                         C.c_void_p(workspace.data_ptr()), workspace.numel(), C.c_void_p(stream.cuda_stream))
    if rc != GS_OK:
        raise GsError(rc, "gs_render")


def _copy_out(ptr, count, dtype, device):
    """Device array at raw pointer -> numpy copy (parity tests only)."""
    if count == 0:
        return np.zeros(0, dtype=dtype)
    nbytes = int(count) * np.dtype(dtype).itemsize
    host = np.empty(nbytes, dtype=np.uint8)
    rc = lib().gs_copy_to_host(host.ctypes.data_as(C.c_void_p), C.c_void_p(int(ptr)), nbytes)
    if rc != GS_OK:
        raise GsError(rc, "gs_copy_to_host")
    return host.view(dtype)


def gs_get_intermediates(workspace, copy=("per_gaussian", "tile_ranges", "sorted_ids")):
    """gs_get_intermediates of include/gs.h; the arrays named in `copy` are copied to numpy.  Raises GsError with
    code GS_ERR_OVERFLOW if the frame needed more than max_dup duplicates (n_dup is attached to the exception)."""
    it = _Intermediates()
    rc = lib().gs_get_intermediates(C.c_void_p(workspace.data_ptr()), C.byref(it))
    if rc not in (GS_OK, GS_ERR_OVERFLOW):
        raise GsError(rc, "gs_get_intermediates")
    out = SimpleNamespace(P=it.P, W=it.W, H=it.H, grid_x=it.grid_x, grid_y=it.grid_y, n_tiles=it.n_tiles,
                          n_visible=int(it.n_visible), n_dup=int(it.n_dup), max_dup=int(it.max_dup), n_coarse=int(it.n_coarse),
                          overflow=rc == GS_ERR_OVERFLOW)
    if rc == GS_ERR_OVERFLOW:
        e = GsError(rc, "gs_get_intermediates")
        e.n_dup = out.n_dup
        raise e
    dev = workspace.device
    if "per_gaussian" in copy:
        pg = _copy_out(it.per_gaussian, 4 * it.P, np.uint32, dev).reshape(it.P, 4)
        out.rect = np.stack([pg[:, 0] & 0xFFFF, pg[:, 0] >> 16, pg[:, 1] & 0xFFFF, pg[:, 1] >> 16], axis=1).astype(np.int32)
        out.depth_bits = pg[:, 2].copy()
        out.radius = pg[:, 3].astype(np.int32)
        out.tiles_touched = ((out.rect[:, 2] - out.rect[:, 0]) * (out.rect[:, 3] - out.rect[:, 1])).astype(np.uint32)
    if "geom" in copy:
        out.record = _copy_out(it.record, 16 * it.P, np.float32, dev).reshape(it.P, 16)
        rc = out.record   # layout: include/gs.h {mu_x, mu_y, b, det | x*, 1/c, c tau, flags | a, c, log2 o, r | g, b, -, -}
        out.geom = np.stack([rc[:, 0], rc[:, 1], rc[:, 8], rc[:, 2], rc[:, 9], rc[:, 10], rc[:, 3], rc[:, 7]], axis=1)  # mu, conic a b c, log2 o, det, flags
        out.colour = np.stack([rc[:, 11], rc[:, 12], rc[:, 13]], axis=1)
    if "depth_sorted" in copy:
        out.depth_sorted = _copy_out(it.depth_sorted, it.n_visible, np.uint64, dev)
        out.dup_offsets = _copy_out(it.dup_offsets, it.n_visible, np.uint32, dev)
    if "tile_ranges" in copy:
        out.tile_ranges = _copy_out(it.tile_ranges, it.n_tiles + 1, np.uint32, dev)
    if "sorted_ids" in copy:
        out.sorted_ids = _copy_out(it.sorted_ids, min(it.n_dup, it.max_dup), np.uint32, dev)
    return out


def gs_set_render_stream(enable: bool) -> None:
    lib().gs_set_render_stream(1 if enable else 0)


def gs_set_timing(enable: bool) -> None:
    lib().gs_set_timing(1 if enable else 0)


def gs_get_timings(workspace) -> dict:
    ms = (C.c_float * GS_N_TIMINGS)()
    rc = lib().gs_get_timings(C.c_void_p(workspace.data_ptr()), ms)
    if rc != GS_OK:
        raise GsError(rc, "gs_get_timings")
    return dict(zip(TIMING_NAMES, [float(x) for x in ms]))


def gs_set_stats(enable: bool) -> None:
    lib().gs_set_stats(1 if enable else 0)


def gs_get_stats(workspace) -> dict:
    out = (C.c_uint64 * GS_N_STATS)()
    rc = lib().gs_get_stats(C.c_void_p(workspace.data_ptr()), out)
    if rc != GS_OK:
        raise GsError(rc, "gs_get_stats")
    return dict(zip(STATS_NAMES, [int(x) for x in out]))


def gs_selftest_atomic_order(iters: int = 50) -> dict:
    out = (C.c_uint64 * 2)()
    rc = lib().gs_selftest_atomic_order(int(iters), out)
    if rc != GS_OK:
        raise GsError(rc, "gs_selftest_atomic_order")
    return {"violations": int(out[0]), "atomics_checked": int(out[1])}


def gs_selftest_issue_peak(iters: int = 2000) -> dict:
    """Measured thread-operations per second of the current device: scalar FFMA, packed FFMA2, MUFU.EX2."""
    out = (C.c_double * 3)()
    rc = lib().gs_selftest_issue_peak(int(iters), out)
    if rc != GS_OK:
        raise GsError(rc, "gs_selftest_issue_peak")
    return {"ffma": float(out[0]), "ffma2": float(out[1]), "ex2": float(out[2])}


def gs_noalloc_max_keys() -> int:
    return int(lib().gs_noalloc_max_keys())


def gs_depth_sort_noalloc(keys_in, keys_out, n: int = None, stream=None) -> None:
    """keys_out[:n] = keys_in[:n] sorted ascending by bits 63..32, stable (include/gs.h).  keys_in / keys_out: distinct
    contiguous int64 CUDA tensors (the 64-bit keys' bit patterns).  Allocates nothing; n <= GS_NOALLOC_MAX_KEYS, else
    GsError(GS_ERR_LIMIT).  All calls share one static device scratch: do not overlap them on the GPU."""
    import torch
    if n is None:
        n = keys_in.numel()
    for t in (keys_in, keys_out):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.int64 and t.numel() >= min(n, GS_NOALLOC_MAX_KEYS)):
            raise ValueError("gs_depth_sort_noalloc: contiguous int64 CUDA tensors of at least n elements expected")
    st = stream if stream is not None else torch.cuda.current_stream(keys_in.device)
    rc = lib().gs_depth_sort_noalloc(C.c_void_p(keys_in.data_ptr()), C.c_void_p(keys_out.data_ptr()), int(n), C.c_void_p(st.cuda_stream))
    if rc != GS_OK:
        raise GsError(rc, "gs_depth_sort_noalloc(n = %d, limit %d)" % (n, GS_NOALLOC_MAX_KEYS))


def gs_set_workspace_option(workspace, option: int, value: int) -> None:
    """Per-workspace switch (include/gs.h): wins over the process-wide setter for calls on this workspace; -1 = follow it."""
    rc = lib().gs_set_workspace_option(C.c_void_p(workspace.data_ptr()), int(option), int(value))
    if rc != GS_OK:
        raise GsError(rc, "gs_set_workspace_option")


def gs_release(workspace) -> None:
    rc = lib().gs_release(C.c_void_p(workspace.data_ptr()))
    if rc != GS_OK:
        raise GsError(rc, "gs_release")


def gs_set_graph(enable: bool) -> None:
    lib().gs_set_graph(1 if enable else 0)


def gs_set_rank_mode(mode: int) -> None:
    rc = lib().gs_set_rank_mode(int(mode))
    if rc != GS_OK:
        raise GsError(rc, "gs_set_rank_mode")


def gs_get_rank_mode() -> int:
    rc = int(lib().gs_get_rank_mode())
    if rc < 0:
        raise GsError(rc, "gs_get_rank_mode")
    return rc


def gs_set_tile_cull(mode: int) -> None:
    rc = lib().gs_set_tile_cull(int(mode))
    if rc != GS_OK:
        raise GsError(rc, "gs_set_tile_cull")


def gs_get_tile_cull() -> int:
    return int(lib().gs_get_tile_cull())


def gs_set_render_variant(variant: int) -> None:
    rc = lib().gs_set_render_variant(int(variant))
    if rc != GS_OK:
        raise GsError(rc, "gs_set_render_variant")


def gs_get_render_variant() -> int:
    return int(lib().gs_get_render_variant())


def gs_last_launch_count() -> int:
    return int(lib().gs_last_launch_count())


def gs_error_string(code: int) -> str:
    return lib().gs_error_string(int(code)).decode()
