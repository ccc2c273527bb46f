"""Parity protocol between the CUDA path (through the C ABI) and the CPU oracle.

1. bit-exact, whole arrays: tiles_touched, radius, rect, depth bits, N_dup, tile counts, tile ranges, sorted id lists;
2. n_contrib equal on every pixel whose oracle `fragile` flag is 0 (an alpha within delta of 1/255 or a T' within delta
   of 1e-4 makes a pixel fragile; delta = 1e-3);
3. image and final_T: |diff| <= 2e-3 on >= 99.9 % of pixels, <= 2/255 on all, and every pixel above 2e-3 is fragile
   (BASELINE.json north_star).
Used by tests/test_gpu_parity.py and __graft_entry__.smoke().  Imports the oracle: test infrastructure only.
"""
from __future__ import annotations

import numpy as np
import torch

from oracle import oracle
from paper_2606_16566_b200 import binding
from paper_2606_16566_b200.renderer import Renderer

TOL_MOST = 2e-3        # north_star: within 2e-3 absolute on >= 99.9 % of pixels
TOL_ALL = 2.0 / 255.0  # and within 2/255 on all pixels
FRAC_MOST = 0.999
DELTA = 1e-3           # fragile-pixel delta of the parity protocol


def run_gpu(scene, cam_index=0, max_dup=None, variant=None, count_contrib=True, device="cuda:0", renderer=None):
    cam = scene.cameras[cam_index]
    if max_dup is None:
        max_dup = 1 << 20
    # the variant is process-wide state of the library: always set it, the product default when none is asked for
    binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT if variant is None else variant)
    r = renderer or Renderer(scene.P, cam.W, cam.H, max_dup, device=device, count_contrib=count_contrib)
    if renderer is None or r.scene is None:
        r.upload(scene)
    r.render(cam)
    torch.cuda.synchronize()
    return r


def run_gpu_auto(scene, cam_index=0, variant=None, count_contrib=True, device="cuda:0", start_dup=1 << 20):
    """Render, growing the workspace when the frame needs more duplicates than it holds (GS_ERR_OVERFLOW)."""
    max_dup = start_dup
    for attempt in range(4):
        r = run_gpu(scene, cam_index, max_dup, variant, count_contrib, device)
        try:
            it = r.intermediates()
            return r, it
        except binding.GsError as e:
            if e.code != binding.GS_ERR_OVERFLOW:
                raise
            assert e.n_dup > max_dup, "overflow reported although the workspace was sized for %d >= %d duplicates" % (max_dup, e.n_dup)
            max_dup = int(e.n_dup * 1.02) + 4096
            del r
            torch.cuda.empty_cache()
    raise AssertionError("workspace still too small after 4 attempts")


def compare(r, it, ref, check_lists=True, check_pixels=True, exact_cull=False):
    """Returns a report dict; raises AssertionError on any violation.  `ref` is an oracle.render() result (possibly a
    tile subset), `r` a Renderer after render(), `it` its intermediates.  exact_cull: both sides ran the exact ellipse-tile
    mode (gs_set_tile_cull(2) / TILE_CULL_EXACT): the tile counts are the exact list lengths, tile_ranges still holds the
    rect-based first slots, and list t is sorted_ids[ranges[t] : ranges[t] + counts[t]]."""
    rep = {}
    # ---- 1. bit-exact integers -----------------------------------------------------------------------------------
    assert it.P == ref.P and it.n_tiles == ref.n_tiles
    for name in ("tiles_touched", "radius", "depth_bits"):
        a, b = getattr(it, name), getattr(ref, name)
        bad = np.flatnonzero(a != b)
        assert bad.size == 0, "%s differs for %d Gaussians, first %s: gpu %s oracle %s" % (
            name, bad.size, bad[:5], a[bad[:5]], b[bad[:5]])
    bad = np.flatnonzero((it.rect != ref.rect).any(axis=1))
    assert bad.size == 0, "rect differs for %d Gaussians, first %s" % (bad.size, bad[:5])
    assert it.n_dup == ref.n_dup, "N_dup gpu %d oracle %d" % (it.n_dup, ref.n_dup)
    assert it.n_visible == int((ref.tiles_touched > 0).sum())
    counts = r.out_tile_counts.cpu().numpy().view(np.uint32)
    assert np.array_equal(counts, ref.tile_counts), "tile counts differ"
    ranges = it.tile_ranges.astype(np.uint64)
    if exact_cull:   # first slots from the rect-based coverage grid; every list fits into its slot range
        assert ranges[0] == 0 and ranges[-1] == it.n_dup and (np.diff(ranges) >= ref.tile_counts.astype(np.uint64)).all(), "tile ranges"
    else:
        assert ranges[0] == 0 and np.array_equal(np.diff(ranges), ref.tile_counts.astype(np.uint64)), "tile ranges differ"
    rep.update(P=int(it.P), n_visible=int(it.n_visible), n_dup=int(it.n_dup))
    if check_lists and exact_cull:
        n_bad = 0
        for l, t in enumerate(ref.list_tile):
            a = it.sorted_ids[int(ranges[t]):int(ranges[t]) + int(counts[t])]
            b = ref.sorted_ids[int(ref.list_offsets[l]):int(ref.list_offsets[l + 1])]
            if not np.array_equal(a, b):
                n_bad += 1
        assert n_bad == 0, "sorted id lists differ in %d of %d tiles" % (n_bad, len(ref.list_tile))
        rep["lists_checked"] = int(len(ref.list_tile))
        rep["list_entries"] = int(counts.sum())
    elif check_lists and ref.full:   # every list: the concatenation IS the sorted id array (ranges already compared)
        assert it.sorted_ids.shape == ref.sorted_ids.shape and np.array_equal(it.sorted_ids, ref.sorted_ids), \
            "sorted id array differs (first at %s)" % (np.flatnonzero(it.sorted_ids != ref.sorted_ids)[:5],)
        rep["lists_checked"] = int(len(ref.list_tile))
    elif check_lists:
        n_bad = 0
        for l, t in enumerate(ref.list_tile):
            a = it.sorted_ids[int(ranges[t]):int(ranges[t + 1])]
            b = ref.sorted_ids[int(ref.list_offsets[l]):int(ref.list_offsets[l + 1])]
            if not np.array_equal(a, b):
                n_bad += 1
        assert n_bad == 0, "sorted id lists differ in %d of %d tiles" % (n_bad, len(ref.list_tile))
        rep["lists_checked"] = int(len(ref.list_tile))
    if not check_pixels:
        return rep
    # ---- pixels of rendered tiles ----------------------------------------------------------------------------------
    H, W, gx = ref.H, ref.W, ref.grid_x
    tmask = ref.rendered.reshape(ref.grid_y, gx).astype(bool)
    pmask = np.repeat(np.repeat(tmask, 16, axis=0), 16, axis=1)[:H, :W]
    img = r.out_rgb.cpu().numpy()
    fT = r.out_final_T.cpu().numpy()
    fragile = ref.fragile != 0
    # ---- 2. contributor counts -------------------------------------------------------------------------------------
    if r.out_n_contrib is not None:
        nc = r.out_n_contrib.cpu().numpy().view(np.uint32)
        diff = (nc != ref.n_contrib) & pmask
        hard = diff & ~fragile
        assert hard.sum() == 0, "n_contrib differs on %d NON-fragile pixels, first %s" % (hard.sum(), np.argwhere(hard)[:5])
        rep["n_contrib_mismatch_fragile"] = int(diff.sum())
    # ---- 3. image and final T --------------------------------------------------------------------------------------
    d_img = np.abs(img - ref.image).max(axis=0)
    d_T = np.abs(fT - ref.final_T)
    d = np.maximum(d_img, d_T)
    d = np.where(pmask, d, 0.0)
    npx = int(pmask.sum())
    over = d > TOL_MOST
    assert not np.isnan(img).any() and not np.isnan(fT).any(), "NaN in the output"
    assert d.max() <= TOL_ALL, "max |diff| %.3g > 2/255 at %s" % (d.max(), np.unravel_index(d.argmax(), d.shape))
    assert over.sum() <= (1.0 - FRAC_MOST) * npx, "%d of %d pixels above 2e-3" % (over.sum(), npx)
    assert (over & ~fragile).sum() == 0, "%d NON-fragile pixels above 2e-3" % (over & ~fragile).sum()
    # the classifier that forgives mismatches must stay near what SURVEY.md 8(c) estimates (~3 % of the pixels at delta = 1e-3; measured 0.6-5.4 %:
    # it grows with the number of Gaussians a pixel traverses, the dense indoor scene being the highest)
    assert (fragile & pmask).sum() <= 0.08 * max(npx, 1) + 8, "fragile share %.3f > 8 %%" % ((fragile & pmask).sum() / max(npx, 1))
    rep.update(pixels=npx, fragile_share=float((fragile & pmask).sum()) / max(npx, 1), max_abs_diff=float(d.max()),
               over_2e3=int(over.sum()), p999_abs_diff=float(np.quantile(d[pmask], 0.999)) if npx else 0.0,
               mean_abs_diff=float(d[pmask].mean()) if npx else 0.0)
    return rep


def oracle_and_compare(scene, cam_index=0, tile_subset=None, n_threads=8, variant=None, count_contrib=True, flags=0, tile_cull=False):
    """tile_cull: both sides in the tighter-rect mode (True / 1: gs_set_tile_cull(1) / oracle flag TILE_CULL; 2: the exact
    ellipse-tile mode gs_set_tile_cull(2) / TILE_CULL_EXACT, which needs a two-level workspace); reset to 0 afterwards."""
    mode = int(tile_cull)
    binding.gs_set_tile_cull(mode)
    try:
        r, it = run_gpu_auto(scene, cam_index, variant=variant, count_contrib=count_contrib, start_dup=(5 << 20) if mode == 2 else (1 << 20))
    finally:
        binding.gs_set_tile_cull(0)
    if mode == 1:
        flags |= oracle.TILE_CULL
    elif mode == 2:
        flags |= oracle.TILE_CULL_EXACT
    ref = oracle.render(scene, cam_index, tile_subset=tile_subset, n_threads=n_threads, flags=flags, fragile_delta=DELTA)
    rep = compare(r, it, ref, check_lists=not (flags & oracle.NO_LISTS),
                  check_pixels=not (flags & (oracle.NO_LISTS | oracle.NO_RENDER)), exact_cull=(mode == 2))
    return rep, r, it, ref
