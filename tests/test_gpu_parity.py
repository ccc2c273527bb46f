"""GPU parity tests: the CUDA path, called through the C ABI (ctypes), against the CPU oracle on the same seeded inputs.

Protocol and tolerances: tests/parity_util.py (BASELINE.json north_star).  Every test needs a B200: `-m gpu`.
"""
import os

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_16566_b200 import binding, scenes
from paper_2606_16566_b200.renderer import Renderer

import parity_util as pu

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _default_variant():
    binding.gs_set_render_variant(4)
    binding.gs_set_tile_cull(0)
    yield
    binding.gs_set_render_variant(4)
    binding.gs_set_tile_cull(0)


# ------------------------------------------------------------------------------------------------------------------
# config 1 (tiny) -- every render variant of the ablation ladder, whole image
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [4, 3, 2, 1, 0])
def test_config1_all_variants(variant):
    sc = scenes.make_scene(1)
    rep, r, it, ref = pu.oracle_and_compare(sc, 0, variant=variant)
    assert rep["n_dup"] == ref.n_dup and rep["lists_checked"] == 64
    print("config1 variant", variant, rep)


# ------------------------------------------------------------------------------------------------------------------
# config 2 (object-centric, the bench workload) -- full size, whole image, several poses
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pose,variant", [(0, 4), (3, 4), (5, 4), (0, 3), (1, 0), (2, 2)])
def test_config2_full(pose, variant):
    sc = scenes.make_scene(2)
    rep, *_ = pu.oracle_and_compare(sc, pose, variant=variant)
    print("config2 pose", pose, "variant", variant, rep)


def test_config2_bench_configuration_without_counts():
    """bench.py renders without the optional n_contrib output: same image bit for bit, parity holds."""
    sc = scenes.make_scene(2)
    r1, it1 = pu.run_gpu_auto(sc, 2, count_contrib=True)
    r2, it2 = pu.run_gpu_auto(sc, 2, count_contrib=False)
    assert torch.equal(r1.out_rgb, r2.out_rgb) and torch.equal(r1.out_final_T, r2.out_final_T)
    ref = oracle.render(sc, 2, n_threads=8, fragile_delta=pu.DELTA)
    print(pu.compare(r2, it2, ref))


# ------------------------------------------------------------------------------------------------------------------
# reduced configs 3-5: same distributions, fewer Gaussians, ragged image sizes (W, H not multiples of 16)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,P,W,H,f,pose", [
    (3, 120_000, 637, 419, 500.0, 0),
    (3, 120_000, 637, 419, 500.0, 7),
    (4, 60_000, 963, 541, 750.0, 0),
    (4, 60_000, 963, 541, 750.0, 5),
    (5, 400_000, 1283, 727, 1000.0, 0),
    (5, 400_000, 1283, 727, 1000.0, 3),
])
def test_reduced_configs(config, P, W, H, f, pose):
    sc = scenes.make_scene(config, P=P, W=W, H=H, f=f)
    rep, *_ = pu.oracle_and_compare(sc, pose)
    print("config", config, "reduced pose", pose, rep)


# ------------------------------------------------------------------------------------------------------------------
# full-size configs 3-5 in the launch configuration bench.py uses: NO sampling of the bit-exact outputs.
#   configs 3 and 5: every per-Gaussian integer, N_dup, every tile count / range, the WHOLE sorted id array and the WHOLE
#     image / final T / n_contrib against the oracle, on two poses each (pose 0 and a mid-orbit pose);
#   config 4 (1.02 G list entries, ~125 000 per tile): every per-Gaussian integer, every tile count / range and the whole
#     4 GB sorted id array on pose 0; pixels on the tiles of the three longest lists, the corners, the centre and random
#     tiles (the oracle blends those one by one); the integers and counts of a second pose.
# ------------------------------------------------------------------------------------------------------------------
_SCENES = {}
N_CPU = os.cpu_count() or 8


def _full_scene(config):
    if config not in _SCENES:
        _SCENES.clear()            # one multi-GB scene at a time
        _SCENES[config] = scenes.make_scene(config)
    return _SCENES[config]


@pytest.mark.parametrize("config,pose", [(3, 0), (3, 9), (5, 0), (5, 5)])
def test_full_size_whole_frame(config, pose):
    sc = _full_scene(config)
    ref = oracle.render(sc, pose, n_threads=N_CPU, fragile_delta=pu.DELTA)
    assert ref.full
    r, it = pu.run_gpu_auto(sc, pose, start_dup=int(ref.n_dup) + 4096)
    rep = pu.compare(r, it, ref)
    assert rep["lists_checked"] == ref.n_tiles and rep["pixels"] == ref.W * ref.H
    print("config", config, "FULL pose", pose, rep)


def test_config4_full_size_every_list_and_sampled_pixels():
    sc = _full_scene(4)
    ref = oracle.render(sc, 0, n_threads=N_CPU, flags=oracle.NO_RENDER)       # every list: 1.02 G entries
    assert ref.full and ref.n_dup > 900_000_000
    r, it = pu.run_gpu_auto(sc, 0, start_dup=int(ref.n_dup) + 4096)
    rep = pu.compare(r, it, ref, check_lists=True, check_pixels=False)
    assert rep["lists_checked"] == ref.n_tiles
    counts, gx, gy = ref.tile_counts.copy(), ref.grid_x, ref.grid_y
    del ref, it
    longest = [int(t) for t in np.argsort(counts)[::-1][:3]]
    fixed = [0, gx - 1, (gy - 1) * gx, gy * gx - 1, (gy // 2) * gx + gx // 2]
    rnd = [int(t) for t in np.random.default_rng(4).choice(gx * gy, size=12, replace=False)]
    tiles = np.array(sorted(set(longest + fixed + rnd)), dtype=np.int32)
    assert all(t in tiles for t in longest) and len(tiles) >= 16
    sub = oracle.render(sc, 0, tile_subset=tiles, n_threads=N_CPU, fragile_delta=pu.DELTA)
    it = r.intermediates()
    rep2 = pu.compare(r, it, sub)
    print("config 4 FULL pose 0: lists", rep, "pixels on", len(tiles), "tiles", rep2)
    del r, it, sub
    torch.cuda.empty_cache()
    rep3, *_ = pu.oracle_and_compare(sc, 9, flags=oracle.NO_LISTS)             # a second pose: integers, N_dup, every tile count
    print("config 4 FULL pose 9:", rep3)


# ------------------------------------------------------------------------------------------------------------------
# closed-form fixtures on the GPU (DESIGN.md pins T1-T3 applied to the CUDA path)
# ------------------------------------------------------------------------------------------------------------------
def test_closed_form_single_gaussian():
    W = H = 33
    sc = scenes.single_gaussian_scene([0.0, 0.0, 4.0], [0.1] * 3, [0.5, -0.5, 0.5, 0.5], 0.7, [0.9, 0.5, 0.1],
                                      [0.2, 0.3, 0.4], W, H, 40.0, 40.0)
    r, it = pu.run_gpu_auto(sc)
    img = r.out_rgb.cpu().numpy()
    fT = r.out_final_T.cpu().numpy()
    sig2 = (40.0 * 0.1 / 4.0) ** 2 + 0.3
    yy, xx = np.mgrid[0:H, 0:W]
    r2 = (xx - 16.0) ** 2 + (yy - 16.0) ** 2
    a = 0.7 * np.exp(-r2 / (2 * sig2))
    a = np.where(a < 1.0 / 255.0, 0.0, np.minimum(a, 0.99))
    inrect = (xx < 32) & (yy < 32)
    a = np.where(inrect, a, 0.0)
    near = np.abs(0.7 * np.exp(-r2 / (2 * sig2)) - 1.0 / 255.0) < 1e-5  # exactly-on-threshold pixels: none here
    assert not near.any()
    for ch, (c, b) in enumerate(zip([0.9, 0.5, 0.1], [0.2, 0.3, 0.4])):
        assert np.abs(img[ch] - (b * (1 - a) + c * a)).max() < 2e-5
    assert np.abs(fT - (1 - a)).max() < 2e-5
    assert it.radius[0] == 4 and list(it.rect[0]) == [0, 0, 2, 2] and it.n_dup == 4


def test_termination_rule_stack():
    """>= 7 identical centred Gaussians, o = 0.8, equal depth: n_contrib = 5, final T = 3.2e-4 at the centre (R1)."""
    W = H = 33
    n = 9
    sc = scenes.single_gaussian_scene([[0.0, 0.0, 4.0]] * n, [0.2] * 3, [1.0, 0.0, 0.0, 0.0], 0.8, [0.3, 0.6, 0.9],
                                      [0.0, 0.0, 0.0], W, H, 40.0, 40.0)
    rep, r, it, ref = pu.oracle_and_compare(sc)
    assert int(r.out_n_contrib[16, 16]) == 5
    assert abs(float(r.out_final_T[16, 16]) - 3.2e-4) < 1e-7


def test_equal_depth_tie_break_and_order_independence():
    W = H = 49
    means = [[0.0, 0.0, 3.0], [0.05, 0.0, 3.0], [0.0, 0.05, 5.0]]
    cols = [[1.0, 0.0, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]]
    sc = scenes.single_gaussian_scene(means, [0.3] * 3, [1.0, 0.0, 0.0, 0.0], [0.6, 0.7, 0.8], cols, [0.1] * 3, W, H, 50.0, 50.0)
    rep, r, it, ref = pu.oracle_and_compare(sc)
    # ids 0 and 1 share their depth bits: 0 comes first in every list
    for t in range(it.n_tiles):
        ids = list(it.sorted_ids[it.tile_ranges[t]:it.tile_ranges[t + 1]])
        if 0 in ids and 1 in ids:
            assert ids.index(0) < ids.index(1)


# ------------------------------------------------------------------------------------------------------------------
# edge cases
# ------------------------------------------------------------------------------------------------------------------
def test_empty_and_all_culled():
    W, H = 70, 45
    bg = np.array([0.25, 0.5, 0.75], np.float32)
    # (a) P = 0
    sc = scenes.make_scene(1, P=0, W=W, H=H)
    sc.bg = bg
    r, it = pu.run_gpu_auto(sc)
    assert it.n_dup == 0 and it.n_visible == 0
    assert torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))
    assert np.array_equal(r.out_rgb.cpu().numpy(), np.broadcast_to(bg[:, None, None], (3, H, W)))
    assert int(r.out_tile_counts.sum()) == 0 and int(r.out_n_contrib.sum()) == 0
    # (b) everything behind the camera
    sc = scenes.make_scene(1, P=500, W=W, H=H)
    sc.means3D[:, 2] = -sc.means3D[:, 2]
    sc.bg = bg
    rep, r, it, ref = pu.oracle_and_compare(sc)
    assert it.n_dup == 0 and torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))


def test_workspace_overflow_is_reported_and_safe():
    sc = scenes.make_scene(1)
    cam = sc.cameras[0]
    r = pu.run_gpu(sc, 0, max_dup=1000)  # the frame needs 5 436 entries
    with pytest.raises(binding.GsError) as ei:
        r.intermediates()
    assert ei.value.code == binding.GS_ERR_OVERFLOW and ei.value.n_dup == oracle.render(sc, flags=oracle.NO_LISTS).n_dup
    assert torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))  # every list treated as empty
    # too small for even max_dup = 0
    small = torch.empty(1024, dtype=torch.uint8, device="cuda:0")
    with pytest.raises(binding.GsError) as ei:
        binding.gs_render(r.scene["means3D"], r.scene["scales"], r.scene["rotations"], r.scene["opacities"], r.scene["sh"], 0,
                          cam.viewmatrix, cam.projmatrix, cam.fx, cam.fy, cam.W, cam.H, sc.bg, r.out_rgb, r.out_final_T,
                          r.out_tile_counts, r.out_n_contrib, small)
    assert ei.value.code == binding.GS_ERR_WORKSPACE
    with pytest.raises(binding.GsError) as ei:
        binding.gs_render(r.scene["means3D"], r.scene["scales"], r.scene["rotations"], r.scene["opacities"], r.scene["sh"], 7,
                          cam.viewmatrix, cam.projmatrix, cam.fx, cam.fy, cam.W, cam.H, sc.bg, r.out_rgb, r.out_final_T,
                          r.out_tile_counts, r.out_n_contrib, r.workspace)
    assert ei.value.code == binding.GS_ERR_BAD_ARG


def test_deterministic_and_reusable_workspace():
    sc = scenes.make_scene(2, P=30_000, W=400, H=300, f=500.0)
    r, it = pu.run_gpu_auto(sc, 0)
    a = (r.out_rgb.clone(), r.out_final_T.clone(), r.out_n_contrib.clone(), it.sorted_ids.copy())
    for pose in (1, 0):
        r.render(sc.cameras[pose])
    torch.cuda.synchronize()
    it2 = r.intermediates()
    assert torch.equal(a[0], r.out_rgb) and torch.equal(a[1], r.out_final_T) and torch.equal(a[2], r.out_n_contrib)
    assert np.array_equal(a[3], it2.sorted_ids)


def test_sh_degrees_and_colour_tolerance():
    """SH degrees 0..3 through the CUDA preprocess: colours within 1e-5 of the oracle's double evaluation."""
    for deg in (0, 1, 2, 3):
        sc = scenes.make_scene(2, P=5_000, W=256, H=192, f=300.0, sh_degree=deg)
        r, it = pu.run_gpu_auto(sc, 1)
        full = r.intermediates(copy=("per_gaussian", "geom", "tile_ranges", "sorted_ids"))
        ref = oracle.render(sc, 1, n_threads=8, fragile_delta=pu.DELTA)
        vis = ref.tiles_touched > 0
        assert np.abs(full.colour[vis, :3] - ref.rgb[vis]).max() < 1e-5
        assert np.array_equal(full.geom[vis, 0:2].view(np.uint32), ref.mu[vis].view(np.uint32))      # mu bit-exact
        assert np.array_equal(full.geom[vis, 2:5].view(np.uint32), ref.conic[vis].view(np.uint32))  # conic bit-exact
        pu.compare(r, it, ref)


def test_per_stage_timings_and_launch_count():
    sc = scenes.make_scene(1)
    binding.gs_set_timing(True)
    try:
        r = pu.run_gpu(sc, 0)
        t = binding.gs_get_timings(r.workspace)
    finally:
        binding.gs_set_timing(False)
    assert set(t) == set(binding.TIMING_NAMES) and all(v >= 0 for v in t.values()) and t["frame"] > 0
    assert binding.gs_last_launch_count() >= 8


def test_shared_atomic_rank_order_selftest():
    """The radix sort ranks keys with one shared-memory atomicAdd each and relies on same-address lanes being served in
    lane order (csrc/binning.cu header); the device self-test checks that property on this GPU."""
    r = binding.gs_selftest_atomic_order(40)
    assert r["atomics_checked"] > 10_000_000
    assert r["violations"] == 0, r


def test_global_coordinate_polynomial_loses_precision_at_4k():
    """PAPER.md Sec. III-B4 / Table V: the expanded polynomial in GLOBAL pixel coordinates loses up to
    4 * 4000^2 * 2^-24 = 3.81 in ln(alpha) at 4K (Eq. 11), the tile-local form 2.4e-4 (Eq. 12).  Variant 6 is variant 3
    with global coordinates and fp32 coefficients; on a 4K frame it must miss the oracle by far more than variant 3,
    which stays inside the parity tolerance."""
    sc = scenes.make_scene(5, P=150_000, poses=1)          # 3840x2160, f = 3000: coordinates up to ~4000
    ref = oracle.render(sc, 0, n_threads=8, fragile_delta=pu.DELTA)
    err = {}
    for variant in (3, 6):
        r, it = pu.run_gpu_auto(sc, 0, variant=variant, start_dup=int(ref.n_dup) + 4096)
        d = np.abs(r.out_rgb.cpu().numpy() - ref.image).max(axis=0)
        err[variant] = (float(d.max()), float((d > pu.TOL_MOST).mean()))
        if variant == 3:
            pu.compare(r, it, ref)                         # the tile-local form is inside the tolerance
    binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT)
    print("max |rgb - oracle|, share of pixels over 2e-3: tile-local %s, global %s" % (err[3], err[6]))
    assert err[3][0] <= pu.TOL_ALL and err[3][1] <= 1e-3
    assert err[6][0] > 10.0 * max(err[3][0], 1e-4) and err[6][0] > pu.TOL_ALL


def test_overlapped_readback_returns_the_same_images():
    """Renderer.render_to_host() double-buffers the device image and copies on a second stream; the host images must be
    the frames a plain render produces, pose by pose."""
    sc = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT)
    r = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
    r.upload(sc)
    n = len(sc.cameras)
    host = [r.render_to_host(cam, i, n) for i, cam in enumerate(sc.cameras)]
    r.synchronize_readback()
    host = [h.clone() for h in host]
    for i, cam in enumerate(sc.cameras):
        r.render(cam, count_contrib=False)
        torch.cuda.synchronize()
        assert torch.equal(host[i], r.out_rgb.cpu()), "pose %d" % i
    assert not torch.equal(host[0], host[1])


@pytest.mark.parametrize("lanes", [1, 2, 3])
def test_render_batch_frames_in_flight_equal_plain_renders(lanes):
    """Renderer.render_batch() keeps several frames in flight, each on its own stream and workspace; every image (written
    to a caller tensor, and copied to host memory on the copy stream) must be bit-identical to the frame a plain
    render() of the same pose produces, and so must the tile counts of the last frame of every lane."""
    sc = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT)
    r = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
    r.upload(sc)
    cams = list(sc.cameras)
    n = len(cams)
    dev_imgs = torch.empty((n, 3, 240, 320), dtype=torch.float32, device="cuda:0")
    for rep in range(2):                                   # the second batch reuses lanes, events and host slots
        host = r.render_batch(cams, lanes=lanes, out_rgb=dev_imgs, to_host=True)
        torch.cuda.current_stream().synchronize()
        host = host.clone()
        host2 = r.render_batch(cams, lanes=lanes, to_host=True)   # images left in the lanes' own buffers
        torch.cuda.current_stream().synchronize()
        assert torch.equal(host, host2.clone())
    plain = torch.empty_like(dev_imgs)                     # no host copy: with one lane this is the plain-stream path
    r.render_batch(cams, lanes=lanes, out_rgb=plain)
    torch.cuda.current_stream().synchronize()
    assert torch.equal(plain, dev_imgs)
    r.render_batch(cams, lanes=lanes, to_host=True)        # leaves the last frame of every lane in the lane's buffers
    torch.cuda.current_stream().synchronize()
    lane_counts = [r._lanes[k]["out_tile_counts"].clone() for k in range(min(lanes, n))]
    for i, cam in enumerate(cams):
        r.render(cam, count_contrib=False)
        torch.cuda.synchronize()
        assert torch.equal(host[i], r.out_rgb.cpu()), "pose %d (host copy)" % i
        assert torch.equal(dev_imgs[i], r.out_rgb), "pose %d (device tensor)" % i
        if i >= n - min(lanes, n):
            assert torch.equal(lane_counts[i % lanes], r.out_tile_counts), "pose %d (tile counts)" % i
    assert not torch.equal(host[0], host[1])


@pytest.mark.parametrize("config,P,W,H,f", [(3, 120_000, 637, 419, 500.0), (5, 1_100_000, 1283, 727, 1000.0)])
def test_one_level_and_two_level_binning_give_the_same_frame(config, P, W, H, f):
    """The binning strategy follows the workspace CAPACITY (<= 4 M entries: one radix sort over tile ids; above: sort
    over 8x8-tile super-tiles + expand_kernel) and the preprocess kernel follows P (below 2^20: no compaction; above:
    two-phase with compaction).  The frame may depend on neither: every integer output, the sorted lists and the
    images must be bit-identical between a small and a large workspace, for a small and a large scene."""
    sc = scenes.make_scene(config, P=P, W=W, H=H, f=f)
    res = []
    for cap in (3 << 20, 9 << 20):
        r = pu.run_gpu(sc, 1, max_dup=cap, count_contrib=True)
        it = r.intermediates(copy=("per_gaussian", "tile_ranges", "sorted_ids"))
        assert it.n_dup <= 3 << 20, "pick a smaller scene: the one-level workspace must hold the frame"
        assert (it.n_coarse > 0) == (cap > 4 << 20)
        res.append((r, it))
    (r1, i1), (r2, i2) = res
    assert i1.n_dup == i2.n_dup and i1.n_visible == i2.n_visible
    assert np.array_equal(i1.rect, i2.rect) and np.array_equal(i1.depth_bits, i2.depth_bits)
    assert np.array_equal(i1.tile_ranges, i2.tile_ranges)
    assert np.array_equal(i1.sorted_ids, i2.sorted_ids)
    assert torch.equal(r1.out_tile_counts, r2.out_tile_counts)
    assert torch.equal(r1.out_rgb, r2.out_rgb) and torch.equal(r1.out_final_T, r2.out_final_T)
    assert torch.equal(r1.out_n_contrib, r2.out_n_contrib)
    ref = oracle.render(sc, 1, n_threads=8, fragile_delta=pu.DELTA)
    print(pu.compare(r2, i2, ref))


@pytest.mark.parametrize("cap", [8000, (256 << 10), (256 << 10) + 1, (4 << 20), (4 << 20) + 1, 6_000_000])
def test_capacity_recovered_from_the_workspace_size_is_never_below_the_one_asked_for(cap):
    """gs_render recovers max_dup from workspace_bytes; the layout changes regime at 256 Ki (radix tile size) and 4 Mi
    entries (binning levels), where its size is not monotone.  A workspace sized by gs_workspace_bytes(.., cap) must give
    back at least `cap`, and the frame must be the same on both sides of every edge."""
    sc = scenes.make_scene(1)
    r = pu.run_gpu(sc, 0, max_dup=cap, count_contrib=True)
    it = r.intermediates(copy=("tile_ranges", "sorted_ids"))
    assert it.max_dup >= cap, (it.max_dup, cap)
    ref = pu.run_gpu(sc, 0, max_dup=1 << 20, count_contrib=True)
    it0 = ref.intermediates(copy=("tile_ranges", "sorted_ids"))
    assert np.array_equal(it.sorted_ids, it0.sorted_ids) and np.array_equal(it.tile_ranges, it0.tile_ranges)
    assert torch.equal(r.out_rgb, ref.out_rgb) and torch.equal(r.out_n_contrib, ref.out_n_contrib)


def test_two_level_binning_edge_cases():
    """The large-capacity path (two-level binning) on the degenerate frames: nothing visible, an overflowing frame
    (every list left empty, the need reported, the workspace reusable afterwards), and a one-tile-wide image whose
    super-tile grid is a single partial cell."""
    cap = 5 << 20                                               # > 4 Mi entries: two levels
    bg = np.array([0.25, 0.5, 0.75], np.float32)
    # (a) everything behind the camera
    sc = scenes.make_scene(1, P=500, W=70, H=45)
    sc.means3D[:, 2] = -sc.means3D[:, 2]
    sc.bg = bg
    r = pu.run_gpu(sc, 0, max_dup=cap)
    it = r.intermediates()
    assert it.n_dup == 0 and it.n_coarse == 0 and int(r.out_tile_counts.sum()) == 0
    assert torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))
    assert np.array_equal(r.out_rgb.cpu().numpy(), np.broadcast_to(bg[:, None, None], (3, 45, 70)))
    # (b) overflow above the two-level threshold: config 3's distribution, ~6.7 M entries into 5 Mi... then enough room
    sc = scenes.make_scene(3, P=500_000, W=1264, H=832)
    need = int(oracle.render(sc, 0, flags=oracle.NO_LISTS).n_dup)
    assert need > cap, need
    r = pu.run_gpu(sc, 0, max_dup=cap)
    with pytest.raises(binding.GsError) as ei:
        r.intermediates()
    assert ei.value.code == binding.GS_ERR_OVERFLOW and ei.value.n_dup == need
    assert torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))
    del r
    torch.cuda.empty_cache()
    rep, *_ = pu.oracle_and_compare(sc, 0)                      # grows the workspace from the reported need
    print(rep)
    # (c) a 16 x 200 image: one tile column, super-tile grid 1 x 2 with partial cells
    sc = scenes.make_scene(1, P=2000, W=16, H=200, f=100.0)
    r = pu.run_gpu(sc, 0, max_dup=cap)
    it = r.intermediates()
    ref = oracle.render(sc, 0, n_threads=4, fragile_delta=pu.DELTA)
    assert it.n_coarse > 0
    print(pu.compare(r, it, ref))


def _same_frame(sc, caps=(3 << 20, 5 << 20)):
    """Renders sc with a one-level and a two-level workspace; every list, range and pixel must be identical."""
    res = []
    for cap in caps:
        r = pu.run_gpu(sc, 0, max_dup=cap, count_contrib=True)
        it = r.intermediates(copy=("per_gaussian", "tile_ranges", "sorted_ids"))
        assert it.n_dup <= caps[0]
        assert (it.n_coarse > 0) == (cap > 4 << 20)
        res.append((r, it))
    (r1, i1), (r2, i2) = res
    assert i1.n_dup == i2.n_dup
    assert np.array_equal(i1.tile_ranges, i2.tile_ranges) and np.array_equal(i1.sorted_ids, i2.sorted_ids)
    assert torch.equal(r1.out_rgb, r2.out_rgb) and torch.equal(r1.out_n_contrib, r2.out_n_contrib)
    return r2, i2


def test_expand_kernel_chunk_and_piece_edges():
    """expand_kernel cuts the sorted super-tile entries into chunks of 2 048, whatever super-tiles they belong to, and chains
    the chunks of one super-tile by look-back.  Adversarial list shapes, each against the one-level sort of the same frame:
    (a) every super-tile list exactly one chunk long (piece boundaries ON chunk boundaries), (b) lists of 5 000 (boundaries inside
    chunks, a chunk holding the tail of one list and the head of the next), (c) ONE super-tile list of 40 000 entries (20 chunks
    chained by look-back), (d) 64 super-tiles of ~50 entries each (dozens of pieces per chunk)."""
    rng = np.random.default_rng(5)

    def blanket(P, W, H):   # P faint Gaussians that each cover the whole W x H image, distinct depths
        z = rng.uniform(3.0, 6.0, P)
        means = np.stack([rng.uniform(-0.2, 0.2, P), rng.uniform(-0.2, 0.2, P), z], 1)
        return scenes.single_gaussian_scene(means, [40.0, 40.0, 40.0], [1, 0, 0, 0], 0.004, rng.uniform(0, 1, (P, 3)), [0.1, 0.2, 0.3],
                                            W, H, 100.0, 100.0)
    # (a) 256 x 256 = 2 x 2 super-tiles, 2 048 entries each
    r, it = _same_frame(blanket(2048, 256, 256))
    assert it.n_coarse == 4 * 2048 and it.n_dup == 2048 * 256
    # (b) 5 000 entries per super-tile list: 20 000 entries, 10 chunks, every piece boundary inside a chunk
    r, it = _same_frame(blanket(5000, 256, 256))
    assert it.n_coarse == 4 * 5000
    # (c) one super-tile (128 x 128), 40 000 entries: 20 chunks of one list
    r, it = _same_frame(blanket(40_000, 128, 128))
    assert it.n_coarse == 40_000 and it.n_dup == 40_000 * 64
    # (d) many short lists: 1 024 x 1 024 = 8 x 8 super-tiles, 3 000 small Gaussians; also against the oracle
    sc = scenes.make_scene(1, P=3000, W=1024, H=1024, f=800.0)
    r, it = _same_frame(sc)
    assert 0 < it.n_coarse < 2 * 2048 * 4
    ref = oracle.render(sc, 0, n_threads=8, fragile_delta=pu.DELTA)
    print(pu.compare(r, it, ref))


def test_two_level_workspace_reused_across_frames_of_different_size():
    """On two-level frames the look-back status words of the tile passes and of expand_kernel are not part of the per-frame
    memset: duplicate_kernel clears the words THIS frame's entry count needs.  One workspace, a sequence of frames whose
    sorted level grows and shrinks (a pulled-back pose with 1.5x the entries between the scene's own poses): every frame must
    equal the frame a fresh renderer produces -- a stale status word read as "published" would corrupt the sort or the offsets."""
    sc = scenes.make_scene(3, P=200_000, W=1264, H=832, poses=4)
    cams = list(sc.cameras)
    V = np.array(cams[0].viewmatrix, dtype=np.float64, copy=True)   # the same camera pulled back: more of the scene in view
    V[2, 3] += 30.0
    far = scenes.make_camera(V, cams[0].fx, cams[0].fy, cams[0].W, cams[0].H)
    seq = [cams[0], far, cams[1], far, cams[2], cams[0]]
    cap = 12 << 20
    want = {}
    for cam in seq:
        if id(cam) in want:
            continue
        r0 = Renderer(sc.P, cam.W, cam.H, cap, device="cuda:0", count_contrib=True)
        r0.upload(sc)
        r0.render(cam)
        torch.cuda.synchronize()
        it = r0.intermediates(copy=("tile_ranges", "sorted_ids"))
        assert it.n_coarse > 0
        want[id(cam)] = (it.n_coarse, it.tile_ranges.copy(), it.sorted_ids[: it.n_dup].copy(), r0.out_rgb.clone())
        del r0
    sizes = [want[id(c)][0] for c in seq]
    assert min(sizes) * 1.5 < max(sizes), sizes               # the sequence really grows and shrinks (radix tiles: 4 096 entries)
    r = Renderer(sc.P, cams[0].W, cams[0].H, cap, device="cuda:0", count_contrib=True)
    r.upload(sc)
    for cam in seq:
        r.render(cam)
        torch.cuda.synchronize()
        it = r.intermediates(copy=("tile_ranges", "sorted_ids"))
        n_coarse, ranges, ids, rgb = want[id(cam)]
        assert it.n_coarse == n_coarse
        assert np.array_equal(it.tile_ranges, ranges) and np.array_equal(it.sorted_ids[: it.n_dup], ids)
        assert torch.equal(r.out_rgb, rgb)


def test_overlapped_scene_upload_switches_buffer_sets_safely():
    """Renderer.upload_async() fills a second set of scene buffers on an upload stream while frames are rendered from the
    active one; activate_uploaded() switches.  Alternating two DIFFERENT scenes of the same size through it must give, for
    each, exactly the frames a fresh renderer produces -- a copy that overtook the frames still reading its target set,
    or a frame that started before its upload finished, would show up as a mismatch."""
    sa = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    sb = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    sb.means3D = (sb.means3D[::-1] * np.float32(0.9)).copy()       # a different scene with the same shapes
    binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT)
    want = []
    for sc in (sa, sb):
        r0 = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
        r0.upload(sc)
        host = r0.render_batch(list(sc.cameras), lanes=1, to_host=True)
        torch.cuda.synchronize()
        want.append(host.clone())
    assert not torch.equal(want[0], want[1])
    for pin in (False, True):                                       # numpy scenes (staged by the Renderer) / pre-pinned tensors
        src = [Renderer.pin_scene(x) for x in (sa, sb)] if pin else [sa, sb]
        r = Renderer(sa.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
        got = []
        r.upload_async(src[0])
        for k in range(6):
            r.activate_uploaded()
            r.upload_async(src[(k + 1) & 1])                        # overlaps the frames of this step
            host = r.render_batch(list(sa.cameras), lanes=3, to_host=True)
            torch.cuda.current_stream().synchronize()
            got.append(host.clone())
        for k in range(6):
            assert torch.equal(got[k], want[k & 1]), "step %d (pinned inputs: %s)" % (k, pin)


def test_upload_restages_the_scene_on_every_call():
    """Renderer.upload() must copy the scene it is GIVEN on every call (round-1 advisor finding: it re-sent the first
    scene's staging), and follow its background colour and SH degree."""
    sa = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    sb = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    sb.means3D = (sb.means3D[::-1] * np.float32(0.9)).copy()
    sb.bg = np.array([0.1, 0.7, 0.3], np.float32)
    want = []
    for sc in (sa, sb):
        r0 = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
        r0.upload(sc)
        r0.render(sc.cameras[1], count_contrib=False)
        torch.cuda.synchronize()
        want.append(r0.out_rgb.clone())
    assert not torch.equal(want[0], want[1])
    r = Renderer(sa.P, 320, 240, 1 << 20, device="cuda:0", count_contrib=False)
    for k in range(4):
        sc = (sa, sb)[k & 1]
        r.upload(sc)
        r.render(sc.cameras[1], count_contrib=False)
        torch.cuda.synchronize()
        assert torch.equal(r.out_rgb, want[k & 1]), "call %d" % k
    with pytest.raises(ValueError):
        r.upload(scenes.make_scene(2, P=10_000, W=320, H=240, f=400.0))


# ------------------------------------------------------------------------------------------------------------------
# tighter tile culling (gs_set_tile_cull(1) / oracle flag TILE_CULL): rects, N_dup, counts, ranges and
# the sorted lists bit-exact against the oracle in the same mode; the image identical to the standard mode's
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,kw,pose", [
    (1, {}, 0), (2, {}, 0), (2, {}, 5),
    (3, dict(P=120_000, W=637, H=419, f=500.0), 7), (4, dict(P=60_000, W=963, H=541, f=750.0), 5),
    (5, dict(P=400_000, W=1283, H=727, f=1000.0), 3)])
def test_tile_cull_mode_matches_the_oracle_in_the_same_mode(config, kw, pose):
    sc = scenes.make_scene(config, **kw)
    rep, r, it, ref = pu.oracle_and_compare(sc, pose, tile_cull=True)
    std = oracle.render(sc, pose, flags=oracle.NO_LISTS)
    assert ref.n_dup < std.n_dup
    print("config", config, "tile cull: N_dup %d -> %d (%.2f)" % (std.n_dup, ref.n_dup, ref.n_dup / std.n_dup), rep)


@pytest.mark.parametrize("config,pose", [(3, 4), (5, 2)])
def test_tile_cull_mode_full_size(config, pose):
    sc = _full_scene(config)
    binding.gs_set_tile_cull(1)
    ref = oracle.render(sc, pose, n_threads=N_CPU, fragile_delta=pu.DELTA, flags=oracle.TILE_CULL)
    r, it = pu.run_gpu_auto(sc, pose, start_dup=int(ref.n_dup) + 4096)
    binding.gs_set_tile_cull(0)
    rep = pu.compare(r, it, ref)
    print("config", config, "FULL, tile cull, pose", pose, rep)


def test_tile_cull_mode_leaves_the_image_unchanged():
    """No pixel outside the tighter rect can be blended (alpha < 1/255 there), so the entries it removes contributed
    exactly nothing: same contributor counts, and the same image and final T up to the rounding of the kernel's stop
    repair (two entries are blended per iteration and a stopping pixel takes its pair back: which entries share a pair
    changes with the list), from 30 % fewer list entries.  (In the oracle the two modes are bit-identical.)"""
    sc = scenes.make_scene(2)
    out = []
    for mode in (0, 1):
        binding.gs_set_tile_cull(mode)
        r, it = pu.run_gpu_auto(sc, 3)
        out.append((r.out_rgb.clone(), r.out_final_T.clone(), r.out_n_contrib.clone(), it.n_dup))
    binding.gs_set_tile_cull(0)
    assert out[1][3] < 0.8 * out[0][3]
    assert torch.equal(out[0][2], out[1][2])
    assert float((out[0][0] - out[1][0]).abs().max()) < 2e-6 and float((out[0][1] - out[1][1]).abs().max()) < 2e-6
    with pytest.raises(binding.GsError):
        binding.gs_set_tile_cull(3)


# exact ellipse-tile culling (gs_set_tile_cull(2) / oracle flag TILE_CULL_EXACT): the per-Gaussian integers and
# N_dup are those of mode 1; the tile counts are the exact list lengths; every list equals the oracle's; image within tolerance
@pytest.mark.parametrize("config,kw,pose", [
    (2, dict(P=30_000, W=480, H=360, f=500.0), 1), (3, dict(P=60_000, W=640, H=416, f=500.0), 2),
    (4, dict(P=20_000, W=480, H=270, f=375.0), 0), (5, dict(P=200_000, W=960, H=540, f=750.0), 3)])
def test_exact_tile_cull_mode_matches_the_oracle_in_the_same_mode(config, kw, pose):
    sc = scenes.make_scene(config, **kw)
    rep, r, it, ref = pu.oracle_and_compare(sc, pose, tile_cull=2)
    assert it.n_coarse > 0
    print("config", config, "exact tile cull", rep, "entries / N_dup %.2f" % (rep["list_entries"] / max(rep["n_dup"], 1)))


@pytest.mark.parametrize("config,pose", [(2, 1), (3, 4), (5, 2)])
def test_exact_tile_cull_mode_full_size(config, pose):
    sc = _full_scene(config)
    binding.gs_set_tile_cull(2)
    ref = oracle.render(sc, pose, n_threads=N_CPU, fragile_delta=pu.DELTA, flags=oracle.TILE_CULL_EXACT)
    r, it = pu.run_gpu_auto(sc, pose, start_dup=max(int(ref.n_dup) + 4096, 5 << 20))
    binding.gs_set_tile_cull(0)
    rep = pu.compare(r, it, ref, exact_cull=True)
    print("config", config, "FULL, exact tile cull, pose", pose, rep)


def test_exact_tile_cull_needs_a_two_level_workspace_and_the_b200_kernel():
    sc = scenes.make_scene(1)
    binding.gs_set_tile_cull(2)
    try:
        with pytest.raises(binding.GsError) as ei:                # capacity <= 4 Mi entries: one-level binning has no expansion stage
            pu.run_gpu(sc, 0, max_dup=1 << 20)
        assert ei.value.code == binding.GS_ERR_WORKSPACE
        with pytest.raises(binding.GsError) as ei:                # the ladder variants walk tile_ranges
            pu.run_gpu(sc, 0, max_dup=5 << 20, variant=3)
        assert ei.value.code == binding.GS_ERR_BAD_ARG
        rep, r, it, ref = pu.oracle_and_compare(sc, 0, tile_cull=2)   # and with both it works on the smallest scene too
        print(rep)
    finally:
        binding.gs_set_tile_cull(0)
        binding.gs_set_render_variant(binding.GS_DEFAULT_RENDER_VARIANT)


def test_exact_tile_cull_overflow_batch_and_per_workspace_switch():
    """Edge cases of gs_set_tile_cull(2): (a) an overflowing frame -- expand_kernel does nothing, no list length is published
    -- must come out as background with the need reported, and the same workspace must render correctly afterwards when it
    is large enough; (b) the mode as a PER-WORKSPACE switch next to a renderer in the standard mode, through render_batch
    with several frames in flight: same images as single renders, the other renderer untouched."""
    bg = np.array([0.25, 0.5, 0.75], np.float32)
    sc = scenes.make_scene(3, P=1_000_000, W=1264, H=832)
    sc.bg = bg
    need = int(oracle.render(sc, 0, flags=oracle.NO_LISTS | oracle.TILE_CULL).n_dup)
    cap = 5 << 20
    assert need > cap, need
    binding.gs_set_tile_cull(2)
    try:
        r = pu.run_gpu(sc, 0, max_dup=cap)
        with pytest.raises(binding.GsError) as ei:
            r.intermediates()
        assert ei.value.code == binding.GS_ERR_OVERFLOW and ei.value.n_dup == need
        assert torch.equal(r.out_final_T, torch.ones_like(r.out_final_T))
        assert np.array_equal(r.out_rgb.cpu().numpy(), np.broadcast_to(bg[:, None, None], (3, 832, 1264)))
        del r
        torch.cuda.empty_cache()
    finally:
        binding.gs_set_tile_cull(0)
    rep, *_ = pu.oracle_and_compare(sc, 0, tile_cull=2)             # grows the workspace from the reported need
    print(rep)
    # (b)
    sc = scenes.make_scene(5, P=150_000, W=960, H=540, f=750.0, poses=4)
    cams = list(sc.cameras)
    ra = Renderer(sc.P, 960, 540, 6 << 20, device="cuda:0", count_contrib=False)
    rb = Renderer(sc.P, 960, 540, 6 << 20, device="cuda:0", count_contrib=False)
    ra.upload(sc); rb.upload(sc)
    ra.set_option(binding.GS_OPT_TILE_CULL, 2)                   # every workspace of ra, the lanes of render_batch included
    singles_a, singles_b, lens = [], [], []
    for cam in cams:
        ra.render(cam); rb.render(cam)
        torch.cuda.synchronize()
        singles_a.append(ra.out_rgb.clone()); singles_b.append(rb.out_rgb.clone())
        lens.append((int(ra.out_tile_counts.sum()), int(rb.out_tile_counts.sum())))
    assert all(a < 0.8 * b for a, b in lens), lens              # a's lists are the exact ones, b's the standard ones
    host_a = ra.render_batch(cams, lanes=3, to_host=True)
    host_b = rb.render_batch(cams, lanes=3, to_host=True)
    torch.cuda.synchronize()
    for k in range(len(cams)):
        assert torch.equal(host_a[k], singles_a[k].cpu()) and torch.equal(host_b[k], singles_b[k].cpu())
        assert float((singles_a[k] - singles_b[k]).abs().max()) < 2e-6   # same image up to the rounding of the stop repair
    assert binding.gs_get_tile_cull() == 0


# ------------------------------------------------------------------------------------------------------------------
# boundary: ranking fallback, per-workspace switches, release
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,kw,pose", [(1, {}, 0), (2, {}, 2), (5, dict(P=1_100_000, W=1283, H=727, f=1000.0), 1)])
def test_ballot_ranking_fallback_gives_the_same_lists(config, kw, pose):
    """gs_set_rank_mode(1): the radix passes rank with ballots (documented semantics only) instead of the shared-memory
    atomic whose lane order is a hardware property; every list must stay bit-exact (one-level and two-level binning)."""
    assert binding.gs_get_rank_mode() == 0          # the self-test found the atomic ranking stable on this device
    sc = scenes.make_scene(config, **kw)
    binding.gs_set_rank_mode(1)
    try:
        assert binding.gs_get_rank_mode() == 1
        rep, r, it, ref = pu.oracle_and_compare(sc, pose)
        if config == 5:
            r2 = pu.run_gpu(sc, pose, max_dup=9 << 20)       # two-level binning
            it2 = r2.intermediates()
            assert it2.n_coarse > 0 and np.array_equal(it2.sorted_ids, it.sorted_ids)
    finally:
        binding.gs_set_rank_mode(-1)
    print("ballot ranking, config", config, rep)


def test_workspace_options_are_per_workspace_and_release_forgets_the_workspace():
    sc = scenes.make_scene(2, P=20_000, W=320, H=240, f=400.0)
    ra = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0")
    rb = Renderer(sc.P, 320, 240, 1 << 20, device="cuda:0")
    ra.upload(sc); rb.upload(sc)
    binding.gs_set_workspace_option(ra.workspace, binding.GS_OPT_TILE_CULL, 1)       # only renderer a
    binding.gs_set_workspace_option(rb.workspace, binding.GS_OPT_STATS, 1)           # only renderer b
    ra.render(sc.cameras[0]); rb.render(sc.cameras[0])
    torch.cuda.synchronize()
    ia, ib = ra.intermediates(copy=()), rb.intermediates(copy=())
    assert ia.n_dup < ib.n_dup and ib.n_dup == oracle.render(sc, 0, flags=oracle.NO_LISTS).n_dup
    assert binding.gs_get_stats(rb.workspace)["pairs_evaluated"] > 0 and binding.gs_get_stats(ra.workspace)["pairs_evaluated"] == 0
    assert binding.gs_get_tile_cull() == 0                                           # the process-wide switch never moved
    binding.gs_set_workspace_option(ra.workspace, binding.GS_OPT_TILE_CULL, -1)      # back to the process-wide value
    ra.render(sc.cameras[0])
    assert ra.intermediates(copy=()).n_dup == ib.n_dup
    assert torch.equal(ra.out_rgb, rb.out_rgb)
    binding.gs_release(ra.workspace)
    with pytest.raises(binding.GsError):
        ra.intermediates(copy=())                                                    # nothing is kept for a released workspace
    ra.render(sc.cameras[1])                                                         # and it can simply be used again
    rb.render(sc.cameras[1])
    assert torch.equal(ra.out_rgb, rb.out_rgb)
    ra.close(); rb.close()


def test_graph_replay_gives_the_same_frames_as_plain_launches():
    """gs_set_graph / GS_OPT_GRAPH: the launch sequence is captured once and replayed with the camera and the caller's
    pointers patched into three kernel nodes.  Poses, output tensors, the optional n_contrib output (another kernel: the
    graph is re-captured) and the tile-cull switch change between calls; every frame must equal the plain-launch frame."""
    sc = scenes.make_scene(2, P=30_000, W=400, H=300, f=500.0)
    rg = Renderer(sc.P, 400, 300, 1 << 20, device="cuda:0", graph=True)
    rp = Renderer(sc.P, 400, 300, 1 << 20, device="cuda:0", graph=False)
    rg.upload(sc); rp.upload(sc)
    other = torch.empty_like(rg.out_rgb)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):                      # a capturable stream (the legacy default stream falls back to plain launches)
        for k, pose in enumerate([0, 3, 3, 5, 1, 0, 7, 2]):
            cc = k not in (3, 4)
            cull = 1 if k in (5, 6) else 0
            binding.gs_set_workspace_option(rg.workspace, binding.GS_OPT_TILE_CULL, cull)
            binding.gs_set_workspace_option(rp.workspace, binding.GS_OPT_TILE_CULL, cull)
            out = other if k % 2 else None
            rg.render(sc.cameras[pose], count_contrib=cc, out_rgb=out)
            rp.render(sc.cameras[pose], count_contrib=cc)
            st.synchronize()
            img = other if k % 2 else rg.out_rgb
            assert torch.equal(img, rp.out_rgb), "frame %d" % k
            assert torch.equal(rg.out_final_T, rp.out_final_T) and torch.equal(rg.out_tile_counts, rp.out_tile_counts)
            if cc:
                assert torch.equal(rg.out_n_contrib, rp.out_n_contrib)
            ig, ip = rg.intermediates(), rp.intermediates()
            assert ig.n_dup == ip.n_dup and np.array_equal(ig.sorted_ids, ip.sorted_ids)
        # batches: several workspaces, render streams, per-frame output tensors
        cams = list(sc.cameras)
        a = torch.empty((len(cams), 3, 300, 400), device="cuda:0")
        b = torch.empty_like(a)
        for rep in range(2):
            rg.render_batch(cams, lanes=3, out_rgb=a)
            rp.render_batch(cams, lanes=3, out_rgb=b)
            st.synchronize()
            assert torch.equal(a, b)
    rep, *_ = pu.oracle_and_compare(sc, 4)           # and the oracle agrees with the plain path as everywhere else
    rg.close(); rp.close()


def test_bounds_checked_build_runs_clean():
    """libgs_dbg.so = the same sources with -DGS_DEBUG_BOUNDS: every index into the workspace and the output arrays is
    checked on the device and a violation traps (the stand-in for compute-sanitizer, closed on this pool).  Configs 1 and 2 at
    full size, a two-level frame, both tile-cull modes, the ballot ranking and the allocation-free depth sort run through it in a
    fresh process and must still agree with the oracle."""
    import subprocess
    import sys
    code = r'''
import sys
sys.path.insert(0, "tests")
import parity_util as pu
from paper_2606_16566_b200 import binding, build, scenes
assert binding.lib()._name == build.LIB_DBG, binding.lib()._name
print(pu.oracle_and_compare(scenes.make_scene(1), 0)[0])
sc = scenes.make_scene(2)
print(pu.oracle_and_compare(sc, 0)[0])
print(pu.oracle_and_compare(sc, 4, tile_cull=True)[0])
binding.gs_set_rank_mode(1)
print(pu.oracle_and_compare(sc, 6)[0])
binding.gs_set_rank_mode(-1)
sc = scenes.make_scene(3, P=300_000)
r = pu.run_gpu(sc, 2, max_dup=9 << 20)
it = r.intermediates()
assert it.n_coarse > 0
from oracle import oracle
print(pu.compare(r, it, oracle.render(sc, 2, n_threads=8, fragile_delta=pu.DELTA)))
print(pu.oracle_and_compare(sc, 5, tile_cull=2)[0])          # exact ellipse-tile mode (expand_kernel<.., true>)
import numpy as np, torch
keys = torch.from_numpy(np.random.default_rng(3).integers(0, 1 << 62, 100_000, dtype=np.int64)).cuda()
out = torch.empty_like(keys)
binding.gs_depth_sort_noalloc(keys, out)                       # the allocation-free depth sort on its static scratch
torch.cuda.synchronize()
hi = keys.cpu().numpy().view(np.uint64) >> np.uint64(32)
assert np.array_equal(out.cpu().numpy().view(np.uint64), keys.cpu().numpy().view(np.uint64)[np.argsort(hi, kind="stable")])
print("BOUNDS OK")
'''
    env = dict(os.environ, GS_DEBUG_BOUNDS="1")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=1200)
    assert res.returncode == 0 and "BOUNDS OK" in res.stdout, res.stdout[-2000:] + res.stderr[-3000:]
