/* gs.h -- C ABI of the B200-native forward 3D Gaussian Splatting tile rasterizer (libgs.so).
 *
 * What it computes: the forward 3DGS render pipeline of PAPER.md:51-53 (Fig. 2: preprocess -> duplication +
 * sort -> render) with the render kernel of Local-GS (Sec. III: tile-local hoisting Eq. 1-10, warp-level
 * culling Eq. 13-21, warp-coherent blending Eq. 22 / Alg. 1).  Everything the paper leaves open (near plane,
 * dilation, rect rounding, SH convention, termination rule ...) follows the readings listed in DESIGN.md.
 *
 * Conventions
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors); "host" pointers are
 *     ordinary host memory read during the call.  The library never allocates or frees caller-visible memory and
 *     keeps no reference to any pointer after the call returns, except that gs_get_intermediates() returns
 *     pointers INTO the caller's workspace.
 *   - Matrices are 16 floats, row-major, column-vector convention (p_cam = V * [p;1]).
 *   - All work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default stream); the tile-grid
 *     kernels run on a library-owned side stream, forked from and joined back into `cuda_stream` with events.
 *     gs_render() returns after enqueueing; it performs NO host synchronisation unless timing is enabled.
 *   - Return value: 0 (GS_OK) or a negative error code; nothing is printed, thrown or exit()ed.
 *   - Not thread-safe per workspace; distinct workspaces on distinct streams may be used concurrently (per-workspace
 *     switches: gs_set_workspace_option).  The workspace must live on the CURRENT device (GS_ERR_BAD_ARG otherwise); the
 *     first call on a device runs a short synchronous self-test (gs_set_rank_mode).  gs_release() frees what the library
 *     keeps per workspace address.
 */
#ifndef GS_H
#define GS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define GS_OK 0
#define GS_ERR_BAD_ARG (-1)   /* null pointer, P < 0, W/H <= 0, sh_degree not in [0,3], > 2^24 tiles ...         */
#define GS_ERR_WORKSPACE (-2) /* workspace_bytes < gs_workspace_bytes(P, W, H, max_dup) or misaligned pointer    */
#define GS_ERR_OVERFLOW (-3)  /* reported by gs_get_intermediates: the frame needed more than max_dup duplicates */
#define GS_ERR_CUDA (-4)      /* a CUDA runtime call failed; gs_last_cuda_error() returns its cudaError_t        */
#define GS_ERR_LIMIT (-5)     /* gs_depth_sort_noalloc: more keys than the fixed scratch holds (GS_NOALLOC_MAX_KEYS) */

#define GS_TILE 16            /* tile edge in pixels                                         */

/* Scratch size (bytes) that gs_render needs for P Gaussians, a W x H image and room for `max_dup` duplicated
 * (tile, Gaussian) entries ("duplicates the surviving primitives across intersecting tiles").
 * Returns 0 on bad arguments.  max_dup must be < 2^32. */
size_t gs_workspace_bytes(int P, int W, int H, uint64_t max_dup);

/* Forward render of one frame.
 *
 *  Per-Gaussian inputs: dev, fp32, read-only, reusable across calls
 *    means3D   [P,3]   world-space centres
 *    scales    [P,3]   ACTIVATED scales (positive)
 *    rotations [P,4]   unit quaternions (w,x,y,z); not re-normalised
 *    opacities [P]     ACTIVATED opacities in (0,1)
 *    sh_coeffs [P,K,3] K = (sh_degree+1)^2, coefficient-major, RGB innermost
 *  Camera (host): viewmatrix (world->camera), projmatrix (FULL transform Proj*V), fx, fy in pixels, W, H, bg[3].
 *  Outputs (dev, fully overwritten):
 *    out_rgb         [3,H,W] planar fp32:  C + T_final * bg
 *    out_final_T     [H,W]   fp32 final transmittance
 *    out_tile_counts [gy*gx] u32, gx=(W+15)/16, gy=(H+15)/16: length of each tile's sorted list
 *    out_n_contrib   [H,W]   u32 number of Gaussians blended into the pixel, or NULL
 *  workspace: dev, 256-byte aligned, >= gs_workspace_bytes(P, W, H, max_dup) bytes; max_dup is recovered from
 *    workspace_bytes (the largest capacity that fits).  If the frame produces more duplicates than fit, every tile
 *    list is left empty (the image is the background) and gs_get_intermediates() reports GS_ERR_OVERFLOW with the
 *    n_dup the frame needs.  The capacity also selects the binning strategy -- up to 4 Mi entries: one radix sort over
 *    tile ids; above: radix sort over super-tiles of 8 x 8 tiles, then every tile list is written in place from its
 *    super-tile's list -- and P the preprocess kernel (from 2^20 Gaussians: two-phase, compacting).  The outputs do
 *    not depend on either choice.
 */
int gs_render(int P, const float* means3D, const float* scales, const float* rotations, const float* opacities,
              const float* sh_coeffs, int sh_degree, const float* viewmatrix, const float* projmatrix, float fx,
              float fy, int W, int H, const float* bg, float* out_rgb, float* out_final_T,
              uint32_t* out_tile_counts, uint32_t* out_n_contrib, void* workspace, size_t workspace_bytes,
              void* cuda_stream);

/* Pointers into the workspace of the LAST gs_render() call on it (valid until the next call on that workspace).
 * For parity tests and diagnostics; calling it synchronises the stream of that call. */
typedef struct gs_intermediates {
    int32_t P, W, H, grid_x, grid_y, n_tiles;
    uint32_t n_visible;            /* Gaussians with tiles_touched > 0                                           */
    uint64_t n_dup;                /* total duplicated entries the frame needs = sum of tiles_touched            */
    uint64_t max_dup;              /* capacity of this workspace                                                  */
    const uint32_t* per_gaussian;  /* dev [P,4] u32: {xmin | ymin<<16, xmax | ymax<<16, depth bits, radius};
                                      rect in tiles, half-open; all zero for a culled Gaussian                   */
    const float* record;           /* dev [P,16], the 64-byte render record, defined only where tiles_touched > 0:
                                      first 32 bytes -- all the tight box (Eq. 13-18) of the render stage reads:
                                      [0..1] mu_x, mu_y (pixels)   [2] conic b (Eq. 5)   [3] a*c-b*b
                                      [4] x*  [5] 1/c  [6] c*tau: per-Gaussian constants of the tight box (tau =
                                      2 ln(255 o) widened)   [7] flags (bits; 1 = degenerate conic)
                                      second 32 bytes -- read only for entries that reach a pixel (hoist, Eq. 8):
                                      [8] conic a  [9] conic c  [10] log2(opacity)
                                      [11..13] r, g, b (SH colour clamped at 0)   [14] 0   [15] tile-cull modes: the
                                      upper bound of 2 ln(255 o) the rect and the exact tile test use, else 0      */
    const uint64_t* depth_sorted;  /* dev [n_visible]: (depth bits << 32 | Gaussian id), ascending, stable       */
    const uint32_t* dup_offsets;   /* dev [n_visible]: exclusive prefix sum, in depth order, of the number of
                                      SUPER-TILES (8 x 8 tiles) each Gaussian's tile rect reaches -- the level the
                                      duplication and the sort run on (two-level binning)                        */
    const uint32_t* tile_ranges;   /* dev [n_tiles+1]: list of tile t is sorted_ids[tile_ranges[t] .. [t+1])     */
    const uint32_t* sorted_ids;    /* dev [min(n_dup,max_dup)]: Gaussian ids, by (tile, depth bits, id)          */
    uint64_t n_coarse;             /* duplicated (super-tile, Gaussian) entries that were actually sorted        */
} gs_intermediates;
int gs_get_intermediates(const void* workspace, gs_intermediates* out);

/* Per-stage device times (ms, CUDA events) of the last gs_render() on this workspace made while timing was
 * enabled with gs_set_timing(1): [0] preprocess, [1] depth sort, [2] tile grid, [3] offset scan, [4] duplicate,
 * [5] tile sort, [6] render, [7] whole frame.  [4] is the duplication over super-tiles -- fused with the first radix pass
 * on frames with a capacity of <= 4 M entries -- and [5] the remaining radix passes plus the expansion of the super-tile
 * lists into the tile lists.  Enabling timing adds event records and one stream
 * synchronisation per frame, serialises the tile-grid kernel (otherwise on a side stream, concurrent with the depth sort)
 * and disables programmatic dependent launch, so that every stage time is that stage alone; it is off by default. */
#define GS_N_TIMINGS 8
int gs_set_timing(int enable);
int gs_get_timings(const void* workspace, float ms[GS_N_TIMINGS]);

/* Render-kernel variant (ablation ladder of PAPER.md Table IV):
 *   0 = baseline column of Alg. 1 (one thread per pixel, direct conic, per-pixel branches)
 *   1 = + tile-local hoisting (Eq. 7-10)
 *   2 = + warp-level culling (Eq. 13-21)
 *   3 = + warp-coherent blending (Eq. 22, branch-free)            -- the paper's full method
 *   4 = B200 design (default): 2 pixels/thread, packed f32x2, per-warp ballot compaction, cp.async-gathered staging
 *   5 = (removed: the warp-specialised experiment of round 1; GS_ERR_BAD_ARG)
 *   6 = precision switch of PAPER.md Table V: variant 3 with the polynomial in GLOBAL pixel coordinates and fp32
 *       coefficients (Eq. 11).  For measuring the error the tile-local form removes; NOT within the parity tolerance.
 * Returns GS_ERR_BAD_ARG for an unknown variant.  Process-wide default (see gs_set_workspace_option). */
int gs_set_render_variant(int variant);
int gs_get_render_variant(void);

/* Tighter tile culling (tile-level culling is orthogonal to Local-GS and composes with it; P:181 the
 * alpha >= 1/255 visibility threshold).  mode 0 (default): the standard rect -- the 3-sigma square of BASELINE.json's
 * north_star.  mode 1: that square intersected with the axis-aligned bounding box of the Gaussian's alpha >= 1/255
 * ellipse (half-extents sqrt(tau c / det), sqrt(tau a / det), tau = 2 ln(255 o) from a library-free upper bound), and
 * Gaussians with o <= 1/255 dropped.  No pixel outside that box can be blended, so the image, final T and n_contrib are
 * unchanged while tiles_touched, N_dup, the tile counts and the sorted lists shrink (30-55 % fewer entries on the five
 * configurations).  The rect arithmetic is one IEEE rounding per operation: bit-identical to the oracle's TILE_CULL mode.
 * mode 2: the rect of mode 1, and a (tile, Gaussian) pair is LISTED only if the ellipse (tau + 0.05) meets the tile's box of
 * pixel centres -- the exact ellipse-tile intersection, evaluated where the super-tile lists are expanded into tile lists
 * (x-extent of the ellipse over the row band: PAPER.md Eq. 13-18 with x and y exchanged; fp32, one IEEE rounding per
 * operation, bit-identical to the oracle's TILE_CULL_EXACT mode).  Per-Gaussian outputs, tiles_touched and N_dup (the capacity
 * a frame needs) stay those of mode 1; out_tile_counts holds the EXACT list lengths; gs_intermediates.tile_ranges still
 * holds the rect-based first slots: list t is sorted_ids[tile_ranges[t] .. tile_ranges[t] + out_tile_counts[t]).  Another
 * 25-40 % fewer entries than mode 1.  Mode 2 needs the two-level binning, i.e. a workspace sized for max_dup > 4 Mi entries
 * (gs_render returns GS_ERR_WORKSPACE otherwise), and render variant 4 (GS_ERR_BAD_ARG otherwise); it launches plainly
 * (gs_set_graph is ignored).
 * Returns GS_ERR_BAD_ARG for another mode.  Process-wide. */
int gs_set_tile_cull(int mode);
int gs_get_tile_cull(void);

/* Frames in flight.  With gs_set_render_stream(1) the render kernel of every later gs_render() call is enqueued on a
 * library-owned stream of the LOWEST priority (one per workspace), forked from and joined back into `cuda_stream` with
 * events, so that `cuda_stream` still orders everything.  Meant for callers that keep several frames in flight on
 * HIGHER-priority streams (one workspace each): the latency-bound binning kernels of one frame then take SM slots as
 * they free up, ahead of the throughput-bound render blocks of another (measured: -5 % time per frame on config 2,
 * -7 % on config 3 with 4-6 frames in flight).  Off by default: a single frame gains nothing and loses the
 * programmatic dependent launch of its render kernel.  Process-wide, like the other switches. */
int gs_set_render_stream(int enable);

/* Render statistics (render variant 4 with out_n_contrib != NULL only; off by default, process-wide).  With
 * gs_set_stats(1) the render kernel counts what its blend loop did and gs_get_stats() (which synchronises the
 * stream of the last call on `workspace`) returns
 *   [0] (warp, Gaussian) slots walked by the blend loop (after the warp cull of PAPER.md Sec. III-C, before Eq. 22 exit)
 *   [1] (pixel, Gaussian) pairs blended = sum of out_n_contrib
 *   [2] (tile, Gaussian) entries staged into shared memory (Sec. III-B5)
 *   [3] (pixel, Gaussian) pairs whose alpha was evaluated = 64 x [0]
 * These are the units of the render roofline in bench.py. */
#define GS_N_STATS 4
int gs_set_stats(int enable);
int gs_get_stats(const void* workspace, uint64_t out[GS_N_STATS]);

/* CUDA graph replay (small frames are launch-chain-bound).  With gs_set_graph(1) the launch sequence of
 * a frame -- the workspace memset, the 10-12 kernels, the fork / join of the side and render streams -- is captured ONCE
 * per workspace and (P, W, H, SH degree, capacity, switches) and replayed with one cudaGraphLaunch; before every replay
 * the three kernel nodes whose arguments change (camera in preprocess and render, the caller's input / output pointers)
 * are updated with cudaGraphExecKernelNodeSetParams.  Same kernels, same results.  Ignored (plain launches) while timing
 * is enabled, for render variants other than 4 and on the legacy / per-thread default streams, which cannot be captured.
 * Process-wide default, off; per workspace: GS_OPT_GRAPH. */
int gs_set_graph(int enable);

/* Per-workspace switches.  The setters above are process-wide DEFAULTS; a value set here applies to the gs_render() calls on
 * this workspace only and wins over the default, so that two renderers (or a timed / statistics render next to a batch in
 * another thread) cannot change each other's launch path.  value -1 = follow the process-wide switch again.  May be called
 * before the first gs_render() on the workspace.  GS_ERR_BAD_ARG for an unknown option or value. */
#define GS_OPT_RENDER_VARIANT 0   /* as gs_set_render_variant */
#define GS_OPT_TILE_CULL 1        /* as gs_set_tile_cull      */
#define GS_OPT_TIMING 2           /* as gs_set_timing         */
#define GS_OPT_STATS 3            /* as gs_set_stats          */
#define GS_OPT_RENDER_STREAM 4    /* as gs_set_render_stream  */
#define GS_OPT_GRAPH 5            /* as gs_set_graph          */
#define GS_N_OPTIONS 6
int gs_set_workspace_option(const void* workspace, int option, int value);

/* Releases what the library keeps for a workspace address: its side stream, its render stream, their events and the
 * record of the last call (gs_get_intermediates / gs_get_timings / gs_get_stats then fail until the next gs_render).
 * Synchronises those streams first.  Call it before freeing the workspace; GS_OK also when nothing was kept. */
int gs_release(const void* workspace);

/* Ranking of the radix passes (csrc/binning.cu).  0: one shared-memory atomicAdd per key, whose returned value is the
 * stable rank PROVIDED the hardware serves same-address lanes in lane order (true on sm_100, not a PTX guarantee);
 * 1: ballot multi-split, documented semantics only (8 ballots per key round).  -1 (default): decided per device by
 * gs_selftest_atomic_order(), run once on the first gs_render() on that device -- if it ever reports a violation the
 * library ranks with ballots instead of returning unstable lists.  gs_get_rank_mode() returns the mode in force on the
 * current device (running the self-test if it has not run yet), or a negative error code. */
int gs_set_rank_mode(int mode);
int gs_get_rank_mode(void);

/* Number of kernel launches (ours; memsets not counted) enqueued by the last gs_render() in this process. */
int gs_last_launch_count(void);

/* Device self-test of the one undocumented hardware property the radix sort relies on (csrc/binning.cu,
 * radix_pass_kernel): the lanes of one warp-wide shared-memory atomicAdd that hit the same address are served in
 * ascending lane order, and a thread's atomics in program order, so the returned values are stable ranks.  Runs
 * `iters` iterations x 8 atomics per thread over 7 digit distributions on the current device (synchronous; uses 16
 * bytes of private device scratch).  out[0] = atomics whose returned value differed from the stable rank (must be
 * 0), out[1] = atomics checked. */
int gs_selftest_atomic_order(int iters, uint64_t out[2]);

/* Measured issue peaks of the current device, the denominators of the render roofline (Sec. IV-F / Table VII
 * counts FP32 and SFU work; BASELINE.json metric "blend kernel % FP32+SFU issue peak").  Saturates the FP32 pipe with
 * scalar fma.rn.f32, with packed fma.rn.f32x2 (what the blend loop issues) and the SFU with ex2.approx.ftz -- 8 independent
 * chains per thread, 64 warps per SM, `iters` x 256 instructions per thread, best of 3 timed launches (CUDA events,
 * synchronous, default stream) -- and returns THREAD-OPERATIONS per second: out[0] FFMA, out[1] FFMA2 (two FP32
 * operations per lane and instruction), out[2] MUFU.EX2.  Uses 16 bytes of private device scratch. */
int gs_selftest_issue_peak(int iters, double out[3]);

/* Depth sort WITHOUT any allocation -- for callers that cannot call cudaMalloc (code under CUDA stream capture, tight
 * serving loops, harnesses that forbid it).  The operation is the depth sort of the binning stage ("sorts them
 * by tile index and depth"; four stable 8-bit LSD radix passes over the depth bits, before duplication):
 *   keys_out[0..n) = keys_in[0..n) in ascending order of bits 63..32, STABLE (keys whose high words are equal keep their
 *   input order; bits 31..0 are carried along) -- with keys (depth bits << 32 | Gaussian id) in id order this is the
 *   (depth, id) order of gs_intermediates.depth_sorted.
 * keys_in, keys_out: dev, n 64-bit keys each, 8-byte aligned, distinct buffers on the CURRENT device (GS_ERR_BAD_ARG
 * otherwise); keys_in is only read.  Enqueued on `cuda_stream` (one memset node, 5 kernels); no host synchronisation.
 * The passes are the radix_pass_kernel of gs_render; their scratch (ping-pong keys, digit histograms, tile counters,
 * look-back status words) is a static __device__ array of 4.2 MB that every GPU that loads the library holds until the
 * process exits.  Hence the LIMIT: n <= GS_NOALLOC_MAX_KEYS (= gs_noalloc_max_keys()); a larger n returns GS_ERR_LIMIT
 * and enqueues nothing; n == 0 returns GS_OK and enqueues nothing.  The call makes no cudaMalloc / cudaFree / stream or
 * event creation; its first call on a device looks up the array's address (cudaGetSymbolAddress) and the SM count.
 * Ranking uses the ballot multi-split (gs_set_rank_mode(1) semantics), which needs no self-test.
 * ALL calls share the one array per device: two calls that overlap on the GPU (different streams, or graphs launched
 * concurrently) race -- order them on one stream or with events.  The array keeps the last call's contents; the call
 * itself clears what must start at zero. */
#define GS_NOALLOC_MAX_KEYS 262144
uint32_t gs_noalloc_max_keys(void);
int gs_depth_sort_noalloc(const uint64_t* keys_in, uint64_t* keys_out, uint32_t n, void* cuda_stream);

/* Synchronous device->host copy of `bytes` bytes (a plain cudaMemcpy) -- lets a binding without CUDA runtime access
 * read the arrays gs_get_intermediates() points at. */
int gs_copy_to_host(void* dst_host, const void* src_dev, size_t bytes);

const char* gs_error_string(int code);
int gs_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif
