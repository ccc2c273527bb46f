/* gs_oracle.h -- C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, obviously-correct CPU implementation of what the forward 3DGS tile rasterizer
 * computes (PAPER.md:51-53 pipeline, Eq. 4-5, baseline column of Alg. 1
 * PAPER.md:260-275), following the readings listed in DESIGN.md (C-P0..C-P9, C-B, C-R).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.  It shares no code, header, table or constant with the CUDA path
 * (include/gs.h, the paper_2606_16566_b200/csrc sources) and must never be linked into the product.
 *
 * All pointers are HOST pointers.  Matrices are row-major, column-vector convention.
 */
#ifndef GS_ORACLE_H
#define GS_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct gs_oracle_result gs_oracle_result;

/* Pointers into a result; valid until gs_oracle_free(result). */
typedef struct gs_oracle_view {
    int32_t P, W, H, grid_x, grid_y, n_tiles, n_lists, full; /* full=1: every tile listed and rendered */
    uint64_t n_dup;              /* total duplicated keys = sum of tiles_touched                        */
    uint64_t n_list_entries;     /* entries stored in sorted_ids (== n_dup when full)                   */
    uint64_t pairs_traversed;    /* (pixel, Gaussian) pairs reached by the blend loop                   */
    uint64_t pairs_blended;      /* pairs actually blended (step 6 of C-R)                              */
    /* per Gaussian (C-P0..C-P9); all zero for a culled Gaussian */
    const uint32_t* depth_bits;  /* [P] bits of fp32 view-space z                                       */
    const int32_t* radius;       /* [P]                                                                 */
    const int32_t* rect;         /* [P,4] xmin, ymin, xmax, ymax in tiles, half-open                    */
    const uint32_t* tiles_touched; /* [P]                                                               */
    const float* mu;             /* [P,2] pixel-space centre                                            */
    const float* conic;          /* [P,3] a, b, c                                                       */
    const float* rgb;            /* [P,3] SH colour, clamped at 0                                       */
    /* binning (C-B) */
    const uint32_t* tile_counts; /* [n_tiles] list length of EVERY tile (also in subset mode)           */
    const int32_t* list_tile;    /* [n_lists] tile id of list l (identity when full)                    */
    const uint64_t* list_offsets;/* [n_lists+1] into sorted_ids                                         */
    const uint32_t* sorted_ids;  /* [n_list_entries] per list: (depth bits asc, Gaussian index asc)     */
    /* per pixel (C-R); pixels of tiles that were not rendered (subset mode) hold zeros */
    const float* image;          /* [3,H,W]                                                             */
    const float* final_T;        /* [H,W]                                                               */
    const uint32_t* n_contrib;   /* [H,W] Gaussians blended                                             */
    const uint32_t* last_k;      /* [H,W] 1 + list position of the last blended Gaussian (0: none)      */
    const uint8_t* fragile;      /* [H,W] bit0: some alpha within delta of 1/255; bit1: some T' within delta of 1e-4 */
    const float* m_alpha;        /* [H,W] min |ln(o)+power-ln(1/255)| over Gaussians reached            */
    const float* m_T;            /* [H,W] min |T'/1e-4 - 1| over Gaussians that passed the alpha test   */
    const uint8_t* rendered;     /* [n_tiles] 1 if the tile's pixels were rendered                      */
} gs_oracle_view;

/* flags */
#define GS_ORACLE_NO_RENDER 1   /* stop after binning */
#define GS_ORACLE_NO_LISTS  2   /* stop after preprocess + tile_counts */
#define GS_ORACLE_TILE_CULL 4   /* C-P8': tile rect intersected with the AABB of the alpha >= 1/255 ellipse;
                                   off by default -- every pin of the standard definition uses the 3-sigma square */

#define GS_ORACLE_TILE_CULL_EXACT 8 /* C-P8'': the C-P8' rect, and a (tile, Gaussian) pair is counted and listed only if the
                                   ellipse alpha >= 1/255 (widened) meets the tile's box of pixel centres (exact
                                   ellipse-tile test).  tile_counts and the lists shrink; rect,
                                   tiles_touched and n_dup stay those of C-P8' */

/* Runs the oracle.  tile_subset == NULL: all tiles (full).  Otherwise only the n_subset listed tiles get
 * lists and pixels; per-Gaussian outputs and tile_counts always cover everything.
 * n_threads <= 1: single-threaded (the definitional baseline); > 1: the per-list stable sorts of C-B and the tiles of
 * C-R are spread over threads (same std::stable_sort per list, same arithmetic per pixel: identical results).  fragile_delta: the delta of the parity protocol (1e-3).
 * Returns NULL on bad arguments. */
gs_oracle_result* gs_oracle_render(int P, const float* means3D, const float* scales, const float* rotations,
                                   const float* opacities, const float* sh_coeffs, int sh_degree,
                                   const float* viewmatrix, const float* projmatrix, float fx, float fy,
                                   int W, int H, const float* bg, const int32_t* tile_subset, int n_subset,
                                   int n_threads, int flags, double fragile_delta);
void gs_oracle_get_view(const gs_oracle_result* r, gs_oracle_view* out);
void gs_oracle_free(gs_oracle_result* r);

/* Brute force (DESIGN.md pin T4): untiled renderer.  For every pixel: all un-culled Gaussians whose rect
 * contains the pixel's tile (use_rect=1) or ALL un-culled Gaussians (use_rect=0), in input order, stably
 * sorted by depth bits, blended by C-R.  Outputs [3,H,W], [H,W], [H,W]. */
int gs_oracle_render_untiled(int P, const float* means3D, const float* scales, const float* rotations,
                             const float* opacities, const float* sh_coeffs, int sh_degree,
                             const float* viewmatrix, const float* projmatrix, float fx, float fy,
                             int W, int H, const float* bg, int use_rect,
                             float* image, float* final_T, uint32_t* n_contrib);

/* The paper's machinery, restated for the invariants I1/I2 (double precision). */
/* Eq. 8 (reading G2): V = [A,B,C,D,E,F] from (a,b,c,o) and (dx,dy) = mu - tile origin. */
void gs_oracle_hoist(double a, double b, double c, double o, double dx, double dy, double V[6]);
/* Eq. 13-21 (reading S13): 8-bit warp mask of the 16x2 strips of the tile at (Tx,Ty).
 * Also returns the continuous span through y_span[2] = {y_min, y_max} (NaN,NaN when empty). */
uint32_t gs_oracle_warp_mask(double a, double b, double c, double o, double mux, double muy,
                             double Tx, double Ty, double y_span[2]);
/* C-P9: signed real-SH basis, out[k] for k < (deg+1)^2, such that colour = 0.5 + sum_k out[k]*sh[k]. */
void gs_oracle_sh_basis(int deg, const double dir[3], double out[16]);

#ifdef __cplusplus
}
#endif
#endif
