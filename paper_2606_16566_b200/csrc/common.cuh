// common.cuh -- workspace layout, control block and small device helpers shared by the CUDA translation units.
// Product code (libgs.so).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// -DGS_DEBUG_BOUNDS (build.py build(debug_bounds=True) -> libgs_dbg.so, loaded with GS_DEBUG_BOUNDS=1): every index into the
// workspace and into the caller's output arrays is checked on the device and a violation traps -- the stand-in for
// compute-sanitizer, which is not available on the GPU pool.  Compiles to nothing in the product build.
#ifdef GS_DEBUG_BOUNDS
#define GS_BOUND(idx, limit) do { if (!((unsigned long long)(idx) < (unsigned long long)(limit))) __trap(); } while (0)
#else
#define GS_BOUND(idx, limit) ((void)0)
#endif

namespace gs {

constexpr int TILE = 16;
// two-level binning: a super-tile is 8 x 8 tiles.  (4 x 4 was measured too: -10 % on the expansion of
// the 10 M-Gaussian scene, +10 % on the indoor scene whose large splats double the sorted level; not worth a heuristic.)
constexpr int SUPER_SHIFT = 3;
constexpr int CDIFF_SMEM = 2304;           // coarse difference grids up to this many cells are accumulated in shared memory
constexpr int MAX_SORT_PASSES_DEPTH = 4;   // 32 depth bits, 8-bit digits
constexpr int MAX_SORT_PASSES_TILE = 3;    // up to 24 tile-id bits
constexpr int SORT_THREADS = 256;
// keys per thread of a radix-pass tile, from the CAPACITY of the array being sorted (host and layout agree on it)
__host__ __device__ inline int sort_items_for(unsigned long long capacity) { return capacity <= (256ull << 10) ? 4 : 16; }
constexpr int PRE_THREADS = 256;                      // threads per preprocess block (one 32-Gaussian sub-tile per warp)
constexpr int COMPACT_MIN_P = 1 << 20;                // scenes below this size skip the compaction of visible Gaussians
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_WARP_TILE = 32 * SCAN_ITEMS;        // 256 depth-sorted Gaussians per offset-scan tile (one warp)
constexpr unsigned long long FUSED_DUP_MAX = 4ull << 20;   // frames up to this capacity fuse the duplication into the first tile pass
constexpr int EXP_SEG = 2048;                         // expand_kernel: super-tile list entries per chunk (8 warps x 8 x 32 lanes)
constexpr int EXP_THREADS = 256;
constexpr int DUP_TILE = 1024;                        // duplication chunk: output slots per staged set of depth ranks
// keys per thread of the fused duplicate + first-tile-pass kernel (its tile also holds the staged ranks of a chunk)
__host__ __device__ inline int dup_items_for(unsigned long long capacity) { return capacity <= (256ull << 10) ? 4 : 8; }

// Control block at the start of the workspace; zeroed (with the tile-difference grid and the look-back status
// arrays that follow it) by one cudaMemsetAsync per frame.
struct Ctrl {
    uint32_t tile_counter[16];          // dynamic tile ids of the chained-scan kernels (forward-progress order)
    unsigned long long n_vis;           // visible Gaussians
    unsigned long long n_sort;          // keys the depth sort runs over: n_vis (compacted) or P (small scenes)
    unsigned long long overflow;        // 1 if n_dup > max_dup
    unsigned long long n_dup;           // duplicates the frame needs
    unsigned long long n_dup_eff;       // duplicates actually produced (0 on overflow)
    uint32_t depth_hist[MAX_SORT_PASSES_DEPTH][256];  // global digit histograms of the depth bits (atomics)
    uint32_t tile_hist[MAX_SORT_PASSES_TILE][256];    // global digit histograms of the tile ids (from tile counts)
    unsigned long long stats[4];        // render statistics (gs_set_stats): warp slots walked, pairs blended, entries staged
};
// The workspace holds TWO control blocks: `ctrl` (frame-level counters + the FINE tile grid: n_dup, overflow) and
// `cctrl` (the same fields for the SUPER-TILE grid that duplication and sort run on: n_vis is copied there,
// n_dup / tile_hist / tile_counter are the coarse ones).
enum { TC_PRE = 0, TC_DEPTH0 = 1, TC_SCAN = 5, TC_TILE0 = 6, TC_EXPAND = 10 };

// Look-back status word: [63:62] flag, [61:0] value.
constexpr unsigned long long ST_EMPTY = 0ull;
constexpr unsigned long long ST_AGG = 1ull << 62;
constexpr unsigned long long ST_INC = 2ull << 62;
constexpr unsigned long long ST_MASK = (1ull << 62) - 1;

struct Frame {              // per-frame constants, passed by value to the kernels
    int P, W, H, gx, gy, n_tiles, deg, K;
    int cshift;                            // log2 of the super-tile edge in tiles (two-level binning; 0 = one level)
    int cgx, cgy, n_ctiles, cdiff_cells;   // super-tile grid and its difference grid
    int tile_bits, n_tile_passes;         // of the grid the duplication + sort runs on (the super-tile grid)
    int compact;                // 1: preprocess compacts the visible Gaussians (P >= COMPACT_MIN_P)
    int rank_mode;              // radix passes: 0 = rank by shared-memory atomics, 1 = by ballots (gs_set_rank_mode)
    int tile_cull;              // 1: tile rect intersected with the bounding box of the alpha >= 1/255 ellipse (gs_set_tile_cull);
                                // 2: that rect, and expand_kernel lists a (tile, Gaussian) pair only if the ellipse meets the tile
    int diff_copies, diff_cells; // replicas of the coverage difference grid (power of two) and cells per replica
    float V[16], PM[16];
    float fx, fy;
    float campos[3];
    float bg[3];
    unsigned long long max_dup;
    const uint32_t* tile_len;   // tile_cull == 2: exact list length of every tile (workspace; written by expand_kernel), else nullptr
};

struct Pointers {           // device pointers carved from the workspace
    Ctrl* ctrl;
    Ctrl* cctrl;                            // control block of the super-tile level
    int* cdiff;                             // [(cgy+1)*(cgx+1)] difference grid of super-tile coverage
    uint32_t* cranges;                      // [n_ctiles + 1] ranges of the super-tile lists in cids
    uint32_t* ccounts;                      // [n_ctiles]
    uint32_t* tile_len;                     // [n_tiles] two-level frames, tile_cull == 2: exact list lengths (expand_kernel)
    uint32_t* cids;                         // [max_dup] Gaussian ids sorted by (super-tile, depth bits, id)
    int* diff;                              // [diff_copies][(gy+1)*(gx+1)] 2-D difference grid of tile coverage
    unsigned long long* st_pre;             // [pre tiles]    look-back status: compaction of visible Gaussians
    unsigned long long* st_scan;            // [scan tiles]   look-back status: duplicate offsets
    unsigned long long* st_depth;           // [4][depth sort tiles][256]
    unsigned long long* st_tile;            // [3][tile sort tiles][256]
    unsigned long long* st_exp;             // [chunks of EXP_SEG super-tile entries][64] look-back status of expand_kernel (two-level frames)
    uint4* per_g;                           // [P] {rect01, rect23, depth bits, radius}
    float4* rec;                            // [P][4] 64-byte render record (layout: include/gs.h, gs_intermediates.record)
    unsigned long long* gkeyA;              // [P] (depth bits << 32 | id), compacted
    unsigned long long* gkeyB;              // [P] ping-pong
    uint32_t* dup_off;                      // [P] exclusive prefix of tiles_touched in depth order
    uint2* rk_rect;                         // [P] tile rect {xmin | ymin<<16, xmax | ymax<<16} in depth order
    uint32_t* chunk_start;                  // [ceil(max_dup / DUP_TILE) + 1] depth rank owning entry c * DUP_TILE
    uint32_t* ranges;                       // [n_tiles + 1]
    uint4* desc;                            // [n_tiles] {tile, start, end, -}: tiles by descending list length (render schedule)
    unsigned long long* entA;               // [max_dup] (tile << 32 | id)
    unsigned long long* entB;               // [max_dup] ping-pong
    uint32_t* ids;                          // [max_dup] final sorted Gaussian ids
    size_t n_depth_tiles, n_tile_tiles;     // status array strides (tiles per pass)
};

// Programmatic dependent launch (PDL): every kernel of the frame starts with griddep_sync() -- wait until the previous
// kernel in the stream has completed and its writes are visible, then allow the NEXT kernel's launch to begin -- so the
// launch latency and block scheduling of kernel k+1 overlap the tail of kernel k (the frame of a 100 000-Gaussian
// scene is 11 kernels of 5-50 us each).  Without the launch attribute both instructions are no-ops.
__device__ __forceinline__ void griddep_sync() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// Kernel functions of the three launches whose arguments change from frame to frame (camera, caller pointers), noted by
// their launchers so that api.cu can find the matching nodes of a captured CUDA graph (gs_set_graph).
struct CaptureLog { const void* preprocess = nullptr; const void* tile_grid = nullptr; const void* render = nullptr; };
extern thread_local CaptureLog g_caplog;
extern thread_local int g_use_pdl;   // api.cu: 1 = launch with the programmatic-serialization attribute (set per frame, by the calling thread)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = g_use_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Warp-parallel decoupled look-back over single-value status words (called by one full warp).
// Returns the exclusive prefix of tile `tile` (sum of the aggregates of tiles 0..tile-1) in every lane.
__device__ __forceinline__ unsigned long long lookback_warp(const unsigned long long* status, int tile) {
    const int lane = threadIdx.x & 31;
    unsigned long long excl = 0;
    int idx = tile - 1;
    while (idx >= 0) {
        const int my = idx - lane;
        unsigned long long s = ST_INC;  // tiles before 0: inclusive prefix 0
        if (my >= 0) {
            do { s = ld_status(status + my); } while ((s >> 62) == 0);
        }
        const unsigned inc = __ballot_sync(0xffffffffu, (s >> 62) == 2);
        unsigned long long v = s & ST_MASK;
        if (inc) {
            const int first = __ffs(inc) - 1;  // nearest tile with an inclusive prefix
            if (lane > first) v = 0;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        excl += v;
        if (inc) break;
        idx -= 32;
    }
    return excl;
}

// Block-wide exclusive scan of one u32 per thread (blockDim.x == 256); returns the exclusive prefix and the total.
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* smem_warp /*[8]*/, uint32_t& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) smem_warp[w] = inc;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const uint32_t s = smem_warp[i];
        if (i < w) base += s;
        tot += s;
    }
    total = tot;
    __syncthreads();
    return base + inc - v;
}

}  // namespace gs
