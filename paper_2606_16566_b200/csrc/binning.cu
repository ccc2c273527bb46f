// binning.cu -- duplication + sort ("parallel prefix scan ... duplicates the surviving primitives across
// intersecting tiles into 64-bit key-value pairs ... sorted by GPU Radix Sort ... tile ranges").
//
// The result is exactly a STABLE LSD radix sort of the keys (tile_id << 32 | depth bits) with value = Gaussian id
// (BASELINE.json north_star (2),(3)); DESIGN.md "Binning" explains the one structural change:
//   all duplicates of a Gaussian share their 32 depth bits, so the LSD digit passes over the depth bits are run
//   BEFORE duplication, on the n_visible per-Gaussian keys (depth << 32 | id)  [4 passes over <= P elements],
//   then the entries (tile << 32 | id) are emitted in that order and only the tile-id digits are sorted after
//   duplication  [ceil(tile_bits / 8) passes over N_dup elements].  Stable passes commute with duplication because
//   duplication preserves relative order, so the final order is (tile, depth bits, id) -- bit-identical.
// Tile counts / ranges come from the 2-D difference grid filled by the preprocess kernel, not from the keys.
//
// Kernels: radix_pass_kernel (one-sweep: block-local ranking + chained decoupled look-back per digit),
//          tile_grid_kernel, scan_offsets_kernel (chained scan), duplicate_kernel (load-balanced by output chunk).
#include <type_traits>

#include "common.cuh"

namespace gs {

// ------------------------------------------------------------------------------------------------------------
// One stable radix pass over u64 elements on digit (key >> shift) & 255.  No payload: the id lives in the low
// 32 bits of the element.  OUT32: write only the low 32 bits (last tile pass -> sorted_ids).
//
// Ranking.  Keys are loaded warp-striped (lane l of warp w holds elements w*32*ITEMS + j*32 + l, j = 0..ITEMS-1), so
// the input order inside a warp is (round j, lane).  The stable rank of a key among the warp's keys of equal digit
// is the value returned by ONE shared-memory atomicAdd on the warp's private digit counter: the ITEMS atomics of a
// thread are issued in program order, and the lanes of one warp-wide ATOMS that hit the same address are served in
// ascending lane order.  The second property is how sm_100 hardware resolves the conflict, not a documented PTX
// guarantee: it is asserted on the device by gs_selftest_atomic_order() (tests/test_gpu_parity.py runs it) and
// every list-parity test would expose a violation.  Why not match.any: measured on B200 it costs ~400 cycles of
// latency and ~40-70 cycles of issue per warp instruction (emulated), against ~2 cycles for the atomic
// (profiles/r01_microbench.md) -- the match-based first version of this kernel spent 35 % of its stall samples there.
// ------------------------------------------------------------------------------------------------------------
template <int ITEMS, typename K>
struct SortSmem {
    K sorted[SORT_THREADS * ITEMS];
    uint32_t hist[SORT_THREADS / 32][256];
    uint32_t bpos[256], gbase[256], gpos[256];
    uint32_t scan[SORT_THREADS / 32];
    int tile;
};

// One tile of a pass, shared by the plain pass kernel and the fused duplicate + first-pass kernel.  key[] holds the
// tile's keys warp-striped (element w*32*ITEMS + j*32 + lane in key[j]); sm.hist is zeroed and sm.gbase holds the
// exclusive scan of the global digit histogram.  digit(key) -> 0..255; store(pos, key) writes one output element.
template <int ITEMS, typename K, typename DigitF, typename StoreF>
__device__ __forceinline__ void radix_tile(SortSmem<ITEMS, K>& sm, K (&key)[ITEMS], const int tile, const uint32_t tile_n,
                                           unsigned long long* __restrict__ status, const int rank_mode, const unsigned long long n_total, DigitF digit, StoreF store) {
    (void)n_total;
    constexpr int NW = SORT_THREADS / 32;
    constexpr int TILE_N = SORT_THREADS * ITEMS;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t wbase = w * (32 * ITEMS) + lane;
    uint32_t rk2[ITEMS / 2];  // two 16-bit ranks per register (a warp holds 32 * ITEMS <= 512 keys)
    if (rank_mode != 0) {
        // Ranking with documented semantics only (gs_set_rank_mode(1), or chosen by the device self-test): the lanes of a
        // round that hold the same digit find each other with 8 ballots (multi-split), rank = the warp's running count of
        // the digit + the number of such lanes below this one; the lowest of them advances the count.  ~10x the issue
        // cost of the atomic form (profiles/r01_microbench.md), same result.
        const unsigned lt = (1u << lane) - 1u;
#pragma unroll
        for (int j = 0; j < ITEMS; j++) {
            const bool valid = wbase + j * 32 < tile_n;
            const uint32_t d = digit(key[j]);
            unsigned peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
            for (int b = 0; b < 8; b++) {
                const unsigned bb = __ballot_sync(0xffffffffu, (d >> b) & 1u);
                peers &= ((d >> b) & 1u) ? bb : ~bb;
            }
            if (!valid) peers = 0u;
            const int leader = peers ? __ffs(peers) - 1 : 0;
            uint32_t base = 0;
            if (valid && lane == leader) {
                base = sm.hist[w][d];
                sm.hist[w][d] = base + __popc(peers);
            }
            __syncwarp();
            base = __shfl_sync(0xffffffffu, base, leader);
            const uint32_t r = valid ? base + __popc(peers & lt) : 0u;
            if (j & 1) rk2[j / 2] |= r << 16; else rk2[j / 2] = r;
        }
    } else if (tile_n == TILE_N) {
#pragma unroll
        for (int j = 0; j < ITEMS; j += 2) {
            const uint32_t ra = atomicAdd(&sm.hist[w][digit(key[j])], 1u);
            const uint32_t rb = atomicAdd(&sm.hist[w][digit(key[j + 1])], 1u);
            rk2[j / 2] = ra | (rb << 16);
        }
    } else {
#pragma unroll
        for (int j = 0; j < ITEMS; j += 2) {
            uint32_t ra = 0, rb = 0;
            if (wbase + j * 32 < tile_n) ra = atomicAdd(&sm.hist[w][digit(key[j])], 1u);
            if (wbase + (j + 1) * 32 < tile_n) rb = atomicAdd(&sm.hist[w][digit(key[j + 1])], 1u);
            rk2[j / 2] = ra | (rb << 16);
        }
    }
    __syncthreads();
    // ---- per digit: exclusive prefix over warps, block count, publish aggregate ------------------------------
    uint32_t cnt = 0;
#pragma unroll
    for (int k = 0; k < NW; k++) {
        const uint32_t t = sm.hist[k][tid];
        sm.hist[k][tid] = cnt;
        cnt += t;
    }
    unsigned long long* st = status + (size_t)tile * 256 + tid;
    st_status(st, (tile == 0 ? ST_INC : ST_AGG) | (unsigned long long)cnt);
    uint32_t tot;
    const uint32_t bpos = block_excl_scan_256(cnt, sm.scan, tot);  // contains __syncthreads
    sm.bpos[tid] = bpos;
    __syncthreads();
    // ---- block-local reorder through shared memory ---------------------------------------------------------
#pragma unroll
    for (int j = 0; j < ITEMS; j++) {
        if (wbase + j * 32 < tile_n) {
            const uint32_t d = digit(key[j]);
            GS_BOUND(sm.bpos[d] + sm.hist[w][d] + ((rk2[j / 2] >> (16 * (j & 1))) & 0xffffu), TILE_N);
            sm.sorted[sm.bpos[d] + sm.hist[w][d] + ((rk2[j / 2] >> (16 * (j & 1))) & 0xffffu)] = key[j];
        }
    }
    // ---- decoupled look-back for digit `tid` ------------------------------------------------------------------
    // Steady state (many waves of tiles): the direct predecessor already holds its inclusive prefix -- one load.
    // First wave (or a sort that fits in one wave): every resident tile only has its aggregate published, and the
    // inclusive prefixes advance a few tiles per L2 round trip; LB_WINDOW status words in flight per step divide
    // that latency chain.
    unsigned long long excl = 0;
    if (tile > 0) {
        constexpr int LB_WINDOW = 16;
        int idx = tile - 1;
        bool done = false;
        {
            const unsigned long long s0 = ld_status(status + (size_t)idx * 256 + tid);
            if ((s0 >> 62) != 0) {
                excl = s0 & ST_MASK;
                idx--;
                done = (s0 >> 62) == 2 || idx < 0;
            }
        }
        while (!done) {
            unsigned long long sv[LB_WINDOW];
#pragma unroll
            for (int k = 0; k < LB_WINDOW; k++)
                sv[k] = (idx - k >= 0) ? ld_status(status + (size_t)(idx - k) * 256 + tid) : ST_INC;
#pragma unroll
            for (int k = 0; k < LB_WINDOW; k++) {
                if (done || (sv[k] >> 62) == 0) break;   // not published yet: poll again from here
                excl += sv[k] & ST_MASK;
                idx--;
                done = (sv[k] >> 62) == 2;
            }
        }
        st_status(st, ST_INC | (excl + cnt));
    }
    sm.gpos[tid] = sm.gbase[tid] + (uint32_t)excl - bpos;
    __syncthreads();
    // ---- coalesced output: runs of equal digits are contiguous ---------------------------------------------
#pragma unroll
    for (int j = 0; j < ITEMS; j++) {
        const uint32_t li = j * SORT_THREADS + tid;
        if (li < tile_n) {
            const K k = sm.sorted[li];
            GS_BOUND(sm.gpos[digit(k)] + li, n_total);
            store(sm.gpos[digit(k)] + li, k);
        }
    }
}

// MODE 0: u64 keys in and out, digit (key >> shift) & 255.
// MODE 1: u64 keys in, only the low 32 bits (the Gaussian id) out -- the last pass of the 64-bit path.
// MODE 2: packed 32-bit entries (tile >> 8) << 24 | id in, digit = entry >> 24, id out -- the last of two tile passes.
// MODE 3: u64 entries (tile << 32 | id) in, packed 32-bit entries out -- the first of two tile passes, P <= 2^24.
template <int ITEMS, int MODE>
__global__ void __launch_bounds__(SORT_THREADS, 4)
radix_pass_kernel(const void* __restrict__ in_v, void* __restrict__ out_v, const unsigned long long* __restrict__ n_ptr,
                  int shift, const uint32_t* __restrict__ ghist, unsigned long long* __restrict__ status,
                  uint32_t* __restrict__ tile_counter, const int rank_mode) {
    using K = typename std::conditional<MODE == 2, uint32_t, unsigned long long>::type;
    constexpr int TILE_N = SORT_THREADS * ITEMS;
    __shared__ SortSmem<ITEMS, K> sm;
    griddep_sync();
    const K* __restrict__ in = static_cast<const K*>(in_v);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned long long n = *n_ptr;
    {   // exclusive scan of the global digit histogram -> first output slot of every digit
        uint32_t tot;
        sm.gbase[tid] = block_excl_scan_256(ghist[tid], sm.scan, tot);
    }
    auto digit = [shift](K k) -> uint32_t {
        if (MODE == 2) return (uint32_t)(k >> 24);
        return (uint32_t)(k >> shift) & 255u;
    };
    auto store = [out_v](uint32_t pos, K k) {
        if (MODE == 0) static_cast<unsigned long long*>(out_v)[pos] = k;
        else if (MODE == 1) static_cast<uint32_t*>(out_v)[pos] = (uint32_t)k;
        else if (MODE == 2) static_cast<uint32_t*>(out_v)[pos] = (uint32_t)k & 0xffffffu;
        else static_cast<uint32_t*>(out_v)[pos] = ((uint32_t)((unsigned long long)k >> 40) << 24) | ((uint32_t)k & 0xffffffu);
    };
    while (true) {
        __syncthreads();
        if (tid == 0) sm.tile = (int)atomicAdd(tile_counter, 1u);
#pragma unroll
        for (int k = 0; k < 8; k++) sm.hist[w][k * 32 + lane] = 0;
        __syncthreads();
        const int tile = sm.tile;
        const unsigned long long tile_base = (unsigned long long)tile * TILE_N;
        if (tile_base >= n) break;
        const uint32_t tile_n = (uint32_t)min((unsigned long long)TILE_N, n - tile_base);
        K key[ITEMS];
        const uint32_t wbase = w * (32 * ITEMS) + lane;
        if (tile_n == TILE_N) {
#pragma unroll
            for (int j = 0; j < ITEMS; j++) key[j] = __ldcs(in + tile_base + wbase + j * 32);
        } else {
#pragma unroll
            for (int j = 0; j < ITEMS; j++) key[j] = (wbase + j * 32 < tile_n) ? in[tile_base + wbase + j * 32] : (K)0;
        }
        radix_tile<ITEMS, K>(sm, key, tile, tile_n, status, rank_mode, n, digit, store);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Tile grid: 2-D inclusive prefix of the difference grid -> tile counts; exclusive scan -> tile ranges, n_dup;
// digit histograms of the tile ids for the tile radix passes.  One block (the grid has <= 2^24 cells).
// ------------------------------------------------------------------------------------------------------------
constexpr int GRID_THREADS = 1024;
// Render schedule: tiles in 8 coarse classes of list length, longest class first, RASTER order inside a class (a
// stable counting sort).  Heavy tiles start first, so the render launch has no tail of a few long tiles; raster order
// inside a class keeps neighbouring tiles -- which share most of their Gaussians -- close in time, i.e. in L2.  (A fine
// sort by length was tried: on the 10 M-Gaussian scene it doubled the render time by scattering the record gathers.)
constexpr int LPT_BUCKETS = 8;
__device__ __forceinline__ int lpt_bucket(uint32_t c) {
    if (c < 64u) return c ? 1 : 0;
    const int l = 31 - __clz(c);      // >= 6
    return l - 4 > 7 ? 7 : l - 4;     // 64..127 -> 2, 128..255 -> 3, ..., >= 2048 -> 7
}
__global__ void __launch_bounds__(GRID_THREADS)
tile_grid_kernel(const Frame f, const Pointers p, uint32_t* __restrict__ counts /* out_tile_counts */, const Ctrl* __restrict__ parent) {
    __shared__ uint32_t s_hist[MAX_SORT_PASSES_TILE][256];
    __shared__ unsigned long long s_part[GRID_THREADS / 32];
    __shared__ unsigned long long s_total;
    __shared__ uint32_t s_wb[GRID_THREADS / 32][LPT_BUCKETS];
    __shared__ uint32_t s_bbase[LPT_BUCKETS];
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gw = f.gx + 1, gh = f.gy + 1;
    int* diff = p.diff;
    for (int k = tid; k < MAX_SORT_PASSES_TILE * 256; k += GRID_THREADS) (&s_hist[0][0])[k] = 0;
    // row-wise inclusive prefix, one warp per row, in place
    for (int y = w; y < gh; y += GRID_THREADS / 32) {
        int carry = 0;
        for (int x0 = 0; x0 < gw; x0 += 32) {
            const int x = x0 + lane;
            int v = 0;
            if (x < gw)
                for (int r = 0; r < f.diff_copies; r++) v += diff[(size_t)r * f.diff_cells + y * gw + x];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, v, o);
                if (lane >= o) v += t;
            }
            v += carry;
            if (x < gw) diff[y * gw + x] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
    }
    __syncthreads();
    // column-wise running sum, one thread per column -> counts
    for (int x = tid; x < f.gx; x += GRID_THREADS) {
        int acc = 0;
#pragma unroll 8
        for (int y = 0; y < f.gy; y++) {
            acc += diff[y * gw + x];
            counts[y * f.gx + x] = (uint32_t)acc;
        }
    }
    __syncthreads();
    // exclusive scan over tiles (row-major) -> ranges; each thread owns a contiguous run of tiles
    const int per = (f.n_tiles + GRID_THREADS - 1) / GRID_THREADS;
    const int t0 = min(f.n_tiles, tid * per), t1 = min(f.n_tiles, t0 + per);
    unsigned long long sum = 0;
    uint32_t cb[LPT_BUCKETS], cinc[LPT_BUCKETS];
#pragma unroll
    for (int k = 0; k < LPT_BUCKETS; k++) cb[k] = 0;
    for (int t = t0; t < t1; t++) {
        const uint32_t c = counts[t];
        sum += c;
        const int bk = lpt_bucket(c);
#pragma unroll
        for (int k = 0; k < LPT_BUCKETS; k++) cb[k] += (k == bk) ? 1u : 0u;
    }
#pragma unroll
    for (int k = 0; k < LPT_BUCKETS; k++) {   // per class: inclusive scan of the thread counts over the warp
        uint32_t v = cb[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        cinc[k] = v;
        if (lane == 31) s_wb[w][k] = v;
    }
    unsigned long long inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_part[w] = inc;
    __syncthreads();
    if (tid == 0) {
        unsigned long long c = 0;
        for (int k = 0; k < GRID_THREADS / 32; k++) { const unsigned long long t = s_part[k]; s_part[k] = c; c += t; }
        s_total = c;
    }
    if (tid >= 32 && tid < 32 + LPT_BUCKETS) {   // per class: exclusive prefix over the warps, class total
        const int k = tid - 32;
        uint32_t c = 0;
        for (int ww = 0; ww < GRID_THREADS / 32; ww++) { const uint32_t t = s_wb[ww][k]; s_wb[ww][k] = c; c += t; }
        s_bbase[k] = c;
    }
    __syncthreads();
    if (tid == 0) {   // first descriptor slot of every class, LONGEST lists first
        uint32_t c = 0;
        for (int k = LPT_BUCKETS - 1; k >= 0; k--) { const uint32_t t = s_bbase[k]; s_bbase[k] = c; c += t; }
    }
    __syncthreads();
    uint32_t pos[LPT_BUCKETS];
#pragma unroll
    for (int k = 0; k < LPT_BUCKETS; k++) pos[k] = s_bbase[k] + s_wb[w][k] + cinc[k] - cb[k];
    const unsigned long long total = s_total;
    // the super-tile level (parent != nullptr) follows the verdict of the tile level: its total is never larger
    const bool overflow = total > f.max_dup || (parent != nullptr && parent->overflow != 0ull);
    unsigned long long run = s_part[w] + inc - sum;
    for (int t = t0; t < t1; t++) {
        const uint32_t c = counts[t];
        GS_BOUND(t, f.n_tiles);
        p.ranges[t] = overflow ? 0u : (uint32_t)run;
        if (p.desc != nullptr) {   // tile descriptor at its slot of the render schedule
            const int bk = lpt_bucket(c);
            uint32_t slot = 0;
#pragma unroll
            for (int k = 0; k < LPT_BUCKETS; k++)
                if (k == bk) slot = pos[k]++;
            GS_BOUND(slot, f.n_tiles);
            p.desc[slot] = overflow ? make_uint4((uint32_t)t, 0u, 0u, 0u) : make_uint4((uint32_t)t, (uint32_t)run, (uint32_t)(run + c), 0u);
        }
        run += c;
        if (!overflow && c) {
#pragma unroll
            for (int k = 0; k < MAX_SORT_PASSES_TILE; k++) atomicAdd(&s_hist[k][((uint32_t)t >> (8 * k)) & 255u], c);
        }
    }
    if (tid == 0) {
        p.ranges[f.n_tiles] = overflow ? 0u : (uint32_t)total;
        p.ctrl->n_dup = total;
        p.ctrl->n_dup_eff = overflow ? 0ull : total;
        p.ctrl->overflow = overflow ? 1ull : 0ull;
        if (parent != nullptr) p.ctrl->n_vis = parent->n_vis;
    }
    __syncthreads();
    for (int k = tid; k < MAX_SORT_PASSES_TILE * 256; k += GRID_THREADS) (&p.ctrl->tile_hist[0][0])[k] = (&s_hist[0][0])[k];
}

// ------------------------------------------------------------------------------------------------------------
// Offsets of every depth-ranked Gaussian's run of duplicates: exclusive prefix sum of tiles_touched in depth
// order ("parallel prefix scan").  Also records, for every DUP_TILE-th output slot, the rank that
// owns it, so that the duplicate kernel needs no search in global memory.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t rect_tiles(const uint4 pg) {
    const uint32_t w = (pg.y & 0xffffu) - (pg.x & 0xffffu), h = (pg.y >> 16) - (pg.x >> 16);
    return w * h;
}

// One WARP per 256-rank tile (8 consecutive ranks per lane), chained through the look-back status words; no block
// barrier.  The rect of every rank is gathered once here and stored in depth order for the duplicate kernel.
__global__ void __launch_bounds__(SCAN_THREADS)
scan_offsets_kernel(const Pointers p, const int cshift, const unsigned long long max_dup) {
    (void)max_dup;
    griddep_sync();
    const int lane = threadIdx.x & 31;
    const unsigned long long n = p.ctrl->n_vis;
    if (p.ctrl->overflow != 0) return;
    while (true) {
        int tile = 0;
        if (lane == 0) tile = (int)atomicAdd(&p.ctrl->tile_counter[TC_SCAN], 1u);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        const unsigned long long base_r = (unsigned long long)tile * SCAN_WARP_TILE + (unsigned long long)lane * SCAN_ITEMS;
        if ((unsigned long long)tile * SCAN_WARP_TILE >= n) break;
        uint32_t id[SCAN_ITEMS], tt[SCAN_ITEMS];
        uint2 rc[SCAN_ITEMS];
        const bool full = (unsigned long long)(tile + 1) * SCAN_WARP_TILE <= n;  // warp-uniform
        if (full) {   // 64 contiguous, 64-byte aligned bytes per lane: four 16-byte loads
            const ulonglong2* src = reinterpret_cast<const ulonglong2*>(p.gkeyA + base_r);
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; k += 2) {
                const ulonglong2 v = __ldg(src + k / 2);
                id[k] = (uint32_t)v.x; id[k + 1] = (uint32_t)v.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; k++) id[k] = (base_r + k < n) ? (uint32_t)p.gkeyA[base_r + k] : 0xffffffffu;
        }
        uint32_t sum = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            tt[k] = 0;
            rc[k] = make_uint2(0u, 0u);
            if (id[k] != 0xffffffffu) {
                uint4 pg = __ldg(p.per_g + id[k]);
                {   // the tile rect on the grid the duplication runs on: cells of 2^cshift x 2^cshift tiles, half-open
                    const uint32_t r = (1u << cshift) - 1u;
                    const uint32_t x0 = (pg.x & 0xffffu) >> cshift, y0 = (pg.x >> 16) >> cshift;
                    const uint32_t x1 = ((pg.y & 0xffffu) + r) >> cshift, y1 = ((pg.y >> 16) + r) >> cshift;
                    pg.x = x0 | (y0 << 16);
                    pg.y = x1 | (y1 << 16);
                }
                rc[k] = make_uint2(pg.x, pg.y);
                tt[k] = rect_tiles(pg);
            }
            sum += tt[k];
        }
        uint32_t inc = sum;   // inclusive scan over the lanes
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        const uint32_t wtotal = __shfl_sync(0xffffffffu, inc, 31);
        if (lane == 0) st_status(p.st_scan + tile, (tile == 0 ? ST_INC : ST_AGG) | (unsigned long long)wtotal);
        unsigned long long excl = 0;
        if (tile > 0) {
            excl = lookback_warp(p.st_scan, tile);
            if (lane == 0) st_status(p.st_scan + tile, ST_INC | (excl + wtotal));
        }
        unsigned long long off = excl + inc - sum;
        if (full) {   // rect in depth order: duplicate_kernel reads it sequentially
            uint32_t o[SCAN_ITEMS];
            unsigned long long run = off;
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; k++) { o[k] = (uint32_t)run; run += tt[k]; }
            uint4* d4 = reinterpret_cast<uint4*>(p.dup_off + base_r);
            d4[0] = make_uint4(o[0], o[1], o[2], o[3]);
            d4[1] = make_uint4(o[4], o[5], o[6], o[7]);
            uint4* r4 = reinterpret_cast<uint4*>(p.rk_rect + base_r);
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; k += 2) r4[k / 2] = make_uint4(rc[k].x, rc[k].y, rc[k + 1].x, rc[k + 1].y);
        }
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            if (base_r + k < n) {
                if (!full) {
                    p.dup_off[base_r + k] = (uint32_t)off;
                    p.rk_rect[base_r + k] = rc[k];
                }
                if (tt[k]) {  // chunk boundaries c*DUP_TILE that fall inside [off, off + tt)
                    const unsigned long long c0 = (off + DUP_TILE - 1) / DUP_TILE, c1 = (off + tt[k] - 1) / DUP_TILE;
                    for (unsigned long long c = c0; c <= c1; c++) { GS_BOUND(c, max_dup / DUP_TILE + 2); p.chunk_start[c] = (uint32_t)(base_r + k); }
                }
            }
            off += tt[k];
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Duplication FUSED with the first tile pass.  Output slot k of the duplication ("duplicates the surviving
// primitives across intersecting tiles") belongs to the depth-ranked Gaussian r with off[r] <= k < off[r] +
// tiles_touched; its j = k - off[r]-th tile in row-major rect order gives the entry (tile << 32 | id).  The entries are
// never written to HBM in that order: every block GENERATES the 256 * ITEMS consecutive entries of its radix tile in
// shared memory (4 consecutive slots per thread and 1 024-slot chunk: one binary search in the chunk's staged
// offsets, then an incremental walk over columns / rows / ranks) and sorts them on the low tile byte straight away.
// Balanced by OUTPUT slot, so a splat covering 10^4 tiles is spread over many blocks.
//   OUTK 0: (tile << 32 | id) out (u64)       -- three tile passes (> 65 536 tiles) or ids that need more than 24 bits
//   OUTK 1: id out (u32)                      -- a single tile pass (<= 256 tiles): this IS the sorted id list
//   OUTK 2: (tile >> 8) << 24 | id out (u32)  -- two tile passes, P <= 2^24: the second pass moves 4-byte entries
// ------------------------------------------------------------------------------------------------------------
constexpr int GEN_ITEMS = 4;   // slots per thread and chunk; DUP_TILE = SORT_THREADS * GEN_ITEMS
template <int ITEMS, int OUTK>
__global__ void __launch_bounds__(SORT_THREADS, 4)
dup_pass_kernel(const Frame f, const Pointers p, void* __restrict__ out_v, const uint32_t* __restrict__ ghist,
                unsigned long long* __restrict__ status, uint32_t* __restrict__ tile_counter) {
    using K = unsigned long long;
    constexpr int TILE_N = SORT_THREADS * ITEMS;
    static_assert(DUP_TILE == SORT_THREADS * GEN_ITEMS && ITEMS % GEN_ITEMS == 0, "chunking");
    __shared__ SortSmem<ITEMS, K> sm;
    __shared__ uint32_t s_off[DUP_TILE + 2];
    __shared__ uint2 s_rect[DUP_TILE + 2];
    __shared__ uint32_t s_id[DUP_TILE + 2];
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned long long n = p.ctrl->n_dup_eff;
    const uint32_t n_vis = (uint32_t)p.ctrl->n_vis;
    const uint32_t gx = (uint32_t)f.gx;
    {
        uint32_t tot;
        sm.gbase[tid] = block_excl_scan_256(ghist[tid], sm.scan, tot);
    }
    auto digit = [](K k) -> uint32_t { return (uint32_t)(k >> 32) & 255u; };
    auto store = [out_v](uint32_t pos, K k) {
        if (OUTK == 0) static_cast<unsigned long long*>(out_v)[pos] = k;
        else if (OUTK == 1) static_cast<uint32_t*>(out_v)[pos] = (uint32_t)k;
        else static_cast<uint32_t*>(out_v)[pos] = ((uint32_t)(k >> 40) << 24) | ((uint32_t)k & 0xffffffu);
    };
    while (true) {
        __syncthreads();
        if (tid == 0) sm.tile = (int)atomicAdd(tile_counter, 1u);
#pragma unroll
        for (int k = 0; k < 8; k++) sm.hist[w][k * 32 + lane] = 0;
        __syncthreads();
        const int tile = sm.tile;
        const unsigned long long tile_base = (unsigned long long)tile * TILE_N;
        if (tile_base >= n) break;
        const uint32_t tile_n = (uint32_t)min((unsigned long long)TILE_N, n - tile_base);
        // ---- generate the tile's entries, chunk by chunk, in slot order into sm.sorted ---------------------------
        for (int c = 0; c < ITEMS / GEN_ITEMS; c++) {
            const unsigned long long k0 = tile_base + (unsigned long long)c * DUP_TILE;
            if (k0 >= n) break;
            const uint32_t cn = (uint32_t)min((unsigned long long)DUP_TILE, n - k0);
            const unsigned long long ci = k0 / DUP_TILE;
            const uint32_t r0 = p.chunk_start[ci];
            const uint32_t r1 = (k0 + DUP_TILE < n) ? p.chunk_start[ci + 1] : (n_vis - 1);
            const uint32_t nr = r1 - r0 + 1;  // <= DUP_TILE + 1 ranks can start inside one chunk
            if (c) __syncthreads();           // the previous chunk's staged ranks are no longer read
            for (uint32_t k = tid; k < nr; k += SORT_THREADS) {  // the chunk's ranks: all sequential reads
                s_off[k] = p.dup_off[r0 + k];
                s_rect[k] = p.rk_rect[r0 + k];
                s_id[k] = (uint32_t)p.gkeyA[r0 + k];
            }
            __syncthreads();
            const uint32_t lk0 = tid * GEN_ITEMS;
            if (lk0 < cn) {
                const uint32_t kk = (uint32_t)k0 + lk0;  // N_dup < 2^32
                uint32_t lo = 0, hi = nr - 1;            // largest local rank with s_off <= kk
                while (lo < hi) {
                    const uint32_t mid = (lo + hi + 1) >> 1;
                    if (s_off[mid] <= kk) lo = mid; else hi = mid - 1;
                }
                uint32_t lr = lo;
                uint2 rc = s_rect[lr];
                uint32_t id = s_id[lr];
                uint32_t x0 = rc.x & 0xffffu, x1 = rc.y & 0xffffu, wdt = x1 - x0;
                uint32_t left = wdt * ((rc.y >> 16) - (rc.x >> 16)) - (kk - s_off[lr]);  // slots of this rank still to emit
                uint32_t ty, tx;
                {   // the one division of this thread and chunk: row-major position of slot kk inside the rect
                    const uint32_t j = kk - s_off[lr], row = j / wdt;
                    ty = (rc.x >> 16) + row;
                    tx = x0 + (j - row * wdt);
                }
                uint32_t tl = ty * gx + tx;
                K* dst = &sm.sorted[c * DUP_TILE + lk0];
#pragma unroll
                for (int q = 0; q < GEN_ITEMS; q++) {
                    if (lk0 + q < cn) dst[q] = ((K)tl << 32) | id;
                    // advance to the next slot: next column, next row of the rect, or the next rank (every visible
                    // rank has >= 1 tile).  Past the end of the chunk the values are never stored.
                    tx++; tl++; left--;
                    if (left == 0) {
                        lr = min(lr + 1, nr - 1);
                        rc = s_rect[lr]; id = s_id[lr];
                        x0 = rc.x & 0xffffu; x1 = rc.y & 0xffffu; wdt = x1 - x0;
                        left = wdt * ((rc.y >> 16) - (rc.x >> 16));
                        tx = x0; ty = rc.x >> 16; tl = ty * gx + tx;
                    } else if (tx == x1) {
                        tx = x0; ty++; tl = ty * gx + tx;
                    }
                }
            }
        }
        __syncthreads();
        // ---- pick the keys up warp-striped (the order radix_tile ranks in) and sort the tile ---------------------------
        K key[ITEMS];
        const uint32_t wbase = w * (32 * ITEMS) + lane;
#pragma unroll
        for (int j = 0; j < ITEMS; j++) key[j] = (wbase + j * 32 < tile_n) ? sm.sorted[wbase + j * 32] : (K)0;
        radix_tile<ITEMS, K>(sm, key, tile, tile_n, status, f.rank_mode, n, digit, store);   // first barrier inside precedes its stores
    }
}

// Stand-alone duplication for LARGE frames: the same walk, entries (tile << 32 | id) written to HBM in duplication
// order.  Measured on the 10 M-Gaussian scene the fused kernel above is slower than this kernel plus a plain first
// pass (its phases serialise inside a block); on small frames the fused kernel wins by a launch and 16 bytes per entry.
__global__ void __launch_bounds__(SORT_THREADS)
duplicate_kernel(const Frame f, const Pointers p, unsigned long long* __restrict__ ent) {
    __shared__ uint32_t s_off[DUP_TILE + 2];
    __shared__ uint2 s_rect[DUP_TILE + 2];
    __shared__ uint32_t s_id[DUP_TILE + 2];
    griddep_sync();
    const int tid = threadIdx.x;
    const unsigned long long n = p.ctrl->n_dup_eff;
    const uint32_t n_vis = (uint32_t)p.ctrl->n_vis;
    const uint32_t gx = (uint32_t)f.gx;
    {   // clear the look-back status words of the tile passes that follow: only the tiles n entries occupy (api.cu make_layout)
        const unsigned long long tile_n = (unsigned long long)SORT_THREADS * sort_items_for(f.max_dup);
        const unsigned long long words = min((n + tile_n - 1) / tile_n + 1, (unsigned long long)p.n_tile_tiles) * 256ull;
        for (int pass = 0; pass < f.n_tile_passes; pass++) {
            unsigned long long* st = p.st_tile + (size_t)pass * p.n_tile_tiles * 256;
            for (unsigned long long i = (unsigned long long)blockIdx.x * SORT_THREADS + tid; i < words; i += (unsigned long long)gridDim.x * SORT_THREADS)
                st[i] = 0ull;
        }
        // ... and those of expand_kernel (64 per chunk of EXP_SEG super-tile entries; n counts super-tile entries here)
        const unsigned long long xwords = ((n + EXP_SEG - 1) / EXP_SEG + 1) * 64ull;
        for (unsigned long long i = (unsigned long long)blockIdx.x * SORT_THREADS + tid; i < xwords; i += (unsigned long long)gridDim.x * SORT_THREADS)
            p.st_exp[i] = 0ull;
    }
    for (unsigned long long chunk = blockIdx.x; chunk * DUP_TILE < n; chunk += gridDim.x) {
        const unsigned long long k0 = chunk * DUP_TILE;
        const uint32_t cn = (uint32_t)min((unsigned long long)DUP_TILE, n - k0);
        const uint32_t r0 = p.chunk_start[chunk];
        const uint32_t r1 = ((chunk + 1) * DUP_TILE < n) ? p.chunk_start[chunk + 1] : (n_vis - 1);
        const uint32_t nr = r1 - r0 + 1;  // <= DUP_TILE + 1 ranks can start inside one chunk
        __syncthreads();
        for (uint32_t k = tid; k < nr; k += SORT_THREADS) {  // the chunk's ranks: offsets, rects, ids -- all sequential reads
            s_off[k] = p.dup_off[r0 + k];
            s_rect[k] = p.rk_rect[r0 + k];
            s_id[k] = (uint32_t)p.gkeyA[r0 + k];
        }
        __syncthreads();
        const uint32_t lk0 = tid * GEN_ITEMS;
        if (lk0 < cn) {
            const uint32_t kk = (uint32_t)k0 + lk0;  // N_dup < 2^32
            uint32_t lo = 0, hi = nr - 1;            // largest local rank with s_off <= kk
            while (lo < hi) {
                const uint32_t mid = (lo + hi + 1) >> 1;
                if (s_off[mid] <= kk) lo = mid; else hi = mid - 1;
            }
            uint32_t lr = lo;
            uint2 rc = s_rect[lr];
            uint32_t id = s_id[lr];
            uint32_t x0 = rc.x & 0xffffu, x1 = rc.y & 0xffffu, wdt = x1 - x0;
            uint32_t left = wdt * ((rc.y >> 16) - (rc.x >> 16)) - (kk - s_off[lr]);  // slots of this rank still to emit
            uint32_t ty, tx;
            {   // the one division of this thread: row-major position of slot kk inside the rect
                const uint32_t j = kk - s_off[lr], row = j / wdt;
                ty = (rc.x >> 16) + row;
                tx = x0 + (j - row * wdt);
            }
            uint32_t tile = ty * gx + tx;
            unsigned long long outv[GEN_ITEMS];
#pragma unroll
            for (int q = 0; q < GEN_ITEMS; q++) {
                outv[q] = ((unsigned long long)tile << 32) | id;
                // advance to the next slot: next column, next row of the rect, or the next rank (every visible rank
                // has >= 1 tile).  Past the end of the chunk the values are never stored.
                tx++; tile++; left--;
                if (left == 0) {
                    lr = min(lr + 1, nr - 1);
                    rc = s_rect[lr]; id = s_id[lr];
                    x0 = rc.x & 0xffffu; x1 = rc.y & 0xffffu; wdt = x1 - x0;
                    left = wdt * ((rc.y >> 16) - (rc.x >> 16));
                    tx = x0; ty = rc.x >> 16; tile = ty * gx + tx;
                } else if (tx == x1) {
                    tx = x0; ty++; tile = ty * gx + tx;
                }
            }
            GS_BOUND(k0 + lk0, f.max_dup);
            unsigned long long* dst = ent + k0 + lk0;
            if (lk0 + GEN_ITEMS <= cn) {
#pragma unroll
                for (int q = 0; q < GEN_ITEMS; q += 2)
                    __stcs(reinterpret_cast<ulonglong2*>(dst + q), make_ulonglong2(outv[q], outv[q + 1]));
            } else {
                for (int q = 0; q < GEN_ITEMS && lk0 + q < cn; q++) dst[q] = outv[q];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// host-side launchers
// ------------------------------------------------------------------------------------------------------------
static int imin(long long a, long long b) { return (int)(a < b ? a : b); }

// Launch one pass with the tile size chosen from the CAPACITY of the sorted array (sort_items_for, common.cuh): small
// arrays use 1 024-key tiles (more blocks, shorter critical path), large ones 4 096-key tiles (less look-back traffic).
template <int MODE>
static void launch_pass(int items, int n_sm, unsigned long long capacity, const void* in, void* out,
                        const unsigned long long* n_ptr, int shift, const uint32_t* ghist, unsigned long long* status,
                        uint32_t* tile_counter, cudaStream_t st, int rank_mode) {
    const long long tile_n = (long long)SORT_THREADS * items;
    const long long cap_tiles = ((long long)capacity + tile_n - 1) / tile_n;
    const int grid = imin(cap_tiles > 0 ? cap_tiles : 1, (long long)n_sm * 4);
    if (items == 16)
        launch_pdl(radix_pass_kernel<16, MODE>, dim3(grid), dim3(SORT_THREADS), st, in, out, n_ptr, shift, ghist, status, tile_counter, rank_mode);
    else
        launch_pdl(radix_pass_kernel<4, MODE>, dim3(grid), dim3(SORT_THREADS), st, in, out, n_ptr, shift, ghist, status, tile_counter, rank_mode);
}

void launch_depth_sort(const Frame& f, const Pointers& p, int n_sm, cudaStream_t st, int* launches) {
    unsigned long long* bufs[2] = {p.gkeyA, p.gkeyB};
    const int items = sort_items_for((unsigned long long)f.P);
    for (int pass = 0; pass < MAX_SORT_PASSES_DEPTH; pass++) {
        launch_pass<0>(items, n_sm, (unsigned long long)f.P, bufs[pass & 1], bufs[(pass + 1) & 1], &p.ctrl->n_sort,
                       32 + 8 * pass, p.ctrl->depth_hist[pass], p.st_depth + (size_t)pass * p.n_depth_tiles * 256,
                       &p.ctrl->tile_counter[TC_DEPTH0 + pass], st, f.rank_mode);
        (*launches)++;
    }
}

void launch_tile_grid(const Frame& f, const Pointers& p, uint32_t* out_tile_counts, const Ctrl* parent, cudaStream_t st, int* launches) {
    g_caplog.tile_grid = (const void*)tile_grid_kernel;
    launch_pdl(tile_grid_kernel, dim3(1), dim3(GRID_THREADS), st, f, p, out_tile_counts, parent);
    (*launches)++;
}

void launch_scan_offsets(const Frame& f, const Pointers& p, int cshift, int n_sm, cudaStream_t st, int* launches) {
    const long long cap_blocks = ((long long)f.P + SCAN_WARP_TILE * (SCAN_THREADS / 32) - 1) / (SCAN_WARP_TILE * (SCAN_THREADS / 32));
    const int grid = imin(cap_blocks > 0 ? cap_blocks : 1, (long long)n_sm * 8);
    launch_pdl(scan_offsets_kernel, dim3(grid), dim3(SCAN_THREADS), st, p, cshift, (unsigned long long)f.max_dup);
    (*launches)++;
}

// Duplication fused with the first tile pass, then the remaining tile passes:
//   1 pass  (<= 256 tiles):                 fused pass writes the sorted ids
//   2 passes, P <= 2^24:                    fused pass writes packed 4-byte entries, second pass (MODE 2) the ids
//   2 passes, P >  2^24 / 3 passes:         fused pass writes 8-byte entries, 64-bit passes follow
template <int OUTK>
static void launch_dup_pass(int items, int n_sm, const Frame& f, const Pointers& p, void* out, cudaStream_t st) {
    const long long tile_n = (long long)SORT_THREADS * items;
    const long long cap_tiles = ((long long)f.max_dup + tile_n - 1) / tile_n;
    const int grid = imin(cap_tiles > 0 ? cap_tiles : 1, (long long)n_sm * 4);
    if (items == 8)
        launch_pdl(dup_pass_kernel<8, OUTK>, dim3(grid), dim3(SORT_THREADS), st, f, p, out, p.ctrl->tile_hist[0], p.st_tile,
                   &p.ctrl->tile_counter[TC_TILE0]);
    else
        launch_pdl(dup_pass_kernel<4, OUTK>, dim3(grid), dim3(SORT_THREADS), st, f, p, out, p.ctrl->tile_hist[0], p.st_tile,
                   &p.ctrl->tile_counter[TC_TILE0]);
}

void launch_duplicate_and_tile_sort(const Frame& f, const Pointers& p, int n_sm, cudaStream_t st, int* launches,
                                    cudaEvent_t ev_after_duplicate) {
    const int gen_items = dup_items_for(f.max_dup), items = sort_items_for(f.max_dup);
    const bool packed = f.n_tile_passes == 2 && f.P <= (1 << 24);
    const bool fused = f.max_dup <= FUSED_DUP_MAX;
    unsigned long long* bufs[2] = {p.entA, p.entB};
    int first_pass = 1;
    if (fused) {
        if (f.n_tile_passes == 1) launch_dup_pass<1>(gen_items, n_sm, f, p, p.ids, st);
        else if (packed) launch_dup_pass<2>(gen_items, n_sm, f, p, p.entA, st);
        else launch_dup_pass<0>(gen_items, n_sm, f, p, p.entA, st);
        (*launches)++;
        if (ev_after_duplicate) cudaEventRecord(ev_after_duplicate, st);
    } else {   // entries to entB, first pass entB -> entA (packed or not), so that the later passes find them as in the fused path
        const long long cap_chunks = ((long long)f.max_dup + DUP_TILE - 1) / DUP_TILE;
        const int dgrid = imin(cap_chunks > 0 ? cap_chunks : 1, (long long)n_sm * 8);
        launch_pdl(duplicate_kernel, dim3(dgrid), dim3(SORT_THREADS), st, f, p, p.entB);
        (*launches)++;
        if (ev_after_duplicate) cudaEventRecord(ev_after_duplicate, st);
        if (f.n_tile_passes == 1)
            launch_pass<1>(items, n_sm, f.max_dup, p.entB, p.ids, &p.ctrl->n_dup_eff, 32, p.ctrl->tile_hist[0], p.st_tile,
                           &p.ctrl->tile_counter[TC_TILE0], st, f.rank_mode);
        else if (packed)
            launch_pass<3>(items, n_sm, f.max_dup, p.entB, p.entA, &p.ctrl->n_dup_eff, 32, p.ctrl->tile_hist[0], p.st_tile,
                           &p.ctrl->tile_counter[TC_TILE0], st, f.rank_mode);
        else {   // three passes: entB -> entA -> entB -> ids
            launch_pass<0>(items, n_sm, f.max_dup, p.entB, p.entA, &p.ctrl->n_dup_eff, 32, p.ctrl->tile_hist[0], p.st_tile,
                           &p.ctrl->tile_counter[TC_TILE0], st, f.rank_mode);
        }
        (*launches)++;
    }
    for (int pass = first_pass; pass < f.n_tile_passes; pass++) {
        const bool last = pass == f.n_tile_passes - 1;
        unsigned long long* status = p.st_tile + (size_t)pass * p.n_tile_tiles * 256;
        const void* in = bufs[(pass - 1) & 1];
        if (packed)
            launch_pass<2>(items, n_sm, f.max_dup, in, p.ids, &p.ctrl->n_dup_eff, 0, p.ctrl->tile_hist[pass], status,
                           &p.ctrl->tile_counter[TC_TILE0 + pass], st, f.rank_mode);
        else if (last)
            launch_pass<1>(items, n_sm, f.max_dup, in, p.ids, &p.ctrl->n_dup_eff, 32 + 8 * pass, p.ctrl->tile_hist[pass], status,
                           &p.ctrl->tile_counter[TC_TILE0 + pass], st, f.rank_mode);
        else
            launch_pass<0>(items, n_sm, f.max_dup, in, bufs[pass & 1], &p.ctrl->n_dup_eff, 32 + 8 * pass, p.ctrl->tile_hist[pass],
                           status, &p.ctrl->tile_counter[TC_TILE0 + pass], st, f.rank_mode);
        (*launches)++;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Expansion of the super-tile lists into the tile lists (second level of the binning).
// cids holds, for every super-tile (8 x 8 tiles), the ids of the Gaussians whose tile rect reaches it, in (depth bits,
// id) order.  A tile's list is the sub-sequence of its super-tile's list whose rects contain the tile, and it starts
// at ranges[tile] (known from the coverage grid) -- so it can be WRITTEN IN PLACE, in order, with no sort.
//
// Work is cut into CHUNKS of EXP_SEG consecutive entries of cids (whatever super-tiles they belong to), handed out in
// order by a ticket.  Inside a chunk every PIECE (the entries of one super-tile) is handled by the whole block:
//   (a) warp w takes 256 consecutive entries, eight per lane: id, rect -> the 64-bit mask of the super-tile's tiles the
//       rect covers (kept in shared memory), and the per-tile counts of its 256 entries (byte-sliced popcounts per lane,
//       one warp reduction per tile -- no ballot per (tile, 32 entries));
//   (b) 64 threads turn the counts into each warp's first slot in each of the 64 tile lists: ranges[tile] + the entries
//       of this super-tile in EARLIER chunks (decoupled look-back over one status word per (chunk, tile); only a
//       super-tile that straddles a chunk boundary needs it) + the counts of the warps before;
//   (c) every warp walks its entries 32 at a time and, tile by tile, ballots "covers this tile" and stores the ids of
//       the set lanes at consecutive slots (coalesced; the 4-byte id is the only HBM traffic per list entry).
// Per (tile, 32 entries) the cost is ~10 instructions, against a ballot, a popcount and a predicated store per tile
// row AND every staged entry of the super-tile in the previous kernel (one block per (super-tile, row) that read the
// whole super-tile list): 2.4x fewer instructions, and the rect of an entry is fetched once instead of eight times.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t spread4(uint32_t x) { return ((x & 15u) * 0x00204081u) & 0x01010101u; }   // bit i -> byte i

// C-P8'' (gs_set_tile_cull(2), exact ellipse-tile intersection): the tiles of super-tile (X0, Y0) whose box
// of pixel centres the ellipse a dx^2 + 2 b dx dy + c dy^2 <= tau + 0.05 meets, as the 64-bit mask (byte r = columns of tile
// row r; lo = rows 0-3, hi = rows 4-7).  Per tile row: the x-extent of the ellipse over the row band -- the paper's tight box
// (Eq. 13-18) with x and y exchanged -- then one interval test per column.  fp32 with ONE explicit IEEE rounding per
// operation, in the order of the oracle's tile_hit(): the decision is an integer and bit-identical on both sides.  Every
// "miss" is an affirmative comparison: a NaN keeps the tile.
__device__ __forceinline__ void exact_tile_mask(const float a, const float b, const float c, const float mux, const float muy,
                                                const float tau, const uint32_t X0, const uint32_t Y0, const uint32_t rows,
                                                uint32_t& lo, uint32_t& hi) {
    lo = hi = 0xffffffffu;
    const float det = __fsub_rn(__fmul_rn(a, c), __fmul_rn(b, b));
    if (!(det > 0.0f) || !(a > 0.0f) || !(c > 0.0f)) return;          // degenerate conic: keep everything
    const float te = __fadd_rn(tau, 0.05f);
    const float at = __fmul_rn(a, te);
    const float ia = __fdiv_rn(1.0f, a);
    const float hx = __fsqrt_rn(__fdiv_rn(__fmul_rn(te, c), det));
    const float ys = __fdiv_rn(__fmul_rn(-b, hx), c);                 // dy of the right-most point; the left-most is at -ys
    const float fx0 = (float)X0;
    lo = hi = 0u;
#pragma unroll
    for (int r = 0; r < 8; r++) {
        if (!((rows >> r) & 1u)) continue;                            // the rect does not reach this tile row
        const float d0 = __fsub_rn((float)(16u * (Y0 + r)), muy), d1 = __fadd_rn(d0, 15.0f);
        const float yu = fminf(fmaxf(ys, d0), d1), yl = fminf(fmaxf(-ys, d0), d1);
        const float du = __fsub_rn(at, __fmul_rn(__fmul_rn(det, yu), yu)), dl = __fsub_rn(at, __fmul_rn(__fmul_rn(det, yl), yl));
        if (du < 0.0f || dl < 0.0f) continue;                         // the band misses the ellipse
        const float xr = __fadd_rn(mux, __fmul_rn(__fadd_rn(__fmul_rn(-b, yu), __fsqrt_rn(fmaxf(du, 0.0f))), ia));
        const float xl = __fadd_rn(mux, __fmul_rn(__fsub_rn(__fmul_rn(-b, yl), __fsqrt_rn(fmaxf(dl, 0.0f))), ia));
        // tile columns ceil((xl - 15) / 16) .. floor(xr / 16), relative to the super-tile, clamped to its 8 columns; fminf /
        // fmaxf return the other operand for a NaN, i.e. a NaN keeps every column (the oracle's comparisons do the same)
        const float thi = fminf(floorf(__fmul_rn(xr, 0.0625f)) - fx0, 7.0f);
        const float tlo = fmaxf(ceilf(__fmul_rn(__fsub_rn(xl, 15.0f), 0.0625f)) - fx0, 0.0f);
        const int ih = (int)thi, il = (int)tlo;
        if (ih < il) continue;
        const uint32_t byte = ((2u << ih) - 1u) & ~((1u << il) - 1u);
        if (r < 4) lo |= byte << (8 * r); else hi |= byte << (8 * (r - 4));
    }
}

template <int SH, bool EXACT>
__global__ void __launch_bounds__(EXP_THREADS, 4)
expand_kernel(const Frame f, const Pointers p, uint32_t* __restrict__ out_counts) {
    static_assert(SH == 3, "the tile masks are 64-bit: 8 x 8 tiles per super-tile");
    constexpr int SUPER = 8;
    __shared__ __align__(16) uint2 s_m[8][8][32];       // [warp][sub-chunk][lane] tile mask (rows 0-3 | rows 4-7)
    __shared__ uint32_t s_id[8][8][32];
    __shared__ __align__(16) uint32_t s_cnt[8][64];     // [warp][tile] count, then first slot relative to s_tb
    __shared__ __align__(16) uint32_t s_tb[64];         // [tile] first slot of this piece in the tile's list
    __shared__ uint32_t s_ticket;
    griddep_sync();
    if (p.ctrl->overflow != 0ull) return;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const uint32_t n = p.cranges[f.n_ctiles];
    const uint32_t n_chunks = (n + EXP_SEG - 1) / EXP_SEG;
    for (;;) {
        __syncthreads();                                 // everything of the previous chunk is done with shared memory
        if (tid == 0) s_ticket = atomicAdd(&p.ctrl->tile_counter[TC_EXPAND], 1u);
        __syncthreads();
        const uint32_t g = s_ticket;
        if (g >= n_chunks) break;
        const uint32_t e0 = g * EXP_SEG, e1 = min(n, e0 + EXP_SEG);
        // super-tile of an entry: the last one with cranges[s] <= e
        auto super_tile_of = [&](const uint32_t e) -> uint32_t {
            uint32_t lo = 0, hi = (uint32_t)f.n_ctiles - 1;
            while (lo < hi) {
                const uint32_t mid = (lo + hi + 1) >> 1;
                if (__ldg(p.cranges + mid) <= e) lo = mid; else hi = mid - 1;
            }
            return lo;
        };
        // Pieces of this chunk, one super-tile each.  The LAST piece is handled FIRST: if its super-tile goes on into the
        // next chunk, the chunks behind wait for this chunk's status words, and those must not wait for the pieces
        // before it (whose own look-back would chain every chunk boundary of the frame into one serial dependency).
        const uint32_t s_first = super_tile_of(e0), s_last = super_tile_of(e1 - 1);
        const uint32_t last_q0 = max(__ldg(p.cranges + s_last), e0);
        uint32_t s = s_last, q0 = last_q0;
        bool last_done = false;
        for (;;) {
            const uint32_t cbeg = __ldg(p.cranges + s), cend = __ldg(p.cranges + s + 1);
            const uint32_t q1 = min(cend, e1);
            const bool from_before = cbeg < e0, goes_on = cend > e1;
            const int sy = (int)s / f.cgx, sx = (int)s - sy * f.cgx;
            const uint32_t X0 = (uint32_t)(sx * SUPER), Y0 = (uint32_t)(sy * SUPER);
            // ---- (a) masks and per-warp counts -----------------------------------------------------------------
            const uint32_t wq0 = q0 + 256u * (uint32_t)w;
            uint32_t id[8];
            uint2 rc[8];
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t e = wq0 + 32u * j + lane;
                id[j] = e < q1 ? __ldg(p.cids + e) : 0u;
            }
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t e = wq0 + 32u * j + lane;
                rc[j] = e < q1 ? __ldg(reinterpret_cast<const uint2*>(p.per_g + id[j])) : make_uint2(0u, 0u);
            }
            uint32_t mlo[8], mhi[8];
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t x0 = rc[j].x & 0xffffu, y0 = rc[j].x >> 16, x1 = rc[j].y & 0xffffu, y1 = rc[j].y >> 16;
                const uint32_t a = max(x0, X0), b = min(x1, X0 + SUPER), ra = max(y0, Y0), rb = min(y1, Y0 + SUPER);
                uint32_t cols = 0, rows = 0;
                if (b > a && rb > ra) {                  // (an entry past the end of the piece has an empty rect)
                    cols = ((1u << (b - a)) - 1u) << (a - X0);
                    rows = ((1u << (rb - ra)) - 1u) << (ra - Y0);
                }
                mlo[j] = cols * spread4(rows);           // byte r = cols if row r is covered
                mhi[j] = cols * spread4(rows >> 4);
                s_m[w][j][lane] = make_uint2(mlo[j], mhi[j]);
                s_id[w][j][lane] = id[j];
            }
            if (EXACT) {   // AND the exact ellipse-tile mask into the rect mask, entry by entry (not unrolled: ~300 instructions each);
                           // the record of entry j + 1 is in flight while entry j is evaluated
                const float4* rec = p.rec + 4 * (size_t)id[0];
                float4 n0 = __ldg(rec), n2 = __ldg(rec + 2), n3 = __ldg(rec + 3);   // {mu_x, mu_y, b, .} {a, c, ., .} {., ., ., tau}
#pragma unroll 1
                for (int j = 0; j < 8; j++) {
                    const float4 r0 = n0, r2 = n2, r3 = n3;
                    if (j < 7) {
                        const float4* nx = p.rec + 4 * (size_t)s_id[w][j + 1][lane];
                        n0 = __ldg(nx); n2 = __ldg(nx + 2); n3 = __ldg(nx + 3);
                    }
                    const uint2 m = s_m[w][j][lane];
                    if ((m.x | m.y) != 0u) {
                        // rows the rect reaches: a byte of the mask is non-zero
                        uint32_t rows = 0;
#pragma unroll
                        for (int r = 0; r < 4; r++) rows |= (((m.x >> (8 * r)) & 255u) ? 1u : 0u) << r | (((m.y >> (8 * r)) & 255u) ? 16u : 0u) << r;
                        uint32_t xl, xh;
                        exact_tile_mask(r2.x, r0.z, r2.y, r0.x, r0.y, r3.w, X0, Y0, rows, xl, xh);
                        s_m[w][j][lane] = make_uint2(m.x & xl, m.y & xh);
                    }
                }
#pragma unroll
                for (int j = 0; j < 8; j++) { const uint2 m = s_m[w][j][lane]; mlo[j] = m.x; mhi[j] = m.y; }
            }
            {   // counts: for tile row r the bytes of this lane's eight entries side by side, popcount of column c's bit
                // in all of them, one warp reduction per tile; lane t & 31 keeps the count of tile t
                uint32_t mine0 = 0, mine1 = 0;
#pragma unroll
                for (int r = 0; r < 8; r++) {
                    const uint32_t sel = 0x0040u + 0x0011u * (uint32_t)(r & 3);   // bytes 0, 1 <- byte r&3 of the first, of the second operand
                    uint32_t A, B;
                    if (r < 4) {
                        A = __byte_perm(__byte_perm(mlo[0], mlo[1], sel), __byte_perm(mlo[2], mlo[3], sel), 0x5410u);
                        B = __byte_perm(__byte_perm(mlo[4], mlo[5], sel), __byte_perm(mlo[6], mlo[7], sel), 0x5410u);
                    } else {
                        A = __byte_perm(__byte_perm(mhi[0], mhi[1], sel), __byte_perm(mhi[2], mhi[3], sel), 0x5410u);
                        B = __byte_perm(__byte_perm(mhi[4], mhi[5], sel), __byte_perm(mhi[6], mhi[7], sel), 0x5410u);
                    }
#pragma unroll
                    for (int c = 0; c < 8; c++) {
                        const uint32_t k = (uint32_t)__popc(A & (0x01010101u << c)) + (uint32_t)__popc(B & (0x01010101u << c));
                        const uint32_t tot = __reduce_add_sync(0xffffffffu, k);
                        const int t = 8 * r + c;
                        if (lane == (t & 31)) { if (t < 32) mine0 = tot; else mine1 = tot; }
                    }
                }
                s_cnt[w][lane] = mine0;
                s_cnt[w][32 + lane] = mine1;
            }
            __syncthreads();
            // ---- (b) first slots ----------------------------------------------------------------------------------
            if (tid < 64) {
                const int t = tid;
                uint32_t run = 0;
#pragma unroll
                for (int k = 0; k < 8; k++) { const uint32_t c = s_cnt[k][t]; s_cnt[k][t] = run; run += c; }
                unsigned long long* st = p.st_exp + (size_t)g * 64 + t;
                if (goes_on && from_before) st_status(st, ST_AGG | (unsigned long long)run);
                unsigned long long prev = 0;
                if (from_before) {
                    // entries of this super-tile in the chunks before this one: back to the nearest inclusive prefix (the
                    // chunk the super-tile starts in publishes one at once), EXP_LB status words in flight per round trip
                    // -- a super-tile of the outdoor scene fills 76 chunks, most of them in flight in the same wave
                    constexpr int EXP_LB = 16;
                    const uint32_t g_first = cbeg / EXP_SEG;
                    uint32_t idx = g - 1;
                    bool done = false;
                    while (!done) {
                        unsigned long long sv[EXP_LB];
#pragma unroll
                        for (int k = 0; k < EXP_LB; k++)
                            sv[k] = (idx >= g_first + (uint32_t)k) ? ld_status(p.st_exp + (size_t)(idx - k) * 64 + t) : ST_INC;
#pragma unroll
                        for (int k = 0; k < EXP_LB; k++) {
                            if (done || (sv[k] >> 62) == 0) break;   // not published yet: poll again from here
                            prev += sv[k] & ST_MASK;
                            idx--;
                            done = (sv[k] >> 62) == 2;
                        }
                    }
                }
                if (goes_on) st_status(st, ST_INC | (prev + run));
                const uint32_t ty = Y0 + (uint32_t)(t >> 3), tx = X0 + (uint32_t)(t & 7);
                const bool inside = ty < (uint32_t)f.gy && tx < (uint32_t)f.gx;
                s_tb[t] = (inside ? p.ranges[ty * f.gx + tx] : 0u) + (uint32_t)prev;
                if (EXACT && !goes_on && inside) {       // the super-tile ends here: the exact length of this tile's list
                    p.tile_len[ty * f.gx + tx] = (uint32_t)prev + run;
                    out_counts[ty * f.gx + tx] = (uint32_t)prev + run;
                }
            }
            __syncthreads();
            // ---- (c) emit ------------------------------------------------------------------------------------------
            if (wq0 < q1) {
                const uint32_t n_sub = (min(q1 - wq0, 256u) + 31u) >> 5;
                const unsigned char* mb = reinterpret_cast<const unsigned char*>(&s_m[w][0][lane]);
#pragma unroll 1
                for (int r = 0; r < 8; r++) {
                    if (Y0 + (uint32_t)r >= (uint32_t)f.gy) break;
                    uint32_t slot[8];
                    {
                        const uint4 c0 = *reinterpret_cast<const uint4*>(&s_cnt[w][8 * r]), c1 = *reinterpret_cast<const uint4*>(&s_cnt[w][8 * r + 4]);
                        const uint4 b0 = *reinterpret_cast<const uint4*>(&s_tb[8 * r]), b1 = *reinterpret_cast<const uint4*>(&s_tb[8 * r + 4]);
                        slot[0] = c0.x + b0.x; slot[1] = c0.y + b0.y; slot[2] = c0.z + b0.z; slot[3] = c0.w + b0.w;
                        slot[4] = c1.x + b1.x; slot[5] = c1.y + b1.y; slot[6] = c1.z + b1.z; slot[7] = c1.w + b1.w;
                    }
#pragma unroll 1
                    for (uint32_t j = 0; j < n_sub; j++) {
                        const uint32_t rowbyte = mb[j * (32 * 8) + r];      // byte r of this lane's mask of sub-chunk j
                        if (!__any_sync(0xffffffffu, rowbyte != 0u)) continue;   // none of the 32 entries reaches this tile row
                        const uint32_t my_id = s_id[w][j][lane];
#pragma unroll
                        for (int c = 0; c < 8; c++) {
                            const bool hit = (rowbyte >> c) & 1u;
                            const unsigned bal = __ballot_sync(0xffffffffu, hit);
                            const uint32_t rank = __popc(bal & lt);
                            if (hit) {
                                GS_BOUND(slot[c] + rank, f.max_dup);
                                p.ids[slot[c] + rank] = my_id;
                            }
                            slot[c] += __popc(bal);
                        }
                    }
                }
            }
            // next piece: after the last one, the others in list order
            if (!last_done) { last_done = true; s = s_first; q0 = e0; }
            else {
                q0 = q1;
                if (q0 < last_q0) { do { s++; } while (__ldg(p.cranges + s + 1) <= q0); }
            }
            if (q0 >= last_q0) break;
            __syncthreads();                             // the next piece overwrites the shared arrays
        }
    }
}

void launch_expand(const Frame& f, const Pointers& p, uint32_t* out_tile_counts, int n_sm, cudaStream_t st, int* launches) {
    const long long cap_chunks = ((long long)f.max_dup + EXP_SEG - 1) / EXP_SEG;
    // three blocks per SM measured best (two to five tried): with more chunks in flight the look-back chains of the long
    // super-tile lists get deeper and the store streams of a tile list interleave more
    const dim3 grid(imin(cap_chunks > 0 ? cap_chunks : 1, (long long)n_sm * 3));
    if (f.tile_cull == 2) launch_pdl(expand_kernel<SUPER_SHIFT, true>, grid, dim3(EXP_THREADS), st, f, p, out_tile_counts);
    else launch_pdl(expand_kernel<SUPER_SHIFT, false>, grid, dim3(EXP_THREADS), st, f, p, out_tile_counts);
    (*launches)++;
}

// ------------------------------------------------------------------------------------------------------------
// Self-test of the hardware property radix_pass_kernel's ranking relies on (see its header): `rounds` back-to-back
// shared-memory atomicAdd per thread on a warp-private counter array return, for every key, exactly its stable rank
// in (round, lane) order -- checked against a shuffle-based count, with random digits drawn from `nbins` bins and a
// divergent subset of lanes every fourth iteration.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
atomic_order_selftest_kernel(unsigned long long* __restrict__ out, int iters, uint32_t seed, int nbins) {
    __shared__ uint32_t hist[8][256];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t s = seed ^ (blockIdx.x * 0x9E3779B9u) ^ (threadIdx.x * 0x85EBCA6Bu);
    unsigned long long bad = 0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int k = 0; k < 8; k++) hist[w][k * 32 + lane] = 0;
        __syncwarp();
        uint32_t d[8], r[8];
#pragma unroll
        for (int j = 0; j < 8; j++) { s = s * 1664525u + 1013904223u; d[j] = (s >> 16) % (uint32_t)nbins; }
        const bool act = (it & 3) != 3 || ((s >> 8) & 1u);
        if (act) {
#pragma unroll
            for (int j = 0; j < 8; j++) r[j] = atomicAdd(&hist[w][d[j]], 1u);
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 8; j++) {
            uint32_t cnt = 0;
            for (int jj = 0; jj <= j; jj++)
                for (int l = 0; l < 32; l++) {
                    const uint32_t od = __shfl_sync(0xffffffffu, d[jj], l);
                    const int oa = __shfl_sync(0xffffffffu, (int)act, l);
                    if (oa && od == d[j] && (jj < j || l < lane)) cnt++;
                }
            if (act && r[j] != cnt) bad++;
        }
        __syncwarp();
    }
    if (bad) atomicAdd(out, bad);
    if (threadIdx.x == 0) atomicAdd(out + 1, (unsigned long long)iters * 8ull * blockDim.x);
}

void launch_atomic_order_selftest(unsigned long long* out, int iters, uint32_t seed, int nbins, int n_sm, cudaStream_t st) {
    atomic_order_selftest_kernel<<<n_sm * 4, 256, 0, st>>>(out, iters, seed, nbins);
}

}  // namespace gs
