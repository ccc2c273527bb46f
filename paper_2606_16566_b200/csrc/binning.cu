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
#include "common.cuh"

namespace gs {

// ------------------------------------------------------------------------------------------------------------
// One stable radix pass over u64 elements on digit (key >> shift) & 255.  No payload: the id lives in the low
// 32 bits of the element.  OUT32: write only the low 32 bits (last tile pass -> sorted_ids).
// ------------------------------------------------------------------------------------------------------------
template <bool OUT32>
__global__ void __launch_bounds__(SORT_THREADS)
radix_pass_kernel(const unsigned long long* __restrict__ in, unsigned long long* __restrict__ out,
                  uint32_t* __restrict__ out32, const unsigned long long* __restrict__ n_ptr, int shift,
                  const uint32_t* __restrict__ ghist, unsigned long long* __restrict__ status,
                  uint32_t* __restrict__ tile_counter) {
    constexpr int NW = SORT_THREADS / 32;
    __shared__ unsigned long long s_sorted[SORT_TILE];
    __shared__ uint32_t s_hist[NW][257];
    __shared__ uint32_t s_bpos[257];
    __shared__ uint32_t s_gbase[256];
    __shared__ uint32_t s_gpos[256];
    __shared__ uint32_t s_scan[NW];
    __shared__ int s_tile;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned long long n = *n_ptr;
    {   // exclusive scan of the global digit histogram -> first output slot of every digit
        uint32_t tot;
        s_gbase[tid] = block_excl_scan_256(ghist[tid], s_scan, tot);
    }
    const unsigned lt_mask = (1u << lane) - 1u;
    while (true) {
        __syncthreads();
        if (tid == 0) s_tile = (int)atomicAdd(tile_counter, 1u);
        __syncthreads();
        const int tile = s_tile;
        const unsigned long long tile_base = (unsigned long long)tile * SORT_TILE;
        if (tile_base >= n) break;
        const uint32_t tile_n = (uint32_t)min((unsigned long long)SORT_TILE, n - tile_base);
        // ---- load (warp-striped: lane l of warp w takes w*512 + j*32 + l) ---------------------------------
        unsigned long long key[SORT_ITEMS];
        uint32_t rk[SORT_ITEMS];
#pragma unroll
        for (int j = 0; j < SORT_ITEMS; j++) {
            const uint32_t li = w * (32 * SORT_ITEMS) + j * 32 + lane;
            key[j] = (li < tile_n) ? in[tile_base + li] : ~0ull;
        }
        for (int k = lane; k < 257; k += 32) s_hist[w][k] = 0;
        __syncwarp();
        // ---- stable rank inside the warp: (round j, lane) order ------------------------------------------
#pragma unroll
        for (int j = 0; j < SORT_ITEMS; j++) {
            const uint32_t li = w * (32 * SORT_ITEMS) + j * 32 + lane;
            const uint32_t d = (li < tile_n) ? (uint32_t)((key[j] >> shift) & 255ull) : 256u;
            const unsigned peers = __match_any_sync(0xffffffffu, d);
            const int leader = __ffs(peers) - 1;
            uint32_t old = 0;
            if (lane == leader) {
                old = s_hist[w][d];
                s_hist[w][d] = old + __popc(peers);
            }
            old = __shfl_sync(0xffffffffu, old, leader);
            rk[j] = old + __popc(peers & lt_mask);
            __syncwarp();
        }
        __syncthreads();
        // ---- per digit: exclusive prefix over warps, block count, publish aggregate ------------------------
        uint32_t cnt = 0;
#pragma unroll
        for (int k = 0; k < NW; k++) {
            const uint32_t t = s_hist[k][tid];
            s_hist[k][tid] = cnt;
            cnt += t;
        }
        unsigned long long* st = status + (size_t)tile * 256 + tid;
        st_status(st, (tile == 0 ? ST_INC : ST_AGG) | (unsigned long long)cnt);
        uint32_t tot;
        const uint32_t bpos = block_excl_scan_256(cnt, s_scan, tot);  // contains __syncthreads
        s_bpos[tid] = bpos;
        if (tid == 0) {
            s_bpos[256] = tot;  // invalid (tail) elements sort behind every digit
            uint32_t c = 0;     // their per-warp offsets
            for (int k = 0; k < NW; k++) { const uint32_t t = s_hist[k][256]; s_hist[k][256] = c; c += t; }
        }
        __syncthreads();
        // ---- block-local reorder through shared memory ---------------------------------------------------
#pragma unroll
        for (int j = 0; j < SORT_ITEMS; j++) {
            const uint32_t li = w * (32 * SORT_ITEMS) + j * 32 + lane;
            const uint32_t d = (li < tile_n) ? (uint32_t)((key[j] >> shift) & 255ull) : 256u;
            s_sorted[s_bpos[d] + s_hist[w][d] + rk[j]] = key[j];
        }
        // ---- decoupled look-back for digit `tid` ---------------------------------------------------------
        unsigned long long excl = 0;
        if (tile > 0) {
            int idx = tile - 1;
            while (true) {
                unsigned long long s;
                do { s = ld_status(status + (size_t)idx * 256 + tid); } while ((s >> 62) == 0);
                excl += s & ST_MASK;
                if ((s >> 62) == 2 || idx == 0) break;
                idx--;
            }
            st_status(st, ST_INC | (excl + cnt));
        }
        s_gpos[tid] = s_gbase[tid] + (uint32_t)excl - bpos;
        __syncthreads();
        // ---- coalesced output: runs of equal digits are contiguous ---------------------------------------
#pragma unroll
        for (int j = 0; j < SORT_ITEMS; j++) {
            const uint32_t li = j * SORT_THREADS + tid;
            if (li < tile_n) {
                const unsigned long long k = s_sorted[li];
                const uint32_t d = (uint32_t)((k >> shift) & 255ull);
                const uint32_t pos = s_gpos[d] + li;
                if (OUT32) out32[pos] = (uint32_t)k;
                else out[pos] = k;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Tile grid: 2-D inclusive prefix of the difference grid -> tile counts; exclusive scan -> tile ranges, n_dup;
// digit histograms of the tile ids for the tile radix passes.  One block (the grid has <= 2^24 cells).
// ------------------------------------------------------------------------------------------------------------
constexpr int GRID_THREADS = 1024;
__global__ void __launch_bounds__(GRID_THREADS)
tile_grid_kernel(const Frame f, const Pointers p, uint32_t* __restrict__ counts /* out_tile_counts */) {
    __shared__ uint32_t s_hist[MAX_SORT_PASSES_TILE][256];
    __shared__ unsigned long long s_part[GRID_THREADS / 32];
    __shared__ unsigned long long s_total;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gw = f.gx + 1, gh = f.gy + 1;
    int* diff = p.diff;
    for (int k = tid; k < MAX_SORT_PASSES_TILE * 256; k += GRID_THREADS) (&s_hist[0][0])[k] = 0;
    // row-wise inclusive prefix, one warp per row, in place
    for (int y = w; y < gh; y += GRID_THREADS / 32) {
        int carry = 0;
        for (int x0 = 0; x0 < gw; x0 += 32) {
            const int x = x0 + lane;
            int v = (x < gw) ? diff[y * gw + x] : 0;
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
    for (int t = t0; t < t1; t++) sum += counts[t];
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
    __syncthreads();
    const unsigned long long total = s_total;
    const bool overflow = total > f.max_dup;
    unsigned long long run = s_part[w] + inc - sum;
    for (int t = t0; t < t1; t++) {
        const uint32_t c = counts[t];
        p.ranges[t] = overflow ? 0u : (uint32_t)run;
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

__global__ void __launch_bounds__(SCAN_THREADS)
scan_offsets_kernel(const Pointers p) {
    __shared__ uint32_t s_scan[SCAN_THREADS / 32];
    __shared__ int s_tile;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x;
    const unsigned long long n = p.ctrl->n_vis;
    const bool dead = p.ctrl->overflow != 0;
    while (true) {
        __syncthreads();
        if (tid == 0) s_tile = (int)atomicAdd(&p.ctrl->tile_counter[TC_SCAN], 1u);
        __syncthreads();
        const int tile = s_tile;
        const unsigned long long base_r = (unsigned long long)tile * SCAN_TILE;
        if (base_r >= n || dead) break;
        uint32_t tt[SCAN_ITEMS];
        uint32_t sum = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            const unsigned long long r = base_r + (unsigned long long)tid * SCAN_ITEMS + k;
            tt[k] = 0;
            if (r < n) {
                const uint32_t id = (uint32_t)p.gkeyA[r];
                tt[k] = rect_tiles(__ldg(p.per_g + id));
            }
            sum += tt[k];
        }
        uint32_t btotal;
        const uint32_t texcl = block_excl_scan_256(sum, s_scan, btotal);
        if (tid < 32) {
            if (tid == 0) st_status(p.st_scan + tile, (tile == 0 ? ST_INC : ST_AGG) | (unsigned long long)btotal);
            unsigned long long excl = 0;
            if (tile > 0) {
                excl = lookback_warp(p.st_scan, tile);
                if (tid == 0) st_status(p.st_scan + tile, ST_INC | (excl + btotal));
            }
            if (tid == 0) s_base = excl;
        }
        __syncthreads();
        unsigned long long off = s_base + texcl;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            const unsigned long long r = base_r + (unsigned long long)tid * SCAN_ITEMS + k;
            if (r < n) {
                p.dup_off[r] = (uint32_t)off;
                if (tt[k]) {  // chunk boundaries c*DUP_TILE that fall inside [off, off + tt)
                    const unsigned long long c0 = (off + DUP_TILE - 1) / DUP_TILE, c1 = (off + tt[k] - 1) / DUP_TILE;
                    for (unsigned long long c = c0; c <= c1; c++) p.chunk_start[c] = (uint32_t)r;
                }
            }
            off += tt[k];
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Duplication: output slot k belongs to the depth-ranked Gaussian r with off[r] <= k < off[r] + tiles_touched;
// its j = k - off[r]-th tile in row-major rect order is written as (tile << 32 | id).  Load-balanced by OUTPUT
// chunk (a splat covering thousands of tiles is spread over many blocks).
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(DUP_THREADS)
duplicate_kernel(const Frame f, const Pointers p, unsigned long long* __restrict__ ent) {
    __shared__ uint32_t s_off[DUP_TILE + 2];
    const int tid = threadIdx.x;
    const unsigned long long n = p.ctrl->n_dup_eff;
    const uint32_t n_vis = (uint32_t)p.ctrl->n_vis;
    for (unsigned long long chunk = blockIdx.x; chunk * DUP_TILE < n; chunk += gridDim.x) {
        const unsigned long long k0 = chunk * DUP_TILE;
        const uint32_t cn = (uint32_t)min((unsigned long long)DUP_TILE, n - k0);
        const uint32_t r0 = p.chunk_start[chunk];
        const uint32_t r1 = ((chunk + 1) * DUP_TILE < n) ? p.chunk_start[chunk + 1] : (n_vis - 1);
        const uint32_t nr = r1 - r0 + 1;  // <= DUP_TILE + 1 ranks can start inside one chunk
        __syncthreads();
        for (uint32_t k = tid; k < nr; k += DUP_THREADS) s_off[k] = p.dup_off[r0 + k];
        __syncthreads();
        const uint32_t lk0 = tid * DUP_ITEMS;
        if (lk0 < cn) {
            const uint32_t kk = (uint32_t)k0 + lk0;  // N_dup < 2^32
            // largest local rank with s_off <= kk
            uint32_t lo = 0, hi = nr - 1;
            while (lo < hi) {
                const uint32_t mid = (lo + hi + 1) >> 1;
                if (s_off[mid] <= kk) lo = mid; else hi = mid - 1;
            }
            uint32_t lr = lo;
            uint32_t id = (uint32_t)p.gkeyA[r0 + lr];
            uint4 pg = __ldg(p.per_g + id);
            uint32_t x0 = pg.x & 0xffffu, y0 = pg.x >> 16, wdt = (pg.y & 0xffffu) - x0;
            uint32_t end = s_off[lr] + rect_tiles(pg);
            unsigned long long outv[DUP_ITEMS];
#pragma unroll
            for (int q = 0; q < DUP_ITEMS; q++) {
                const uint32_t k = kk + q;
                if (lk0 + q < cn) {
                    while (k >= end) {  // advance to the rank owning slot k (every visible rank has >= 1 tile)
                        lr++;
                        id = (uint32_t)p.gkeyA[r0 + lr];
                        pg = __ldg(p.per_g + id);
                        x0 = pg.x & 0xffffu; y0 = pg.x >> 16; wdt = (pg.y & 0xffffu) - x0;
                        end = s_off[lr] + rect_tiles(pg);
                    }
                    const uint32_t j = k - s_off[lr];
                    const uint32_t ty = y0 + j / wdt, tx = x0 + j % wdt;
                    outv[q] = ((unsigned long long)(ty * (uint32_t)f.gx + tx) << 32) | id;
                } else {
                    outv[q] = 0;
                }
            }
            unsigned long long* dst = ent + k0 + lk0;
            if (lk0 + DUP_ITEMS <= cn) {
#pragma unroll
                for (int q = 0; q < DUP_ITEMS; q += 2)
                    *reinterpret_cast<ulonglong2*>(dst + q) = make_ulonglong2(outv[q], outv[q + 1]);
            } else {
                for (int q = 0; q < DUP_ITEMS && lk0 + q < cn; q++) dst[q] = outv[q];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// host-side launchers
// ------------------------------------------------------------------------------------------------------------
static int imin(long long a, long long b) { return (int)(a < b ? a : b); }

void launch_depth_sort(const Frame& f, const Pointers& p, int n_sm, cudaStream_t st, int* launches) {
    const long long cap_tiles = ((long long)f.P + SORT_TILE - 1) / SORT_TILE;
    const int grid = imin(cap_tiles > 0 ? cap_tiles : 1, (long long)n_sm * 4);
    unsigned long long* bufs[2] = {p.gkeyA, p.gkeyB};
    for (int pass = 0; pass < MAX_SORT_PASSES_DEPTH; pass++) {
        radix_pass_kernel<false><<<grid, SORT_THREADS, 0, st>>>(
            bufs[pass & 1], bufs[(pass + 1) & 1], nullptr, &p.ctrl->n_vis, 32 + 8 * pass, p.ctrl->depth_hist[pass],
            p.st_depth + (size_t)pass * p.n_depth_tiles * 256, &p.ctrl->tile_counter[TC_DEPTH0 + pass]);
        (*launches)++;
    }
}

void launch_tile_grid(const Frame& f, const Pointers& p, uint32_t* out_tile_counts, cudaStream_t st, int* launches) {
    tile_grid_kernel<<<1, GRID_THREADS, 0, st>>>(f, p, out_tile_counts);
    (*launches)++;
}

void launch_scan_offsets(const Frame& f, const Pointers& p, int n_sm, cudaStream_t st, int* launches) {
    const long long cap_tiles = ((long long)f.P + SCAN_TILE - 1) / SCAN_TILE;
    const int grid = imin(cap_tiles > 0 ? cap_tiles : 1, (long long)n_sm * 8);
    scan_offsets_kernel<<<grid, SCAN_THREADS, 0, st>>>(p);
    (*launches)++;
}

// Entries are first written into the buffer from which n_tile_passes ping-pong passes end in `ids`.
void launch_duplicate_and_tile_sort(const Frame& f, const Pointers& p, int n_sm, cudaStream_t st, int* launches,
                                    cudaEvent_t ev_after_duplicate) {
    const long long cap_chunks = ((long long)f.max_dup + DUP_TILE - 1) / DUP_TILE;
    const int dgrid = imin(cap_chunks > 0 ? cap_chunks : 1, (long long)n_sm * 8);
    duplicate_kernel<<<dgrid, DUP_THREADS, 0, st>>>(f, p, p.entA);
    (*launches)++;
    if (ev_after_duplicate) cudaEventRecord(ev_after_duplicate, st);
    const long long cap_tiles = ((long long)f.max_dup + SORT_TILE - 1) / SORT_TILE;
    const int grid = imin(cap_tiles > 0 ? cap_tiles : 1, (long long)n_sm * 4);
    unsigned long long* bufs[2] = {p.entA, p.entB};
    for (int pass = 0; pass < f.n_tile_passes; pass++) {
        const bool last = pass == f.n_tile_passes - 1;
        unsigned long long* status = p.st_tile + (size_t)pass * p.n_tile_tiles * 256;
        if (last)
            radix_pass_kernel<true><<<grid, SORT_THREADS, 0, st>>>(bufs[pass & 1], nullptr, p.ids, &p.ctrl->n_dup_eff,
                                                                  32 + 8 * pass, p.ctrl->tile_hist[pass], status,
                                                                  &p.ctrl->tile_counter[TC_TILE0 + pass]);
        else
            radix_pass_kernel<false><<<grid, SORT_THREADS, 0, st>>>(bufs[pass & 1], bufs[(pass + 1) & 1], nullptr,
                                                                   &p.ctrl->n_dup_eff, 32 + 8 * pass,
                                                                   p.ctrl->tile_hist[pass], status,
                                                                   &p.ctrl->tile_counter[TC_TILE0 + pass]);
        (*launches)++;
    }
}

}  // namespace gs
