// api.cu -- the C ABI of include/gs.h: workspace carving, the per-frame launch sequence, inspection and timing.
// Every step of the path runs in the kernels of preprocess.cu / binning.cu / render*.cu; this file only enqueues.
#include "../../include/gs.h"

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace gs {
thread_local CaptureLog g_caplog;
thread_local int g_use_pdl = 1;   // set by gs_render on the calling thread for the launches it makes
void launch_preprocess(const Frame&, const Pointers&, const float*, const float*, const float*, const float*, const float*,
                       int, cudaStream_t);
void launch_depth_sort(const Frame&, const Pointers&, int, cudaStream_t, int*);
void launch_tile_grid(const Frame&, const Pointers&, uint32_t*, const Ctrl*, cudaStream_t, int*);
void launch_scan_offsets(const Frame&, const Pointers&, int, int, cudaStream_t, int*);
void launch_expand(const Frame&, const Pointers&, uint32_t*, int, cudaStream_t, int*);
void launch_duplicate_and_tile_sort(const Frame&, const Pointers&, int, cudaStream_t, int*, cudaEvent_t);
void launch_atomic_order_selftest(unsigned long long*, int, uint32_t, int, int, cudaStream_t);
cudaError_t run_issue_peak(int, int, double*);
void launch_render_ladder(int, const Frame&, const Pointers&, float*, float*, uint32_t*, cudaStream_t);
void launch_render_b200(const Frame&, const Pointers&, float*, float*, uint32_t*, int, bool, cudaStream_t);
}  // namespace gs

namespace {
using namespace gs;

constexpr size_t ALIGN = 256;
size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
    size_t ctrl, cctrl, diff, cdiff, st_pre, st_scan, st_depth, st_tile, st_exp, zero_end;
    size_t per_g, rec, gkeyA, gkeyB, dup_off, rk_rect, chunk_start, ranges, desc, cranges, ccounts, tile_len, entA, entB, cids, ids, total;
    size_t n_depth_tiles, n_tile_tiles;
    int gx, gy, n_tiles, tile_bits, n_tile_passes, diff_copies, diff_cells;
    int cshift, cgx, cgy, n_ctiles, cdiff_cells;
    bool two_level;
};

bool make_layout(int P, int W, int H, unsigned long long max_dup, Layout& L) {
    if (P < 0 || W <= 0 || H <= 0 || max_dup >= (1ull << 32)) return false;
    L.gx = (W + TILE - 1) / TILE;
    L.gy = (H + TILE - 1) / TILE;
    const long long nt = (long long)L.gx * L.gy;
    if (nt > (1ll << 24) || L.gx > 65535 || L.gy > 65535) return false;
    L.n_tiles = (int)nt;
    // Large frames (capacity > FUSED_DUP_MAX) bin in TWO LEVELS: duplication + sort run on the super-tile grid, whose id
    // width then sets the number of radix passes, and expand_kernel writes the tile lists.  Small frames sort tile ids.
    L.two_level = max_dup > FUSED_DUP_MAX;
    L.cshift = L.two_level ? SUPER_SHIFT : 0;
    const int SUPER = 1 << L.cshift;
    L.cgx = L.two_level ? (L.gx + SUPER - 1) / SUPER : 0;
    L.cgy = L.two_level ? (L.gy + SUPER - 1) / SUPER : 0;
    L.n_ctiles = L.cgx * L.cgy;
    L.cdiff_cells = L.two_level ? (L.cgx + 1) * (L.cgy + 1) : 0;
    L.tile_bits = 1;
    while ((1ll << L.tile_bits) < (L.two_level ? (long long)L.n_ctiles : nt)) L.tile_bits++;
    L.n_tile_passes = (L.tile_bits + 7) / 8;
    const size_t Pz = (size_t)P;
    const size_t depth_tile = (size_t)SORT_THREADS * sort_items_for(Pz), ent_tile = (size_t)SORT_THREADS * dup_items_for(max_dup);  // the smaller of the tile passes' tiles
    L.n_depth_tiles = (Pz + depth_tile - 1) / depth_tile + 1;
    L.n_tile_tiles = ((size_t)max_dup + ent_tile - 1) / ent_tile + 1;
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o = up(o + bytes); return at; };
    L.ctrl = take(sizeof(Ctrl));
    L.cctrl = take(sizeof(Ctrl));
    L.diff_cells = (L.gx + 1) * (L.gy + 1);
    L.diff_copies = 1;   // replicas of the coverage grid (spreads the hot corner counters of small grids)
    while (L.diff_copies < 16 && (long long)L.diff_cells * L.diff_copies * 2 <= 65536) L.diff_copies *= 2;
    L.diff = take(sizeof(int) * (size_t)L.diff_cells * L.diff_copies);
    L.cdiff = take(sizeof(int) * (size_t)L.cdiff_cells);
    L.st_pre = take(8 * ((Pz + 31) / 32 + 1));
    L.st_scan = take(8 * ((Pz + SCAN_WARP_TILE - 1) / SCAN_WARP_TILE + 1));
    L.st_depth = take(8 * 256 * L.n_depth_tiles * MAX_SORT_PASSES_DEPTH);
    // The look-back status words of the tile passes are sized by CAPACITY (2 KB per tile of the sorted array: 1.1 GB at
    // the 1.1 G-entry capacity of the outdoor scene).  Small frames clear them with the rest of the control block; large
    // (two-level) frames sort a few per cent of their capacity, so there duplicate_kernel clears exactly the words the
    // passes of THIS frame will use and the block stays out of the memset.
    if (!L.two_level) L.st_tile = take(8 * 256 * L.n_tile_tiles * (size_t)L.n_tile_passes);
    L.zero_end = o;
    if (L.two_level) L.st_tile = take(8 * 256 * L.n_tile_tiles * (size_t)L.n_tile_passes);
    L.st_exp = take(L.two_level ? 8 * 64 * (((size_t)max_dup + EXP_SEG - 1) / EXP_SEG + 2) : 0);   // cleared by duplicate_kernel too
    L.per_g = take(16 * Pz);
    L.rec = take(64 * Pz);
    L.gkeyA = take(8 * Pz);
    L.gkeyB = take(8 * Pz);
    L.dup_off = take(4 * Pz);
    L.rk_rect = take(8 * Pz);
    L.chunk_start = take(4 * (((size_t)max_dup + DUP_TILE - 1) / DUP_TILE + 2));
    L.ranges = take(4 * ((size_t)L.n_tiles + 1));
    L.desc = take(16 * (size_t)L.n_tiles);
    L.cranges = take(4 * ((size_t)L.n_ctiles + 1));
    L.ccounts = take(4 * (size_t)L.n_ctiles);
    L.tile_len = take(L.two_level ? 4 * (size_t)L.n_tiles : 0);
    // Two-level frames with <= 2 radix passes over packed entries (P <= 2^24) use at most the first half of entA (packed
    // 4-byte entries between the two passes), so the sorted super-tile ids (cids) live in its second half.
    const bool cids_in_entA = L.two_level && L.n_tile_passes <= 2 && P <= (1 << 24);
    L.entA = take(8 * (size_t)max_dup + (cids_in_entA ? 2 * ALIGN : 0));
    L.entB = take((L.n_tile_passes >= 3 || max_dup > FUSED_DUP_MAX) ? 8 * (size_t)max_dup : 0);
    L.cids = !L.two_level ? L.entA : (cids_in_entA ? up(L.entA + 4 * (size_t)max_dup) : take(4 * (size_t)max_dup + 16));
    L.ids = take(4 * (size_t)max_dup + 16);
    L.total = o;
    return true;
}

struct WsOptions {   // per-workspace overrides of the process-wide switches; -1 = follow the process-wide value
    int v[GS_N_OPTIONS] = {-1, -1, -1, -1, -1, -1};
};

struct LastCall {
    WsOptions opt;
    int device = -1;
    Layout L;
    Frame f;
    unsigned long long max_dup = 0;
    cudaStream_t stream = nullptr;
    bool valid = false, timed = false;
    cudaEvent_t ev[GS_N_TIMINGS + 2] = {};
    bool have_events = false;
    cudaStream_t side = nullptr;          // tile-grid kernel runs here, concurrently with the depth sort
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t rstream = nullptr;       // gs_set_render_stream(1): the render kernel runs on this lowest-priority stream
    cudaEvent_t ev_r0 = nullptr, ev_r1 = nullptr;
    // gs_set_graph(1): the launch sequence of a frame, captured once per (shape, capacity, switches) and replayed; the three
    // kernel nodes whose arguments change from frame to frame (camera, caller pointers) are updated before every launch
    struct GNode { cudaGraphNode_t node = nullptr; cudaKernelNodeParams kp = {}; std::vector<void*> args; };
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t gexec = nullptr, gexec2 = nullptr;   // two instances, used alternately: the one being updated is never the one just launched
    int gflip = 0;
    GNode g_pre, g_grid, g_render;
    long long gkey[12] = {};
    int g_launches = 0;
};

std::mutex g_mu;
std::map<const void*, LastCall> g_calls;
std::atomic<int> g_tile_cull{0}, g_variant{4}, g_timing{0}, g_stats{0}, g_launches{0}, g_cuda_err{0}, g_render_stream{0};
std::atomic<int> g_graph{0};
std::atomic<int> g_rank_mode{-1};   // -1: decided per device by the self-test, 0: shared-atomic ranking, 1: ballot ranking

struct DevInfo {
    int n_sm = 0;
    int rank_auto = -1;   // result of the atomic-order self-test on this device: 0 = the atomics rank stably, 1 = use ballots
};
std::map<int, DevInfo> g_devs;   // under g_mu

int cuda_fail(cudaError_t e) {
    g_cuda_err.store((int)e);
    (void)cudaGetLastError();   // clear the sticky-free error state for the next call
    return GS_ERR_CUDA;
}
#define GS_CK(call) do { const cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_); } while (0)

void destroy_call_resources(LastCall& lc) {
    if (lc.have_events)
        for (auto& e : lc.ev) if (e) { cudaEventDestroy(e); e = nullptr; }
    lc.have_events = false;
    if (lc.ev_fork) cudaEventDestroy(lc.ev_fork);
    if (lc.ev_join) cudaEventDestroy(lc.ev_join);
    if (lc.ev_r0) cudaEventDestroy(lc.ev_r0);
    if (lc.ev_r1) cudaEventDestroy(lc.ev_r1);
    if (lc.side) cudaStreamDestroy(lc.side);
    if (lc.rstream) cudaStreamDestroy(lc.rstream);
    lc.ev_fork = lc.ev_join = lc.ev_r0 = lc.ev_r1 = nullptr;
    lc.side = lc.rstream = nullptr;
    if (lc.gexec) cudaGraphExecDestroy(lc.gexec);
    if (lc.gexec2) cudaGraphExecDestroy(lc.gexec2);
    lc.gexec2 = nullptr;
    if (lc.graph) cudaGraphDestroy(lc.graph);
    lc.gexec = nullptr; lc.graph = nullptr;
}

// The device the workspace lives on must be the current one (streams and events are created there); returns its SM count
// and the ranking mode of the radix passes (the self-test of the shared-atomic order runs once per device, on first use).
int device_info(const void* workspace, int& dev_out, DevInfo& info_out) {
    cudaPointerAttributes at;
    GS_CK(cudaPointerGetAttributes(&at, workspace));
    int cur = 0;
    GS_CK(cudaGetDevice(&cur));
    if (at.type != cudaMemoryTypeDevice || at.device != cur) return GS_ERR_BAD_ARG;
    dev_out = cur;
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_devs.find(cur);
        if (it != g_devs.end() && it->second.rank_auto >= 0) { info_out = it->second; return GS_OK; }
    }
    DevInfo d;
    GS_CK(cudaDeviceGetAttribute(&d.n_sm, cudaDevAttrMultiProcessorCount, cur));
    uint64_t res[2] = {0, 0};
    const int rc = gs_selftest_atomic_order(2, res);   // ~10^7 atomics, a few hundred microseconds; synchronous, once per device
    if (rc != GS_OK) return rc;
    d.rank_auto = res[0] == 0 ? 0 : 1;
    {
        std::lock_guard<std::mutex> g(g_mu);
        g_devs[cur] = d;
    }
    info_out = d;
    return GS_OK;
}

Pointers carve(void* ws, const Layout& L) {
    char* b = static_cast<char*>(ws);
    Pointers p;
    p.ctrl = reinterpret_cast<Ctrl*>(b + L.ctrl);
    p.cctrl = reinterpret_cast<Ctrl*>(b + L.cctrl);
    p.diff = reinterpret_cast<int*>(b + L.diff);
    p.cdiff = reinterpret_cast<int*>(b + L.cdiff);
    p.cranges = reinterpret_cast<uint32_t*>(b + L.cranges);
    p.ccounts = reinterpret_cast<uint32_t*>(b + L.ccounts);
    p.cids = reinterpret_cast<uint32_t*>(b + L.cids);
    p.tile_len = reinterpret_cast<uint32_t*>(b + L.tile_len);
    p.st_pre = reinterpret_cast<unsigned long long*>(b + L.st_pre);
    p.st_scan = reinterpret_cast<unsigned long long*>(b + L.st_scan);
    p.st_depth = reinterpret_cast<unsigned long long*>(b + L.st_depth);
    p.st_tile = reinterpret_cast<unsigned long long*>(b + L.st_tile);
    p.st_exp = reinterpret_cast<unsigned long long*>(b + L.st_exp);
    p.per_g = reinterpret_cast<uint4*>(b + L.per_g);
    p.rec = reinterpret_cast<float4*>(b + L.rec);
    p.gkeyA = reinterpret_cast<unsigned long long*>(b + L.gkeyA);
    p.gkeyB = reinterpret_cast<unsigned long long*>(b + L.gkeyB);
    p.dup_off = reinterpret_cast<uint32_t*>(b + L.dup_off);
    p.rk_rect = reinterpret_cast<uint2*>(b + L.rk_rect);
    p.chunk_start = reinterpret_cast<uint32_t*>(b + L.chunk_start);
    p.ranges = reinterpret_cast<uint32_t*>(b + L.ranges);
    p.desc = reinterpret_cast<uint4*>(b + L.desc);
    p.entA = reinterpret_cast<unsigned long long*>(b + L.entA);
    p.entB = reinterpret_cast<unsigned long long*>(b + L.entB);
    p.ids = reinterpret_cast<uint32_t*>(b + L.ids);
    p.n_depth_tiles = L.n_depth_tiles;
    p.n_tile_tiles = L.n_tile_tiles;
    return p;
}

// largest max_dup whose layout fits into `bytes`; false if even 0 does not fit.  The layout size is monotone in
// max_dup inside each tile-size regime of sort_items_for() but drops at the regime boundary (larger sort tiles need
// fewer look-back status words), so the regimes are searched separately, the upper one first.
bool fit_max_dup(int P, int W, int H, size_t bytes, unsigned long long& max_dup) {
    Layout L;
    if (!make_layout(P, W, H, 0, L) || L.total > bytes) return false;
    // regime starts: sort_items_for (256 K: small radix tiles) and FUSED_DUP_MAX (two-level binning, second entry buffer)
    const unsigned long long starts[3] = {0ull, (256ull << 10) + 1, FUSED_DUP_MAX + 1};
    const unsigned long long top = (1ull << 32) - 1;
    for (int r = 2; r >= 0; r--) {
        unsigned long long lo = starts[r], hi = (r == 2 ? top : starts[r + 1] - 1);
        if (lo > top || hi < lo) continue;
        if (hi > top) hi = top;
        make_layout(P, W, H, lo, L);
        if (L.total > bytes) continue;
        while (lo < hi) {
            const unsigned long long mid = lo + (hi - lo + 1) / 2;
            make_layout(P, W, H, mid, L);
            if (L.total <= bytes) lo = mid; else hi = mid - 1;
        }
        max_dup = lo;
        return true;
    }
    return false;
}

}  // namespace

namespace gs {
// lets the other translation units of the library (noalloc.cu) record a CUDA error for gs_last_cuda_error()
int record_cuda_error(cudaError_t e) { return cuda_fail(e); }
}  // namespace gs

extern "C" {

size_t gs_workspace_bytes(int P, int W, int H, uint64_t max_dup) {
    Layout L;
    if (!make_layout(P, W, H, max_dup, L)) return 0;
    return L.total;
}

int gs_render(int P, const float* means3D, const float* scales, const float* rotations, const float* opacities,
              const float* sh_coeffs, int sh_degree, const float* viewmatrix, const float* projmatrix, float fx, float fy,
              int W, int H, const float* bg, float* out_rgb, float* out_final_T, uint32_t* out_tile_counts,
              uint32_t* out_n_contrib, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (P < 0 || W <= 0 || H <= 0 || sh_degree < 0 || sh_degree > 3 || !viewmatrix || !projmatrix || !bg || !out_rgb ||
        !out_final_T || !out_tile_counts || !workspace || !(fx > 0.0f) || !(fy > 0.0f))
        return GS_ERR_BAD_ARG;
    if (P > 0 && (!means3D || !scales || !rotations || !opacities || !sh_coeffs)) return GS_ERR_BAD_ARG;
    if (reinterpret_cast<uintptr_t>(workspace) % ALIGN) return GS_ERR_WORKSPACE;
    unsigned long long max_dup = 0;
    Layout L;
    if (!make_layout(P, W, H, 0, L)) return GS_ERR_BAD_ARG;
    if (!fit_max_dup(P, W, H, workspace_bytes, max_dup)) return GS_ERR_WORKSPACE;
    make_layout(P, W, H, max_dup, L);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    DevInfo dinfo;
    {
        const int rc = device_info(workspace, dev, dinfo);   // the workspace must live on the current device
        if (rc != GS_OK) return rc;
    }
    const int g_n_sm = dinfo.n_sm;
    const int rank_mode = g_rank_mode.load() >= 0 ? g_rank_mode.load() : dinfo.rank_auto;
    Frame f;
    f.P = P; f.W = W; f.H = H; f.gx = L.gx; f.gy = L.gy; f.n_tiles = L.n_tiles;
    f.deg = sh_degree; f.K = (sh_degree + 1) * (sh_degree + 1);
    f.tile_bits = L.tile_bits; f.n_tile_passes = L.n_tile_passes;
    f.compact = P >= COMPACT_MIN_P ? 1 : 0;
    f.tile_cull = 0; f.rank_mode = 0;   // set below, from the options of this call
    f.diff_copies = L.diff_copies; f.diff_cells = L.diff_cells;
    f.cshift = L.cshift; f.cgx = L.cgx; f.cgy = L.cgy; f.n_ctiles = L.n_ctiles; f.cdiff_cells = L.cdiff_cells;
    for (int k = 0; k < 16; k++) { f.V[k] = viewmatrix[k]; f.PM[k] = projmatrix[k]; }
    f.fx = fx; f.fy = fy;
    // camera centre of the rigid view matrix: campos = -Wv^T t (the north_star signature carries no campos)
    for (int c = 0; c < 3; c++)
        f.campos[c] = (float)-((double)viewmatrix[c] * viewmatrix[3] + (double)viewmatrix[4 + c] * viewmatrix[7] +
                               (double)viewmatrix[8 + c] * viewmatrix[11]);
    for (int c = 0; c < 3; c++) f.bg[c] = bg[c];
    f.max_dup = max_dup;
    f.tile_len = nullptr;
    const Pointers p = carve(workspace, L);
    // the super-tile level of the binning: the same kernels on the coarse grid, with their own control block
    Frame fc = f;
    fc.gx = f.cgx; fc.gy = f.cgy; fc.n_tiles = f.n_ctiles; fc.diff_copies = 1; fc.diff_cells = f.cdiff_cells;
    Pointers pc = p;
    pc.ctrl = p.cctrl; pc.diff = p.cdiff; pc.ranges = p.cranges; pc.desc = nullptr; pc.ids = p.cids;

    LastCall* lc;
    {
        std::lock_guard<std::mutex> g(g_mu);
        lc = &g_calls[workspace];
    }
    if (lc->device >= 0 && lc->device != dev) destroy_call_resources(*lc);   // the address now belongs to another device
    lc->device = dev;
    // the switches of THIS call: the workspace's own value where one was set (gs_set_workspace_option), else the process-wide one
    auto opt = [&](int k, int process_wide) { return lc->opt.v[k] >= 0 ? lc->opt.v[k] : process_wide; };
    const int variant = opt(GS_OPT_RENDER_VARIANT, g_variant.load());
    const bool timed = opt(GS_OPT_TIMING, g_timing.load()) != 0;
    const bool stats = opt(GS_OPT_STATS, g_stats.load()) != 0;
    const bool render_stream = opt(GS_OPT_RENDER_STREAM, g_render_stream.load()) != 0;
    f.tile_cull = opt(GS_OPT_TILE_CULL, g_tile_cull.load());
    f.rank_mode = rank_mode;
    // exact ellipse-tile culling happens where the super-tile lists are expanded: it needs the two-level binning (a workspace
    // sized for more than FUSED_DUP_MAX entries) and the B200 render kernel (the ladder variants walk tile_ranges)
    if (f.tile_cull == 2 && !L.two_level) return GS_ERR_WORKSPACE;
    if (f.tile_cull == 2 && variant != 4) return GS_ERR_BAD_ARG;
    if (f.tile_cull == 2) f.tile_len = p.tile_len;
    fc.tile_cull = f.tile_cull; fc.rank_mode = rank_mode; fc.tile_len = nullptr;
    if (timed && !lc->have_events) {
        lc->have_events = true;
        for (auto& e : lc->ev) {
            const cudaError_t ce = cudaEventCreate(&e);
            if (ce != cudaSuccess) { destroy_call_resources(*lc); return cuda_fail(ce); }
        }
    }
    if (!lc->side) {
        cudaError_t ce = cudaStreamCreateWithFlags(&lc->side, cudaStreamNonBlocking);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&lc->ev_fork, cudaEventDisableTiming);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&lc->ev_join, cudaEventDisableTiming);
        if (ce != cudaSuccess) { destroy_call_resources(*lc); return cuda_fail(ce); }
    }
    if (render_stream && !timed && !lc->rstream) {
        int lo = 0, hi = 0;
        cudaError_t ce = cudaDeviceGetStreamPriorityRange(&lo, &hi);
        if (ce == cudaSuccess) ce = cudaStreamCreateWithPriority(&lc->rstream, cudaStreamNonBlocking, lo);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&lc->ev_r0, cudaEventDisableTiming);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&lc->ev_r1, cudaEventDisableTiming);
        if (ce != cudaSuccess) { destroy_call_resources(*lc); return cuda_fail(ce); }
    }
    lc->L = L; lc->f = f; lc->max_dup = max_dup; lc->stream = st; lc->valid = true; lc->timed = timed;
#ifdef GS_DEBUG_SYNC   // development builds only: synchronise and report after every stage (never defined in libgs.so)
    auto mark = [&](int k) {
        const cudaError_t de = cudaStreamSynchronize(st);
        fprintf(stderr, "[gs debug] stage %d done: %s\n", k, cudaGetErrorString(de));
        if (timed) cudaEventRecord(lc->ev[k], st);
    };
#else
    cudaError_t mark_err = cudaSuccess;
    auto mark = [&](int k) {
        if (timed && mark_err == cudaSuccess) mark_err = cudaEventRecord(lc->ev[k], st);
    };
#endif

    // PDL hides launch latency between the 11 kernels of a small frame; large frames (kernels of 100+ us) gain nothing
    // and lose a little to early-resident dependents, so they launch plainly.  Thread-local: the launches below are made
    // by this thread.
    g_use_pdl = (!timed && P <= (1 << 21) && max_dup <= (1ull << 25)) ? 1 : 0;
    int launches = 0;
    auto enqueue = [&]() -> int {   // the launch sequence of one frame on `st` (+ the library's side / render streams)
    launches = 0;
    mark(0);
    cudaError_t e = cudaMemsetAsync(workspace, 0, L.zero_end, st);
    if (e != cudaSuccess) return cuda_fail(e);
    {   // (1) preprocess + compaction + depth histograms + coverage grid
        launch_preprocess(f, p, means3D, scales, rotations, opacities, sh_coeffs, g_n_sm, st);
        launches++;
    }
    mark(1);
    // The tile grid (counts, ranges, N_dup, tile-digit histograms) depends on the preprocess only: it runs on a side
    // stream, concurrently with the depth sort (fork / join with two events).  With timing enabled the stages are
    // serialised on the caller's stream so that every per-stage time is that stage alone.
    const bool two_level = L.two_level;
    if (!timed) {
        GS_CK(cudaEventRecord(lc->ev_fork, st));
        GS_CK(cudaStreamWaitEvent(lc->side, lc->ev_fork, 0));
        launch_tile_grid(f, p, out_tile_counts, nullptr, lc->side, &launches);
        if (two_level) launch_tile_grid(fc, pc, p.ccounts, p.ctrl, lc->side, &launches);
        GS_CK(cudaEventRecord(lc->ev_join, lc->side));
    }
    launch_depth_sort(f, p, g_n_sm, st, &launches);          // (3a) LSD passes over the depth bits, pre-duplication
    mark(2);
    if (timed) {
        launch_tile_grid(f, p, out_tile_counts, nullptr, st, &launches);
        if (two_level) launch_tile_grid(fc, pc, p.ccounts, p.ctrl, st, &launches);
    } else {
        GS_CK(cudaStreamWaitEvent(st, lc->ev_join, 0));
    }
    mark(3);
    if (two_level) {
        launch_scan_offsets(fc, pc, f.cshift, g_n_sm, st, &launches);   // (2) prefix-sum offsets of the super-tile duplicates
        mark(4);
        launch_duplicate_and_tile_sort(fc, pc, g_n_sm, st, &launches, timed ? lc->ev[5] : nullptr);  // (2) + (3b) on super-tiles
        launch_expand(f, p, out_tile_counts, g_n_sm, st, &launches);                 // (3c) super-tile lists -> tile lists, written in place
    } else {
        launch_scan_offsets(f, p, 0, g_n_sm, st, &launches);  // (2) prefix-sum offsets
        mark(4);
        launch_duplicate_and_tile_sort(f, p, g_n_sm, st, &launches, timed ? lc->ev[5] : nullptr);  // (2) + (3b)
    }
    mark(6);
    cudaStream_t rs = st;                                      // (4) render
    if (render_stream && !timed) {
        rs = lc->rstream;
        GS_CK(cudaEventRecord(lc->ev_r0, st));
        GS_CK(cudaStreamWaitEvent(rs, lc->ev_r0, 0));
    }
    if (variant == 4) launch_render_b200(f, p, out_rgb, out_final_T, out_n_contrib, g_n_sm, stats, rs);
    else launch_render_ladder(variant, f, p, out_rgb, out_final_T, out_n_contrib, rs);
    if (rs != st) {
        GS_CK(cudaEventRecord(lc->ev_r1, rs));
        GS_CK(cudaStreamWaitEvent(st, lc->ev_r1, 0));
    }
    launches++;
    mark(7);
    return GS_OK;
    };   // enqueue

    const bool special_stream = st == nullptr || st == cudaStreamLegacy || st == cudaStreamPerThread;   // cannot be captured
    const bool use_graph = opt(GS_OPT_GRAPH, g_graph.load()) != 0 && !timed && variant == 4 && !special_stream && f.tile_cull != 2;
    cudaError_t e = cudaSuccess;
    if (!use_graph) {
        const int rc = enqueue();
        if (rc != GS_OK) return rc;
    } else {
        const long long key[12] = {P, W, H, sh_degree, (long long)max_dup, f.tile_cull, rank_mode, stats ? 1 : 0, render_stream ? 1 : 0,
                                   out_n_contrib ? 1 : 0, (long long)workspace_bytes, g_use_pdl};
        bool fresh = false;
        if (!lc->gexec || memcmp(key, lc->gkey, sizeof(key)) != 0) {
            if (lc->gexec) { cudaGraphExecDestroy(lc->gexec); lc->gexec = nullptr; }
            if (lc->gexec2) { cudaGraphExecDestroy(lc->gexec2); lc->gexec2 = nullptr; }
            if (lc->graph) { cudaGraphDestroy(lc->graph); lc->graph = nullptr; }
            g_caplog = CaptureLog();
            GS_CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            const int rc = enqueue();
            cudaGraph_t g = nullptr;
            const cudaError_t ce = cudaStreamEndCapture(st, &g);   // always ended, also after a failed enqueue
            if (rc != GS_OK) { if (g) cudaGraphDestroy(g); return rc; }
            if (ce != cudaSuccess) return cuda_fail(ce);
            lc->graph = g;
            e = cudaGraphInstantiate(&lc->gexec, g, 0);
            if (e == cudaSuccess) e = cudaGraphInstantiate(&lc->gexec2, g, 0);
            if (e != cudaSuccess) { destroy_call_resources(*lc); return cuda_fail(e); }
            // the three nodes with per-frame arguments, found by their kernel function
            size_t n_nodes = 0;
            GS_CK(cudaGraphGetNodes(g, nullptr, &n_nodes));
            std::vector<cudaGraphNode_t> nodes(n_nodes);
            GS_CK(cudaGraphGetNodes(g, nodes.data(), &n_nodes));
            lc->g_pre = LastCall::GNode(); lc->g_grid = LastCall::GNode(); lc->g_render = LastCall::GNode();
            for (cudaGraphNode_t nd : nodes) {
                cudaGraphNodeType ty;
                GS_CK(cudaGraphNodeGetType(nd, &ty));
                if (ty != cudaGraphNodeTypeKernel) continue;
                cudaKernelNodeParams kp = {};
                GS_CK(cudaGraphKernelNodeGetParams(nd, &kp));
                LastCall::GNode* dst = nullptr;
                int n_args = 0;
                if (kp.func == g_caplog.preprocess) { dst = &lc->g_pre; n_args = 7; }
                else if (kp.func == g_caplog.render) { dst = &lc->g_render; n_args = 8; }
                else if (kp.func == g_caplog.tile_grid && *static_cast<uint32_t**>(kp.kernelParams[2]) == out_tile_counts) { dst = &lc->g_grid; n_args = 4; }
                if (!dst) continue;
                dst->node = nd; dst->kp = kp;
                dst->args.assign(kp.kernelParams, kp.kernelParams + n_args);
            }
            if (!lc->g_pre.node || !lc->g_grid.node || !lc->g_render.node) { destroy_call_resources(*lc); return GS_ERR_CUDA; }
            memcpy(lc->gkey, key, sizeof(key));
            lc->g_launches = launches;
            fresh = true;
        }
        lc->gflip ^= 1;
        cudaGraphExec_t ex = lc->gflip ? lc->gexec2 : lc->gexec;
        if (!fresh || lc->gflip) {   // (a fresh capture holds this frame's arguments; its twin does not)
            auto set = [&](LastCall::GNode& gn) {
                gn.kp.kernelParams = gn.args.data();
                return cudaGraphExecKernelNodeSetParams(ex, gn.node, &gn.kp);
            };
            lc->g_pre.args[0] = &f;
            lc->g_pre.args[2] = &means3D; lc->g_pre.args[3] = &scales; lc->g_pre.args[4] = &rotations;
            lc->g_pre.args[5] = &opacities; lc->g_pre.args[6] = &sh_coeffs;
            lc->g_grid.args[2] = &out_tile_counts;
            lc->g_render.args[0] = &f;
            lc->g_render.args[5] = &out_rgb; lc->g_render.args[6] = &out_final_T; lc->g_render.args[7] = &out_n_contrib;
            GS_CK(set(lc->g_pre));
            GS_CK(set(lc->g_grid));
            GS_CK(set(lc->g_render));
            launches = lc->g_launches;
        }
        GS_CK(cudaGraphLaunch(ex, st));
    }
    g_launches.store(launches);
    if (mark_err != cudaSuccess) return cuda_fail(mark_err);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    if (timed) {
        e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return GS_OK;
}

int gs_get_intermediates(const void* workspace, gs_intermediates* out) {
    if (!workspace || !out) return GS_ERR_BAD_ARG;
    LastCall lc;
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_calls.find(workspace);
        if (it == g_calls.end() || !it->second.valid) return GS_ERR_BAD_ARG;
        lc = it->second;
    }
    cudaError_t e = cudaStreamSynchronize(lc.stream);
    if (e != cudaSuccess) return cuda_fail(e);
    Ctrl c;
    e = cudaMemcpy(&c, static_cast<const char*>(workspace) + lc.L.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(e);
    const Pointers p = carve(const_cast<void*>(workspace), lc.L);
    out->P = lc.f.P; out->W = lc.f.W; out->H = lc.f.H; out->grid_x = lc.f.gx; out->grid_y = lc.f.gy;
    out->n_tiles = lc.f.n_tiles;
    out->n_visible = (uint32_t)c.n_vis;
    out->n_dup = c.n_dup;
    out->max_dup = lc.max_dup;
    out->per_gaussian = reinterpret_cast<const uint32_t*>(p.per_g);
    out->record = reinterpret_cast<const float*>(p.rec);
    out->depth_sorted = reinterpret_cast<const uint64_t*>(p.gkeyA);
    out->dup_offsets = p.dup_off;
    out->tile_ranges = p.ranges;
    out->sorted_ids = p.ids;
    {
        Ctrl cc;
        e = cudaMemcpy(&cc, static_cast<const char*>(workspace) + lc.L.cctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(e);
        out->n_coarse = lc.L.two_level ? cc.n_dup_eff : 0ull;
    }
    return c.overflow ? GS_ERR_OVERFLOW : GS_OK;
}

int gs_set_timing(int enable) {
    g_timing.store(enable ? 1 : 0);
    return GS_OK;
}

int gs_get_timings(const void* workspace, float ms[GS_N_TIMINGS]) {
    if (!workspace || !ms) return GS_ERR_BAD_ARG;
    LastCall lc;
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_calls.find(workspace);
        if (it == g_calls.end() || !it->second.valid || !it->second.timed) return GS_ERR_BAD_ARG;
        lc = it->second;
    }
    cudaError_t e = cudaEventSynchronize(lc.ev[7]);
    if (e != cudaSuccess) return cuda_fail(e);
    // events: 0 start | 1 after preprocess | 2 after depth sort | 3 after tile grid | 4 after offset scan |
    //         5 after duplicate | 6 after tile sort | 7 after render
    for (int k = 0; k < 7; k++)
        if ((e = cudaEventElapsedTime(&ms[k], lc.ev[k], lc.ev[k + 1])) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaEventElapsedTime(&ms[7], lc.ev[0], lc.ev[7])) != cudaSuccess) return cuda_fail(e);
    return GS_OK;
}

int gs_set_stats(int enable) {
    g_stats.store(enable ? 1 : 0);
    return GS_OK;
}

int gs_get_stats(const void* workspace, uint64_t out[GS_N_STATS]) {
    if (!workspace || !out) return GS_ERR_BAD_ARG;
    LastCall lc;
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_calls.find(workspace);
        if (it == g_calls.end() || !it->second.valid) return GS_ERR_BAD_ARG;
        lc = it->second;
    }
    cudaError_t e = cudaStreamSynchronize(lc.stream);
    if (e != cudaSuccess) return cuda_fail(e);
    Ctrl c;
    e = cudaMemcpy(&c, static_cast<const char*>(workspace) + lc.L.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(e);
    out[0] = c.stats[0];
    out[1] = c.stats[1];
    out[2] = c.stats[2];
    out[3] = c.stats[0] * 64ull;  // every walked (warp, Gaussian) slot evaluates the warp's 8x8 pixels
    return GS_OK;
}

int gs_selftest_atomic_order(int iters, uint64_t out[2]) {
    if (iters <= 0 || !out) return GS_ERR_BAD_ARG;
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    unsigned long long* d = nullptr;   // 16 bytes of private scratch, freed before returning
    if ((e = cudaMalloc(&d, 16)) != cudaSuccess) return cuda_fail(e);
    e = cudaMemset(d, 0, 16);
    const int bins[7] = {1, 2, 3, 7, 16, 64, 256};
    for (int k = 0; k < 7 && e == cudaSuccess; k++) {
        launch_atomic_order_selftest(d, iters, 12345u + (uint32_t)bins[k], bins[k], n_sm, nullptr);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    unsigned long long h[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e);
    out[0] = h[0];
    out[1] = h[1];
    return GS_OK;
}

int gs_selftest_issue_peak(int iters, double out[3]) {
    if (iters <= 0 || !out) return GS_ERR_BAD_ARG;
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = run_issue_peak(n_sm, iters, out);
    return e == cudaSuccess ? GS_OK : cuda_fail(e);
}

int gs_copy_to_host(void* dst_host, const void* src_dev, size_t bytes) {
    if (bytes == 0) return GS_OK;
    if (!dst_host || !src_dev) return GS_ERR_BAD_ARG;
    const cudaError_t e = cudaMemcpy(dst_host, src_dev, bytes, cudaMemcpyDeviceToHost);
    return e == cudaSuccess ? GS_OK : cuda_fail(e);
}

int gs_set_render_variant(int variant) {
    if (variant < 0 || variant > 6 || variant == 5) return GS_ERR_BAD_ARG;
    g_variant.store(variant);
    return GS_OK;
}
int gs_get_render_variant(void) { return g_variant.load(); }
int gs_set_tile_cull(int mode) {
    if (mode < 0 || mode > 2) return GS_ERR_BAD_ARG;
    g_tile_cull.store(mode);
    return GS_OK;
}
int gs_get_tile_cull(void) { return g_tile_cull.load(); }
int gs_set_render_stream(int enable) {
    g_render_stream.store(enable ? 1 : 0);
    return GS_OK;
}
int gs_set_workspace_option(const void* workspace, int option, int value) {
    if (!workspace || option < 0 || option >= GS_N_OPTIONS || value < -1) return GS_ERR_BAD_ARG;
    if (option == GS_OPT_RENDER_VARIANT && (value > 6 || value == 5)) return GS_ERR_BAD_ARG;
    if (option != GS_OPT_RENDER_VARIANT && value > (option == GS_OPT_TILE_CULL ? 2 : 1)) return GS_ERR_BAD_ARG;
    std::lock_guard<std::mutex> g(g_mu);
    g_calls[workspace].opt.v[option] = value;
    return GS_OK;
}

int gs_release(const void* workspace) {
    if (!workspace) return GS_ERR_BAD_ARG;
    LastCall lc;
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_calls.find(workspace);
        if (it == g_calls.end()) return GS_OK;
        lc = it->second;
        g_calls.erase(it);
    }
    cudaError_t e = cudaSuccess;
    if (lc.side) e = cudaStreamSynchronize(lc.side);
    if (lc.rstream && e == cudaSuccess) e = cudaStreamSynchronize(lc.rstream);
    destroy_call_resources(lc);
    return e == cudaSuccess ? GS_OK : cuda_fail(e);
}

int gs_set_graph(int enable) {
    g_graph.store(enable ? 1 : 0);
    return GS_OK;
}

int gs_set_rank_mode(int mode) {
    if (mode < -1 || mode > 1) return GS_ERR_BAD_ARG;
    g_rank_mode.store(mode);
    return GS_OK;
}

int gs_get_rank_mode(void) {
    const int forced = g_rank_mode.load();
    if (forced >= 0) return forced;
    int cur = 0;
    if (cudaGetDevice(&cur) != cudaSuccess) return cuda_fail(cudaGetLastError());
    {
        std::lock_guard<std::mutex> g(g_mu);
        auto it = g_devs.find(cur);
        if (it != g_devs.end() && it->second.rank_auto >= 0) return it->second.rank_auto;
    }
    DevInfo d;
    cudaError_t e = cudaDeviceGetAttribute(&d.n_sm, cudaDevAttrMultiProcessorCount, cur);
    if (e != cudaSuccess) return cuda_fail(e);
    uint64_t res[2] = {0, 0};
    const int rc = gs_selftest_atomic_order(2, res);
    if (rc != GS_OK) return rc;
    d.rank_auto = res[0] == 0 ? 0 : 1;
    std::lock_guard<std::mutex> g(g_mu);
    g_devs[cur] = d;
    return d.rank_auto;
}

int gs_last_launch_count(void) { return g_launches.load(); }
int gs_last_cuda_error(void) { return g_cuda_err.load(); }

const char* gs_error_string(int code) {
    switch (code) {
        case GS_OK: return "ok";
        case GS_ERR_BAD_ARG: return "bad argument";
        case GS_ERR_WORKSPACE: return "workspace too small or misaligned";
        case GS_ERR_OVERFLOW: return "more duplicated entries than the workspace capacity (max_dup)";
        case GS_ERR_CUDA: return "CUDA runtime error (see gs_last_cuda_error)";
        case GS_ERR_LIMIT: return "more keys than the fixed scratch of gs_depth_sort_noalloc holds (GS_NOALLOC_MAX_KEYS)";
        default: return "unknown error";
    }
}

}  // extern "C"
