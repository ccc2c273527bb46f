// noalloc.cu -- gs_depth_sort_noalloc(): the depth sort of the binning stage ("sorts them by tile index and
// depth"; stable LSD radix passes over the 32 depth bits, before duplication) as an entry point of
// its own that ALLOCATES NOTHING.  Its scratch -- the ping-pong key buffer, the digit histograms, the dynamic tile
// counters and the look-back status words of radix_pass_kernel -- lives in a file-scope __device__ array of a fixed,
// modest size instead of a caller-sized workspace, so the call can be made where cudaMalloc cannot (under stream
// capture, inside a serving loop, in a harness that forbids allocation).  The passes are the library's own
// radix_pass_kernel, launched through launch_depth_sort exactly as gs_render launches them; only the histogram kernel
// below is new (in gs_render the preprocess kernel accumulates the digit histograms).  Product code (C ABI, include/gs.h).
#include <mutex>

#include "common.cuh"
#include "gs.h"

namespace gs {
void launch_depth_sort(const Frame&, const Pointers&, int, cudaStream_t, int*);   // binning.cu
int record_cuda_error(cudaError_t);                                                // api.cu: feeds gs_last_cuda_error()
}  // namespace gs

namespace {
using namespace gs;

constexpr size_t NA_ALIGN = 256;
constexpr size_t na_up(size_t x) { return (x + NA_ALIGN - 1) / NA_ALIGN * NA_ALIGN; }
constexpr unsigned long long NA_MAX_KEYS = GS_NOALLOC_MAX_KEYS;
// the radix tile follows the CAPACITY (sort_items_for, common.cuh): 256 threads x 4 keys up to 256 Ki keys
constexpr size_t NA_TILE = (size_t)SORT_THREADS * 4;
constexpr size_t NA_TILES = (NA_MAX_KEYS + NA_TILE - 1) / NA_TILE + 1;             // per pass; + 1 as in make_layout
// layout of the scratch array: [control block | status words of the 4 passes | ping-pong keys]; the first two are zeroed
// by one cudaMemsetAsync per call
constexpr size_t NA_OFF_STATUS = na_up(sizeof(Ctrl));
constexpr size_t NA_OFF_PONG = na_up(NA_OFF_STATUS + 8 * 256 * NA_TILES * MAX_SORT_PASSES_DEPTH);
constexpr size_t NA_BYTES = na_up(NA_OFF_PONG + 8 * NA_MAX_KEYS);
static_assert(NA_MAX_KEYS <= (256ull << 10), "sort_items_for(capacity) must stay 4: the status stride assumes 1 024-key tiles");
static_assert(NA_BYTES <= (5u << 20), "gs.h states 4.2 MB");

// THE scratch: 4.2 MB held by every GPU that loads the library, until the process exits.  In host code this name is a
// host-side stand-in, not a device address; the address comes from cudaGetSymbolAddress (na_setup below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_BYTES];

// Copies the keys into the output buffer (which then plays gkeyA: the passes go out -> pong -> out -> pong -> out) and
// accumulates the four digit histograms of bits 32..63; block 0 also publishes the key count the passes read.
__global__ void __launch_bounds__(256)
noalloc_hist_kernel(const unsigned long long* __restrict__ in, unsigned long long* __restrict__ out, const uint32_t n,
                    Ctrl* __restrict__ ctrl) {
    __shared__ uint32_t s_hist[MAX_SORT_PASSES_DEPTH][256];
    const int tid = threadIdx.x;
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += 256) (&s_hist[0][0])[k] = 0;
    __syncthreads();
    for (uint32_t i = blockIdx.x * 256u + tid; i < n; i += gridDim.x * 256u) {
        const unsigned long long k = in[i];
        out[i] = k;
#pragma unroll
        for (int pass = 0; pass < MAX_SORT_PASSES_DEPTH; pass++) atomicAdd(&s_hist[pass][(uint32_t)(k >> (32 + 8 * pass)) & 255u], 1u);
    }
    __syncthreads();
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += 256) {
        const uint32_t c = (&s_hist[0][0])[k];
        if (c) atomicAdd(&ctrl->depth_hist[0][0] + k, c);
    }
    if (blockIdx.x == 0 && tid == 0) ctrl->n_sort = (unsigned long long)n;
}

struct NaDevice {
    unsigned char* base = nullptr;   // device address of g_noalloc_scratch on this device
    int n_sm = 0;
};
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mu;
NaDevice g_na_dev[NA_MAX_DEVICES];   // under g_na_mu

// Set-up, once per device, with that device current: the device address of the scratch array and the SM count.
int na_setup(int dev, NaDevice& out) {
    std::lock_guard<std::mutex> g(g_na_mu);
    NaDevice& d = g_na_dev[dev];
    if (d.base == nullptr) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return record_cuda_error(e);
        int n_sm = 0;
        e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return record_cuda_error(e);
        if (ptr == nullptr || n_sm <= 0) return GS_ERR_CUDA;
        d.n_sm = n_sm;
        d.base = static_cast<unsigned char*>(ptr);
    }
    out = d;
    return GS_OK;
}

bool na_on_device(const void* p, int dev) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) && at.device == dev;
}
}  // namespace

extern "C" {

uint32_t gs_noalloc_max_keys(void) { return (uint32_t)NA_MAX_KEYS; }

int gs_depth_sort_noalloc(const uint64_t* keys_in, uint64_t* keys_out, uint32_t n, void* cuda_stream) {
    if (n > NA_MAX_KEYS) return GS_ERR_LIMIT;     // before anything else: the limit is the contract of this entry point
    if (n == 0) return GS_OK;
    if (keys_in == nullptr || keys_out == nullptr || keys_in == keys_out) return GS_ERR_BAD_ARG;
    if ((reinterpret_cast<uintptr_t>(keys_in) | reinterpret_cast<uintptr_t>(keys_out)) & 7u) return GS_ERR_BAD_ARG;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return record_cuda_error(e);
    if (dev < 0 || dev >= NA_MAX_DEVICES) return GS_ERR_BAD_ARG;
    if (!na_on_device(keys_in, dev) || !na_on_device(keys_out, dev)) return GS_ERR_BAD_ARG;
    NaDevice d;
    const int rc = na_setup(dev, d);
    if (rc != GS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    Frame f = {};
    f.P = (int)NA_MAX_KEYS;    // the CAPACITY: fixes the radix tile (1 024 keys) and the grid, whatever n is
    f.rank_mode = 1;           // ballot multi-split: documented semantics only (the atomic-order self-test allocates)
    Pointers p = {};
    p.ctrl = reinterpret_cast<Ctrl*>(d.base);
    p.st_depth = reinterpret_cast<unsigned long long*>(d.base + NA_OFF_STATUS);
    p.n_depth_tiles = NA_TILES;
    p.gkeyA = reinterpret_cast<unsigned long long*>(keys_out);
    p.gkeyB = reinterpret_cast<unsigned long long*>(d.base + NA_OFF_PONG);

    // the array keeps the last call's contents: counters, histograms and status words must start at zero
    e = cudaMemsetAsync(d.base, 0, NA_OFF_PONG, st);
    if (e != cudaSuccess) return record_cuda_error(e);
    const uint32_t blocks = (n + 256u * 16u - 1u) / (256u * 16u);
    const int grid = (int)(blocks < (uint32_t)d.n_sm * 4u ? blocks : (uint32_t)d.n_sm * 4u);
    noalloc_hist_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const unsigned long long*>(keys_in), p.gkeyA, n, p.ctrl);
    e = cudaGetLastError();
    if (e != cudaSuccess) return record_cuda_error(e);
    g_use_pdl = 0;             // plain launches (thread-local switch of launch_pdl; gs_render sets it on every call)
    int launches = 0;
    launch_depth_sort(f, p, d.n_sm, st, &launches);   // 4 passes: out -> pong -> out -> pong -> out
    e = cudaGetLastError();
    if (e != cudaSuccess) return record_cuda_error(e);
    return GS_OK;
}

}  // extern "C"
