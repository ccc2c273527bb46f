// selftest.cu -- device micro-benchmarks behind the render roofline (SURVEY.md 8(d) "% of FP32 + SFU issue peak": the
// denominators are MEASURED per-SM rates, not derived ones).  gs_selftest_issue_peak() saturates the FP32 pipe with
// scalar FFMA, with packed FFMA2 (fma.rn.f32x2, what the blend loop issues) and the SFU with ex2.approx, each from 8
// independent dependency chains per thread, and reports thread-operations per second.  Product code (C ABI).
#include "common.cuh"

namespace gs {

constexpr int PK_THREADS = 256;
constexpr int PK_CHAINS = 8;
constexpr int PK_UNROLL = 32;   // instructions per chain and loop iteration

// MODE 0: FFMA, 1: FFMA2 (two FP32 operations per lane and instruction), 2: MUFU.EX2
template <int MODE>
__global__ void __launch_bounds__(PK_THREADS)
issue_peak_kernel(float* __restrict__ sink, int iters, float seed) {
    float a[PK_CHAINS];
    unsigned long long p[PK_CHAINS];
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) {
        a[c] = seed + (float)(threadIdx.x + c) * 1e-3f;
        asm("mov.b64 %0, {%1, %1};" : "=l"(p[c]) : "f"(a[c]));
    }
    const float m = 0.999f + seed * 1e-6f, b = 1e-3f;
    unsigned long long m2, b2;
    asm("mov.b64 %0, {%1, %1};" : "=l"(m2) : "f"(m));
    asm("mov.b64 %0, {%1, %1};" : "=l"(b2) : "f"(b));
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < PK_UNROLL; u++) {
#pragma unroll
            for (int c = 0; c < PK_CHAINS; c++) {
                if (MODE == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(m), "f"(b));
                else if (MODE == 1) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[c]) : "l"(m2), "l"(b2));
                else asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[c]));
            }
        }
    }
    float acc = 0.0f;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p[c]));
        acc += a[c] + lo + hi;
    }
    if (acc == 123.456f) sink[0] = acc;   // never true: keeps the chains alive
}

template <int MODE>
static cudaError_t time_mode(int n_sm, int iters, float* sink, double ops_per_instr, double* rate) {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    const int grid = n_sm * 8;   // 8 blocks of 8 warps: every scheduler has 16 warps to pick from
    double best = 0.0;
    for (int rep = 0; rep < 4 && e == cudaSuccess; rep++) {   // first repetition = warm-up / clock ramp; best of the rest
        cudaEventRecord(e0, nullptr);
        issue_peak_kernel<MODE><<<grid, PK_THREADS>>>(sink, iters, 1.0f);
        cudaEventRecord(e1, nullptr);
        e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        const double ops = (double)grid * PK_THREADS * (double)iters * PK_UNROLL * PK_CHAINS * ops_per_instr;
        if (rep > 0 && ms > 0.0f && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    *rate = best;
    return e;
}

cudaError_t run_issue_peak(int n_sm, int iters, double out[3]) {
    float* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 16);
    if (e != cudaSuccess) return e;
    e = time_mode<0>(n_sm, iters, sink, 1.0, &out[0]);
    if (e == cudaSuccess) e = time_mode<1>(n_sm, iters, sink, 2.0, &out[1]);
    if (e == cudaSuccess) e = time_mode<2>(n_sm, iters, sink, 1.0, &out[2]);
    cudaFree(sink);
    return e;
}

}  // namespace gs
