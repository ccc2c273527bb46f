// render.cu -- render kernels, ablation ladder of PAPER.md Table IV, one thread per pixel, a 16x16 tile
// per 256-thread block, warp w owns the 16x2 strip of rows 2w, 2w+1:
//   variant 0  baseline column of Alg. 1: direct conic exponent (Table I left), per-pixel branches
//   variant 1  + tile-local hoisting: log2(alpha) = V_hoisted . B_local, 5 FMA (Eq. 7-10)
//   variant 2  + warp-level culling: 8-bit visibility mask, uniform skip (Eq. 13-21)
//   variant 3  + warp-coherent blending: branch-free predicated blend, warp-uniform exit (Eq. 22)
//   variant 6  = variant 3 with the polynomial in GLOBAL pixel coordinates and fp32 coefficients: the precision switch of
//              PAPER.md Sec. III-B4 / Table V (Eq. 11: error bound 4 * 4000^2 * 2^-24 = 3.81 in ln alpha at 4K).  It
//              exists to MEASURE that failure against the oracle; it does not meet the parity tolerance by design.
// All variants implement termination rule R1 (reading S11) and produce the same image up to rounding.
// The B200 design (variant 4) lives in render_b200.cu.  This TU may use approximate intrinsics.
#include "render_common.cuh"

namespace gs {

constexpr int RB = 256;  // batch = block size

// Eq. 8 evaluated the naive way: fp32 throughout, about an arbitrary origin (the global-coordinate variant uses (0, 0)).
__device__ __forceinline__ Hoisted hoist_f32(float mux, float muy, float a, float b, float c, float log2o, float ox, float oy) {
    const float k = LOG2E;
    const float dx = mux - ox, dy = muy - oy;
    Hoisted h;
    h.A = -0.5f * k * a;
    h.B = -k * b;
    h.C = -0.5f * k * c;
    h.D = k * (a * dx + b * dy);
    h.E = k * (b * dx + c * dy);
    h.F = log2o - 0.5f * k * (a * dx * dx + 2.0f * b * dx * dy + c * dy * dy);
    return h;
}

template <int VAR, bool GLOBAL = false>
__global__ void __launch_bounds__(256)
render_ladder_kernel(const Frame f, const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ ids,
                     const float4* __restrict__ rec, float* __restrict__ out_rgb,
                     float* __restrict__ out_T, uint32_t* __restrict__ out_n) {
    constexpr bool HOIST = VAR >= 1, CULL = VAR >= 2, COHERENT = VAR >= 3;
    // staged batch: HOIST ? (A,B,C,F) : (mux,muy,a,b) ; HOIST ? (D,E,guard,-) : (c,o,-,-)
    __shared__ float4 s_q0[RB];
    __shared__ float4 s_q1[RB];
    __shared__ float4 s_col[RB];
    __shared__ uint32_t s_mask[RB];
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.y * f.gx + blockIdx.x;
    const int Tx = blockIdx.x * TILE, Ty = blockIdx.y * TILE;
    const int lx = lane & 15, ly = 2 * w + (lane >> 4);  // tile-local pixel (16x2 strip per warp)
    const int px = Tx + lx, py = Ty + ly;
    const bool inside = px < f.W && py < f.H;
    const float fx_ = (float)px, fy_ = (float)py;     // baseline: global pixel coordinates
    const float xl = GLOBAL ? fx_ : (float)lx, yl = GLOBAL ? fy_ : (float)ly;  // hoisted: tile-local coordinates (Eq. 1)
    const float bx2 = xl * xl, bxy = xl * yl, by2 = yl * yl;  // B_local (Eq. 9)
    const uint32_t start = ranges[tile], end = ranges[tile + 1];
    float T = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    uint32_t n = 0;
    bool done = !inside;
    for (uint32_t base = start; base < end; base += RB) {
        // block-level exit once every pixel of the tile is done (baseline) / every warp is done
        if (__syncthreads_and(done)) break;
        {   // ---- cooperative staging ---------------------------------------------------------
            const uint32_t k = base + tid;
            if (k < end) {
                const uint32_t id = ids[k];
                // 64-byte render record (include/gs.h): {mu_x, mu_y, b, det | x*, 1/c, c tau, flags | a, c, log2 o, r | g, b, -, -}
                const float4 k0 = __ldg(rec + 4 * (size_t)id), k1 = __ldg(rec + 4 * (size_t)id + 1),
                             k2 = __ldg(rec + 4 * (size_t)id + 2), k3 = __ldg(rec + 4 * (size_t)id + 3);
                const float4 g0 = make_float4(k0.x, k0.y, k2.x, k0.z), g1 = make_float4(k2.y, k2.z, k0.w, k1.w);
                s_col[tid] = make_float4(k2.w, k3.x, k3.y, 0.0f);
                const bool indefinite = __float_as_uint(g1.w) & 1u;
                if (HOIST) {
                    const Hoisted h = GLOBAL ? hoist_f32(g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, 0.0f, 0.0f)
                                             : hoist(g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, (float)Tx, (float)Ty);
                    s_q0[tid] = make_float4(h.A, h.B, h.C, h.F);
                    // power > 0  <=>  log2(alpha) > log2(o): only an indefinite conic can get there (C-R step 2)
                    s_q1[tid] = make_float4(h.D, h.E, indefinite ? g1.y : 3.0e38f, 0.0f);
                } else {
                    s_q0[tid] = g0;
                    s_q1[tid] = make_float4(g1.x, ex2_approx(g1.y), 0.0f, 0.0f);
                }
                if (CULL) {
                    uint32_t m = 0;
                    const float tau = tau_widened(g1.y);
                    if (tau > 0.0f) {
                        int r0, r1;
                        column_rows(g0.x - (float)Tx, g0.y - (float)Ty, g0.z, g0.w, g1.x, g1.z, tau, 0.0f, 15.0f, r0, r1);
                        if (r0 <= r1) {  // Eq. 20-21
                            const int w0 = r0 >> 1, w1 = r1 >> 1;
                            m = ((1u << (w1 - w0 + 1)) - 1u) << w0;
                        }
                    }
                    s_mask[tid] = m;
                }
            }
        }
        __syncthreads();
        const int cnt = (int)min((uint32_t)RB, end - base);
        if (COHERENT) {
            // ---- warp-coherent blending (Alg. 1 right column; readings S11, S12) ------------------------------
            for (int j = 0; j < cnt; j++) {
                if (CULL && !((s_mask[j] >> w) & 1u)) continue;  // warp-uniform skip
                if (__all_sync(0xffffffffu, done)) break;          // Eq. 22
                const float4 q0 = s_q0[j], q1 = s_q1[j], c = s_col[j];
                float L = fmaf(q0.x, bx2, q0.w);
                L = fmaf(q0.y, bxy, L);
                L = fmaf(q0.z, by2, L);
                L = fmaf(q1.x, xl, L);
                L = fmaf(q1.y, yl, L);
                const float alpha = fminf(ALPHA_MAX, ex2_approx(L));
                const bool valid = (L >= L2_ALPHA_MIN) && (L <= q1.z);
                float wgt = alpha * T;
                const bool stop = valid && (T - wgt < T_MIN);
                done = done || stop;
                const bool take = valid && !done;
                wgt = take ? wgt : 0.0f;
                Cr = fmaf(c.x, wgt, Cr);
                Cg = fmaf(c.y, wgt, Cg);
                Cb = fmaf(c.z, wgt, Cb);
                T -= wgt;
                n += take ? 1u : 0u;
            }
        } else {
            // ---- baseline blending (Alg. 1 left column): per-pixel branches -----------------------------------
            for (int j = 0; !done && j < cnt; j++) {
                if (CULL && !((s_mask[j] >> w) & 1u)) continue;
                const float4 q0 = s_q0[j], q1 = s_q1[j];
                float alpha;
                if (HOIST) {
                    float L = fmaf(q0.x, bx2, q0.w);
                    L = fmaf(q0.y, bxy, L);
                    L = fmaf(q0.z, by2, L);
                    L = fmaf(q1.x, xl, L);
                    L = fmaf(q1.y, yl, L);
                    if (L > q1.z) continue;
                    alpha = fminf(ALPHA_MAX, ex2_approx(L));
                } else {
                    const float dx = fx_ - q0.x, dy = fy_ - q0.y;  // Table I left: 3 SUB + 8 MUL + 1 ADD
                    const float power = -0.5f * (q0.z * dx * dx + q1.x * dy * dy) - q0.w * dx * dy;
                    if (power > 0.0f) continue;
                    alpha = fminf(ALPHA_MAX, q1.y * __expf(power));
                }
                if (alpha < ALPHA_MIN) continue;
                const float test_T = T * (1.0f - alpha);
                if (test_T < T_MIN) { done = true; continue; }
                const float4 c = s_col[j];
                Cr += c.x * alpha * T;
                Cg += c.y * alpha * T;
                Cb += c.z * alpha * T;
                T = test_T;
                n++;
            }
        }
    }
    if (inside) {
        const size_t npix = (size_t)f.W * f.H, pix = (size_t)py * f.W + px;
        out_rgb[pix] = fmaf(T, f.bg[0], Cr);
        out_rgb[npix + pix] = fmaf(T, f.bg[1], Cg);
        out_rgb[2 * npix + pix] = fmaf(T, f.bg[2], Cb);
        out_T[pix] = T;
        if (out_n) out_n[pix] = n;
    }
}

void launch_render_ladder(int variant, const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n,
                          cudaStream_t st) {
    const dim3 grid(f.gx, f.gy), block(256);
    switch (variant) {
        case 0: render_ladder_kernel<0><<<grid, block, 0, st>>>(f, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n); break;
        case 1: render_ladder_kernel<1><<<grid, block, 0, st>>>(f, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n); break;
        case 2: render_ladder_kernel<2><<<grid, block, 0, st>>>(f, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n); break;
        case 6: render_ladder_kernel<3, true><<<grid, block, 0, st>>>(f, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n); break;
        default: render_ladder_kernel<3><<<grid, block, 0, st>>>(f, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n); break;
    }
}

}  // namespace gs
