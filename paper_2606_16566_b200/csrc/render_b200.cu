// render_b200.cu -- the B200 render kernel (variant 4): Local-GS (Sec. III) re-laid-out for sm_100a.
//
//   * 128 threads per 16x16 tile, TWO horizontally adjacent pixels per thread, every per-pixel operation issued as a
//     packed f32x2 instruction (FFMA2 / FMUL2 / FADD2 with scalar-broadcast coefficient operands): the exponent
//     log2(alpha) = V_hoisted . B_local (Eq. 9-10) is 5 FFMA2 for two pixels, the blend w = alpha T; C += f w;
//     T -= w (Alg. 1 right column) is FMUL2 + 3 FFMA2 + FADD2.
//   * warp w owns the 8x8 quadrant (w&1, w>>1); the tight box (Eq. 13-19) is evaluated once per (tile, Gaussian) for
//     the two 8-pixel sub-columns and turned into a 4-bit warp mask (Eq. 20-21 with 8-row bands).
//   * the uniform skip of Sec. III-C4 is taken one step further: while staging, every warp gets its own compacted,
//     order-preserving LIST of the batch slots whose mask bit is set, so a culled (warp, Gaussian) pair costs no
//     instruction at all in the blend loop and every loop branch is warp-uniform.
//   * coefficients are pre-scaled by log2(e) so alpha = ex2.approx(L) directly; the 1/255 floor is a compare in the
//     log2 domain followed by a select (readings S12); hoisting is done in double, about the tile CENTRE (S14).
//   * termination rule R1 (reading S11) without any per-pixel state test in the hot loop: the only test is
//     T - w < 1e-4, voted across the warp; the rare taken branch un-blends the stopping pixel and POISONS its x^2
//     basis element (1e36), which drives every later log2(alpha) to -huge, i.e. alpha = 0 exactly.
#include "render_common.cuh"

namespace gs {

constexpr int QB = 128;            // threads per block == staged entries per batch
constexpr float POISON = 1.0e36f;  // x'^2 of a finished pixel: A * POISON <= -1e3 for every conic with a >= 1e-33

typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) {
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 fmul2(u64 a, u64 b) {
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 fsub2(u64 a, u64 b) {
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 bc(float v) { return pk(v, v); }  // scalar broadcast (a .F32 operand in SASS)

struct PixelPair {
    u64 bx2, bxy, by2, bx, by;  // B_local (Eq. 9) of the two pixels, tile-centre origin
    u64 T, Cr, Cg, Cb;
    uint32_t n0, n1;
    int ndone;                  // finished pixels of this thread (0..2)
};

// One (warp, Gaussian) step for two pixels.  Returns true when the whole warp is finished (Eq. 22).
template <bool COUNT, bool GUARD>
__device__ __forceinline__ bool blend_step(PixelPair& s, const float4 q0, const float4 q1, const float cb, const float guard) {
    // Eq. 10 in the log2 domain: 5 FFMA2 for two pixels (Table I: "5 FMA")
    u64 L2 = ffma2(bc(q0.x), s.bx2, bc(q0.w));
    L2 = ffma2(bc(q0.y), s.bxy, L2);
    L2 = ffma2(bc(q0.z), s.by2, L2);
    L2 = ffma2(bc(q1.x), s.bx, L2);
    L2 = ffma2(bc(q1.y), s.by, L2);
    float L0, L1;
    unpk(L2, L0, L1);
    bool v0 = L0 >= L2_ALPHA_MIN, v1 = L1 >= L2_ALPHA_MIN;          // opacity floor 1/255 (reading S12)
    if (GUARD) { v0 = v0 && (L0 <= guard); v1 = v1 && (L1 <= guard); }  // power > 0 (indefinite conic): skip
    const float a0 = v0 ? fminf(ALPHA_MAX, ex2_approx(L0)) : 0.0f;    // clamp to [0, 0.99]
    const float a1 = v1 ? fminf(ALPHA_MAX, ex2_approx(L1)) : 0.0f;
    u64 w2 = fmul2(pk(a0, a1), s.T);                                  // w = alpha T (Alg. 1 right)
    u64 Tn = fsub2(s.T, w2);                                          // T - w
    float t0, t1;
    unpk(Tn, t0, t1);
    const bool stop0 = t0 < T_MIN, stop1 = t1 < T_MIN;                // R1: this Gaussian would take T below 1e-4
    bool all_done = false;
    if (__any_sync(0xffffffffu, stop0 || stop1)) {                    // rare, warp-uniform
        float w0, w1, T0, T1, x0, x1;
        unpk(w2, w0, w1);
        unpk(s.T, T0, T1);
        unpk(s.bx2, x0, x1);
        if (stop0) { w0 = 0.0f; t0 = T0; x0 = POISON; s.ndone++; v0 = false; }
        if (stop1) { w1 = 0.0f; t1 = T1; x1 = POISON; s.ndone++; v1 = false; }
        w2 = pk(w0, w1);
        Tn = pk(t0, t1);
        s.bx2 = pk(x0, x1);
        all_done = __all_sync(0xffffffffu, s.ndone == 2);
    }
    s.Cr = ffma2(bc(q1.z), w2, s.Cr);                                 // C += f w
    s.Cg = ffma2(bc(q1.w), w2, s.Cg);
    s.Cb = ffma2(bc(cb), w2, s.Cb);
    s.T = Tn;
    if (COUNT) { s.n0 += v0 ? 1u : 0u; s.n1 += v1 ? 1u : 0u; }
    return all_done;
}

template <bool COUNT, bool STATS>
__global__ void __launch_bounds__(QB)
render_b200_kernel(const Frame f, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ ids,
                   const float4* __restrict__ geom, const float4* __restrict__ colour, float* __restrict__ out_rgb,
                   float* __restrict__ out_T, uint32_t* __restrict__ out_n) {
    __shared__ float4 s_q0[QB];       // A, B, C, F
    __shared__ float4 s_q1[QB];       // D, E, r, g
    __shared__ float s_cb[QB];        // b
    __shared__ float s_guard[QB];     // log2(o) of entries with an indefinite conic
    __shared__ uint8_t s_list[4][QB]; // per-warp compacted slot lists
    __shared__ uint32_t s_cnt[4][4];  // [quadrant][staging warp]
    __shared__ uint32_t s_flag[2];    // batch holds an indefinite conic (double-buffered by batch parity)
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.y * f.gx + blockIdx.x;
    const int Tx = blockIdx.x * TILE, Ty = blockIdx.y * TILE;
    // warp w = quadrant (w&1, w>>1); lane -> row lane>>2, column pair lane&3
    const int lx = 8 * (w & 1) + 2 * (lane & 3), ly = 8 * (w >> 1) + (lane >> 2);
    const int px = Tx + lx, py = Ty + ly;
    const bool in0 = px < f.W && py < f.H, in1 = (px + 1) < f.W && py < f.H;
    const float ox = (float)Tx + 7.5f, oy = (float)Ty + 7.5f;  // tile-centre origin (Eq. 1 with T at the centre)
    PixelPair s;
    {
        const float x0 = (float)lx - 7.5f, x1 = x0 + 1.0f, y = (float)ly - 7.5f;
        s.bx2 = pk(in0 ? x0 * x0 : POISON, in1 ? x1 * x1 : POISON);
        s.bxy = pk(x0 * y, x1 * y);
        s.by2 = pk(y * y, y * y);
        s.bx = pk(x0, x1);
        s.by = pk(y, y);
        s.T = pk(1.0f, 1.0f);
        s.Cr = s.Cg = s.Cb = pk(0.0f, 0.0f);
        s.n0 = s.n1 = 0;
        s.ndone = (in0 ? 0 : 1) + (in1 ? 0 : 1);
    }
    bool wdone = __all_sync(0xffffffffu, s.ndone == 2);
    const uint32_t start = ranges[tile], end = ranges[tile + 1];
    const unsigned lt = (1u << lane) - 1u;
    int parity = 0;
    uint32_t st_walk = 0, st_staged = 0;  // STATS only
    for (uint32_t base = start; base < end; base += QB, parity ^= 1) {
        if (tid == 0) s_flag[parity] = 0;
        if (__syncthreads_and(wdone)) break;  // every warp of the tile is finished
        // ---- staging: gather, tight box -> 4-bit warp mask, per-warp compacted lists, hoist -----------------------
        uint32_t m = 0;
        float4 g0 = make_float4(0.f, 0.f, 0.f, 0.f), g1 = g0;
        uint32_t id = 0;
        const uint32_t k = base + tid;
        if (STATS && tid == 0) st_staged += min((uint32_t)QB, end - base);
        if (k < end) {
            id = ids[k];
            g0 = __ldg(geom + 2 * (size_t)id);
            g1 = __ldg(geom + 2 * (size_t)id + 1);
            const float tau = tau_widened(g1.y);
            if (tau > 0.0f) {
                const float dxc = g0.x - (float)Tx, dyc = g0.y - (float)Ty;
                int r0, r1;
                column_rows(dxc, dyc, g0.z, g0.w, g1.x, g1.z, tau, 0.0f, 7.0f, r0, r1);
                if (r0 <= r1) m |= (r0 <= 7 ? 1u : 0u) | (r1 >= 8 ? 4u : 0u);
                column_rows(dxc, dyc, g0.z, g0.w, g1.x, g1.z, tau, 8.0f, 15.0f, r0, r1);
                if (r0 <= r1) m |= (r0 <= 7 ? 2u : 0u) | (r1 >= 8 ? 8u : 0u);
            }
        }
        const bool indefinite = (__float_as_uint(g1.w) & 1u) && m;
        const unsigned b0 = __ballot_sync(0xffffffffu, m & 1u), b1 = __ballot_sync(0xffffffffu, m & 2u),
                       b2 = __ballot_sync(0xffffffffu, m & 4u), b3 = __ballot_sync(0xffffffffu, m & 8u);
        if (lane < 4) s_cnt[lane][w] = __popc(lane == 0 ? b0 : lane == 1 ? b1 : lane == 2 ? b2 : b3);
        if (__any_sync(0xffffffffu, indefinite) && lane == 0) s_flag[parity] = 1;
        if (m) {  // only entries that reach some warp are hoisted and coloured
            const float4 c = __ldg(colour + id);
            const Hoisted h = hoist(g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, ox, oy);
            s_q0[tid] = make_float4(h.A, h.B, h.C, h.F);
            s_q1[tid] = make_float4(h.D, h.E, c.x, c.y);
            s_cb[tid] = c.z;
            s_guard[tid] = (__float_as_uint(g1.w) & 1u) ? g1.y : 3.0e38f;
        }
        __syncthreads();
        {
            uint32_t o0 = 0, o1 = 0, o2 = 0, o3 = 0;
            for (int sw = 0; sw < w; sw++) { o0 += s_cnt[0][sw]; o1 += s_cnt[1][sw]; o2 += s_cnt[2][sw]; o3 += s_cnt[3][sw]; }
            if (m & 1u) s_list[0][o0 + __popc(b0 & lt)] = (uint8_t)tid;
            if (m & 2u) s_list[1][o1 + __popc(b1 & lt)] = (uint8_t)tid;
            if (m & 4u) s_list[2][o2 + __popc(b2 & lt)] = (uint8_t)tid;
            if (m & 8u) s_list[3][o3 + __popc(b3 & lt)] = (uint8_t)tid;
        }
        __syncthreads();
        // ---- blend: this warp walks ITS list only ---------------------------------------------------------------
        if (!wdone) {
            const int cnt = (int)(s_cnt[w][0] + s_cnt[w][1] + s_cnt[w][2] + s_cnt[w][3]);
            const uint8_t* list = s_list[w];
            if (s_flag[parity] == 0) {
                for (int i = 0; i < cnt; i++) {
                    const int j = list[i];
                    if (STATS) st_walk++;
                    if (blend_step<COUNT, false>(s, s_q0[j], s_q1[j], s_cb[j], 0.0f)) { wdone = true; break; }
                }
            } else {
                for (int i = 0; i < cnt; i++) {
                    const int j = list[i];
                    if (STATS) st_walk++;
                    if (blend_step<COUNT, true>(s, s_q0[j], s_q1[j], s_cb[j], s_guard[j])) { wdone = true; break; }
                }
            }
        }
    }
    if (STATS) {  // gs_set_stats(1): what the blend loop actually did (bench.py roofline)
        uint32_t nb = s.n0 + s.n1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nb += __shfl_xor_sync(0xffffffffu, nb, o);
        if (lane == 0) {
            atomicAdd(&ctrl->stats[0], (unsigned long long)st_walk);
            atomicAdd(&ctrl->stats[1], (unsigned long long)nb);
        }
        if (tid == 0) atomicAdd(&ctrl->stats[2], (unsigned long long)st_staged);
    }
    // ---- epilogue: out = C + T bg (reading S16) -------------------------------------------------------------------
    float T0, T1, r0, r1, g0_, g1_, b0_, b1_;
    unpk(s.T, T0, T1); unpk(s.Cr, r0, r1); unpk(s.Cg, g0_, g1_); unpk(s.Cb, b0_, b1_);
    const size_t npix = (size_t)f.W * f.H, pix = (size_t)py * f.W + px;
    if (in0) {
        out_rgb[pix] = fmaf(T0, f.bg[0], r0);
        out_rgb[npix + pix] = fmaf(T0, f.bg[1], g0_);
        out_rgb[2 * npix + pix] = fmaf(T0, f.bg[2], b0_);
        out_T[pix] = T0;
        if (COUNT) out_n[pix] = s.n0;
    }
    if (in1) {
        out_rgb[pix + 1] = fmaf(T1, f.bg[0], r1);
        out_rgb[npix + pix + 1] = fmaf(T1, f.bg[1], g1_);
        out_rgb[2 * npix + pix + 1] = fmaf(T1, f.bg[2], b1_);
        out_T[pix + 1] = T1;
        if (COUNT) out_n[pix + 1] = s.n1;
    }
}

void launch_render_b200(const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n, int n_sm,
                        bool stats, cudaStream_t st) {
    (void)n_sm;
    const dim3 grid(f.gx, f.gy), block(QB);
    if (stats && out_n)
        render_b200_kernel<true, true><<<grid, block, 0, st>>>(f, p.ctrl, p.ranges, p.ids, p.geom, p.colour, out_rgb, out_T, out_n);
    else if (out_n)
        render_b200_kernel<true, false><<<grid, block, 0, st>>>(f, p.ctrl, p.ranges, p.ids, p.geom, p.colour, out_rgb, out_T, out_n);
    else
        render_b200_kernel<false, false><<<grid, block, 0, st>>>(f, p.ctrl, p.ranges, p.ids, p.geom, p.colour, out_rgb, out_T, nullptr);
}

}  // namespace gs
