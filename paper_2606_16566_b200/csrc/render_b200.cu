// render_b200.cu -- the B200 render kernel (variant 4): Local-GS (Sec. III) re-laid-out for sm_100a.
//
//   * 128 threads per 16x16 tile, TWO horizontally adjacent pixels per thread, every per-pixel operation issued as a
//     packed f32x2 instruction (FFMA2 / FMUL2 with scalar-broadcast coefficient operands): the exponent
//     log2(alpha) = V_hoisted . B_local (Eq. 9-10) is 5 FFMA2 for two pixels, the blend w = alpha T; C += f w;
//     T -= w (Alg. 1 right column) is FMUL2 + 4 FFMA2.
//   * warp w owns the 8x8 quadrant (w&1, w>>1); the tight box (Eq. 13-19) is evaluated once per (tile, Gaussian) for
//     the two 8-pixel sub-columns and turned into a 4-bit warp mask (Eq. 20-21 with 8-row bands); its per-Gaussian
//     part (x*, 1/c, c tau) comes precomputed from preprocess, the per-tile part is branch-free.
//   * the uniform skip of Sec. III-C4 is taken one step further: every warp turns the mask ballots of a staged batch
//     into its own compacted, order-preserving LIST of record offsets, so a culled (warp, Gaussian) pair costs no
//     instruction at all in the blend loop and every loop branch is warp-uniform.
//   * the opacity floor costs no instruction: the exponent carries the bias -126 - log2(1/255), so
//     ex2.approx.ftz flushes every alpha < 1/255 to exactly 0 (readings S12, G4); alpha and T live scaled by
//     K = 2^126 / 255 and 1/K folds into the w = alpha T product.  No compare, no select, no predicate.
//   * hoisting is done in double, about the tile CENTRE (S14), once per (tile, Gaussian).
//   * termination rule R1 (reading S11) without any per-pixel state test in the hot loop: the only test is
//     T - w < 1e-4, voted across the warp; the rare taken branch un-blends the stopping pixel and POISONS its x^2
//     basis element (1e36), which drives every later log2(alpha) to -huge, i.e. alpha = 0 exactly.
//   * staging is software-pipelined: the ids of batch k+2 and the 64-byte records of batch k+1 are in flight while
//     batch k is blended; shared memory is double-buffered, so a batch costs ONE block barrier.
#include "render_common.cuh"

namespace gs {

constexpr int QB = 128;            // threads per block == staged entries per batch
constexpr float POISON = 1.0e36f;  // x'^2 of a finished pixel: A * POISON <= -1e3 for every conic with a >= 1e-33
// alpha' = 2^(L + L_BIAS) = alpha / K:  alpha' < 2^-126 (flushed to 0 by ex2.approx.ftz)  <=>  alpha < 1/255
constexpr float L_BIAS = -118.00564575195312f;   // fl32(-126 - log2(1/255))
constexpr float K_SCALE = 3.33609985e+35f;       // 2^(-L_BIAS): alpha = K alpha', T_s = K T
constexpr float K_INV = 2.99751221e-36f;
constexpr float AMAX_S = 2.96753725e-36f;        // 0.99 / K   (PAPER.md:277 clamp)
constexpr float TMIN_S = 3.33609971e+31f;        // 1e-4 K
constexpr int REC = 48;                          // bytes of one staged record: (A,B,C,F) (D,E,r,g) (b,guard,-,-)

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
__device__ __forceinline__ u64 bc(float v) { return pk(v, v); }  // scalar broadcast (a .F32 operand in SASS)
// acc <- a * b + acc, in place (the accumulator is one read-modify-write operand, so no copy is ever needed)
__device__ __forceinline__ void ffma2_acc(u64& acc, u64 a, u64 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b)); }

struct PixelPair {
    u64 bx2, bxy, by2, bx, by;  // B_local (Eq. 9) of the two pixels, tile-centre origin
    u64 T, Cr, Cg, Cb;          // T scaled by K; touched by the unconditional blend only
    u64 thr;                    // per pixel: 1e-4 K while the pixel is live, -(K w of the un-blended entries) once stopped
    u64 dCr, dCg, dCb;          // colour of the un-blended entries (written by the rare branch only; added at the end)
    uint32_t n0, n1;
};

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint2 lds64u(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
    return v;
}

// Exponent and alpha of one staged record for the two pixels of this thread: alpha / K, clamped (Eq. 10 in the biased
// log2 domain: 5 FFMA2, "5 FMA" of Table I; exactly 0 below the 1/255 floor; min(0.99, .)).
template <bool GUARD>
__device__ __forceinline__ u64 alpha_pair(const PixelPair& s, const float4 q0, const float4 q1, const float guard, float& e0,
                                          float& e1) {
    u64 L2 = ffma2(bc(q0.x), s.bx2, bc(q0.w));
    L2 = ffma2(bc(q0.y), s.bxy, L2);
    L2 = ffma2(bc(q0.z), s.by2, L2);
    L2 = ffma2(bc(q1.x), s.bx, L2);
    L2 = ffma2(bc(q1.y), s.by, L2);
    float L0, L1;
    unpk(L2, L0, L1);
    e0 = ex2_approx(L0);
    e1 = ex2_approx(L1);
    if (GUARD) {                                      // power > 0 (indefinite conic): skip (C-R step 2)
        e0 = (L0 <= guard) ? e0 : 0.0f;
        e1 = (L1 <= guard) ? e1 : 0.0f;
    }
    return pk(fminf(AMAX_S, e0), fminf(AMAX_S, e1));
}

// TWO consecutive list entries (records at shared-memory addresses a1, a2) for the two pixels of this thread.
// Everything is updated IN PLACE and unconditionally -- w = alpha T; T <- T - K w; C <- C + f w (Alg. 1 right column),
// twice -- followed by ONE warp vote: T only decreases, so "some T ended below 1e-4" catches a crossing in either entry.
// The rare branch REPAIRS the stopping pixels (rule R1: the crossing Gaussian and everything after it is not blended):
// their f w are subtracted again and T is restored, packed and in place (wm = w on the stopping pixels, 0 elsewhere:
// exact no-ops for the others; the restored values are within two roundings of the old ones -- toleranced outputs),
// then the pixels are poisoned.  When the whole warp is finished (Eq. 22) the branch zeroes `lend`, the warp-uniform
// end of the list walk, so the loop has one exit and no flag to test.
template <bool COUNT, bool GUARD>
__device__ __forceinline__ void blend_pair(PixelPair& s, const uint32_t a1, const uint32_t a2, uint32_t& lend) {
    const float4 p0 = lds128(a1), p1 = lds128(a1 + 16);   // (A, B, C, F) (D, E, r, g)
    const float2 p2 = lds64(a1 + 32);                     // (b, guard)
    const float4 q0 = lds128(a2), q1 = lds128(a2 + 16);
    const float2 q2 = lds64(a2 + 32);
    float e0, e1, g0, g1;
    const u64 al1 = alpha_pair<GUARD>(s, p0, p1, p2.y, e0, e1);
    const u64 al2 = alpha_pair<GUARD>(s, q0, q1, q2.y, g0, g1);
    const u64 w1 = fmul2(al1, s.T);
    const u64 T1 = ffma2(bc(-K_SCALE), w1, s.T);
    const u64 w2 = fmul2(al2, T1);
    s.T = ffma2(bc(-K_SCALE), w2, T1);
    ffma2_acc(s.Cr, bc(p1.z), w1);
    ffma2_acc(s.Cg, bc(p1.w), w1);
    ffma2_acc(s.Cb, bc(p2.x), w1);
    ffma2_acc(s.Cr, bc(q1.z), w2);
    ffma2_acc(s.Cg, bc(q1.w), w2);
    ffma2_acc(s.Cb, bc(q2.x), w2);
    if (COUNT) {
        s.n0 += ((e0 > 0.0f) ? 1u : 0u) + ((g0 > 0.0f) ? 1u : 0u);
        s.n1 += ((e1 > 0.0f) ? 1u : 0u) + ((g1 > 0.0f) ? 1u : 0u);
    }
    float t0, t1, h0, h1;
    unpk(s.T, t0, t1);
    unpk(s.thr, h0, h1);
    if (__any_sync(0xffffffffu, (t0 < h0) || (t1 < h1))) {   // rare; a stopped pixel has thr < 0 <= T: it never fires again
        float u0, u1, w10, w11, w20, w21;
        unpk(T1, u0, u1); unpk(w1, w10, w11); unpk(w2, w20, w21);
        const bool sa0 = u0 < h0, sa1 = u1 < h1;              // stopped at the first entry
        const bool sb0 = t0 < h0, sb1 = t1 < h1;              // stopped at the first or the second entry
        const u64 wm2 = pk(sb0 ? w20 : 0.0f, sb1 ? w21 : 0.0f), wm1 = pk(sa0 ? w10 : 0.0f, sa1 ? w11 : 0.0f);
        // thr <- -(K wm1 + K wm2) on the stopping pixels (final T = T - thr there), unchanged elsewhere
        const u64 live = pk(sb0 ? 0.0f : 1.0f, sb1 ? 0.0f : 1.0f);
        s.thr = ffma2(bc(-K_SCALE), wm2, fmul2(s.thr, live));
        ffma2_acc(s.thr, bc(-K_SCALE), wm1);
        ffma2_acc(s.dCr, bc(-q1.z), wm2);
        ffma2_acc(s.dCg, bc(-q1.w), wm2);
        ffma2_acc(s.dCb, bc(-q2.x), wm2);
        ffma2_acc(s.dCr, bc(-p1.z), wm1);
        ffma2_acc(s.dCg, bc(-p1.w), wm1);
        ffma2_acc(s.dCb, bc(-p2.x), wm1);
        ffma2_acc(s.bx2, pk(sb0 ? 1.0f : 0.0f, sb1 ? 1.0f : 0.0f), bc(POISON));
        if (COUNT) {  // a pixel stopped at the first entry also counted the second one when its alpha was > 0
            s.n0 -= (sa0 ? 1u + ((g0 > 0.0f) ? 1u : 0u) : (sb0 ? 1u : 0u));
            s.n1 -= (sa1 ? 1u + ((g1 > 0.0f) ? 1u : 0u) : (sb1 ? 1u : 0u));
        }
        float x0, x1;
        unpk(s.bx2, x0, x1);
        if (__all_sync(0xffffffffu, x0 >= 0.5f * POISON && x1 >= 0.5f * POISON)) lend = 0;
    }
}

// Walk of one warp's list (two entries per iteration; the list is padded to an even length with the null record).
template <bool COUNT, bool GUARD>
__device__ __forceinline__ void blend_list(PixelPair& s, uint32_t& lp, uint32_t& lend) {
    while (lp < lend) {
        const uint2 aa = lds64u(lp);
        lp += 8;
        blend_pair<COUNT, GUARD>(s, aa.x, aa.y, lend);
    }
}

template <bool COUNT, bool STATS>
__global__ void __launch_bounds__(QB, 6)
render_b200_kernel(const Frame f, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ ids,
                   const float4* __restrict__ rec, float* __restrict__ out_rgb, float* __restrict__ out_T,
                   uint32_t* __restrict__ out_n) {
    __shared__ __align__(16) unsigned char s_rec[2][(QB + 1) * REC];  // staged, hoisted records (double-buffered) + a null record
    __shared__ __align__(16) uint32_t s_ball[2][4][4];          // [buffer][staging warp][quadrant] mask ballots
    __shared__ __align__(16) uint32_t s_indef[2][4];                        // [buffer][staging warp] batch holds an indefinite conic
    __shared__ __align__(16) uint32_t s_list[4][QB + 2];        // per-warp compacted lists of record addresses (padded to even length)
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31;
    // warp index through a warp reduction: ptxas then KNOWS it is warp-uniform (it lives in a uniform register), so
    // every trip count derived from it is uniform and the votes of the blend loop need no divergence guard
    const int w = __reduce_max_sync(0xffffffffu, tid >> 5);
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
        s.T = pk(K_SCALE, K_SCALE);
        s.Cr = s.Cg = s.Cb = s.dCr = s.dCg = s.dCb = pk(0.0f, 0.0f);
        s.thr = pk(TMIN_S, TMIN_S);
        s.n0 = s.n1 = 0;
    }
    if (tid < 6) {  // null record of both buffers: F = -huge, alpha = 0 exactly; colours 0
        float4* d = reinterpret_cast<float4*>(&s_rec[tid & 1][QB * REC]) + (tid >> 1);
        *d = make_float4(0.0f, 0.0f, 0.0f, (tid >> 1) == 0 ? -1.0e30f : 0.0f);
        if ((tid >> 1) == 2) d->y = 3.0e38f;
    }
    bool wdone = __all_sync(0xffffffffu, !in0 && !in1);
    const uint32_t start = ranges[tile], end = ranges[tile + 1];
    const unsigned lt = (1u << lane) - 1u;
    uint32_t st_walk = 0, st_staged = 0;  // STATS only
    // ---- software pipeline prologue: records of batch 0, ids of batch 1 ------------------------------------------
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0, r3 = r0;
    uint32_t id_next = 0;
    if (start + tid < end) {
        const uint32_t id = ids[start + tid];
        const float4* p = rec + 4 * (size_t)id;
        r0 = __ldg(p); r1 = __ldg(p + 1); r2 = __ldg(p + 2); r3 = __ldg(p + 3);
    }
    if (start + QB + tid < end) id_next = ids[start + QB + tid];
    int buf = 0;
    for (uint32_t base = start; base < end; base += QB, buf ^= 1) {
        // ---- staging of batch `base` from registers: tight box -> 4-bit warp mask, hoist -> shared memory ----------
        uint32_t m = 0;
        bool indefinite = false;
        if (STATS && tid == 0) st_staged += min((uint32_t)QB, end - base);
        if (base + tid < end) {
            m = quadrant_mask(r0.x - (float)Tx, r0.y - (float)Ty, r0.w, r1.z, r2.w, r3.x, r3.y);
            if (__float_as_uint(r1.w) & 1u) { m = 15u; indefinite = true; }  // degenerate conic: keep everything
        }
        const unsigned b0 = __ballot_sync(0xffffffffu, m & 1u), b1 = __ballot_sync(0xffffffffu, m & 2u),
                       b2 = __ballot_sync(0xffffffffu, m & 4u), b3 = __ballot_sync(0xffffffffu, m & 8u);
        const unsigned bi = __ballot_sync(0xffffffffu, indefinite);
        if (lane == 0) *reinterpret_cast<uint4*>(&s_ball[buf][w][0]) = make_uint4(b0, b1, b2, b3);
        if (lane == 4) s_indef[buf][w] = bi;
        if (m) {  // only entries that reach some warp are hoisted
            const Hoisted h = hoist(r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, ox, oy, L_BIAS);
            float4* d = reinterpret_cast<float4*>(&s_rec[buf][tid * REC]);
            d[0] = make_float4(h.A, h.B, h.C, h.F);
            d[1] = make_float4(h.D, h.E, r2.x, r2.y);
            d[2] = make_float4(r2.z, indefinite ? r1.y + L_BIAS : 3.0e38f, 0.0f, 0.0f);
        }
        // ---- prefetch: records of the next batch, ids of the one after -------------------------------------------
        if (base + QB + tid < end) {
            const float4* p = rec + 4 * (size_t)id_next;
            r0 = __ldg(p); r1 = __ldg(p + 1); r2 = __ldg(p + 2); r3 = __ldg(p + 3);
        }
        if (base + 2 * QB + tid < end) id_next = ids[base + 2 * QB + tid];
        // ---- the batch's only barrier; also the block-level exit (every warp of the tile finished, Eq. 22) ----------
        if (__syncthreads_and(wdone)) break;
        if (wdone) continue;
        // ---- this warp's compacted list: addresses of the staged records whose mask bit w is set, in list order -----
        const uint4 bb = make_uint4(s_ball[buf][0][w], s_ball[buf][1][w], s_ball[buf][2][w], s_ball[buf][3][w]);
        const uint4 iv = *reinterpret_cast<const uint4*>(&s_indef[buf][0]);
        const int c0 = __popc(bb.x), c1 = c0 + __popc(bb.y), c2 = c1 + __popc(bb.z), cnt = c2 + __popc(bb.w);
        const uint32_t rec_addr = (uint32_t)__cvta_generic_to_shared(&s_rec[buf][0]);
        uint32_t* list = &s_list[w][0];
        if ((bb.x >> lane) & 1u) list[__popc(bb.x & lt)] = rec_addr + lane * REC;
        if ((bb.y >> lane) & 1u) list[c0 + __popc(bb.y & lt)] = rec_addr + (32 + lane) * REC;
        if ((bb.z >> lane) & 1u) list[c1 + __popc(bb.z & lt)] = rec_addr + (64 + lane) * REC;
        if ((bb.w >> lane) & 1u) list[c2 + __popc(bb.w & lt)] = rec_addr + (96 + lane) * REC;
        if (lane == 0) list[cnt] = rec_addr + QB * REC;  // pad to an even length with the null record (alpha = 0)
        __syncwarp();
        // ---- blend: this warp walks ITS list only, two entries per iteration ---------------------------------------
        uint32_t lp = (uint32_t)__cvta_generic_to_shared(list);
        const uint32_t lp0 = lp;
        uint32_t lend = lp + 4 * cnt;
        if ((iv.x | iv.y | iv.z | iv.w) == 0u) blend_list<COUNT, false>(s, lp, lend);
        else blend_list<COUNT, true>(s, lp, lend);
        wdone = lend == 0;
        if (STATS) st_walk += min((lp - lp0) / 4, (uint32_t)cnt);
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
    float T0, T1, c0r, c1r, c0g, c1g, c0b, c1b;
    {   // fold the repairs of the stopped pixels in: T = T - thr where thr < 0, C = C + dC
        float h0, h1, d0, d1;
        unpk(s.T, T0, T1); unpk(s.thr, h0, h1);
        T0 = (h0 < 0.0f ? T0 - h0 : T0) * K_INV;
        T1 = (h1 < 0.0f ? T1 - h1 : T1) * K_INV;
        unpk(s.Cr, c0r, c1r); unpk(s.dCr, d0, d1); c0r += d0; c1r += d1;
        unpk(s.Cg, c0g, c1g); unpk(s.dCg, d0, d1); c0g += d0; c1g += d1;
        unpk(s.Cb, c0b, c1b); unpk(s.dCb, d0, d1); c0b += d0; c1b += d1;
    }
    const size_t npix = (size_t)f.W * f.H, pix = (size_t)py * f.W + px;
    if (in1 && !(f.W & 1)) {  // both pixels inside, 8-byte aligned pair
        *reinterpret_cast<float2*>(out_rgb + pix) = make_float2(fmaf(T0, f.bg[0], c0r), fmaf(T1, f.bg[0], c1r));
        *reinterpret_cast<float2*>(out_rgb + npix + pix) = make_float2(fmaf(T0, f.bg[1], c0g), fmaf(T1, f.bg[1], c1g));
        *reinterpret_cast<float2*>(out_rgb + 2 * npix + pix) = make_float2(fmaf(T0, f.bg[2], c0b), fmaf(T1, f.bg[2], c1b));
        *reinterpret_cast<float2*>(out_T + pix) = make_float2(T0, T1);
        if (COUNT) *reinterpret_cast<uint2*>(out_n + pix) = make_uint2(s.n0, s.n1);
    } else {
        if (in0) {
            out_rgb[pix] = fmaf(T0, f.bg[0], c0r);
            out_rgb[npix + pix] = fmaf(T0, f.bg[1], c0g);
            out_rgb[2 * npix + pix] = fmaf(T0, f.bg[2], c0b);
            out_T[pix] = T0;
            if (COUNT) out_n[pix] = s.n0;
        }
        if (in1) {
            out_rgb[pix + 1] = fmaf(T1, f.bg[0], c1r);
            out_rgb[npix + pix + 1] = fmaf(T1, f.bg[1], c1g);
            out_rgb[2 * npix + pix + 1] = fmaf(T1, f.bg[2], c1b);
            out_T[pix + 1] = T1;
            if (COUNT) out_n[pix + 1] = s.n1;
        }
    }
}

void launch_render_b200(const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n, int n_sm,
                        bool stats, cudaStream_t st) {
    (void)n_sm;
    const dim3 grid(f.gx, f.gy), block(QB);
    if (stats && out_n)
        launch_pdl(render_b200_kernel<true, true>, grid, block, st, f, p.ctrl, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n);
    else if (out_n)
        launch_pdl(render_b200_kernel<true, false>, grid, block, st, f, p.ctrl, p.ranges, p.ids, p.rec, out_rgb, out_T, out_n);
    else
        launch_pdl(render_b200_kernel<false, false>, grid, block, st, f, p.ctrl, p.ranges, p.ids, p.rec, out_rgb, out_T, (uint32_t*)nullptr);
}

}  // namespace gs
