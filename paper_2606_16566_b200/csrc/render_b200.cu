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
    u64 T, Cr, Cg, Cb;          // T scaled by K
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
    float t0, t1;
    unpk(s.T, t0, t1);
    if (__any_sync(0xffffffffu, (t0 < TMIN_S) || (t1 < TMIN_S))) {   // rare; a stopped pixel keeps T >= 1e-4 K: it never fires again
        float u0, u1, w10, w11, w20, w21;
        unpk(T1, u0, u1); unpk(w1, w10, w11); unpk(w2, w20, w21);
        const bool sa0 = u0 < TMIN_S, sa1 = u1 < TMIN_S;      // stopped at the first entry
        const bool sb0 = t0 < TMIN_S, sb1 = t1 < TMIN_S;      // stopped at the first or the second entry
        const u64 wm2 = pk(sb0 ? w20 : 0.0f, sb1 ? w21 : 0.0f), wm1 = pk(sa0 ? w10 : 0.0f, sa1 ? w11 : 0.0f);
        ffma2_acc(s.Cr, bc(-q1.z), wm2);
        ffma2_acc(s.Cg, bc(-q1.w), wm2);
        ffma2_acc(s.Cb, bc(-q2.x), wm2);
        ffma2_acc(s.Cr, bc(-p1.z), wm1);
        ffma2_acc(s.Cg, bc(-p1.w), wm1);
        ffma2_acc(s.Cb, bc(-p2.x), wm1);
        ffma2_acc(s.T, bc(K_SCALE), wm2);
        ffma2_acc(s.T, bc(K_SCALE), wm1);
        float r0, r1;
        unpk(s.T, r0, r1);   // the T of rule R1 passed the test when it was formed: >= 1e-4 K up to the rounding of the repair
        s.T = pk(sb0 ? fmaxf(r0, TMIN_S) : r0, sb1 ? fmaxf(r1, TMIN_S) : r1);
        ffma2_acc(s.bx2, pk(sb0 ? 1.0f : 0.0f, sb1 ? 1.0f : 0.0f), bc(POISON));
        if (COUNT) {
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
    uint2 aa = lds64u(lp);
    while (lp < lend) {
        lp += 8;
        const uint2 nx = lds64u(lp);   // the pair after this one (the list buffer has room for one pair past the padding)
        blend_pair<COUNT, GUARD>(s, aa.x, aa.y, lend);
        aa = nx;
    }
}

template <bool COUNT, bool STATS>
__global__ void __launch_bounds__(QB, 6)
render_b200_kernel(const Frame f, Ctrl* __restrict__ ctrl, const uint4* __restrict__ desc, const uint32_t* __restrict__ ids,
                   const float4* __restrict__ rec, float* __restrict__ out_rgb, float* __restrict__ out_T,
                   uint32_t* __restrict__ out_n) {
    __shared__ __align__(16) unsigned char s_rec[2][(QB + 1) * REC];  // staged, hoisted records (double-buffered) + a null record
    __shared__ __align__(16) uint32_t s_ball[2][4][4];          // [buffer][staging warp][quadrant] mask ballots
    __shared__ __align__(16) uint32_t s_indef[2][4];                        // [buffer][staging warp] batch holds an indefinite conic
    __shared__ __align__(16) uint32_t s_list[4][QB + 4];        // per-warp compacted lists of record addresses (padded to even length)
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31;
    // warp index through a warp reduction: ptxas then KNOWS it is warp-uniform (it lives in a uniform register), so
    // every trip count derived from it is uniform and the votes of the blend loop need no divergence guard
    const int w = __reduce_max_sync(0xffffffffu, tid >> 5);
    // blocks are dispatched in index order: descriptor b follows the render schedule of tile_grid_kernel (classes of
    // list length, longest first, raster order inside), so the long tiles start first and the launch has no tail
    const uint4 dsc = desc[blockIdx.x];
    const int tile = (int)dsc.x;
    const int tyi = tile / f.gx, txi = tile - tyi * f.gx;
    const int Tx = txi * TILE, Ty = tyi * TILE;
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
        s.Cr = s.Cg = s.Cb = pk(0.0f, 0.0f);
        s.n0 = s.n1 = 0;
    }
    if (tid < 6) {  // null record of both buffers: F = -huge, alpha = 0 exactly; colours 0
        float4* d = reinterpret_cast<float4*>(&s_rec[tid & 1][QB * REC]) + (tid >> 1);
        *d = make_float4(0.0f, 0.0f, 0.0f, (tid >> 1) == 0 ? -1.0e30f : 0.0f);
        if ((tid >> 1) == 2) d->y = 3.0e38f;
    }
    bool wdone = __all_sync(0xffffffffu, !in0 && !in1);
    const uint32_t start = dsc.y, end = dsc.z;
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
        // every lane stores the same words (one wavefront, no branch on the lane index)
        *reinterpret_cast<uint4*>(&s_ball[buf][w][0]) = make_uint4(b0, b1, b2, b3);
        s_indef[buf][w] = bi;
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
        list[cnt] = rec_addr + QB * REC;  // pad to an even length with the null record (alpha = 0); same word from every lane
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
    unpk(s.T, T0, T1);
    T0 *= K_INV; T1 *= K_INV;
    unpk(s.Cr, c0r, c1r); unpk(s.Cg, c0g, c1g); unpk(s.Cb, c0b, c1b);
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

// ====================================================================================================================
// Variant 5: the same blend loop, warp-specialised and persistent.
//
//   * 192 threads per CTA: 4 CONSUMER warps (one 8x8 quadrant of the current tile each, running blend_list above) and
//     2 PRODUCER warps that do all the staging (gather, tight box -> quadrant masks, double-precision hoist, per-quadrant
//     compacted lists).  Staging costs a quarter of the instructions of the kernel and all of its global-memory
//     latency; on its own warps it overlaps the blend instead of preceding it.
//   * a ring of NSTAGE stages of 64 list entries in shared memory, handed over with mbarriers (full: 64 producer
//     arrivals, empty: 4 consumer-warp arrivals) -- no CTA-wide barrier anywhere; a consumer warp is never held back by
//     a slower quadrant inside a tile, only by the ring depth.
//   * persistent CTAs walk a STATIC tile schedule in longest-list-first order (tile descriptors written by
//     tile_grid_kernel): CTA c takes descriptors c, c + G, c + 2G, ...  No tail of a few long tiles at the end of the
//     launch, and the next tile is known in advance: its descriptor, first ids and first records are prefetched while
//     the current tile is staged, so a tile switch costs no global round trip.
//   * termination (Eq. 22): a consumer warp whose 64 pixels are finished reports to a per-tile counter; when all four
//     have, the producers abandon the tile (at most NSTAGE - 1 staged batches are wasted) and the consumers skip
//     whatever stale stages of it remain.
// ====================================================================================================================
constexpr int WS_SB = 64;            // list entries per stage
constexpr int WS_NSTAGE = 3;
constexpr int WS_THREADS = 192;      // 4 consumer warps + 2 producer warps
constexpr uint32_t WS_FIRST = 1u, WS_LAST = 2u, WS_EXIT = 4u, WS_INDEF = 8u;

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}

struct WsShared {
    __align__(16) unsigned char rec[WS_NSTAGE][WS_SB * REC];  // staged, hoisted records
    __align__(16) unsigned char null_rec[REC];                // F = -huge: alpha = 0 exactly (list padding)
    __align__(16) uint32_t list[WS_NSTAGE][4][WS_SB + 4];     // per stage, per quadrant: record addresses, in list order
    __align__(16) uint4 hdr[WS_NSTAGE];                       // {flags, tile, tile sequence number, 4 x 8-bit list lengths}
    __align__(8) unsigned long long full[WS_NSTAGE], empty[WS_NSTAGE];
    uint32_t qid[2 * WS_SB];                                  // producers: queue of Gaussian ids that reach the tile
    uint32_t xchg[2][2][8];                                   // [iteration parity][producer warp]: ballot counts
    uint32_t abort_flag[2];                                   // [iteration parity]
    uint32_t done[8];                                         // consumer warps finished with tile sequence number & 7
};

// out = C + T bg (reading S16), final T, optional counts, for the two pixels of this thread
template <bool COUNT>
__device__ __forceinline__ void ws_write_pixels(const Frame& f, const PixelPair& s, int px, int py, bool in0, bool in1,
                                                float* __restrict__ out_rgb, float* __restrict__ out_T,
                                                uint32_t* __restrict__ out_n) {
    float T0, T1, c0r, c1r, c0g, c1g, c0b, c1b;
    unpk(s.T, T0, T1);
    T0 *= K_INV; T1 *= K_INV;
    unpk(s.Cr, c0r, c1r); unpk(s.Cg, c0g, c1g); unpk(s.Cb, c0b, c1b);
    const size_t npix = (size_t)f.W * f.H, pix = (size_t)py * f.W + px;
    if (in1 && !(f.W & 1)) {  // both pixels inside, 8-byte aligned pair
        __stcs(reinterpret_cast<float2*>(out_rgb + pix), make_float2(fmaf(T0, f.bg[0], c0r), fmaf(T1, f.bg[0], c1r)));
        __stcs(reinterpret_cast<float2*>(out_rgb + npix + pix), make_float2(fmaf(T0, f.bg[1], c0g), fmaf(T1, f.bg[1], c1g)));
        __stcs(reinterpret_cast<float2*>(out_rgb + 2 * npix + pix), make_float2(fmaf(T0, f.bg[2], c0b), fmaf(T1, f.bg[2], c1b)));
        __stcs(reinterpret_cast<float2*>(out_T + pix), make_float2(T0, T1));
        if (COUNT) __stcs(reinterpret_cast<uint2*>(out_n + pix), make_uint2(s.n0, s.n1));
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

// Consumer warp w = quadrant (w & 1, w >> 1) of whatever tile the stage headers announce.
template <bool COUNT, bool STATS>
__device__ __forceinline__ void ws_consumer(const Frame& f, WsShared& sm, Ctrl* __restrict__ ctrl, float* __restrict__ out_rgb,
                                            float* __restrict__ out_T, uint32_t* __restrict__ out_n, const int w,
                                            const int lane) {
    const uint32_t full0 = (uint32_t)__cvta_generic_to_shared(&sm.full[0]);
    const uint32_t empty0 = (uint32_t)__cvta_generic_to_shared(&sm.empty[0]);
    const uint32_t list0 = (uint32_t)__cvta_generic_to_shared(&sm.list[0][w][0]);
    const int lx = 8 * (w & 1) + 2 * (lane & 3), ly = 8 * (w >> 1) + (lane >> 2);
    const float x0 = (float)lx - 7.5f, x1 = x0 + 1.0f, y = (float)ly - 7.5f;  // tile-centre origin (Eq. 1)
    PixelPair s;
    s.bxy = pk(x0 * y, x1 * y);
    s.by2 = pk(y * y, y * y);
    s.bx = pk(x0, x1);
    s.by = pk(y, y);
    s.bx2 = s.T = s.Cr = s.Cg = s.Cb = pk(0.0f, 0.0f);
    s.n0 = s.n1 = 0;
    bool wdone = true, written = true, in0 = false, in1 = false;
    int px = 0, py = 0;
    uint32_t seq = 0;
    unsigned long long st_walk = 0, st_blend = 0;  // STATS only
    for (uint32_t g = 0;; g++) {
        const uint32_t slot = g % WS_NSTAGE;
        mbar_wait(full0 + 8 * slot, (g / WS_NSTAGE) & 1u);
        const uint4 h = sm.hdr[slot];
        if (h.x & WS_EXIT) break;
        if (h.x & WS_FIRST) {   // a new tile: reset the pixel state
            const int ty = (int)h.y / f.gx, tx = (int)h.y - ty * f.gx;
            px = tx * TILE + lx; py = ty * TILE + ly;
            in0 = px < f.W && py < f.H; in1 = (px + 1) < f.W && py < f.H;
            s.bx2 = pk(in0 ? x0 * x0 : POISON, in1 ? x1 * x1 : POISON);
            s.T = pk(K_SCALE, K_SCALE);
            s.Cr = s.Cg = s.Cb = pk(0.0f, 0.0f);
            s.n0 = s.n1 = 0;
            seq = h.z;
            written = false;
            wdone = __all_sync(0xffffffffu, !in0 && !in1);
            if (wdone && lane == 0) atomicAdd(&sm.done[seq & 7u], 1u);
        }
        if (!wdone) {
            const uint32_t cnt = (h.w >> (8 * w)) & 255u;
            uint32_t lp = list0 + slot * (uint32_t)(4 * (WS_SB + 4) * 4);
            const uint32_t lp0 = lp;
            uint32_t lend = lp + 4 * cnt;
            if (h.x & WS_INDEF) blend_list<COUNT, true>(s, lp, lend);
            else blend_list<COUNT, false>(s, lp, lend);
            wdone = lend == 0;
            if (STATS) st_walk += min((lp - lp0) / 4, cnt);
            if (wdone && lane == 0) atomicAdd(&sm.done[seq & 7u], 1u);
        }
        if (!written && (wdone || (h.x & WS_LAST))) {
            ws_write_pixels<COUNT>(f, s, px, py, in0, in1, out_rgb, out_T, out_n);
            if (STATS) st_blend += s.n0 + s.n1;
            written = true;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
    }
    if (STATS) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) st_blend += __shfl_xor_sync(0xffffffffu, st_blend, o);
        if (lane == 0) {
            atomicAdd(&ctrl->stats[0], st_walk);
            atomicAdd(&ctrl->stats[1], st_blend);
        }
    }
}

// The two producer warps (pt = 0..63), in lockstep through named barrier 1.
//
// Phase 1, per RAW batch of 64 list entries of the tile (one per thread; records prefetched one batch ahead, ids two):
//   the tight box of the entry against the WHOLE tile (tile_reach, ~40 instructions).  On the dense scenes 50-85 % of
//   the entries a 3-sigma rect brings into a list reach no pixel of the tile; they end here.  Survivors are appended,
//   in list order, to a queue of Gaussian ids.
// Phase 2, whenever 64 survivors are queued (or the list ends): one STAGE -- records re-read (L1), 4-bit quadrant
//   masks (Eq. 13-21), per-quadrant compacted lists, double-precision hoist (Eq. 8) -- handed to the consumers.
// So a stage holds 64 LIVE entries however sparse the list is, and the expensive part of staging runs on dense lanes.
template <bool STATS>
__device__ __forceinline__ void ws_producer(const Frame& f, WsShared& sm, Ctrl* __restrict__ ctrl, const uint4* __restrict__ desc,
                                            const uint32_t* __restrict__ ids, const float4* __restrict__ rec, const int pt) {
    const int lane = pt & 31, pw = pt >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const uint32_t full0 = (uint32_t)__cvta_generic_to_shared(&sm.full[0]);
    const uint32_t empty0 = (uint32_t)__cvta_generic_to_shared(&sm.empty[0]);
    const uint32_t null_addr = (uint32_t)__cvta_generic_to_shared(&sm.null_rec[0]);
    const int G = gridDim.x;
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    // ---- current tile: descriptor, records of the raw batch to test next, ids of the batch after -------------------
    int kn = blockIdx.x;
    uint4 dc = desc[kn];
    bool have = true;                       // false once the schedule of this CTA is exhausted
    uint32_t tile = dc.x, base = dc.y, end = dc.z;
    float4 r0 = z4, r1 = z4, r2 = z4, r3 = z4;
    uint32_t idc = 0, idn = 0;
    if (base + pt < end) {
        idc = ids[base + pt];
        const float4* q = rec + 4 * (size_t)idc;
        r0 = __ldg(q); r1 = __ldg(q + 1); r2 = __ldg(q + 2); r3 = __ldg(q + 3);
    }
    if (base + WS_SB + pt < end) idn = ids[base + WS_SB + pt];
    // ---- next tile: descriptor now, first ids and first records during the batches of the current tile ------------
    kn += G;
    bool have_n = kn < f.n_tiles;
    uint4 dn = have_n ? desc[kn] : make_uint4(0u, 0u, 0u, 0u);
    int nstate = 0;                         // 0: nothing requested, 1: ids requested, 2: records requested
    uint32_t nid = 0;
    float4 n0 = z4, n1 = z4, n2 = z4, n3 = z4;
    uint32_t seq = 0, g = 0, it = 0;
    uint32_t qhead = 0, qn = 0;             // survivor queue (circular, 2 * WS_SB ids), identical in all 64 threads
    bool emitted = false;                   // a stage of the current tile has been handed over
    unsigned long long st_staged = 0;       // STATS only

    auto next_tile = [&]() {   // switch to the next tile of the schedule (completing its prefetch when the tile was short)
        have = have_n;
        qn = 0;
        emitted = false;
        if (!have) return;
        if (nstate == 0 && dn.y + pt < dn.z) nid = ids[dn.y + pt];
        if (nstate <= 1) {
            n0 = n1 = n2 = n3 = z4;
            if (dn.y + pt < dn.z) {
                const float4* q = rec + 4 * (size_t)nid;
                n0 = __ldg(q); n1 = __ldg(q + 1); n2 = __ldg(q + 2); n3 = __ldg(q + 3);
            }
        }
        tile = dn.x; base = dn.y; end = dn.z;
        r0 = n0; r1 = n1; r2 = n2; r3 = n3;
        idc = nid;
        idn = (base + WS_SB + pt < end) ? ids[base + WS_SB + pt] : 0u;
        seq++;
        if (pt == 0) sm.done[seq & 7u] = 0;   // published to the consumers with the FIRST stage of this tile
        kn += G;
        have_n = kn < f.n_tiles;
        if (have_n) dn = desc[kn];
        nstate = 0;
    };

    while (true) {
        if (!have) {   // schedule exhausted: tell the consumers
            const uint32_t slot = g % WS_NSTAGE;
            if (g >= WS_NSTAGE) mbar_wait(empty0 + 8 * slot, ((g / WS_NSTAGE) - 1u) & 1u);
            if (pt == 0) sm.hdr[slot] = make_uint4(WS_EXIT, 0u, 0u, 0u);
            mbar_arrive(full0 + 8 * slot);
            break;
        }
        const int ty = (int)tile / f.gx, tx = (int)tile - ty * f.gx;
        const float Txf = (float)(tx * TILE), Tyf = (float)(ty * TILE);
        // ---- phase 1: which entries of the raw batch can reach the tile at all ------------------------------------
        bool alive = false;
        if (base + pt < end)
            alive = tile_reach(r0.x - Txf, r0.y - Tyf, r0.w, r1.z, r2.w, r3.x, r3.y) || (__float_as_uint(r1.w) & 1u);
        const unsigned ba = __ballot_sync(0xffffffffu, alive);
        uint32_t par = it & 1u;
        it++;
        if (lane == 0) sm.xchg[par][pw][0] = __popc(ba);
        if (pt == 0) sm.abort_flag[par] = *reinterpret_cast<volatile uint32_t*>(&sm.done[seq & 7u]) >= 4u ? 1u : 0u;
        asm volatile("bar.sync 1, 64;" ::: "memory");   // the two producer warps only
        if (sm.abort_flag[par]) {   // every pixel of the tile is finished (Eq. 22): abandon it
            next_tile();
            continue;
        }
        {
            const uint32_t a0 = sm.xchg[par][0][0], a1 = sm.xchg[par][1][0];
            if (alive) sm.qid[(qhead + qn + (pw ? a0 : 0u) + __popc(ba & lt)) & (2 * WS_SB - 1)] = idc;
            qn += a0 + a1;
        }
        if (STATS && pt == 0) st_staged += min((uint32_t)WS_SB, end - base);
        const bool raw_last = base + WS_SB >= end;
        if (!raw_last) {   // advance the raw pipeline: records of the next batch, ids of the one after
            base += WS_SB;
            idc = idn;
            r0 = r1 = r2 = r3 = z4;
            if (base + pt < end) {
                const float4* q = rec + 4 * (size_t)idc;
                r0 = __ldg(q); r1 = __ldg(q + 1); r2 = __ldg(q + 2); r3 = __ldg(q + 3);
            }
            if (base + WS_SB + pt < end) idn = ids[base + WS_SB + pt];
            if (have_n) {   // one step of the next tile's prefetch
                if (nstate == 0) {
                    if (dn.y + pt < dn.z) nid = ids[dn.y + pt];
                    nstate = 1;
                } else if (nstate == 1) {
                    n0 = n1 = n2 = n3 = z4;
                    if (dn.y + pt < dn.z) {
                        const float4* q = rec + 4 * (size_t)nid;
                        n0 = __ldg(q); n1 = __ldg(q + 1); n2 = __ldg(q + 2); n3 = __ldg(q + 3);
                    }
                    nstate = 2;
                }
            }
        }
        // ---- phase 2: hand over full stages (and the partial one when the list ends) --------------------------------
        bool aborted = false, last_done = false;   // the list's final stage (possibly empty) always carries LAST
        while (qn >= (uint32_t)WS_SB || (raw_last && !last_done)) {
            const uint32_t n = min(qn, (uint32_t)WS_SB);
            const bool last = raw_last && qn == n;
            const uint32_t slot = g % WS_NSTAGE;
            if (g >= WS_NSTAGE) mbar_wait(empty0 + 8 * slot, ((g / WS_NSTAGE) - 1u) & 1u);
            asm volatile("bar.sync 1, 64;" ::: "memory");   // the queue writes of phase 1 are visible
            float4 s0 = z4, s1 = z4, s2 = z4, s3 = z4;
            uint32_t m = 0;
            bool indefinite = false;
            if (pt < n) {
                const float4* q = rec + 4 * (size_t)sm.qid[(qhead + pt) & (2 * WS_SB - 1)];
                s0 = __ldg(q); s1 = __ldg(q + 1); s2 = __ldg(q + 2); s3 = __ldg(q + 3);
                m = quadrant_mask(s0.x - Txf, s0.y - Tyf, s0.w, s1.z, s2.w, s3.x, s3.y);
                if (__float_as_uint(s1.w) & 1u) { m = 15u; indefinite = true; }  // degenerate conic: keep everything
            }
            const unsigned b0 = __ballot_sync(0xffffffffu, m & 1u), b1 = __ballot_sync(0xffffffffu, m & 2u),
                           b2 = __ballot_sync(0xffffffffu, m & 4u), b3 = __ballot_sync(0xffffffffu, m & 8u);
            const unsigned bi = __ballot_sync(0xffffffffu, indefinite);
            par = it & 1u;
            it++;
            if (lane == 0) {
                *reinterpret_cast<uint4*>(&sm.xchg[par][pw][0]) = make_uint4(__popc(b0), __popc(b1), __popc(b2), __popc(b3));
                sm.xchg[par][pw][4] = bi ? 1u : 0u;
            }
            if (pt == 0) sm.abort_flag[par] = *reinterpret_cast<volatile uint32_t*>(&sm.done[seq & 7u]) >= 4u ? 1u : 0u;
            asm volatile("bar.sync 1, 64;" ::: "memory");
            if (sm.abort_flag[par]) { aborted = true; break; }
            const uint4 c0 = *reinterpret_cast<const uint4*>(&sm.xchg[par][0][0]), c1 = *reinterpret_cast<const uint4*>(&sm.xchg[par][1][0]);
            const bool any_indef = (sm.xchg[par][0][4] | sm.xchg[par][1][4]) != 0u;
            // per-quadrant compacted lists of record addresses, in list order (warp 0's entries first)
            const uint32_t rec_addr = (uint32_t)__cvta_generic_to_shared(&sm.rec[slot][pt * REC]);
            uint32_t* L0 = &sm.list[slot][0][0];
            constexpr int LS = WS_SB + 4;
            if (m & 1u) L0[0 * LS + (pw ? c0.x : 0u) + __popc(b0 & lt)] = rec_addr;
            if (m & 2u) L0[1 * LS + (pw ? c0.y : 0u) + __popc(b1 & lt)] = rec_addr;
            if (m & 4u) L0[2 * LS + (pw ? c0.z : 0u) + __popc(b2 & lt)] = rec_addr;
            if (m & 8u) L0[3 * LS + (pw ? c0.w : 0u) + __popc(b3 & lt)] = rec_addr;
            const uint32_t t0 = c0.x + c1.x, t1 = c0.y + c1.y, t2 = c0.z + c1.z, t3 = c0.w + c1.w;
            if (pt < 4) {   // pad every list to an even length with the null record (alpha = 0)
                const uint32_t tq = pt == 0 ? t0 : (pt == 1 ? t1 : (pt == 2 ? t2 : t3));
                L0[pt * LS + tq] = null_addr;
            }
            if (m) {  // hoist (Eq. 8) in double about the tile centre (reading S14)
                const Hoisted h = hoist(s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, Txf + 7.5f, Tyf + 7.5f, L_BIAS);
                float4* d = reinterpret_cast<float4*>(&sm.rec[slot][pt * REC]);
                d[0] = make_float4(h.A, h.B, h.C, h.F);
                d[1] = make_float4(h.D, h.E, s2.x, s2.y);
                d[2] = make_float4(s2.z, indefinite ? s1.y + L_BIAS : 3.0e38f, 0.0f, 0.0f);
            }
            if (pt == 0)
                sm.hdr[slot] = make_uint4((emitted ? 0u : WS_FIRST) | (last ? WS_LAST : 0u) | (any_indef ? WS_INDEF : 0u), tile, seq,
                                          t0 | (t1 << 8) | (t2 << 16) | (t3 << 24));
            mbar_arrive(full0 + 8 * slot);   // release: records, lists and header of this thread are visible to the waiters
            g++;
            emitted = true;
            last_done = last;
            qhead = (qhead + n) & (2 * WS_SB - 1);
            qn -= n;
        }
        if (aborted || raw_last) next_tile();
    }
    if (STATS && pt == 0) atomicAdd(&ctrl->stats[2], st_staged);
}

template <bool COUNT, bool STATS>
__global__ void __launch_bounds__(WS_THREADS, 4)
render_ws_kernel(const Frame f, Ctrl* __restrict__ ctrl, const uint4* __restrict__ desc, const uint32_t* __restrict__ ids,
                 const float4* __restrict__ rec, float* __restrict__ out_rgb, float* __restrict__ out_T,
                 uint32_t* __restrict__ out_n) {
    __shared__ WsShared sm;
    griddep_sync();
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int k = 0; k < WS_NSTAGE; k++) {
            mbar_init((uint32_t)__cvta_generic_to_shared(&sm.full[k]), WS_SB);
            mbar_init((uint32_t)__cvta_generic_to_shared(&sm.empty[k]), 4);
        }
    }
    if (tid < 8) sm.done[tid] = 0;
    if (tid >= 32 && tid < 35) {   // null record: F = -huge -> alpha = 0 exactly; colours 0; guard never trips
        float4* d = reinterpret_cast<float4*>(&sm.null_rec[0]) + (tid - 32);
        *d = make_float4(0.0f, tid == 34 ? 3.0e38f : 0.0f, 0.0f, tid == 32 ? -1.0e30f : 0.0f);
    }
    __syncthreads();
    // warp index through a warp reduction: ptxas then knows it is warp-uniform
    const int w = __reduce_max_sync(0xffffffffu, tid >> 5);
    if (w < 4) ws_consumer<COUNT, STATS>(f, sm, ctrl, out_rgb, out_T, out_n, w, tid & 31);
    else ws_producer<STATS>(f, sm, ctrl, desc, ids, rec, tid - 128);
}

void launch_render_ws(const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n, int n_sm, bool stats,
                      cudaStream_t st) {
    const int g = f.n_tiles < n_sm * 4 ? f.n_tiles : n_sm * 4;
    const dim3 grid(g), block(WS_THREADS);
    if (stats && out_n)
        launch_pdl(render_ws_kernel<true, true>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else if (out_n)
        launch_pdl(render_ws_kernel<true, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else
        launch_pdl(render_ws_kernel<false, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, (uint32_t*)nullptr);
}

void launch_render_b200(const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n, int n_sm,
                        bool stats, cudaStream_t st) {
    (void)n_sm;
    const dim3 grid(f.n_tiles), block(QB);
    if (stats && out_n)
        launch_pdl(render_b200_kernel<true, true>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else if (out_n)
        launch_pdl(render_b200_kernel<true, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else
        launch_pdl(render_b200_kernel<false, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, (uint32_t*)nullptr);
}

}  // namespace gs
