// render_blend.cuh -- what the B200 render kernels share: the packed f32x2 pixel-pair
// state, the biased-exponent alpha (Eq. 9-10 in the log2 domain), shared-memory loads, cp.async / mbarrier
// helpers and the epilogue.  Product code; shares nothing with oracle/.
#pragma once
#include "render_common.cuh"

namespace gs {

constexpr int QB = 128;            // threads per block == staged entries per batch
constexpr float POISON = 1.0e18f;  // x' of a finished pixel: (A * POISON + H) * POISON <= -1e3 for every conic with a >= 1e-33 and |H| < 1e-15 a
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
    u64 bx;                     // x' of the two pixels, tile-centre origin (B_local of Eq. 9 in separable form, see alpha_pair)
    float y, y2;                // y' and y'^2: the two pixels of a thread share their row
    u64 T, Cr, Cg, Cb;          // T scaled by K
    uint32_t n0, n1;
};

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts128f(uint32_t addr, float x, float y, float z, float w) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds32u(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint2 lds64u(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
    return v;
}

// Exponent and alpha of one staged record for the two pixels of this thread: alpha / K, clamped (Eq. 10 in the biased
// log2 domain, separable form: 3 FFMA for the shared row part + 2 FFMA2 -- Table I has "5 FMA" per pixel; exactly 0 below
// the 1/255 floor; min(0.99, .)).
template <bool GUARD>
__device__ __forceinline__ u64 alpha_pair(const PixelPair& s, const float4 q0, const float4 q1, const float guard, float& e0,
                                          float& e1) {
    const float H = fmaf(q0.y, s.y, q1.x);                       // B y' + D
    const float G = fmaf(q0.z, s.y2, fmaf(q1.y, s.y, q0.w));     // C y'^2 + E y' + F
    const u64 L2 = ffma2(ffma2(bc(q0.x), s.bx, bc(H)), s.bx, bc(G));   // (A x' + H) x' + G
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

// out = C + T bg (reading S16), final T, optional counts, for the two pixels of this thread
template <bool COUNT>
__device__ __forceinline__ void write_pixels(const Frame& f, const PixelPair& s, int px, int py, bool in0,
                                             bool in1, float* __restrict__ out_rgb, float* __restrict__ out_T,
                                             uint32_t* __restrict__ out_n) {
    float T0, T1, c0r, c1r, c0g, c1g, c0b, c1b;
    unpk(s.T, T0, T1);
    unpk(s.Cr, c0r, c1r); unpk(s.Cg, c0g, c1g); unpk(s.Cb, c0b, c1b);
    T0 *= K_INV; T1 *= K_INV;
    const size_t npix = (size_t)f.W * f.H, pix = (size_t)py * f.W + px;
    if (in0) GS_BOUND(pix, npix);
    if (in1) GS_BOUND(pix + 1, npix);
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

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

}  // namespace gs
