// render_common.cuh -- device helpers of the render kernels: tile-local hoisting (Eq. 1-10) and the
// tight box / warp visibility mask (Eq. 13-21).  Product code; shares nothing with oracle/.
#pragma once
#include "common.cuh"

namespace gs {

constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
constexpr float L2_ALPHA_MIN = -7.994353436858858f;  // log2(1/255): the opacity floor in the log2 domain
constexpr float ALPHA_MIN = 1.0f / 255.0f;
constexpr float ALPHA_MAX = 0.99f;
constexpr float T_MIN = 0.0001f;

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Hoist transformation (Eq. 8, reading G2), in the log2 domain:
//   log2(alpha)(x', y') = A x'^2 + B x'y' + C y'^2 + D x' + E y' + F,   (x', y') relative to the origin (ox, oy),
//   A = -a k/2, B = -b k, C = -c k/2, D = (a dx + b dy) k, E = (b dx + c dy) k,
//   F = log2(o) - (a dx^2 + 2 b dx dy + c dy^2) k / 2,   (dx, dy) = mu - origin (Eq. 2),  k = log2(e).
// Evaluated in double and rounded once: D, E, F are sums of large cancelling terms for far-centred splats
// (reading S14), and this runs once per (tile, Gaussian), off the per-pixel path.
struct Hoisted { float A, B, C, D, E, F; };
// exact fp32 -> fp64 conversion (plain cvt: under -use_fast_math a C++ cast first flushes denormals with an FMUL)
__device__ __forceinline__ double f2d(float x) {
    double d;
    asm("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(x));
    return d;
}
// round-to-nearest fp64 -> fp32 conversion (plain cvt: under -use_fast_math a C++ cast adds a compare and a multiply per
// value to flush denormal results, which no coefficient here can be)
__device__ __forceinline__ float d2f(double x) {
    float f;
    asm("cvt.rn.f32.f64 %0, %1;" : "=f"(f) : "d"(x));
    return f;
}
__device__ __forceinline__ Hoisted hoist(float mux, float muy, float a, float b, float c, float log2o, float ox, float oy,
                                         float bias = 0.0f) {
    const double k = 1.4426950408889634;
    const double dx = f2d(mux) - f2d(ox), dy = f2d(muy) - f2d(oy);
    const double da = f2d(a), db = f2d(b), dc = f2d(c);
    const double gx = da * dx + db * dy, gy = db * dx + dc * dy;
    Hoisted h;
    // A, B, C: one fp32 multiplication each (within 1 ulp of the double product rounded once; they multiply |x'|, |y'| <= 7.5).
    // D, E, F are sums of large cancelling terms for far-centred splats and stay in double (reading S14); conversions
    // run at a quarter of the issue rate, so only what needs them goes through double.
    h.A = a * -0.7213475204444817f;   // -k/2
    h.B = b * -1.4426950408889634f;   // -k
    h.C = c * -0.7213475204444817f;
    h.D = d2f(k * gx);
    h.E = d2f(k * gy);
    h.F = d2f((f2d(log2o) + f2d(bias)) - 0.5 * k * (gx * dx + gy * dy));
    return h;
}

// Tight box (Eq. 13-19): vertical extent [ymin, ymax] (centre-relative) of the ellipse
// a x^2 + 2 b x y + c y^2 <= tau restricted to the column x in [x0, x1] (centre-relative, Eq. 14).
// Returns false when the ellipse misses the column.  det = a c - b^2 > 0 is required.
__device__ __forceinline__ bool column_span(float a, float b, float c, float det, float tau, float x0, float x1,
                                            float& ymin, float& ymax) {
    const float dy = sqrtf(__fdividef(a * tau, det));   // Eq. 16
    const float ct = c * tau;
    const float ic = __fdividef(1.0f, c);
    const float ax0 = a * x0, ax1 = a * x1;
    // upper branch: peak vertex at x = -b dy / a (division-free test)
    const float tu = -b * dy;
    if (tu < ax0 || tu > ax1) {
        const float xs = (tu < ax0) ? x0 : x1;           // Case A (Eq. 17) / Case B (Eq. 18)
        const float disc = ct - det * xs * xs;
        if (disc < 0.0f) return false;
        ymax = (-b * xs + sqrtf(disc)) * ic;
    } else {
        ymax = dy;                                       // Case C
    }
    // lower branch: "identical conditional logic with reversed signs for the linear terms"
    const float tl = b * dy;
    if (tl < ax0 || tl > ax1) {
        const float xs = (tl < ax0) ? x0 : x1;
        const float disc = ct - det * xs * xs;
        if (disc < 0.0f) return false;
        ymin = (-b * xs - sqrtf(disc)) * ic;
    } else {
        ymin = -dy;
    }
    return true;
}

// Threshold of the alpha >= 1/255 ellipse, tau = 2 ln(255 o), from log2(o), widened so that fp32
// rounding in column_span can never cull a contributing pixel (any conservative mask is correct; S13).
__device__ __forceinline__ float tau_widened(float log2o) {
    const float tau = 2.0f * LN2 * (log2o - L2_ALPHA_MIN);
    return tau + 0.02f + 1e-5f * fabsf(tau);
}
constexpr float SPAN_EPS = 2e-3f;  // widening of the vertical span, pixels

// ---- B200 staging: the same tight box (Eq. 13-19), branch-free, with its per-Gaussian part hoisted into preprocess ----
// Per Gaussian (once per frame, preprocess.cu): the vertex abscissa of the upper boundary x* = -b d_y / a
// (Eq. 16 + PAPER.md:198), 1/c and c tau.  Per (tile, Gaussian) (render_b200.cu): Cases A/B/C of Eq. 17-18 collapse to
// x_s = clamp(+-x*, x0, x1) because the upper boundary y(x) = (-b x + sqrt(c tau - det x^2)) / c is concave with its
// maximum at x* (the lower one convex with its minimum at -x*); the column misses the ellipse iff c tau - det x_s^2 < 0.
struct TightBox { float xstar, ic, ct; bool degenerate; };
__device__ __forceinline__ TightBox tight_box_constants(float a, float b, float c, float det, float log2o) {
    TightBox t;
    const float tau = tau_widened(log2o);
    t.degenerate = !(det > 0.0f) || !(a > 0.0f) || !(c > 0.0f);
    const float dy = sqrtf(a * tau / det);        // Eq. 16
    t.xstar = -b * dy / a;
    t.ic = 1.0f / c;
    t.ct = c * tau;
    if (!(tau > 0.0f)) { t.xstar = 0.0f; t.ct = -1.0f; }  // o <= 1/255: never visible (reading S13)
    if (!(fabsf(t.xstar) <= 3.0e38f) || !(fabsf(t.ic) <= 3.0e38f) || !(fabsf(t.ct) <= 3.0e38f)) t.degenerate = true;
    return t;
}

// Quadrant hits of one (tile, Gaussian): q[col + 2 band] is set when the alpha >= 1/255 ellipse can reach a pixel of
// the 8x8 quadrant (columns 8 col .. 8 col + 7, rows 8 band .. 8 band + 7) -- Eq. 19-21 with 8-row bands, evaluated for
// the two 8-pixel sub-columns.  (dxc, dyc) = centre relative to the tile corner.  Conservative by the widening of tau
// and SPAN_EPS; a row band is hit iff an INTEGER row lies in [ymin, ymax] (PAPER.md:216 ceil/floor).  The four results
// are predicates (they feed the warp ballots directly; no mask word is assembled and taken apart again).
__device__ __forceinline__ void quadrant_hits(float dxc, float dyc, float b, float det, float xstar, float ic, float ct,
                                              bool (&q)[4]) {
#pragma unroll
    for (int col = 0; col < 2; col++) {
        const float x0 = 8.0f * col - dxc, x1 = x0 + 7.0f;      // Eq. 14, centre-relative
        const float xu = fminf(fmaxf(xstar, x0), x1), xl = fminf(fmaxf(-xstar, x0), x1);
        const float du = fmaf(-det * xu, xu, ct), dl = fmaf(-det * xl, xl, ct);
        const float ymax = fmaf(fmaf(-b, xu, sqrtf(fmaxf(du, 0.0f))), ic, dyc + SPAN_EPS);   // Eq. 17 / 18 / Case C
        const float ymin = fmaf(fmaf(-b, xl, -sqrtf(fmaxf(dl, 0.0f))), ic, dyc - SPAN_EPS);
        // misses (du or dl < 0) are folded into the comparison operand, so the whole test is straight-line selects
        const float top = floorf((fminf(du, dl) >= 0.0f) ? ymax : -1.0f);   // floor(min(top, 7)) = min(floor(top), 7)
        q[col] = fminf(top, 7.0f) >= fmaxf(ymin, 0.0f);
        q[col + 2] = fminf(top, 15.0f) >= fmaxf(ymin, 8.0f);
    }
}

// Rows [r0, r1] (tile-local, clamped to [0, 15]) of the tile column [ox + cx0, ox + cx1] that the ellipse can reach;
// r0 > r1 when empty.  (mux, muy) - (ox, oy) = centre relative to the tile corner.
__device__ __forceinline__ void column_rows(float dxc, float dyc, float a, float b, float c, float det, float tau,
                                            float cx0, float cx1, int& r0, int& r1) {
    float ymin, ymax;
    r0 = 1; r1 = 0;
    if (!(det > 0.0f) || !(a > 0.0f) || !(c > 0.0f)) { r0 = 0; r1 = 15; return; }  // degenerate conic: keep everything
    if (!column_span(a, b, c, det, tau, cx0 - dxc, cx1 - dxc, ymin, ymax)) return;
    const float lo = ceilf(dyc + ymin - SPAN_EPS), hi = floorf(dyc + ymax + SPAN_EPS);  // Eq. 19 + ceil/floor
    if (!(lo <= hi)) {  // NaN-safe: a NaN keeps everything
        if (lo != lo || hi != hi) { r0 = 0; r1 = 15; }
        return;
    }
    r0 = (int)fmaxf(lo, 0.0f);
    r1 = (int)fminf(hi, 15.0f);
}

}  // namespace gs
