// preprocess.cu -- per-Gaussian preprocess (DESIGN.md steps C-P0..C-P9), fused with
//   * order-preserving compaction of the visible Gaussians (single-pass chained scan, decoupled look-back),
//   * the global digit histograms of the depth bits (for the depth radix sort),
//   * the 2-D difference grid of tile coverage (from which tile counts and tile ranges follow without ever
//     reading the duplicated keys).
//
// Arithmetic contract: C-P0..C-P8 are evaluated in IEEE binary32 with ONE rounding per written operation, in the
// canonical order of DESIGN.md -- every operation below is an explicit round-to-nearest intrinsic
// (__fmul_rn/__fadd_rn/__fsub_rn/__fdiv_rn/__fsqrt_rn are never contracted into FMAs and ignore -use_fast_math),
// so depth bits, radius, rect and tiles_touched are unique integers any conforming implementation reproduces.
// C-P9 (SH colour) is free-order fp32 (a toleranced output).
#include "render_common.cuh"

namespace gs {

__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float dvd(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float sqr(float a) { return __fsqrt_rn(a); }
// ((m0*x + m1*y) + m2*z) + m3
__device__ __forceinline__ float affine(const float* m, float x, float y, float z) {
    return add(add(add(mul(m[0], x), mul(m[1], y)), mul(m[2], z)), m[3]);
}
__device__ __forceinline__ float dot3(float a0, float a1, float a2, float b0, float b1, float b2) {
    return add(add(mul(a0, b0), mul(a1, b1)), mul(a2, b2));
}

struct float5 { float a, b, c, d, e; };
struct Splat {
    float mux, muy, ca, cb, cc, depth;
    float tau;   // tile-cull modes: the upper bound of 2 ln(255 o) of C-P8' (0 in the standard mode)
    int radius, xmin, ymin, xmax, ymax;
};

// Library-free UPPER bound of tau = 2 ln(255 o), o > 1/255: 255 o = 2^e m, ln m <= (m - 1) / sqrt(m) on
// [1, 2] (at most 0.014 above), + 1e-5; fp32, one rounding per operation (C-P8').
__device__ __forceinline__ float tau_upper(float opacity) {
    const float x255 = mul(255.0f, opacity);
    const uint32_t xb = __float_as_uint(x255);
    const int e2 = (int)(xb >> 23) - 127;
    const float m = __uint_as_float((xb & 0x007fffffu) | 0x3f800000u);
    const float lnm = dvd(sub(m, 1.0f), sqr(m));
    return add(mul(2.0f, add(mul((float)e2, 0.693147182f), lnm)), 1e-5f);
}

// C-P0..C-P8.  Returns false when the Gaussian is culled.
__device__ __forceinline__ bool project(const Frame& f, float px, float py, float pz, float sx, float sy, float sz,
                                        float qw, float qx, float qy, float qz, float opacity, Splat& o) {
    const float* V = f.V;
    const float* PM = f.PM;
    const float Wf = (float)f.W, Hf = (float)f.H;
    // C-P0 camera space; near plane 0.2 (reading S2)
    const float pc0 = affine(V + 0, px, py, pz), pc1 = affine(V + 4, px, py, pz), pc2 = affine(V + 8, px, py, pz);
    if (!(pc2 > 0.2f)) return false;
    // C-P1 clip -> pixel (reading S1)
    const float h0 = affine(PM + 0, px, py, pz), h1 = affine(PM + 4, px, py, pz), h3 = affine(PM + 12, px, py, pz);
    const float iw = dvd(1.0f, add(h3, 1e-7f));
    const float ndcx = mul(h0, iw), ndcy = mul(h1, iw);
    const float mux = mul(sub(mul(add(ndcx, 1.0f), Wf), 1.0f), 0.5f);
    const float muy = mul(sub(mul(add(ndcy, 1.0f), Hf), 1.0f), 0.5f);
    if (!(fabsf(mux) <= 1.0e9f) || !(fabsf(muy) <= 1.0e9f)) return false;
    // C-P2 rotation (reading S19)
    const float R00 = sub(1.0f, mul(2.0f, add(mul(qy, qy), mul(qz, qz))));
    const float R01 = mul(2.0f, sub(mul(qx, qy), mul(qw, qz)));
    const float R02 = mul(2.0f, add(mul(qx, qz), mul(qw, qy)));
    const float R10 = mul(2.0f, add(mul(qx, qy), mul(qw, qz)));
    const float R11 = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qz, qz))));
    const float R12 = mul(2.0f, sub(mul(qy, qz), mul(qw, qx)));
    const float R20 = mul(2.0f, sub(mul(qx, qz), mul(qw, qy)));
    const float R21 = mul(2.0f, add(mul(qy, qz), mul(qw, qx)));
    const float R22 = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qy, qy))));
    // C-P3 Sigma = (R S)(R S)^T
    const float M00 = mul(R00, sx), M01 = mul(R01, sy), M02 = mul(R02, sz);
    const float M10 = mul(R10, sx), M11 = mul(R11, sy), M12 = mul(R12, sz);
    const float M20 = mul(R20, sx), M21 = mul(R21, sy), M22 = mul(R22, sz);
    const float S00 = dot3(M00, M01, M02, M00, M01, M02);
    const float S01 = dot3(M00, M01, M02, M10, M11, M12);
    const float S02 = dot3(M00, M01, M02, M20, M21, M22);
    const float S11 = dot3(M10, M11, M12, M10, M11, M12);
    const float S12 = dot3(M10, M11, M12, M20, M21, M22);
    const float S22 = dot3(M20, M21, M22, M20, M21, M22);
    // C-P4 Jacobian with the 1.3 guard band (reading S3)
    const float limx = mul(1.3f, dvd(mul(0.5f, Wf), f.fx));
    const float limy = mul(1.3f, dvd(mul(0.5f, Hf), f.fy));
    const float tx = mul(fminf(limx, fmaxf(-limx, dvd(pc0, pc2))), pc2);
    const float ty = mul(fminf(limy, fmaxf(-limy, dvd(pc1, pc2))), pc2);
    const float tz = pc2;
    const float j00 = dvd(f.fx, tz);
    const float j02 = -dvd(mul(f.fx, tx), mul(tz, tz));
    const float j11 = dvd(f.fy, tz);
    const float j12 = -dvd(mul(f.fy, ty), mul(tz, tz));
    // C-P5 cov2D = T Sigma T^T, T = J W, + 0.3 px dilation (reading S4)
    const float T00 = add(mul(j00, V[0]), mul(j02, V[8])), T01 = add(mul(j00, V[1]), mul(j02, V[9])),
                T02 = add(mul(j00, V[2]), mul(j02, V[10]));
    const float T10 = add(mul(j11, V[4]), mul(j12, V[8])), T11 = add(mul(j11, V[5]), mul(j12, V[9])),
                T12 = add(mul(j11, V[6]), mul(j12, V[10]));
    const float U00 = dot3(T00, T01, T02, S00, S01, S02), U01 = dot3(T00, T01, T02, S01, S11, S12),
                U02 = dot3(T00, T01, T02, S02, S12, S22);
    const float U10 = dot3(T10, T11, T12, S00, S01, S02), U11 = dot3(T10, T11, T12, S01, S11, S12),
                U12 = dot3(T10, T11, T12, S02, S12, S22);
    float c00 = dot3(U00, U01, U02, T00, T01, T02);
    const float c01 = dot3(U00, U01, U02, T10, T11, T12);
    float c11 = dot3(U10, U11, U12, T10, T11, T12);
    c00 = add(c00, 0.3f);
    c11 = add(c11, 0.3f);
    // C-P6 conic (Eq. 5); cull if !(det > 0) (reading S7)
    const float det = sub(mul(c00, c11), mul(c01, c01));
    if (!(det > 0.0f)) return false;
    const float inv = dvd(1.0f, det);
    o.ca = mul(c11, inv);
    o.cb = -mul(c01, inv);
    o.cc = mul(c00, inv);
    // C-P7 3-sigma radius (reading S5)
    const float mid = mul(0.5f, add(c00, c11));
    const float sq = sqr(fmaxf(0.1f, sub(mul(mid, mid), det)));
    const float lam = fmaxf(add(mid, sq), sub(mid, sq));
    const float rf_ = ceilf(mul(3.0f, sqr(lam)));
    if (!(rf_ <= 1.0e9f)) return false;
    const int radius = (int)rf_;
    // C-P8 tile rect, half-open, clamped to the grid (reading S6)
    const float rf = (float)radius;
    float rxf = rf, ryf = rf;
    o.tau = 0.0f;
    if (f.tile_cull) {
        // C-P8' (gs_set_tile_cull(1)): the square intersected with the bounding box of the ellipse
        // alpha >= 1/255, i.e. a dx^2 + 2 b dx dy + c dy^2 <= tau = 2 ln(255 o), half-extents
        // sqrt(tau c / det) and sqrt(tau a / det).  tau is a library-free UPPER bound (255 o = 2^e m, ln m <= (m - 1) /
        // sqrt(m) on [1, 2], + 1e-5); the extents are formed in double from the fp32 conic the blend uses; every operation
        // is one explicit IEEE rounding, as in the rest of this function, so the rect is bit-reproducible.
        if (!(mul(255.0f, opacity) > 1.0f)) return false;   // alpha < 1/255 everywhere: never blended
        const float tau = tau_upper(opacity);
        o.tau = tau;
        const double dd = __dsub_rn(__dmul_rn((double)o.ca, (double)o.cc), __dmul_rn((double)o.cb, (double)o.cb));
        if (dd > 0.0 && o.ca > 0.0f && o.cc > 0.0f) {
            const double hx = __dsqrt_rn(__ddiv_rn(__dmul_rn((double)tau, (double)o.cc), dd));
            const double hy = __dsqrt_rn(__ddiv_rn(__dmul_rn((double)tau, (double)o.ca), dd));
            if (hx < 1.0e9) rxf = fminf(rf, add((float)ceil(hx), 1.0f));
            if (hy < 1.0e9) ryf = fminf(rf, add((float)ceil(hy), 1.0f));
        }
    }
    const float gxf = (float)f.gx, gyf = (float)f.gy;
    const int xmin = (int)fminf(gxf, fmaxf(0.0f, floorf(dvd(sub(mux, rxf), 16.0f))));
    const int xmax = (int)fminf(gxf, fmaxf(0.0f, floorf(dvd(add(add(mux, rxf), 15.0f), 16.0f))));
    const int ymin = (int)fminf(gyf, fmaxf(0.0f, floorf(dvd(sub(muy, ryf), 16.0f))));
    const int ymax = (int)fminf(gyf, fmaxf(0.0f, floorf(dvd(add(add(muy, ryf), 15.0f), 16.0f))));
    if ((xmax - xmin) * (ymax - ymin) <= 0) return false;
    o.mux = mux; o.muy = muy; o.depth = pc2; o.radius = radius;
    o.xmin = xmin; o.ymin = ymin; o.xmax = xmax; o.ymax = ymax;
    return true;
}

// C-P9: colour = max(0, 0.5 + sum_k (-1)^m Y_lm(d) sh[k]), k = l^2 + l + m, d = unit vector camera -> Gaussian
// ("view-dependent color parameterized by spherical harmonics"; reading S8).  DEG is a template parameter
// so that the basis lives in registers (a runtime degree indexes the array dynamically and spills it to local memory).
template <int DEG>
__device__ __forceinline__ void sh_basis(const Frame& f, float px, float py, float pz, float* Y) {
    float x = px - f.campos[0], y = py - f.campos[1], z = pz - f.campos[2];
    const float rn = rsqrtf(x * x + y * y + z * z);
    x *= rn; y *= rn; z *= rn;
    Y[0] = 0.28209479177387814f;
    if (DEG >= 1) {
        Y[1] = -0.4886025119029199f * y;
        Y[2] = 0.4886025119029199f * z;
        Y[3] = -0.4886025119029199f * x;
    }
    if (DEG >= 2) {
        const float xx = x * x, yy = y * y, zz = z * z;
        Y[4] = 1.0925484305920792f * x * y;
        Y[5] = -1.0925484305920792f * y * z;
        Y[6] = 0.31539156525252005f * (2.0f * zz - xx - yy);
        Y[7] = -1.0925484305920792f * x * z;
        Y[8] = 0.5462742152960396f * (xx - yy);
        if (DEG >= 3) {
            Y[9] = -0.5900435899266435f * y * (3.0f * xx - yy);
            Y[10] = 2.890611442640554f * x * y * z;
            Y[11] = -0.4570457994644658f * y * (4.0f * zz - xx - yy);
            Y[12] = 0.3731763325901154f * z * (2.0f * zz - 3.0f * xx - 3.0f * yy);
            Y[13] = -0.4570457994644658f * x * (4.0f * zz - xx - yy);
            Y[14] = 1.445305721320277f * z * (xx - yy);
            Y[15] = -0.5900435899266435f * x * (xx - 3.0f * yy);
        }
    }
}

// The lane reads its own coefficients (3, 12, 27 or 48 floats; 16-byte loads where the count allows).
template <int DEG>
__device__ __forceinline__ float3 sh_colour_direct(const Frame& f, const float* __restrict__ sh, int i, float px, float py,
                                                   float pz) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    float Y[K];
    sh_basis<DEG>(f, px, py, pz, Y);
    float c[3 * K];
    if (K % 4 == 0) {
        const float4* s4 = reinterpret_cast<const float4*>(sh + (size_t)i * (3 * K));
#pragma unroll
        for (int k = 0; k < 3 * K / 4; k++) {
            const float4 v = __ldcs(s4 + k);
            c[4 * k] = v.x; c[4 * k + 1] = v.y; c[4 * k + 2] = v.z; c[4 * k + 3] = v.w;
        }
    } else {
        const float* s1 = sh + (size_t)i * (3 * K);
#pragma unroll
        for (int k = 0; k < 3 * K; k++) c[k] = __ldcs(s1 + k);
    }
    float r = 0.5f, g = 0.5f, b = 0.5f;
#pragma unroll
    for (int k = 0; k < K; k++) {
        r = fmaf(Y[k], c[3 * k], r); g = fmaf(Y[k], c[3 * k + 1], g); b = fmaf(Y[k], c[3 * k + 2], b);
    }
    return make_float3(fmaxf(r, 0.0f), fmaxf(g, 0.0f), fmaxf(b, 0.0f));
}

// Small scenes (P < COMPACT_MIN_P, one wave of warps): one WARP processes one 32-Gaussian sub-tile at a time, sub-tiles
// assigned statically, no inter-warp dependency and no block barrier inside the loop.  Nothing is compacted: a single
// wave gives a chained scan nothing to overlap with (its inclusive prefixes advance 32 sub-tiles per L2 round trip,
// ~25 us for 100 000 Gaussians), so every Gaussian writes a key -- culled ones the all-ones key that sorts behind every
// depth -- and the depth sort runs over all P keys.
template <int DEG>
__global__ void __launch_bounds__(PRE_THREADS)
preprocess_kernel(const Frame f, const Pointers p, const float* __restrict__ means, const float* __restrict__ scales,
                  const float* __restrict__ rots, const float* __restrict__ opac, const float* __restrict__ sh) {
    __shared__ uint32_t s_hist[MAX_SORT_PASSES_DEPTH][256];
    __shared__ uint32_t s_nvis;
    __shared__ int s_cdiff[CDIFF_SMEM];   // super-tile coverage (difference grid) of this block's Gaussians
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31;
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += PRE_THREADS) (&s_hist[0][0])[k] = 0;
    const bool cdiff_shared = f.cdiff_cells <= CDIFF_SMEM;
    if (cdiff_shared)
        for (int k = tid; k < f.cdiff_cells; k += PRE_THREADS) s_cdiff[k] = 0;
    int* const cdiff = cdiff_shared ? s_cdiff : p.cdiff;
    const int cgw = f.cgx + 1;
    if (tid == 0) s_nvis = 0;
    __syncthreads();
    const int n_tiles = (f.P + 31) / 32;
    const int gw = f.gx + 1;
    const int gwarp = blockIdx.x * (PRE_THREADS / 32) + (tid >> 5), n_warps = gridDim.x * (PRE_THREADS / 32);
    // coverage grid copy of this warp: the corner counters of a small grid are hot (hundreds of atomics per address,
    // serialised in L2), so they are spread over diff_copies replicas that tile_grid_kernel adds up
    int* diff = p.diff + (size_t)(gwarp & (f.diff_copies - 1)) * f.diff_cells;
    for (int tile = gwarp; tile < n_tiles; tile += n_warps) {
        const int i = tile * 32 + lane;
        Splat s = {};
        bool vis = false;
        float px = 0.f, py = 0.f, pz = 0.f;
        if (i < f.P) {
            // plain loads: the three components of a lane share their cache lines with the neighbouring lanes
            px = __ldg(means + 3 * (size_t)i); py = __ldg(means + 3 * (size_t)i + 1); pz = __ldg(means + 3 * (size_t)i + 2);
            const float sx = __ldg(scales + 3 * (size_t)i), sy = __ldg(scales + 3 * (size_t)i + 1), sz = __ldg(scales + 3 * (size_t)i + 2);
            const float4 q = __ldcs(reinterpret_cast<const float4*>(rots) + i);
            vis = project(f, px, py, pz, sx, sy, sz, q.x, q.y, q.z, q.w, f.tile_cull ? __ldg(opac + i) : 1.0f, s);
        }
        const uint32_t cnt = __popc(__ballot_sync(0xffffffffu, vis));
        if (lane == 0 && cnt) atomicAdd(&s_nvis, cnt);
        if (i < f.P) {
            uint4 pg = make_uint4(0u, 0u, 0u, 0u);
            if (vis) {
                pg.x = (uint32_t)s.xmin | ((uint32_t)s.ymin << 16);
                pg.y = (uint32_t)s.xmax | ((uint32_t)s.ymax << 16);
                pg.z = __float_as_uint(s.depth);
                pg.w = (uint32_t)s.radius;
            }
            GS_BOUND(i, f.P);
            p.per_g[i] = pg;
            // a culled Gaussian sorts behind every depth: digit 255 in all four passes
            const uint32_t db = vis ? __float_as_uint(s.depth) : 0xffffffffu;
            atomicAdd(&s_hist[0][db & 255u], 1u);
            atomicAdd(&s_hist[1][(db >> 8) & 255u], 1u);
            atomicAdd(&s_hist[2][(db >> 16) & 255u], 1u);
            atomicAdd(&s_hist[3][db >> 24], 1u);
            p.gkeyA[i] = vis ? (((unsigned long long)db << 32) | (unsigned)i) : ~0ull;
        }
        if (vis) {
            GS_BOUND(s.ymax * gw + s.xmax, f.diff_cells); GS_BOUND(s.ymin * gw + s.xmin, f.diff_cells);
            atomicAdd(diff + s.ymin * gw + s.xmin, 1);
            atomicAdd(diff + s.ymin * gw + s.xmax, -1);
            atomicAdd(diff + s.ymax * gw + s.xmin, -1);
            atomicAdd(diff + s.ymax * gw + s.xmax, 1);
            if (f.n_ctiles) {   // the same rect on the super-tile grid (two-level binning: the grid duplication + sort run on)
                const int cs = f.cshift, cr = (1 << cs) - 1;
                const int cx0 = s.xmin >> cs, cy0 = s.ymin >> cs;
                const int cx1 = (s.xmax + cr) >> cs, cy1 = (s.ymax + cr) >> cs;
                GS_BOUND(cy1 * cgw + cx1, f.cdiff_cells);
                atomicAdd(cdiff + cy0 * cgw + cx0, 1);
                atomicAdd(cdiff + cy0 * cgw + cx1, -1);
                atomicAdd(cdiff + cy1 * cgw + cx0, -1);
                atomicAdd(cdiff + cy1 * cgw + cx1, 1);
            }
            const float o = __ldcs(opac + i);
            const float3 col = sh_colour_direct<DEG>(f, sh, i, px, py, pz);
            // det of the STORED conic, exact products in double (24+24 bits): the form is indefinite iff det <= 0,
            // and the tight box of the render stage needs det without fp32 cancellation (needle-like splats)
            const double dd = (double)s.ca * (double)s.cc - (double)s.cb * (double)s.cb;
            const float l2o = log2f(o);
            const TightBox tb = tight_box_constants(s.ca, s.cb, s.cc, (float)dd, l2o);
            const uint32_t flags = (!(dd > 0.0) || tb.degenerate) ? 1u : 0u;
            float4* rec = p.rec + 4 * (size_t)i;  // 64-byte render record (include/gs.h: gs_intermediates.record)
            rec[0] = make_float4(s.mux, s.muy, s.cb, (float)dd);          // the half the tight box needs ...
            rec[1] = make_float4(tb.xstar, tb.ic, tb.ct, __uint_as_float(flags));
            rec[2] = make_float4(s.ca, s.cc, l2o, col.x);                   // ... and the half only the hoist needs
            rec[3] = make_float4(col.y, col.z, 0.0f, s.tau);                 // [15]: C-P8' tau (0 in the standard mode)
        }
    }
    __syncthreads();
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += PRE_THREADS) {
        const uint32_t c = (&s_hist[0][0])[k];
        if (c) atomicAdd(&p.ctrl->depth_hist[0][0] + k, c);
    }
    if (cdiff_shared)
        for (int k = tid; k < f.cdiff_cells; k += PRE_THREADS) {
            const int c = s_cdiff[k];
            if (c) atomicAdd(p.cdiff + k, c);
        }
    if (tid == 0) {
        if (s_nvis) atomicAdd(&p.ctrl->n_vis, (unsigned long long)s_nvis);
        if (blockIdx.x == 0) p.ctrl->n_sort = (unsigned long long)f.P;
    }
}

// Large scenes (P >= COMPACT_MIN_P): TWO-PHASE preprocess with order-preserving compaction of the visible Gaussians.
// A warp takes 96 consecutive Gaussians per atomic ticket.
//   Phase A (all 96, three rounds): the mean only -- view-space depth against the near plane (C-P0, the exact test
//     project() starts with).  In the camera-inside scenes about half of the Gaussians end here, having cost ~30
//     instructions instead of ~1 000; the survivors' indices are queued, in index order, in shared memory.
//   Phase B (survivors, DENSE lanes: two rounds when <= 64 survived): C-P0..C-P8, then -- visible ones only -- SH
//     colour, render record, coverage grids, depth histograms.
// The tile's count of visible Gaussians is published before the heavy part of phase B and the exclusive prefix is
// looked back for after it ("parallel prefix scan"; decoupled look-back), by which time the predecessors
// have long published.  Index order is kept throughout (queue in index order, rounds in order), which the stable
// depth sort needs for the tie-break of reading S10.
constexpr int PRE2_TILE = 96;
template <int DEG>
__global__ void __launch_bounds__(PRE_THREADS, 4)
preprocess2_kernel(const Frame f, const Pointers p, const float* __restrict__ means, const float* __restrict__ scales,
                   const float* __restrict__ rots, const float* __restrict__ opac, const float* __restrict__ sh) {
    __shared__ uint32_t s_hist[MAX_SORT_PASSES_DEPTH][256];
    __shared__ int s_cdiff[CDIFF_SMEM];
    __shared__ uint32_t s_q[PRE_THREADS / 32][PRE2_TILE];
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += PRE_THREADS) (&s_hist[0][0])[k] = 0;
    const bool cdiff_shared = f.cdiff_cells <= CDIFF_SMEM;
    if (cdiff_shared)
        for (int k = tid; k < f.cdiff_cells; k += PRE_THREADS) s_cdiff[k] = 0;
    int* const cdiff = cdiff_shared ? s_cdiff : p.cdiff;
    const int cgw = f.cgx + 1;
    __syncthreads();
    const int n_tiles = (f.P + PRE2_TILE - 1) / PRE2_TILE;
    const int gw = f.gx + 1;
    const unsigned lt = (1u << lane) - 1u;
    const int gwarp = blockIdx.x * (PRE_THREADS / 32) + w;
    int* diff = p.diff + (size_t)(gwarp & (f.diff_copies - 1)) * f.diff_cells;
    const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
    while (true) {
        int tile = 0;
        if (lane == 0) tile = (int)atomicAdd(&p.ctrl->tile_counter[TC_PRE], 1u);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        if (tile >= n_tiles) break;
        const int i0 = tile * PRE2_TILE;
        // ---- phase A: near-plane test on the mean, survivors queued in index order ---------------------------------
        uint32_t n_alive = 0;
#pragma unroll
        for (int r = 0; r < PRE2_TILE / 32; r++) {
            const int i = i0 + 32 * r + lane;
            bool alive = false;
            if (i < f.P) {
                const float px = __ldg(means + 3 * (size_t)i), py = __ldg(means + 3 * (size_t)i + 1), pz = __ldg(means + 3 * (size_t)i + 2);
                alive = affine(f.V + 8, px, py, pz) > 0.2f;     // C-P0 (reading S2), the operation project() repeats
                if (!alive) p.per_g[i] = zero4;
            }
            const unsigned ba = __ballot_sync(0xffffffffu, alive);
            if (alive) GS_BOUND(n_alive + __popc(ba & lt), PRE2_TILE);
            if (alive) s_q[w][n_alive + __popc(ba & lt)] = (uint32_t)i;
            n_alive += __popc(ba);
        }
        __syncwarp();
        // ---- phase B, part 1: projection of the survivors, dense lanes ------------------------------------------------
        // carried to part 2 per round: index, 2-D mean and conic (rect / depth / radius are re-read from per_g)
        float5 g[PRE2_TILE / 32];
        bool vis[PRE2_TILE / 32];
        int idx[PRE2_TILE / 32];
        unsigned vb[PRE2_TILE / 32];
        uint32_t cnt = 0;
#pragma unroll
        for (int h = 0; h < PRE2_TILE / 32; h++) {
            vis[h] = false; idx[h] = 0; vb[h] = 0u; g[h] = float5{};
            if (32u * h < n_alive) {   // warp-uniform
                if (32u * h + lane < n_alive) {
                    const int i = (int)s_q[w][32 * h + lane];
                    idx[h] = i;
                    const float px = __ldg(means + 3 * (size_t)i), py = __ldg(means + 3 * (size_t)i + 1), pz = __ldg(means + 3 * (size_t)i + 2);
                    const float sx = __ldg(scales + 3 * (size_t)i), sy = __ldg(scales + 3 * (size_t)i + 1), sz = __ldg(scales + 3 * (size_t)i + 2);
                    const float4 q = __ldcs(reinterpret_cast<const float4*>(rots) + i);
                    Splat t;
                    vis[h] = project(f, px, py, pz, sx, sy, sz, q.x, q.y, q.z, q.w, f.tile_cull ? __ldg(opac + i) : 1.0f, t);
                    uint4 pg = zero4;
                    if (vis[h]) {
                        pg.x = (uint32_t)t.xmin | ((uint32_t)t.ymin << 16);
                        pg.y = (uint32_t)t.xmax | ((uint32_t)t.ymax << 16);
                        pg.z = __float_as_uint(t.depth);
                        pg.w = (uint32_t)t.radius;
                        g[h] = float5{t.mux, t.muy, t.ca, t.cb, t.cc};
                        // the SH block is read in part 2: start it towards L2 now (12 K floats = 1-2 lines of 128 bytes)
                        const char* shp = reinterpret_cast<const char*>(sh + (size_t)i * (3 * (DEG + 1) * (DEG + 1)));
#pragma unroll
                        for (int o = 0; o < 12 * (DEG + 1) * (DEG + 1); o += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(shp + o));
                    }
                    p.per_g[i] = pg;
                }
                vb[h] = __ballot_sync(0xffffffffu, vis[h]);
                cnt += __popc(vb[h]);
            }
        }
        __syncwarp();   // the queue is re-used by the next ticket
        if (lane == 0) st_status(p.st_pre + tile, (tile == 0 ? ST_INC : ST_AGG) | (unsigned long long)cnt);
        // ---- phase B, part 2: everything that does not need the compact index --------------------------------------
        uint32_t depth_bits[PRE2_TILE / 32];
#pragma unroll
        for (int h = 0; h < PRE2_TILE / 32; h++) depth_bits[h] = 0u;
#pragma unroll
        for (int h = 0; h < PRE2_TILE / 32; h++) {
            if (vb[h] == 0u) continue;   // warp-uniform
            if (vis[h]) {
                const int i = idx[h];
                const uint4 pg = p.per_g[i];     // this thread's own store of part 1
                struct { int xmin, ymin, xmax, ymax; float mux, muy, ca, cb, cc; } t = {
                    (int)(pg.x & 0xffffu), (int)(pg.x >> 16), (int)(pg.y & 0xffffu), (int)(pg.y >> 16),
                    g[h].a, g[h].b, g[h].c, g[h].d, g[h].e};
                depth_bits[h] = pg.z;
                const float px = __ldg(means + 3 * (size_t)i), py = __ldg(means + 3 * (size_t)i + 1), pz = __ldg(means + 3 * (size_t)i + 2);
                GS_BOUND(t.ymax * gw + t.xmax, f.diff_cells); GS_BOUND(t.ymin * gw + t.xmin, f.diff_cells); GS_BOUND(i, f.P);
                atomicAdd(diff + t.ymin * gw + t.xmin, 1);
                atomicAdd(diff + t.ymin * gw + t.xmax, -1);
                atomicAdd(diff + t.ymax * gw + t.xmin, -1);
                atomicAdd(diff + t.ymax * gw + t.xmax, 1);
                if (f.n_ctiles) {   // the same rect on the super-tile grid (two-level binning)
                    const int cs = f.cshift, cr = (1 << cs) - 1;
                    const int cx0 = t.xmin >> cs, cy0 = t.ymin >> cs;
                    const int cx1 = (t.xmax + cr) >> cs, cy1 = (t.ymax + cr) >> cs;
                    GS_BOUND(cy1 * cgw + cx1, f.cdiff_cells);
                    atomicAdd(cdiff + cy0 * cgw + cx0, 1);
                    atomicAdd(cdiff + cy0 * cgw + cx1, -1);
                    atomicAdd(cdiff + cy1 * cgw + cx0, -1);
                    atomicAdd(cdiff + cy1 * cgw + cx1, 1);
                }
                const uint32_t db = pg.z;
                atomicAdd(&s_hist[0][db & 255u], 1u);
                atomicAdd(&s_hist[1][(db >> 8) & 255u], 1u);
                atomicAdd(&s_hist[2][(db >> 16) & 255u], 1u);
                atomicAdd(&s_hist[3][db >> 24], 1u);
                const float o = __ldcs(opac + i);
                const float3 col = sh_colour_direct<DEG>(f, sh, i, px, py, pz);
                // det of the STORED conic, exact products in double (24+24 bits): the form is indefinite iff det <= 0,
                // and the tight box of the render stage needs det without fp32 cancellation (needle-like splats)
                const double dd = (double)t.ca * (double)t.cc - (double)t.cb * (double)t.cb;
                const float l2o = log2f(o);
                const TightBox tb = tight_box_constants(t.ca, t.cb, t.cc, (float)dd, l2o);
                const uint32_t flags = (!(dd > 0.0) || tb.degenerate) ? 1u : 0u;
                float4* rec = p.rec + 4 * (size_t)i;  // 64-byte render record (include/gs.h: gs_intermediates.record)
                rec[0] = make_float4(t.mux, t.muy, t.cb, (float)dd);          // the half the tight box needs ...
                rec[1] = make_float4(tb.xstar, tb.ic, tb.ct, __uint_as_float(flags));
                rec[2] = make_float4(t.ca, t.cc, l2o, col.x);                   // ... and the half only the hoist needs
                rec[3] = make_float4(col.y, col.z, 0.0f, f.tile_cull ? tau_upper(o) : 0.0f);   // [15]: C-P8' tau, read by expand_kernel (tile_cull 2)
            }
        }
        // ---- exclusive prefix by decoupled look-back; keys of the visible Gaussians in index order ------------------
        const unsigned long long excl = tile > 0 ? lookback_warp(p.st_pre, tile) : 0ull;
        const unsigned long long run = excl + cnt;
        if (lane == 0) {
            st_status(p.st_pre + tile, ST_INC | run);
            if (tile == n_tiles - 1) { p.ctrl->n_vis = run; p.ctrl->n_sort = run; }
        }
        uint32_t before = 0;
#pragma unroll
        for (int h = 0; h < PRE2_TILE / 32; h++) {
            if (vis[h]) GS_BOUND(excl + before + __popc(vb[h] & lt), f.P);
            if (vis[h]) p.gkeyA[excl + before + __popc(vb[h] & lt)] = ((unsigned long long)depth_bits[h] << 32) | (unsigned)idx[h];
            before += __popc(vb[h]);
        }
    }
    __syncthreads();
    for (int k = tid; k < MAX_SORT_PASSES_DEPTH * 256; k += PRE_THREADS) {
        const uint32_t c = (&s_hist[0][0])[k];
        if (c) atomicAdd(&p.ctrl->depth_hist[0][0] + k, c);
    }
    if (cdiff_shared)
        for (int k = tid; k < f.cdiff_cells; k += PRE_THREADS) {
            const int c = s_cdiff[k];
            if (c) atomicAdd(p.cdiff + k, c);
        }
}

template <int DEG>
static void launch_pre(const Frame& f, const Pointers& p, const float* means, const float* scales, const float* rots,
                       const float* opac, const float* sh, int grid, cudaStream_t st) {
    g_caplog.preprocess = f.compact ? (const void*)preprocess2_kernel<DEG> : (const void*)preprocess_kernel<DEG>;
    if (f.compact) launch_pdl(preprocess2_kernel<DEG>, dim3(grid), dim3(PRE_THREADS), st, f, p, means, scales, rots, opac, sh);
    else launch_pdl(preprocess_kernel<DEG>, dim3(grid), dim3(PRE_THREADS), st, f, p, means, scales, rots, opac, sh);
}

void launch_preprocess(const Frame& f, const Pointers& p, const float* means, const float* scales, const float* rots,
                       const float* opac, const float* sh, int n_sm, cudaStream_t st) {
    const long long warps = ((long long)f.P + 31) / 32, blocks = (warps + PRE_THREADS / 32 - 1) / (PRE_THREADS / 32);
    const int grid = (int)(blocks < 1 ? 1 : (blocks < (long long)n_sm * 8 ? blocks : (long long)n_sm * 8));
    switch (f.deg) {
        case 0: launch_pre<0>(f, p, means, scales, rots, opac, sh, grid, st); break;
        case 1: launch_pre<1>(f, p, means, scales, rots, opac, sh, grid, st); break;
        case 2: launch_pre<2>(f, p, means, scales, rots, opac, sh, grid, st); break;
        default: launch_pre<3>(f, p, means, scales, rots, opac, sh, grid, st); break;
    }
}

}  // namespace gs
