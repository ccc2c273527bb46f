// gs_oracle.cpp -- CPU ORACLE of the forward 3DGS tile rasterizer.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// What it is: the plain definition of the standard forward 3DGS render that Local-GS reproduces exactly
// ("mathematically equivalent ... no approximation errors"; "strict mathematical adherence to the
// alpha-blending formulation"), computed slowly and without any of the paper's machinery:
//   C-P  per-Gaussian preprocess            -> preprocess_one()
//   C-B  duplication + sort by (tile, depth bits, index) -> bin()
//   C-R  per-pixel front-to-back blend, baseline column of Alg. 1 -> blend_pixel()
// Readings of everything the paper leaves open (near plane, dilation, rect rounding, SH convention, which T is
// tested ...) are the ones listed in DESIGN.md ("Readings"), numbered as in SURVEY.md §8(c).
//
// Precision: C-P0..C-P8 in IEEE binary32, one rounding per written operation, no FMA contraction, no
// reassociation (build with -O2 -ffp-contract=off, no -ffast-math) so that every integer it produces is the
// unique result of a pinned arithmetic.  C-P9 (colour) and C-R (blend) in double from the fp32 C-P outputs.
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): closed form T1-T3, brute force T4, hoist identity I1,
// mask soundness I2, partition of unity I3, monotone T I4, Eq. 11-12 constants I5, sort vs numpy stable sort T6,
// SH orthonormality / Unsoeld / scipy T7, permutation T8, EWA vs finite differences + scipy rotations T9.
// Parity unpinned (paper silent, fixed by declaration in DESIGN.md): near plane 0.2, guard band 1.3,
// eigenvalue floor 0.1, the 1e-7 in C-P1, SH sign convention S8 (pinned to the mathematical definition only).
//
// Shares no code with the CUDA path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it.
#include "gs_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

constexpr int TILE = 16;

struct Pre {  // per-Gaussian outputs of C-P (all zero when culled)
    std::vector<uint32_t> depth_bits, tiles_touched;
    std::vector<int32_t> radius, rect;
    std::vector<float> mu, conic, rgb, opacity;
    std::vector<float> tau;   // C-P8': the upper bound of 2 ln(255 o) the tile-cull modes use (0 in the standard mode)
};

inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

// ---------------------------------------------------------------------------------------------------------
// C-P9: signed real spherical-harmonics basis (reading S8).  Index k = l^2 + l + m; the value is
// (-1)^m * Y_lm(d) with Y_lm the orthonormal real SH (its normalisation constant included), so that
// colour = 0.5 + sum_k basis[k] * sh[k]   ("view-dependent color parameterized by SH").
// ---------------------------------------------------------------------------------------------------------
void sh_basis(int deg, const double d[3], double out[16]) {
    const double pi = 3.14159265358979323846;
    const double x = d[0], y = d[1], z = d[2];
    out[0] = 1.0 / (2.0 * std::sqrt(pi));
    if (deg < 1) return;
    const double c1 = std::sqrt(3.0) / (2.0 * std::sqrt(pi));
    out[1] = -c1 * y;  // m=-1
    out[2] = c1 * z;   // m= 0
    out[3] = -c1 * x;  // m=+1
    if (deg < 2) return;
    const double xx = x * x, yy = y * y, zz = z * z;
    const double c2a = std::sqrt(15.0) / (2.0 * std::sqrt(pi));
    const double c2b = std::sqrt(5.0) / (4.0 * std::sqrt(pi));
    const double c2c = std::sqrt(15.0) / (4.0 * std::sqrt(pi));
    out[4] = c2a * x * y;                  // m=-2
    out[5] = -c2a * y * z;                 // m=-1
    out[6] = c2b * (2.0 * zz - xx - yy);   // m= 0
    out[7] = -c2a * x * z;                 // m=+1
    out[8] = c2c * (xx - yy);              // m=+2
    if (deg < 3) return;
    const double c3a = 0.25 * std::sqrt(35.0 / (2.0 * pi));
    const double c3b = 0.5 * std::sqrt(105.0 / pi);
    const double c3c = 0.25 * std::sqrt(21.0 / (2.0 * pi));
    const double c3d = 0.25 * std::sqrt(7.0 / pi);
    const double c3e = 0.25 * std::sqrt(105.0 / pi);
    out[9] = -c3a * y * (3.0 * xx - yy);               // m=-3
    out[10] = c3b * x * y * z;                         // m=-2
    out[11] = -c3c * y * (4.0 * zz - xx - yy);         // m=-1
    out[12] = c3d * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);  // m= 0
    out[13] = -c3c * x * (4.0 * zz - xx - yy);         // m=+1
    out[14] = c3e * z * (xx - yy);                     // m=+2
    out[15] = -c3a * x * (xx - 3.0 * yy);              // m=+3
}

struct Frame {
    int P, W, H, gx, gy, deg, K;
    const float *means, *scales, *rots, *opac, *sh, *V, *PM;
    float fx, fy;
    double campos[3];
    int tile_cull = 0;   // 0: standard 3-sigma square rect (C-P8); 1: intersected with the AABB of the alpha >= 1/255 ellipse (C-P8');
                         // 2: that rect, and a (tile, Gaussian) pair is listed only if tile_hit() below holds (C-P8'')
};

// ---------------------------------------------------------------------------------------------------------
// C-P0..C-P9 for Gaussian i.  Every line is one step of the table in DESIGN.md; parentheses give the
// evaluation order, each operation rounds to binary32 once.
// ---------------------------------------------------------------------------------------------------------
void preprocess_one(const Frame& f, int i, Pre& o) {
    const float* V = f.V;
    const float* PM = f.PM;
    const float px = f.means[3 * i + 0], py = f.means[3 * i + 1], pz = f.means[3 * i + 2];
    const float Wf = (float)f.W, Hf = (float)f.H;
    // C-P0 camera space; cull if !(depth > 0.2)                                    (reading S2)
    float pc[3];
    for (int r = 0; r < 3; r++) pc[r] = ((V[4 * r + 0] * px + V[4 * r + 1] * py) + V[4 * r + 2] * pz) + V[4 * r + 3];
    const float depth = pc[2];
    if (!(depth > 0.2f)) return;
    // C-P1 clip -> pixel; pixel (x,y) is sampled at the point (x,y)                 (reading S1)
    const float h0 = ((PM[0] * px + PM[1] * py) + PM[2] * pz) + PM[3];
    const float h1 = ((PM[4] * px + PM[5] * py) + PM[6] * pz) + PM[7];
    const float h3 = ((PM[12] * px + PM[13] * py) + PM[14] * pz) + PM[15];
    const float iw = 1.0f / (h3 + 1e-7f);
    const float ndcx = h0 * iw, ndcy = h1 * iw;
    const float mux = ((ndcx + 1.0f) * Wf - 1.0f) * 0.5f;
    const float muy = ((ndcy + 1.0f) * Hf - 1.0f) * 0.5f;
    if (!(std::fabs(mux) <= 1.0e9f) || !(std::fabs(muy) <= 1.0e9f)) return;  // non-finite centre
    // C-P2 rotation from the unit quaternion (w,x,y,z)                               (reading S19)
    const float qw = f.rots[4 * i + 0], qx = f.rots[4 * i + 1], qy = f.rots[4 * i + 2], qz = f.rots[4 * i + 3];
    float R[3][3];
    R[0][0] = 1.0f - 2.0f * ((qy * qy) + (qz * qz));
    R[0][1] = 2.0f * ((qx * qy) - (qw * qz));
    R[0][2] = 2.0f * ((qx * qz) + (qw * qy));
    R[1][0] = 2.0f * ((qx * qy) + (qw * qz));
    R[1][1] = 1.0f - 2.0f * ((qx * qx) + (qz * qz));
    R[1][2] = 2.0f * ((qy * qz) - (qw * qx));
    R[2][0] = 2.0f * ((qx * qz) - (qw * qy));
    R[2][1] = 2.0f * ((qy * qz) + (qw * qx));
    R[2][2] = 1.0f - 2.0f * ((qx * qx) + (qy * qy));
    // C-P3 Sigma = (R S)(R S)^T
    const float s[3] = {f.scales[3 * i + 0], f.scales[3 * i + 1], f.scales[3 * i + 2]};
    float M[3][3], S3[3][3];
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) M[r][c] = R[r][c] * s[c];
    for (int r = 0; r < 3; r++)
        for (int c = r; c < 3; c++) {
            S3[r][c] = ((M[r][0] * M[c][0]) + (M[r][1] * M[c][1])) + (M[r][2] * M[c][2]);
            S3[c][r] = S3[r][c];
        }
    // C-P4 Jacobian of the perspective projection with the 1.3 guard band            (reading S3)
    const float limx = 1.3f * ((0.5f * Wf) / f.fx);
    const float limy = 1.3f * ((0.5f * Hf) / f.fy);
    const float tx = std::fmin(limx, std::fmax(-limx, pc[0] / pc[2])) * pc[2];
    const float ty = std::fmin(limy, std::fmax(-limy, pc[1] / pc[2])) * pc[2];
    const float tz = pc[2];
    const float j00 = f.fx / tz;
    const float j02 = -((f.fx * tx) / (tz * tz));
    const float j11 = f.fy / tz;
    const float j12 = -((f.fy * ty) / (tz * tz));
    // C-P5 2D covariance  T Sigma T^T, T = J W, plus the 0.3-pixel dilation          (reading S4)
    float Tm[2][3];
    for (int k = 0; k < 3; k++) {
        Tm[0][k] = (j00 * V[4 * 0 + k]) + (j02 * V[4 * 2 + k]);
        Tm[1][k] = (j11 * V[4 * 1 + k]) + (j12 * V[4 * 2 + k]);
    }
    float U[2][3];
    for (int r = 0; r < 2; r++)
        for (int j = 0; j < 3; j++) U[r][j] = ((Tm[r][0] * S3[0][j]) + (Tm[r][1] * S3[1][j])) + (Tm[r][2] * S3[2][j]);
    float c00 = ((U[0][0] * Tm[0][0]) + (U[0][1] * Tm[0][1])) + (U[0][2] * Tm[0][2]);
    const float c01 = ((U[0][0] * Tm[1][0]) + (U[0][1] * Tm[1][1])) + (U[0][2] * Tm[1][2]);
    float c11 = ((U[1][0] * Tm[1][0]) + (U[1][1] * Tm[1][1])) + (U[1][2] * Tm[1][2]);
    c00 = c00 + 0.3f;
    c11 = c11 + 0.3f;
    // C-P6 conic = inverse covariance (Eq. 5); cull if !(det > 0)  (reading S7)
    const float det = (c00 * c11) - (c01 * c01);
    if (!(det > 0.0f)) return;
    const float inv = 1.0f / det;
    const float ca = c11 * inv, cb = -(c01 * inv), cc = c00 * inv;
    // C-P7 3-sigma radius from the larger eigenvalue                                 (reading S5)
    const float mid = 0.5f * (c00 + c11);
    const float sq = std::sqrt(std::fmax(0.1f, (mid * mid) - det));
    const float lam = std::fmax(mid + sq, mid - sq);
    const float rf_ = std::ceil(3.0f * std::sqrt(lam));
    if (!(rf_ <= 1.0e9f)) return;  // non-finite radius
    const int radius = (int)rf_;
    // C-P8 tile rectangle, half-open, clamped to the grid                            (reading S6)
    const float rf = (float)radius;
    float rxf = rf, ryf = rf;
    float tau_out = 0.0f;
    if (f.tile_cull) {
        // C-P8' ("tighter tile culling", off by default): the square is intersected with the axis-aligned
        // bounding box of the ellipse alpha >= 1/255, i.e. a dx^2 + 2 b dx dy + c dy^2 <= tau, tau = 2 ln(255 o)
        // (PAPER.md:181), whose half-extents are sqrt(tau c / det) and sqrt(tau a / det), det = a c - b^2.  No pixel outside
        // it can pass step 4 of C-R, so the image does not change.  tau is a library-free UPPER bound: 255 o = 2^e m,
        // m in [1, 2), ln m <= (m - 1) / sqrt(m), plus 1e-5.  Extents in double from the fp32 conic the blend uses; one
        // pixel is added because the rounding of S6 can leave out a last pixel that is the first column of its tile.
        const float x255 = 255.0f * f.opac[i];
        if (!(x255 > 1.0f)) return;                       // alpha < 1/255 everywhere: never blended
        const uint32_t xb = f2u(x255);
        const int e2 = (int)(xb >> 23) - 127;
        const uint32_t mb = (xb & 0x007fffffu) | 0x3f800000u;
        float m;
        std::memcpy(&m, &mb, 4);
        const float lnm = (m - 1.0f) / std::sqrt(m);
        const float tau = (2.0f * (((float)e2 * 0.693147182f) + lnm)) + 1e-5f;
        tau_out = tau;
        const double dd = ((double)ca * (double)cc) - ((double)cb * (double)cb);
        if (dd > 0.0 && ca > 0.0f && cc > 0.0f) {
            const double hx = std::sqrt(((double)tau * (double)cc) / dd), hy = std::sqrt(((double)tau * (double)ca) / dd);
            if (hx < 1.0e9) rxf = std::fmin(rf, (float)std::ceil(hx) + 1.0f);
            if (hy < 1.0e9) ryf = std::fmin(rf, (float)std::ceil(hy) + 1.0f);
        }
    }
    const int xmin = (int)std::fmin((float)f.gx, std::fmax(0.0f, std::floor((mux - rxf) / 16.0f)));
    const int xmax = (int)std::fmin((float)f.gx, std::fmax(0.0f, std::floor(((mux + rxf) + 15.0f) / 16.0f)));
    const int ymin = (int)std::fmin((float)f.gy, std::fmax(0.0f, std::floor((muy - ryf) / 16.0f)));
    const int ymax = (int)std::fmin((float)f.gy, std::fmax(0.0f, std::floor(((muy + ryf) + 15.0f) / 16.0f)));
    const int tt = (xmax - xmin) * (ymax - ymin);
    if (tt <= 0) return;
    // C-P9 colour (double, any order)                                                (reading S8)
    double dir[3] = {(double)px - f.campos[0], (double)py - f.campos[1], (double)pz - f.campos[2]};
    const double nrm = std::sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    for (double& v : dir) v /= nrm;
    double basis[16];
    sh_basis(f.deg, dir, basis);
    for (int ch = 0; ch < 3; ch++) {
        double acc = 0.5;
        for (int k = 0; k < f.K; k++) acc += basis[k] * (double)f.sh[((size_t)i * f.K + k) * 3 + ch];
        o.rgb[3 * (size_t)i + ch] = (float)std::max(0.0, acc);
    }
    o.depth_bits[i] = f2u(depth);
    o.radius[i] = radius;
    o.rect[4 * (size_t)i + 0] = xmin;
    o.rect[4 * (size_t)i + 1] = ymin;
    o.rect[4 * (size_t)i + 2] = xmax;
    o.rect[4 * (size_t)i + 3] = ymax;
    o.tiles_touched[i] = (uint32_t)tt;
    o.mu[2 * (size_t)i + 0] = mux;
    o.mu[2 * (size_t)i + 1] = muy;
    o.conic[3 * (size_t)i + 0] = ca;
    o.conic[3 * (size_t)i + 1] = cb;
    o.conic[3 * (size_t)i + 2] = cc;
    o.opacity[i] = f.opac[i];
    o.tau[i] = tau_out;
}

bool make_frame(Frame& f, int P, const float* means, const float* scales, const float* rots, const float* opac,
                const float* sh, int deg, const float* V, const float* PM, float fx, float fy, int W, int H) {
    if (P < 0 || W <= 0 || H <= 0 || deg < 0 || deg > 3 || !V || !PM) return false;
    if (P > 0 && (!means || !scales || !rots || !opac || !sh)) return false;
    f.P = P; f.W = W; f.H = H; f.gx = (W + TILE - 1) / TILE; f.gy = (H + TILE - 1) / TILE;
    f.deg = deg; f.K = (deg + 1) * (deg + 1);
    f.means = means; f.scales = scales; f.rots = rots; f.opac = opac; f.sh = sh; f.V = V; f.PM = PM;
    f.fx = fx; f.fy = fy;
    // camera centre from the rigid view matrix: campos = -Wv^T t                     (C-P9)
    for (int c = 0; c < 3; c++)
        f.campos[c] = -((double)V[4 * 0 + c] * V[3] + (double)V[4 * 1 + c] * V[7] + (double)V[4 * 2 + c] * V[11]);
    return true;
}

void alloc_pre(Pre& o, int P) {
    o.depth_bits.assign(P, 0); o.tiles_touched.assign(P, 0); o.radius.assign(P, 0); o.rect.assign(4 * (size_t)P, 0);
    o.mu.assign(2 * (size_t)P, 0.f); o.conic.assign(3 * (size_t)P, 0.f); o.rgb.assign(3 * (size_t)P, 0.f);
    o.opacity.assign(P, 0.f);
    o.tau.assign(P, 0.f);
}

// ---------------------------------------------------------------------------------------------------------
// C-R: per-pixel blend, termination rule R1 = the paper's BASELINE column (reading S11).
// ---------------------------------------------------------------------------------------------------------
// C-P8'' (SURVEY.md 8(f) N2 "exact ellipse-tile intersection"; flag TILE_CULL_EXACT, off by default): does the ellipse
//   E = { a dx^2 + 2 b dx dy + c dy^2 <= tau_e },  (dx, dy) relative to the 2-D mean,  tau_e = tau + 0.05
// (tau: the upper bound of 2 ln(255 o) of C-P8'; PAPER.md:181 alpha >= 1/255) meet the box of pixel CENTRES of tile
// (tx, ty), [16 tx, 16 tx + 15] x [16 ty, 16 ty + 15]?  E restricted to the row band is convex, so the tile is met iff the
// x-extent of that restriction reaches the tile's columns.  The extent comes from the paper's tight box (Eq. 13-18) with
// the roles of x and y exchanged: the right-most point of E lies at dy* = -b h_x / c, h_x = sqrt(tau_e c / det); over the
// band dy in [d0, d1] the right boundary x(dy) = (-b dy + sqrt(a tau_e - det dy^2)) / a is concave, so its maximum is at
// clamp(dy*, d0, d1) (the left boundary: convex, minimum at clamp(-dy*, d0, d1)).  fp32, ONE rounding per operation in
// this order (the CUDA side restates it with __f*_rn intrinsics): the decision is an integer and must be bit-identical.
// Every "miss" is an affirmative comparison, so a NaN keeps the tile; the 0.05 added to tau (>= 4e-3 relative, >= 4e-3 px of
// extent for the sharpest conic the dilation allows) covers the fp32 rounding of the pixel positions (<= 5e-4 px at 8 K), of
// the reciprocal (1e-7 relative) and of the discriminants (1e-6 relative).
bool tile_hit(const Pre& pre, int i, int tx, int ty) {
    const float a = pre.conic[3 * (size_t)i], b = pre.conic[3 * (size_t)i + 1], c = pre.conic[3 * (size_t)i + 2];
    const float mux = pre.mu[2 * (size_t)i], muy = pre.mu[2 * (size_t)i + 1];
    const float det = (a * c) - (b * b);
    if (!(det > 0.0f) || !(a > 0.0f) || !(c > 0.0f)) return true;      // degenerate conic: keep everything
    const float te = pre.tau[i] + 0.05f;
    const float at = a * te;
    const float ia = 1.0f / a;
    const float hx = std::sqrt((te * c) / det);
    const float ys = ((-b) * hx) / c;                                  // dy of the right-most point; the left-most is at -ys
    const float d0 = (float)(16 * ty) - muy, d1 = d0 + 15.0f;          // the band, relative to the mean
    const float yu = std::fmin(std::fmax(ys, d0), d1), yl = std::fmin(std::fmax(-ys, d0), d1);
    const float du = at - ((det * yu) * yu), dl = at - ((det * yl) * yl);
    if (du < 0.0f || dl < 0.0f) return false;                          // the band misses the ellipse
    // right-most / left-most pixel abscissa of the ellipse over the band, then the tile columns they fall in: tile tx holds
    // the pixels 16 tx .. 16 tx + 15, so it is met iff ceil((xl - 15) / 16) <= tx <= floor(xr / 16) (the scaling is exact)
    const float xr = mux + ((((-b) * yu) + std::sqrt(std::fmax(du, 0.0f))) * ia);
    const float xl = mux + ((((-b) * yl) - std::sqrt(std::fmax(dl, 0.0f))) * ia);
    const float thi = std::floor(xr * 0.0625f), tlo = std::ceil((xl - 15.0f) * 0.0625f);
    if ((float)tx > thi || (float)tx < tlo) return false;
    return true;
}

struct PixelOut {
    double C[3], T;
    uint32_t n, last_k;
    double m_alpha, m_T;
    uint64_t traversed;
};

void blend_pixel(double x, double y, const uint32_t* ids, size_t n_ids, const Pre& pre, PixelOut& o) {
    const double alpha_min = (double)(1.0f / 255.0f);  // PAPER.md:181 epsilon = 1/255
    const double T_min = (double)0.0001f;
    const double alpha_max = (double)0.99f;            // PAPER.md:277 clamp to [0, 0.99]
    const double ln_alpha_min = std::log(alpha_min);
    double T = 1.0, C[3] = {0.0, 0.0, 0.0};
    uint32_t n = 0, last_k = 0;
    double m_alpha = std::numeric_limits<double>::infinity(), m_T = m_alpha;
    uint64_t traversed = 0;
    for (size_t k = 0; k < n_ids; k++) {
        const uint32_t g = ids[k];
        traversed++;
        // 1. Eq. 4-5, Table I left column
        const double dx = x - (double)pre.mu[2 * (size_t)g], dy = y - (double)pre.mu[2 * (size_t)g + 1];
        const double a = pre.conic[3 * (size_t)g], b = pre.conic[3 * (size_t)g + 1], c = pre.conic[3 * (size_t)g + 2];
        const double op = pre.opacity[g];
        const double power = -0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy;
        m_alpha = std::min(m_alpha, std::fabs(std::log(op) + power - ln_alpha_min));
        // 2. guard
        if (power > 0.0) continue;
        // 3. clamp
        const double alpha = std::min(alpha_max, op * std::exp(power));
        // 4. opacity floor
        if (alpha < alpha_min) continue;
        // 5. transmittance test BEFORE blending
        const double Tn = T * (1.0 - alpha);
        m_T = std::min(m_T, std::fabs(Tn / T_min - 1.0));
        if (Tn < T_min) break;
        // 6. blend
        for (int ch = 0; ch < 3; ch++) C[ch] += (double)pre.rgb[3 * (size_t)g + ch] * alpha * T;
        T = Tn;
        n++;
        last_k = (uint32_t)(k + 1);
    }
    o.C[0] = C[0]; o.C[1] = C[1]; o.C[2] = C[2]; o.T = T; o.n = n; o.last_k = last_k;
    o.m_alpha = m_alpha; o.m_T = m_T; o.traversed = traversed;
}

}  // namespace

struct gs_oracle_result {
    Frame f;
    Pre pre;
    bool full = true;
    uint64_t n_dup = 0, pairs_traversed = 0, pairs_blended = 0;
    std::vector<uint32_t> tile_counts, sorted_ids, n_contrib, last_k;
    std::vector<int32_t> list_tile;
    std::vector<uint64_t> list_offsets;
    std::vector<float> image, final_T, m_alpha, m_T;
    std::vector<uint8_t> fragile, rendered;
};

extern "C" {

gs_oracle_result* gs_oracle_render(int P, const float* means3D, const float* scales, const float* rotations,
                                   const float* opacities, const float* sh_coeffs, int sh_degree,
                                   const float* viewmatrix, const float* projmatrix, float fx, float fy, int W,
                                   int H, const float* bg, const int32_t* tile_subset, int n_subset, int n_threads,
                                   int flags, double fragile_delta) {
    Frame f;
    if (!make_frame(f, P, means3D, scales, rotations, opacities, sh_coeffs, sh_degree, viewmatrix, projmatrix, fx, fy, W, H))
        return nullptr;
    if (!bg) return nullptr;
    f.tile_cull = (flags & GS_ORACLE_TILE_CULL_EXACT) ? 2 : ((flags & GS_ORACLE_TILE_CULL) ? 1 : 0);
    gs_oracle_result* r = new gs_oracle_result();
    r->f = f;
    const int n_tiles = f.gx * f.gy;
    // ---- C-P -------------------------------------------------------------------------------------------
    alloc_pre(r->pre, P);
    for (int i = 0; i < P; i++) preprocess_one(f, i, r->pre);
    const Pre& pre = r->pre;
    // ---- C-B: count, prefix, fill buckets in Gaussian order, stable sort each bucket on depth bits --------
    r->tile_counts.assign(n_tiles, 0);
    r->rendered.assign(n_tiles, 0);
    r->full = (tile_subset == nullptr);
    std::vector<int32_t> slot(n_tiles, -1);
    if (r->full) {
        r->list_tile.resize(n_tiles);
        for (int t = 0; t < n_tiles; t++) { r->list_tile[t] = t; slot[t] = t; }
    } else {
        for (int k = 0; k < n_subset; k++) {
            const int t = tile_subset[k];
            if (t < 0 || t >= n_tiles || slot[t] >= 0) { delete r; return nullptr; }
            slot[t] = (int32_t)r->list_tile.size();
            r->list_tile.push_back(t);
        }
    }
    const size_t n_lists = r->list_tile.size();
    for (int i = 0; i < P; i++) {
        if (!pre.tiles_touched[i]) continue;
        const int32_t* rc = &pre.rect[4 * (size_t)i];
        for (int ty = rc[1]; ty < rc[3]; ty++)
            for (int tx = rc[0]; tx < rc[2]; tx++) {
                if (f.tile_cull == 2 && !tile_hit(pre, i, tx, ty)) continue;
                r->tile_counts[(size_t)ty * f.gx + tx]++;
            }
        r->n_dup += pre.tiles_touched[i];   // the rect area in every mode: the capacity a frame needs
    }
    r->list_offsets.assign(n_lists + 1, 0);
    if (!(flags & GS_ORACLE_NO_LISTS)) {
        for (size_t l = 0; l < n_lists; l++) r->list_offsets[l + 1] = r->list_offsets[l] + r->tile_counts[r->list_tile[l]];
        r->sorted_ids.resize(r->list_offsets[n_lists]);
        std::vector<uint64_t> cursor(r->list_offsets.begin(), r->list_offsets.end() - 1);
        for (int i = 0; i < P; i++) {  // duplication in Gaussian-index order
            if (!pre.tiles_touched[i]) continue;
            const int32_t* rc = &pre.rect[4 * (size_t)i];
            for (int ty = rc[1]; ty < rc[3]; ty++)
                for (int tx = rc[0]; tx < rc[2]; tx++) {
                    if (f.tile_cull == 2 && !tile_hit(pre, i, tx, ty)) continue;
                    const int32_t l = slot[(size_t)ty * f.gx + tx];
                    if (l >= 0) r->sorted_ids[cursor[l]++] = (uint32_t)i;
                }
        }
        // key = (tile << 32) | depth bits, stable => ties by index (S10).  The lists are independent: with n_threads > 1 they
        // are sorted by several threads (same std::stable_sort per list, identical result).
        auto sort_lists = [&](size_t first, size_t stride) {
            for (size_t l = first; l < n_lists; l += stride)
                std::stable_sort(r->sorted_ids.begin() + r->list_offsets[l], r->sorted_ids.begin() + r->list_offsets[l + 1],
                                 [&](uint32_t p, uint32_t q) { return pre.depth_bits[p] < pre.depth_bits[q]; });
        };
        if (n_threads <= 1) {
            sort_lists(0, 1);
        } else {
            std::vector<std::thread> th;
            for (int k = 0; k < n_threads; k++) th.emplace_back(sort_lists, (size_t)k, (size_t)n_threads);
            for (auto& t : th) t.join();
        }
    }
    // ---- C-R ---------------------------------------------------------------------------------------------
    const size_t npix = (size_t)W * H;
    r->image.assign(3 * npix, 0.f); r->final_T.assign(npix, 0.f); r->n_contrib.assign(npix, 0); r->last_k.assign(npix, 0);
    r->fragile.assign(npix, 0); r->m_alpha.assign(npix, 0.f); r->m_T.assign(npix, 0.f);
    if (!(flags & (GS_ORACLE_NO_RENDER | GS_ORACLE_NO_LISTS))) {
        const int nt = std::max(1, n_threads);
        std::vector<uint64_t> trav(nt, 0), blen(nt, 0);
        auto work = [&](int tid) {
            for (size_t l = tid; l < n_lists; l += nt) {
                const int t = r->list_tile[l];
                const int tx0 = (t % f.gx) * TILE, ty0 = (t / f.gx) * TILE;
                const uint32_t* ids = r->sorted_ids.data() + r->list_offsets[l];
                const size_t n_ids = r->list_offsets[l + 1] - r->list_offsets[l];
                for (int y = ty0; y < std::min(ty0 + TILE, H); y++)
                    for (int x = tx0; x < std::min(tx0 + TILE, W); x++) {
                        PixelOut po;
                        blend_pixel((double)x, (double)y, ids, n_ids, pre, po);
                        const size_t p = (size_t)y * W + x;
                        for (int ch = 0; ch < 3; ch++) r->image[ch * npix + p] = (float)(po.C[ch] + po.T * (double)bg[ch]);
                        r->final_T[p] = (float)po.T;
                        r->n_contrib[p] = po.n;
                        r->last_k[p] = po.last_k;
                        r->m_alpha[p] = (float)po.m_alpha;
                        r->m_T[p] = (float)po.m_T;
                        r->fragile[p] = (uint8_t)((po.m_alpha < fragile_delta ? 1 : 0) | (po.m_T < fragile_delta ? 2 : 0));
                        trav[tid] += po.traversed;
                        blen[tid] += po.n;
                    }
                r->rendered[t] = 1;
            }
        };
        if (nt == 1) {
            work(0);
        } else {
            std::vector<std::thread> th;
            for (int k = 0; k < nt; k++) th.emplace_back(work, k);
            for (auto& t : th) t.join();
        }
        for (int k = 0; k < nt; k++) { r->pairs_traversed += trav[k]; r->pairs_blended += blen[k]; }
    }
    return r;
}

void gs_oracle_get_view(const gs_oracle_result* r, gs_oracle_view* v) {
    std::memset(v, 0, sizeof(*v));
    v->P = r->f.P; v->W = r->f.W; v->H = r->f.H; v->grid_x = r->f.gx; v->grid_y = r->f.gy;
    v->n_tiles = r->f.gx * r->f.gy; v->n_lists = (int32_t)r->list_tile.size(); v->full = r->full ? 1 : 0;
    v->n_dup = r->n_dup; v->n_list_entries = r->sorted_ids.size();
    v->pairs_traversed = r->pairs_traversed; v->pairs_blended = r->pairs_blended;
    v->depth_bits = r->pre.depth_bits.data(); v->radius = r->pre.radius.data(); v->rect = r->pre.rect.data();
    v->tiles_touched = r->pre.tiles_touched.data(); v->mu = r->pre.mu.data(); v->conic = r->pre.conic.data();
    v->rgb = r->pre.rgb.data();
    v->tile_counts = r->tile_counts.data(); v->list_tile = r->list_tile.data(); v->list_offsets = r->list_offsets.data();
    v->sorted_ids = r->sorted_ids.data();
    v->image = r->image.data(); v->final_T = r->final_T.data(); v->n_contrib = r->n_contrib.data();
    v->last_k = r->last_k.data(); v->fragile = r->fragile.data(); v->m_alpha = r->m_alpha.data(); v->m_T = r->m_T.data();
    v->rendered = r->rendered.data();
}

void gs_oracle_free(gs_oracle_result* r) { delete r; }

int gs_oracle_render_untiled(int P, const float* means3D, const float* scales, const float* rotations,
                             const float* opacities, const float* sh_coeffs, int sh_degree, const float* viewmatrix,
                             const float* projmatrix, float fx, float fy, int W, int H, const float* bg, int use_rect,
                             float* image, float* final_T, uint32_t* n_contrib) {
    Frame f;
    if (!make_frame(f, P, means3D, scales, rotations, opacities, sh_coeffs, sh_degree, viewmatrix, projmatrix, fx, fy, W, H))
        return -1;
    Pre pre;
    alloc_pre(pre, P);
    for (int i = 0; i < P; i++) preprocess_one(f, i, pre);
    const size_t npix = (size_t)W * H;
    std::vector<uint32_t> ids;
    for (int y = 0; y < H; y++)
        for (int x = 0; x < W; x++) {
            const int tx = x / TILE, ty = y / TILE;
            ids.clear();
            for (int i = 0; i < P; i++) {  // input order
                if (!pre.tiles_touched[i]) continue;
                const int32_t* rc = &pre.rect[4 * (size_t)i];
                if (use_rect && !(tx >= rc[0] && tx < rc[2] && ty >= rc[1] && ty < rc[3])) continue;
                ids.push_back((uint32_t)i);
            }
            std::stable_sort(ids.begin(), ids.end(), [&](uint32_t p, uint32_t q) { return pre.depth_bits[p] < pre.depth_bits[q]; });
            PixelOut po;
            blend_pixel((double)x, (double)y, ids.data(), ids.size(), pre, po);
            const size_t p = (size_t)y * W + x;
            for (int ch = 0; ch < 3; ch++) image[ch * npix + p] = (float)(po.C[ch] + po.T * (double)bg[ch]);
            final_T[p] = (float)po.T;
            n_contrib[p] = po.n;
        }
    return 0;
}

// Eq. 8 with the garbled rows restored by expanding Eq. 6 (reading G2):
//   A = -a/2, B = -b, C = -c/2, D = a dx + b dy, E = b dx + c dy, F = ln o - a dx^2/2 - b dx dy - c dy^2/2
// where (dx,dy) = mu - tile origin (Eq. 2) and ln(alpha) = A x'^2 + B x'y' + C y'^2 + D x' + E y' + F (Eq. 7).
void gs_oracle_hoist(double a, double b, double c, double o, double dx, double dy, double V[6]) {
    const double ln_o = std::log(o);
    V[0] = -0.5 * a;
    V[1] = -1.0 * b;
    V[2] = -0.5 * c;
    V[3] = dx * a + dy * b;
    V[4] = dx * b + dy * c;
    V[5] = -0.5 * dx * dx * a - dx * dy * b - 0.5 * dy * dy * c + 1.0 * ln_o;
}

// Eq. 13-21, reading S13: X0 = Tx, X1 = Tx + 15 are sample points; negative discriminant in
// case A/B => the ellipse misses the column => M = 0; tau <= 0 => M = 0.
uint32_t gs_oracle_warp_mask(double a, double b, double c, double o, double mux, double muy, double Tx, double Ty,
                             double y_span[2]) {
    const double nan = std::numeric_limits<double>::quiet_NaN();
    if (y_span) { y_span[0] = nan; y_span[1] = nan; }
    const double tau = 2.0 * std::log(255.0 * o);
    if (!(tau > 0.0)) return 0;
    const double det = a * c - b * b;
    const double x0 = Tx - mux, x1 = (Tx + 15.0) - mux;  // Eq. 14
    const double dy = std::sqrt(a * tau / det);          // Eq. 16
    double ymax, ymin;
    // upper branch
    if (-b * dy < a * x0) {  // Case A, Eq. 17
        const double disc = c * tau - det * x0 * x0;
        if (disc < 0.0) return 0;
        ymax = (-b * x0 + std::sqrt(disc)) / c;
    } else if (-b * dy > a * x1) {  // Case B, Eq. 18
        const double disc = c * tau - det * x1 * x1;
        if (disc < 0.0) return 0;
        ymax = (-b * x1 + std::sqrt(disc)) / c;
    } else {  // Case C
        ymax = dy;
    }
    // lower branch: "identical conditional logic with reversed signs for the linear terms"
    if (b * dy < a * x0) {
        const double disc = c * tau - det * x0 * x0;
        if (disc < 0.0) return 0;
        ymin = (-b * x0 - std::sqrt(disc)) / c;
    } else if (b * dy > a * x1) {
        const double disc = c * tau - det * x1 * x1;
        if (disc < 0.0) return 0;
        ymin = (-b * x1 - std::sqrt(disc)) / c;
    } else {
        ymin = -dy;
    }
    const double gy_min = muy + ymin, gy_max = muy + ymax;  // Eq. 19
    if (y_span) { y_span[0] = gy_min; y_span[1] = gy_max; }
    const double y_start = std::max(Ty, std::ceil(gy_min));
    const double y_end = std::min(Ty + 15.0, std::floor(gy_max));
    if (y_start > y_end) return 0;
    const int w_start = ((int)(y_start - Ty)) >> 1;  // Eq. 20
    const int w_end = ((int)(y_end - Ty)) >> 1;
    return ((1u << (w_end - w_start + 1)) - 1u) << w_start;  // Eq. 21
}

void gs_oracle_sh_basis(int deg, const double dir[3], double out[16]) {
    for (int k = 0; k < 16; k++) out[k] = 0.0;
    sh_basis(deg, dir, out);
}

}  // extern "C"
