// render_b200.cu -- the B200 render kernel (variant 4): Local-GS (Sec. III) re-laid-out for sm_100a.
//
//   * 128 threads per 16x16 tile, TWO horizontally adjacent pixels per thread, the per-pixel operations issued as
//     packed f32x2 instructions (FFMA2 / FMUL2 with scalar-broadcast coefficient operands).  The two pixels share their
//     row, so the exponent log2(alpha) = V_hoisted . B_local (Eq. 9-10) is evaluated as (A x' + H) x' + G with the row
//     part H = B y' + D, G = C y'^2 + E y' + F computed once for both: 3 scalar FFMA + 2 FFMA2 per entry; the blend
//     w = alpha T; C += f w; T -= w (Alg. 1 right column) is FMUL2 + 4 FFMA2.
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
//     T - w < 1e-4, voted across the warp; the rare taken branch un-blends the stopping pixel and POISONS its x'
//     (1e18), which drives every later log2(alpha) to -huge, i.e. alpha = 0 exactly.
//   * staging is software-pipelined: the ids of batch k+2 and the 64-byte records of batch k+1 are in flight while
//     batch k is blended; shared memory is double-buffered, so a batch costs ONE block barrier.
#include "render_blend.cuh"

namespace gs {

// Walk of one warp's list, TWO consecutive entries per iteration (the list is padded to an even length with the null
// record) for the two pixels of this thread.  The HOT loop updates everything IN PLACE and unconditionally -- w = alpha T;
// T <- T - K w; C <- C + f w (Alg. 1 right column), twice -- and ends with ONE warp vote: T only decreases, so "some T
// ended below 1e-4" catches a crossing in either entry.  The loop is a single basic block that is left when the vote
// fires (or the list ends): the repair below is OUTSIDE it, so that the accumulators stay in their registers across the
// back edge (with the repair inlined in the loop body ptxas carried them through 10 register moves per iteration).
// The rare REPAIR (rule R1: the crossing Gaussian and everything after it is not blended): the f w of the stopping
// pixels are subtracted again and T is restored, packed and in place (wm = w on the stopping pixels, 0 elsewhere: exact
// no-ops for the others; the restored values are within two roundings of the old ones -- toleranced outputs), then the
// pixels are poisoned.  When the whole warp is finished (Eq. 22) `lend` is zeroed: the warp-uniform end of the walk.
template <bool COUNT, bool GUARD>
__device__ __forceinline__ void blend_list(PixelPair& s, uint32_t& lp, uint32_t& lend) {
    while (lp < lend) {
        float4 p1, q1;
        float2 p2, q2;
        float e0, e1, g0, g1;
        u64 w1, w2;
        bool hit;
        do {
            const uint2 aa = lds64u(lp);   // no prefetch across the back edge: ptxas carried a prefetched pair through two moves
            const uint32_t a1 = aa.x, a2 = aa.y;
            lp += 8;
            const float4 p0 = lds128(a1);                     // (A, B, C, F)
            p1 = lds128(a1 + 16);                             // (D, E, r, g)
            p2 = lds64(a1 + 32);                              // (b, guard)
            const float4 q0 = lds128(a2);
            q1 = lds128(a2 + 16);
            q2 = lds64(a2 + 32);
            const u64 al1 = alpha_pair<GUARD>(s, p0, p1, p2.y, e0, e1);
            const u64 al2 = alpha_pair<GUARD>(s, q0, q1, q2.y, g0, g1);
            w1 = fmul2(al1, s.T);
            ffma2_acc(s.T, bc(-K_SCALE), w1);
            w2 = fmul2(al2, s.T);
            ffma2_acc(s.T, bc(-K_SCALE), w2);
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
            hit = __any_sync(0xffffffffu, fminf(t0, t1) < TMIN_S);   // rare; a stopped pixel keeps T >= 1e-4 K: it never fires again
        } while (!hit && lp < lend);
        if (hit) {
            float t0, t1, w10, w11, w20, w21;
            unpk(s.T, t0, t1);
            unpk(w1, w10, w11); unpk(w2, w20, w21);
            const bool sb0 = t0 < TMIN_S, sb1 = t1 < TMIN_S;      // stopped at the first or the second entry
            const u64 wm2 = pk(sb0 ? w20 : 0.0f, sb1 ? w21 : 0.0f);
            ffma2_acc(s.T, bc(K_SCALE), wm2);                     // on the stopped pixels: the T before the second entry
            float u0, u1;
            unpk(s.T, u0, u1);
            const bool sa0 = sb0 && u0 < TMIN_S, sa1 = sb1 && u1 < TMIN_S;   // stopped at the first entry already
            const u64 wm1 = pk(sa0 ? w10 : 0.0f, sa1 ? w11 : 0.0f);
            ffma2_acc(s.T, bc(K_SCALE), wm1);
            ffma2_acc(s.Cr, bc(-q1.z), wm2);
            ffma2_acc(s.Cg, bc(-q1.w), wm2);
            ffma2_acc(s.Cb, bc(-q2.x), wm2);
            ffma2_acc(s.Cr, bc(-p1.z), wm1);
            ffma2_acc(s.Cg, bc(-p1.w), wm1);
            ffma2_acc(s.Cb, bc(-p2.x), wm1);
            float r0, r1;
            unpk(s.T, r0, r1);   // the T of rule R1 passed the test when it was formed: >= 1e-4 K up to the rounding of the repair
            s.T = pk(sb0 ? fmaxf(r0, TMIN_S) : r0, sb1 ? fmaxf(r1, TMIN_S) : r1);
            ffma2_acc(s.bx, pk(sb0 ? 1.0f : 0.0f, sb1 ? 1.0f : 0.0f), bc(POISON));
            if (COUNT) {
                s.n0 -= (sa0 ? 1u + ((g0 > 0.0f) ? 1u : 0u) : (sb0 ? 1u : 0u));
                s.n1 -= (sa1 ? 1u + ((g1 > 0.0f) ? 1u : 0u) : (sb1 ? 1u : 0u));
            }
            float x0, x1;
            unpk(s.bx, x0, x1);
            if (__all_sync(0xffffffffu, x0 >= 0.5f * POISON && x1 >= 0.5f * POISON)) lend = 0;
        }
    }
}

// 8 blocks per SM at 64 registers: since the separable exponent (three scalars and one packed x' instead of five packed
// basis elements) the loop fits without a register move; at 9 blocks (56 registers) ptxas brings six moves back.
template <bool COUNT, bool STATS>
__global__ void __launch_bounds__(QB, 8)
render_b200_kernel(const Frame f, Ctrl* __restrict__ ctrl, const uint4* __restrict__ desc, const uint32_t* __restrict__ ids,
                   const float4* __restrict__ rec, float* __restrict__ out_rgb, float* __restrict__ out_T,
                   uint32_t* __restrict__ out_n) {
    __shared__ __align__(16) unsigned char s_raw[QB * 64];            // 64-byte records of the NEXT batch as gathered (cp.async)
    __shared__ __align__(16) unsigned char s_rec[2][(QB + 1) * REC];  // staged, hoisted records (double-buffered) + a null record
    __shared__ __align__(16) uint32_t s_ball[2][4][4];          // [buffer][staging warp][quadrant] mask ballots
    __shared__ __align__(16) uint32_t s_indef[2][4];            // [buffer][staging warp] the batch holds an indefinite conic
    __shared__ __align__(16) uint32_t s_list[4][QB + 4];        // per-warp compacted lists of record addresses (padded to even length)
    griddep_sync();
    const int tid = threadIdx.x, lane = tid & 31;
    // warp index through a warp reduction: ptxas then KNOWS it is warp-uniform (it lives in a uniform register), so
    // every trip count derived from it is uniform and the votes of the blend loop need no divergence guard
    const int w = __reduce_max_sync(0xffffffffu, tid >> 5);
    // blocks are dispatched in index order: descriptor b follows the render schedule of tile_grid_kernel (classes of
    // list length, longest first, raster order inside), so the long tiles start first and the launch has no tail
    const uint4 dsc = desc[blockIdx.x];
    GS_BOUND(dsc.x, f.n_tiles); GS_BOUND(dsc.z, f.max_dup + 1); GS_BOUND(dsc.y, (unsigned long long)dsc.z + 1);
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
        s.bx = pk(in0 ? x0 : POISON, in1 ? x1 : POISON);
        s.y = y;
        s.y2 = y * y;
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
    uint32_t end_ = dsc.z;
    if (f.tile_len != nullptr && dsc.z > dsc.y) end_ = dsc.y + __ldg(f.tile_len + tile);   // gs_set_tile_cull(2): exact list length (expand_kernel)
    const uint32_t start = __reduce_max_sync(0xffffffffu, dsc.y), end = __reduce_max_sync(0xffffffffu, end_);   // warp-uniform to ptxas
    const unsigned lt = (1u << lane) - 1u;
    uint32_t st_walk = 0, st_staged = 0;  // STATS only
    // ---- gather of a batch: FOUR LANES PER RECORD.  A lane that fetches its own 64-byte record with four 16-byte loads
    // makes every one of them a 32-line request (the L1 tag stage serves one line per cycle: 128 cycles per warp and
    // batch, and the unit was 72 % busy, profiles/r02_render_base.md); here lanes 4j..4j+3 copy the four 16-byte chunks
    // of record 8k + j in copy k = 0..3 (8 lines per request), straight into shared memory with cp.async, so that no
    // register holds a prefetched record across the blend loop.  Chunk c of record j is stored at chunk position
    // c ^ ((j >> 1) & 3): the 16-byte reads of the staging thread (stride 64 bytes across lanes) are then conflict-free.
    // Warp w gathers, and later stages, entries 32 w .. 32 w + 31 of the batch: the raw records are warp-private.
    const uint32_t raw_w = (uint32_t)__cvta_generic_to_shared(&s_raw[w * 32 * 64]);
    // this thread's own raw record: chunk c sits at raw_me ^ (c << 4) (the swizzle above, (lane >> 1) & 3 for record `lane`)
    const uint32_t raw_me = raw_w + lane * 64 + (((uint32_t)(lane >> 1) & 3u) << 4);
    // Unconditional: a slot past the end of the list copies the record of whatever valid id its lane still holds (0 or an
    // id of the previous batch -- a cache hit, masked out at staging); four predicates and their compares per batch saved.
    auto gather = [&](const uint32_t id_mine) {
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int j = 8 * k + (lane >> 2), c = lane & 3;
            const uint32_t id = __shfl_sync(0xffffffffu, id_mine, j);
            cp_async16(raw_w + j * 64 + ((c ^ ((j >> 1) & 3)) << 4), rec + 4 * (size_t)id + c);
        }
        cp_async_commit();
    };
    // ---- software pipeline prologue: records of batch 0 (in flight), ids of batch 1 -------------------------------------
    uint32_t id_next = 0;
    {
        const uint32_t id0 = (start + tid < end) ? ids[start + tid] : 0u;
        if (start < end) gather(id0);
    }
    if (start + QB + tid < end) id_next = ids[start + QB + tid];
    int buf = 0;
    for (uint32_t base = start; base < end; base += QB, buf ^= 1) {
        // ---- staging of batch `base`: tight box -> four quadrant hits -> ballots, hoist -> shared memory -------------
        if (STATS && tid == 0) st_staged += min((uint32_t)QB, end - base);
        cp_async_wait_all();
        __syncwarp();               // the four chunks of this thread's record were copied by four lanes of this warp
        // straight-line for every lane: a lane past the end of the list works on whatever its raw slot holds (stale
        // bytes, never a trap) and is masked out of the predicates -- no divergent region, the four hits go to the votes
        const bool valid = base + tid < end;
        const float4 r0 = lds128(raw_me), r1 = lds128(raw_me ^ 0x10u), r2 = lds128(raw_me ^ 0x20u), r3 = lds128(raw_me ^ 0x30u);
        bool q[4];
        quadrant_hits(r0.x - (float)Tx, r0.y - (float)Ty, r0.z, r0.w, r1.x, r1.y, r1.z, q);
        const bool indefinite = valid && (__float_as_uint(r1.w) & 1u);   // degenerate conic: keep everything
#pragma unroll
        for (int k = 0; k < 4; k++) q[k] = (valid && q[k]) || indefinite;
        const unsigned b0 = __ballot_sync(0xffffffffu, q[0]), b1 = __ballot_sync(0xffffffffu, q[1]),
                       b2 = __ballot_sync(0xffffffffu, q[2]), b3 = __ballot_sync(0xffffffffu, q[3]);
        const unsigned bi = __ballot_sync(0xffffffffu, indefinite);
        const bool any = q[0] | q[1] | q[2] | q[3];
        // every lane stores the same words (one wavefront, no branch on the lane index)
        *reinterpret_cast<uint4*>(&s_ball[buf][w][0]) = make_uint4(b0, b1, b2, b3);
        s_indef[buf][w] = bi;
        // the hoist itself is straight-line too (some lane of the warp needs it in practically every batch; a branch
        // around it only adds a divergent region), only the stores are kept to the entries that reach some warp
        const Hoisted h = hoist(r0.x, r0.y, r2.x, r0.z, r2.y, r2.z, ox, oy, L_BIAS);
        if (any) {
            float4* d = reinterpret_cast<float4*>(&s_rec[buf][tid * REC]);
            d[0] = make_float4(h.A, h.B, h.C, h.F);
            d[1] = make_float4(h.D, h.E, r2.w, r3.x);
            d[2] = make_float4(r3.y, indefinite ? r2.z + L_BIAS : 3.0e38f, 0.0f, 0.0f);
        }
        // ---- gather of the next batch into the raw slots just consumed (the hoist above read them), ids of the one after ---
        __syncwarp();
        if (base + QB < end) gather(id_next);
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
        GS_BOUND(cnt, QB + 1);
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
    cp_async_wait_all();   // nothing of this block may still be landing in shared memory when it retires
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
    write_pixels<COUNT>(f, s, px, py, in0, in1, out_rgb, out_T, out_n);   // epilogue: out = C + T bg (reading S16)
}

void launch_render_b200(const Frame& f, const Pointers& p, float* out_rgb, float* out_T, uint32_t* out_n, int n_sm,
                        bool stats, cudaStream_t st) {
    (void)n_sm;
    const dim3 grid(f.n_tiles), block(QB);
    g_caplog.render = (stats && out_n) ? (const void*)render_b200_kernel<true, true>
                                       : (out_n ? (const void*)render_b200_kernel<true, false> : (const void*)render_b200_kernel<false, false>);
    if (stats && out_n)
        launch_pdl(render_b200_kernel<true, true>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else if (out_n)
        launch_pdl(render_b200_kernel<true, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, out_n);
    else
        launch_pdl(render_b200_kernel<false, false>, grid, block, st, f, p.ctrl, p.desc, p.ids, p.rec, out_rgb, out_T, (uint32_t*)nullptr);
}

}  // namespace gs
