// raster.cu -- steps a7 macro-tile rasterizer and a8 post-blend merge
// (section 3.4 with Alg. 1 MacroTileRasterize and Alg. 2 RasterizeTile,
//  PAPER.md:278-301 section 4.5, Eq. (1)).
//
// A work unit is one (macro-tile, batch of <= B_r gaussians).  A persistent CTA claims
// units from a device counter.  Phase 1 (Alg. 1 lines 1-8): the unit's records are gathered by sorted
// id into shared memory, every thread derives the 32-bit render-tile overlap mask of its gaussian, and a
// warp ballot transposes 32 gaussians x 32 tiles so that one word per (tile, mini-batch) says which
// gaussians touch the tile.  Phase 2 (Alg. 1 lines 9-17, Alg. 2): warps claim render tiles from a shared
// counter; a warp owns the tile (TILE^2 / 32 pixels per lane, all in one pixel column so that the dx terms are
// shared, in pairs of rows), walks the tile's mask words, reads each listed gaussian with broadcast shared
// loads and composites front to back; after every drain a unanimous vote on T < eps ends the tile early
// (Alg. 2 line 8).  Partial (r,g,b,T) per pixel goes to the dense (unit, tile) buffer, the unit's 32-bit
// active mask out of band.  The merge kernel gives one warp per render tile and folds the
// macro-tile's units in depth order with Eq. (1), stopping once every pixel is saturated.
//
// Two data paths, one kernel template:
//   fp32 (default, the parity path): the skip decision q <= tau uses the pinned sequence N-Q (DESIGN.md
//     section 3) in absolute pixel coordinates, bit-identical to the oracle's; alpha, colour and T are
//     "smooth" (ex2.approx, fp32 accumulation); 48-byte staged records, packed f32x2 arithmetic.
//   fp16 (HIGS_FLAG_FP16; section 3.5): Cholesky factors of the inverse
//     covariance prescaled by sqrt(log2 e / 2) * tile_size, positions in tile units relative to the macro-tile
//     centre, q = (l0 dx + l1 dy)^2 + (l2 dy)^2 as a sum of squares, alpha = o * exp2(-q) with
//     ex2.approx.f16x2, half2 accumulators for two pixel rows, 20-byte staged records, fp16 RGBT partials
//     (16 KB per unit at 8x8 tiles).  Accepted by PSNR against the fp32 oracle, not bit-pinned.
// TILE = 8 (the paper's default) or 16 (the variant of Table 2).
#include <stdio.h>
#include <cuda_fp16.h>
#include "higs_internal.cuh"

namespace {

constexpr int RAS_THREADS = 256;
constexpr int RAS_WARPS = RAS_THREADS / 32;
constexpr int RAS_SUB = HIGS_BATCH_CAP;           // gaussians per unit
constexpr int RAS_MB = RAS_SUB / 32;              // mini-batches of 32 gaussians per unit
constexpr int MASK_PITCH = RAS_MB + 1;
constexpr float LOGT_SCALE = 1024.0f;             // fixed point of the log2 transmittance bounds
constexpr int LOGT_EPS = -13608;                  // floor(log2(1e-4) * 1024): a sum below it proves T < eps
constexpr int RING = 512;                         // per-warp scheduling buffer of staged-record addresses, drained 8 at a time
constexpr int NULL_IDX = RAS_SUB;                 // index of the "null" gaussian that pads the last drain

// fp32 staged record: the first 48 B of the global record, as gathered:
//   f4[0] = mux, muy, A, B2      f4[1] = C, tau, log2 o, r      f4[2] = g, b, cov a, cov b
// Packed f32x2 instructions (FFMA2 / FMUL2 / FADD2) take a plain 32-bit register as a broadcast operand, so the values
// that multiply both pixels of a pair need no duplicated copy in shared memory.
// fp16 staged record (20 B in a 32-byte slot): recA (16 B) = half2 (x, y) | half2 (l0', l1') | half2 (l2', o) | half2 (r, g), recB (4 B) = half2 (b, -);
// x, y in tile units relative to the macro-tile centre.  HFMA2 / HMUL2 broadcast either half of a register for free.
constexpr int REC_F4 = 3;
template <bool HALF> struct RasLayout;
template <> struct RasLayout<false> {
    static constexpr size_t rec_bytes = sizeof(float4) * (RAS_SUB + 1) * REC_F4;
    static constexpr uint32_t stride = REC_F4 * 16u;
    static constexpr uint32_t b_off = 0;
};
template <> struct RasLayout<true> {
    static constexpr size_t rec_bytes = 32u * (RAS_SUB + 1);      // 20 B used of a 32-byte slot: recB sits at +16, an immediate offset of the LDS
    static constexpr uint32_t stride = 32u;
    static constexpr uint32_t b_off = 16u;
};
struct RasCtl {
    uint32_t masks[HIGS_MT_TILES * MASK_PITCH];   // [tile][mini-batch]: bit j = gaussian k*32+j touches the tile
    uint32_t ring[RAS_WARPS][RING + 8];          // shared-window byte addresses of the records: an entry is an LDS operand as it stands
    uint32_t unit, next_tile, active, cut;
};
template <bool HALF> constexpr size_t ras_smem_bytes() { return RasLayout<HALF>::rec_bytes + sizeof(RasCtl); }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(s), "l"(gmem));
}
__device__ __forceinline__ float4 lds128(uint32_t saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint4 lds128u(uint32_t saddr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint32_t lds32u(uint32_t saddr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint32_t h22u(__half2 v) { return *reinterpret_cast<uint32_t*>(&v); }
__device__ __forceinline__ __half2 u2h2(uint32_t v) { return *reinterpret_cast<__half2*>(&v); }
__device__ __forceinline__ __half2 ex2_h2(__half2 x)
{
    uint32_t yi;
    asm("ex2.approx.f16x2 %0, %1;" : "=r"(yi) : "r"(h22u(x)));
    return u2h2(yi);
}

// Conservative render-tile overlap mask of one gaussian inside a macro-tile (reading Q9: internal, never
// compared with the oracle): N-SCAN on the covariance (a, b, c), det = a c - b^2 given by the caller from an identity
// that does not cancel, threshold tau_m, over a grid of MTX x (32 / MTX) cells of size `cell` whose origin is (X0, Y0); the image
// ends at (fW, fH) in the same units.  Approximate rcp / sqrt: every extent is good to ~1e-6 relative; extents are widened
// by `slack` on top (pixel centres sit half a pixel inside their tile) and a gaussian whose extent exceeds `huge` takes
// every tile.
template <int MTX>
__device__ __forceinline__ uint32_t tile_mask_cov(float mux, float muy, float a, float b, float c, float det, float tau_m,
                                                  float X0, float Y0, float cell, float rcell, float fW, float fH, float slack, float huge)
{
    const float hx = sqrt_approx(tau_m * a) + slack, hy = sqrt_approx(tau_m * c) + slack;
    if (!(det > 0.0f) || !(c > 0.0f) || !(hx < huge) || !(hy < huge)) return 0xffffffffu;
    const float rc = rcp_approx(c);
    const float boc = b * rc, sdet = det * rc;
    const float yR = b * sqrt_approx(tau_m * rcp_approx(a));          // dy of the rightmost point
    const float ytop = muy - hy, ybot = muy + hy;
    uint32_t mask = 0;
#pragma unroll
    for (int tr = 0; tr < 32 / MTX; ++tr) {
        const float y0 = Y0 + cell * tr;
        const float y1 = fminf(y0 + cell, fH);
        const float ylo = fmaxf(y0, ytop) - muy, yhi = fminf(y1, ybot) - muy;
        if (!(yhi >= ylo)) continue;
        const float rlo = sqrt_approx(fmaxf(0.0f, sdet * fmaf(-ylo * ylo, rc, tau_m)));
        const float rhi = sqrt_approx(fmaxf(0.0f, sdet * fmaf(-yhi * yhi, rc, tau_m)));
        float xmax = (ylo <= yR && yR <= yhi) ? hx : fmaxf(fmaf(boc, ylo, rlo), fmaf(boc, yhi, rhi)) + slack;
        float xmin = (ylo <= -yR && -yR <= yhi) ? -hx : fminf(fmaf(boc, ylo, -rlo), fmaf(boc, yhi, -rhi)) - slack;
        xmax = fminf(xmax + mux, fW) - X0; xmin = fmaxf(xmin + mux, X0) - X0;
        if (!(xmax >= 0.0f) || !(xmin < (float)MTX * cell) || !(xmax >= xmin)) continue;
        const int c0 = max(0, (int)floorf(xmin * rcell)), c1 = min(MTX - 1, (int)floorf(xmax * rcell));
        if (c0 > c1) continue;
        mask |= ((2u << c1) - (1u << c0)) << (tr * MTX);
    }
    return mask;
}

// ---- cross-batch cut (not in the paper, which lets the batches behind an opaque one run) -------------
// Every (unit, tile) publishes a TERM: log2 of the largest transmittance it left in the tile, fixed point, rounded
// towards zero (so a sum of terms never understates the product of the transmittances).  cut_term[u][t] holds it as
// term - 1 (< 0); 0 = not published (the buffer is zeroed every frame by k_fill).  Unit (m, j) may skip tile t when
// the terms of batches 0 .. j-1 of macro-tile m sum below log2(eps): everything it could add sits behind T < eps.
// The sum is taken IN BATCH ORDER and only over j' < j by construction: cut_word[m][t] = (k << 32 | sum of the terms
// of batches 0 .. k-1) is a cache of a prefix; a reader starts from it, walks terms k, k+1, ... < j until one is
// not published yet, and writes the longer prefix back with atomicMax (equal k means equal sum, so the largest word is
// the longest prefix).  No ordering between units is assumed: a term that is not visible yet only loses some cut.
__device__ __forceinline__ int cut_prefix(unsigned long long* __restrict__ word, const int* __restrict__ term_mt /* cut_term + u0*32 + t */,
                                          uint32_t j)
{
    const unsigned long long w0 = __ldcg(word);
    uint32_t k = (uint32_t)(w0 >> 32);
    int sum = (int)(uint32_t)w0;
    const uint32_t k0 = k;
    while (k < j && sum >= LOGT_EPS) {
        const int tk = __ldcg(term_mt + (size_t)k * HIGS_MT_TILES);
        if (tk == 0) break;
        sum += tk + 1; ++k;
    }
    if (k != k0) atomicMax(word, ((unsigned long long)k << 32) | (unsigned long long)(uint32_t)sum);
    return sum;
}

// MTX x MTY render tiles per macro-tile: 8 x 4; 4 x 8 and 16 x 2 for the shape sweep (higs_set_macro_tile).  Tile t of a
// macro-tile sits in column t % MTX, row t / MTX.
template <int TILE, int MTX = 8> struct TileGeo {
    static constexpr int MTY = 32 / MTX, MT_SH = MTX == 4 ? 2 : (MTX == 8 ? 3 : 4);
    static constexpr int MT_W = MTX * TILE, MT_H = MTY * TILE;
    static constexpr int PPL = TILE * TILE / 32;   // pixels per lane
    static constexpr int NP = PPL / 2;             // pairs of pixels per lane
    static constexpr int RS = 32 / TILE;           // rows between consecutive pixels of a lane: lane -> column lane % TILE, rows lane / TILE + RS * i
};

template <bool COUNT, int TILE, bool HALF, int MTX = 8>
__global__ void __launch_bounds__(RAS_THREADS, HALF ? 3 : (TILE == 8 ? 3 : 2))
k_raster(const unsigned long long* __restrict__ pairs, const float4* __restrict__ rec, const uint4* __restrict__ rec16,
         const uint32_t* __restrict__ mt_offset, const uint32_t* __restrict__ mt_count,
         const uint32_t* __restrict__ batch_offset, const uint32_t* __restrict__ unit_mt,
         const uint32_t* __restrict__ unit_order,
         const FrameParams P, FrameHeader* __restrict__ hdr,
         float4* __restrict__ partial, uint32_t* __restrict__ unit_active,
         unsigned long long* __restrict__ cut_word, int* __restrict__ cut_term, uint32_t* __restrict__ tile_load)
{
    typedef TileGeo<TILE, MTX> G;
    static_assert(MTX == 8 || (TILE == 8 && !HALF), "other macro-tile shapes: fp32 path, 8 x 8 tiles (the fp16 path's coordinate range is the 8 x 4 macro-tile's, PAPER.md:280)");
    constexpr int NP = G::NP;
    extern __shared__ __align__(16) unsigned char s_raw[];
    RasCtl& S = *reinterpret_cast<RasCtl*>(s_raw + RasLayout<HALF>::rec_bytes);
    float4* s_rec = reinterpret_cast<float4*>(s_raw);                 // fp32 records
    uint4* s_rec16 = reinterpret_cast<uint4*>(s_raw);                 // fp16 records: [i][2], second half holds recB in its first word
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    pdl_trigger();                                                    // k_merge_image may be scheduled as this grid drains
    const uint32_t n_units = hdr->n_units;
    const bool use_cut = !(P.flags & HIGS_FLAG_NO_XBATCH_CUT);
    const float fW = (float)P.W, fH = (float)P.H;
    unsigned long long n_eval_g = 0, n_tp = 0;
    if (threadIdx.x == 0) {                                           // the null gaussian: never contributes
        if constexpr (HALF) { s_rec16[2 * NULL_IDX] = make_uint4(0u, 0u, 0u, 0u); s_rec16[2 * NULL_IDX + 1] = make_uint4(0u, 0u, 0u, 0u); }      // opacity 0
        else {
            s_rec[NULL_IDX * REC_F4] = make_float4(0.f, 0.f, 0.f, 0.f); s_rec[NULL_IDX * REC_F4 + 1] = make_float4(0.f, -1.0f, 0.f, 0.f);   // tau < 0
            s_rec[NULL_IDX * REC_F4 + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    uint32_t* ring = S.ring[w];
    const uint32_t rec_s = (uint32_t)__cvta_generic_to_shared(s_raw);

    // Warp 0 claims units until one has something left to show.  Tiles wholly outside the image are never active
    // (Alg. 1 line 11, InBounds); tiles whose bound from the batches in front is below eps are cut (lane = tile).
    // A unit with every tile cut costs one atomic and a few loads: it is never gathered.
    auto claim_unit = [&]() {
        uint32_t u_sel = 0xffffffffu, cut_sel = 0;
        for (;;) {
            uint32_t c = 0;
            if (lane == 0) c = atomicAdd(&hdr->raster_cursor, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= n_units) break;
            const uint32_t uc = unit_order[c];
            const uint32_t mc = unit_mt[uc];
            const uint32_t u0c = batch_offset[mc];
            const uint32_t jc = uc - u0c;
            const int mtx = (int)(mc % (uint32_t)P.n_mx), mty = (int)(mc / (uint32_t)P.n_mx);
            const int tiles_x = min(MTX, (P.W - mtx * G::MT_W + TILE - 1) / TILE);
            const int tiles_y = min(G::MTY, (P.H - mty * G::MT_H + TILE - 1) / TILE);
            bool saturated = false;
            if (use_cut && jc > 0)
                saturated = cut_prefix(cut_word + (size_t)mc * HIGS_MT_TILES + lane, cut_term + (size_t)u0c * HIGS_MT_TILES + lane, jc) < LOGT_EPS;
            const bool inb = (lane & (MTX - 1)) < tiles_x && (lane >> G::MT_SH) < tiles_y;
            const uint32_t cut = __ballot_sync(0xffffffffu, saturated || !inb);
            if (cut == 0xffffffffu) {                                 // nothing left to see behind the earlier batches
                if (lane == 0) unit_active[uc] = 0;
                continue;
            }
            u_sel = uc; cut_sel = cut;
            break;
        }
        if (lane == 0) { S.unit = u_sel; S.cut = cut_sel; }
    };
    uint32_t u_prev = 0xffffffffu;

    // Per unit four block barriers: top, unit claimed, records staged, masks written; every warp ranks the tiles for itself
    // instead of waiting for one warp to do it.  (Claiming the next unit early, during the compositing of the current one,
    // was measured: the cut then sees older bounds and the frame executes 19 % more evaluations - 0.407 against 0.349 ms.)
    for (;;) {
        __syncthreads();                                              // everyone is done with the previous unit's shared state
        if (w == 0) {
            if (lane == 0) {
                if (u_prev != 0xffffffffu) unit_active[u_prev] = S.active;
                S.active = 0; S.next_tile = 0;
            }
            claim_unit();
        }
        __syncthreads();
        const uint32_t u = S.unit;
        const uint32_t cut = S.cut;
        if (u == 0xffffffffu) break;
        u_prev = u;
        const uint32_t m = unit_mt[u];
        const uint32_t u0 = batch_offset[m];
        const uint32_t j = u - u0;
        const uint32_t seg_n = mt_count[m];
        const uint32_t start = mt_offset[m] + j * (uint32_t)P.batch_cap;
        const int len = (int)min((uint32_t)P.batch_cap, seg_n - j * (uint32_t)P.batch_cap);
        const int mtx = (int)(m % (uint32_t)P.n_mx), mty = (int)(m / (uint32_t)P.n_mx);
        const float X0 = (float)(mtx * G::MT_W), Y0 = (float)(mty * G::MT_H);
        HIGS_ASSERT(u < P.max_units && m < (uint32_t)P.n_m && len > 0 && len <= RAS_SUB && start + (uint32_t)len <= hdr->n_pairs);

        if constexpr (!HALF) {
            // ---- Phase 1a: gather of this unit's records (Alg. 1 line 4), first 48 B of each, by sorted id ----
            for (int i = threadIdx.x; i < len; i += RAS_THREADS) {
                const uint32_t id = (uint32_t)pairs[start + i];
                const float4* src = rec + 4 * (size_t)id;
                cp_async16(&s_rec[REC_F4 * i], src);
                cp_async16(&s_rec[REC_F4 * i + 1], src + 1);
                cp_async16(&s_rec[REC_F4 * i + 2], src + 2);
            }
            cp_async_wait_all();                                      // each thread waits for the records it asked for
            __syncthreads();
        }
        // ---- Phase 1b: per-gaussian tile masks (Alg. 1 lines 5-6), transposed by ballot ----
        // fp16 path: the 32-byte global record is loaded to registers here, converted to the macro-tile-local frame
        // ("convert to tile space") and stored as the 20-byte staged record.
        constexpr int KPW = RAS_MB / RAS_WARPS;                       // mini-batches per warp
        uint4 g0[HALF ? KPW : 1], g1[HALF ? KPW : 1];
        if constexpr (HALF) {
#pragma unroll
            for (int kk = 0; kk < KPW; ++kk) {
                const int i = (w + kk * RAS_WARPS) * 32 + lane;
                g0[kk] = make_uint4(0u, 0u, 0u, 0u); g1[kk] = g0[kk];
                if (i < len) {
                    const uint32_t id = (uint32_t)pairs[start + i];
                    g0[kk] = __ldg(rec16 + 2 * (size_t)id); g1[kk] = __ldg(rec16 + 2 * (size_t)id + 1);
                }
            }
        }
#pragma unroll (HALF ? KPW : 1)
        for (int kk = 0; kk < KPW; ++kk) {
            const int k = w + kk * RAS_WARPS;
            const int i = k * 32 + lane;                              // fp32: the slot this thread gathered
            if (k * 32 >= len) { S.masks[lane * MASK_PITCH + k] = 0; continue; }
            uint32_t gm = 0;
            if (i < len) {
                if constexpr (HALF) {
                    // tile units relative to the macro-tile centre (|x| <= 4, |y| <= 2 inside the macro-tile)
                    const float mux = __uint_as_float(g0[kk].x), muy = __uint_as_float(g0[kk].y);
                    const float xt = (mux - (X0 + 0.5f * G::MT_W)) * (1.0f / TILE), yt = (muy - (Y0 + 0.5f * G::MT_H)) * (1.0f / TILE);
                    const float2 l01 = __half22float2(u2h2(g0[kk].z)), l2o = __half22float2(u2h2(g0[kk].w));
                    const __half2 xy = __floats2half2_rn(fminf(fmaxf(xt, -4000.0f), 4000.0f), fminf(fmaxf(yt, -4000.0f), 4000.0f));
                    s_rec16[2 * i] = make_uint4(h22u(xy), g0[kk].z, g0[kk].w, g1[kk].x);
                    reinterpret_cast<uint32_t*>(s_rec16 + 2 * i + 1)[0] = g1[kk].y;
                    // covariance of the prescaled Cholesky form, without cancellation: inverse = L L^T, L = [[l0,0],[l1,l2]]
                    //   det(inverse) = (l0 l2)^2, c = 1 / l2^2, a = (l1^2 + l2^2) / (l0 l2)^2, b = -l1 / (l0 l2^2)
                    // threshold in the same units: q' <= log2(255 o); 2 % + 0.05 on top for the half-precision q
                    const float il2 = rcp_approx(l2o.x), il0 = rcp_approx(l01.x);
                    const float c = il2 * il2, det = c * il0 * il0;
                    const float a = (l01.y * l01.y + l2o.x * l2o.x) * det, b = -l01.y * il0 * c;
                    const float tau_m = 1.02f * (7.99435344f + __log2f(l2o.y)) + 0.05f;
                    gm = tile_mask_cov<8>(xt, yt, a, b, c, det, tau_m, -4.0f, -2.0f, 1.0f, 1.0f, (fW - (X0 + 0.5f * G::MT_W)) * (1.0f / TILE),
                                       (fH - (Y0 + 0.5f * G::MT_H)) * (1.0f / TILE), 0.05f, 3000.0f) & ~cut;
                } else {
                    // c and det from the identities det = a / C, c = A det, cond = a c / det = A a (recomputing det from the
                    // conic as A C - B2^2/4 loses all digits for elongated gaussians); threshold = the oracle's tau_s
                    // (tau_scan, higs_internal.cuh) with 0.2 % on top
                    const float4 q0 = s_rec[REC_F4 * i], q1 = s_rec[REC_F4 * i + 1], q2 = s_rec[REC_F4 * i + 2];
                    const float det = q2.z * rcp_approx(q1.x);
                    const float tau_m = q1.y * fmaf(q0.z * q2.z, 9.5367431640625e-07f, 1.002f);
                    gm = tile_mask_cov<MTX>(q0.x, q0.y, q2.z, q2.w, q0.z * det, det, tau_m, X0, Y0, (float)TILE, 1.0f / TILE, fW, fH, 0.25f, 3.0e4f) & ~cut;
                }
            }
            uint32_t mine = 0;
            int lane_t = lane;
            asm volatile("" : "+r"(lane_t));                          // keeps the 32 lane == t predicates from being hoisted out of the loop
#pragma unroll                                                        // (kept alive across it they are packed into a register bit by bit and unpacked again)
            for (int t = 0; t < 32; ++t) {
                const uint32_t bt = __ballot_sync(0xffffffffu, (gm >> t) & 1u);
                if (lane_t == t) mine = bt;
            }
            S.masks[lane * MASK_PITCH + k] = mine;
        }
        __syncthreads();
        // tiles are handed out most-gaussians-first (the longest tile bounds the unit's tail); tiles nobody touches get
        // no claim at all: they publish the term of T = 1 here so that the prefix of later batches runs through.  lane = tile;
        // every warp computes the ranking for itself (no barrier, no shared table).
        uint32_t t_cnt = 0;
#pragma unroll
        for (int kk = 0; kk < RAS_MB; ++kk) t_cnt += __popc(S.masks[lane * MASK_PITCH + kk]);
        uint32_t t_rank = 0;
        {
            const uint32_t key = (t_cnt << 5) | (uint32_t)(31 - lane);
#pragma unroll
            for (int o = 0; o < 32; ++o) t_rank += __shfl_sync(0xffffffffu, key, o) > key ? 1u : 0u;
        }
        const int n_tiles = __popc(__ballot_sync(0xffffffffu, t_cnt != 0u));
        if (w == 0) {
            if (COUNT && t_cnt) atomicAdd(tile_load + (size_t)m * HIGS_MT_TILES + lane, t_cnt);   // Fig. 1 load map
            if (!t_cnt && use_cut && !((cut >> lane) & 1u)) cut_term[(size_t)u * HIGS_MT_TILES + lane] = -1;
        }

        // ---- Phase 2: warps claim render tiles (Alg. 1 lines 9-17), RasterizeTile (Alg. 2) ----
        for (;;) {
            int t = 0;
            if (lane == 0) t = (int)atomicAdd(&S.next_tile, 1u);
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t >= n_tiles) break;
            t = __ffs(__ballot_sync(0xffffffffu, t_cnt != 0u && t_rank == (uint32_t)t)) - 1;
            const uint32_t mine = lane < RAS_MB ? S.masks[t * MASK_PITCH + lane] : 0u;   // lane k holds mini-batch k's word
            const int col = (t & (MTX - 1)) * TILE + (lane % TILE), row0 = (t >> G::MT_SH) * TILE + (lane / TILE);   // inside the macro-tile
            uint32_t wr = 0, rd = 0, n_done = 0;
            bool sat = false;
            float tm;                                                 // largest transmittance left in the tile

            // Alg. 2: the tile's mask bits are compacted into the scheduling buffer and drained 8 gaussians at a time.  The paper
            // compacts one mask word at a time into a ring; a word holds 3 gaussians on average here, so the whole tile (or half
            // of it, when more than RING gaussians touch it) is compacted at once: a warp scan over the words' population counts
            // gives every lane the position of its word's first gaussian, and each lane writes out its own bits in order.
            auto walk = [&](auto&& drain8, auto&& saturated) {
                const uint32_t total = __reduce_add_sync(0xffffffffu, __popc(mine));
                const int n_parts = total > (uint32_t)RING ? 2 : 1;    // half of the words hold at most 16 x 32 = RING gaussians
                for (int part = 0; part < n_parts && !sat; ++part) {
                    uint32_t bits = (n_parts == 1 || (lane >> 4) == part) ? mine : 0u;
                    uint32_t incl = __popc(bits);
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
                    const uint32_t n = __shfl_sync(0xffffffffu, incl, 31);
                    uint32_t pos = incl - __popc(bits);
                    const uint32_t base = rec_s + (uint32_t)(lane * 32) * RasLayout<HALF>::stride;
                    while (bits) {
                        HIGS_ASSERT(pos < (uint32_t)RING);
                        ring[pos++] = base + (uint32_t)(__ffs(bits) - 1) * RasLayout<HALF>::stride;
                        bits &= bits - 1;
                    }
                    if (lane < 8) ring[n + lane] = rec_s + (uint32_t)NULL_IDX * RasLayout<HALF>::stride;   // the null gaussian pads the last drain
                    __syncwarp();
                    wr += n;
                    for (rd = 0; rd < n; ) {
                        drain8();
                        if (COUNT) n_done += 8;
                        if (__all_sync(0xffffffffu, saturated())) { sat = true; break; }   // Alg. 2 line 8
                    }
                    __syncwarp();                                     // buffer reads done before the next writes
                }
            };

            if constexpr (!HALF) {
                const float pxf = X0 + (float)col + 0.5f;
                float2 py2[NP], T2[NP], r2[NP], g2[NP], b2[NP];
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const float py = Y0 + (float)(row0 + G::RS * 2 * p) + 0.5f;
                    py2[p] = make_float2(py, py + (float)G::RS);
                    T2[p] = make_float2(1.0f, 1.0f); r2[p] = make_float2(0.f, 0.f); g2[p] = r2[p]; b2[p] = r2[p];
                }
                const float2 kexp = make_float2(-0.72134752f, -0.72134752f), neg1 = make_float2(-1.0f, -1.0f);
                auto drain8 = [&]() {                                 // 8 ring entries starting at rd (a multiple of 8), composited in order
                    const uint4 pk0 = *reinterpret_cast<const uint4*>(ring + rd);
                    const uint4 pk1 = *reinterpret_cast<const uint4*>(ring + rd + 4);
                    const uint32_t pkw[8] = { pk0.x, pk0.y, pk0.z, pk0.w, pk1.x, pk1.y, pk1.z, pk1.w };
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float4 a = lds128(pkw[e]), bq = lds128(pkw[e] + 16), cq = lds128(pkw[e] + 32);
                        // N-Q, pinned: dx, u = A dx, a0 = u dx, b0 = B2 dx, t = fma(C, dy, b0), q = fma(t, dy, a0)
                        const float dx = __fsub_rn(pxf, a.x);
                        const float2 ub = __fmul2_rn(make_float2(a.z, a.w), make_float2(dx, dx));   // u = A dx and b0 = B2 dx in one packed multiply
                        const float a0 = __fmul_rn(ub.x, dx);
                        const float bb = ub.y;
                        const float nmy = -a.y;
#pragma unroll
                        for (int p = 0; p < NP; ++p) {
                            const float2 dy = __fadd2_rn(py2[p], make_float2(nmy, nmy));    // py - muy for both rows (same rounding as a subtraction)
                            const float2 tq = __ffma2_rn(make_float2(bq.x, bq.x), dy, make_float2(bb, bb));
                            const float2 q = __ffma2_rn(tq, dy, make_float2(a0, a0));
                            const float2 ex = __ffma2_rn(q, kexp, make_float2(bq.z, bq.z));
                            float al0 = fminf(HIGS_ALPHA_MAX, ex2_approx(ex.x));
                            float al1 = fminf(HIGS_ALPHA_MAX, ex2_approx(ex.y));
                            al0 = (q.x <= bq.y) ? al0 : 0.0f;         // alpha < 1/255: skipped
                            al1 = (q.y <= bq.y) ? al1 : 0.0f;
                            const float2 wgt = __fmul2_rn(T2[p], make_float2(al0, al1));
                            r2[p] = __ffma2_rn(wgt, make_float2(bq.w, bq.w), r2[p]);
                            g2[p] = __ffma2_rn(wgt, make_float2(cq.x, cq.x), g2[p]);
                            b2[p] = __ffma2_rn(wgt, make_float2(cq.y, cq.y), b2[p]);
                            T2[p] = __ffma2_rn(wgt, neg1, T2[p]);
                        }
                    }
                    rd += 8;
                };
                auto tmax = [&]() {
                    float v = fmaxf(T2[0].x, T2[0].y);
#pragma unroll
                    for (int p = 1; p < NP; ++p) v = fmaxf(v, fmaxf(T2[p].x, T2[p].y));
                    return v;
                };
                walk(drain8, [&]() { return tmax() < HIGS_EPS_T; });
                float4* out = partial + ((size_t)u * HIGS_MT_TILES + t) * (TILE * TILE);
#pragma unroll
                for (int p = 0; p < NP; ++p) {                        // partial layout: [pixel i of the lane][lane]
                    __stcs(out + (2 * p) * 32 + lane, make_float4(r2[p].x, g2[p].x, b2[p].x, T2[p].x));
                    __stcs(out + (2 * p + 1) * 32 + lane, make_float4(r2[p].y, g2[p].y, b2[p].y, T2[p].y));
                }
                tm = tmax();
            } else {
                // tile units relative to the macro-tile centre: exact in half (multiples of 1/(2 TILE), |x| < 4, |y| < 2)
                const __half2 px2 = __float2half2_rn(((float)col + 0.5f - 0.5f * G::MT_W) * (1.0f / TILE));
                // T and the colour sums of one drain (8 gaussians) are half2; after every drain the colour sums are folded into
                // fp32 totals, so the half-precision additions only ever see the small sums of 8 terms (fp16 accumulation over
                // the 30-70 contributions of a pixel at paper scale costs 8 dB of PSNR: 59 instead of 67)
                __half2 py2[NP], T2[NP];
                float2 rf[NP], gf[NP], bf[NP];
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const float py = ((float)(row0 + G::RS * 2 * p) + 0.5f - 0.5f * G::MT_H) * (1.0f / TILE);
                    py2[p] = __floats2half2_rn(py, py + (float)G::RS * (1.0f / TILE));
                    T2[p] = __float2half2_rn(1.0f); rf[p] = make_float2(0.f, 0.f); gf[p] = rf[p]; bf[p] = rf[p];
                }
                const __half2 amax = __float2half2_rn(HIGS_ALPHA_MAX), amin = __float2half2_rn(1.0f / 255.0f);
                auto drain8 = [&]() {
                    const uint4 pk0 = *reinterpret_cast<const uint4*>(ring + rd);
                    const uint4 pk1 = *reinterpret_cast<const uint4*>(ring + rd + 4);
                    const uint32_t pkw[8] = { pk0.x, pk0.y, pk0.z, pk0.w, pk1.x, pk1.y, pk1.z, pk1.w };
                    __half2 r2[NP], g2[NP], b2[NP];
#pragma unroll
                    for (int p = 0; p < NP; ++p) { r2[p] = __float2half2_rn(0.0f); g2[p] = r2[p]; b2[p] = r2[p]; }
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint4 ra = lds128u(pkw[e]);
                        const uint32_t rb = lds32u(pkw[e] + RasLayout<HALF>::b_off);
                        const __half2 xy = u2h2(ra.x), l01 = u2h2(ra.y), l2o = u2h2(ra.z), rg = u2h2(ra.w), bb = u2h2(rb);
                        // q = (l0 dx + l1 dy)^2 + (l2 dy)^2, a sum of squares; alpha = o exp2(-q)
                        const __half2 dx = __hsub2(px2, __low2half2(xy));
                        const __half2 u0 = __hmul2(__low2half2(l01), dx);             // hoisted over the pixel pairs
#pragma unroll
                        for (int p = 0; p < NP; ++p) {
                            const __half2 dy = __hsub2(py2[p], __high2half2(xy));
                            const __half2 t1 = __hfma2(__high2half2(l01), dy, u0);
                            const __half2 t2 = __hmul2(__low2half2(l2o), dy);
                            const __half2 nq = __hfma2(__hneg2(t2), t2, __hmul2(__hneg2(t1), t1));
                            __half2 al = __hmin2(__hmul2(__high2half2(l2o), ex2_h2(nq)), amax);
                            al = __hmul2(al, __hge2(al, amin));           // alpha < 1/255: skipped
                            const __half2 wgt = __hmul2(T2[p], al);
                            r2[p] = __hfma2(wgt, __low2half2(rg), r2[p]);
                            g2[p] = __hfma2(wgt, __high2half2(rg), g2[p]);
                            b2[p] = __hfma2(wgt, __low2half2(bb), b2[p]);
                            T2[p] = __hsub2(T2[p], wgt);
                        }
                    }
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        const float2 dr = __half22float2(r2[p]), dg = __half22float2(g2[p]), db = __half22float2(b2[p]);
                        rf[p] = __fadd2_rn(rf[p], dr); gf[p] = __fadd2_rn(gf[p], dg); bf[p] = __fadd2_rn(bf[p], db);
                    }
                    rd += 8;
                };
                auto tmax2 = [&]() {
                    __half2 v = T2[0];
#pragma unroll
                    for (int p = 1; p < NP; ++p) v = __hmax2(v, T2[p]);
                    return fmaxf(__low2float(v), __high2float(v));
                };
                walk(drain8, [&]() { return tmax2() < HIGS_EPS_T; });
                // fp16 partials: per lane and pixel pair 16 B = half2 r, g, b, T of the pair (16 KB per unit)
                uint4* out16 = reinterpret_cast<uint4*>(partial) + ((size_t)u * HIGS_MT_TILES + t) * (TILE * TILE / 2);
#pragma unroll
                for (int p = 0; p < NP; ++p)
                    __stcs(out16 + p * 32 + lane, make_uint4(h22u(__float22half2_rn(rf[p])), h22u(__float22half2_rn(gf[p])), h22u(__float22half2_rn(bf[p])), h22u(T2[p])));
                tm = tmax2();
            }
            if (COUNT) { n_tp += wr; n_eval_g += n_done; }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, d));
            if (lane == 0) {
                if (use_cut) {                                        // log2 of the largest transmittance left, rounded towards zero
                    const int q = max(-32768, min(0, (int)ceilf(__log2f(fmaxf(tm, 1e-30f)) * LOGT_SCALE) + 2));
                    cut_term[(size_t)u * HIGS_MT_TILES + t] = q - 1;
                }
                atomicOr(&S.active, 1u << t);
            }
        }
    }
    if (COUNT && lane == 0) {                                         // both counters are warp-uniform
        atomicAdd(&hdr->n_evals, n_eval_g * (unsigned long long)(TILE * TILE));
        atomicAdd(&hdr->n_tile_pairs, n_tp);
    }
}

// a8: one warp per render tile; Eq. (1): C = C_0 + T_0 C_1 + T_0 T_1 C_2 + ...  fp32 accumulation on both paths.
template <int TILE, bool HALF, int MTX = 8>
__global__ void __launch_bounds__(256)
k_merge_image(const float4* __restrict__ partial, const uint32_t* __restrict__ unit_active,
              const uint32_t* __restrict__ batch_offset, const FrameParams P, const FrameHeader* __restrict__ hdr,
              float* __restrict__ out_rgb)
{
    typedef TileGeo<TILE, MTX> G;
    constexpr int PPL = G::PPL;
    const int lane = threadIdx.x & 31;
    pdl_wait();
    const int gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int m = gw >> 5, t = gw & 31;
    if (m >= P.n_m) return;
    const int mtx = m % P.n_mx, mty = m / P.n_mx;
    const int tcol = (t & (MTX - 1)) * TILE, trow = (t >> G::MT_SH) * TILE;
    const int x = mtx * G::MT_W + tcol + (lane % TILE);
    const int y0 = mty * G::MT_H + trow + (lane / TILE);
    if (mtx * G::MT_W + tcol >= P.W || mty * G::MT_H + trow >= P.H) return;
    uint32_t u0 = 0, nb = 0;
    if (!hdr->overflow) { u0 = batch_offset[m]; nb = batch_offset[m + 1] - u0; }   // this macro-tile's units, in depth order
    float T[PPL], r[PPL], g[PPL], b[PPL];
#pragma unroll
    for (int i = 0; i < PPL; ++i) { T[i] = 1.0f; r[i] = 0.f; g[i] = 0.f; b[i] = 0.f; }
    for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t act = __ldg(unit_active + u0 + j);
        if (!((act >> t) & 1u)) continue;
        const float4* p = partial + ((size_t)(u0 + j) * HIGS_MT_TILES + t) * (HALF ? 32 : 64) * (TILE * TILE / 64);
        bool all_sat = true;
        if constexpr (HALF) {
            const uint4* p16 = reinterpret_cast<const uint4*>(p);
#pragma unroll
            for (int q = 0; q < PPL / 2; ++q) {
                const uint4 c = __ldcs(p16 + q * 32 + lane);
                const float2 cr = __half22float2(u2h2(c.x)), cg = __half22float2(u2h2(c.y)), cb = __half22float2(u2h2(c.z)), cT = __half22float2(u2h2(c.w));
                r[2 * q] = fmaf(T[2 * q], cr.x, r[2 * q]); g[2 * q] = fmaf(T[2 * q], cg.x, g[2 * q]); b[2 * q] = fmaf(T[2 * q], cb.x, b[2 * q]); T[2 * q] *= cT.x;
                r[2 * q + 1] = fmaf(T[2 * q + 1], cr.y, r[2 * q + 1]); g[2 * q + 1] = fmaf(T[2 * q + 1], cg.y, g[2 * q + 1]);
                b[2 * q + 1] = fmaf(T[2 * q + 1], cb.y, b[2 * q + 1]); T[2 * q + 1] *= cT.y;
                all_sat = all_sat && T[2 * q] < HIGS_EPS_T && T[2 * q + 1] < HIGS_EPS_T;
            }
        } else {
#pragma unroll
            for (int i = 0; i < PPL; ++i) {
                const float4 c = __ldcs(p + i * 32 + lane);
                r[i] = fmaf(T[i], c.x, r[i]); g[i] = fmaf(T[i], c.y, g[i]); b[i] = fmaf(T[i], c.z, b[i]); T[i] *= c.w;
                all_sat = all_sat && T[i] < HIGS_EPS_T;
            }
        }
        if (__all_sync(0xffffffffu, all_sat)) break;
    }
    if (x < P.W) {
#pragma unroll
        for (int i = 0; i < PPL; ++i) {
            const int y = y0 + G::RS * i;
            if (y < P.H) { float* o = out_rgb + ((size_t)y * P.W + x) * 3; o[0] = r[i]; o[1] = g[i]; o[2] = b[i]; }
        }
    }
}

template <bool COUNT, int TILE, bool HALF, int MTX = 8>
int setup_one(higs_ctx* ctx, int* occ_out)
{
    const int smem = (int)ras_smem_bytes<HALF>();
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_raster<COUNT, TILE, HALF, MTX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (occ_out) {
        int occ = 0;
        HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_raster<COUNT, TILE, HALF, MTX>, RAS_THREADS, smem));
        *occ_out = occ > 0 ? occ : 1;
    }
    return HIGS_OK;
}

template <bool COUNT, int TILE, bool HALF, int MTX = 8>
void launch_one(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    const int grid = ctx->n_sm * ctx->raster_ctas_per_sm[TILE == 16][HALF];
    k_raster<COUNT, TILE, HALF, MTX><<<grid, RAS_THREADS, ras_smem_bytes<HALF>(), st>>>(
        ctx->pairs, ctx->rec, ctx->rec16, ctx->mt_offset, ctx->mt_count, ctx->batch_offset, ctx->unit_mt, ctx->unit_order, P, ctx->hdr,
        ctx->partial, ctx->unit_active, ctx->cut_word, ctx->cut_term, ctx->tile_load);
}

} // namespace

int higs_raster_setup(higs_ctx* ctx)
{
    int rc;
    if ((rc = setup_one<false, 8, false>(ctx, &ctx->raster_ctas_per_sm[0][0]))) return rc;
    if ((rc = setup_one<true, 8, false>(ctx, nullptr))) return rc;
    if ((rc = setup_one<false, 8, true>(ctx, &ctx->raster_ctas_per_sm[0][1]))) return rc;
    if ((rc = setup_one<true, 8, true>(ctx, nullptr))) return rc;
    if ((rc = setup_one<false, 16, false>(ctx, &ctx->raster_ctas_per_sm[1][0]))) return rc;
    if ((rc = setup_one<true, 16, false>(ctx, nullptr))) return rc;
    if ((rc = setup_one<false, 16, true>(ctx, &ctx->raster_ctas_per_sm[1][1]))) return rc;
    if ((rc = setup_one<true, 16, true>(ctx, nullptr))) return rc;
    if ((rc = setup_one<false, 8, false, 4>(ctx, nullptr))) return rc;
    if ((rc = setup_one<true, 8, false, 4>(ctx, nullptr))) return rc;
    if ((rc = setup_one<false, 8, false, 16>(ctx, nullptr))) return rc;
    if ((rc = setup_one<true, 8, false, 16>(ctx, nullptr))) return rc;
    return HIGS_OK;
}

int launch_raster(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    const bool count = (P.flags & HIGS_FLAG_COUNT_EVALS) != 0, half = (P.flags & HIGS_FLAG_FP16) != 0;
#define HIGS_RAS(T, H) do { if (count) launch_one<true, T, H>(ctx, P, st); else launch_one<false, T, H>(ctx, P, st); } while (0)
    if (P.mt_tx != 8) {                                               // shape sweep: fp32 path, 8 x 8 tiles (render_impl checks the combination)
        if (P.tile != 8 || half) return HIGS_E_ARG;
        if (P.mt_tx == 4) { if (count) launch_one<true, 8, false, 4>(ctx, P, st); else launch_one<false, 8, false, 4>(ctx, P, st); }
        else              { if (count) launch_one<true, 8, false, 16>(ctx, P, st); else launch_one<false, 8, false, 16>(ctx, P, st); }
    }
    else if (P.tile == 16) { if (half) HIGS_RAS(16, true); else HIGS_RAS(16, false); }
    else              { if (half) HIGS_RAS(8, true);  else HIGS_RAS(8, false); }
#undef HIGS_RAS
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int launch_merge(higs_ctx* ctx, const FrameParams& P, float* out_rgb, cudaStream_t st)
{
    const int warps = P.n_m * HIGS_MT_TILES;
    const bool half = (P.flags & HIGS_FLAG_FP16) != 0;
#define HIGS_MRG(T, H) HIGS_CUDA(ctx, launch_pdl(k_merge_image<T, H>, dim3((warps + 7) / 8), dim3(256), 0, st, ctx->partial, ctx->unit_active, \
                                                 ctx->batch_offset, P, ctx->hdr, out_rgb))
#define HIGS_MRG_MT(X) HIGS_CUDA(ctx, launch_pdl(k_merge_image<8, false, X>, dim3((warps + 7) / 8), dim3(256), 0, st, ctx->partial, ctx->unit_active, \
                                                 ctx->batch_offset, P, ctx->hdr, out_rgb))
    if (P.mt_tx == 4) HIGS_MRG_MT(4);
    else if (P.mt_tx == 16) HIGS_MRG_MT(16);
    else if (P.tile == 16) { if (half) HIGS_MRG(16, true); else HIGS_MRG(16, false); }
    else              { if (half) HIGS_MRG(8, true);  else HIGS_MRG(8, false); }
#undef HIGS_MRG
#undef HIGS_MRG_MT
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}
