// raster.cu -- steps a7 macro-tile rasterizer and a8 post-blend merge
// (section 3.4 with Alg. 1 MacroTileRasterize and Alg. 2 RasterizeTile,
//  PAPER.md:278-301 section 4.5, Eq. (1)).
//
// A work unit is one (macro-tile, batch of <= B_r gaussians).  A persistent CTA claims
// units from a device counter.  Phase 1 (Alg. 1 lines 1-8): the unit's records are gathered by sorted
// id straight into shared memory with cp.async (LDGSTS), every thread derives the 32-bit render-tile
// overlap mask of its gaussian, and a warp ballot transposes 32 gaussians x 32 tiles so that one
// word per (tile, mini-batch) says which gaussians touch the tile.  Phase 2 (Alg. 1 lines 9-17,
// Alg. 2): warps claim render tiles from a shared counter; a warp owns the 8x8 tile (two pixels per
// lane, rows y and y+4 of one column, so the dx terms are shared), walks the tile's mask words,
// reads each listed gaussian as three broadcast LDS.128 (48 B, as gathered) and composites front to back; after every
// mask word a unanimous vote on T < eps ends the tile early (Alg. 2 line 8).  Partial (r,g,b,T) per
// pixel goes to the dense (unit, tile) buffer, the unit's 32-bit active mask out of band
// (PAPER.md:284).  The merge kernel gives one warp per render tile and folds the macro-tile's units
// in depth order with Eq. (1), stopping once every pixel is saturated.
//
// fp32 throughout.  The skip decision q <= tau uses the pinned sequence N-Q
// in absolute pixel coordinates, so it is bit-identical to the oracle's; alpha, colour and T are
// "smooth" and use ex2.approx.
#include <stdio.h>
#include "higs_internal.cuh"

namespace {

constexpr int RAS_THREADS = 256;                  // 3 CTAs per SM at 80 registers (4 at 64 registers measured 2 % slower)
constexpr int RAS_WARPS = RAS_THREADS / 32;
constexpr int RAS_SUB = HIGS_BATCH_CAP;           // gaussians per unit
constexpr int RAS_MB = RAS_SUB / 32;              // mini-batches of 32 gaussians per unit
constexpr int MASK_PITCH = RAS_MB + 1;
constexpr float LOGT_SCALE = 1024.0f;             // fixed point of the running log2 transmittance bounds
constexpr int LOGT_EPS = -13608;                  // floor(log2(1e-4) * 1024): a sum below it proves T < eps
constexpr int RING = 64;                          // per-warp ring of staged-record addresses, drained 8 at a time (B_d, 8x unroll)
constexpr int NULL_IDX = RAS_SUB;                 // index of the "null" gaussian that pads the last drain

// Shared-memory record of one staged gaussian: the first 48 B of its global record, as gathered:
//   f4[0] = mux, muy, A, B2      f4[1] = C, tau, log2 o, r      f4[2] = g, b, cov a, cov b
// Packed f32x2 instructions (FFMA2 / FMUL2 / FADD2) take a plain 32-bit register as a broadcast operand, so the values
// that multiply both pixels of a lane need no duplicated copy in shared memory.
constexpr int REC_F4 = 3;
struct __align__(16) RasSmem {
    float4 rec[(RAS_SUB + 1) * REC_F4];
    uint32_t masks[HIGS_MT_TILES * MASK_PITCH];   // [tile][mini-batch]: bit j = gaussian k*32+j touches the tile
    uint32_t ring[RAS_WARPS][RING];              // shared-window byte addresses of the records: an entry is an LDS operand as it stands
    uint32_t unit, next_tile, n_tiles, active, cut;
    uint8_t order[HIGS_MT_TILES];                 // tile of the i-th tile claim: most gaussians first
};

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
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Conservative render-tile overlap mask of one gaussian inside macro-tile (X0, Y0) (reading Q9:
// internal, never compared with the oracle).  N-SCAN at 8-px cells on the COVARIANCE (a, b, c), on the threshold
//   tau_m = tau (1.002 + 2^-20 cond),  cond = a c / det,
// i.e. the oracle's tau_s (the region the fp32 pixel test accepts stays inside the ellipse of tau_s, see tau_scan)
// with 0.2 % on top.  The staged record has a, b and the conic; c and det come from the identities det = a / C,
// c = A det, cond = A a, which do not cancel - recomputing det from the conic as A C - B2^2/4 loses all digits for
// elongated gaussians (cond ~ 1/eps).  With approximate rcp / sqrt every extent is good to ~1e-6 relative; extents are
// widened by 0.25 px on top, pixel centres sit 0.5 px inside their tile, and gaussians larger than 3e4 px take every tile.
__device__ __forceinline__ uint32_t tile_mask_cov(float mux, float muy, float A, float C, float tau, float a, float b,
                                                  float X0, float Y0, float fW, float fH)
{
    const float det = a * rcp_approx(C);
    const float c = A * det;
    const float tau_m = tau * fmaf(A * a, 9.5367431640625e-07f, 1.002f);
    const float hx = sqrt_approx(tau_m * a) + 0.25f, hy = sqrt_approx(tau_m * c) + 0.25f;
    if (!(det > 0.0f) || !(c > 0.0f) || !(hx < 3.0e4f) || !(hy < 3.0e4f)) return 0xffffffffu;
    const float rc = rcp_approx(c);
    const float boc = b * rc, sdet = det * rc;
    const float yR = b * sqrt_approx(tau_m * rcp_approx(a));          // dy of the rightmost point
    const float ytop = muy - hy, ybot = muy + hy;
    uint32_t mask = 0;
#pragma unroll
    for (int tr = 0; tr < 4; ++tr) {
        const float y0 = Y0 + 8.0f * tr;
        const float y1 = fminf(y0 + 8.0f, fH);
        const float ylo = fmaxf(y0, ytop) - muy, yhi = fminf(y1, ybot) - muy;
        if (!(yhi >= ylo)) continue;
        const float rlo = sqrt_approx(fmaxf(0.0f, sdet * fmaf(-ylo * ylo, rc, tau_m)));
        const float rhi = sqrt_approx(fmaxf(0.0f, sdet * fmaf(-yhi * yhi, rc, tau_m)));
        float xmax = (ylo <= yR && yR <= yhi) ? hx : fmaxf(fmaf(boc, ylo, rlo), fmaf(boc, yhi, rhi)) + 0.25f;
        float xmin = (ylo <= -yR && -yR <= yhi) ? -hx : fminf(fmaf(boc, ylo, -rlo), fmaf(boc, yhi, -rhi)) - 0.25f;
        xmax = fminf(xmax + mux, fW) - X0; xmin = fmaxf(xmin + mux, 0.0f) - X0;
        if (!(xmax >= 0.0f) || !(xmin < 64.0f) || !(xmax >= xmin)) continue;
        const int c0 = max(0, (int)floorf(xmin * 0.125f)), c1 = min(7, (int)floorf(xmax * 0.125f));
        if (c0 > c1) continue;
        mask |= ((2u << c1) - (1u << c0)) << (tr * 8);
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

template <bool COUNT>
__global__ void __launch_bounds__(RAS_THREADS, 3)
k_raster(const unsigned long long* __restrict__ pairs, const float4* __restrict__ rec,
         const uint32_t* __restrict__ mt_offset, const uint32_t* __restrict__ mt_count,
         const uint32_t* __restrict__ batch_offset, const uint32_t* __restrict__ unit_mt,
         const uint32_t* __restrict__ unit_order,
         const FrameParams P, FrameHeader* __restrict__ hdr,
         float4* __restrict__ partial, uint32_t* __restrict__ unit_active,
         unsigned long long* __restrict__ cut_word, int* __restrict__ cut_term)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    RasSmem& S = *reinterpret_cast<RasSmem*>(s_raw);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    pdl_trigger();                                                    // k_merge_image may be scheduled as this grid drains
    const uint32_t n_units = hdr->n_units;
    const bool use_cut = !(P.flags & HIGS_FLAG_NO_XBATCH_CUT);
    const float fW = (float)P.W, fH = (float)P.H;
    unsigned long long n_eval_g = 0, n_tp = 0;
    if (threadIdx.x == 0) {                                           // the null gaussian: tau < 0, never passes q <= tau
        S.rec[NULL_IDX * REC_F4] = make_float4(0.f, 0.f, 0.f, 0.f); S.rec[NULL_IDX * REC_F4 + 1] = make_float4(0.f, -1.0f, 0.f, 0.f);
        S.rec[NULL_IDX * REC_F4 + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    uint32_t* ring = S.ring[w];
    const uint32_t rec_s = (uint32_t)__cvta_generic_to_shared(S.rec);

    for (;;) {
        __syncthreads();                                              // everyone is done with the previous unit's shared state
        // Warp 0 claims units until one has something left to show.  Tiles wholly outside the image are never active
        // (Alg. 1 line 11, InBounds); tiles whose bound from the batches in front is below eps are cut (lane = tile).
        // A unit with every tile cut costs one atomic and a few loads: it is never gathered.
        if (w == 0) {
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
                const int tiles_x = min(8, (P.W - mtx * HIGS_MT_W + HIGS_TILE - 1) / HIGS_TILE);
                const int tiles_y = min(4, (P.H - mty * HIGS_MT_H + HIGS_TILE - 1) / HIGS_TILE);
                bool saturated = false;
                if (use_cut && jc > 0)
                    saturated = cut_prefix(cut_word + (size_t)mc * HIGS_MT_TILES + lane, cut_term + (size_t)u0c * HIGS_MT_TILES + lane, jc) < LOGT_EPS;
                const bool inb = (lane & 7) < tiles_x && (lane >> 3) < tiles_y;
                const uint32_t cut = __ballot_sync(0xffffffffu, saturated || !inb);
                if (cut == 0xffffffffu) {                             // nothing left to see behind the earlier batches
                    if (lane == 0) unit_active[uc] = 0;
                    continue;
                }
                u_sel = uc; cut_sel = cut;
                break;
            }
            if (lane == 0) { S.unit = u_sel; S.cut = cut_sel; S.next_tile = 0; S.active = 0; }
        }
        __syncthreads();
        const uint32_t u = S.unit;
        if (u == 0xffffffffu) break;
        const uint32_t cut = S.cut;
        const uint32_t m = unit_mt[u];
        const uint32_t u0 = batch_offset[m];
        const uint32_t j = u - u0;
        const uint32_t seg_n = mt_count[m];
        const uint32_t start = mt_offset[m] + j * (uint32_t)P.batch_cap;
        const int len = (int)min((uint32_t)P.batch_cap, seg_n - j * (uint32_t)P.batch_cap);
        const int mtx = (int)(m % (uint32_t)P.n_mx), mty = (int)(m / (uint32_t)P.n_mx);
        const float X0 = (float)(mtx * HIGS_MT_W), Y0 = (float)(mty * HIGS_MT_H);

        // ---- Phase 1a: gather of this unit's records (Alg. 1 line 4), first 48 B of each, by sorted id ----
        for (int i = threadIdx.x; i < len; i += RAS_THREADS) {
            const uint32_t id = (uint32_t)pairs[start + i];
            const float4* src = rec + 4 * (size_t)id;
            cp_async16(&S.rec[REC_F4 * i], src);
            cp_async16(&S.rec[REC_F4 * i + 1], src + 1);
            cp_async16(&S.rec[REC_F4 * i + 2], src + 2);
        }
        cp_async_wait_all();                                          // each thread waits for the records it asked for
        __syncthreads();

        // ---- Phase 1b: per-gaussian tile masks (Alg. 1 lines 5-6), transposed by ballot ----
        for (int k = w; k < RAS_MB; k += RAS_WARPS) {
            const int i = k * 32 + lane;                              // == threadIdx.x + RAS_THREADS*(k/RAS_WARPS): the slot this thread gathered
            if (k * 32 >= len) { S.masks[lane * MASK_PITCH + k] = 0; continue; }
            uint32_t gm = 0;
            if (i < len) {
                const float4 a = S.rec[REC_F4 * i], b = S.rec[REC_F4 * i + 1], c = S.rec[REC_F4 * i + 2];
                gm = tile_mask_cov(a.x, a.y, a.z, b.x, b.y, c.z, c.w, X0, Y0, fW, fH) & ~cut;
            }
            uint32_t mine = 0;
#pragma unroll
            for (int t = 0; t < 32; ++t) {
                const uint32_t bt = __ballot_sync(0xffffffffu, (gm >> t) & 1u);
                if (lane == t) mine = bt;
            }
            S.masks[lane * MASK_PITCH + k] = mine;
        }
        __syncthreads();
        // tiles are handed out most-gaussians-first (the longest tile bounds the unit's tail); tiles nobody touches get
        // no claim at all: they publish the term of T = 1 here so that the prefix of later batches runs through.  lane = tile.
        if (w == 0) {
            uint32_t cnt = 0;
#pragma unroll
            for (int kk = 0; kk < RAS_MB; ++kk) cnt += __popc(S.masks[lane * MASK_PITCH + kk]);
            const uint32_t key = (cnt << 5) | (uint32_t)(31 - lane);
            uint32_t rank = 0;
#pragma unroll
            for (int o = 0; o < 32; ++o) rank += __shfl_sync(0xffffffffu, key, o) > key ? 1u : 0u;
            if (cnt) S.order[rank] = (uint8_t)lane;
            else if (use_cut && !((cut >> lane) & 1u)) cut_term[(size_t)u * HIGS_MT_TILES + lane] = -1;
            const uint32_t nt = __popc(__ballot_sync(0xffffffffu, cnt != 0u));
            if (lane == 0) S.n_tiles = nt;
        }
        __syncthreads();
        const int n_tiles = (int)S.n_tiles;

        // ---- Phase 2: warps claim render tiles (Alg. 1 lines 9-17), RasterizeTile (Alg. 2) ----
        for (;;) {
            int t = 0;
            if (lane == 0) t = (int)atomicAdd(&S.next_tile, 1u);
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t >= n_tiles) break;
            t = (int)S.order[t];
            const uint32_t mine = lane < RAS_MB ? S.masks[t * MASK_PITCH + lane] : 0u;   // lane k holds mini-batch k's word
            uint32_t rest = __ballot_sync(0xffffffffu, mine != 0u);
            const float pxf = X0 + (float)((t & 7) * HIGS_TILE + (lane & 7)) + 0.5f;
            const float py0 = Y0 + (float)((t >> 3) * HIGS_TILE + (lane >> 3)) + 0.5f;
            const float py1 = py0 + 4.0f;
            const float2 py2 = make_float2(py0, py1);
            float2 T2 = make_float2(1.0f, 1.0f), r2 = make_float2(0.f, 0.f), g2 = r2, b2 = r2;
            const float2 kexp = make_float2(-0.72134752f, -0.72134752f), neg1 = make_float2(-1.0f, -1.0f);
            uint32_t wr = 0, rd = 0;
            bool sat = false;
            // one drain: 8 ring entries starting at rd (a multiple of 8), composited in order
            auto drain8 = [&]() {
                const uint4 pk0 = *reinterpret_cast<const uint4*>(ring + (rd & (RING - 1)));
                const uint4 pk1 = *reinterpret_cast<const uint4*>(ring + (rd & (RING - 1)) + 4);
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
                    const float2 dy = __fadd2_rn(py2, make_float2(nmy, nmy));    // py - muy for both rows (same rounding as a subtraction)
                    const float2 tq = __ffma2_rn(make_float2(bq.x, bq.x), dy, make_float2(bb, bb));
                    const float2 q = __ffma2_rn(tq, dy, make_float2(a0, a0));
                    const float2 ex = __ffma2_rn(q, kexp, make_float2(bq.z, bq.z));
                    float al0 = fminf(HIGS_ALPHA_MAX, ex2_approx(ex.x));
                    float al1 = fminf(HIGS_ALPHA_MAX, ex2_approx(ex.y));
                    al0 = (q.x <= bq.y) ? al0 : 0.0f;                 // alpha < 1/255: skipped
                    al1 = (q.y <= bq.y) ? al1 : 0.0f;
                    const float2 wgt = __fmul2_rn(T2, make_float2(al0, al1));
                    r2 = __ffma2_rn(wgt, make_float2(bq.w, bq.w), r2);
                    g2 = __ffma2_rn(wgt, make_float2(cq.x, cq.x), g2);
                    b2 = __ffma2_rn(wgt, make_float2(cq.y, cq.y), b2);
                    T2 = __ffma2_rn(wgt, neg1, T2);
                }
                rd += 8;
            };
            while (rest) {
                const int k = __ffs(rest) - 1;
                rest &= rest - 1;
                const uint32_t bits = __shfl_sync(0xffffffffu, mine, k);
                if ((bits >> lane) & 1u) ring[(wr + __popc(bits & lt_mask)) & (RING - 1)] = rec_s + (uint32_t)(k * 32 + lane) * (REC_F4 * 16u);
                wr += __popc(bits);
                __syncwarp();
                while (wr - rd >= 8u) {
                    drain8();
                    if (__all_sync(0xffffffffu, fmaxf(T2.x, T2.y) < HIGS_EPS_T)) { sat = true; break; }   // Alg. 2 line 8
                }
                if (sat) break;
            }
            if (!sat && wr > rd) {                                    // flush: pad the last drain with the null gaussian
                if (lane < 8) ring[(wr + lane) & (RING - 1)] = rec_s + (uint32_t)NULL_IDX * (REC_F4 * 16u);
                __syncwarp();
                drain8();
            }
            __syncwarp();                                             // ring reads done before the next tile's writes
            if (COUNT) { n_tp += wr; n_eval_g += min(rd, wr); }
            float4* out = partial + ((size_t)u * HIGS_MT_TILES + t) * 64;
            __stcs(out + lane, make_float4(r2.x, g2.x, b2.x, T2.x));
            __stcs(out + 32 + lane, make_float4(r2.y, g2.y, b2.y, T2.y));
            float tm = fmaxf(T2.x, T2.y);
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
        __syncthreads();
        if (threadIdx.x == 0) unit_active[u] = S.active;
    }
    if (COUNT && lane == 0) {                                         // both counters are warp-uniform
        atomicAdd(&hdr->n_evals, n_eval_g * 64ull);
        atomicAdd(&hdr->n_tile_pairs, n_tp);
    }
}

// a8: one warp per render tile; Eq. (1): C = C_0 + T_0 C_1 + T_0 T_1 C_2 + ...
__global__ void __launch_bounds__(256)
k_merge_image(const float4* __restrict__ partial, const uint32_t* __restrict__ unit_active,
              const uint32_t* __restrict__ batch_offset, const FrameParams P, const FrameHeader* __restrict__ hdr,
              float* __restrict__ out_rgb)
{
    const int lane = threadIdx.x & 31;
    pdl_wait();
    const int gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int m = gw >> 5, t = gw & 31;
    if (m >= P.n_m) return;
    const int mtx = m % P.n_mx, mty = m / P.n_mx;
    const int x = mtx * HIGS_MT_W + (t & 7) * HIGS_TILE + (lane & 7);
    const int y0 = mty * HIGS_MT_H + (t >> 3) * HIGS_TILE + (lane >> 3);
    if (mtx * HIGS_MT_W + (t & 7) * HIGS_TILE >= P.W || mty * HIGS_MT_H + (t >> 3) * HIGS_TILE >= P.H) return;
    uint32_t u0 = 0, nb = 0;
    if (!hdr->overflow) { u0 = batch_offset[m]; nb = batch_offset[m + 1] - u0; }   // this macro-tile's units, in depth order
    float T0 = 1.0f, T1 = 1.0f, r0 = 0, g0 = 0, b0 = 0, r1 = 0, g1 = 0, b1 = 0;
    for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t act = __ldg(unit_active + u0 + j);
        if (!((act >> t) & 1u)) continue;
        const float4* p = partial + ((size_t)(u0 + j) * HIGS_MT_TILES + t) * 64;
        const float4 c0 = __ldcs(p + lane), c1 = __ldcs(p + 32 + lane);
        r0 = fmaf(T0, c0.x, r0); g0 = fmaf(T0, c0.y, g0); b0 = fmaf(T0, c0.z, b0); T0 *= c0.w;
        r1 = fmaf(T1, c1.x, r1); g1 = fmaf(T1, c1.y, g1); b1 = fmaf(T1, c1.z, b1); T1 *= c1.w;
        if (__all_sync(0xffffffffu, T0 < HIGS_EPS_T && T1 < HIGS_EPS_T)) break;
    }
    if (x < P.W) {
        if (y0 < P.H) { float* o = out_rgb + ((size_t)y0 * P.W + x) * 3; o[0] = r0; o[1] = g0; o[2] = b0; }
        if (y0 + 4 < P.H) { float* o = out_rgb + ((size_t)(y0 + 4) * P.W + x) * 3; o[0] = r1; o[1] = g1; o[2] = b1; }
    }
}

} // namespace

int higs_raster_setup(higs_ctx* ctx)
{
    const int smem = (int)sizeof(RasSmem);
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_raster<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_raster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_raster<false>, RAS_THREADS, smem));
    ctx->raster_ctas_per_sm = occ > 0 ? occ : 1;
    return HIGS_OK;
}

int launch_raster(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    const int smem = (int)sizeof(RasSmem);
    const int grid = ctx->n_sm * ctx->raster_ctas_per_sm;
    if (P.flags & HIGS_FLAG_COUNT_EVALS)
        k_raster<true><<<grid, RAS_THREADS, smem, st>>>(ctx->pairs, ctx->rec, ctx->mt_offset, ctx->mt_count, ctx->batch_offset,
                                                        ctx->unit_mt, ctx->unit_order, P, ctx->hdr, ctx->partial, ctx->unit_active, ctx->cut_word, ctx->cut_term);
    else
        k_raster<false><<<grid, RAS_THREADS, smem, st>>>(ctx->pairs, ctx->rec, ctx->mt_offset, ctx->mt_count, ctx->batch_offset,
                                                         ctx->unit_mt, ctx->unit_order, P, ctx->hdr, ctx->partial, ctx->unit_active, ctx->cut_word, ctx->cut_term);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int launch_merge(higs_ctx* ctx, const FrameParams& P, float* out_rgb, cudaStream_t st)
{
    const int warps = P.n_m * HIGS_MT_TILES;
    HIGS_CUDA(ctx, launch_pdl(k_merge_image, dim3((warps + 7) / 8), dim3(256), 0, st, ctx->partial, ctx->unit_active, ctx->batch_offset, P,
                              ctx->hdr, out_rgb));
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}
