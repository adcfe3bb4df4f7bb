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
// reads each listed gaussian as three broadcast LDS.128 and composites front to back; after every
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

constexpr int RAS_THREADS = 256;
constexpr int RAS_WARPS = RAS_THREADS / 32;
constexpr int MASK_PITCH = 33;

struct __align__(16) RasSmem {
    float4 rec[HIGS_BATCH_CAP * 3];               // 48 B per gaussian: mux,muy,A,B2 | C,tau,log2o,r | g,b,-,-
    uint32_t masks[HIGS_MT_TILES * MASK_PITCH];   // [tile][mini-batch]
    uint32_t unit, next_tile, active, cut;
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Conservative render-tile overlap mask of one gaussian inside macro-tile (mtx, mty): the row scan
// at 8-px cells on a threshold inflated by 1e-3 (internal; reading Q9 -- never compared
// with the oracle, only required to keep every pixel centre with q <= tau).
__device__ __forceinline__ uint32_t tile_mask(const float4 g0, const float4 g1, int mtx, int mty, const FrameParams& P)
{
    const float A = g0.z, B2 = g0.w, C = g1.x;
    const float tau = g1.y * 1.001f;
    const float det = A * C - 0.25f * B2 * B2;
    if (!(det > 0.0f)) return 0xffffffffu;
    const float rd = 1.0f / det;
    const float a = C * rd, b = -0.5f * B2 * rd, c = A * rd;
    const int ncx = (P.W + HIGS_TILE - 1) / HIGS_TILE, ncy = (P.H + HIGS_TILE - 1) / HIGS_TILE;
    RowScan rs;
    rs.init(g0.x, g0.y, a, b, c, tau, (float)HIGS_TILE, ncy);
    const int R0 = mty * 4, C0 = mtx * 8;
    const int ra = max(rs.r0, R0), rb = min(rs.r1, R0 + 3);
    uint32_t mask = 0;
    for (int r = ra; r <= rb; ++r) {
        int m0, m1;
        if (!rs.row(r, (float)HIGS_TILE, (float)HIGS_TILE, (float)P.W, (float)P.H, ncx, m0, m1)) continue;
        m0 = max(m0, C0); m1 = min(m1, C0 + 7);
        if (m0 > m1) continue;
        const uint32_t bits = (2u << (m1 - C0)) - (1u << (m0 - C0));
        mask |= bits << ((r - R0) * 8);
    }
    return mask;
}

template <bool COUNT>
__global__ void __launch_bounds__(RAS_THREADS, 4)
k_raster(const unsigned long long* __restrict__ pairs, const float4* __restrict__ ras,
         const uint32_t* __restrict__ mt_offset, const uint32_t* __restrict__ mt_count,
         const uint32_t* __restrict__ batch_offset, const uint32_t* __restrict__ unit_mt,
         const FrameParams P, FrameHeader* __restrict__ hdr,
         float4* __restrict__ partial, uint32_t* __restrict__ unit_active, float* __restrict__ tile_maxT)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    RasSmem& S = *reinterpret_cast<RasSmem*>(s_raw);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t n_units = hdr->n_units;
    const bool use_cut = !(P.flags & HIGS_FLAG_NO_XBATCH_CUT);
    unsigned long long n_eval_g = 0, n_tp = 0;

    for (;;) {
        __syncthreads();                                              // everyone is done with the previous unit's shared state
        if (threadIdx.x == 0) { S.unit = atomicAdd(&hdr->raster_cursor, 1u); S.next_tile = 0; S.active = 0; S.cut = 0; }
        __syncthreads();
        const uint32_t u = S.unit;
        if (u >= n_units) break;
        const uint32_t m = unit_mt[u];
        const uint32_t u0 = batch_offset[m];
        const uint32_t j = u - u0;
        const uint32_t seg_n = mt_count[m];
        const uint32_t start = mt_offset[m] + j * (uint32_t)P.batch_cap;
        const int len = (int)min((uint32_t)P.batch_cap, seg_n - j * (uint32_t)P.batch_cap);
        const int mtx = (int)(m % (uint32_t)P.n_mx), mty = (int)(m / (uint32_t)P.n_mx);

        // tiles wholly outside the image are never active (Alg. 1 line 11, InBounds)
        const int tiles_x = min(8, (P.W - mtx * HIGS_MT_W + HIGS_TILE - 1) / HIGS_TILE);
        const int tiles_y = min(4, (P.H - mty * HIGS_MT_H + HIGS_TILE - 1) / HIGS_TILE);

        // cross-batch saturation cut-off: product over the earlier units of the largest transmittance
        // they left in tile t bounds the transmittance in front of this unit
        if (use_cut && j > 0 && w == 0) {
            float bound = 1.0f;
            for (uint32_t jj = 0; jj < j; ++jj) {
                const float v = __ldcg(tile_maxT + (size_t)(u0 + jj) * HIGS_MT_TILES + lane);
                bound *= (v > 0.0f ? v : 1.0f);                       // 0 = not published yet
                if (__all_sync(0xffffffffu, bound < HIGS_EPS_T)) break;
            }
            const bool inb = (lane & 7) < tiles_x && (lane >> 3) < tiles_y;
            const uint32_t cut = __ballot_sync(0xffffffffu, bound < HIGS_EPS_T || !inb);
            if (lane == 0) S.cut = cut;
        }
        __syncthreads();
        const uint32_t cut = S.cut;
        if (cut == 0xffffffffu) {                                     // nothing left to see behind the earlier batches
            if (threadIdx.x == 0) unit_active[u] = 0;
            continue;
        }

        // ---- Phase 1: gather records into shared memory ----
        for (int i = threadIdx.x; i < len; i += RAS_THREADS) {
            const uint32_t id = (uint32_t)pairs[start + i];
            const float4* src = ras + 3 * (size_t)id;
            cp_async16(&S.rec[3 * i], src);
            cp_async16(&S.rec[3 * i + 1], src + 1);
            cp_async16(&S.rec[3 * i + 2], src + 2);
        }
        cp_async_wait_all();
        __syncthreads();
        // per-gaussian tile masks, transposed by ballot: masks[t][k] bit jj = gaussian k*32+jj touches tile t
        for (int k = w; k < HIGS_BATCH_CAP / 32; k += RAS_WARPS) {
            const int i = k * 32 + lane;
            uint32_t gm = 0;
            if (i < len) gm = tile_mask(S.rec[3 * i], S.rec[3 * i + 1], mtx, mty, P) & ~cut;
            uint32_t mine = 0;
#pragma unroll
            for (int t = 0; t < 32; ++t) {
                const uint32_t b = __ballot_sync(0xffffffffu, (gm >> t) & 1u);
                if (lane == t) mine = b;
            }
            S.masks[lane * MASK_PITCH + k] = mine;
        }
        __syncthreads();

        // ---- Phase 2: warps claim render tiles ----
        for (;;) {
            int t = 0;
            if (lane == 0) t = (int)atomicAdd(&S.next_tile, 1u);
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t >= HIGS_MT_TILES) break;
            const uint32_t mine = S.masks[t * MASK_PITCH + lane];      // lane k holds mini-batch k's word
            const uint32_t nonempty = __ballot_sync(0xffffffffu, mine != 0u);
            if (!nonempty) continue;
            const int tx = t & 7, ty = t >> 3;
            const float pxf = (float)(mtx * HIGS_MT_W + tx * HIGS_TILE + (lane & 7)) + 0.5f;
            const float py0 = (float)(mty * HIGS_MT_H + ty * HIGS_TILE + (lane >> 3)) + 0.5f;
            const float py1 = py0 + 4.0f;
            float T0 = 1.0f, T1 = 1.0f, r0 = 0, g0c = 0, b0c = 0, r1 = 0, g1c = 0, b1c = 0;
            uint32_t rest = nonempty;
            while (rest) {
                const int k = __ffs(rest) - 1;
                rest &= rest - 1;
                uint32_t bits = __shfl_sync(0xffffffffu, mine, k);
                if (COUNT) n_tp += __popc(bits);
                do {
                    const int i = k * 32 + __ffs(bits) - 1;
                    bits &= bits - 1;
                    const float4 a = S.rec[3 * i], bq = S.rec[3 * i + 1], cq = S.rec[3 * i + 2];
                    // N-Q, pinned: dx, u = A dx, a0 = u dx, b0 = B2 dx, t = fma(C, dy, b0), q = fma(t, dy, a0)
                    const float dx = __fsub_rn(pxf, a.x);
                    const float uu = __fmul_rn(a.z, dx);
                    const float a0 = __fmul_rn(uu, dx);
                    const float bb = __fmul_rn(a.w, dx);
                    const float dy0 = __fsub_rn(py0, a.y), dy1 = __fsub_rn(py1, a.y);
                    const float q0 = __fmaf_rn(__fmaf_rn(bq.x, dy0, bb), dy0, a0);
                    const float q1 = __fmaf_rn(__fmaf_rn(bq.x, dy1, bb), dy1, a0);
                    float al0 = fminf(HIGS_ALPHA_MAX, ex2_approx(fmaf(q0, -0.72134752f, bq.z)));
                    float al1 = fminf(HIGS_ALPHA_MAX, ex2_approx(fmaf(q1, -0.72134752f, bq.z)));
                    al0 = (q0 <= bq.y) ? al0 : 0.0f;                  // alpha < 1/255: skipped
                    al1 = (q1 <= bq.y) ? al1 : 0.0f;
                    const float w0 = T0 * al0, w1 = T1 * al1;
                    r0 = fmaf(w0, bq.w, r0); g0c = fmaf(w0, cq.x, g0c); b0c = fmaf(w0, cq.y, b0c);
                    r1 = fmaf(w1, bq.w, r1); g1c = fmaf(w1, cq.x, g1c); b1c = fmaf(w1, cq.y, b1c);
                    T0 -= w0; T1 -= w1;
                    if (COUNT) ++n_eval_g;
                } while (bits);
                if (__all_sync(0xffffffffu, T0 < HIGS_EPS_T && T1 < HIGS_EPS_T)) break;   // Alg. 2 line 8
            }
            float4* out = partial + ((size_t)u * HIGS_MT_TILES + t) * 64;
            __stcs(out + lane, make_float4(r0, g0c, b0c, T0));
            __stcs(out + 32 + lane, make_float4(r1, g1c, b1c, T1));
            float tm = fmaxf(T0, T1);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) tm = fmaxf(tm, __shfl_xor_sync(0xffffffffu, tm, d));
            if (lane == 0) {
                __stcg(tile_maxT + (size_t)u * HIGS_MT_TILES + t, fmaxf(tm, 1e-30f));
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
    const int gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int m = gw >> 5, t = gw & 31;
    if (m >= P.n_m) return;
    const int mtx = m % P.n_mx, mty = m / P.n_mx;
    const int x = mtx * HIGS_MT_W + (t & 7) * HIGS_TILE + (lane & 7);
    const int y0 = mty * HIGS_MT_H + (t >> 3) * HIGS_TILE + (lane >> 3);
    if (mtx * HIGS_MT_W + (t & 7) * HIGS_TILE >= P.W || mty * HIGS_MT_H + (t >> 3) * HIGS_TILE >= P.H) return;
    uint32_t u0 = 0, nb = 0;
    if (!hdr->overflow) { u0 = batch_offset[m]; nb = batch_offset[m + 1] - u0; }
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

static int g_raster_ctas_per_sm = 0;

int higs_raster_setup(higs_ctx* ctx)
{
    const int smem = (int)sizeof(RasSmem);
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_raster<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_raster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_raster<false>, RAS_THREADS, smem));
    g_raster_ctas_per_sm = occ > 0 ? occ : 1;
    return HIGS_OK;
}

int launch_raster(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    const int smem = (int)sizeof(RasSmem);
    const int grid = ctx->n_sm * g_raster_ctas_per_sm;
    if (P.flags & HIGS_FLAG_COUNT_EVALS)
        k_raster<true><<<grid, RAS_THREADS, smem, st>>>(ctx->pairs, ctx->ras, ctx->mt_offset, ctx->mt_count, ctx->batch_offset,
                                                        ctx->unit_mt, P, ctx->hdr, ctx->partial, ctx->unit_active, ctx->tile_maxT);
    else
        k_raster<false><<<grid, RAS_THREADS, smem, st>>>(ctx->pairs, ctx->ras, ctx->mt_offset, ctx->mt_count, ctx->batch_offset,
                                                         ctx->unit_mt, P, ctx->hdr, ctx->partial, ctx->unit_active, ctx->tile_maxT);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int launch_merge(higs_ctx* ctx, const FrameParams& P, float* out_rgb, cudaStream_t st)
{
    const int warps = P.n_m * HIGS_MT_TILES;
    k_merge_image<<<(warps + 7) / 8, 256, 0, st>>>(ctx->partial, ctx->unit_active, ctx->batch_offset, P, ctx->hdr, out_rgb);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}
