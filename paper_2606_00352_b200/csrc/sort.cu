// sort.cu -- step a5: segmented depth sort (section 3.3, section 4.4).
//
// One segment per macro-tile, items are 64-bit (depth key << 32 | gaussian id); the required order
// is ascending (key, id) (reading Q7), i.e. ascending as unsigned 64-bit integers.
//   * tier cascade: segments of <= 1024 / 2048 / 4096 / 8192 items are sorted by ONE CTA in shared
//     memory (CTA 128 / 256 / 512 / 1024 threads), four stable 8-bit LSD radix passes on the depth
//     key, passes whose digit is constant over the segment are skipped, then
//     equal-key runs (rare) are put in id order by an odd-even transposition confined to the run;
//   * overflow path: longer segments are cut into 8192-item blocks sorted by the top tier, then
//     merged level by level (run size doubling) with merge-path partitioning.
// All sizes are read from device memory; the kernels are persistent over device work counters, so
// nothing here needs a host synchronisation.
#include <stdio.h>
#include <cooperative_groups.h>
#include "higs_internal.cuh"

namespace cg = cooperative_groups;
typedef unsigned long long u64;

namespace {

__device__ __forceinline__ int tier_of(uint32_t n) { return n <= 1024u ? 0 : (n <= 2048u ? 1 : (n <= 4096u ? 2 : 3)); }

// ---- sort plan: job lists per tier + merge plan for oversize segments -------------------------
template <int NV>
__device__ __forceinline__ void plan_scan(uint32_t (&v)[NV], uint32_t (&carry)[NV], uint32_t* s_warp)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t incl[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        uint32_t x = v[q];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
        incl[q] = x;
        if (lane == 31) s_warp[wid * NV + q] = x;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const uint32_t x = s_warp[lane * NV + q];
            uint32_t t = x;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, t, d); if (lane >= d) t += y; }
            s_warp[lane * NV + q] = t - x;
            if (lane == 31) s_warp[32 * NV + q] = t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        const uint32_t excl = carry[q] + s_warp[wid * NV + q] + incl[q] - v[q];
        carry[q] += s_warp[32 * NV + q];
        v[q] = excl;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(1024)
k_sort_plan(const uint32_t* __restrict__ seg_offset, int n_seg, int honour_overflow, SortJob* __restrict__ jobs,
            size_t max_jobs, OverSeg* __restrict__ over, FrameHeader* __restrict__ hdr)
{
    __shared__ uint32_t s_warp[33 * 6];
    __shared__ uint32_t s_maxlev;
    if (threadIdx.x == 0) s_maxlev = 0;
    const bool dead = honour_overflow && hdr->overflow;
    uint32_t carry[6] = {0, 0, 0, 0, 0, 0};
    __syncthreads();
    for (int s0 = 0; s0 < n_seg; s0 += 1024) {
        const int s = s0 + threadIdx.x;
        uint32_t start = 0, n = 0;
        if (s < n_seg && !dead) { start = seg_offset[s]; n = seg_offset[s + 1] - start; }
        uint32_t v[6] = {0, 0, 0, 0, 0, 0};
        uint32_t nc = 0, levels = 0;
        if (n > 1) {
            if (n <= HIGS_SORT_BLOCK) v[tier_of(n)] = 1;
            else {
                nc = (n + HIGS_SORT_BLOCK - 1) / HIGS_SORT_BLOCK;
                levels = 32 - __clz(nc - 1);
                v[3] = nc; v[4] = 1; v[5] = (n + HIGS_MERGE_TILE - 1) / HIGS_MERGE_TILE;
                atomicMax(&s_maxlev, levels);
            }
        }
        const uint32_t cnt3 = v[3], tiles = v[5];
        const int t = n > 1 ? (n <= HIGS_SORT_BLOCK ? tier_of(n) : 3) : -1;
        plan_scan<6>(v, carry, s_warp);
        if (t >= 0) {
            if (nc == 0) {
                jobs[(size_t)t * max_jobs + v[t]] = SortJob{start, n, 0u, 0u};
            } else {
                for (uint32_t c = 0; c < cnt3; ++c) {
                    const uint32_t cs = c * HIGS_SORT_BLOCK;
                    jobs[(size_t)3 * max_jobs + v[3] + c] = SortJob{start + cs, min((uint32_t)HIGS_SORT_BLOCK, n - cs), levels & 1u, 0u};
                }
                over[v[4]] = OverSeg{start, n, levels, v[5]};
                (void)tiles;
            }
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int t = 0; t < HIGS_N_TIERS; ++t) { hdr->n_sort_jobs[t] = carry[t]; hdr->sort_cursor[t] = 0; }
        hdr->n_oversize = carry[4];
        hdr->n_merge_tiles = carry[5];
        hdr->max_levels = s_maxlev;
    }
}

// ---- tier kernel: one CTA sorts one segment (or one 8192-item block) in shared memory ---------
template <int CAP, int THREADS>
__global__ void __launch_bounds__(THREADS)
k_block_sort(const SortJob* __restrict__ jobs, FrameHeader* __restrict__ hdr, int tier,
             u64* __restrict__ pairs, u64* __restrict__ pairs_alt)
{
    constexpr int NW = THREADS / 32;
    extern __shared__ __align__(16) unsigned char s_raw[];
    u64* buf0 = reinterpret_cast<u64*>(s_raw);
    u64* buf1 = buf0 + CAP;
    uint32_t* cnt = reinterpret_cast<uint32_t*>(buf1 + CAP);      // [NW][256]
    uint32_t* dbase = cnt + NW * 256;                             // [256] exclusive digit bases
    __shared__ uint32_t s_job;
    __shared__ int s_skip;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;

    for (;;) {
        if (threadIdx.x == 0) s_job = atomicAdd(&hdr->sort_cursor[tier], 1u);
        __syncthreads();
        const uint32_t jb = s_job;
        if (jb >= hdr->n_sort_jobs[tier]) return;
        const SortJob job = jobs[jb];
        const int n = (int)job.len;
        u64* gsrc = pairs + job.start;
        for (int i = threadIdx.x; i < n; i += THREADS) buf0[i] = gsrc[i];
        u64* src = buf0; u64* dst = buf1;
        const int per = (((n + NW - 1) / NW) + 31) & ~31;         // contiguous chunk per warp, multiple of 32
        const int beg = min(n, w * per), end = min(n, beg + per);

        for (int pass = 0; pass < 4; ++pass) {
            const int shift = 32 + 8 * pass;
            for (int i = threadIdx.x; i < NW * 256; i += THREADS) cnt[i] = 0;
            __syncthreads();                                     // also covers the load of buf0
            for (int v = beg + lane; v < end; v += 32)
                atomicAdd(&cnt[w * 256 + (int)((src[v] >> shift) & 255u)], 1u);
            __syncthreads();
            for (int d = threadIdx.x; d < 256; d += THREADS) {    // per digit: exclusive scan over warps
                uint32_t run = 0;
#pragma unroll
                for (int ww = 0; ww < NW; ++ww) { const uint32_t t = cnt[ww * 256 + d]; cnt[ww * 256 + d] = run; run += t; }
                dbase[d] = run;
            }
            __syncthreads();
            if (w == 0) {                                        // exclusive scan over the 256 digit totals
                uint32_t t[8], sum = 0; bool full = false;
#pragma unroll
                for (int k = 0; k < 8; ++k) { t[k] = dbase[lane * 8 + k]; full |= (t[k] == (uint32_t)n); sum += t[k]; }
                uint32_t x = sum;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
                uint32_t run = x - sum;
#pragma unroll
                for (int k = 0; k < 8; ++k) { dbase[lane * 8 + k] = run; run += t[k]; }
                const bool any_full = __any_sync(0xffffffffu, full);
                if (lane == 0) s_skip = any_full ? 1 : 0;
            }
            __syncthreads();
            if (s_skip) continue;                                // digit constant over the segment: nothing moves
            for (int vb = beg; vb < end; vb += 32) {             // stable scatter, warp walks its chunk in order
                const int v = vb + lane;
                const bool act = v < end;
                const u64 item = act ? src[v] : 0ull;
                const uint32_t d = act ? (uint32_t)((item >> shift) & 255u) : (256u + (uint32_t)lane);
                const uint32_t peers = __match_any_sync(0xffffffffu, d);
                const uint32_t rank = __popc(peers & lt_mask);
                uint32_t pos = 0;
                if (act) pos = cnt[w * 256 + d] + dbase[d] + rank;
                __syncwarp();
                if (act && rank == 0) cnt[w * 256 + d] += __popc(peers);
                __syncwarp();
                if (act) dst[pos] = item;
            }
            __syncthreads();
            u64* tmp = src; src = dst; dst = tmp;
        }
        // equal depth keys: order by id (odd-even transposition confined to equal-key neighbours)
        for (;;) {
            int swapped = 0;
#pragma unroll
            for (int phase = 0; phase < 2; ++phase) {
                for (int i = 2 * threadIdx.x + phase; i + 1 < n; i += 2 * THREADS) {
                    const u64 a = src[i], b = src[i + 1];
                    if ((a >> 32) == (b >> 32) && a > b) { src[i] = b; src[i + 1] = a; swapped = 1; }
                }
                __syncthreads();
            }
            if (!__syncthreads_or(swapped)) break;
        }
        u64* gdst = (job.dst_alt ? pairs_alt : pairs) + job.start;
        for (int i = threadIdx.x; i < n; i += THREADS) gdst[i] = src[i];
        __syncthreads();
    }
}

// ---- overflow path: level-by-level merge of the sorted 8192-item blocks ------------------------
// smallest a with: merging the first `diag` outputs takes a items from A (and diag - a from B)
__device__ __forceinline__ int merge_path(const u64* A, int na, const u64* B, int nb, int diag)
{
    int lo = max(0, diag - nb), hi = min(diag, na);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (A[mid] < B[diag - 1 - mid]) lo = mid + 1; else hi = mid;
    }
    return lo;
}

constexpr int MERGE_THREADS = 512;
constexpr int MERGE_ITEMS = HIGS_MERGE_TILE / MERGE_THREADS;

__global__ void __launch_bounds__(MERGE_THREADS)
k_merge_levels(const OverSeg* __restrict__ over, const FrameHeader* __restrict__ hdr, u64* __restrict__ pairs, u64* __restrict__ pairs_alt)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ u64 s_in[HIGS_MERGE_TILE];
    __shared__ int s_part[4];
    const uint32_t n_tiles = hdr->n_merge_tiles, n_over = hdr->n_oversize, max_levels = hdr->max_levels;
    for (uint32_t lev = 0; lev < max_levels; ++lev) {
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            int lo = 0, hi = (int)n_over - 1;                     // last segment with tile_base <= tile
            while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (over[mid].tile_base <= tile) lo = mid; else hi = mid - 1; }
            const OverSeg sg = over[lo];
            if (lev >= sg.levels) continue;                       // uniform per CTA
            const bool from_main = ((sg.levels - lev) & 1u) == 0u;
            const u64* src = (from_main ? pairs : pairs_alt) + sg.start;
            u64* dst = (from_main ? pairs_alt : pairs) + sg.start;
            const uint32_t run = (uint32_t)HIGS_SORT_BLOCK << lev;
            const uint32_t o0 = (tile - sg.tile_base) * HIGS_MERGE_TILE, o1 = min(sg.len, o0 + HIGS_MERGE_TILE);
            const uint32_t ps = (o0 / (2u * run)) * (2u * run);
            const uint32_t a_beg = ps, a_end = min(sg.len, ps + run), b_end = min(sg.len, ps + 2u * run);
            const u64* A = src + a_beg; const int na = (int)(a_end - a_beg);
            const u64* B = src + a_end; const int nb = (int)(b_end - a_end);
            if (threadIdx.x < 2) {
                const int diag = (int)((threadIdx.x == 0 ? o0 : o1) - ps);
                s_part[threadIdx.x] = merge_path(A, na, B, nb, diag);
            }
            __syncthreads();
            const int a0 = s_part[0], a1 = s_part[1];
            const int b0 = (int)(o0 - ps) - a0, b1 = (int)(o1 - ps) - a1;
            const int ca = a1 - a0, cb = b1 - b0, tot = ca + cb;
            for (int i = threadIdx.x; i < tot; i += MERGE_THREADS) s_in[i] = i < ca ? A[a0 + i] : B[b0 + (i - ca)];
            __syncthreads();
            const u64* SA = s_in; const u64* SB = s_in + ca;
            const int d0 = min(tot, (int)threadIdx.x * MERGE_ITEMS);
            int ia = merge_path(SA, ca, SB, cb, d0), ib = d0 - ia;
            u64 outv[MERGE_ITEMS];
#pragma unroll
            for (int k = 0; k < MERGE_ITEMS; ++k) {
                const bool has_a = ia < ca, has_b = ib < cb;
                const u64 va = has_a ? SA[ia] : ~0ull, vb = has_b ? SB[ib] : ~0ull;
                const bool take_a = has_a && (!has_b || va < vb);
                outv[k] = take_a ? va : vb;
                ia += take_a ? 1 : 0; ib += take_a ? 0 : 1;
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < MERGE_ITEMS; ++k) if (d0 + k < tot) s_in[d0 + k] = outv[k];
            __syncthreads();
            for (int i = threadIdx.x; i < tot; i += MERGE_THREADS) dst[o0 + i] = s_in[i];
            __syncthreads();
        }
        grid.sync();
    }
}

int g_merge_ctas_per_sm = 1;

template <int CAP, int THREADS>
constexpr size_t sort_smem() { return (size_t)CAP * 16 + (size_t)(THREADS / 32) * 256 * 4 + 256 * 4; }

template <int CAP, int THREADS>
int launch_tier(higs_ctx* ctx, int tier, int ctas, u64* pairs, cudaStream_t st)
{
    k_block_sort<CAP, THREADS><<<ctas, THREADS, sort_smem<CAP, THREADS>(), st>>>(
        ctx->sort_jobs + (size_t)tier * ctx->max_jobs, ctx->hdr, tier, pairs, ctx->pairs_alt);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int run_sort(higs_ctx* ctx, u64* pairs, const uint32_t* seg_offset, int n_seg, int honour_overflow, cudaStream_t st)
{
    k_sort_plan<<<1, 1024, 0, st>>>(seg_offset, n_seg, honour_overflow, ctx->sort_jobs, (size_t)ctx->max_jobs, ctx->over_segs, ctx->hdr);
    HIGS_LAUNCHED(ctx);
    int rc;
    if ((rc = launch_tier<1024, 128>(ctx, 0, ctx->n_sm * 8, pairs, st))) return rc;
    if ((rc = launch_tier<2048, 256>(ctx, 1, ctx->n_sm * 4, pairs, st))) return rc;
    if ((rc = launch_tier<4096, 512>(ctx, 2, ctx->n_sm * 2, pairs, st))) return rc;
    if ((rc = launch_tier<8192, 1024>(ctx, 3, ctx->n_sm, pairs, st))) return rc;
    const OverSeg* over = ctx->over_segs; const FrameHeader* hdr = ctx->hdr; u64* alt = ctx->pairs_alt;
    void* args[] = { (void*)&over, (void*)&hdr, (void*)&pairs, (void*)&alt };
    HIGS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)k_merge_levels, dim3(ctx->n_sm * g_merge_ctas_per_sm), dim3(MERGE_THREADS), args, 0, st));
    ++ctx->n_launches;
    return HIGS_OK;
}

} // namespace

int higs_sort_smem_setup(higs_ctx* ctx)
{
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<1024, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<1024, 128>()));
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<2048, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<2048, 256>()));
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<4096, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<4096, 512>()));
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<8192, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<8192, 1024>()));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_merge_levels, MERGE_THREADS, 0));
    g_merge_ctas_per_sm = occ < 1 ? 1 : (occ > 2 ? 2 : occ);
    return HIGS_OK;
}

int launch_sort(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    return run_sort(ctx, ctx->pairs, ctx->mt_offset, P.n_m, 1, st);
}

int launch_sort_only(higs_ctx* ctx, unsigned long long* pairs, const uint32_t* seg_offset, int n_seg, cudaStream_t st)
{
    return run_sort(ctx, pairs, seg_offset, n_seg, 0, st);
}
