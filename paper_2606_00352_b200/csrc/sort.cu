// sort.cu -- step a5: segmented depth sort (section 3.3, section 4.4).
//
// One segment per macro-tile, items are 64-bit (depth key << 32 | gaussian slot); the required order
// is ascending (key, id) (reading Q7), i.e. ascending as unsigned 64-bit integers.  Slots are
// unique inside a segment, so all items are distinct and no stability question arises.
//   * tier cascade: segments of <= 1024 / 2048 / 4096 / 8192 items are sorted by ONE
//     CTA of 64 / 128 / 256 / 512 threads, 16 items per thread.  Where the paper runs four 8-bit radix
//     passes, this build runs a block merge sort on the whole 64-bit item: a 63-exchange Batcher network
//     in registers, then log2(threads) merge-path levels through shared memory.  It needs no tie pass for
//     equal depth keys and its cost does not depend on the key distribution.
//     The tier kernels run concurrently on forked streams (the paper overlaps them with PDL).
//   * oversize segments (PAPER.md:272-274 sorts 8192-blocks and merges them level by level): here they are
//     first split by depth into buckets of about 1.5 k items (sample sort): a strided sample of the segment
//     is sorted by one CTA and every `oversample`-th element becomes a splitter; a count pass and a scatter
//     pass move every item to its bucket in the alternate buffer; the buckets then go through the tier
//     kernels like ordinary segments and land in place.  One pass over the data instead of one per merge
//     level.  A bucket that still exceeds 8192 items (possible only for segments beyond ~0.8 M items or a
//     very unlucky sample) takes the paper's route: 8192-blocks + merge levels with merge-path partitioning.
// All sizes are read from device memory; the kernels are persistent over device work counters, so
// nothing here needs a host synchronisation.
#include <stdio.h>
#include <cooperative_groups.h>
#include "higs_internal.cuh"
#include "sort_plan.cuh"

namespace cg = cooperative_groups;
typedef unsigned long long u64;

namespace {

constexpr int IPT = 16;                                   // items per thread of the block sort

__global__ void __launch_bounds__(1024)
k_sort_plan(const uint32_t* __restrict__ seg_offset, int n_seg, SortJob* __restrict__ jobs,
            size_t max_jobs, SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr)
{
    __shared__ uint32_t s_warp[33 * 8];
    sort_plan_body(seg_offset, n_seg, false, jobs, max_jobs, split, hdr, s_warp);
}

// ---- block merge sort of up to THREADS*16 items held in shared memory ------------------------------
__device__ __forceinline__ void cex(u64& a, u64& b)
{
    const bool sw = b < a;
    const u64 lo = sw ? b : a, hi = sw ? a : b;
    a = lo; b = hi;
}

// Batcher's odd-even merge sort network for 16 items: 63 compare-exchanges, written out so that every
// index is static and the items stay in registers
__device__ __forceinline__ void reg_sort16(u64 (&v)[IPT])
{
#define X(a, b) cex(v[a], v[b]);
    X(0,1) X(2,3) X(4,5) X(6,7) X(8,9) X(10,11) X(12,13) X(14,15)
    X(0,2) X(1,3) X(4,6) X(5,7) X(8,10) X(9,11) X(12,14) X(13,15)
    X(1,2) X(5,6) X(9,10) X(13,14) X(0,4) X(1,5) X(2,6) X(3,7)
    X(8,12) X(9,13) X(10,14) X(11,15) X(2,4) X(3,5) X(10,12) X(11,13)
    X(1,2) X(3,4) X(5,6) X(9,10) X(11,12) X(13,14) X(0,8) X(1,9)
    X(2,10) X(3,11) X(4,12) X(5,13) X(6,14) X(7,15) X(4,8) X(5,9)
    X(6,10) X(7,11) X(2,4) X(3,5) X(6,8) X(7,9) X(10,12) X(11,13)
    X(1,2) X(3,4) X(5,6) X(7,8) X(9,10) X(11,12) X(13,14)
#undef X
}

// shared-memory index with one padding slot per 16 items: thread t's blocked items t*16.. start at
// t*17, so a half-warp's 64-bit accesses to "item k of each thread" fall in 16 distinct bank pairs
__device__ __forceinline__ int sidx(int i) { return i + (i >> 4); }

// Sorts buf[sidx(0 .. n_pad-1)] (n items, padded with ~0 up to a whole number of threads' worth) in place.
// Every thread of the CTA must call it; on return (after a __syncthreads) buf holds the sorted items.
template <int THREADS>
__device__ __forceinline__ void block_sort_smem(u64* buf, int n, int n_pad)
{
    const int t = threadIdx.x;
    u64 v[IPT];
    const bool live = t * IPT < n;                               // threads past the data hold nothing
    if (live) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) v[k] = buf[t * (IPT + 1) + k];
        reg_sort16(v);
    }
    // merge levels: sorted runs of `run` items -> 2*run, each live thread produces its own 16 outputs
    for (int run = IPT; run < n; run <<= 1) {
        __syncthreads();
        if (live) {
#pragma unroll
            for (int k = 0; k < IPT; ++k) buf[t * (IPT + 1) + k] = v[k];
        }
        __syncthreads();
        if (live) {
            const int o0 = t * IPT;
            const int pb = o0 & ~(2 * run - 1);                  // start of this pair of runs
            const int na = min(run, n_pad - pb), nb = max(0, min(run, n_pad - pb - run));
            const int A = pb, B = pb + run, diag = o0 - pb;
            int lo = max(0, diag - nb), hi = min(diag, na);
            while (lo < hi) {                                    // merge path: first `diag` outputs take `lo` items of A
                const int mid = (lo + hi) >> 1;
                if (buf[sidx(A + mid)] < buf[sidx(B + diag - 1 - mid)]) lo = mid + 1; else hi = mid;
            }
            int ia = lo, ib = diag - lo;
            u64 ka = ia < na ? buf[sidx(A + ia)] : ~0ull, kb = ib < nb ? buf[sidx(B + ib)] : ~0ull;
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const bool take_a = ib >= nb || (ia < na && ka < kb);
                v[k] = take_a ? ka : kb;
                if (take_a) { ++ia; ka = ia < na ? buf[sidx(A + ia)] : ~0ull; }
                else        { ++ib; kb = ib < nb ? buf[sidx(B + ib)] : ~0ull; }
            }
        }
    }
    __syncthreads();
    if (live) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) buf[t * (IPT + 1) + k] = v[k];
    }
    __syncthreads();
}

// ---- tier kernel: one CTA sorts one segment, one bucket, or one 8192-item block ---------------------
template <int THREADS>
__global__ void __launch_bounds__(THREADS)
k_block_sort(const SortJob* __restrict__ jobs, FrameHeader* __restrict__ hdr, int list, int tier,
             u64* __restrict__ pairs, u64* __restrict__ pairs_alt)
{
    constexpr int CAP = THREADS * IPT;
    extern __shared__ __align__(16) unsigned char s_raw[];
    u64* buf = reinterpret_cast<u64*>(s_raw);                     // sidx(CAP) items
    __shared__ uint32_t s_job;
    const int t = threadIdx.x;

    for (;;) {
        __syncthreads();                                         // previous job's shared state is free
        if (t == 0) s_job = atomicAdd(&hdr->sort_cursor[list][tier], 1u);
        __syncthreads();
        const uint32_t jb = s_job;
        if (jb >= hdr->n_sort_jobs[list][tier]) return;
        const SortJob job = jobs[jb];
        const int n = (int)job.len;
        const u64* gsrc = ((job.flags & 2u) ? pairs_alt : pairs) + job.start;
        const int n_pad = min(CAP, ((n + IPT - 1) / IPT) * IPT);  // whole threads
        for (int i = t; i < n_pad; i += THREADS) buf[sidx(i)] = i < n ? gsrc[i] : ~0ull;
        __syncthreads();
        block_sort_smem<THREADS>(buf, n, n_pad);
        u64* gdst = ((job.flags & 1u) ? pairs_alt : pairs) + job.start;
        for (int i = t; i < n; i += THREADS) gdst[i] = buf[sidx(i)];
    }
}

// ---- oversize segments, step 1: splitters from a sorted strided sample -------------------------------
constexpr int SPLIT_THREADS = 512;

__global__ void __launch_bounds__(SPLIT_THREADS)
k_over_split(const SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr, const u64* __restrict__ pairs,
             u64* __restrict__ splitters, uint32_t* __restrict__ bucket_count, uint32_t* __restrict__ bucket_seg)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    u64* buf = reinterpret_cast<u64*>(s_raw);
    __shared__ uint32_t s_seg;
    const int t = threadIdx.x;
    pdl_trigger();
    for (;;) {
        __syncthreads();
        if (t == 0) s_seg = atomicAdd(&hdr->split_cursor[0], 1u);
        __syncthreads();
        const uint32_t si = s_seg;
        if (si >= hdr->n_oversize) return;
        const SplitSeg sg = split[si];
        const int m = (int)(sg.oversample * sg.nb);              // sample size, <= 8192 <= len
        const int m_pad = ((m + IPT - 1) / IPT) * IPT;
        const u64* src = pairs + sg.start;
        for (int i = t; i < m_pad; i += SPLIT_THREADS)
            buf[sidx(i)] = i < m ? src[(uint32_t)(((u64)i * sg.len) / (uint32_t)m)] : ~0ull;
        __syncthreads();
        block_sort_smem<SPLIT_THREADS>(buf, m, m_pad);
        for (uint32_t b = t; b < sg.nb; b += SPLIT_THREADS) {
            if (b + 1 < sg.nb) splitters[sg.bucket_base + b] = buf[sidx((int)((b + 1) * sg.oversample))];
            bucket_count[sg.bucket_base + b] = 0;
            bucket_seg[sg.bucket_base + b] = si;
        }
    }
}

// ---- oversize segments, steps 2 and 4: bucket count and scatter ----------------------------------------
// bucket of item x = number of splitters <= x (splitters ascending, nb - 1 of them)
__device__ __forceinline__ uint32_t bucket_of(const u64* s_split, uint32_t n_split, u64 x)
{
    uint32_t lo = 0, hi = n_split;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (s_split[mid] <= x) lo = mid + 1; else hi = mid; }
    return lo;
}

constexpr int SCAT_THREADS = 512;
constexpr int SCAT_ITEMS = HIGS_SPLIT_TILE / SCAT_THREADS;

// SCATTER = false: per-bucket totals.  SCATTER = true: every tile reserves its share of each bucket with one atomic
// on the bucket cursor and writes its items there (order inside a bucket is arbitrary: the tier sort follows).
template <bool SCATTER>
__global__ void __launch_bounds__(SCAT_THREADS)
k_over_buckets(const SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr, const u64* __restrict__ pairs,
               const u64* __restrict__ splitters, uint32_t* __restrict__ bucket_count, uint32_t* __restrict__ bucket_cursor,
               u64* __restrict__ pairs_alt)
{
    __shared__ u64 s_split[HIGS_MAX_SPLIT];
    __shared__ uint32_t s_hist[HIGS_MAX_SPLIT];
    __shared__ uint32_t s_base[HIGS_MAX_SPLIT];
    __shared__ uint32_t s_tile;
    const int t = threadIdx.x;
    pdl_wait(); pdl_trigger();
    const uint32_t n_over = hdr->n_oversize, n_tiles = hdr->n_split_tiles;
    for (;;) {
        __syncthreads();
        if (t == 0) s_tile = atomicAdd(&hdr->split_cursor[SCATTER ? 2 : 1], 1u);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) return;
        int lo = 0, hi = (int)n_over - 1;                         // last segment with tile_base <= tile
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (split[mid].tile_base <= tile) lo = mid; else hi = mid - 1; }
        const SplitSeg sg = split[lo];
        for (uint32_t b = t; b < sg.nb; b += SCAT_THREADS) {
            if (b + 1 < sg.nb) s_split[b] = splitters[sg.bucket_base + b];
            s_hist[b] = 0;
        }
        __syncthreads();
        const uint32_t o0 = (tile - sg.tile_base) * HIGS_SPLIT_TILE;
        const u64* src = pairs + sg.start;
        u64 x[SCAT_ITEMS]; uint32_t bk[SCAT_ITEMS], rk[SCAT_ITEMS];
#pragma unroll
        for (int k = 0; k < SCAT_ITEMS; ++k) {
            const uint32_t i = o0 + k * SCAT_THREADS + t;
            x[k] = i < sg.len ? src[i] : 0ull;
        }
#pragma unroll
        for (int k = 0; k < SCAT_ITEMS; ++k) {
            const uint32_t i = o0 + k * SCAT_THREADS + t;
            bk[k] = 0; rk[k] = 0;
            if (i < sg.len) {
                bk[k] = bucket_of(s_split, sg.nb - 1, x[k]);
                rk[k] = atomicAdd(&s_hist[bk[k]], 1u);
            }
        }
        __syncthreads();
        for (uint32_t b = t; b < sg.nb; b += SCAT_THREADS) {
            const uint32_t h = s_hist[b];
            if (h) {
                if (SCATTER) s_base[b] = atomicAdd(&bucket_cursor[sg.bucket_base + b], h);
                else atomicAdd(&bucket_count[sg.bucket_base + b], h);
            }
        }
        if (SCATTER) {
            __syncthreads();
#pragma unroll
            for (int k = 0; k < SCAT_ITEMS; ++k) {
                const uint32_t i = o0 + k * SCAT_THREADS + t;
                if (i < sg.len) pairs_alt[s_base[bk[k]] + rk[k]] = x[k];
            }
        }
    }
}

// ---- plan B: buckets -> tier job lists (list 1), scatter cursors, fallback merge plan -------------------
__global__ void __launch_bounds__(1024)
k_bucket_plan(const SplitSeg* __restrict__ split, const uint32_t* __restrict__ bucket_count, const uint32_t* __restrict__ bucket_seg,
              uint32_t* __restrict__ bucket_cursor, SortJob* __restrict__ jobs /* list 1 */, size_t max_jobs,
              OverSeg* __restrict__ over, FrameHeader* __restrict__ hdr)
{
    __shared__ uint32_t s_warp[33 * 7];
    __shared__ uint32_t s_maxlev;
    pdl_wait(); pdl_trigger();
    if (threadIdx.x == 0) s_maxlev = 0;
    __syncthreads();
    const uint32_t n_buckets = hdr->n_buckets;
    uint32_t carry[7] = {0, 0, 0, 0, 0, 0, 0};          // tiers 0-3 (3 counts fallback blocks too), fallback buckets, merge tiles, items
    for (uint32_t b0 = 0; b0 < n_buckets; b0 += 1024) {
        const uint32_t b = b0 + threadIdx.x;
        uint32_t n = 0, seg_start = 0, seg_before = 0;
        if (b < n_buckets) {
            n = bucket_count[b];
            const SplitSeg sg = split[bucket_seg[b]];
            seg_start = sg.start; seg_before = sg.items_before;
        }
        uint32_t v[7] = {0, 0, 0, 0, 0, 0, n};
        const bool fall = n > HIGS_SORT_BLOCK;
        const int t = n >= 1 ? (fall ? 3 : tier_of(n)) : -1;     // a one-item bucket still has to travel back from the alternate buffer
        uint32_t nc = 0, levels = 0;
        if (fall) {
            nc = (n + HIGS_SORT_BLOCK - 1) / HIGS_SORT_BLOCK;
            levels = 32 - __clz(nc - 1);
            v[3] = nc; v[4] = 1; v[5] = (n + HIGS_MERGE_TILE - 1) / HIGS_MERGE_TILE;
            atomicMax(&s_maxlev, levels);
        } else if (t >= 0) v[t] = 1;
        plan_scan<7>(v, carry, s_warp);
        if (b < n_buckets) {
            const uint32_t start = seg_start + (v[6] - seg_before);   // buckets of a segment are consecutive, in depth order
            bucket_cursor[b] = start;
            if (fall) {
                for (uint32_t c = 0; c < nc; ++c) {
                    const uint32_t cs = c * HIGS_SORT_BLOCK;
                    jobs[(size_t)3 * max_jobs + v[3] + c] = SortJob{start + cs, min((uint32_t)HIGS_SORT_BLOCK, n - cs), 2u | (levels & 1u), 0u};
                }
                over[v[4]] = OverSeg{start, n, levels, v[5]};
            } else if (t >= 0) {
                jobs[(size_t)t * max_jobs + v[t]] = SortJob{start, n, 2u, 0u};
            }
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int t = 0; t < HIGS_N_TIERS; ++t) hdr->n_sort_jobs[1][t] = carry[t];
        hdr->n_fallback = carry[4];
        hdr->n_merge_tiles = carry[5];
        hdr->max_levels = s_maxlev;
    }
}

// ---- fallback path: level-by-level merge of the sorted 8192-item blocks of a bucket that stayed too large ----
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

// The same search done by one warp on global memory, 32 probes per step instead of one.  The predicate
// A[mid] < B[diag-1-mid] is monotone in mid (true ... true false ... false); the answer is the first false.
__device__ __forceinline__ int merge_path_warp(const u64* A, int na, const u64* B, int nb, int diag, int lane)
{
    int lo = max(0, diag - nb), hi = min(diag, na);              // answer in [lo, hi]
    while (lo < hi) {
        const int step = (hi - lo + 31) >> 5;
        const int mid = min(hi - 1, lo + step * (lane + 1) - 1); // lane 31 always probes hi-1
        const uint32_t bal = __ballot_sync(0xffffffffu, A[mid] < B[diag - 1 - mid]);
        const int ff = bal == 0xffffffffu ? 32 : __ffs(~bal) - 1;   // first probe that answered false
        const int new_lo = ff == 0 ? lo : min(hi - 1, lo + step * ff - 1) + 1;
        const int new_hi = ff == 32 ? hi : min(hi - 1, lo + step * (ff + 1) - 1);
        lo = new_lo; hi = new_hi;
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
    const uint32_t n_tiles = hdr->n_merge_tiles, n_over = hdr->n_fallback, max_levels = hdr->max_levels;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (uint32_t lev = 0; lev < max_levels; ++lev) {
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            int lo = 0, hi = (int)n_over - 1;                     // last bucket with tile_base <= tile
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
            if (wid < 2) {                                        // warp 0: tile start, warp 1: tile end
                const int diag = (int)((wid == 0 ? o0 : o1) - ps);
                const int a = merge_path_warp(A, na, B, nb, diag, lane);
                if (lane == 0) s_part[wid] = a;
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

template <int THREADS>
constexpr size_t sort_smem() { return (size_t)(THREADS * IPT + THREADS) * sizeof(u64); }

template <int THREADS>
int launch_tier(higs_ctx* ctx, int list, int tier, u64* pairs, cudaStream_t st)
{
    const int ctas = ctx->n_sm * ctx->tier_ctas_per_sm[tier];
    k_block_sort<THREADS><<<ctas, THREADS, sort_smem<THREADS>(), st>>>(
        ctx->sort_jobs + (size_t)(list * HIGS_N_TIERS + tier) * ctx->max_jobs, ctx->hdr, list, tier, pairs, ctx->pairs_alt);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

template <int THREADS>
int setup_tier(higs_ctx* ctx, int tier)
{
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<THREADS>()));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_block_sort<THREADS>, THREADS, sort_smem<THREADS>()));
    ctx->tier_ctas_per_sm[tier] = occ < 1 ? 1 : occ;
    return HIGS_OK;
}

int run_sort(higs_ctx* ctx, u64* pairs, const uint32_t* seg_offset, int n_seg, bool plan_done, cudaStream_t st)
{
    SortJob* jobs0 = ctx->sort_jobs;
    SortJob* jobs1 = ctx->sort_jobs + (size_t)HIGS_N_TIERS * ctx->max_jobs;
    u64* alt = ctx->pairs_alt;
    int rc;
    if (!plan_done) {                                             // inside a frame k_plan has already done this (binning.cu)
        k_sort_plan<<<1, 1024, 0, st>>>(seg_offset, n_seg, jobs0, (size_t)ctx->max_jobs, ctx->split_segs, ctx->hdr);
        HIGS_LAUNCHED(ctx);
    }
    // fork: whole segments go through the tier kernels on side streams (the paper overlaps tiers with PDL)
    // while the main stream splits the oversize segments into buckets
    HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_fork, st));
    for (int k = 0; k < 4; ++k) HIGS_CUDA(ctx, cudaStreamWaitEvent(ctx->aux_stream[k], ctx->ev_fork, 0));
    if ((rc = launch_tier<512>(ctx, 0, 3, pairs, ctx->aux_stream[0]))) return rc;
    if ((rc = launch_tier<256>(ctx, 0, 2, pairs, ctx->aux_stream[1]))) return rc;
    if ((rc = launch_tier<128>(ctx, 0, 1, pairs, ctx->aux_stream[2]))) return rc;
    if ((rc = launch_tier<64>(ctx, 0, 0, pairs, ctx->aux_stream[3]))) return rc;
    k_over_split<<<ctx->n_sm, SPLIT_THREADS, sort_smem<SPLIT_THREADS>(), st>>>(ctx->split_segs, ctx->hdr, pairs, ctx->splitters,
                                                                              ctx->bucket_count, ctx->bucket_seg);
    HIGS_LAUNCHED(ctx);
    HIGS_CUDA(ctx, launch_pdl(k_over_buckets<false>, dim3(ctx->n_sm * 2), dim3(SCAT_THREADS), 0, st, ctx->split_segs, ctx->hdr, pairs,
                              ctx->splitters, ctx->bucket_count, ctx->bucket_cursor, alt));
    HIGS_LAUNCHED(ctx);
    HIGS_CUDA(ctx, launch_pdl(k_bucket_plan, dim3(1), dim3(1024), 0, st, ctx->split_segs, ctx->bucket_count, ctx->bucket_seg, ctx->bucket_cursor,
                              jobs1, (size_t)ctx->max_jobs, ctx->over_segs, ctx->hdr));
    HIGS_LAUNCHED(ctx);
    HIGS_CUDA(ctx, launch_pdl(k_over_buckets<true>, dim3(ctx->n_sm * 2), dim3(SCAT_THREADS), 0, st, ctx->split_segs, ctx->hdr, pairs,
                              ctx->splitters, ctx->bucket_count, ctx->bucket_cursor, alt));
    HIGS_LAUNCHED(ctx);
    HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_fork2, st));
    for (int k = 1; k < 4; ++k) HIGS_CUDA(ctx, cudaStreamWaitEvent(ctx->aux_stream[k], ctx->ev_fork2, 0));
    if ((rc = launch_tier<512>(ctx, 1, 3, pairs, st))) return rc;
    if ((rc = launch_tier<256>(ctx, 1, 2, pairs, ctx->aux_stream[1]))) return rc;
    if ((rc = launch_tier<128>(ctx, 1, 1, pairs, ctx->aux_stream[2]))) return rc;
    if ((rc = launch_tier<64>(ctx, 1, 0, pairs, ctx->aux_stream[3]))) return rc;
    const OverSeg* over = ctx->over_segs; const FrameHeader* hdr = ctx->hdr;
    void* args[] = { (void*)&over, (void*)&hdr, (void*)&pairs, (void*)&alt };
    HIGS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)k_merge_levels, dim3(ctx->n_sm * ctx->merge_ctas_per_sm), dim3(MERGE_THREADS), args, 0, st));
    ++ctx->n_launches;
    for (int k = 0; k < 4; ++k) {
        HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_join[k], ctx->aux_stream[k]));
        HIGS_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_join[k], 0));
    }
    return HIGS_OK;
}

} // namespace

int higs_sort_smem_setup(higs_ctx* ctx)
{
    int rc;
    if ((rc = setup_tier<64>(ctx, 0))) return rc;
    if ((rc = setup_tier<128>(ctx, 1))) return rc;
    if ((rc = setup_tier<256>(ctx, 2))) return rc;
    if ((rc = setup_tier<512>(ctx, 3))) return rc;
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_over_split, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<SPLIT_THREADS>()));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_merge_levels, MERGE_THREADS, 0));
    ctx->merge_ctas_per_sm = occ < 1 ? 1 : (occ > 2 ? 2 : occ);
    return HIGS_OK;
}

int launch_sort(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    return run_sort(ctx, ctx->pairs, ctx->mt_offset, P.n_m, true, st);
}

int launch_sort_only(higs_ctx* ctx, unsigned long long* pairs, const uint32_t* seg_offset, int n_seg, cudaStream_t st)
{
    return run_sort(ctx, pairs, seg_offset, n_seg, false, st);
}
