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
// Compare-exchange.  Written as `sw ? b : a, sw ? a : b` on 64-bit values, the compiler (and ptxas again from selp.b64) takes the
// second select for a maximum and computes a second predicate for it: 4 ISETP + 4 SEL.  One 64-bit compare and four 32-bit
// selects on the halves stay as written: 2 ISETP + 4 SEL, a quarter fewer ALU-pipe instructions in the networks that bound
// these kernels.
__device__ __forceinline__ void cex(u64& a, u64& b)
{
    const uint32_t al = (uint32_t)a, ah = (uint32_t)(a >> 32), bl = (uint32_t)b, bh = (uint32_t)(b >> 32);
    uint32_t l0, l1, h0, h1;
    asm("{\n\t.reg .pred p;\n\t.reg .b64 x, y;\n\tmov.b64 x, {%4, %5};\n\tmov.b64 y, {%6, %7};\n\tsetp.lt.u64 p, y, x;\n\t"
        "selp.b32 %0, %6, %4, p;\n\tselp.b32 %1, %7, %5, p;\n\tselp.b32 %2, %4, %6, p;\n\tselp.b32 %3, %5, %7, p;\n\t}"
        : "=r"(l0), "=r"(l1), "=r"(h0), "=r"(h1) : "r"(al), "r"(ah), "r"(bl), "r"(bh));
    a = ((u64)l1 << 32) | l0; b = ((u64)h1 << 32) | h0;
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
    int* s_split = reinterpret_cast<int*>(buf + (THREADS * IPT + THREADS + 2));      // [THREADS + 1] merge-path splits of the threads
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
            s_split[t] = lo;
        }
        __syncthreads();
        if (live) {
            // This thread's 16 outputs are the merge of A[ia .. ia+ca) and B[ib .. ib+cb), ca + cb = 16, where ia + ca is the
            // next thread's split (or the end of A when the next thread starts another pair of runs).  Loaded as A ascending
            // followed by B descending they form a bitonic sequence: a 32-exchange bitonic merge network with static register
            // indices sorts them - no data-dependent loads, no pointer bookkeeping (a two-pointer merge was 25 instructions
            // per output, most of them on the ALU pipe that bounds this kernel).
            const int o0 = t * IPT;
            const int pb = o0 & ~(2 * run - 1);
            const int na = min(run, n_pad - pb), nb = max(0, min(run, n_pad - pb - run));
            const int A = pb, B = pb + run, diag = o0 - pb;
            const int ia = s_split[t], ib = diag - ia;
            const bool last = diag + IPT >= na + nb;             // the next thread belongs to another pair (or there is none)
            const int ca = (last ? na : s_split[t + 1]) - ia;
            const int pa = A + ia, pbd = B + ib + (IPT - 1);
#pragma unroll
            for (int k = 0; k < IPT; ++k) v[k] = buf[sidx(k < ca ? pa + k : pbd - k)];
#define X(a, b) cex(v[a], v[b]);
            X(0,8) X(1,9) X(2,10) X(3,11) X(4,12) X(5,13) X(6,14) X(7,15)
            X(0,4) X(1,5) X(2,6) X(3,7) X(8,12) X(9,13) X(10,14) X(11,15)
            X(0,2) X(1,3) X(4,6) X(5,7) X(8,10) X(9,11) X(12,14) X(13,15)
            X(0,1) X(2,3) X(4,5) X(6,7) X(8,9) X(10,11) X(12,13) X(14,15)
#undef X
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
        HIGS_ASSERT(n >= 1 && n <= CAP);
        const u64* gsrc = ((job.flags & 2u) ? pairs_alt : pairs) + job.start;
        const int n_pad = min(CAP, ((n + IPT - 1) / IPT) * IPT);  // whole threads
        for (int i = t; i < n_pad; i += THREADS) buf[sidx(i)] = i < n ? gsrc[i] : ~0ull;
        __syncthreads();
        block_sort_smem<THREADS>(buf, n, n_pad);
        u64* gdst = ((job.flags & 1u) ? pairs_alt : pairs) + job.start;
        for (int i = t; i < n; i += THREADS) gdst[i] = buf[sidx(i)];
    }
}

// ---- block radix sort ("4 x 8-bit radix passes") ------------------------------------------
// LSD passes of 8 bits over the bits of the depth key that actually vary inside the job (depth inside one
// macro-tile spans a narrow range: the top bits are common, typically 3 passes instead of 4).  Ranking is
// warp-private: a warp owns a contiguous chunk of the items and walks it 32 at a time; match.any finds the lanes
// with the same digit, the lowest of them bumps the warp's counter of that digit, so an item's rank inside
// (warp, digit) follows item order and the pass is stable.  A column scan over the NW x 256 counters gives the
// global bases.  Required order is the whole 64-bit item (key, slot) (reading Q7): equal keys are rare,
// so after the key passes runs of two equal keys are fixed by one compare-exchange; a job with a longer run of
// equal keys (duplicate depths) is sorted again, stably, by the varying bits of the slot and then by the key.
template <int THREADS, int IPT>
struct RadixLayout {
    static constexpr int NW = THREADS / 32;
    static constexpr int CAP = THREADS * IPT;
    static constexpr int G = THREADS >= 256 ? THREADS / 256 : 1;   // thread groups of the column scan
    static constexpr size_t bytes = sizeof(u64) * CAP + sizeof(uint32_t) * (NW * 256 + 256 + G * 256 + 4 * NW + 4);
    u64* buf; uint32_t* cnt; uint32_t* tot; uint32_t* grp; uint32_t* red;
    __device__ explicit RadixLayout(unsigned char* raw)
    {
        buf = reinterpret_cast<u64*>(raw);
        cnt = reinterpret_cast<uint32_t*>(buf + CAP);
        tot = cnt + NW * 256;
        grp = tot + 256;
        red = grp + G * 256;
    }
};

// one stable counting pass on digit (x >> shift) & 255 of the n items in L.buf; cpw = items per warp chunk (multiple of 32)
template <int THREADS, int IPT>
__device__ __forceinline__ void radix_pass(const RadixLayout<THREADS, IPT>& L, int n, int cpw, int shift)
{
    constexpr int NW = THREADS / 32;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    for (int i = t; i < NW * 256; i += THREADS) L.cnt[i] = 0;
    __syncthreads();
    const int wbeg = w * cpw, wend = min(n, wbeg + cpw);
    uint32_t* my_cnt = L.cnt + w * 256;
    const int kpw = cpw >> 5;                                        // items per lane (warp-uniform)
    u64 x[IPT];
    uint32_t off[IPT];                                               // first the peer mask, then the rank inside (warp, digit)
#pragma unroll
    for (int k = 0; k < IPT; ++k) {                                  // the matches of a chunk are independent: issued back to back
        if (k < kpw) {
            const int i = wbeg + k * 32 + lane;
            x[k] = i < wend ? L.buf[i] : ~0ull;
            const uint32_t dgt = i < wend ? (uint32_t)(x[k] >> shift) & 255u : 256u + (uint32_t)lane;
            off[k] = __match_any_sync(0xffffffffu, dgt);
        }
    }
#pragma unroll
    for (int k = 0; k < IPT; ++k) {                                  // in item order: the lowest lane of a digit bumps the warp's counter
        if (k < kpw) {
            const uint32_t peers = off[k];
            const int leader = __ffs(peers) - 1;
            const uint32_t dgt = (uint32_t)(x[k] >> shift) & 255u;
            uint32_t old = 0;
            if (lane == leader && wbeg + k * 32 + lane < wend) { old = my_cnt[dgt]; my_cnt[dgt] = old + __popc(peers); }
            old = __shfl_sync(0xffffffffu, old, leader);
            off[k] = old + __popc(peers & lt);
            __syncwarp();
        }
    }
    __syncthreads();
    if constexpr (THREADS >= 256) {                                  // per digit: exclusive prefix over the warps, 8 warps per thread
        constexpr int G = THREADS / 256;
        const int d = t & 255, g = t >> 8;
        uint32_t c[8], run = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) c[q] = L.cnt[(g * 8 + q) * 256 + d];
#pragma unroll
        for (int q = 0; q < 8; ++q) { const uint32_t v = c[q]; c[q] = run; run += v; }
        if (G > 1) { L.grp[g * 256 + d] = run; __syncthreads(); }
        uint32_t base = 0;
#pragma unroll
        for (int gg = 0; gg < G - 1; ++gg) if (gg < g) base += L.grp[gg * 256 + d];
#pragma unroll
        for (int q = 0; q < 8; ++q) L.cnt[(g * 8 + q) * 256 + d] = base + c[q];
        if (g == G - 1) L.tot[d] = base + run;
    } else {
        for (int d = t; d < 256; d += THREADS) {
            uint32_t run = 0;
#pragma unroll
            for (int ww = 0; ww < NW; ++ww) { const uint32_t c = L.cnt[ww * 256 + d]; L.cnt[ww * 256 + d] = run; run += c; }
            L.tot[d] = run;
        }
    }
    __syncthreads();
    if (w == 0) {                                                    // exclusive scan of the 256 digit totals
        uint32_t v[8], sum = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) { v[q] = L.tot[lane * 8 + q]; sum += v[q]; }
        uint32_t incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
        uint32_t run = incl - sum;
#pragma unroll
        for (int q = 0; q < 8; ++q) { L.tot[lane * 8 + q] = run; run += v[q]; }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        if (k < kpw && wbeg + k * 32 + lane < wend) {
            const uint32_t dgt = (uint32_t)(x[k] >> shift) & 255u;
            L.buf[L.tot[dgt] + my_cnt[dgt] + off[k]] = x[k];
        }
    }
    __syncthreads();
}

// Sorts L.buf[0 .. n) ascending as 64-bit integers, in place.  Every thread of the CTA calls it; n <= THREADS*IPT.
template <int THREADS, int IPT>
__device__ __forceinline__ void block_radix_sort(const RadixLayout<THREADS, IPT>& L, int n)
{
    constexpr int NW = THREADS / 32;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    uint32_t kmin = 0xffffffffu, kmax = 0u;
    for (int i = t; i < n; i += THREADS) { const uint32_t k = (uint32_t)(L.buf[i] >> 32); kmin = min(kmin, k); kmax = max(kmax, k); }
    kmin = __reduce_min_sync(0xffffffffu, kmin); kmax = __reduce_max_sync(0xffffffffu, kmax);
    if (lane == 0) { L.red[w] = kmin; L.red[NW + w] = kmax; }
    __syncthreads();
    for (int ww = 0; ww < NW; ++ww) { kmin = min(kmin, L.red[ww]); kmax = max(kmax, L.red[NW + ww]); }
    const uint32_t kdiff = kmin ^ kmax;
    const int nk = kdiff ? (32 - __clz(kdiff) + 7) >> 3 : 0;       // 8-bit passes over the varying key bits
    const int cpw = ((n + NW * 32 - 1) / (NW * 32)) * 32;
    int ns = 0;                                                      // slot passes: none in the first round
    for (int round = 0; ; ++round) {
#pragma unroll 1
        for (int p = 0; p < ns + nk; ++p) radix_pass<THREADS, IPT>(L, n, cpw, p < ns ? 8 * p : 32 + 8 * (p - ns));
        if (round == 1) return;
        // equal keys: the thread at the start of a run of up to MAXRUN equal keys puts it in slot order by insertion
        // (runs are disjoint); a longer run (duplicate depths) needs the slot passes
        constexpr int MAXRUN = 16;
        int longrun = 0;
        for (int i = t; i + 1 < n; i += THREADS) {
            const uint32_t k0 = (uint32_t)(L.buf[i] >> 32);
            if (k0 != (uint32_t)(L.buf[i + 1] >> 32) || (i > 0 && (uint32_t)(L.buf[i - 1] >> 32) == k0)) continue;
            int e = i + 2;
            while (e < n && e - i <= MAXRUN && (uint32_t)(L.buf[e] >> 32) == k0) ++e;
            if (e - i > MAXRUN) { longrun = 1; continue; }
            for (int a = i + 1; a < e; ++a) {
                const u64 v = L.buf[a];
                int b = a - 1;
                while (b >= i && L.buf[b] > v) { L.buf[b + 1] = L.buf[b]; --b; }
                L.buf[b + 1] = v;
            }
        }
        longrun = __syncthreads_or(longrun);
        if (!longrun) return;
        // second round: stable LSD over the varying slot bits, then the key bits again
        uint32_t smin = 0xffffffffu, smax = 0u;
        for (int i = t; i < n; i += THREADS) { const uint32_t sl = (uint32_t)L.buf[i]; smin = min(smin, sl); smax = max(smax, sl); }
        smin = __reduce_min_sync(0xffffffffu, smin); smax = __reduce_max_sync(0xffffffffu, smax);
        if (lane == 0) { L.red[2 * NW + w] = smin; L.red[3 * NW + w] = smax; }
        __syncthreads();
        for (int ww = 0; ww < NW; ++ww) { smin = min(smin, L.red[2 * NW + ww]); smax = max(smax, L.red[3 * NW + ww]); }
        const uint32_t sdiff = smin ^ smax;
        ns = sdiff ? (32 - __clz(sdiff) + 7) >> 3 : 0;
    }
}

// ---- radix tier kernel: one CTA sorts one segment, one bucket, or one 8192-item block ------------------
template <int THREADS, int IPT>
__global__ void __launch_bounds__(THREADS)
k_tier_radix(const SortJob* __restrict__ jobs, FrameHeader* __restrict__ hdr, int list, int tier,
             u64* __restrict__ pairs, u64* __restrict__ pairs_alt)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    const RadixLayout<THREADS, IPT> L(s_raw);
    __shared__ uint32_t s_job;
    const int t = threadIdx.x;
    for (;;) {
        __syncthreads();
        if (t == 0) s_job = atomicAdd(&hdr->sort_cursor[list][tier], 1u);
        __syncthreads();
        const uint32_t jb = s_job;
        if (jb >= hdr->n_sort_jobs[list][tier]) return;
        const SortJob job = jobs[jb];
        const int n = (int)job.len;
        const u64* gsrc = ((job.flags & 2u) ? pairs_alt : pairs) + job.start;
        for (int i = t; i < n; i += THREADS) L.buf[i] = gsrc[i];
        __syncthreads();
        block_radix_sort<THREADS, IPT>(L, n);
        u64* gdst = ((job.flags & 1u) ? pairs_alt : pairs) + job.start;
        for (int i = t; i < n; i += THREADS) gdst[i] = L.buf[i];
    }
}

// ---- oversize segments: one kernel, three phases ------------------------------------------
// bucket of item x = number of splitters <= x (splitters ascending, nb - 1 of them)
__device__ __forceinline__ uint32_t bucket_of(const u64* s_split, uint32_t n_split, u64 x)
{
    uint32_t lo = 0, hi = n_split;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (s_split[mid] <= x) lo = mid + 1; else hi = mid; }
    return lo;
}

constexpr int OVER_THREADS = 256;
constexpr int SCAT_ITEMS = HIGS_SPLIT_TILE / OVER_THREADS;
static_assert(HIGS_MAX_SPLIT <= OVER_THREADS && HIGS_MAX_SPLIT <= 256, "one thread per bucket in the bucket scan; bucket ids are bytes");
constexpr size_t OVER_BUF = sizeof(u64) * (OVER_THREADS * IPT + OVER_THREADS + 2) + sizeof(int) * (OVER_THREADS + 2);    // sidx(4096) items of the sample sort
constexpr size_t OVER_SMEM = OVER_BUF + sizeof(u64) * HIGS_MAX_SPLIT + sizeof(uint32_t) * (2 * HIGS_MAX_SPLIT + 64);

// last segment with tile_base <= tile
__device__ __forceinline__ int seg_of_tile(const SplitSeg* __restrict__ split, uint32_t n_over, uint32_t tile)
{
    int lo = 0, hi = (int)n_over - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (split[mid].tile_base <= tile) lo = mid; else hi = mid - 1; }
    return lo;
}

// Phase 0: splitters of every oversize segment from a sorted strided sample.  Phase 1: per-bucket totals.
// Phase 2: every tile reserves its share of each bucket with one atomic on the bucket cursor and writes its items
// there in the alternate buffer (order inside a bucket is arbitrary: the tier sort follows); the CTA that owns a
// segment's first tile turns its buckets into tier jobs (list 1).  The phases are separated by completion counters
// (see below); the kernel replaces a chain of four dependent launches.
__global__ void __launch_bounds__(OVER_THREADS)
k_oversize(const SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr, const u64* __restrict__ pairs, u64* __restrict__ pairs_alt,
           u64* __restrict__ splitters, uint32_t* __restrict__ bucket_count, uint32_t* __restrict__ bucket_cursor,
           SortJob* __restrict__ jobs /* list 1 */, size_t max_jobs, OverSeg* __restrict__ over, uint8_t* __restrict__ bucket_id)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    __shared__ uint32_t s_claim;
    u64* buf = reinterpret_cast<u64*>(s_raw);
    u64* s_split = reinterpret_cast<u64*>(s_raw + OVER_BUF);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(s_split + HIGS_MAX_SPLIT);
    uint32_t* s_base = s_hist + HIGS_MAX_SPLIT;
    uint32_t* s_scan = s_base + HIGS_MAX_SPLIT;                     // [33] warp totals of the bucket scan
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    pdl_wait();
    const uint32_t n_over = hdr->n_oversize, n_tiles = hdr->n_split_tiles;
    if (n_over == 0) return;
    // Work items of a phase are claimed from a device counter and counted when done; a CTA enters the next phase once
    // every item of the previous one is done.  Whoever holds an item is running, so the wait cannot deadlock whether or
    // not the whole grid is resident (the tier kernels of the whole segments share the SMs with this kernel).
    auto claim = [&](int phase) -> uint32_t {
        __syncthreads();
        if (t == 0) s_claim = atomicAdd(&hdr->split_cursor[phase], 1u);
        __syncthreads();
        return s_claim;
    };
    auto done = [&](int phase) {
        __syncthreads();
        if (t == 0) { __threadfence(); atomicAdd(&hdr->split_done[phase], 1u); }
    };
    auto wait_all = [&](int phase, uint32_t n_work) {
        if (t == 0) {
            while (*reinterpret_cast<volatile uint32_t*>(&hdr->split_done[phase]) < n_work) __nanosleep(200);
            __threadfence();
        }
        __syncthreads();
    };

    for (;;) {
        const uint32_t si = claim(0);
        if (si >= n_over) break;
        const SplitSeg sg = split[si];
        const int m = (int)(sg.oversample * sg.nb);                  // sample size, <= 4096 <= len
        const u64* src = pairs + sg.start;
        __syncthreads();
        const int m_pad = ((m + IPT - 1) / IPT) * IPT;
        for (int i = t; i < m_pad; i += OVER_THREADS) buf[sidx(i)] = i < m ? src[(uint32_t)(((u64)i * sg.len) / (uint32_t)m)] : ~0ull;
        __syncthreads();
        block_sort_smem<OVER_THREADS>(buf, m, m_pad);
        for (uint32_t b = t; b < sg.nb; b += OVER_THREADS) {
            if (b + 1 < sg.nb) splitters[sg.bucket_base + b] = buf[sidx((int)((b + 1) * sg.oversample))];
            bucket_count[sg.bucket_base + b] = 0;
            bucket_cursor[sg.bucket_base + b] = 0;
        }
        done(0);
    }
    wait_all(0, n_over);

    for (int phase = 1; phase <= 2; ++phase) {
        for (;;) {
            const uint32_t tile = claim(phase);
            if (tile >= n_tiles) break;
            const int si = seg_of_tile(split, n_over, tile);
            const SplitSeg sg = split[si];
            __syncthreads();                                          // previous tile's shared state is free
            for (uint32_t b = t; b < sg.nb; b += OVER_THREADS) {
                if (phase == 1 && b + 1 < sg.nb) s_split[b] = splitters[sg.bucket_base + b];
                s_hist[b] = 0;
            }
            uint32_t my_count = 0, my_start = 0;
            if (phase == 2) {                                         // bucket b starts at the exclusive prefix of the totals (thread = bucket)
                my_count = (uint32_t)t < sg.nb ? bucket_count[sg.bucket_base + t] : 0u;
                uint32_t incl = my_count;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
                if (lane == 31) s_scan[w] = incl;
                __syncthreads();
                if (w == 0) {
                    const uint32_t x = lane < OVER_THREADS / 32 ? s_scan[lane] : 0u;
                    uint32_t sc = x;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, sc, d); if (lane >= d) sc += y; }
                    if (lane < OVER_THREADS / 32) s_scan[lane] = sc - x;
                }
                __syncthreads();
                my_start = sg.start + s_scan[w] + incl - my_count;
            }
            __syncthreads();
            const uint32_t o0 = (tile - sg.tile_base) * HIGS_SPLIT_TILE;
            const u64* src = pairs + sg.start;
            u64 x[SCAT_ITEMS]; uint32_t bk[SCAT_ITEMS], rk[SCAT_ITEMS];
#pragma unroll
            for (int k = 0; k < SCAT_ITEMS; ++k) {
                const uint32_t i = o0 + k * OVER_THREADS + t;
                x[k] = i < sg.len ? src[i] : 0ull;
            }
#pragma unroll
            for (int k = 0; k < SCAT_ITEMS; ++k) {
                const uint32_t i = o0 + k * OVER_THREADS + t;
                bk[k] = 0; rk[k] = 0;
                if (i < sg.len) {                                    // the search runs once: phase 2 reads the bucket back (nb <= 256)
                    if (phase == 1) { bk[k] = bucket_of(s_split, sg.nb - 1, x[k]); bucket_id[sg.start + i] = (uint8_t)bk[k]; }
                    else bk[k] = bucket_id[sg.start + i];
                    rk[k] = atomicAdd(&s_hist[bk[k]], 1u);
                }
            }
            __syncthreads();
            if ((uint32_t)t < sg.nb) {
                const uint32_t h = s_hist[t];
                if (phase == 1) { if (h) atomicAdd(&bucket_count[sg.bucket_base + t], h); }
                else s_base[t] = my_start + (h ? atomicAdd(&bucket_cursor[sg.bucket_base + t], h) : 0u);
            }
            if (phase == 2) {
                __syncthreads();
#pragma unroll
                for (int k = 0; k < SCAT_ITEMS; ++k) {
                    const uint32_t i = o0 + k * OVER_THREADS + t;
                    if (i < sg.len) {
                        HIGS_ASSERT(s_base[bk[k]] + rk[k] >= sg.start && s_base[bk[k]] + rk[k] < sg.start + sg.len);
                        pairs_alt[s_base[bk[k]] + rk[k]] = x[k];
                    }
                }
                if (tile == sg.tile_base && (uint32_t)t < sg.nb && my_count) {   // this segment's buckets -> tier jobs
                    const uint32_t n = my_count;
                    if (n <= HIGS_SORT_BLOCK) {
                        const int tr = tier_of(n);                   // a one-item bucket still has to travel back from the alternate buffer
                        jobs[(size_t)tr * max_jobs + atomicAdd(&hdr->n_sort_jobs[1][tr], 1u)] = SortJob{my_start, n, 2u, 0u};
                    } else {                                         // still too large: 8192-blocks + merge levels (k_merge_levels)
                        const uint32_t nc = (n + HIGS_SORT_BLOCK - 1) / HIGS_SORT_BLOCK, levels = 32 - __clz(nc - 1);
                        const uint32_t j0 = atomicAdd(&hdr->n_sort_jobs[1][3], nc);
                        for (uint32_t c = 0; c < nc; ++c) {
                            const uint32_t cs = c * HIGS_SORT_BLOCK;
                            jobs[(size_t)3 * max_jobs + j0 + c] = SortJob{my_start + cs, min((uint32_t)HIGS_SORT_BLOCK, n - cs), 2u | (levels & 1u), 0u};
                        }
                        // (index, first merge tile) handed out together, so that tile_base grows with the index
                        const unsigned long long fp = atomicAdd(&hdr->fallback_pack, (1ull << 32) | (unsigned long long)((n + HIGS_MERGE_TILE - 1) / HIGS_MERGE_TILE));
                        over[(uint32_t)(fp >> 32)] = OverSeg{my_start, n, levels, (uint32_t)fp};
                        atomicMax(&hdr->max_levels, levels);
                    }
                }
            }
            done(phase);
        }
        if (phase == 1) wait_all(1, n_tiles);
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
    const unsigned long long fp = hdr->fallback_pack;                 // (fallback buckets << 32 | merge tiles)
    const uint32_t n_tiles = (uint32_t)fp, n_over = (uint32_t)(fp >> 32), max_levels = hdr->max_levels;
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
constexpr size_t sort_smem() { return (size_t)(THREADS * IPT + THREADS + 2) * sizeof(u64) + (THREADS + 2) * sizeof(int); }   // sidx(CAP) items + the threads' splits

// tier t: segments / buckets of up to 1024 << t items
template <int TIER> struct TierCfg;
template <> struct TierCfg<0> { static constexpr int R_THREADS = 128, R_IPT = 8,  M_THREADS = 64; };
template <> struct TierCfg<1> { static constexpr int R_THREADS = 256, R_IPT = 8,  M_THREADS = 128; };
template <> struct TierCfg<2> { static constexpr int R_THREADS = 512, R_IPT = 8,  M_THREADS = 256; };
template <> struct TierCfg<3> { static constexpr int R_THREADS = 1024, R_IPT = 8, M_THREADS = 512; };

template <int TIER>
int launch_tier(higs_ctx* ctx, int list, u64* pairs, bool merge_sort, cudaStream_t st)
{
    typedef TierCfg<TIER> C;
    const SortJob* jobs = ctx->sort_jobs + (size_t)(list * HIGS_N_TIERS + TIER) * ctx->max_jobs;
    const int ctas = ctx->n_sm * ctx->tier_ctas_per_sm[merge_sort ? 1 : 0][TIER];
    if (merge_sort)
        k_block_sort<C::M_THREADS><<<ctas, C::M_THREADS, sort_smem<C::M_THREADS>(), st>>>(jobs, ctx->hdr, list, TIER, pairs, ctx->pairs_alt);
    else
        k_tier_radix<C::R_THREADS, C::R_IPT><<<ctas, C::R_THREADS, RadixLayout<C::R_THREADS, C::R_IPT>::bytes, st>>>(jobs, ctx->hdr, list, TIER, pairs, ctx->pairs_alt);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

template <int TIER>
int setup_tier(higs_ctx* ctx)
{
    typedef TierCfg<TIER> C;
    int occ = 0;
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_block_sort<C::M_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem<C::M_THREADS>()));
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_block_sort<C::M_THREADS>, C::M_THREADS, sort_smem<C::M_THREADS>()));
    ctx->tier_ctas_per_sm[1][TIER] = occ < 1 ? 1 : occ;
    constexpr size_t rb = RadixLayout<C::R_THREADS, C::R_IPT>::bytes;
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_tier_radix<C::R_THREADS, C::R_IPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb));
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tier_radix<C::R_THREADS, C::R_IPT>, C::R_THREADS, rb));
    ctx->tier_ctas_per_sm[0][TIER] = occ < 1 ? 1 : occ;
    return HIGS_OK;
}

int run_sort(higs_ctx* ctx, u64* pairs, const uint32_t* seg_offset, int n_seg, const FrameParams* frame, cudaStream_t st)
{
    const bool plan_done = frame != nullptr;
    SortJob* jobs0 = ctx->sort_jobs;
    SortJob* jobs1 = ctx->sort_jobs + (size_t)HIGS_N_TIERS * ctx->max_jobs;
    u64* alt = ctx->pairs_alt;
    const bool ms = (ctx->flags & HIGS_FLAG_RADIX_SORT) == 0;
    int rc;
    if (!plan_done) {                                             // inside a frame k_plan has already done this (binning.cu)
        k_sort_plan<<<1, 1024, 0, st>>>(seg_offset, n_seg, jobs0, (size_t)ctx->max_jobs, ctx->split_segs, ctx->hdr);
        HIGS_LAUNCHED(ctx);
    }
    // fork: whole segments go through the tier kernels on side streams (the paper overlaps tiers with PDL)
    // while the main stream splits the oversize segments into buckets
    HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_fork, st));
    for (int k = 0; k < 4; ++k) HIGS_CUDA(ctx, cudaStreamWaitEvent(ctx->aux_stream[k], ctx->ev_fork, 0));
    {
        const SplitSeg* split = ctx->split_segs; FrameHeader* hdr = ctx->hdr; const u64* src = pairs;
        u64* splitters = ctx->splitters; uint32_t* bc = ctx->bucket_count; uint32_t* bcur = ctx->bucket_cursor;
        size_t mj = (size_t)ctx->max_jobs; OverSeg* over = ctx->over_segs;
        HIGS_CUDA(ctx, launch_pdl(k_oversize, dim3(ctx->n_sm * ctx->over_ctas_per_sm), dim3(OVER_THREADS), OVER_SMEM, st, split, hdr, src, alt, splitters, bc, bcur,
                                  jobs1, mj, over, ctx->bucket_id));
        HIGS_LAUNCHED(ctx);
    }
    if ((rc = launch_tier<3>(ctx, 0, pairs, ms, ctx->aux_stream[0]))) return rc;
    if (frame && (rc = launch_units(ctx, *frame, ctx->aux_stream[0]))) return rc;   // the unit table: needed by the rasterizer only
    if ((rc = launch_tier<2>(ctx, 0, pairs, ms, ctx->aux_stream[1]))) return rc;
    if ((rc = launch_tier<1>(ctx, 0, pairs, ms, ctx->aux_stream[2]))) return rc;
    if ((rc = launch_tier<0>(ctx, 0, pairs, ms, ctx->aux_stream[3]))) return rc;
    HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_fork2, st));
    for (int k = 1; k < 4; ++k) HIGS_CUDA(ctx, cudaStreamWaitEvent(ctx->aux_stream[k], ctx->ev_fork2, 0));
    if ((rc = launch_tier<1>(ctx, 1, pairs, ms, st))) return rc;              // buckets average HIGS_BUCKET_TARGET items: tier 1 carries most
    if ((rc = launch_tier<0>(ctx, 1, pairs, ms, ctx->aux_stream[1]))) return rc;
    if ((rc = launch_tier<2>(ctx, 1, pairs, ms, ctx->aux_stream[2]))) return rc;
    if ((rc = launch_tier<3>(ctx, 1, pairs, ms, ctx->aux_stream[3]))) return rc;
    HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_join[3], ctx->aux_stream[3]));     // the merge levels follow the 8192-blocks of tier 3
    HIGS_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_join[3], 0));
    const OverSeg* over = ctx->over_segs; const FrameHeader* hdr = ctx->hdr;
    void* args[] = { (void*)&over, (void*)&hdr, (void*)&pairs, (void*)&alt };
    HIGS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)k_merge_levels, dim3(ctx->n_sm * ctx->merge_ctas_per_sm), dim3(MERGE_THREADS), args, 0, st));
    ++ctx->n_launches;
    for (int k = 0; k < 3; ++k) {
        HIGS_CUDA(ctx, cudaEventRecord(ctx->ev_join[k], ctx->aux_stream[k]));
        HIGS_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_join[k], 0));
    }
    return HIGS_OK;
}

} // namespace

int higs_sort_smem_setup(higs_ctx* ctx)
{
    int rc;
    if ((rc = setup_tier<0>(ctx))) return rc;
    if ((rc = setup_tier<1>(ctx))) return rc;
    if ((rc = setup_tier<2>(ctx))) return rc;
    if ((rc = setup_tier<3>(ctx))) return rc;
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_oversize, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)OVER_SMEM));
    int occ = 0;
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_oversize, OVER_THREADS, OVER_SMEM));
    ctx->over_ctas_per_sm = occ < 1 ? 1 : (occ > 4 ? 4 : occ);
    HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_merge_levels, MERGE_THREADS, 0));
    ctx->merge_ctas_per_sm = occ < 1 ? 1 : (occ > 2 ? 2 : occ);
    return HIGS_OK;
}

int launch_sort(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    return run_sort(ctx, ctx->pairs, ctx->mt_offset, P.n_m, &P, st);
}

int launch_sort_only(higs_ctx* ctx, unsigned long long* pairs, const uint32_t* seg_offset, int n_seg, cudaStream_t st)
{
    return run_sort(ctx, pairs, seg_offset, n_seg, nullptr, st);
}
