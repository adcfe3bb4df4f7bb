// sort_plan.cuh -- plan A of the segmented sort (sort.cu): whole segments -> tier job lists (list 0), oversize
// segments -> split plan.  A device function for one CTA of 1024 threads, shared by k_sort_plan (sort.cu, used when
// the sort runs alone) and k_plan (binning.cu, which appends it to the scan so a frame saves a launch).
#pragma once
#include "higs_internal.cuh"

__device__ __forceinline__ int tier_of(uint32_t n) { return n <= 1024u ? 0 : (n <= 2048u ? 1 : (n <= 4096u ? 2 : 3)); }

// exclusive block scan (1024 threads) of NV values per thread position, with a running carry
template <int NV>
__device__ __forceinline__ void plan_scan(uint32_t (&v)[NV], uint32_t (&carry)[NV], uint32_t* s_warp /* [33*NV] */)
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

// ---- plan A: whole segments -> tier job lists (list 0); oversize segments -> split plan --------------
__device__ __forceinline__ uint32_t buckets_of(uint32_t n)
{
    const uint32_t nb = (n + HIGS_BUCKET_TARGET - 1) / HIGS_BUCKET_TARGET;
    return nb > HIGS_MAX_SPLIT ? HIGS_MAX_SPLIT : nb;
}

__device__ __forceinline__ void sort_plan_body(const uint32_t* __restrict__ seg_offset, int n_seg, bool dead, SortJob* __restrict__ jobs,
                                               size_t max_jobs, SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr,
                                               uint32_t* s_warp /* [33*8] shared */)
{
    uint32_t carry[8] = {0, 0, 0, 0, 0, 0, 0, 0};       // tiers 0-3, oversize segments, split tiles, buckets, oversize items
    for (int s0 = 0; s0 < n_seg; s0 += 1024) {
        const int s = s0 + threadIdx.x;
        uint32_t start = 0, n = 0;
        if (s < n_seg && !dead) { start = seg_offset[s]; n = seg_offset[s + 1] - start; }
        uint32_t v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const bool over = n > HIGS_SORT_BLOCK;
        const int t = n > 1 && !over ? tier_of(n) : -1;
        uint32_t nb = 0;
        if (t >= 0) v[t] = 1;
        if (over) { nb = buckets_of(n); v[4] = 1; v[5] = (n + HIGS_SPLIT_TILE - 1) / HIGS_SPLIT_TILE; v[6] = nb; v[7] = n; }
        plan_scan<8>(v, carry, s_warp);
        if (t >= 0) jobs[(size_t)t * max_jobs + v[t]] = SortJob{start, n, 0u, 0u};
        if (over) {
            const uint32_t a = nb > 64u ? 8u : 16u;     // sample = a * nb <= 2048 items, sorted by one CTA; 16 sample items per
                                                        // bucket keep bucket sizes within about +-25 % (1 sigma), 8 within +-35 %
            split[v[4]] = SplitSeg{start, n, nb, v[6], v[5], v[7], a, 0u};
        }
    }
    if (threadIdx.x == 0) {
        for (int t = 0; t < HIGS_N_TIERS; ++t) {
            hdr->n_sort_jobs[0][t] = carry[t]; hdr->sort_cursor[0][t] = 0;
            hdr->n_sort_jobs[1][t] = 0; hdr->sort_cursor[1][t] = 0;
        }
        hdr->n_oversize = carry[4];
        hdr->n_split_tiles = carry[5];
        hdr->n_buckets = carry[6];
        hdr->fallback_pack = 0ull; hdr->max_levels = 0;
        for (int q = 0; q < 3; ++q) { hdr->split_cursor[q] = 0; hdr->split_done[q] = 0; }
    }
}

