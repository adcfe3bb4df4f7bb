// binning.cu -- steps a3 scan, a4 fill, a6 batch schedule (section 3.2,
// PAPER.md:247-257 section 4.3, section 3.1).  The count pass (a2) lives in project.cu.
//
// Count and fill each run one CTA per partitioning batch.  Here a batch is the set of
// HIGS_CHUNK-id chunks one persistent projection CTA claimed (project.cu), so N_B = a whole number of CTAs per SM;
// fill only touches the dense survivor slots, so culled gaussians never reach it.  The
// count CTA's histogram is one row of the N_B x N_M matrix and is also added to mt_count[m] by atomics, so the
// segment bounds are one scan over m (k_plan); a fill CTA reserves its share of a segment with one atomic on
// mt_fill[m].  The fill CTA replays the intersection -- from the 64-bit span descriptor the count left in the
// record, or by redoing the row scan N-SCAN when the span did not fit -- and drops
// (depth key << 32 | id) at base + local rank.
#include <stdio.h>
#include "higs_internal.cuh"
#include "sort_plan.cuh"

namespace {

constexpr int FILL_QCAP = 1024;      // wide-span gaussians a fill CTA can defer (more are handled in place)
constexpr int BIN_THREADS = 1024;   // two CTAs per SM at 32 registers: the pass is latency-bound, so warps in flight decide

// Scan (a3) + batch schedule (a6) + sort plan, one CTA of 1024 threads:
//   mt_count[m] was accumulated by the projection CTAs (one atomicAdd per touched macro-tile per CTA);
//   mt_offset = exclusive scan over m; nb[m] = ceil(n_m / B_r); batch_offset = exclusive scan; unit_mt[u] = m
//   (PAPER.md:81); then the tier job lists of the segmented sort (sort_plan.cuh) and the order of the units.
__global__ void __launch_bounds__(1024)
k_plan(const FrameParams P,
       const uint32_t* __restrict__ mt_count, uint32_t* __restrict__ mt_offset, uint32_t* __restrict__ batch_offset,
       SortJob* __restrict__ sort_jobs, size_t max_jobs, SplitSeg* __restrict__ split, FrameHeader* __restrict__ hdr,
       uint4* __restrict__ pairs_touch, uint32_t touch_max_pairs)
{
    __shared__ uint32_t s_warp[33 * 8];
    __shared__ uint32_t s_max;
    __shared__ unsigned long long s_total;
    if (threadIdx.x == 0) { s_max = 0; s_total = 0ull; }
    pdl_wait(); pdl_trigger();
    __syncthreads();
    // CTAs 1 .. gridDim.x - 1: beside the one CTA that plans, the rest of the GPU has nothing to do for these 13 us.  They write
    // zeros over the part of the pair list the fill pass is about to fill.  The fill pass drops 8-byte items at scattered places:
    // partial-sector writes, which L2 answers with a fill read of the sector from DRAM when the line is not resident (it never is:
    // the list was last touched a frame ago) - ncu counted 47 MB of such reads, and the kernel ran at the pace of those fills,
    // whatever its occupancy or instruction count (0.082 ms).  Whole lines written here are resident and dirty when the fill pass
    // comes (41 MB, L2 holds 126 MB), its partial writes hit, and it runs 0.060 ms, as it does on a spatially ordered scene whose
    // stores coalesce; this kernel grows from 0.013 to 0.019 ms (the zeros are 8 us of L2 write bandwidth).  Every item zeroed
    // here is overwritten by the fill pass, which starts after this grid has completed.  (The same treatment of the alternate
    // buffer the oversize split scatters into was measured and bought nothing.)
    if (blockIdx.x > 0) {
        unsigned long long tot = 0;
        for (int m = threadIdx.x; m < P.n_m; m += 1024) tot += mt_count[m];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, d);
        if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&s_total, tot);
        __syncthreads();
        if (s_total > (unsigned long long)P.max_pairs || s_total > (unsigned long long)touch_max_pairs) return;   // a list that does not fit in L2 gains nothing
        const size_t n16 = (size_t)s_total / 2;                       // whole 16-byte pieces (an odd last item stays a partial write)
        const size_t per = (n16 + (gridDim.x - 1) - 1) / (gridDim.x - 1);
        const size_t a = (size_t)(blockIdx.x - 1) * per, b = a + per < n16 ? a + per : n16;
        for (size_t i = a + threadIdx.x; i < b; i += 1024) pairs_touch[i] = make_uint4(0u, 0u, 0u, 0u);
        return;
    }
    uint32_t carry[2] = {0, 0};
    unsigned long long my_total = 0;
    const uint32_t br = (uint32_t)P.batch_cap;
    // pass 1: totals and offsets
    for (int m0 = 0; m0 < P.n_m; m0 += 1024) {
        const int m = m0 + threadIdx.x;
        uint32_t n = 0;
        if (m < P.n_m) {
            n = mt_count[m];
            my_total += n;
            if (n) atomicMax(&s_max, n);
        }
        uint32_t v[2] = { n, (n + br - 1) / br };
        plan_scan<2>(v, carry, s_warp);
        if (m < P.n_m) { mt_offset[m] = v[0]; batch_offset[m] = v[1]; }
    }
    // the 32-bit scan wraps beyond 2^32 pairs: the capacity check is on a 64-bit total (one shared atomic per warp)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) my_total += __shfl_xor_sync(0xffffffffu, my_total, d);
    if ((threadIdx.x & 31) == 0 && my_total) atomicAdd(&s_total, my_total);
    __syncthreads();
    const uint32_t n_pairs = carry[0], n_units = carry[1];
    const bool overflow = s_total > (unsigned long long)P.max_pairs || n_units > P.max_units;
    if (threadIdx.x == 0) {
        mt_offset[P.n_m] = n_pairs; batch_offset[P.n_m] = n_units;
        hdr->n_pairs = overflow ? 0u : n_pairs;
        hdr->n_units = overflow ? 0u : n_units;
        hdr->overflow = overflow ? 1u : 0u;
        hdr->max_segment = s_max;
    }
    __syncthreads();                                              // mt_offset is complete (and visible to this CTA)
    sort_plan_body(mt_offset, P.n_m, overflow, sort_jobs, max_jobs, split, hdr, s_warp);
}

// a6, second part (off the critical path: it runs beside the sort and is needed by the rasterizer only): the unit table and
// the order the rasterizer claims units in - batch index j major ("level" j = the j-th batch of every macro-tile that has one),
// so that by the time a deep batch starts the batches in front of it have published their transmittance bounds (cross-batch
// cut).
__global__ void __launch_bounds__(1024)
k_units(const FrameParams P, const uint32_t* __restrict__ mt_count, const uint32_t* __restrict__ batch_offset,
        uint32_t* __restrict__ unit_mt, uint32_t* __restrict__ unit_order, uint32_t* __restrict__ level_hist,
        uint32_t* __restrict__ level_cur, const FrameHeader* __restrict__ hdr)
{
    extern __shared__ uint32_t s_bo[];                            // [n_m + 1] copy of batch_offset for the unit -> macro-tile search
    __shared__ uint32_t s_warp[33 * 8];
    if (hdr->overflow) return;
    const uint32_t br = (uint32_t)P.batch_cap, s_max = hdr->max_segment, n_units = hdr->n_units;
    for (int m = threadIdx.x; m <= P.n_m; m += 1024) s_bo[m] = batch_offset[m];
    const uint32_t max_nb = (s_max + br - 1) / br;
    for (uint32_t v = threadIdx.x; v <= max_nb + 1; v += 1024) level_hist[v] = 0;
    __syncthreads();
    for (int m = threadIdx.x; m < P.n_m; m += 1024) {
        const uint32_t nb = (mt_count[m] + br - 1) / br;
        if (nb) atomicAdd(&level_hist[nb], 1u);               // macro-tiles with exactly nb batches
    }
    __syncthreads();
    // units in level j = macro-tiles with more than j batches = n_nonempty - #{nb <= j}; level bases = exclusive
    // prefix of that over j.  Two chained block scans over j in chunks of 1024.
    {
        uint32_t c_hist[1] = {0}, c_base[1] = {0};
        __shared__ uint32_t s_nonempty;
        if (threadIdx.x == 0) s_nonempty = 0;
        __syncthreads();
        uint32_t mine = 0;
        for (uint32_t v = threadIdx.x; v <= max_nb; v += 1024) mine += level_hist[v];
        mine = __reduce_add_sync(0xffffffffu, mine);
        if ((threadIdx.x & 31) == 0 && mine) atomicAdd(&s_nonempty, mine);
        __syncthreads();
        const uint32_t n_nonempty = s_nonempty;
        for (uint32_t j0 = 0; j0 < max_nb; j0 += 1024) {
            const uint32_t j = j0 + threadIdx.x;
            const uint32_t h = (j < max_nb) ? level_hist[j + 1] : 0u;       // hist[0] is unused (nb = 0 is never counted)
            uint32_t v[1] = { h };
            plan_scan<1>(v, c_hist, s_warp);                        // v = #{1 <= nb <= j}
            const uint32_t cnt = (j < max_nb) ? n_nonempty - v[0] : 0u;     // macro-tiles with nb > j
            uint32_t b[1] = { cnt };
            plan_scan<1>(b, c_base, s_warp);
            if (j < max_nb) level_cur[j] = b[0];
        }
    }
    __syncthreads();
    for (uint32_t u = threadIdx.x; u < n_units; u += 1024) {
        int lo = 0, hi = P.n_m - 1;                                       // last m with batch_offset[m] <= u and a batch there
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_bo[mid] <= u) lo = mid; else hi = mid - 1; }
        unit_mt[u] = (uint32_t)lo;
        const uint32_t lvl = u - s_bo[lo];
        const uint32_t at = atomicAdd(&level_cur[lvl], 1u);
        HIGS_ASSERT(at < n_units && lvl < max_nb);
        unit_order[at] = u;
    }
}

#define HIGS_DESC_FALLBACK 0x8000000000000000ull   // see project.cu

// a4: one CTA per partition batch = per CTA of the projection kernel, which left the list of chunks it claimed.
// The survivors of those chunks sit densely in `bin`; the CTA flattens them (prefix sum over the chunk counts) and
// strides over them with all its threads, so the loads are coalesced, independent, and every lane has work.
// Items are (depth key << 32 | slot).
__global__ void __launch_bounds__(BIN_THREADS, 2)
k_fill(const uint32_t* __restrict__ chunk_count, const uint32_t* __restrict__ part_list, const uint2* __restrict__ part_desc, int lcap,
       const uint4* __restrict__ bin, const float4* __restrict__ rec,
       const FrameParams P, const uint32_t* __restrict__ hist, uint32_t* __restrict__ mt_fill, const uint32_t* __restrict__ mt_offset,
       unsigned long long* __restrict__ pairs, const FrameHeader* __restrict__ hdr,
       unsigned long long* __restrict__ cut_word, int* __restrict__ cut_term, uint32_t* __restrict__ tile_load)
{
    extern __shared__ uint32_t s_cursor[];
    uint32_t* s_chunk = s_cursor + P.n_m;           // [lcap]
    uint32_t* s_pref = s_chunk + lcap;              // [lcap + 1] survivors of each chunk of the list
    uint32_t* s_queue = s_pref + lcap + 1;          // [2 * FILL_QCAP] (slot, key) of the gaussians with wide spans
    __shared__ uint32_t s_nq, s_next;
    if (threadIdx.x == 0) s_nq = 0;
    pdl_wait(); pdl_trigger();
    if (hdr->overflow) return;                      // capacity exceeded: write nothing (HIGS_E_CAPACITY)
    // the rasterizer's cross-batch cut state starts every frame at zero (raster.cu): cleared here, where the grid is wide
    // and the unit count is known, instead of by a memset sized for the capacity
    if (!(P.flags & HIGS_FLAG_NO_XBATCH_CUT)) {
        const size_t n_word = (size_t)P.n_m * HIGS_MT_TILES, n_term = (size_t)hdr->n_units * HIGS_MT_TILES;
        const size_t stride = (size_t)gridDim.x * BIN_THREADS;
        for (size_t i = (size_t)blockIdx.x * BIN_THREADS + threadIdx.x; i < n_word; i += stride) cut_word[i] = 0ull;
        for (size_t i = (size_t)blockIdx.x * BIN_THREADS + threadIdx.x; i < n_term; i += stride) cut_term[i] = 0;
    }
    if (P.flags & HIGS_FLAG_COUNT_EVALS)
        for (size_t i = (size_t)blockIdx.x * BIN_THREADS + threadIdx.x; i < (size_t)P.n_m * HIGS_MT_TILES; i += (size_t)gridDim.x * BIN_THREADS) tile_load[i] = 0u;
    const uint32_t b = blockIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint2 pd = part_desc[b];
    const uint32_t n_list = min(pd.y, (uint32_t)lcap);
    if (w == 0) {                                   // chunk list + prefix of the counts (a few dozen entries)
        uint32_t run = 0;
        for (uint32_t e0 = 0; e0 < n_list; e0 += 32) {
            const uint32_t e = e0 + lane;
            const uint32_t c = e < n_list ? part_list[pd.x + e] : 0u;
            const uint32_t n = e < n_list ? chunk_count[c] : 0u;
            uint32_t x = n;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
            if (e < n_list) { s_chunk[e] = c; s_pref[e] = n; }
            run += __shfl_sync(0xffffffffu, x, 31);
        }
        if (lane == 0) s_pref[n_list] = run;
    }
    if (threadIdx.x == 0) s_next = 0;
    // this batch's share of every macro-tile it touches: reserved with one atomic on the macro-tile's fill counter
    // (which batch lands where inside a segment is arbitrary; the depth sort orders the segment anyway)
    for (int m = threadIdx.x; m < P.n_m; m += BIN_THREADS) {
        const uint32_t h = hist[(size_t)b * P.n_m + m];
        s_cursor[m] = h ? mt_offset[m] + atomicAdd(&mt_fill[m], h) : 0u;
    }
    __syncthreads();
    // A gaussian whose span did not fit the descriptor (more than 4 macro-tile rows: 0.8 % of the survivors at 1080p,
    // 4.5 % at 4K) redoes the row scan, some hundreds of instructions.  Done in place it would run with one lane of the
    // warp active in a quarter (1080p) to three quarters (4K) of all warp iterations, so such gaussians are queued and
    // handled after the main loop, one per lane.
    auto emit_wide = [&](size_t slot, uint32_t key) {
        const unsigned long long item = ((unsigned long long)key << 32) | (unsigned long long)(uint32_t)slot;
        const float4 s0 = __ldcs(rec + 4 * slot), s1 = __ldcs(rec + 4 * slot + 1), s2 = __ldcs(rec + 4 * slot + 2),
                     s3 = __ldcs(rec + 4 * slot + 3);
        RowScan rs{};
        rs.init(s0.x, s0.y, s2.z, s2.w, s3.x, tau_scan(s2.z, s2.w, s3.x, s1.y), (float)(P.mt_ty * P.tile), P.n_my);
        const float fW = (float)P.W, fH = (float)P.H;
        for (int r = rs.r0; r <= rs.r1; ++r) {
            int m0, m1;
            if (!rs.row(r, (float)(P.mt_tx * P.tile), (float)(P.mt_ty * P.tile), fW, fH, P.n_mx, m0, m1)) continue;
            for (int m = m0; m <= m1; ++m) {
                const uint32_t at = atomicAdd(&s_cursor[r * P.n_mx + m], 1u);
                HIGS_ASSERT(at >= mt_offset[r * P.n_mx + m] && at < mt_offset[r * P.n_mx + m + 1]);
                pairs[at] = item;
            }
        }
    };
    auto emit = [&](size_t slot, const uint4 bn) {  // bn = key, desc lo, desc hi, id
        const unsigned long long item = ((unsigned long long)bn.x << 32) | (unsigned long long)(uint32_t)slot;
        const unsigned long long desc = ((unsigned long long)bn.z << 32) | bn.y;
        if (!(desc & HIGS_DESC_FALLBACK)) {
            const int r0 = (int)(desc & 511u), nr = (int)((desc >> 9) & 3u);
            for (int rr = 0; rr <= nr; ++rr) {
                const uint32_t f = (uint32_t)(desc >> (11 + 13 * rr)) & 0x1fffu;
                const int m0 = (int)(f & 511u);
                if (m0 == 511) continue;
                const int cell0 = (r0 + rr) * P.n_mx + m0, wd = (int)(f >> 9);
                for (int m = 0; m <= wd; ++m) {
                    const uint32_t at = atomicAdd(&s_cursor[cell0 + m], 1u);
                    HIGS_ASSERT(cell0 + m < P.n_m && at >= mt_offset[cell0 + m] && at < mt_offset[cell0 + m + 1]);
                    pairs[at] = item;
                }
            }
        } else {                                    // span too large for the descriptor: queue it (or, queue full, do it here)
            const uint32_t qpos = atomicAdd(&s_nq, 1u);
            if (qpos < (uint32_t)FILL_QCAP) { s_queue[2 * qpos] = (uint32_t)slot; s_queue[2 * qpos + 1] = bn.x; }
            else emit_wide(slot, bn.x);
        }
    };
    // warps claim chunks (up to 128 dense survivor slots: four warp iterations) from a shared counter: no search for the
    // slot of the k-th survivor of the batch (it was a third of the kernel's instructions and the time did not move; neither did it
    // with half the warps, with the records requested four deep or prefetched: the kernel ran at the pace of L2's fill reads for
    // its partial-sector stores, see k_plan), tail of at most one chunk.
    for (;;) {
        uint32_t q = 0;
        if (lane == 0) q = atomicAdd(&s_next, 1u);
        q = __shfl_sync(0xffffffffu, q, 0);
        if (q >= n_list) break;
        const uint32_t n = s_pref[q];
        const size_t slot0 = (size_t)s_chunk[q] * HIGS_CHUNK;
        for (uint32_t k = lane; k < n; k += 32) emit(slot0 + k, __ldcs(bin + slot0 + k));
    }
    __syncthreads();
    const uint32_t n_wide = min(s_nq, (uint32_t)FILL_QCAP);
    for (uint32_t k = threadIdx.x; k < n_wide; k += BIN_THREADS) emit_wide((size_t)s_queue[2 * k], s_queue[2 * k + 1]);
}

// test-facing exports (higs_get_lists / higs_get_records; never part of a frame)
__global__ void k_export_lists(const unsigned long long* __restrict__ pairs, const uint4* __restrict__ bin, uint32_t n,
                               unsigned long long* __restrict__ out)
{
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const unsigned long long it = pairs[p];
    out[p] = (it & 0xffffffff00000000ull) | (unsigned long long)bin[(uint32_t)it].w;
}

__global__ void k_export_records(const uint32_t* __restrict__ chunk_count, const float4* __restrict__ rec, const uint4* __restrict__ bin,
                                 int64_t n_slots, float* __restrict__ out)
{
    const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= n_slots) return;
    if ((uint32_t)(slot % HIGS_CHUNK) >= chunk_count[slot / HIGS_CHUNK]) return;
    const float4 q0 = rec[4 * slot], q1 = rec[4 * slot + 1], q2 = rec[4 * slot + 2], q3 = rec[4 * slot + 3];
    const uint4 bn = bin[slot];
    float* o = out + (size_t)bn.w * 16;               // mux, muy, A, B2, C, tau, log2 o, r, g, b, bits(key), desc lo, desc hi, a, b, c
    o[0] = q0.x; o[1] = q0.y; o[2] = q0.z; o[3] = q0.w; o[4] = q1.x; o[5] = q1.y; o[6] = q1.z; o[7] = q1.w;
    o[8] = q2.x; o[9] = q2.y; o[10] = __uint_as_float(bn.x); o[11] = __uint_as_float(bn.y); o[12] = __uint_as_float(bn.z);
    o[13] = q2.z; o[14] = q2.w; o[15] = q3.x;
}

__global__ void k_zero_lists(uint32_t* mt_count, uint32_t* mt_offset, uint32_t* batch_offset, int n_m)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m < n_m) mt_count[m] = 0;
    if (m <= n_m) { mt_offset[m] = 0; batch_offset[m] = 0; }
}

} // namespace

int launch_binning(higs_ctx* ctx, const FrameParams& P, int64_t N, cudaStream_t st, cudaEvent_t ev_count, cudaEvent_t ev_scan)
{
    const int n_b = N > 0 ? higs_part_grid(ctx, N) : 0;
    if (n_b == 0) {
        k_zero_lists<<<(P.n_m + 256) / 256, 256, 0, st>>>(ctx->mt_count, ctx->mt_offset, ctx->batch_offset, P.n_m);
        HIGS_LAUNCHED(ctx);
        if (ev_count) { cudaEventRecord(ev_count, st); cudaEventRecord(ev_scan, st); }
        return HIGS_OK;
    }
    const int lcap = higs_part_lcap((N + HIGS_CHUNK - 1) / HIGS_CHUNK, n_b);
    const size_t smem = sizeof(uint32_t) * ((size_t)P.n_m + 2 * (size_t)lcap + 1 + 2 * FILL_QCAP);
    if (ev_count) cudaEventRecord(ev_count, st);    // the count pass ran inside k_project: this stage is empty
    HIGS_CUDA(ctx, launch_pdl(k_plan, dim3(1 + ctx->n_sm), dim3(1024), 0, st, P, ctx->mt_count, ctx->mt_offset, ctx->batch_offset, ctx->sort_jobs,
                              (size_t)ctx->max_jobs, ctx->split_segs, ctx->hdr, reinterpret_cast<uint4*>(ctx->pairs), ctx->touch_max_pairs));
    HIGS_LAUNCHED(ctx);
    if (ev_scan) cudaEventRecord(ev_scan, st);
    HIGS_CUDA(ctx, launch_pdl(k_fill, dim3(n_b), dim3(BIN_THREADS), smem, st, ctx->chunk_count, ctx->part_list, ctx->part_desc, lcap, ctx->bin,
                              ctx->rec, P, ctx->hist, ctx->mt_fill, ctx->mt_offset, ctx->pairs, ctx->hdr, ctx->cut_word, ctx->cut_term, ctx->tile_load));
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

// enqueued on a side stream of the sort (sort.cu), behind the event recorded after k_fill
int launch_units(higs_ctx* ctx, const FrameParams& P, cudaStream_t st)
{
    k_units<<<1, 1024, sizeof(uint32_t) * ((size_t)P.n_m + 1), st>>>(P, ctx->mt_count, ctx->batch_offset, ctx->unit_mt, ctx->unit_order,
                                                                     ctx->level_hist, ctx->level_cur, ctx->hdr);
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int launch_export_lists(higs_ctx* ctx, uint32_t n_pairs, cudaStream_t st)
{
    k_export_lists<<<(n_pairs + 255) / 256, 256, 0, st>>>(ctx->pairs, ctx->bin, n_pairs, ctx->pairs_alt);
    HIGS_CUDA(ctx, cudaGetLastError());
    return HIGS_OK;
}

int launch_export_records(higs_ctx* ctx, int64_t N, cudaStream_t st)
{
    const int64_t n_slots = ((N + HIGS_CHUNK - 1) / HIGS_CHUNK) * HIGS_CHUNK;
    k_export_records<<<(unsigned)((n_slots + 255) / 256), 256, 0, st>>>(ctx->chunk_count, ctx->rec, ctx->bin, n_slots, ctx->rec_export);
    HIGS_CUDA(ctx, cudaGetLastError());
    return HIGS_OK;
}

int higs_binning_smem_setup(higs_ctx* ctx)
{
    int lcap_max = higs_part_lcap(ctx->n_chunks_max, ctx->n_sm);
    if (lcap_max < 96) lcap_max = 96;
    const int bytes = (int)(sizeof(uint32_t) * ((size_t)ctx->max_nm + 2 * (size_t)lcap_max + 1 + 2 * FILL_QCAP));
    if (bytes > 48 * 1024) {
        HIGS_CUDA(ctx, cudaFuncSetAttribute(k_fill, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    }
    const int plan_bytes = (int)(sizeof(uint32_t) * ((size_t)ctx->max_nm + 1));
    if (plan_bytes > 40 * 1024) HIGS_CUDA(ctx, cudaFuncSetAttribute(k_units, cudaFuncAttributeMaxDynamicSharedMemorySize, plan_bytes));
    return HIGS_OK;
}
