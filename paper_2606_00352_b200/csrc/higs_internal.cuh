// higs_internal.cuh -- context layout, constants and small device helpers shared by the
// kernels of libhigs.so.  Nothing here is visible through the C ABI (include/higs.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/higs.h"

#define HIGS_EPS_T      1e-4f        // transmittance threshold, reading Q1
#define HIGS_ALPHA_MAX  0.99f
#define HIGS_HDR_WORDS  64           // 32-bit words reserved for the FrameHeader at the head of its block
#define HIGS_MAX_NM     32768        // macro-tiles per frame the shared-memory histograms are sized for
#define HIGS_N_TIERS    4            // block-sort tiers, capacities 1024 / 2048 / 4096 / 8192
#define HIGS_CHUNK      128          // consecutive ids projected by one warp; survivors are stored densely per chunk
#define HIGS_MERGE_TILE 4096         // output items per merge-path tile (overflow path)
#define HIGS_SPLIT_TILE 2048         // items per CTA pass of the bucket count / scatter kernels
#define HIGS_BUCKET_TARGET 1536      // mean items per depth bucket of an oversize segment
#define HIGS_MAX_SPLIT  256          // most buckets per oversize segment (splitters live in shared memory)

// ---- per-frame device header: every data-dependent size lives here, never on the host ----------
struct FrameHeader {
    uint32_t n_pairs;          // sum of mt_count (0 when overflow)
    uint32_t n_units;          // N_R (0 when overflow)
    uint32_t overflow;         // pairs or units exceeded the preallocated capacity
    uint32_t max_segment;
    uint32_t n_oversize;       // segments > HIGS_SORT_BLOCK: split into depth buckets first (sort.cu)
    uint32_t n_split_tiles;    // sum over oversize segments of ceil(n / HIGS_SPLIT_TILE)
    uint32_t n_buckets;        // buckets of all oversize segments
    uint32_t max_levels;       // merge levels needed by the longest fallback bucket
    uint32_t pad0;
    uint32_t n_sort_jobs[2][HIGS_N_TIERS];   // [0] whole segments, [1] buckets of oversize segments
    uint32_t sort_cursor[2][HIGS_N_TIERS];   // work counters (persistent kernels)
    uint32_t split_cursor[3];  // k_oversize: work items claimed per phase (segments, tiles, tiles)
    uint32_t split_done[3];    // k_oversize: work items finished per phase
    uint32_t raster_cursor;
    uint32_t merge_barrier;    // software grid barrier of the merge kernel
    uint32_t n_visible;
    uint32_t proj_cursor;      // chunk counter of the projection kernel
    uint32_t part_list_cursor; // entries of part_list handed out
    uint32_t pad1;
    unsigned long long fallback_pack;   // (buckets that still exceed HIGS_SORT_BLOCK << 32 | their merge tiles): block sort + merge levels
    unsigned long long n_evals;
    unsigned long long n_tile_pairs;
};

struct SortJob   { uint32_t start, len, flags, pad; };             // flags bit 0: write the sorted run to the alternate buffer, bit 1: read it there
struct OverSeg   { uint32_t start, len, levels, tile_base; };     // a fallback bucket and its merge plan
struct SplitSeg  { uint32_t start, len, nb, bucket_base, tile_base, items_before, oversample, pad; };   // an oversize segment and its bucket plan

// camera + frame constants handed to the kernels by value
struct FrameParams {
    float V[12];
    float fx, fy, cx, cy, near_z;
    float cam[3];
    int   W, H;
    int   n_mx, n_my, n_m;
    int   degree;
    int   batch_cap;
    int   tile;                // render-tile edge, 8 or 16
    int   mt_tx, mt_ty;        // render tiles per macro-tile in x and y: 8 x 4, or 4 x 8 / 16 x 2 (higs_set_macro_tile)
    float limx, limy;          // (0.65 W) / fx, (0.65 H) / fy: the clamp of the Jacobian (N-PROJ step 3), the same for every gaussian
    uint32_t flags;
    uint32_t max_pairs, max_units;
};

struct ShScales { float s[48]; };   // 32-byte SH code: scale of (basis k, channel Y / Co / Cg) at [k*3 + c], passed to kernels by value

struct higs_ctx {
    int device;
    int64_t max_gaussians;
    int max_W, max_H, max_nm;
    int64_t max_pairs, max_units;
    int n_part_max;            // partition CTAs (= histogram rows): n_sm x resident k_project CTAs
    int64_t n_chunks_max;
    int n_sm;
    uint32_t flags;
    int batch_cap;
    int tile;                  // render-tile edge in effect (8 or 16)
    int mt_tx, mt_ty;          // macro-tile shape in render tiles (8 x 4 unless higs_set_macro_tile changed it)
    uint32_t touch_max_pairs;  // k_plan pre-writes the pair list when it has at most this many items (3/4 of L2)
    // scratch (device)
    uint32_t* valid_bits;      // [ceil(maxN/32)]
    float4*   rec;             // [slots][4]  mux,muy,A,B2 | C,tau,log2o,r | g,b,a,b | c,bits(key),id,-   (64 B; the rasterizer gathers the
                               //             first 48 B).  A slot is the dense position of a surviving gaussian: survivor k of the
                               //             HIGS_CHUNK-id chunk c sits at c*HIGS_CHUNK + k (monotone in the id)
    uint4*    rec16;           // [slots][2]  fp16 data path (HIGS_FLAG_FP16): mux, muy (fp32) | half2 (l0', l1') | half2 (l2', o) ;
                               //             half2 (r, g) | half2 (b, 0) | - | -   (32 B = one sector)
    uint4*    bin;             // [slots]     bits(key), span descriptor lo, hi, id   (16 B, read by fill)
    uint32_t* chunk_count;     // [chunks]    survivors of the chunk
    uint32_t* part_list;       // [chunks]    chunk ids grouped by the partition CTA that claimed them
    uint2*    part_desc;       // [N_B]       (first entry, entries) of each partition CTA in part_list
    float*    rec_export;      // [maxN][16]  test-facing copy indexed by gaussian id, allocated by the first higs_get_records
    uint32_t* hist;            // [N_B][N_M]
    uint32_t* hdr_block;       // one allocation, zeroed per frame: FrameHeader (HIGS_HDR_WORDS words) | mt_count | mt_fill
    uint32_t* mt_count;        // [max_nm+1]  pairs per macro-tile, accumulated by the projection CTAs
    uint32_t* mt_fill;         // [max_nm+1]  pairs of the macro-tile handed out so far (fill pass)
    uint32_t* mt_offset;       // [max_nm+1]
    uint32_t* batch_offset;    // [max_nm+1]
    uint32_t* unit_mt;         // [max_units] macro-tile of unit u
    uint32_t* unit_active;     // [max_units] 32-bit active-tile mask per unit
    uint32_t* unit_order;      // [max_units] units in the order the rasterizer claims them: batch index j major
    uint32_t* level_hist;      // [max_units+2] scratch of k_plan: macro-tiles per batch count, then level cursors
    uint32_t* level_cur;       // [max_units+2] write cursor of each level in unit_order
    unsigned long long* pairs; // [max_pairs]
    unsigned long long* pairs_alt; // [max_pairs] ping-pong buffer of the overflow merge
    SortJob*  sort_jobs;       // [2][HIGS_N_TIERS][max_jobs]  list 0: whole segments, list 1: buckets
    int64_t   max_jobs;
    OverSeg*  over_segs;       // [max_over]   fallback buckets (merge path)
    SplitSeg* split_segs;      // [max_over]   oversize segments
    int64_t   max_over;
    unsigned long long* splitters;   // [max_buckets]  bucket b of a segment holds items in [splitter[b-1], splitter[b])
    uint32_t* bucket_count;    // [max_buckets]
    uint32_t* bucket_cursor;   // [max_buckets]  write position of the scatter pass
    uint8_t*  bucket_id;       // [max_pairs]  bucket of every item of an oversize segment (phase 1 of k_oversize writes, phase 2 reads)
    int64_t   max_buckets;
    float4*   partial;         // [max_units][32 tiles][64 px] (r,g,b,T)
    unsigned long long* cut_word;  // [max_nm][32] cross-batch cut: (k << 32 | sum of the terms of batches 0 .. k-1), a cached prefix (raster.cu)
    int*      cut_term;        // [max_units][32] log2(largest transmittance the unit left in the tile) x 1024, rounded towards zero, minus 1;
                               //             0 = not published.  Both are zeroed every frame by k_fill
    uint32_t* tile_load;       // [max_nm][32] gaussians that passed the per-tile visibility test, summed over the macro-tile's units;
                               //             only with HIGS_FLAG_COUNT_EVALS (zeroed by k_fill)
    FrameHeader* hdr;          // device
    FrameHeader* hdr_host;     // pinned
    // resident scene / host staging
    float *s_means, *s_scales, *s_quats, *s_opac, *s_sh, *s_img;
    uint4* s_sh32;             // [s_n][2] 32-byte SH codes of the resident scene (higs_scene_compress_sh), or null
    int64_t s_sh32_cap;
    bool s_sh32_valid;
    float sh32_scales_host[48];
    uint32_t* sh32_work;       // device scratch of the encoder: hist [48][256] | prefix [48] | rank lo/hi [48][2] | scales [48]
    int64_t s_cap_n, s_cap_sh, s_img_cap;
    int64_t s_n; int s_degree;
    // last frame
    int64_t last_n; int last_W, last_H, last_nm; int last_mx, last_my;
    cudaStream_t last_stream;
    cudaStream_t own_stream;
    cudaStream_t aux_stream[4];   // forked from the render stream for the sort tiers
    cudaEvent_t ev_fork, ev_fork2, ev_join[4];
    cudaEvent_t ev[9];
    bool timers_valid;
    int n_launches;            // kernels enqueued by the current / last frame
    // resident CTAs per SM of the persistent kernels (occupancy queried at create time, per device)
    bool proj_staged_ok;                                   // the staged-row projection variants fit in shared memory
    int raster_ctas_per_sm[2][2], merge_ctas_per_sm, over_ctas_per_sm, tier_ctas_per_sm[2][HIGS_N_TIERS];   // tiers: [0] radix, [1] merge sort
    char err[512];
};

#define HIGS_CUDA(ctx, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
    return HIGS_E_CUDA; } } while (0)

// every kernel launch site of a frame calls this right after the <<<>>> (stats: n_launches)
#define HIGS_LAUNCHED(ctx) do { HIGS_CUDA(ctx, cudaGetLastError()); ++(ctx)->n_launches; } while (0)

// ---- programmatic dependent launch (PDL): a kernel launched with launch_pdl right behind another kernel on the same
// stream may be scheduled while its predecessor drains; it must call pdl_wait() before touching anything the
// predecessor wrote, and calls pdl_trigger() so that its own successor can be scheduled early in turn.
__device__ __forceinline__ void pdl_wait()    { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KP, typename... A>
inline cudaError_t launch_pdl(void (*kernel)(KP...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KP(args)...);
}

// ---- launch entry points, one per pipeline step (defined in the .cu files) ----------------------
// sh_mode of launch_project: where the SH coefficients come from
#define HIGS_SH_ROWS   0        /* fp32 rows, device memory */
#define HIGS_SH_CODES  1        /* 32-byte codes of the resident scene */
#define HIGS_SH_STAGED 2        /* fp32 rows in mapped host memory, copied to shared memory by whole warps */
int launch_project(higs_ctx*, const FrameParams&, const float* means, const float* scales, const float* quats,
                   const float* opac, const float* sh, int sh_mode, int64_t N, cudaStream_t);
int launch_sh32_encode(higs_ctx*, cudaStream_t);
int launch_scene_sort(higs_ctx*, uint32_t* d_perm, cudaStream_t);
int higs_part_grid(const higs_ctx*, int64_t N);
int higs_part_lcap(int64_t n_chunks, int grid);
int launch_binning(higs_ctx*, const FrameParams&, int64_t N, cudaStream_t, cudaEvent_t ev_count, cudaEvent_t ev_scan);
int launch_sort(higs_ctx*, const FrameParams&, cudaStream_t);
int launch_units(higs_ctx*, const FrameParams&, cudaStream_t);
int launch_sort_only(higs_ctx*, unsigned long long* pairs, const uint32_t* seg_offset, int n_seg, cudaStream_t);
int launch_raster(higs_ctx*, const FrameParams&, cudaStream_t);
int launch_merge(higs_ctx*, const FrameParams&, float* out_rgb, cudaStream_t);

// ---- bounds checks of a debug build (python -m paper_2606_00352_b200.build --debug-bounds): compute-sanitizer is not
// available on the GPU pool, so the indexed writes of the frame carry device asserts that the test suite runs through once
// per round (profiles/r02_sanitizer.md).  A failed assert traps: the next CUDA call of the test fails loudly.
#ifdef HIGS_DEBUG_BOUNDS
#include <assert.h>
#define HIGS_ASSERT(c) assert(c)
#else
#define HIGS_ASSERT(c) ((void)0)
#endif

// ---- device helpers ----------------------------------------------------------------------------
__device__ __forceinline__ float clampf_(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

// Threshold of the bounding box and of the macro-tile row scan (N-PROJ step 9):
//   tau_s = tau * fma(cond, 2^-20, 1),  cond = (a c) / det,  det = fma(a, c, -(b b)).
// The fp32 pixel test q <= tau is evaluated on the conic, whose cross term cancels for elongated gaussians
// (PAPER.md:180-226), so the region it accepts leaves the covariance ellipse of tau by ~3 * 2^-24 * cond in tau;
// everything that must be conservative with respect to the pixel test runs on tau_s.  Pinned: same ops as the oracle.
__device__ __forceinline__ float tau_scan(float a, float b, float c, float tau)
{
    const float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
    const float cond = __fmul_rn(__fmul_rn(a, c), __frcp_rn(det));
    return __fmul_rn(tau, __fmaf_rn(cond, 9.5367431640625e-07f, 1.0f));
}

// The row scan of DESIGN.md section 3 (N-SCAN): exact x-extent of the threshold ellipse
// {q <= tau_s} inside each row band of a grid of cw x ch cells, clipped to [0,W] x [0,H]; the caller passes
// tau_s = tau_scan(a, b, c, tau).
// Every operation is a single correctly rounded fp32 op in the written order (no contraction):
// the set of cells it yields is part of the bit-exact contract with the oracle.
struct RowScan {
    float mux, muy, tau, hx, hy, boc, rc, sdet, yR, nyR, ytop, ybot;
    int r0, r1;
    // tau_ = tau_s.  LEAN: cell sizes are powers of two, so x * (1 / size) is the correctly rounded x / size of the pinned
    // sequence at the price of one multiply, and rcp.rn(c) is the correctly rounded 1 / c: same bits, fewer instructions.
    // The lean form is used where it was measured faster (the projection kernel reading SH codes, which is bound by issue);
    // on the DRAM-bound fp32-SH kernel it was slower (0.286 against 0.268 ms), so that one keeps the divisions.
    template <bool LEAN = false>
    __device__ __forceinline__ void init(float mux_, float muy_, float a, float b, float c, float tau_, float fch, int ncy)
    {
        mux = mux_; muy = muy_; tau = tau_;
        hx = __fsqrt_rn(__fmul_rn(tau, a));
        hy = __fsqrt_rn(__fmul_rn(tau, c));
        ytop = __fsub_rn(muy, hy); ybot = __fadd_rn(muy, hy);
        const float rfch = 1.0f / fch;
        r0 = (int)clampf_(floorf(LEAN ? __fmul_rn(ytop, rfch) : __fdiv_rn(ytop, fch)), 0.0f, (float)(ncy - 1));
        r1 = (int)clampf_(floorf(LEAN ? __fmul_rn(ybot, rfch) : __fdiv_rn(ybot, fch)), 0.0f, (float)(ncy - 1));
        boc = __fdiv_rn(b, c);
        rc = LEAN ? __frcp_rn(c) : __fdiv_rn(1.0f, c);
        sdet = fmaxf(0.0f, __fmaf_rn(-b, boc, a));
        yR = __fmul_rn(b, __fsqrt_rn(__fdiv_rn(tau, a)));
        nyR = -yR;
    }
    // columns [m0, m1] of row r; returns false when the row is not touched
    template <bool LEAN = false>
    __device__ __forceinline__ bool row(int r, float fcw, float fch, float fW, float fH, int ncx, int& m0, int& m1) const
    {
        const float rfcw = 1.0f / fcw;
        float y0 = __fmul_rn((float)r, fch);
        float y1 = fminf(__fmul_rn((float)(r + 1), fch), fH);
        float ylo = __fsub_rn(fmaxf(y0, ytop), muy);
        float yhi = __fsub_rn(fminf(y1, ybot), muy);
        if (!(yhi >= ylo)) return false;
        float rlo = __fsqrt_rn(fmaxf(0.0f, __fmul_rn(sdet, __fmaf_rn(-__fmul_rn(ylo, ylo), rc, tau))));
        float rhi = __fsqrt_rn(fmaxf(0.0f, __fmul_rn(sdet, __fmaf_rn(-__fmul_rn(yhi, yhi), rc, tau))));
        float xmax = (ylo <= yR && yR <= yhi) ? hx : fmaxf(__fmaf_rn(boc, ylo, rlo), __fmaf_rn(boc, yhi, rhi));
        float xmin = (ylo <= nyR && nyR <= yhi) ? -hx : fminf(__fmaf_rn(boc, ylo, -rlo), __fmaf_rn(boc, yhi, -rhi));
        xmin = __fadd_rn(xmin, mux); xmax = __fadd_rn(xmax, mux);
        if (!(xmax > 0.0f) || !(xmin < fW)) return false;
        m0 = (int)clampf_(floorf(LEAN ? __fmul_rn(xmin, rfcw) : __fdiv_rn(xmin, fcw)), 0.0f, (float)(ncx - 1));
        m1 = (int)clampf_(floorf(LEAN ? __fmul_rn(xmax, rfcw) : __fdiv_rn(xmax, fcw)), 0.0f, (float)(ncx - 1));
        return true;
    }
};
