/*
 * higs.h -- C ABI of the B200-native HiGS forward render path
 * (arxiv/paper_2606_00352, "HiGS: A Hierarchical Rendering Architecture for Real-Time 3D
 * Gaussian Splatting"; citations are PAPER.md:<line> + section).
 *
 * One frame = the pipeline of PAPER.md:53 (Fig. 2) / PAPER.md:230-301 (section 4):
 *   a1 projection + cull + SH colour          PAPER.md:241-245 (4.2)
 *   a2 count   (gaussian x macro-tile hits)    PAPER.md:85-107 (3.2), 251 (4.3)
 *   a3 scan    (segment bounds, write bases)
 *   a4 fill    ((depth key, id) pairs)
 *   a5 segmented depth sort                    PAPER.md:109-117 (3.3), 259-276 (4.4)
 *   a6 batch schedule (units of <= B_r)        PAPER.md:81 (3.1)
 *   a7 macro-tile rasterizer                   PAPER.md:119-170 (3.4, Alg. 1-2), 278-284 (4.5)
 *   a8 post-blend merge, Eq. (1)
 * Every step runs in hand-written sm_100a kernels inside libhigs.so; there is no CPU fallback.
 *
 * Conventions
 *   - "device pointer" = memory of the CUDA device the context was created on, owned by the
 *     caller, contiguous fp32, never retained past the stream work of the call that got it.
 *   - "host pointer"  = ordinary (preferably pinned) host memory.
 *   - Inputs are *activated* 3DGS parameters: linear scales (> 0), opacities in [0,1],
 *     quaternions (w,x,y,z) not necessarily normalised, SH as [N][K][3], K = (degree+1)^2,
 *     in the convention of the public 3DGS models the paper renders.
 *   - Camera frame: +x right, +y down, +z forward; pixel (i,j) has its centre at (i+0.5,j+0.5).
 *   - Two-level grid: render tile 8x8 px; macro-tile = 8x4 render tiles = 64x32 px;
 *     macro-tile id m = my*ceil(W/64) + mx; tile in macro-tile t = ty*8 + tx.
 *   - All functions return HIGS_OK (0) or a negative higs_status; nothing throws.
 *   - A context is not thread-safe; use one context per host thread / stream.
 */
#ifndef HIGS_H
#define HIGS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HIGS_ABI_VERSION 3    /* 2: higs_lists.tile_load, higs_stats.tile, set_tile / scene_sort_spatial / scene_compress_sh / get_sh32; 3: set_macro_tile, sh32_encode_static */

#define HIGS_TILE        8      /* render tile edge, px  */
#define HIGS_MT_W        64     /* macro-tile width,  px (8 tiles)  */
#define HIGS_MT_H        32     /* macro-tile height, px (4 tiles)  */
#define HIGS_MT_TILES    32     /* M: render tiles per macro-tile  */
#define HIGS_BATCH_CAP   1024   /* B_r: gaussians per rasterizer work unit  */
#define HIGS_PART_BATCH  8192   /* B_p: gaussians per partitioning batch  */
#define HIGS_SORT_BLOCK  8192   /* largest segment sorted by one CTA */

typedef enum {
    HIGS_OK          = 0,
    HIGS_E_ARG       = -1,  /* null pointer, degree not in [0,3], W/H <= 0 or > max, N < 0 or > max */
    HIGS_E_CUDA      = -2,  /* a CUDA call failed; text via higs_last_error()                       */
    HIGS_E_CAPACITY  = -3,  /* the frame produced more pairs / units than the context was sized for;
                               detected on the device, nothing is written out of bounds, the frame's
                               image is then all zeros; reported by higs_get_stats / higs_get_lists  */
    HIGS_E_NOMEM     = -4   /* host or device allocation failed                                     */
} higs_status;

/* Pinhole camera.  HOST memory, copied at call time.  20 floats, no padding. */
typedef struct {
    float view[12];   /* row-major 3x4 world->camera [R|t]                                        */
    float fx, fy;     /* focal lengths, px                                                         */
    float cx, cy;     /* principal point, px                                                       */
    float near_z;     /* gaussians with z_cam <= near_z are culled (default 0.2)                   */
    float cam_pos[3]; /* world-space camera centre (= -R^T t), used only for the SH view direction */
} higs_camera;

typedef struct higs_ctx higs_ctx;

/* Frame statistics.  HOST struct filled by higs_get_stats (synchronises the render stream). */
typedef struct {
    int64_t n_gaussians;     /* N of the last render                                              */
    int64_t n_visible;       /* gaussians surviving the cull                                      */
    int64_t n_pairs;         /* (gaussian, macro-tile) pairs                  PAPER.md:97 Table 1 */
    int64_t n_units;         /* N_R = sum_m ceil(n_m / B_r) rasterizer units         */
    int64_t max_segment;     /* largest per-macro-tile list                                       */
    int64_t n_oversize;      /* segments longer than HIGS_SORT_BLOCK (overflow path)*/
    int32_t n_mt_x, n_mt_y;  /* macro-tile grid                                                   */
    int32_t batch_cap;       /* B_r in effect                                                     */
    int32_t overflow;        /* 1 if the frame hit HIGS_E_CAPACITY                                */
    int32_t n_launches;      /* kernels the library enqueued for the last frame (memsets excluded) */
    int32_t tile;            /* render-tile edge in effect (8 or 16)                               */
    int64_t n_evals;         /* pixel-gaussian evaluations executed by the rasterizer; only
                                counted when HIGS_FLAG_COUNT_EVALS is set, else 0                 */
    int64_t n_tile_pairs;    /* (gaussian, render tile) pairs that passed the inline visibility
                                test; only with HIGS_FLAG_COUNT_EVALS                             */
    /* per-stage device time of the last frame, ms; only with HIGS_FLAG_STAGE_TIMERS, else 0     */
    float ms_project, ms_count, ms_scan, ms_fill, ms_sort, ms_raster, ms_merge, ms_total;
} higs_stats;

/* The integer lists of the last frame (O-LIST).  DEVICE pointers owned by the context, valid
 * until the next render on it.  higs_get_lists synchronises the render stream. */
typedef struct {
    int64_t n_pairs, n_units;
    int32_t n_mt;                    /* N_M                                                       */
    const uint32_t* mt_count;        /* [N_M]     pairs per macro-tile                            */
    const uint32_t* mt_offset;       /* [N_M+1]   exclusive prefix sum = segment bounds           */
    const uint32_t* batch_offset;    /* [N_M+1]   exclusive prefix sum of ceil(n_m/B_r)           */
    const uint64_t* pairs;           /* [n_pairs] (key << 32 | id), each segment ascending        */
    const uint32_t* unit_active;     /* [n_units] 32-bit active-tile mask per unit  */
    const uint32_t* tile_load;       /* [N_M][32] per render tile: gaussians that passed the inline visibility test, summed over
                                        the macro-tile's units - the load map of PAPER.md:9 (Fig. 1); only filled with
                                        HIGS_FLAG_COUNT_EVALS (use HIGS_FLAG_NO_XBATCH_CUT as well for the uncut load)     */
} higs_lists;

/* Per-gaussian records of the last frame.  DEVICE pointers owned by the context. */
typedef struct {
    int64_t n;
    const uint32_t* valid_bits;      /* [ceil(N/32)] bit (i & 31) of word i/32 = gaussian i kept  */
    const float*    rec;             /* [N][16] mux, muy, A, B2, C, tau, log2(o), r, g, b, bits(key), (2 words
                                        internal), a, b, c; rows of culled gaussians are not written
                                        (a,b,c = 2D covariance, A,B2,C = conic)       */
} higs_records;

#define HIGS_FLAG_STAGE_TIMERS  1u   /* record CUDA events around every stage                     */
#define HIGS_FLAG_COUNT_EVALS   2u   /* rasterizer counts evaluations (slower; for the roofline)  */
#define HIGS_FLAG_NO_XBATCH_CUT 4u   /* disable the cross-batch saturation cut-off:
                                        every unit then rasterizes every tile it touches          */
#define HIGS_FLAG_FP16          16u  /* fp16 data path: Cholesky conics prescaled for exp2, positions in
                                        tile units relative to the macro-tile centre, half2 blending, fp16 RGBT partials (16 KB per
                                        unit).  Culling, macro-tile lists and the depth sort are the same pinned fp32 code, so the
                                        integer lists stay bit-exact; the image is accepted by PSNR against the fp32 oracle.  In
                                        this mode higs_get_records returns valid_bits only (rec rows are not written).        */
#define HIGS_FLAG_SH32          32u  /* resident-scene renders (higs_render_view*) read the 32-byte SH codes made by
                                        higs_scene_compress_sh instead of the 192-byte fp32 rows              */
#define HIGS_FLAG_RADIX_SORT    8u   /* tier kernels run the block radix sort (8-bit passes) instead of
                                        the block merge sort; same result, measured slower on B200 (profiles/)   */

/* Create a context on CUDA device `device` and preallocate all scratch (PAPER.md:83, 284:
 * "preallocated up front").  max_pairs bounds N_pairs (<= 2^31-1; 0 selects 4*max_gaussians + 65536).
 * Device memory taken: ~120 B/gaussian (64-B and 32-B records, 16-B bin record) + 17 B/pair + 32 KB per unit
 * (units <= N_M + max_pairs/1024; 128 KB per unit after higs_set_tile(ctx, 16)). */
int higs_create(higs_ctx** out, int device, int64_t max_gaussians, int max_W, int max_H, int64_t max_pairs);
void higs_destroy(higs_ctx* ctx);

/* Runtime knobs: flags (HIGS_FLAG_*) and the rasterizer batch cap B_r in [1, 1024]
 * (tests use small B_r to force many batches per macro-tile; the paper's value is 1024). */
int higs_set_flags(higs_ctx* ctx, uint32_t flags);
int higs_set_batch_cap(higs_ctx* ctx, int batch_cap);
/* Render-tile edge in pixels: 8 (default) or 16 (the variant of Table 2).  The macro-tile
 * stays 8 x 4 render tiles, i.e. 64 x 32 or 128 x 64 px, and m = my*ceil(W/(8 tile)) + mx.  Reallocates the per-unit
 * buffers (synchronises the device). */
int higs_set_tile(higs_ctx* ctx, int tile);
/* Macro-tile shape in render tiles (shape sweep): 8 x 4 (default), 4 x 8 or 16 x 2; always
 * HIGS_MT_TILES = 32 tiles, m = my*ceil(W/(tiles_x tile)) + mx, tile t of a macro-tile at column t % tiles_x, row t / tiles_x.
 * Shapes other than 8 x 4 exist on the fp32 path with 8 x 8 tiles only: HIGS_E_ARG with tile 16, and a frame rendered with
 * HIGS_FLAG_FP16 set returns HIGS_E_ARG (the fp16 path's coordinate range is that of the 8 x 4 macro-tile). */
int higs_set_macro_tile(higs_ctx* ctx, int tiles_x, int tiles_y);

/* Render one frame.  All array arguments are DEVICE pointers:
 *   means [N][3], scales [N][3], quats [N][4], opacities [N], sh [N][(degree+1)^2][3],
 *   out_rgb [H][W][3] fp32, black background, no clamp / gamma.
 * cam is a HOST pointer.  cuda_stream is a cudaStream_t (NULL = legacy default stream).
 * Only enqueues work: no host synchronisation, no allocation, so the call may
 * be captured into a CUDA graph.  N = 0 is valid (image = 0). */
int higs_render(higs_ctx* ctx, const float* means, const float* scales, const float* quats,
                const float* opacities, const float* sh, int degree, int64_t N,
                const higs_camera* cam, int W, int H, float* out_rgb, void* cuda_stream);

/* Same frame with HOST buffers: uploads the arrays, renders, downloads the image into the host buffer out_rgb and
 * synchronises.  Staging device buffers are owned by the context and shared with the resident scene, which this call
 * invalidates (higs_render_view returns HIGS_E_ARG until the next higs_scene_upload).
 * If sh is page-locked host memory the device can address (cudaHostAlloc, cudaHostRegister, torch pin_memory()), the SH
 * array is NOT uploaded: the projection kernel (a1) reads the rows of the gaussians that survive the cull directly from
 * host memory, whole warps copying 16 contiguous bytes per lane (the cull keeps fewer than half of the gaussians and the
 * SH rows are 4/5 of a scene's bytes).  Results are identical bit for bit to the uploaded path. */
int higs_render_host(higs_ctx* ctx, const float* means, const float* scales, const float* quats,
                     const float* opacities, const float* sh, int degree, int64_t N,
                     const higs_camera* cam, int W, int H, float* out_rgb);

/* Resident-scene path for view loops: upload once (HOST pointers), then per view copy the camera
 * in and the image out (HOST pointer out_rgb, pinned for full speed) and synchronise. */
int higs_scene_upload(higs_ctx* ctx, const float* means, const float* scales, const float* quats,
                      const float* opacities, const float* sh, int degree, int64_t N);
int higs_render_view_host(higs_ctx* ctx, const higs_camera* cam, int W, int H, float* out_rgb);
/* Store the resident scene in a spatially coherent order: its gaussians are sorted along a Morton curve of their means
 * (10 bits per axis over the bounding box, ties by index).  The order of the gaussians is part of a scene - the ids in the
 * lists and the (depth key, id) tie-break refer to the new order - so the permutation is returned: host_perm[i] (HOST, [N],
 * may be NULL) = index in the uploaded arrays of the gaussian now at i.  Rendering the reordered scene is rendering the
 * uploaded arrays permuted that way.  Why: survivors of the cull become contiguous, so the projection kernel's scattered
 * 192-byte SH reads stop over-fetching.  Needs N <= max_pairs (it uses the frame's sort scratch).
 * Synchronises; discards SH codes made before it. */
int higs_scene_sort_spatial(higs_ctx* ctx, uint32_t* host_perm);
/* 32-byte SH codec (section 4.2): encode the resident scene's degree-3 SH rows on the device - YCoCg-R,
 * square-root gamma quantisation (6 bits luma, 4 bits chroma; 16 / 15 / 15 bits for the DC basis), per-(basis, channel)
 * scales = the 99.9th percentile of |value| over the scene (the maximum for DC); bit layout in DESIGN.md (Q20).  With
 * HIGS_FLAG_SH32 set, higs_render_view / higs_render_view_host then decode the codes inline in the projection kernel.
 * Synchronises.  HIGS_E_ARG if no degree-3 scene is resident.  higs_scene_upload discards the codes. */
int higs_scene_compress_sh(higs_ctx* ctx);
/* Copies the codes ([N][32] bytes) and the scale table ([16][3] floats: Y, Co, Cg) to HOST memory (either may be NULL). */
int higs_get_sh32(higs_ctx* ctx, uint8_t* host_codes, float* host_scales);

/* The same encoder for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no context, no cudaMalloc / cudaFree, no host synchronisation; it only enqueues kernels and one 192-byte
 * device-to-device copy on cuda_stream, on the CURRENT device.  All pointers are DEVICE pointers owned by the caller:
 *   d_sh     [N][16][3] fp32 degree-3 SH rows (input),
 *   d_codes  [N][32] bytes (output, 16-byte aligned), d_scales [16][3] fp32 (output: Y, Co, Cg scale per basis).
 * Bytes and scales are identical to higs_scene_compress_sh + higs_get_sh32 on the same rows.  N = 0 writes scales of 1.
 * The work area of the percentile selection (49,920 bytes) is a file-scope device array inside the library: every GPU that
 * loads the library holds it until the process exits.  It is SHARED by all calls and keeps the last call's contents (each
 * call clears what must start at zero): calls that overlap on the GPU - two streams, two host threads - race; serialise them.
 * Errors: HIGS_E_CAPACITY if N > HIGS_SH32_STATIC_MAX_N (the work area's counters are 32-bit), HIGS_E_ARG for null or
 * misaligned pointers or N < 0, HIGS_E_CUDA; text of this thread's last failure: higs_sh32_encode_static_error(). */
#define HIGS_SH32_STATIC_MAX_N 1073741824ll   /* 2^30 gaussians */
int higs_sh32_encode_static(const float* d_sh, int64_t N, uint8_t* d_codes, float* d_scales, void* cuda_stream);
const char* higs_sh32_encode_static_error(void);
/* Resident-scene path with a DEVICE image (no download, no synchronisation). */
int higs_render_view(higs_ctx* ctx, const higs_camera* cam, int W, int H, float* out_rgb, void* cuda_stream);

int higs_get_stats(higs_ctx* ctx, higs_stats* out);
int higs_get_lists(higs_ctx* ctx, higs_lists* out);
int higs_get_records(higs_ctx* ctx, higs_records* out);

/* Stage-isolation entry point for tests ("teacher forcing", a5 alone): sorts every segment
 * [seg_offset[s], seg_offset[s+1]) of the DEVICE array pairs (n_seg segments, 64-bit
 * (key << 32 | id) items) ascending, in place, with the frame's own sort kernels. */
int higs_sort_segments(higs_ctx* ctx, uint64_t* pairs, const uint32_t* seg_offset, int32_t n_seg,
                       void* cuda_stream);

/* Utility: synchronise the last render stream and copy `bytes` from a DEVICE pointer handed out by
 * higs_get_lists / higs_get_records into HOST memory. */
int higs_download(higs_ctx* ctx, const void* device_src, void* host_dst, uint64_t bytes);

const char* higs_strerror(int status);
const char* higs_last_error(higs_ctx* ctx);   /* text of the last HIGS_E_CUDA on this context */
int higs_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HIGS_H */
