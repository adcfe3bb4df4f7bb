// api.cu -- the C ABI of include/higs.h: context, frame orchestration, stats.  Host code only
// enqueues kernels; every data-dependent size stays on the device.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "higs_internal.cuh"

int higs_binning_smem_setup(higs_ctx*);
int higs_project_smem_setup(higs_ctx*);
int higs_sort_smem_setup(higs_ctx*);
int higs_raster_setup(higs_ctx*);
int launch_export_lists(higs_ctx*, uint32_t n_pairs, cudaStream_t);      // binning.cu: pairs (key, slot) -> pairs_alt (key, id)
int launch_export_records(higs_ctx*, int64_t N, cudaStream_t);           // binning.cu: rec[slot] -> rec_export[id]

namespace {

template <typename T>
int dev_alloc(higs_ctx* ctx, T** p, size_t count)
{
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, (count ? count : 1) * sizeof(T));
    if (e != cudaSuccess) {
        snprintf(ctx->err, sizeof(ctx->err), "cudaMalloc(%zu B): %s", count * sizeof(T), cudaGetErrorString(e));
        cudaGetLastError();
        return HIGS_E_NOMEM;
    }
    *p = static_cast<T*>(q);
    return HIGS_OK;
}

template <typename T> void dev_free(T*& p) { if (p) cudaFree(p); p = nullptr; }

int alloc_unit_buffers(higs_ctx* ctx)
{
    dev_free(ctx->unit_mt); dev_free(ctx->unit_active); dev_free(ctx->partial);
    dev_free(ctx->unit_order); dev_free(ctx->level_hist); dev_free(ctx->level_cur); dev_free(ctx->cut_term);
    ctx->max_units = ctx->max_nm + (ctx->max_pairs + ctx->batch_cap - 1) / ctx->batch_cap + 1;
    int rc;
    if ((rc = dev_alloc(ctx, &ctx->unit_mt, (size_t)ctx->max_units))) return rc;
    if ((rc = dev_alloc(ctx, &ctx->unit_active, (size_t)ctx->max_units))) return rc;
    if ((rc = dev_alloc(ctx, &ctx->unit_order, (size_t)ctx->max_units))) return rc;
    if ((rc = dev_alloc(ctx, &ctx->level_hist, (size_t)ctx->max_units + 2))) return rc;
    if ((rc = dev_alloc(ctx, &ctx->level_cur, (size_t)ctx->max_units + 2))) return rc;
    if ((rc = dev_alloc(ctx, &ctx->partial, (size_t)ctx->max_units * HIGS_MT_TILES * ctx->tile * ctx->tile))) return rc;   // float4 per pixel
    if ((rc = dev_alloc(ctx, &ctx->cut_term, (size_t)ctx->max_units * HIGS_MT_TILES))) return rc;
    return HIGS_OK;
}

int check_frame_args(higs_ctx* ctx, int degree, int64_t N, const higs_camera* cam, int W, int H, const void* out)
{
    if (!ctx || !cam || !out) return HIGS_E_ARG;
    if (degree < 0 || degree > 3) return HIGS_E_ARG;
    if (N < 0 || N > ctx->max_gaussians) return HIGS_E_ARG;
    if (W <= 0 || H <= 0 || W > ctx->max_W || H > ctx->max_H) return HIGS_E_ARG;
    const int mw = 8 * ctx->tile, mh = 4 * ctx->tile;
    const int64_t nm = (int64_t)((W + mw - 1) / mw) * ((H + mh - 1) / mh);
    if (nm > ctx->max_nm) return HIGS_E_ARG;
    return HIGS_OK;
}

int render_impl(higs_ctx* ctx, const float* means, const float* scales, const float* quats, const float* opac,
                const float* sh, int degree, int64_t N, const higs_camera* cam, int W, int H, float* out_rgb,
                cudaStream_t st, int sh_mode = HIGS_SH_ROWS)
{
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    FrameParams P;
    memcpy(P.V, cam->view, sizeof(P.V));
    P.fx = cam->fx; P.fy = cam->fy; P.cx = cam->cx; P.cy = cam->cy; P.near_z = cam->near_z;
    memcpy(P.cam, cam->cam_pos, sizeof(P.cam));
    P.W = W; P.H = H;
    P.tile = ctx->tile; P.mt_tx = ctx->mt_tx; P.mt_ty = ctx->mt_ty;
    if (P.mt_tx != 8 && (P.tile != 8 || (ctx->flags & HIGS_FLAG_FP16))) return HIGS_E_ARG;   // other shapes: fp32 path, 8 x 8 tiles
    { const float tx = 0.65f * (float)W, ty = 0.65f * (float)H; P.limx = tx / P.fx; P.limy = ty / P.fy; }   // one rounding per op, as N-PROJ writes it
    P.n_mx = (W + P.mt_tx * P.tile - 1) / (P.mt_tx * P.tile); P.n_my = (H + P.mt_ty * P.tile - 1) / (P.mt_ty * P.tile); P.n_m = P.n_mx * P.n_my;
    if (P.n_m > ctx->max_nm) return HIGS_E_ARG;
    P.degree = degree; P.batch_cap = ctx->batch_cap; P.flags = ctx->flags;
    P.max_pairs = (uint32_t)ctx->max_pairs; P.max_units = (uint32_t)ctx->max_units;
    const bool timers = (ctx->flags & HIGS_FLAG_STAGE_TIMERS) != 0;
    cudaEvent_t* ev = ctx->ev;
    int rc;

    ctx->n_launches = 0;
    // one memset: frame header, per-macro-tile pair counts and fill cursors (one allocation)
    HIGS_CUDA(ctx, cudaMemsetAsync(ctx->hdr, 0, sizeof(uint32_t) * (HIGS_HDR_WORDS + 2 * ((size_t)ctx->max_nm + 1)), st));
    if (timers) cudaEventRecord(ev[0], st);
    if ((rc = launch_project(ctx, P, means, scales, quats, opac, sh, sh_mode, N, st))) return rc;
    if (timers) cudaEventRecord(ev[1], st);
    if ((rc = launch_binning(ctx, P, N, st, timers ? ev[2] : nullptr, timers ? ev[3] : nullptr))) return rc;
    if (timers) cudaEventRecord(ev[4], st);
    if ((rc = launch_sort(ctx, P, st))) return rc;
    if (timers) cudaEventRecord(ev[5], st);
    if ((rc = launch_raster(ctx, P, st))) return rc;
    if (timers) cudaEventRecord(ev[6], st);
    if ((rc = launch_merge(ctx, P, out_rgb, st))) return rc;
    if (timers) cudaEventRecord(ev[7], st);
    ctx->timers_valid = timers;
    ctx->last_n = N; ctx->last_W = W; ctx->last_H = H; ctx->last_nm = P.n_m; ctx->last_mx = P.n_mx; ctx->last_my = P.n_my;
    ctx->last_stream = st;
    return HIGS_OK;
}

int fetch_header(higs_ctx* ctx)
{
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    HIGS_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
    HIGS_CUDA(ctx, cudaMemcpy(ctx->hdr_host, ctx->hdr, sizeof(FrameHeader), cudaMemcpyDeviceToHost));
    return HIGS_OK;
}

// Device copies of a scene: the four small arrays grow together (s_cap_n gaussians), the SH array on its own
// (s_cap_sh floats; need_sh = false when the rows stay in mapped host memory).
int ensure_scene_capacity(higs_ctx* ctx, int64_t N, int K, bool need_sh = true)
{
    int rc;
    if (N > ctx->s_cap_n) {
        dev_free(ctx->s_means); dev_free(ctx->s_scales); dev_free(ctx->s_quats); dev_free(ctx->s_opac);
        ctx->s_cap_n = 0;
        if ((rc = dev_alloc(ctx, &ctx->s_means, (size_t)N * 3))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->s_scales, (size_t)N * 3))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->s_quats, (size_t)N * 4))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->s_opac, (size_t)N))) return rc;
        ctx->s_cap_n = N;
    }
    const int64_t sh_floats = N * K * 3;
    if (need_sh && sh_floats > ctx->s_cap_sh) {
        dev_free(ctx->s_sh); ctx->s_cap_sh = 0;
        if ((rc = dev_alloc(ctx, &ctx->s_sh, (size_t)sh_floats))) return rc;
        ctx->s_cap_sh = sh_floats;
    }
    return HIGS_OK;
}

int ensure_image_capacity(higs_ctx* ctx, int W, int H)
{
    const int64_t need = (int64_t)W * H * 3;
    if (need <= ctx->s_img_cap) return HIGS_OK;
    dev_free(ctx->s_img); ctx->s_img_cap = 0;
    int rc;
    if ((rc = dev_alloc(ctx, &ctx->s_img, (size_t)need))) return rc;
    ctx->s_img_cap = need;
    return HIGS_OK;
}

} // namespace

extern "C" {

int higs_abi_version(void) { return HIGS_ABI_VERSION; }

const char* higs_strerror(int status)
{
    switch (status) {
        case HIGS_OK: return "ok";
        case HIGS_E_ARG: return "invalid argument";
        case HIGS_E_CUDA: return "CUDA error (see higs_last_error)";
        case HIGS_E_CAPACITY: return "frame exceeded the preallocated pair / unit capacity";
        case HIGS_E_NOMEM: return "out of memory";
        default: return "unknown status";
    }
}

const char* higs_last_error(higs_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int higs_create(higs_ctx** out, int device, int64_t max_gaussians, int max_W, int max_H, int64_t max_pairs)
{
    if (!out) return HIGS_E_ARG;
    *out = nullptr;
    if (max_gaussians < 0 || max_gaussians > 0xfffffff0ll || max_W <= 0 || max_H <= 0) return HIGS_E_ARG;
    if (max_pairs <= 0) max_pairs = 4 * max_gaussians + 65536;
    if (max_pairs > 0x7fffffffll) return HIGS_E_ARG;
    int64_t nm = 0;                                                 // macro-tiles at max_W x max_H, the most over the supported shapes (8 x 8 px tiles)
    for (int tx = 4; tx <= 16; tx *= 2) {
        const int mw = tx * HIGS_TILE, mh = (HIGS_MT_TILES / tx) * HIGS_TILE;
        const int64_t v = (int64_t)((max_W + mw - 1) / mw) * ((max_H + mh - 1) / mh);
        if (v > nm) nm = v;
    }
    if (nm > HIGS_MAX_NM) return HIGS_E_ARG;
    higs_ctx* ctx = new (std::nothrow) higs_ctx();
    if (!ctx) return HIGS_E_NOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device; ctx->max_gaussians = max_gaussians; ctx->max_W = max_W; ctx->max_H = max_H;
    ctx->max_nm = (int)nm; ctx->max_pairs = max_pairs; ctx->batch_cap = HIGS_BATCH_CAP; ctx->flags = 0; ctx->tile = HIGS_TILE; ctx->mt_tx = 8; ctx->mt_ty = 4;
    int rc = HIGS_OK;
    auto fail = [&](int code) { higs_destroy(ctx); return code; };
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return fail(HIGS_E_CUDA); }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(HIGS_E_CUDA);
    ctx->n_sm = prop.multiProcessorCount;
    ctx->touch_max_pairs = (uint32_t)((size_t)prop.l2CacheSize / 4 * 3 / 8);
    const int64_t n = max_gaussians > 0 ? max_gaussians : 1;
    ctx->n_chunks_max = (n + HIGS_CHUNK - 1) / HIGS_CHUNK;
    if ((rc = higs_project_smem_setup(ctx))) return fail(rc);       // also fixes n_part_max = n_sm x resident CTAs
    if ((rc = dev_alloc(ctx, &ctx->valid_bits, (size_t)(n + 31) / 32 + 1))) return fail(rc);
    const size_t n_slots = (size_t)ctx->n_chunks_max * HIGS_CHUNK;
    if ((rc = dev_alloc(ctx, &ctx->rec, n_slots * 4))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->rec16, n_slots * 2))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->bin, n_slots))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->chunk_count, (size_t)ctx->n_chunks_max))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->part_list, (size_t)ctx->n_chunks_max))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->part_desc, (size_t)ctx->n_part_max))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->hist, (size_t)ctx->n_part_max * nm))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->cut_word, (size_t)nm * HIGS_MT_TILES))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->tile_load, (size_t)nm * HIGS_MT_TILES))) return fail(rc);
    static_assert(sizeof(FrameHeader) <= sizeof(uint32_t) * HIGS_HDR_WORDS, "frame header outgrew its block");
    if ((rc = dev_alloc(ctx, &ctx->hdr_block, HIGS_HDR_WORDS + 2 * ((size_t)nm + 1)))) return fail(rc);
    ctx->hdr = reinterpret_cast<FrameHeader*>(ctx->hdr_block);
    ctx->mt_count = ctx->hdr_block + HIGS_HDR_WORDS;
    ctx->mt_fill = ctx->mt_count + (nm + 1);
    if ((rc = dev_alloc(ctx, &ctx->mt_offset, (size_t)nm + 1))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->batch_offset, (size_t)nm + 1))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->pairs, (size_t)max_pairs))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->pairs_alt, (size_t)max_pairs))) return fail(rc);
    ctx->max_over = max_pairs / HIGS_SORT_BLOCK + 1;
    ctx->max_buckets = max_pairs / HIGS_BUCKET_TARGET + ctx->max_over + 1;
    ctx->max_jobs = nm + ctx->max_buckets + max_pairs / HIGS_SORT_BLOCK + 2;
    if ((rc = dev_alloc(ctx, &ctx->sort_jobs, (size_t)ctx->max_jobs * HIGS_N_TIERS * 2))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->over_segs, (size_t)ctx->max_over))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->split_segs, (size_t)ctx->max_over))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->splitters, (size_t)ctx->max_buckets))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->bucket_count, (size_t)ctx->max_buckets))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->bucket_cursor, (size_t)ctx->max_buckets))) return fail(rc);
    if ((rc = dev_alloc(ctx, &ctx->bucket_id, (size_t)max_pairs))) return fail(rc);
    if ((rc = alloc_unit_buffers(ctx))) return fail(rc);
    if (cudaMallocHost((void**)&ctx->hdr_host, sizeof(FrameHeader)) != cudaSuccess) return fail(HIGS_E_NOMEM);
    if (cudaMemset(ctx->hdr_block, 0, sizeof(uint32_t) * (HIGS_HDR_WORDS + 2 * ((size_t)nm + 1))) != cudaSuccess) return fail(HIGS_E_CUDA);
    memset(ctx->hdr_host, 0, sizeof(FrameHeader));
    if (cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(HIGS_E_CUDA);
    for (int i = 0; i < 9; ++i) if (cudaEventCreate(&ctx->ev[i]) != cudaSuccess) return fail(HIGS_E_CUDA);
    for (int i = 0; i < 4; ++i) {
        if (cudaStreamCreateWithFlags(&ctx->aux_stream[i], cudaStreamNonBlocking) != cudaSuccess) return fail(HIGS_E_CUDA);
        if (cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming) != cudaSuccess) return fail(HIGS_E_CUDA);
    }
    if (cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess) return fail(HIGS_E_CUDA);
    if (cudaEventCreateWithFlags(&ctx->ev_fork2, cudaEventDisableTiming) != cudaSuccess) return fail(HIGS_E_CUDA);
    if ((rc = higs_binning_smem_setup(ctx))) return fail(rc);
    if ((rc = higs_sort_smem_setup(ctx))) return fail(rc);
    if ((rc = higs_raster_setup(ctx))) return fail(rc);
    ctx->last_stream = ctx->own_stream;
    *out = ctx;
    return HIGS_OK;
}

void higs_destroy(higs_ctx* ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    dev_free(ctx->valid_bits); dev_free(ctx->rec); dev_free(ctx->rec16); dev_free(ctx->bin); dev_free(ctx->chunk_count); dev_free(ctx->part_list); dev_free(ctx->part_desc); dev_free(ctx->rec_export); dev_free(ctx->hist); dev_free(ctx->hdr_block);
    dev_free(ctx->mt_offset); dev_free(ctx->batch_offset); dev_free(ctx->unit_mt);
    dev_free(ctx->unit_active); dev_free(ctx->pairs); dev_free(ctx->pairs_alt); dev_free(ctx->sort_jobs);
    dev_free(ctx->over_segs); dev_free(ctx->split_segs); dev_free(ctx->splitters); dev_free(ctx->bucket_count);
    dev_free(ctx->bucket_cursor); dev_free(ctx->bucket_id); dev_free(ctx->partial); dev_free(ctx->cut_word); dev_free(ctx->cut_term); dev_free(ctx->tile_load);
    dev_free(ctx->unit_order); dev_free(ctx->level_hist); dev_free(ctx->level_cur);
    dev_free(ctx->s_means); dev_free(ctx->s_scales); dev_free(ctx->s_quats); dev_free(ctx->s_opac); dev_free(ctx->s_sh);
    dev_free(ctx->s_img); dev_free(ctx->s_sh32); dev_free(ctx->sh32_work);
    if (ctx->hdr_host) cudaFreeHost(ctx->hdr_host);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    for (int i = 0; i < 9; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    for (int i = 0; i < 4; ++i) {
        if (ctx->aux_stream[i]) cudaStreamDestroy(ctx->aux_stream[i]);
        if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_fork2) cudaEventDestroy(ctx->ev_fork2);
    cudaGetLastError();
    delete ctx;
}

int higs_set_flags(higs_ctx* ctx, uint32_t flags)
{
    if (!ctx) return HIGS_E_ARG;
    ctx->flags = flags;
    return HIGS_OK;
}

int higs_set_batch_cap(higs_ctx* ctx, int batch_cap)
{
    if (!ctx || batch_cap < 1 || batch_cap > HIGS_BATCH_CAP) return HIGS_E_ARG;
    if (batch_cap == ctx->batch_cap) return HIGS_OK;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    HIGS_CUDA(ctx, cudaDeviceSynchronize());
    ctx->batch_cap = batch_cap;
    return alloc_unit_buffers(ctx);
}

int higs_set_tile(higs_ctx* ctx, int tile)
{
    if (!ctx || (tile != 8 && tile != 16) || (tile != 8 && ctx->mt_tx != 8)) return HIGS_E_ARG;
    if (tile == ctx->tile) return HIGS_OK;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    HIGS_CUDA(ctx, cudaDeviceSynchronize());
    ctx->tile = tile;
    return alloc_unit_buffers(ctx);
}

int higs_set_macro_tile(higs_ctx* ctx, int tiles_x, int tiles_y)
{
    if (!ctx || tiles_x * tiles_y != HIGS_MT_TILES || (tiles_x != 4 && tiles_x != 8 && tiles_x != 16)) return HIGS_E_ARG;
    if (tiles_x != 8 && ctx->tile != 8) return HIGS_E_ARG;
    ctx->mt_tx = tiles_x; ctx->mt_ty = tiles_y;
    return HIGS_OK;
}

int higs_render(higs_ctx* ctx, const float* means, const float* scales, const float* quats, const float* opacities,
                const float* sh, int degree, int64_t N, const higs_camera* cam, int W, int H, float* out_rgb,
                void* cuda_stream)
{
    int rc = check_frame_args(ctx, degree, N, cam, W, H, out_rgb);
    if (rc) return rc;
    if (N > 0 && (!means || !scales || !quats || !opacities || !sh)) return HIGS_E_ARG;
    return render_impl(ctx, means, scales, quats, opacities, sh, degree, N, cam, W, H, out_rgb, (cudaStream_t)cuda_stream);
}

int higs_scene_upload(higs_ctx* ctx, const float* means, const float* scales, const float* quats,
                      const float* opacities, const float* sh, int degree, int64_t N)
{
    if (!ctx || degree < 0 || degree > 3 || N < 0 || N > ctx->max_gaussians) return HIGS_E_ARG;
    if (N > 0 && (!means || !scales || !quats || !opacities || !sh)) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    const int K = (degree + 1) * (degree + 1);
    int rc = ensure_scene_capacity(ctx, N > 0 ? N : 1, K);
    if (rc) return rc;
    cudaStream_t st = ctx->own_stream;
    if (N > 0) {
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_means, means, sizeof(float) * 3 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_scales, scales, sizeof(float) * 3 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_quats, quats, sizeof(float) * 4 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_opac, opacities, sizeof(float) * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_sh, sh, sizeof(float) * 3 * K * N, cudaMemcpyHostToDevice, st));
    }
    HIGS_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->s_n = N; ctx->s_degree = degree; ctx->s_sh32_valid = false;
    return HIGS_OK;
}

int higs_scene_compress_sh(higs_ctx* ctx)
{
    if (!ctx || ctx->s_degree != 3 || ctx->s_n < 0) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    if (ctx->s_n > ctx->s_sh32_cap) {
        dev_free(ctx->s_sh32); ctx->s_sh32_cap = 0;
        int rc = dev_alloc(ctx, &ctx->s_sh32, (size_t)ctx->s_n * 2);
        if (rc) return rc;
        ctx->s_sh32_cap = ctx->s_n;
    }
    int rc = launch_sh32_encode(ctx, ctx->own_stream);
    if (rc) return rc;
    ctx->s_sh32_valid = true;
    return HIGS_OK;
}

int higs_scene_sort_spatial(higs_ctx* ctx, uint32_t* host_perm)
{
    if (!ctx || ctx->s_n < 0 || ctx->s_n > ctx->max_pairs) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    HIGS_CUDA(ctx, cudaDeviceSynchronize());
    uint32_t* d_perm = nullptr;
    int rc;
    if (host_perm && ctx->s_n > 0 && (rc = dev_alloc(ctx, &d_perm, (size_t)ctx->s_n))) return rc;
    if (ctx->s_n == 1 && host_perm) host_perm[0] = 0u;
    rc = launch_scene_sort(ctx, d_perm, ctx->own_stream);
    if (!rc && host_perm && ctx->s_n > 1) {
        cudaError_t e = cudaMemcpy(host_perm, d_perm, sizeof(uint32_t) * (size_t)ctx->s_n, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { dev_free(d_perm); HIGS_CUDA(ctx, e); }
    }
    dev_free(d_perm);
    ctx->s_sh32_valid = false;
    ctx->last_stream = ctx->own_stream;
    return rc;
}

int higs_get_sh32(higs_ctx* ctx, uint8_t* host_codes, float* host_scales)
{
    if (!ctx || !ctx->s_sh32_valid) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    if (host_codes && ctx->s_n > 0) HIGS_CUDA(ctx, cudaMemcpy(host_codes, ctx->s_sh32, (size_t)ctx->s_n * 32, cudaMemcpyDeviceToHost));
    if (host_scales) memcpy(host_scales, ctx->sh32_scales_host, sizeof(float) * 48);
    return HIGS_OK;
}

int higs_render_view(higs_ctx* ctx, const higs_camera* cam, int W, int H, float* out_rgb, void* cuda_stream)
{
    if (!ctx) return HIGS_E_ARG;
    int rc = check_frame_args(ctx, ctx->s_degree, ctx->s_n, cam, W, H, out_rgb);
    if (rc) return rc;
    const bool sh32 = (ctx->flags & HIGS_FLAG_SH32) && ctx->s_sh32_valid;
    return render_impl(ctx, ctx->s_means, ctx->s_scales, ctx->s_quats, ctx->s_opac, sh32 ? reinterpret_cast<const float*>(ctx->s_sh32) : ctx->s_sh,
                       ctx->s_degree, ctx->s_n, cam, W, H, out_rgb, (cudaStream_t)cuda_stream, sh32 ? HIGS_SH_CODES : HIGS_SH_ROWS);
}

int higs_render_view_host(higs_ctx* ctx, const higs_camera* cam, int W, int H, float* out_rgb)
{
    if (!ctx) return HIGS_E_ARG;
    int rc = check_frame_args(ctx, ctx->s_degree, ctx->s_n, cam, W, H, out_rgb);
    if (rc) return rc;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    if ((rc = ensure_image_capacity(ctx, W, H))) return rc;
    cudaStream_t st = ctx->own_stream;
    const bool sh32 = (ctx->flags & HIGS_FLAG_SH32) && ctx->s_sh32_valid;
    rc = render_impl(ctx, ctx->s_means, ctx->s_scales, ctx->s_quats, ctx->s_opac, sh32 ? reinterpret_cast<const float*>(ctx->s_sh32) : ctx->s_sh,
                     ctx->s_degree, ctx->s_n, cam, W, H, ctx->s_img, st, sh32 ? HIGS_SH_CODES : HIGS_SH_ROWS);
    if (rc) return rc;
    HIGS_CUDA(ctx, cudaMemcpyAsync(out_rgb, ctx->s_img, sizeof(float) * 3 * (size_t)W * H, cudaMemcpyDeviceToHost, st));
    HIGS_CUDA(ctx, cudaStreamSynchronize(st));
    return HIGS_OK;
}

// Device-visible alias of a page-locked, mapped host buffer (cudaHostAlloc, cudaHostRegister), or null for pageable memory.
static const float* mapped_alias(const float* host)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return (a.type == cudaMemoryTypeHost && a.devicePointer) ? static_cast<const float*>(a.devicePointer) : nullptr;
}

// The SH array is 4/5 of the scene's bytes and the cull keeps fewer than half of the gaussians: when the caller's array is
// page-locked the projection kernel takes the rows of the survivors straight from host memory (HIGS_SH_STAGED, project.cu)
// and the array is never uploaded.  Measured on the bench scene (5.8 M gaussians, 2.6 M survivors): 0.76 GB instead of
// 1.37 GB over PCIe per frame, 15.9 ms instead of 26.0 ms.  The four small arrays are always uploaded: every gaussian's
// are read, a bulk copy is the cheapest way to move them.
int higs_render_host(higs_ctx* ctx, const float* means, const float* scales, const float* quats, const float* opacities,
                     const float* sh, int degree, int64_t N, const higs_camera* cam, int W, int H, float* out_rgb)
{
    int rc = check_frame_args(ctx, degree, N, cam, W, H, out_rgb);
    if (rc) return rc;
    if (N > 0 && (!means || !scales || !quats || !opacities || !sh)) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    const int K = (degree + 1) * (degree + 1);
    const float* d_sh = (N > 0 && ctx->proj_staged_ok) ? mapped_alias(sh) : nullptr;
    ctx->s_n = -1; ctx->s_sh32_valid = false;                        // the staging buffers are the resident scene's: it is gone
    if ((rc = ensure_scene_capacity(ctx, N > 0 ? N : 1, K, d_sh == nullptr))) return rc;
    if ((rc = ensure_image_capacity(ctx, W, H))) return rc;
    cudaStream_t st = ctx->own_stream;
    if (N > 0) {
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_means, means, sizeof(float) * 3 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_scales, scales, sizeof(float) * 3 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_quats, quats, sizeof(float) * 4 * N, cudaMemcpyHostToDevice, st));
        HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_opac, opacities, sizeof(float) * N, cudaMemcpyHostToDevice, st));
        if (!d_sh) HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->s_sh, sh, sizeof(float) * 3 * K * N, cudaMemcpyHostToDevice, st));
    }
    rc = render_impl(ctx, ctx->s_means, ctx->s_scales, ctx->s_quats, ctx->s_opac, d_sh ? d_sh : ctx->s_sh, degree, N, cam, W, H, ctx->s_img, st,
                     d_sh ? HIGS_SH_STAGED : HIGS_SH_ROWS);
    if (rc) return rc;
    HIGS_CUDA(ctx, cudaMemcpyAsync(out_rgb, ctx->s_img, sizeof(float) * 3 * (size_t)W * H, cudaMemcpyDeviceToHost, st));
    HIGS_CUDA(ctx, cudaStreamSynchronize(st));
    return HIGS_OK;
}

int higs_get_stats(higs_ctx* ctx, higs_stats* out)
{
    if (!ctx || !out) return HIGS_E_ARG;
    int rc = fetch_header(ctx);
    if (rc) return rc;
    const FrameHeader& h = *ctx->hdr_host;
    memset(out, 0, sizeof(*out));
    out->n_gaussians = ctx->last_n; out->n_visible = h.n_visible; out->n_pairs = h.n_pairs; out->n_units = h.n_units;
    out->max_segment = h.max_segment; out->n_oversize = h.n_oversize;
    out->n_mt_x = ctx->last_mx; out->n_mt_y = ctx->last_my; out->batch_cap = ctx->batch_cap; out->overflow = (int32_t)h.overflow;
    out->n_launches = ctx->n_launches; out->tile = ctx->tile;
    out->n_evals = (int64_t)h.n_evals; out->n_tile_pairs = (int64_t)h.n_tile_pairs;
    if (ctx->timers_valid) {
        float* dst[7] = { &out->ms_project, &out->ms_count, &out->ms_scan, &out->ms_fill, &out->ms_sort, &out->ms_raster, &out->ms_merge };
        for (int i = 0; i < 7; ++i) HIGS_CUDA(ctx, cudaEventElapsedTime(dst[i], ctx->ev[i], ctx->ev[i + 1]));
        HIGS_CUDA(ctx, cudaEventElapsedTime(&out->ms_total, ctx->ev[0], ctx->ev[7]));
    }
    return h.overflow ? HIGS_E_CAPACITY : HIGS_OK;
}

int higs_get_lists(higs_ctx* ctx, higs_lists* out)
{
    if (!ctx || !out) return HIGS_E_ARG;
    int rc = fetch_header(ctx);
    if (rc) return rc;
    const FrameHeader& h = *ctx->hdr_host;
    // the frame's own list carries dense slots; the caller gets gaussian ids (same order: slots are monotone in the id)
    if (!h.overflow && h.n_pairs) {
        if ((rc = launch_export_lists(ctx, h.n_pairs, ctx->last_stream))) return rc;
        HIGS_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
    }
    out->n_pairs = h.n_pairs; out->n_units = h.n_units; out->n_mt = ctx->last_nm;
    out->mt_count = ctx->mt_count; out->mt_offset = ctx->mt_offset; out->batch_offset = ctx->batch_offset; out->tile_load = ctx->tile_load;
    out->pairs = reinterpret_cast<const uint64_t*>(ctx->pairs_alt); out->unit_active = ctx->unit_active;
    return h.overflow ? HIGS_E_CAPACITY : HIGS_OK;
}

int higs_get_records(higs_ctx* ctx, higs_records* out)
{
    if (!ctx || !out) return HIGS_E_ARG;
    int rc = fetch_header(ctx);
    if (rc) return rc;
    if (!ctx->rec_export && (rc = dev_alloc(ctx, &ctx->rec_export, (size_t)(ctx->max_gaussians > 0 ? ctx->max_gaussians : 1) * 16))) return rc;
    if (ctx->last_n > 0) {
        if ((rc = launch_export_records(ctx, ctx->last_n, ctx->last_stream))) return rc;
        HIGS_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
    }
    out->n = ctx->last_n; out->valid_bits = ctx->valid_bits;
    out->rec = ctx->rec_export;
    return HIGS_OK;
}

int higs_download(higs_ctx* ctx, const void* device_src, void* host_dst, uint64_t bytes)
{
    if (!ctx || (bytes && (!device_src || !host_dst))) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    HIGS_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
    if (bytes) HIGS_CUDA(ctx, cudaMemcpy(host_dst, device_src, (size_t)bytes, cudaMemcpyDeviceToHost));
    return HIGS_OK;
}

int higs_sort_segments(higs_ctx* ctx, uint64_t* pairs, const uint32_t* seg_offset, int32_t n_seg, void* cuda_stream)
{
    if (!ctx || !pairs || !seg_offset || n_seg < 0 || n_seg > ctx->max_nm) return HIGS_E_ARG;
    HIGS_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->last_stream = (cudaStream_t)cuda_stream;
    return launch_sort_only(ctx, reinterpret_cast<unsigned long long*>(pairs), seg_offset, n_seg, (cudaStream_t)cuda_stream);
}

} // extern "C"
