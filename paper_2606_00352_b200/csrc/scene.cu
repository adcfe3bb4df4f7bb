// scene.cu -- spatial ordering of a resident scene (higs_scene_sort_spatial).
//
// The projection kernel (a1) reads the 192-byte SH row of every gaussian that survives the cull.  With the ids in
// arbitrary order the survivors are scattered, and DRAM delivers about 1.6 x the bytes asked for (profiles/r02_final.md);
// the cull itself diverges inside every warp.  A resident scene is owned by the library, so it may be stored in an order
// that makes neighbours in memory neighbours in space: gaussians are sorted along a Morton (Z-order) curve of their means,
// 10 bits per axis over the scene's bounding box, ties by original index.  Whole warps are then culled or kept together,
// the SH rows of the survivors are contiguous, and the records a rasterizer unit gathers sit close to each other.
// The order of the gaussians is part of the scene: ids in the lists and the (key, id) tie-break refer to the NEW order.
// The permutation is handed back, so a caller (or the test oracle) can apply it to its own copy of the arrays.
// Runs once per scene; it reuses the frame's segmented sort (sort.cu) on one segment of N (Morton key << 32 | index) items.
#include <stdio.h>
#include "higs_internal.cuh"

namespace {

// order-preserving map float -> uint32 (for atomicMin / atomicMax on floats of either sign)
__device__ __forceinline__ uint32_t f2ord(float f) { const uint32_t u = __float_as_uint(f); return (u & 0x80000000u) ? ~u : (u | 0x80000000u); }
__device__ __forceinline__ float ord2f(uint32_t o) { return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o); }

__global__ void k_bbox_init(uint32_t* __restrict__ box) { if (threadIdx.x < 3) { box[threadIdx.x] = 0xffffffffu; box[3 + threadIdx.x] = 0u; } }

__global__ void __launch_bounds__(256)
k_bbox(const float* __restrict__ means, int64_t N, uint32_t* __restrict__ box /* min x,y,z | max x,y,z (ordered ints) */)
{
    uint32_t lo[3] = { 0xffffffffu, 0xffffffffu, 0xffffffffu }, hi[3] = { 0u, 0u, 0u };
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < N; i += (int64_t)gridDim.x * 256) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float v = means[3 * i + a];
            if (v == v && fabsf(v) <= 3.402823466e+38f) { const uint32_t o = f2ord(v); lo[a] = min(lo[a], o); hi[a] = max(hi[a], o); }
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = __reduce_min_sync(0xffffffffu, lo[a]); hi[a] = __reduce_max_sync(0xffffffffu, hi[a]);
        if ((threadIdx.x & 31) == 0) { atomicMin(&box[a], lo[a]); atomicMax(&box[3 + a], hi[a]); }
    }
}

__device__ __forceinline__ uint32_t spread10(uint32_t v)       // 10 bits -> every third bit
{
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__global__ void __launch_bounds__(256)
k_morton(const float* __restrict__ means, int64_t N, const uint32_t* __restrict__ box, unsigned long long* __restrict__ items)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    uint32_t q[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float lo = ord2f(box[a]), hi = ord2f(box[3 + a]);
        const float v = means[3 * i + a];
        const float t = (hi > lo && v == v) ? (v - lo) / (hi - lo) : 0.0f;
        q[a] = (uint32_t)fminf(fmaxf(t * 1024.0f, 0.0f), 1023.0f);
    }
    const uint32_t code = spread10(q[0]) | (spread10(q[1]) << 1) | (spread10(q[2]) << 2);
    items[i] = ((unsigned long long)code << 32) | (unsigned long long)(uint32_t)i;
}

__global__ void k_one_segment(uint32_t* __restrict__ seg, uint32_t n) { if (threadIdx.x == 0) { seg[0] = 0u; seg[1] = n; } }

// out row i = in row perm(i); rows of `words` 32-bit words; one thread per word
__global__ void __launch_bounds__(256)
k_gather_rows(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, const unsigned long long* __restrict__ items, int64_t N, int words)
{
    const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= N * words) return;
    const int64_t i = e / words;
    const int wd = (int)(e - i * words);
    out[e] = in[(int64_t)(uint32_t)items[i] * words + wd];
}

__global__ void __launch_bounds__(256)
k_perm_out(const unsigned long long* __restrict__ items, int64_t N, uint32_t* __restrict__ perm)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i < N) perm[i] = (uint32_t)items[i];
}

} // namespace

// Reorders ctx->s_means / s_scales / s_quats / s_opac / s_sh in place (through one scratch buffer) and leaves the permutation
// in ctx->pairs as the low words of the sorted items.  d_perm: device buffer [N] or null.
int launch_scene_sort(higs_ctx* ctx, uint32_t* d_perm, cudaStream_t st)
{
    const int64_t N = ctx->s_n;
    if (N <= 1) return HIGS_OK;
    const int K = (ctx->s_degree + 1) * (ctx->s_degree + 1);
    uint32_t* box = ctx->mt_count;                                  // scratch: any six words that the next frame rewrites
    unsigned long long* items = ctx->pairs;
    k_bbox_init<<<1, 32, 0, st>>>(box);
    k_bbox<<<ctx->n_sm * 4, 256, 0, st>>>(ctx->s_means, N, box);
    k_morton<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(ctx->s_means, N, box, items);
    k_one_segment<<<1, 32, 0, st>>>(ctx->mt_offset, (uint32_t)N);
    HIGS_CUDA(ctx, cudaGetLastError());
    int rc = launch_sort_only(ctx, items, ctx->mt_offset, 1, st);
    if (rc) return rc;
    float* tmp = nullptr;
    HIGS_CUDA(ctx, cudaMalloc((void**)&tmp, sizeof(float) * (size_t)N * (size_t)(3 * K > 4 ? 3 * K : 4)));
    float* arrays[5] = { ctx->s_means, ctx->s_scales, ctx->s_quats, ctx->s_opac, ctx->s_sh };
    const int words[5] = { 3, 3, 4, 1, 3 * K };
    for (int a = 0; a < 5; ++a) {
        const int64_t total = N * words[a];
        k_gather_rows<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(reinterpret_cast<const uint32_t*>(arrays[a]), reinterpret_cast<uint32_t*>(tmp), items, N, words[a]);
        cudaError_t e = cudaMemcpyAsync(arrays[a], tmp, sizeof(float) * (size_t)total, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) { cudaFree(tmp); HIGS_CUDA(ctx, e); }
    }
    if (d_perm) k_perm_out<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(items, N, d_perm);
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(tmp);
    HIGS_CUDA(ctx, e);
    HIGS_CUDA(ctx, cudaGetLastError());
    return HIGS_OK;
}
