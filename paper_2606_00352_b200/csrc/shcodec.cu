// shcodec.cu -- encoder of the 32-byte SH representation (section 4.2: "YCoCg-R color-space conversion to
// decorrelate channels, square-root gamma quantization (6 bits luma, 4 bits chroma), and per-basis percentile scaling
// ... Per-gaussian SH bandwidth drops from 192 bytes (fp32) to 32 bytes").  The paper gives no bit layout; DESIGN.md
// reading Q20 fixes one:
//   per basis k = 0..15: (r, g, b) -> (Y, Co, Cg) by the lifting steps Co = r - b; t = b + Co/2; Cg = g - t; Y = t + Cg/2;
//   scale s(k, channel) = |v| at sorted index min(N-1, floor(0.999 N)) over the scene (index N-1 for the DC basis);
//   code = bias + sign(u) rint(sqrt(min(|u|, 1)) L), u = v / s, (L, bias) = (31, 32) luma / (7, 8) chroma; decode v = s w|w|,
//   w = (code - bias) / L; the DC basis has 16-bit luma (L = 32767) and 15-bit chroma (L = 16383) codes whose top 6 / 4
//   bits sit in the regular fields and whose low bits sit in the last word;
//   bytes 0-11 luma bit stream (6 bits per basis, little endian), byte 12+k = Cg_k << 4 | Co_k, bytes 28-31 =
//   DC Y low 10 | DC Co low 11 << 10 | DC Cg low 11 << 21.
// Runs once per scene (higs_scene_compress_sh); the decoder is inline in k_project (project.cu).  Encoding is byte
// work: every arithmetic step is one correctly rounded fp32 op in the written order, so the bytes are identical to the
// CPU oracle's.  The percentile is an exact selection: four 8-bit passes of a radix select on the bit patterns of |v|
// (non-negative floats order like unsigned integers), 48 columns at a time.
#include <pthread.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include "higs_internal.cuh"

namespace {

constexpr int ENC_THREADS = 256;

__device__ __forceinline__ void ycocg_fwd(float r, float g, float b, float& y, float& co, float& cg)
{
    co = __fsub_rn(r, b);
    const float t = __fadd_rn(b, __fmul_rn(0.5f, co));
    cg = __fsub_rn(g, t);
    y = __fadd_rn(t, __fmul_rn(0.5f, cg));
}

// work layout (uint32 words): hist [48][256] | prefix [48] | rank [48] lo, hi | scales [48] (float bits)
constexpr int W_HIST = 0, W_PREFIX = 48 * 256, W_RANK = W_PREFIX + 48, W_SCALE = W_RANK + 96, W_TOTAL = W_SCALE + 48;

__global__ void k_sh_select_init(uint32_t* __restrict__ work, int64_t N)
{
    const int c = threadIdx.x;
    if (c < 48) {
        const int k = c / 3;
        long long idx = k == 0 ? N - 1 : (long long)((double)N * 0.999);
        if (idx > N - 1) idx = N - 1;
        if (idx < 0) idx = 0;
        work[W_PREFIX + c] = 0u;
        work[W_RANK + 2 * c] = (uint32_t)idx; work[W_RANK + 2 * c + 1] = (uint32_t)((unsigned long long)idx >> 32);
    }
    for (int e = threadIdx.x; e < 48 * 256; e += blockDim.x) work[W_HIST + e] = 0u;
}

// pass p = 0..3 looks at bits [31 - 8p - 7, 31 - 8p] of the keys whose higher bits equal the column's prefix
__global__ void __launch_bounds__(ENC_THREADS)
k_sh_select_hist(const float* __restrict__ sh, int64_t N, int pass, uint32_t* __restrict__ work)
{
    extern __shared__ uint32_t s_hist[];                             // [48][256] then the 48 prefixes
    uint32_t* s_prefix = s_hist + 48 * 256;
    for (int e = threadIdx.x; e < 48 * 256; e += ENC_THREADS) s_hist[e] = 0u;
    if (threadIdx.x < 48) s_prefix[threadIdx.x] = work[W_PREFIX + threadIdx.x];
    __syncthreads();
    const int shift = 24 - 8 * pass;
    for (int64_t i = (int64_t)blockIdx.x * ENC_THREADS + threadIdx.x; i < N; i += (int64_t)gridDim.x * ENC_THREADS) {
        const float* q = sh + i * 48;
#pragma unroll 4
        for (int k = 0; k < 16; ++k) {
            float v[3];
            ycocg_fwd(q[3 * k], q[3 * k + 1], q[3 * k + 2], v[0], v[1], v[2]);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const uint32_t key = __float_as_uint(fabsf(v[c]));
                const bool match = pass == 0 || (key >> (shift + 8)) == (s_prefix[k * 3 + c] >> (shift + 8));
                if (match) atomicAdd(&s_hist[(k * 3 + c) * 256 + ((key >> shift) & 255u)], 1u);
            }
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < 48 * 256; e += ENC_THREADS) if (s_hist[e]) atomicAdd(&work[W_HIST + e], s_hist[e]);
}

// one warp per column: the digit in which the running count passes the rank; the rank becomes relative to that digit
__global__ void k_sh_select_step(uint32_t* __restrict__ work, int pass)
{
    const int c = blockIdx.x, lane = threadIdx.x;
    const int shift = 24 - 8 * pass;
    unsigned long long rank = (unsigned long long)work[W_RANK + 2 * c] | ((unsigned long long)work[W_RANK + 2 * c + 1] << 32);
    uint32_t h[8]; unsigned long long sum = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { h[q] = work[W_HIST + c * 256 + lane * 8 + q]; sum += h[q]; }
    unsigned long long incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const unsigned long long y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
    unsigned long long run = incl - sum;
    int digit = -1; unsigned long long before = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (digit < 0 && rank < run + h[q]) { digit = lane * 8 + q; before = run; }
        run += h[q];
    }
    const uint32_t found = __ballot_sync(0xffffffffu, digit >= 0);
    const int src = __ffs(found) - 1;                                // the first lane whose range holds the rank
    digit = __shfl_sync(0xffffffffu, digit, src); before = __shfl_sync(0xffffffffu, before, src);
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 8; ++q) work[W_HIST + c * 256 + lane * 8 + q] = 0u;
    if (lane == 0) {
        const uint32_t prefix = work[W_PREFIX + c] | ((uint32_t)digit << shift);
        work[W_PREFIX + c] = prefix;
        rank -= before;
        work[W_RANK + 2 * c] = (uint32_t)rank; work[W_RANK + 2 * c + 1] = (uint32_t)(rank >> 32);
        if (pass == 3) {
            const float sc = __uint_as_float(prefix);
            work[W_SCALE + c] = __float_as_uint((sc > 0.0f && sc <= 3.402823466e+38f) ? sc : 1.0f);
        }
    }
}

__device__ __forceinline__ uint32_t sh32_quant(float v, float s, int L)
{
    const float u = __fdiv_rn(v, s);
    const float a = fminf(fabsf(u), 1.0f);
    const float w = __fsqrt_rn(a);
    const int c = (int)rintf(__fmul_rn(w, (float)L));
    return (uint32_t)((L + 1) + (u < 0.0f ? -c : c));
}

__global__ void __launch_bounds__(ENC_THREADS)
k_sh_encode(const float* __restrict__ sh, int64_t N, const uint32_t* __restrict__ work, uint4* __restrict__ out)
{
    __shared__ float s_scale[48];
    if (threadIdx.x < 48) s_scale[threadIdx.x] = __uint_as_float(work[W_SCALE + threadIdx.x]);
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * ENC_THREADS + threadIdx.x;
    if (i >= N) return;
    const float* q = sh + i * 48;
    uint32_t lw[3] = { 0u, 0u, 0u }, cw[4] = { 0u, 0u, 0u, 0u }, ext = 0u;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        float y, co, cg;
        ycocg_fwd(q[3 * k], q[3 * k + 1], q[3 * k + 2], y, co, cg);
        uint32_t cy, cco, ccg;
        if (k == 0) {
            const uint32_t y16 = sh32_quant(y, s_scale[0], 32767), co15 = sh32_quant(co, s_scale[1], 16383), cg15 = sh32_quant(cg, s_scale[2], 16383);
            ext = (y16 & 0x3ffu) | ((co15 & 0x7ffu) << 10) | ((cg15 & 0x7ffu) << 21);
            cy = y16 >> 10; cco = co15 >> 11; ccg = cg15 >> 11;
        } else {
            cy = sh32_quant(y, s_scale[3 * k], 31); cco = sh32_quant(co, s_scale[3 * k + 1], 7); ccg = sh32_quant(cg, s_scale[3 * k + 2], 7);
        }
        const int bit = 6 * k, wd = bit >> 5, sf = bit & 31;
        lw[wd] |= cy << sf;
        if (sf > 26 && wd < 2) lw[wd + 1] |= cy >> (32 - sf);
        cw[k >> 2] |= ((ccg << 4) | cco) << (8 * (k & 3));
    }
    out[2 * i] = make_uint4(lw[0], lw[1], lw[2], cw[0]);
    out[2 * i + 1] = make_uint4(cw[1], cw[2], cw[3], ext);
}

} // namespace

// Encodes the resident scene's SH rows (ctx->s_sh, degree 3) into ctx->s_sh32 and leaves the scale table in
// ctx->sh32_scales_host.  Synchronises the stream (scene set-up, not part of a frame).
int launch_sh32_encode(higs_ctx* ctx, cudaStream_t st)
{
    const int64_t N = ctx->s_n;
    if (N <= 0) { for (int c = 0; c < 48; ++c) ctx->sh32_scales_host[c] = 1.0f; return HIGS_OK; }
    const size_t hist_smem = sizeof(uint32_t) * (48 * 256 + 48);
    HIGS_CUDA(ctx, cudaFuncSetAttribute(k_sh_select_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hist_smem));
    if (!ctx->sh32_work) {
        void* q = nullptr;
        HIGS_CUDA(ctx, cudaMalloc(&q, sizeof(uint32_t) * W_TOTAL));
        ctx->sh32_work = static_cast<uint32_t*>(q);
    }
    uint32_t* work = ctx->sh32_work;
    k_sh_select_init<<<1, 256, 0, st>>>(work, N);
    HIGS_CUDA(ctx, cudaGetLastError());
    const int grid = ctx->n_sm * 2;
    for (int pass = 0; pass < 4; ++pass) {
        k_sh_select_hist<<<grid, ENC_THREADS, hist_smem, st>>>(ctx->s_sh, N, pass, work);
        HIGS_CUDA(ctx, cudaGetLastError());
        k_sh_select_step<<<48, 32, 0, st>>>(work, pass);
        HIGS_CUDA(ctx, cudaGetLastError());
    }
    if (N > 0) {
        k_sh_encode<<<(unsigned)((N + ENC_THREADS - 1) / ENC_THREADS), ENC_THREADS, 0, st>>>(ctx->s_sh, N, work, ctx->s_sh32);
        HIGS_CUDA(ctx, cudaGetLastError());
    }
    HIGS_CUDA(ctx, cudaMemcpyAsync(ctx->sh32_scales_host, work + W_SCALE, sizeof(float) * 48, cudaMemcpyDeviceToHost, st));
    HIGS_CUDA(ctx, cudaStreamSynchronize(st));
    return HIGS_OK;
}

// ---- higs_sh32_encode_static: the encoder for callers that cannot allocate ------------------------------------------
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.)  Same kernels as above; the radix-select work
// area (W_TOTAL words = 49,920 bytes: 48 x 256 counters, prefixes, ranks, scales) lives in a file-scope device array
// instead of ctx->sh32_work, so the call needs no context and allocates nothing.  Every GPU that loads the library holds
// these 49,920 bytes until the process exits.  The array is shared by all calls and keeps the last call's contents:
// k_sh_select_init clears what must start at zero; calls that overlap on the GPU (two streams, two threads) race on it.
static __device__ __align__(256) uint32_t g_sh32_static_work[W_TOTAL];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDev { bool ready; uint32_t* work; int n_sm; };
StaticDev g_static_dev[STATIC_MAX_DEVICES];                          // set up once per device (guarded by g_static_mutex)
pthread_mutex_t g_static_mutex = PTHREAD_MUTEX_INITIALIZER;
thread_local char g_static_err[256] = "";

__global__ void k_sh_static_ones(float* __restrict__ scales) { if (threadIdx.x < 48) scales[threadIdx.x] = 1.0f; }   // N = 0: as launch_sh32_encode

int static_fail(int code, const char* what, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess) { snprintf(g_static_err, sizeof(g_static_err), "%s: %s", what, cudaGetErrorString(e)); cudaGetLastError(); }
    else snprintf(g_static_err, sizeof(g_static_err), "%s", what);
    return code;
}
} // namespace

const char* higs_sh32_encode_static_error(void) { return g_static_err; }

int higs_sh32_encode_static(const float* d_sh, int64_t N, uint8_t* d_codes, float* d_scales, void* cuda_stream)
{
    g_static_err[0] = 0;
    if (N < 0) return static_fail(HIGS_E_ARG, "higs_sh32_encode_static: N < 0");
    if (N > HIGS_SH32_STATIC_MAX_N) {
        snprintf(g_static_err, sizeof(g_static_err), "higs_sh32_encode_static: N = %lld exceeds HIGS_SH32_STATIC_MAX_N = %lld (32-bit counters of the static work area)",
                 (long long)N, (long long)HIGS_SH32_STATIC_MAX_N);
        return HIGS_E_CAPACITY;
    }
    if (!d_scales || (N > 0 && (!d_sh || !d_codes))) return static_fail(HIGS_E_ARG, "higs_sh32_encode_static: null pointer");
    if ((reinterpret_cast<uintptr_t>(d_sh) & 3u) || (reinterpret_cast<uintptr_t>(d_codes) & 15u))
        return static_fail(HIGS_E_ARG, "higs_sh32_encode_static: d_sh must be 4-byte and d_codes 16-byte aligned");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(HIGS_E_CUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return static_fail(HIGS_E_ARG, "higs_sh32_encode_static: device index beyond 63");
    const size_t hist_smem = sizeof(uint32_t) * (48 * 256 + 48);
    pthread_mutex_lock(&g_static_mutex);
    StaticDev sd = g_static_dev[dev];
    if (!sd.ready) {
        // once per device, with that device current: the array's name is a host-side stand-in here, not a device address
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sh32_static_work);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sh_select_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hist_smem);
        int n_sm = 0;
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || !p || n_sm <= 0) {
            pthread_mutex_unlock(&g_static_mutex);
            return static_fail(HIGS_E_CUDA, "higs_sh32_encode_static set-up (cudaGetSymbolAddress / attributes)", e);
        }
        sd.ready = true; sd.work = static_cast<uint32_t*>(p); sd.n_sm = n_sm;
        g_static_dev[dev] = sd;
    }
    pthread_mutex_unlock(&g_static_mutex);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint32_t* work = sd.work;
    if (N == 0) {
        k_sh_static_ones<<<1, 64, 0, st>>>(d_scales);
        if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(HIGS_E_CUDA, "higs_sh32_encode_static launch", e);
        return HIGS_OK;
    }
    k_sh_select_init<<<1, 256, 0, st>>>(work, N);                    // clears the counters and prefixes the last call left behind
    for (int pass = 0; pass < 4; ++pass) {
        k_sh_select_hist<<<sd.n_sm * 2, ENC_THREADS, hist_smem, st>>>(d_sh, N, pass, work);
        k_sh_select_step<<<48, 32, 0, st>>>(work, pass);
    }
    k_sh_encode<<<(unsigned)((N + ENC_THREADS - 1) / ENC_THREADS), ENC_THREADS, 0, st>>>(d_sh, N, work, reinterpret_cast<uint4*>(d_codes));
    if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(HIGS_E_CUDA, "higs_sh32_encode_static launch", e);
    if ((e = cudaMemcpyAsync(d_scales, work + W_SCALE, sizeof(float) * 48, cudaMemcpyDeviceToDevice, st)) != cudaSuccess)
        return static_fail(HIGS_E_CUDA, "higs_sh32_encode_static scale copy", e);
    return HIGS_OK;
}
