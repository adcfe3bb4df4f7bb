// project.cu -- steps a1 + a2: fused EWA projection + cull + SH colour (section 4.2), with the
// count pass of the partitioning folded in: every persistent CTA is one partition batch
// (the chunks of HIGS_CHUNK = 128 consecutive ids its warps claim), keeps the private shared-memory histogram with one counter
// per macro-tile and flushes it as one row of the N_B x N_M matrix (N_B = CTAs = a whole number per SM).  The kernel is HBM-latency-bound, so the row scan runs in issue
// slots that were idle; the macro-tile span it finds is also packed into a 64-bit descriptor in the record, so
// the fill pass replays it without redoing the arithmetic.  (Section 4.2:
// "Each thread processes one gaussian end-to-end: camera-space transformation, 2D covariance via
// Jacobian projection, ... inline view-direction computation, and degree-3 spherical harmonics
// evaluation.  The outputs -- 2D positions, ... conics, colors, and a compact per-warp visibility
// bitfield -- are consumed by the partitioning and rasterization stages.")
//
// HBM-bound: 44 B read per gaussian + 12*K B of SH read and 64 B written per *visible* gaussian.
// Everything that later decides an integer (cull, macro-tile set, depth key, the 1/255 skip) follows
// the pinned fp32 sequence N-PROJ of DESIGN.md section 3, one correctly rounded op per written op:
// the __f*_rn intrinsics are never contracted into FMAs by nvcc.
#include <stdio.h>
#include <string.h>
#include <cuda_fp16.h>
#include "higs_internal.cuh"

// inputs go through the read-only L1 path: consecutive loads of a warp share sectors (12-byte strides, halves of a
// 32-byte sector of an SH row), and streaming / L1-bypassing loads were measured to re-fetch them from L2 and DRAM
#define HIGS_LD __ldg
namespace {

// (ld.global.nc.L2::64B on the scattered 192-byte SH rows was measured: no change, 0.273 against 0.268 ms)
#ifndef HIGS_LD_SH
#define HIGS_LD_SH HIGS_LD
#endif

// ln_spec (DESIGN.md N-LN): frexp + atanh series, separate mul and add, x in (1, 255].
__device__ __forceinline__ float ln_spec(float x)
{
    uint32_t u = __float_as_uint(x);
    int e = (int)((u >> 23) & 0xffu) - 126;                      // x = mant * 2^e, mant in [0.5, 1)
    float mant = __uint_as_float((u & 0x007fffffu) | 0x3f000000u);
    if (mant < 0.70710678f) { mant = __fmul_rn(2.0f, mant); e = e - 1; }
    float f = __fsub_rn(mant, 1.0f);
    float s = __fdiv_rn(f, __fadd_rn(2.0f, f));
    float z = __fmul_rn(s, s);
    float p = 1.0f / 11.0f;
    p = __fmul_rn(p, z); p = __fadd_rn(p, 1.0f / 9.0f);
    p = __fmul_rn(p, z); p = __fadd_rn(p, 1.0f / 7.0f);
    p = __fmul_rn(p, z); p = __fadd_rn(p, 1.0f / 5.0f);
    p = __fmul_rn(p, z); p = __fadd_rn(p, 1.0f / 3.0f);
    p = __fmul_rn(p, z); p = __fadd_rn(p, 1.0f);
    float hi = __fmul_rn((float)e, 0.69314718f);
    float lo = __fmul_rn(__fmul_rn(2.0f, s), p);
    return __fadd_rn(hi, lo);
}

__device__ __forceinline__ bool finite_pos(float v) { return (v > 0.0f) && (v <= 3.402823466e+38f); }

// Real SH basis in the convention of the public 3DGS models (reading Q12), fp32 (smooth).
// STAGED: shp points at the row's copy in shared memory (k_project's SH_STAGED mode), else at the row in global memory.
template <int DEG, bool STAGED>
__device__ __forceinline__ void sh_accumulate(const float* __restrict__ shp, float x, float y, float z,
                                              float& r, float& g, float& b)
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    float c[K * 3];
    if constexpr (DEG == 3 || DEG == 1) {                        // 192 B / 48 B rows: 16-byte aligned
        const float4* p4 = reinterpret_cast<const float4*>(shp);
#pragma unroll
        for (int k = 0; k < K * 3 / 4; ++k) {
            float4 v;
            if constexpr (STAGED) v = p4[k]; else v = HIGS_LD_SH(p4 + k);
            c[4 * k] = v.x; c[4 * k + 1] = v.y; c[4 * k + 2] = v.z; c[4 * k + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < K * 3; ++k) { if constexpr (STAGED) c[k] = shp[k]; else c[k] = HIGS_LD(shp + k); }
    }
    float Y[K];
    Y[0] = 0.28209479177387814f;
    if constexpr (DEG >= 1) {
        const float C1 = 0.4886025119029199f;
        Y[1] = -C1 * y; Y[2] = C1 * z; Y[3] = -C1 * x;
    }
    if constexpr (DEG >= 2) {
        const float xx = x * x, yy = y * y, zz = z * z;
        const float C2a = 1.0925484305920792f, C2b = 0.31539156525252005f, C2c = 0.5462742152960396f;
        Y[4] = C2a * x * y;
        Y[5] = -C2a * y * z;
        Y[6] = C2b * (2.0f * zz - xx - yy);
        Y[7] = -C2a * x * z;
        Y[8] = C2c * (xx - yy);
        if constexpr (DEG >= 3) {
            const float C3a = 0.5900435899266435f, C3b = 2.890611442640554f, C3c = 0.4570457994644658f,
                        C3d = 0.3731763325901154f, C3e = 1.445305721320277f;
            Y[9]  = -C3a * y * (3.0f * xx - yy);
            Y[10] = C3b * x * y * z;
            Y[11] = -C3c * y * (4.0f * zz - xx - yy);
            Y[12] = C3d * z * (2.0f * zz - 3.0f * xx - 3.0f * yy);
            Y[13] = -C3c * x * (4.0f * zz - xx - yy);
            Y[14] = C3e * z * (xx - yy);
            Y[15] = -C3a * x * (xx - 3.0f * yy);
        }
    }
    r = 0.5f; g = 0.5f; b = 0.5f;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        r = fmaf(Y[k], c[3 * k], r);
        g = fmaf(Y[k], c[3 * k + 1], g);
        b = fmaf(Y[k], c[3 * k + 2], b);
    }
    r = fmaxf(r, 0.0f); g = fmaxf(g, 0.0f); b = fmaxf(b, 0.0f);
}

// Colour from the 32-byte SH code (layout and quantiser: DESIGN.md reading Q20, shcodec.cu).  The evaluation is
// linear, so it runs in YCoCg space - sum_k Y_k(dir) * (y, co, cg)_k - and one inverse YCoCg-R lifting at the end gives
// r, g, b.  lut: [16][64] luma then [16][2][16] chroma dequantised values s * w|w| (built per CTA from the scale table),
// so a coefficient costs a bit-field extract, one shared load and one FMA.  The DC basis (16 / 15 / 15 bits) is
// dequantised arithmetically.
__device__ __forceinline__ void sh32_colour(const uint4* __restrict__ codes, int64_t i, const float* __restrict__ lut,
                                            const ShScales& sc, float x, float y, float z, float& r, float& g, float& b)
{
    const uint4 c0 = HIGS_LD(codes + 2 * i), c1 = HIGS_LD(codes + 2 * i + 1);
    const uint32_t lw[4] = { c0.x, c0.y, c0.z, 0u };               // luma bit stream
    const uint32_t cw[4] = { c0.w, c1.x, c1.y, c1.z };             // chroma bytes: Cg << 4 | Co
    float Y[16];
    Y[0] = 0.28209479177387814f;
    {
        const float C1 = 0.4886025119029199f;
        Y[1] = -C1 * y; Y[2] = C1 * z; Y[3] = -C1 * x;
        const float xx = x * x, yy = y * y, zz = z * z;
        const float C2a = 1.0925484305920792f, C2b = 0.31539156525252005f, C2c = 0.5462742152960396f;
        Y[4] = C2a * x * y; Y[5] = -C2a * y * z; Y[6] = C2b * (2.0f * zz - xx - yy); Y[7] = -C2a * x * z; Y[8] = C2c * (xx - yy);
        const float C3a = 0.5900435899266435f, C3b = 2.890611442640554f, C3c = 0.4570457994644658f,
                    C3d = 0.3731763325901154f, C3e = 1.445305721320277f;
        Y[9]  = -C3a * y * (3.0f * xx - yy); Y[10] = C3b * x * y * z; Y[11] = -C3c * y * (4.0f * zz - xx - yy);
        Y[12] = C3d * z * (2.0f * zz - 3.0f * xx - 3.0f * yy); Y[13] = -C3c * x * (4.0f * zz - xx - yy);
        Y[14] = C3e * z * (xx - yy); Y[15] = -C3a * x * (xx - 3.0f * yy);
    }
    // DC: 16-bit luma, 15-bit chroma codes = (field of k = 0) << 10 / 11 | extension bits
    const uint32_t ext = c1.w;
    const uint32_t y16 = ((c0.x & 63u) << 10) | (ext & 0x3ffu);
    const uint32_t co15 = ((c0.w & 15u) << 11) | ((ext >> 10) & 0x7ffu), cg15 = (((c0.w >> 4) & 15u) << 11) | (ext >> 21);
    const float wy = ((float)(int)y16 - 32768.0f) * (1.0f / 32767.0f), wco = ((float)(int)co15 - 16384.0f) * (1.0f / 16383.0f),
                wcg = ((float)(int)cg15 - 16384.0f) * (1.0f / 16383.0f);
    float ay = Y[0] * (sc.s[0] * wy * fabsf(wy)), aco = Y[0] * (sc.s[1] * wco * fabsf(wco)), acg = Y[0] * (sc.s[2] * wcg * fabsf(wcg));
#pragma unroll
    for (int k = 1; k < 16; ++k) {
        const int bit = 6 * k, wd = bit >> 5, sh_ = bit & 31;
        const uint32_t cy = __funnelshift_r(lw[wd], lw[wd + 1 < 4 ? wd + 1 : 3], sh_) & 63u;
        const uint32_t cb = cw[k >> 2] >> (8 * (k & 3));
        ay = fmaf(Y[k], lut[k * 64 + cy], ay);
        aco = fmaf(Y[k], lut[1024 + k * 32 + (cb & 15u)], aco);
        acg = fmaf(Y[k], lut[1024 + k * 32 + 16 + ((cb >> 4) & 15u)], acg);
    }
    const float t = ay - 0.5f * acg;
    g = acg + t;
    b = t - 0.5f * aco;
    r = b + aco;
    r = fmaxf(r + 0.5f, 0.0f); g = fmaxf(g + 0.5f, 0.0f); b = fmaxf(b + 0.5f, 0.0f);
}

// Threads per CTA (two CTAs per SM).  The fp32-record kernel on fp32 SH rows is bound by DRAM and spills at 64 registers
// (512 threads: 40 bytes of stack, 5 M local-memory warp accesses per frame that all travel to L2); 384 threads (80 registers)
// has none: 0.268 -> 0.262 ms, DRAM traffic 1.36 -> 1.27 GB.  The other variants are bound by instruction issue and keep 32 warps per SM.
__host__ __device__ constexpr int proj_threads(bool half, int shm) { return (!half && shm == 0) ? 384 : 512; }
constexpr int PROJ_WARPS_MAX = 16;
constexpr int PROJ_QCAP = 64;                              // per-warp survivor queue (entries), >= 31 + 32
constexpr int PROJ_QF = 15;                                // words per queued survivor

// where phase B takes a survivor's SH coefficients from
constexpr int SH_ROWS = 0;                                 // fp32 rows in device memory: every lane reads its own row
constexpr int SH_CODES = 1;                                // 32-byte codes of the resident scene (shcodec.cu)
constexpr int SH_STAGED = 2;                               // fp32 rows in mapped host memory: the warp copies the rows of its 32 survivors into
                                                           // shared memory with contiguous 16-byte pieces first (one lane per row over PCIe: 12 GB/s;
                                                           // contiguous pieces: 49 GB/s, the rate of a bulk copy, for the surviving rows only)
// staged row: pieces of 16 bytes when the row is a whole number of them (degrees 1, 3), else of 4 bytes; one piece of padding
// per row keeps the per-lane reads free of bank conflicts
template <int DEG> struct ShStage {
    static constexpr int ROW_W = 3 * (DEG + 1) * (DEG + 1);
    static constexpr bool V4 = ROW_W % 4 == 0;
    static constexpr int PIECES = V4 ? ROW_W / 4 : ROW_W;
    static constexpr int STRIDE_W = V4 ? 4 * (PIECES + 1) : ROW_W + 1;     // words
};
constexpr int SH_STAGE_WORDS_MAX = 32 * ShStage<3>::STRIDE_W;               // per warp

// 64-bit macro-tile span descriptor (internal): bit 63 = "not representable, rerun the row scan";
// bits 0-8 first macro-tile row r0, bits 9-10 rows-1 (<= 4 rows), then 13 bits per row:
// first column m0 (9 bits, 511 = row not touched) and columns-1 (4 bits, <= 16 columns).
#define HIGS_DESC_FALLBACK 0x8000000000000000ull

// One 256-bit store (sm_100: STG.256).  A record written as 16-byte halves reaches L2 as partial-sector writes, and L2 answers a
// partial write that misses with a fill read of the sector from DRAM: ncu counted 11.7 M write-miss sectors per frame in this
// kernel and 0.2 GB of DRAM reads nobody asked for.  A whole 32-byte sector in one store needs no fill.  p: 32-byte aligned.
__device__ __forceinline__ void st_global_256(void* p, uint4 lo, uint4 hi)
{
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 :: "l"(__cvta_generic_to_global(p)), "r"(lo.x), "r"(lo.y), "r"(lo.z), "r"(lo.w), "r"(hi.x), "r"(hi.y), "r"(hi.z), "r"(hi.w) : "memory");
}
__device__ __forceinline__ uint4 f4_bits(float a, float b, float c, float d) { return make_uint4(__float_as_uint(a), __float_as_uint(b), __float_as_uint(c), __float_as_uint(d)); }

// what phase A hands to phase B for a surviving gaussian
struct Survivor { float mux, muy, a, b, c, A, B2, C, tau, zc, o, mx, my, mz; uint32_t local; };

// The 44 input bytes of one gaussian.  All eleven words are requested up front, one iteration ahead of their use
// (register double buffer in k_project), so a warp pays one exposed DRAM round trip per 32 gaussians at most
// instead of four dependent ones (means -> quats -> scales -> opacity).
struct RawIn { float mx, my, mz, s0, s1, s2, o; float4 q; };

__device__ __forceinline__ RawIn load_raw(const float* __restrict__ means, const float* __restrict__ scales,
                                          const float* __restrict__ quats, const float* __restrict__ opac, int64_t i)
{
    RawIn r;
    r.mx = HIGS_LD(means + 3 * i); r.my = HIGS_LD(means + 3 * i + 1); r.mz = HIGS_LD(means + 3 * i + 2);
    r.q = HIGS_LD(reinterpret_cast<const float4*>(quats) + i);
    r.s0 = HIGS_LD(scales + 3 * i); r.s1 = HIGS_LD(scales + 3 * i + 1); r.s2 = HIGS_LD(scales + 3 * i + 2);
    r.o = HIGS_LD(opac + i);
    return r;
}

// Phase A: N-PROJ steps 1-10 for one gaussian; false = culled.
template <bool LEAN>
__device__ __forceinline__ bool project_cull(const RawIn& in, const FrameParams& P, Survivor& s)
{
    const float mx = in.mx, my = in.my, mz = in.mz;
    const float* V = P.V;
    // 1. camera transform
    const float xc = __fmaf_rn(V[2], mz, __fmaf_rn(V[1], my, __fmaf_rn(V[0], mx, V[3])));
    const float yc = __fmaf_rn(V[6], mz, __fmaf_rn(V[5], my, __fmaf_rn(V[4], mx, V[7])));
    const float zc = __fmaf_rn(V[10], mz, __fmaf_rn(V[9], my, __fmaf_rn(V[8], mx, V[11])));
    if (!((zc > P.near_z) && (zc <= 3.402823466e+38f))) return false;
    // 2. perspective
    const float rz = __frcp_rn(zc);
    const float xz = __fmul_rn(xc, rz), yz = __fmul_rn(yc, rz);
    const float mux = __fmaf_rn(P.fx, xz, P.cx), muy = __fmaf_rn(P.fy, yz, P.cy);
    // 3. clamp inside the Jacobian only
    const float limx = LEAN ? P.limx : __fdiv_rn(__fmul_rn(0.65f, (float)P.W), P.fx);     // LEAN: see RowScan (higs_internal.cuh)
    const float limy = LEAN ? P.limy : __fdiv_rn(__fmul_rn(0.65f, (float)P.H), P.fy);
    const float txz = fminf(limx, fmaxf(-limx, xz));
    const float tyz = fminf(limy, fmaxf(-limy, yz));
    // 4. rotation from the normalised quaternion
    const float4 q4 = in.q;
    float qw = q4.x, qx = q4.y, qy = q4.z, qz = q4.w;
    const float n2 = __fmaf_rn(qz, qz, __fmaf_rn(qy, qy, __fmaf_rn(qx, qx, __fmul_rn(qw, qw))));
    if (!finite_pos(n2)) return false;
    const float inv = __frcp_rn(__fsqrt_rn(n2));
    qw = __fmul_rn(qw, inv); qx = __fmul_rn(qx, inv); qy = __fmul_rn(qy, inv); qz = __fmul_rn(qz, inv);
    const float Q00 = __fmaf_rn(-2.0f, __fmaf_rn(qy, qy, __fmul_rn(qz, qz)), 1.0f);
    const float Q01 = __fmul_rn(2.0f, __fmaf_rn(qx, qy, -__fmul_rn(qw, qz)));
    const float Q02 = __fmul_rn(2.0f, __fmaf_rn(qx, qz, __fmul_rn(qw, qy)));
    const float Q10 = __fmul_rn(2.0f, __fmaf_rn(qx, qy, __fmul_rn(qw, qz)));
    const float Q11 = __fmaf_rn(-2.0f, __fmaf_rn(qx, qx, __fmul_rn(qz, qz)), 1.0f);
    const float Q12 = __fmul_rn(2.0f, __fmaf_rn(qy, qz, -__fmul_rn(qw, qx)));
    const float Q20 = __fmul_rn(2.0f, __fmaf_rn(qx, qz, -__fmul_rn(qw, qy)));
    const float Q21 = __fmul_rn(2.0f, __fmaf_rn(qy, qz, __fmul_rn(qw, qx)));
    const float Q22 = __fmaf_rn(-2.0f, __fmaf_rn(qx, qx, __fmul_rn(qy, qy)), 1.0f);
    // 5. M = Q diag(s)
    const float s0 = in.s0, s1 = in.s1, s2 = in.s2;
    const float M00 = __fmul_rn(Q00, s0), M01 = __fmul_rn(Q01, s1), M02 = __fmul_rn(Q02, s2);
    const float M10 = __fmul_rn(Q10, s0), M11 = __fmul_rn(Q11, s1), M12 = __fmul_rn(Q12, s2);
    const float M20 = __fmul_rn(Q20, s0), M21 = __fmul_rn(Q21, s1), M22 = __fmul_rn(Q22, s2);
    // 6. J, G = J R_view, Tm = G M
    const float J00 = __fmul_rn(P.fx, rz), J02 = __fmul_rn(-__fmul_rn(P.fx, txz), rz);
    const float J11 = __fmul_rn(P.fy, rz), J12 = __fmul_rn(-__fmul_rn(P.fy, tyz), rz);
    const float G00 = __fmaf_rn(J02, V[8], __fmul_rn(J00, V[0]));
    const float G01 = __fmaf_rn(J02, V[9], __fmul_rn(J00, V[1]));
    const float G02 = __fmaf_rn(J02, V[10], __fmul_rn(J00, V[2]));
    const float G10 = __fmaf_rn(J12, V[8], __fmul_rn(J11, V[4]));
    const float G11 = __fmaf_rn(J12, V[9], __fmul_rn(J11, V[5]));
    const float G12 = __fmaf_rn(J12, V[10], __fmul_rn(J11, V[6]));
    const float T00 = __fmaf_rn(G02, M20, __fmaf_rn(G01, M10, __fmul_rn(G00, M00)));
    const float T01 = __fmaf_rn(G02, M21, __fmaf_rn(G01, M11, __fmul_rn(G00, M01)));
    const float T02 = __fmaf_rn(G02, M22, __fmaf_rn(G01, M12, __fmul_rn(G00, M02)));
    const float T10 = __fmaf_rn(G12, M20, __fmaf_rn(G11, M10, __fmul_rn(G10, M00)));
    const float T11 = __fmaf_rn(G12, M21, __fmaf_rn(G11, M11, __fmul_rn(G10, M01)));
    const float T12 = __fmaf_rn(G12, M22, __fmaf_rn(G11, M12, __fmul_rn(G10, M02)));
    // 7. 2D covariance + 0.3 I
    const float a = __fadd_rn(__fmaf_rn(T02, T02, __fmaf_rn(T01, T01, __fmul_rn(T00, T00))), 0.3f);
    const float b = __fmaf_rn(T02, T12, __fmaf_rn(T01, T11, __fmul_rn(T00, T10)));
    const float c = __fadd_rn(__fmaf_rn(T12, T12, __fmaf_rn(T11, T11, __fmul_rn(T10, T10))), 0.3f);
    // 8. conic
    const float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
    if (!finite_pos(det)) return false;
    const float rd = __frcp_rn(det);
    const float A = __fmul_rn(c, rd), B2 = -__fmul_rn(__fadd_rn(b, b), rd), C = __fmul_rn(a, rd);
    if (!((A <= 3.402823466e+38f) && (C <= 3.402823466e+38f) && (fabsf(B2) <= 3.402823466e+38f))) return false;
    // 9. opacity threshold: alpha >= 1/255 <=> q <= tau = 2 ln(255 o)
    const float o = in.o;
    const float x255 = __fmul_rn(255.0f, o);
    if (!((x255 > 1.0f) && (x255 <= 3.402823466e+38f))) return false;
    const float tau = __fmul_rn(2.0f, ln_spec(x255));
    if (!(tau > 0.0f)) return false;
    // 10. off-screen cull on the bounding box of the threshold ellipse, on tau_s (conservative for the fp32 pixel test)
    const float tau_s = __fmul_rn(tau, __fmaf_rn(__fmul_rn(__fmul_rn(a, c), rd), 9.5367431640625e-07f, 1.0f));
    const float hx = __fsqrt_rn(__fmul_rn(tau_s, a)), hy = __fsqrt_rn(__fmul_rn(tau_s, c));
    if (!((__fadd_rn(mux, hx) > 0.0f) && (__fsub_rn(mux, hx) < (float)P.W) &&
          (__fadd_rn(muy, hy) > 0.0f) && (__fsub_rn(muy, hy) < (float)P.H))) return false;
    s.mux = mux; s.muy = muy; s.a = a; s.b = b; s.c = c; s.A = A; s.B2 = B2; s.C = C; s.tau = tau; s.zc = zc; s.o = o;
    s.mx = mx; s.my = my; s.mz = mz;
    return true;
}

// Phase B for one survivor: a2 macro-tile row scan (N-SCAN, pinned) -> private histogram + span descriptor,
// SH colour, and the two records at dense slot `slot`.
template <int DEG, bool HALF, int SHM>
__device__ __forceinline__ void emit_survivor(const Survivor& s, int64_t i, size_t slot, const float* __restrict__ sh, const float* __restrict__ lut, const ShScales& sc,
                                              const FrameParams& P, uint32_t* s_hist, float4* __restrict__ rec,
                                              uint4* __restrict__ rec16, uint4* __restrict__ bin, int lane, uint32_t n_live)
{
    constexpr bool SHC = SHM == SH_CODES;
    unsigned long long desc = 0;
    {
        RowScan rs{};
        rs.template init<SHC>(s.mux, s.muy, s.a, s.b, s.c, tau_scan(s.a, s.b, s.c, s.tau), (float)(P.mt_ty * P.tile), P.n_my);
        const float fW = (float)P.W, fH = (float)P.H;
        bool fits = (rs.r1 - rs.r0) <= 3 && P.n_mx <= 511 && rs.r0 <= 511;
        desc = (unsigned long long)(uint32_t)rs.r0 | ((unsigned long long)(uint32_t)((rs.r1 - rs.r0) & 3) << 9);
        for (int r = rs.r0; r <= rs.r1; ++r) {
            int m0, m1;
            uint32_t field = 511u;
            if (rs.template row<SHC>(r, (float)(P.mt_tx * P.tile), (float)(P.mt_ty * P.tile), fW, fH, P.n_mx, m0, m1)) {
                HIGS_ASSERT(r >= 0 && r < P.n_my && m0 >= 0 && m1 < P.n_mx);
                for (int m = m0; m <= m1; ++m) atomicAdd(&s_hist[r * P.n_mx + m], 1u);
                fits = fits && (m1 - m0) <= 15;
                field = (uint32_t)m0 | ((uint32_t)((m1 - m0) & 15) << 9);
            }
            if (r - rs.r0 <= 3) desc |= (unsigned long long)field << (11 + 13 * (r - rs.r0));
        }
        if (!fits) desc = HIGS_DESC_FALLBACK;
    }
    // 11./12. depth key, colour
    const float dx = s.mx - P.cam[0], dy = s.my - P.cam[1], dz = s.mz - P.cam[2];
    const float len2 = dx * dx + dy * dy + dz * dz;
    const float rl = len2 > 0.0f ? rsqrtf(len2) : 0.0f;
    float r, g, bl;
    if constexpr (SHC) sh32_colour(reinterpret_cast<const uint4*>(sh), i, lut, sc, dx * rl, dy * rl, dz * rl, r, g, bl);
    else if constexpr (SHM == SH_STAGED) sh_accumulate<DEG, true>(sh, dx * rl, dy * rl, dz * rl, r, g, bl);       // sh = this lane's staged row
    else sh_accumulate<DEG, false>(sh + i * (int64_t)((DEG + 1) * (DEG + 1) * 3), dx * rl, dy * rl, dz * rl, r, g, bl);
    const uint32_t key = __float_as_uint(s.zc);
    if constexpr (HALF) {
        // fp16 data path: inverse covariance as Cholesky factors L = [[l0, 0], [l1, l2]], L L^T = conic,
        // from the covariance without cancellation: l0 = sqrt(c / det), l1 = -b / (det l0), l2 = 1 / sqrt(c); prescaled by
        // sqrt(log2 e / 2) * tile so that alpha = o * exp2(-q') with q' = (l0' dx + l1' dy)^2 + (l2' dy)^2 in tile units
        // (smooth values, stored as half: approximate rsqrt is ample)  sqrt(c det) = det l0, so l0 = c r, l1 = -b r with r = rsqrt(c det)
        const float det = __fmaf_rn(s.a, s.c, -__fmul_rn(s.b, s.b));
        const float rr = rsqrtf(s.c * det);
        const float l0 = s.c * rr, l1 = -s.b * rr, l2 = rsqrtf(s.c);
        const float ks = 0.84932180f * (float)P.tile;                // sqrt(log2(e) / 2) * tile_size
        const __half2 h01 = __floats2half2_rn(l0 * ks, l1 * ks), h2o = __floats2half2_rn(l2 * ks, s.o);
        const __half2 hrg = __floats2half2_rn(r, g), hb = __floats2half2_rn(bl, 0.0f);
        st_global_256(rec16 + 2 * slot, make_uint4(__float_as_uint(s.mux), __float_as_uint(s.muy), *reinterpret_cast<const uint32_t*>(&h01), *reinterpret_cast<const uint32_t*>(&h2o)),
                      make_uint4(*reinterpret_cast<const uint32_t*>(&hrg), *reinterpret_cast<const uint32_t*>(&hb), 0u, 0u));
    }
    if (!HALF || desc == HIGS_DESC_FALLBACK) {                       // fp16 path: the fill pass reads rec only to redo the row scan of wide gaussians
        float4* rp = rec + 4 * slot;
        st_global_256(rp, f4_bits(s.mux, s.muy, s.A, s.B2), f4_bits(s.C, s.tau, SHC ? __log2f(s.o) : log2f(s.o), r));
        st_global_256(rp + 2, f4_bits(g, bl, s.a, s.b), f4_bits(s.c, __uint_as_float(key), __uint_as_float((uint32_t)i), 0.0f));
    }
    // bin records are 16 bytes: lanes 2j and 2j+1 hold neighbouring slots (the first slot of a drain is even) and the even lane
    // stores both.  Worth its four shuffles only where DRAM is the limit (fp32 records from fp32 SH rows: 0.266 -> 0.262 ms); the
    // variants bound by instruction issue lose (32-byte codes: 0.220 -> 0.237 ms) and store their own 16 bytes.
    const uint4 mine = make_uint4(key, (uint32_t)desc, (uint32_t)(desc >> 32), (uint32_t)i);
    if constexpr (HALF || SHM != SH_ROWS) { bin[slot] = mine; return; }
    const uint32_t live = n_live >= 32u ? 0xffffffffu : (1u << n_live) - 1u;
    uint4 next;
    next.x = __shfl_xor_sync(live, mine.x, 1); next.y = __shfl_xor_sync(live, mine.y, 1);
    next.z = __shfl_xor_sync(live, mine.z, 1); next.w = __shfl_xor_sync(live, mine.w, 1);
    if (!(lane & 1)) {
        if ((uint32_t)lane + 1u < n_live) st_global_256(bin + slot, mine, next);
        else bin[slot] = mine;
    }
}

// Persistent CTAs (a whole number per SM), one histogram row per CTA.  A warp claims chunks of HIGS_CHUNK = 128
// consecutive ids from a device counter, so the load balances itself and the grid never has a partial wave; the
// paper's fixed partition batch of B_p consecutive ids becomes "the chunks one CTA happened to
// claim", listed in part_list / part_desc for the fill pass.  A warp runs phase A on 32 gaussians at a time
// and queues the survivors (about 4 in 10 at paper scale) in shared memory; whenever 32 are queued it runs phase B
// on them with every lane busy.  Survivor k of chunk c gets dense slot c*HIGS_CHUNK + k: slots are monotone in the
// gaussian id, so (key, slot) order = (key, id) order (Q7).
template <int DEG, bool HALF, int SHM>
__global__ void __launch_bounds__(proj_threads(HALF, SHM), 2)
k_project(const float* __restrict__ means, const float* __restrict__ scales, const float* __restrict__ quats,
          const float* __restrict__ opac, const float* __restrict__ sh, int64_t N, const FrameParams P,
          uint32_t* __restrict__ valid_bits, float4* __restrict__ rec, uint4* __restrict__ rec16, uint4* __restrict__ bin,
          uint32_t* __restrict__ chunk_count, uint32_t* __restrict__ hist, uint32_t* __restrict__ mt_count, uint32_t* __restrict__ part_list,
          uint2* __restrict__ part_desc, int lcap, FrameHeader* __restrict__ hdr, const ShScales sc)
{
    constexpr int PROJ_THREADS = proj_threads(HALF, SHM), PROJ_WARPS = PROJ_THREADS / 32;
    extern __shared__ uint32_t s_dyn[];
    __shared__ uint32_t s_nvis, s_nlist, s_lbase;
    uint32_t* s_hist = s_dyn;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    pdl_trigger();                                                   // k_plan may be scheduled as this grid drains
    float* q = reinterpret_cast<float*>(s_dyn + ((P.n_m + 3) & ~3)) + w * (PROJ_QF * PROJ_QCAP);
    uint32_t* s_list = s_dyn + ((P.n_m + 3) & ~3) + PROJ_WARPS * PROJ_QF * PROJ_QCAP;   // [lcap] chunks this CTA claimed
    float* s_lut = reinterpret_cast<float*>(s_list + lcap);         // [1536] dequantisation tables of the 32-byte SH code (SHC only)
    constexpr bool SHC = SHM == SH_CODES;
    uint32_t* s_stage = reinterpret_cast<uint32_t*>(s_lut + 1536) + w * SH_STAGE_WORDS_MAX;   // SH_STAGED only
    if constexpr (SHC) {
        for (int e = threadIdx.x; e < 1536; e += PROJ_THREADS) {
            const bool luma = e < 1024;
            const int k = luma ? e >> 6 : (e - 1024) >> 5, c = luma ? 0 : 1 + (((e - 1024) >> 4) & 1), code = luma ? e & 63 : e & 15;
            const float wq = luma ? (float)(code - 32) * (1.0f / 31.0f) : (float)(code - 8) * (1.0f / 7.0f);
            s_lut[e] = sc.s[k * 3 + c] * wq * fabsf(wq);
        }
    }
    for (int m = threadIdx.x; m < P.n_m; m += PROJ_THREADS) s_hist[m] = 0;
    if (threadIdx.x == 0) { s_nvis = 0; s_nlist = 0; }
    __syncthreads();
    const uint32_t n_chunks = (uint32_t)((N + HIGS_CHUNK - 1) / HIGS_CHUNK);
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t n_mine = 0;

    for (;;) {
        uint32_t chunk = 0xffffffffu;
        if (lane == 0) {                                             // a list entry first, then the chunk that goes in it
            const uint32_t e = atomicAdd(&s_nlist, 1u);
            if (e < (uint32_t)lcap) {
                chunk = atomicAdd(&hdr->proj_cursor, 1u);
                s_list[e] = chunk < n_chunks ? chunk : 0xffffffffu;
            }
        }
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk >= n_chunks) break;
        const int64_t c0 = (int64_t)chunk * HIGS_CHUNK;
        const size_t slot0 = (size_t)c0;
        uint32_t head = 0, tail = 0;

        auto drain = [&](uint32_t n_live) {                          // phase B on queue entries head .. head+n_live-1
            if constexpr (SHM == SH_STAGED) {
                using SG = ShStage<DEG>;
                const uint32_t my_local = (uint32_t)lane < n_live ? __float_as_uint(q[14 * PROJ_QCAP + (int)((head + lane) & (PROJ_QCAP - 1))]) : 0u;
                const uint32_t n_pieces = n_live * SG::PIECES;
                for (uint32_t p0 = 0; p0 < n_pieces; p0 += 32) {     // piece p = row p / PIECES, part p % PIECES: consecutive lanes, consecutive bytes
                    const uint32_t p = p0 + lane;
                    const uint32_t r = min(p / SG::PIECES, n_live - 1u), part = p - r * SG::PIECES;
                    const int64_t id = c0 + __shfl_sync(0xffffffffu, my_local, (int)r);
                    if (p < n_pieces) {
                        if constexpr (SG::V4) *reinterpret_cast<uint4*>(s_stage + r * SG::STRIDE_W + 4 * part) = __ldg(reinterpret_cast<const uint4*>(sh + id * SG::ROW_W) + part);
                        else s_stage[r * SG::STRIDE_W + part] = __ldg(reinterpret_cast<const uint32_t*>(sh + id * SG::ROW_W) + part);
                    }
                }
                __syncwarp();
            }
            if ((uint32_t)lane < n_live) {
                const int e = (int)((head + lane) & (PROJ_QCAP - 1));
                Survivor s;
                s.mux = q[0 * PROJ_QCAP + e]; s.muy = q[1 * PROJ_QCAP + e]; s.a = q[2 * PROJ_QCAP + e]; s.b = q[3 * PROJ_QCAP + e];
                s.c = q[4 * PROJ_QCAP + e]; s.A = q[5 * PROJ_QCAP + e]; s.B2 = q[6 * PROJ_QCAP + e]; s.C = q[7 * PROJ_QCAP + e];
                s.tau = q[8 * PROJ_QCAP + e]; s.zc = q[9 * PROJ_QCAP + e]; s.o = q[10 * PROJ_QCAP + e];
                s.mx = q[11 * PROJ_QCAP + e]; s.my = q[12 * PROJ_QCAP + e]; s.mz = q[13 * PROJ_QCAP + e];
                s.local = __float_as_uint(q[14 * PROJ_QCAP + e]);
                const float* shp = SHM == SH_STAGED ? reinterpret_cast<const float*>(s_stage + lane * ShStage<DEG>::STRIDE_W) : sh;
                emit_survivor<DEG, HALF, SHM>(s, c0 + s.local, slot0 + head + lane, shp, s_lut, sc, P, s_hist, rec, rec16, bin, lane, n_live);
            }
            head += n_live;
            __syncwarp();
        };

        RawIn nxt = {};
        if (c0 + lane < N) nxt = load_raw(means, scales, quats, opac, c0 + lane);
        for (int it = 0; it < HIGS_CHUNK / 32; ++it) {
            const int64_t i = c0 + it * 32 + lane;
            if (c0 + it * 32 >= N) break;                            // warp-uniform
            const RawIn cur = nxt;
            if (it + 1 < HIGS_CHUNK / 32 && i + 32 < N) nxt = load_raw(means, scales, quats, opac, i + 32);
            Survivor s;
            const bool ok = (i < N) && project_cull<SHC>(cur, P, s);
            const uint32_t vmask = __ballot_sync(0xffffffffu, ok);
            if (lane == 0) valid_bits[i >> 5] = vmask;               // chunk bases are multiples of 32
            if (ok) {
                const int e = (int)((tail + __popc(vmask & lt)) & (PROJ_QCAP - 1));
                q[0 * PROJ_QCAP + e] = s.mux; q[1 * PROJ_QCAP + e] = s.muy; q[2 * PROJ_QCAP + e] = s.a; q[3 * PROJ_QCAP + e] = s.b;
                q[4 * PROJ_QCAP + e] = s.c; q[5 * PROJ_QCAP + e] = s.A; q[6 * PROJ_QCAP + e] = s.B2; q[7 * PROJ_QCAP + e] = s.C;
                q[8 * PROJ_QCAP + e] = s.tau; q[9 * PROJ_QCAP + e] = s.zc; q[10 * PROJ_QCAP + e] = s.o;
                q[11 * PROJ_QCAP + e] = s.mx; q[12 * PROJ_QCAP + e] = s.my; q[13 * PROJ_QCAP + e] = s.mz;
                q[14 * PROJ_QCAP + e] = __uint_as_float((uint32_t)(it * 32 + lane));
            }
            tail += __popc(vmask);
            __syncwarp();
            if (tail - head >= 32u) drain(32u);
        }
        if (tail > head) drain(tail - head);
        if (lane == 0) chunk_count[chunk] = tail;
        n_mine += tail;
    }
    if (lane == 0 && n_mine) atomicAdd(&s_nvis, n_mine);
    __syncthreads();
    // this CTA's partition batch = the chunks it claimed: compacted into the global list for the fill pass
    if (w == 0) {
        const uint32_t n_e = min(s_nlist, (uint32_t)lcap);
        uint32_t n_valid = 0;
        for (uint32_t e0 = 0; e0 < n_e; e0 += 32) n_valid += __popc(__ballot_sync(0xffffffffu, e0 + lane < n_e && s_list[e0 + lane] != 0xffffffffu));
        if (lane == 0) {
            s_lbase = atomicAdd(&hdr->part_list_cursor, n_valid);
            part_desc[blockIdx.x] = make_uint2(s_lbase, n_valid);
        }
        __syncwarp();
        uint32_t at = s_lbase;
        for (uint32_t e0 = 0; e0 < n_e; e0 += 32) {
            const uint32_t c = e0 + lane < n_e ? s_list[e0 + lane] : 0xffffffffu;
            const uint32_t ok = __ballot_sync(0xffffffffu, c != 0xffffffffu);
            if (c != 0xffffffffu) part_list[at + __popc(ok & lt)] = c;
            at += __popc(ok);
        }
    }
    uint32_t* row = hist + (size_t)blockIdx.x * P.n_m;
    for (int m = threadIdx.x; m < P.n_m; m += PROJ_THREADS) {
        const uint32_t h = s_hist[m];
        row[m] = h;
        if (h) atomicAdd(&mt_count[m], h);                           // segment sizes accumulate here: no scan over the batches
    }
    if (threadIdx.x == 0 && s_nvis) atomicAdd(&hdr->n_visible, s_nvis);
}

} // namespace

static size_t project_smem_bytes(int n_m, int lcap, int warps, bool staged = false)
{
    return sizeof(uint32_t) * (size_t)((n_m + 3) & ~3) + sizeof(float) * (size_t)warps * PROJ_QF * PROJ_QCAP + sizeof(uint32_t) * (size_t)lcap
           + sizeof(float) * 1536 + (staged ? sizeof(uint32_t) * (size_t)warps * SH_STAGE_WORDS_MAX : 0);
}

// list capacity of one partition CTA: four times its fair share of the chunks, so a CTA that fills its list and
// retires early always leaves others with room (sum of capacities > chunks: every chunk finds a taker)
int higs_part_lcap(int64_t n_chunks, int grid) { return (int)(4 * ((n_chunks + grid - 1) / grid) + 2 * PROJ_WARPS_MAX); }

// CTAs of the partition passes (project+count, fill) for N gaussians: a whole number per SM, fewer only when
// there are not enough chunks to give every warp one
int higs_part_grid(const higs_ctx* ctx, int64_t N)
{
    const int64_t n_chunks = (N + HIGS_CHUNK - 1) / HIGS_CHUNK;
    const int64_t want = (n_chunks + PROJ_WARPS_MAX - 1) / PROJ_WARPS_MAX;
    const int64_t cap = (int64_t)ctx->n_part_max;
    return (int)(want < 1 ? 1 : (want > cap ? cap : want));
}

int launch_project(higs_ctx* ctx, const FrameParams& P, const float* means, const float* scales, const float* quats,
                   const float* opac, const float* sh, int sh_mode, int64_t N, cudaStream_t st)
{
    if (N <= 0) return HIGS_OK;
    if (sh_mode == HIGS_SH_STAGED && !ctx->proj_staged_ok) return HIGS_E_ARG;
    const unsigned grid = (unsigned)higs_part_grid(ctx, N);
    const int lcap = higs_part_lcap((N + HIGS_CHUNK - 1) / HIGS_CHUNK, (int)grid);
#define HIGS_PROJ_(D, H, C) k_project<D, H, C><<<grid, proj_threads(H, C), project_smem_bytes(P.n_m, lcap, proj_threads(H, C) / 32, C == SH_STAGED), st>>>(means, scales, quats, opac, sh, N, P, ctx->valid_bits, ctx->rec, \
                                                                   ctx->rec16, ctx->bin, ctx->chunk_count, ctx->hist, ctx->mt_count, ctx->part_list, ctx->part_desc, lcap, ctx->hdr, sc)
#define HIGS_PROJ(D) do { if (sh_mode == HIGS_SH_STAGED) { if (P.flags & HIGS_FLAG_FP16) HIGS_PROJ_(D, true, SH_STAGED); else HIGS_PROJ_(D, false, SH_STAGED); } \
                          else if (P.flags & HIGS_FLAG_FP16) HIGS_PROJ_(D, true, SH_ROWS); else HIGS_PROJ_(D, false, SH_ROWS); } while (0)
    ShScales sc;
    memset(&sc, 0, sizeof(sc));
    if (sh_mode == HIGS_SH_CODES) {                                  // sh = the 32-byte codes of the resident scene (degree 3)
        memcpy(sc.s, ctx->sh32_scales_host, sizeof(sc.s));
        if (P.flags & HIGS_FLAG_FP16) HIGS_PROJ_(3, true, SH_CODES); else HIGS_PROJ_(3, false, SH_CODES);
    } else switch (P.degree) {
        case 0: HIGS_PROJ(0); break;
        case 1: HIGS_PROJ(1); break;
        case 2: HIGS_PROJ(2); break;
        default: HIGS_PROJ(3); break;
    }
#undef HIGS_PROJ
#undef HIGS_PROJ_
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}

int higs_project_smem_setup(higs_ctx* ctx)
{
    // The chunk list of a CTA (four times its fair share of the chunks of max_gaussians) is part of its shared memory, and the
    // fair share depends on how many CTAs the grid has: the largest number of CTAs per SM whose list still lets that many CTAs
    // be resident (sizing the list for one CTA per SM made it so long at 75 M gaussians that only one fitted).  The 512-thread
    // variants carry the largest queue: they decide.
    int per_sm = 1, lcap_max = 0;
    for (int c = 4; c >= 1; --c) {
        lcap_max = higs_part_lcap(ctx->n_chunks_max, ctx->n_sm * c) > 6 * PROJ_WARPS_MAX ? higs_part_lcap(ctx->n_chunks_max, ctx->n_sm * c) : 6 * PROJ_WARPS_MAX;
        const size_t b = project_smem_bytes(ctx->max_nm, lcap_max, PROJ_WARPS_MAX);
        int occ = 0;
        if (cudaFuncSetAttribute(k_project<3, true, SH_ROWS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)b) != cudaSuccess) { cudaGetLastError(); continue; }
        HIGS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_project<3, true, SH_ROWS>, proj_threads(true, SH_ROWS), b));
        per_sm = c;
        if (occ >= c) break;
    }
    const int bytes = (int)project_smem_bytes(ctx->max_nm, lcap_max, PROJ_WARPS_MAX);
#define HIGS_ATTR(D, H, C) HIGS_CUDA(ctx, cudaFuncSetAttribute(k_project<D, H, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))
    HIGS_ATTR(0, false, SH_ROWS); HIGS_ATTR(1, false, SH_ROWS); HIGS_ATTR(2, false, SH_ROWS); HIGS_ATTR(3, false, SH_ROWS);
    HIGS_ATTR(0, true, SH_ROWS); HIGS_ATTR(1, true, SH_ROWS); HIGS_ATTR(2, true, SH_ROWS); HIGS_ATTR(3, true, SH_ROWS);
    HIGS_ATTR(3, false, SH_CODES); HIGS_ATTR(3, true, SH_CODES);
#undef HIGS_ATTR
    // the staged-row variants (mapped host memory) need room for the rows of 32 survivors per warp; without it
    // higs_render_host keeps uploading the SH array
    int optin = 0;
    HIGS_CUDA(ctx, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device));
    const int bytes_staged = (int)project_smem_bytes(ctx->max_nm, lcap_max, PROJ_WARPS_MAX, true);
    ctx->proj_staged_ok = bytes_staged <= optin;
    if (ctx->proj_staged_ok) {
#define HIGS_ATTR(D, H) HIGS_CUDA(ctx, cudaFuncSetAttribute(k_project<D, H, SH_STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes_staged))
        HIGS_ATTR(0, false); HIGS_ATTR(1, false); HIGS_ATTR(2, false); HIGS_ATTR(3, false);
        HIGS_ATTR(0, true); HIGS_ATTR(1, true); HIGS_ATTR(2, true); HIGS_ATTR(3, true);
#undef HIGS_ATTR
    }
    ctx->n_part_max = ctx->n_sm * per_sm;
    return HIGS_OK;
}
