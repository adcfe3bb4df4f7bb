// project.cu -- step a1: fused EWA projection + cull + SH colour (section 4.2:
// "Each thread processes one gaussian end-to-end: camera-space transformation, 2D covariance via
// Jacobian projection, ... inline view-direction computation, and degree-3 spherical harmonics
// evaluation.  The outputs -- 2D positions, ... conics, colors, and a compact per-warp visibility
// bitfield -- are consumed by the partitioning and rasterization stages.")
//
// HBM-bound: 44 B read per gaussian + 12*K B of SH read and 80 B written per *visible* gaussian.
// Everything that later decides an integer (cull, macro-tile set, depth key, the 1/255 skip) follows
// the pinned fp32 sequence N-PROJ of DESIGN.md section 3, one correctly rounded op per written op:
// the __f*_rn intrinsics are never contracted into FMAs by nvcc.
#include <stdio.h>
#include "higs_internal.cuh"

namespace {

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
template <int DEG>
__device__ __forceinline__ void sh_accumulate(const float* __restrict__ shp, float x, float y, float z,
                                              float& r, float& g, float& b)
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    float c[K * 3];
    if constexpr (DEG == 3 || DEG == 1) {                        // 192 B / 48 B rows: 16-byte aligned
        const float4* p4 = reinterpret_cast<const float4*>(shp);
#pragma unroll
        for (int k = 0; k < K * 3 / 4; ++k) {
            float4 v = __ldcs(p4 + k);
            c[4 * k] = v.x; c[4 * k + 1] = v.y; c[4 * k + 2] = v.z; c[4 * k + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < K * 3; ++k) c[k] = __ldcs(shp + k);
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

template <int DEG>
__global__ void __launch_bounds__(256)
k_project(const float* __restrict__ means, const float* __restrict__ scales, const float* __restrict__ quats,
          const float* __restrict__ opac, const float* __restrict__ sh, int64_t N, const FrameParams P,
          uint32_t* __restrict__ valid_bits, float4* __restrict__ geo, float4* __restrict__ ras)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool ok = i < N;
    float mx = 0, my = 0, mz = 0;
    float mux = 0, muy = 0, a = 0, b = 0, c = 0, A = 0, B2 = 0, C = 0, tau = 0, zc = 0, o = 0;
    if (ok) {
        mx = __ldcs(means + 3 * i); my = __ldcs(means + 3 * i + 1); mz = __ldcs(means + 3 * i + 2);
        const float* V = P.V;
        // 1. camera transform
        float xc = __fmaf_rn(V[2], mz, __fmaf_rn(V[1], my, __fmaf_rn(V[0], mx, V[3])));
        float yc = __fmaf_rn(V[6], mz, __fmaf_rn(V[5], my, __fmaf_rn(V[4], mx, V[7])));
        zc = __fmaf_rn(V[10], mz, __fmaf_rn(V[9], my, __fmaf_rn(V[8], mx, V[11])));
        ok = (zc > P.near_z) && (zc <= 3.402823466e+38f);
        if (ok) {
            // 2. perspective
            float rz = __frcp_rn(zc);
            float xz = __fmul_rn(xc, rz), yz = __fmul_rn(yc, rz);
            mux = __fmaf_rn(P.fx, xz, P.cx); muy = __fmaf_rn(P.fy, yz, P.cy);
            // 3. clamp inside the Jacobian only
            float limx = __fdiv_rn(__fmul_rn(0.65f, (float)P.W), P.fx);
            float limy = __fdiv_rn(__fmul_rn(0.65f, (float)P.H), P.fy);
            float txz = fminf(limx, fmaxf(-limx, xz));
            float tyz = fminf(limy, fmaxf(-limy, yz));
            // 4. rotation from the normalised quaternion
            float4 q4 = __ldcs(reinterpret_cast<const float4*>(quats) + i);
            float qw = q4.x, qx = q4.y, qy = q4.z, qz = q4.w;
            float n2 = __fmaf_rn(qz, qz, __fmaf_rn(qy, qy, __fmaf_rn(qx, qx, __fmul_rn(qw, qw))));
            ok = finite_pos(n2);
            if (ok) {
                float inv = __frcp_rn(__fsqrt_rn(n2));
                qw = __fmul_rn(qw, inv); qx = __fmul_rn(qx, inv); qy = __fmul_rn(qy, inv); qz = __fmul_rn(qz, inv);
                float Q00 = __fmaf_rn(-2.0f, __fmaf_rn(qy, qy, __fmul_rn(qz, qz)), 1.0f);
                float Q01 = __fmul_rn(2.0f, __fmaf_rn(qx, qy, -__fmul_rn(qw, qz)));
                float Q02 = __fmul_rn(2.0f, __fmaf_rn(qx, qz, __fmul_rn(qw, qy)));
                float Q10 = __fmul_rn(2.0f, __fmaf_rn(qx, qy, __fmul_rn(qw, qz)));
                float Q11 = __fmaf_rn(-2.0f, __fmaf_rn(qx, qx, __fmul_rn(qz, qz)), 1.0f);
                float Q12 = __fmul_rn(2.0f, __fmaf_rn(qy, qz, -__fmul_rn(qw, qx)));
                float Q20 = __fmul_rn(2.0f, __fmaf_rn(qx, qz, -__fmul_rn(qw, qy)));
                float Q21 = __fmul_rn(2.0f, __fmaf_rn(qy, qz, __fmul_rn(qw, qx)));
                float Q22 = __fmaf_rn(-2.0f, __fmaf_rn(qx, qx, __fmul_rn(qy, qy)), 1.0f);
                // 5. M = Q diag(s)
                float s0 = __ldcs(scales + 3 * i), s1 = __ldcs(scales + 3 * i + 1), s2 = __ldcs(scales + 3 * i + 2);
                float M00 = __fmul_rn(Q00, s0), M01 = __fmul_rn(Q01, s1), M02 = __fmul_rn(Q02, s2);
                float M10 = __fmul_rn(Q10, s0), M11 = __fmul_rn(Q11, s1), M12 = __fmul_rn(Q12, s2);
                float M20 = __fmul_rn(Q20, s0), M21 = __fmul_rn(Q21, s1), M22 = __fmul_rn(Q22, s2);
                // 6. J, G = J R_view, Tm = G M
                float J00 = __fmul_rn(P.fx, rz), J02 = __fmul_rn(-__fmul_rn(P.fx, txz), rz);
                float J11 = __fmul_rn(P.fy, rz), J12 = __fmul_rn(-__fmul_rn(P.fy, tyz), rz);
                float G00 = __fmaf_rn(J02, V[8], __fmul_rn(J00, V[0]));
                float G01 = __fmaf_rn(J02, V[9], __fmul_rn(J00, V[1]));
                float G02 = __fmaf_rn(J02, V[10], __fmul_rn(J00, V[2]));
                float G10 = __fmaf_rn(J12, V[8], __fmul_rn(J11, V[4]));
                float G11 = __fmaf_rn(J12, V[9], __fmul_rn(J11, V[5]));
                float G12 = __fmaf_rn(J12, V[10], __fmul_rn(J11, V[6]));
                float T00 = __fmaf_rn(G02, M20, __fmaf_rn(G01, M10, __fmul_rn(G00, M00)));
                float T01 = __fmaf_rn(G02, M21, __fmaf_rn(G01, M11, __fmul_rn(G00, M01)));
                float T02 = __fmaf_rn(G02, M22, __fmaf_rn(G01, M12, __fmul_rn(G00, M02)));
                float T10 = __fmaf_rn(G12, M20, __fmaf_rn(G11, M10, __fmul_rn(G10, M00)));
                float T11 = __fmaf_rn(G12, M21, __fmaf_rn(G11, M11, __fmul_rn(G10, M01)));
                float T12 = __fmaf_rn(G12, M22, __fmaf_rn(G11, M12, __fmul_rn(G10, M02)));
                // 7. 2D covariance + 0.3 I
                a = __fadd_rn(__fmaf_rn(T02, T02, __fmaf_rn(T01, T01, __fmul_rn(T00, T00))), 0.3f);
                b = __fmaf_rn(T02, T12, __fmaf_rn(T01, T11, __fmul_rn(T00, T10)));
                c = __fadd_rn(__fmaf_rn(T12, T12, __fmaf_rn(T11, T11, __fmul_rn(T10, T10))), 0.3f);
                // 8. conic
                float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
                ok = finite_pos(det);
                if (ok) {
                    float rd = __frcp_rn(det);
                    A = __fmul_rn(c, rd); B2 = -__fmul_rn(__fadd_rn(b, b), rd); C = __fmul_rn(a, rd);
                    ok = (A <= 3.402823466e+38f) && (C <= 3.402823466e+38f) && (fabsf(B2) <= 3.402823466e+38f);
                }
                if (ok) {
                    // 9. opacity threshold: alpha >= 1/255 <=> q <= tau = 2 ln(255 o)
                    o = __ldcs(opac + i);
                    float x255 = __fmul_rn(255.0f, o);
                    ok = (x255 > 1.0f) && (x255 <= 3.402823466e+38f);
                    if (ok) {
                        tau = __fmul_rn(2.0f, ln_spec(x255));
                        ok = tau > 0.0f;
                    }
                }
                if (ok) {
                    // 10. off-screen cull on the threshold ellipse's bounding box
                    float hx = __fsqrt_rn(__fmul_rn(tau, a)), hy = __fsqrt_rn(__fmul_rn(tau, c));
                    ok = (__fadd_rn(mux, hx) > 0.0f) && (__fsub_rn(mux, hx) < (float)P.W) &&
                         (__fadd_rn(muy, hy) > 0.0f) && (__fsub_rn(muy, hy) < (float)P.H);
                }
            }
        }
    }
    const uint32_t vmask = __ballot_sync(0xffffffffu, ok);
    if ((threadIdx.x & 31) == 0 && i < ((N + 31) / 32) * 32) valid_bits[i >> 5] = vmask;
    if (!ok) return;
    // 11./12. depth key, colour
    float dx = mx - P.cam[0], dy = my - P.cam[1], dz = mz - P.cam[2];
    float len2 = dx * dx + dy * dy + dz * dz;
    float rl = len2 > 0.0f ? rsqrtf(len2) : 0.0f;
    float r, g, bl;
    sh_accumulate<DEG>(sh + i * (int64_t)((DEG + 1) * (DEG + 1) * 3), dx * rl, dy * rl, dz * rl, r, g, bl);
    float4* gp = geo + 2 * i;
    gp[0] = make_float4(mux, muy, a, b);
    gp[1] = make_float4(c, tau, __uint_as_float(__float_as_uint(zc)), 0.0f);
    float4* rp = ras + 3 * i;
    rp[0] = make_float4(mux, muy, A, B2);
    rp[1] = make_float4(C, tau, log2f(o), r);
    rp[2] = make_float4(g, bl, 0.0f, 0.0f);
}

} // namespace

int launch_project(higs_ctx* ctx, const FrameParams& P, const float* means, const float* scales, const float* quats,
                   const float* opac, const float* sh, int64_t N, cudaStream_t st)
{
    if (N <= 0) return HIGS_OK;
    const unsigned grid = (unsigned)((N + 255) / 256);
    switch (P.degree) {
        case 0: k_project<0><<<grid, 256, 0, st>>>(means, scales, quats, opac, sh, N, P, ctx->valid_bits, ctx->geo, ctx->ras); break;
        case 1: k_project<1><<<grid, 256, 0, st>>>(means, scales, quats, opac, sh, N, P, ctx->valid_bits, ctx->geo, ctx->ras); break;
        case 2: k_project<2><<<grid, 256, 0, st>>>(means, scales, quats, opac, sh, N, P, ctx->valid_bits, ctx->geo, ctx->ras); break;
        default: k_project<3><<<grid, 256, 0, st>>>(means, scales, quats, opac, sh, N, P, ctx->valid_bits, ctx->geo, ctx->ras); break;
    }
    HIGS_LAUNCHED(ctx);
    return HIGS_OK;
}
