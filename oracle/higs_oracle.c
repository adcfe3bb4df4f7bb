/*
 * higs_oracle.c -- plain, slow, obviously-correct CPU oracle for the HiGS forward render path
 * (arxiv/paper_2606_00352, "HiGS: A Hierarchical Rendering Architecture for Real-Time 3D
 * Gaussian Splatting").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with the CUDA path under paper_2606_00352_b200/ and neither
 * imports the other.  It is never tuned for speed.
 *
 * What it computes (DESIGN.md sections 2-3 give the readings of the paper this follows):
 *
 *  O-IMG   the image HiGS reaches exactly ("preserving exact front-to-back alpha compositing",
 *          PAPER.md:13, 55, 127): per pixel centre, all gaussians surviving the cull in
 *          ascending (depth key, id) order, alpha = min(0.99, o*exp(-q/2)),
 *          contributions below 1/255 skipped, C += T*alpha*rgb, T *= 1-alpha,
 *          stop once T < 1e-4.  orc_render() is the gaussian-major,
 *          untiled form; orc_brute() is the every-pixel-times-every-gaussian form with no
 *          bounding box at all; orc_render_batched() follows the method itself (per
 *          macro-tile sorted lists, batches of B_r, Eq. (1) merge).
 *  O-LIST  the integer lists the method builds, step by step: per-gaussian cull + depth key
 *          (PAPER.md:243, 255), macro-tile row scan, per-macro-tile
 *          counts/offsets, (key,id)-sorted segments,
 *          batch boundaries ceil(n/B_r).
 *
 * Precision.  Everything that decides an integer (cull, macro-tile set, depth key, the 1/255
 * skip test) is evaluated in IEEE binary32 with the op order written in DESIGN.md section 3
 * ("pinned arithmetic"): one rounding per written op, fmaf() where an fma is written, and
 * this file MUST be compiled with -ffp-contract=off -fno-fast-math.  Everything smooth
 * (SH colour, alpha, compositing) is fp64.  orc_project_f64() is the same projection written
 * as the plain fp64 definition; the tests use it to pin the fp32 sequence.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms for one isotropic gaussian, EWA
 * covariance on/off axis, two-gaussian compositing by hand, the 0.99 clamp, termination
 * counts, monotone T, SH orthonormality by quadrature, row scan vs. an independent
 * min-of-quadratic-over-rectangle test, lists vs. numpy sort, orc_render == orc_brute ==
 * orc_render_batched.  Parity unpinned: image quality on the paper's real scenes (Table 5),
 * which needs datasets that are not available.
 */
#include <math.h>
#include <float.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <pthread.h>

/* macro-tile = 8x4 render tiles of 8x8 px = 64x32 px, PAPER.md:73 (128x64 px in the 16x16-tile variant, Table 2) */
#define ORC_EPS_T 1e-4   /* transmittance threshold epsilon, reading Q1 */
#define ORC_ALPHA_MAX 0.99

/* geo record, 9 floats per gaussian: mux, muy, a, b, c (2D covariance), tau, hx, hy, tau_s.
 * tau decides the per-pixel 1/255 skip; tau_s >= tau is the same threshold with the margin the
 * bounding box and the row scan need to stay conservative (see project_one step 9). */
enum { G_MUX = 0, G_MUY, G_A, G_B, G_C, G_TAU, G_HX, G_HY, G_TAUS, G_STRIDE };

static inline uint32_t f2u(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* ---------------------------------------------------------------------------------------
 * ln_spec: reproducible natural log for x in (1, 255] (N-LN).
 * frexp + atanh series, every op a single fp32 rounding.
 * ------------------------------------------------------------------------------------- */
float orc_ln_spec(float x)
{
    int e;
    float mant = frexpf(x, &e);            /* x = mant * 2^e, mant in [0.5, 1) */
    if (mant < 0.70710678f) { mant = 2.0f * mant; e = e - 1; }
    float f = mant - 1.0f;
    float s = f / (2.0f + f);
    float z = s * s;
    float p = 1.0f / 11.0f;
    p = p * z; p = p + 1.0f / 9.0f;
    p = p * z; p = p + 1.0f / 7.0f;
    p = p * z; p = p + 1.0f / 5.0f;
    p = p * z; p = p + 1.0f / 3.0f;
    p = p * z; p = p + 1.0f;
    float hi = (float)e * 0.69314718f;
    float lo = (2.0f * s) * p;
    return hi + lo;
}

/* ---------------------------------------------------------------------------------------
 * Real spherical harmonics, degree <= 3, in the convention of the public 3DGS models the
 * paper renders ("degree-3 spherical harmonics evaluation").
 * d = unit direction from the camera centre to the gaussian mean.
 * ------------------------------------------------------------------------------------- */
void orc_sh_basis(const double d[3], double Y[16])
{
    const double PI = 3.14159265358979323846;
    const double n = sqrt(PI);
    const double x = d[0], y = d[1], z = d[2];
    const double xx = x * x, yy = y * y, zz = z * z;
    const double C0 = 1.0 / (2.0 * n);
    const double C1 = sqrt(3.0) / (2.0 * n);
    const double C2a = sqrt(15.0) / (2.0 * n), C2b = sqrt(5.0) / (4.0 * n), C2c = sqrt(15.0) / (4.0 * n);
    const double C3a = sqrt(35.0 / 2.0) / (4.0 * n), C3b = sqrt(105.0) / (2.0 * n),
                 C3c = sqrt(21.0 / 2.0) / (4.0 * n), C3d = sqrt(7.0) / (4.0 * n),
                 C3e = sqrt(105.0) / (4.0 * n);
    Y[0] = C0;
    Y[1] = -C1 * y;  Y[2] = C1 * z;  Y[3] = -C1 * x;
    Y[4] = C2a * x * y;
    Y[5] = -C2a * y * z;
    Y[6] = C2b * (2.0 * zz - xx - yy);
    Y[7] = -C2a * x * z;
    Y[8] = C2c * (xx - yy);
    Y[9]  = -C3a * y * (3.0 * xx - yy);
    Y[10] = C3b * x * y * z;
    Y[11] = -C3c * y * (4.0 * zz - xx - yy);
    Y[12] = C3d * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);
    Y[13] = -C3c * x * (4.0 * zz - xx - yy);
    Y[14] = C3e * z * (xx - yy);
    Y[15] = -C3a * x * (xx - 3.0 * yy);
}

/* rgb = max(0, 0.5 + sum_k Y_k(dir) * sh[k][:]), no upper clamp (reading Q12). fp64. */
static void sh_colour(const float* mean, const float* cam_pos, const float* sh, int degree, double rgb[3])
{
    double d[3] = { (double)mean[0] - (double)cam_pos[0], (double)mean[1] - (double)cam_pos[1],
                    (double)mean[2] - (double)cam_pos[2] };
    double len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (len > 0.0) { d[0] /= len; d[1] /= len; d[2] /= len; }
    double Y[16];
    orc_sh_basis(d, Y);
    int K = (degree + 1) * (degree + 1);
    for (int ch = 0; ch < 3; ++ch) {
        double acc = 0.5;
        for (int k = 0; k < K; ++k) acc += Y[k] * (double)sh[k * 3 + ch];
        rgb[ch] = acc > 0.0 ? acc : 0.0;
    }
}

/* ---------------------------------------------------------------------------------------
 * N-PROJ: per-gaussian EWA projection + cull, fp32 pinned sequence.
 * cam = 20 floats: view[12] (row-major 3x4 [R|t]), fx, fy, cx, cy, near_z, cam_pos[3].
 * Outputs per gaussian i (written for valid gaussians; zeroed otherwise):
 *   valid[i]   1 / 0          reason[i] (may be NULL): 0 ok, 1 near, 2 quaternion, 3 det,
 *                              4 opacity, 5 off-screen
 *   key[i]     bits(z_cam)    (raw IEEE-754 bits, unsigned order = depth order)
 *   geo[i][9]  mux, muy, a, b, c, tau, hx, hy, tau_s
 *   conic[i][3] A, B2, C      (q = A dx^2 + B2 dx dy + C dy^2)
 *   rgb[i][3]  fp64 colour
 * Returns the number of valid gaussians.
 * ------------------------------------------------------------------------------------- */
static int project_one(const float* m, const float* s, const float* qt, float o,
                       const float* cam, int W, int H,
                       uint32_t* key, float* geo, float* conic)
{
    const float* V = cam;
    const float fx = cam[12], fy = cam[13], cx = cam[14], cy = cam[15], near_z = cam[16];
    const float mx = m[0], my = m[1], mz = m[2];
    /* 1. camera transform */
    float xc = fmaf(V[2], mz, fmaf(V[1], my, fmaf(V[0], mx, V[3])));
    float yc = fmaf(V[6], mz, fmaf(V[5], my, fmaf(V[4], mx, V[7])));
    float zc = fmaf(V[10], mz, fmaf(V[9], my, fmaf(V[8], mx, V[11])));
    if (!(zc > near_z) || !(zc <= FLT_MAX)) return 1;
    /* 2. perspective */
    float rz = 1.0f / zc;
    float xz = xc * rz, yz = yc * rz;
    float mux = fmaf(fx, xz, cx), muy = fmaf(fy, yz, cy);
    /* 3. clamp of x/z, y/z inside the Jacobian only (reading Q11) */
    float limx = (0.65f * (float)W) / fx, limy = (0.65f * (float)H) / fy;
    float txz = fminf(limx, fmaxf(-limx, xz));
    float tyz = fminf(limy, fmaxf(-limy, yz));
    /* 4. rotation from the normalised quaternion (w,x,y,z) */
    float qw = qt[0], qx = qt[1], qy = qt[2], qz = qt[3];
    float n2 = fmaf(qz, qz, fmaf(qy, qy, fmaf(qx, qx, qw * qw)));
    if (!(n2 > 0.0f) || !(n2 <= FLT_MAX)) return 2;
    float inv = 1.0f / sqrtf(n2);
    qw = qw * inv; qx = qx * inv; qy = qy * inv; qz = qz * inv;
    float Q00 = fmaf(-2.0f, fmaf(qy, qy, qz * qz), 1.0f);
    float Q01 = 2.0f * fmaf(qx, qy, -(qw * qz));
    float Q02 = 2.0f * fmaf(qx, qz, qw * qy);
    float Q10 = 2.0f * fmaf(qx, qy, qw * qz);
    float Q11 = fmaf(-2.0f, fmaf(qx, qx, qz * qz), 1.0f);
    float Q12 = 2.0f * fmaf(qy, qz, -(qw * qx));
    float Q20 = 2.0f * fmaf(qx, qz, -(qw * qy));
    float Q21 = 2.0f * fmaf(qy, qz, qw * qx);
    float Q22 = fmaf(-2.0f, fmaf(qx, qx, qy * qy), 1.0f);
    /* 5. M = Q diag(s) */
    float M00 = Q00 * s[0], M01 = Q01 * s[1], M02 = Q02 * s[2];
    float M10 = Q10 * s[0], M11 = Q11 * s[1], M12 = Q12 * s[2];
    float M20 = Q20 * s[0], M21 = Q21 * s[1], M22 = Q22 * s[2];
    /* 6. J (2x3), G = J R_view (2x3), Tm = G M (2x3) */
    float J00 = fx * rz, J02 = -(fx * txz) * rz;
    float J11 = fy * rz, J12 = -(fy * tyz) * rz;
    float G00 = fmaf(J02, V[8], J00 * V[0]), G01 = fmaf(J02, V[9], J00 * V[1]), G02 = fmaf(J02, V[10], J00 * V[2]);
    float G10 = fmaf(J12, V[8], J11 * V[4]), G11 = fmaf(J12, V[9], J11 * V[5]), G12 = fmaf(J12, V[10], J11 * V[6]);
    float T00 = fmaf(G02, M20, fmaf(G01, M10, G00 * M00));
    float T01 = fmaf(G02, M21, fmaf(G01, M11, G00 * M01));
    float T02 = fmaf(G02, M22, fmaf(G01, M12, G00 * M02));
    float T10 = fmaf(G12, M20, fmaf(G11, M10, G10 * M00));
    float T11 = fmaf(G12, M21, fmaf(G11, M11, G10 * M01));
    float T12 = fmaf(G12, M22, fmaf(G11, M12, G10 * M02));
    /* 7. 2D covariance Tm Tm^T + 0.3 I (reading Q4) */
    float a = fmaf(T02, T02, fmaf(T01, T01, T00 * T00)) + 0.3f;
    float b = fmaf(T02, T12, fmaf(T01, T11, T00 * T10));
    float c = fmaf(T12, T12, fmaf(T11, T11, T10 * T10)) + 0.3f;
    /* 8. conic */
    float det = fmaf(a, c, -(b * b));
    if (!(det > 0.0f) || !(det <= FLT_MAX)) return 3;
    float rd = 1.0f / det;
    float A = c * rd, B2 = -((b + b) * rd), C = a * rd;
    if (!(A <= FLT_MAX) || !(C <= FLT_MAX) || !(fabsf(B2) <= FLT_MAX)) return 3;
    /* 9. opacity threshold: alpha >= 1/255  <=>  q <= tau = 2 ln(255 o) */
    float x255 = 255.0f * o;
    if (!(x255 > 1.0f) || !(x255 <= FLT_MAX)) return 4;
    float tau = 2.0f * orc_ln_spec(x255);
    if (!(tau > 0.0f)) return 4;
    /* The bounding box and the macro-tile row scan must be CONSERVATIVE with respect to the pixel
     * test q <= tau ("conservative per-row ellipse-contour scan"; DESIGN.md reading
     * Q8).  q is evaluated in fp32 from the conic (A, B2, C), whose cross term cancels for elongated
     * gaussians (the hazard PAPER.md:180-226 describes): the region the pixel test accepts differs
     * from the ellipse of the covariance (a, b, c) by a relative ~3 * 2^-24 * cond in tau, with
     * cond = a c / det (measured over needles up to cond = 1e7).  The box and the scan therefore use
     * tau_s = tau * (1 + 2^-20 cond), five times that; for ordinary gaussians (cond < 100) the
     * margin is below 1e-4 of tau. */
    float cond = (a * c) * rd;
    float tau_s = tau * fmaf(cond, 9.5367431640625e-07f, 1.0f);
    float hx = sqrtf(tau_s * a), hy = sqrtf(tau_s * c);
    /* 10. off-screen cull on the threshold ellipse's bounding box */
    float fW = (float)W, fH = (float)H;
    if (!(mux + hx > 0.0f) || !(mux - hx < fW) || !(muy + hy > 0.0f) || !(muy - hy < fH)) return 5;
    /* 11. depth key */
    *key = f2u(zc);
    geo[G_MUX] = mux; geo[G_MUY] = muy; geo[G_A] = a; geo[G_B] = b; geo[G_C] = c;
    geo[G_TAU] = tau; geo[G_HX] = hx; geo[G_HY] = hy; geo[G_TAUS] = tau_s;
    conic[0] = A; conic[1] = B2; conic[2] = C;
    return 0;
}

int64_t orc_project(int64_t N, const float* means, const float* scales, const float* quats,
                    const float* opac, const float* sh, int degree, const float* cam, int W, int H,
                    uint8_t* valid, uint8_t* reason, uint32_t* key, float* geo, float* conic, double* rgb)
{
    int K = (degree + 1) * (degree + 1);
    int64_t nvis = 0;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t k = 0;
        float g[G_STRIDE] = {0}, cn[3] = {0};
        int r = project_one(means + 3 * i, scales + 3 * i, quats + 4 * i, opac[i], cam, W, H, &k, g, cn);
        valid[i] = (r == 0);
        if (reason) reason[i] = (uint8_t)r;
        key[i] = r == 0 ? k : 0;
        memcpy(geo + G_STRIDE * i, g, sizeof g);
        memcpy(conic + 3 * i, cn, sizeof cn);
        if (r == 0) {
            sh_colour(means + 3 * i, cam + 17, sh + (int64_t)K * 3 * i, degree, rgb + 3 * i);
            ++nvis;
        } else {
            rgb[3 * i] = rgb[3 * i + 1] = rgb[3 * i + 2] = 0.0;
        }
    }
    return nvis;
}

/* The same projection as the plain fp64 definition (EWA: Sigma2D = J W Sigma3D W^T J^T + 0.3 I,
 * Sigma3D = R S S^T R^T), no culls.  out[9] = mux, muy, a, b, c, A, B2, C, tau; zc separately.
 * Used only to pin the fp32 sequence above. */
void orc_project_f64(const float* m, const float* s, const float* qt, float o, const float* cam,
                     int W, int H, double out[9], double* zc_out)
{
    double V[12]; for (int i = 0; i < 12; ++i) V[i] = cam[i];
    double fx = cam[12], fy = cam[13], cx = cam[14], cy = cam[15];
    double p[3] = { m[0], m[1], m[2] };
    double xc = V[0] * p[0] + V[1] * p[1] + V[2] * p[2] + V[3];
    double yc = V[4] * p[0] + V[5] * p[1] + V[6] * p[2] + V[7];
    double zc = V[8] * p[0] + V[9] * p[1] + V[10] * p[2] + V[11];
    double xz = xc / zc, yz = yc / zc;
    double limx = 0.65 * W / fx, limy = 0.65 * H / fy;
    double txz = fmin(limx, fmax(-limx, xz)), tyz = fmin(limy, fmax(-limy, yz));
    double qw = qt[0], qx = qt[1], qy = qt[2], qz = qt[3];
    double qn = sqrt(qw * qw + qx * qx + qy * qy + qz * qz);
    qw /= qn; qx /= qn; qy /= qn; qz /= qn;
    double Q[3][3] = {
        { 1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy) },
        { 2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx) },
        { 2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy) } };
    double S3[3][3];   /* Sigma3D = Q diag(s^2) Q^T */
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
        double acc = 0; for (int k = 0; k < 3; ++k) acc += Q[i][k] * (double)s[k] * (double)s[k] * Q[j][k];
        S3[i][j] = acc;
    }
    double J[2][3] = { { fx / zc, 0, -fx * txz / zc }, { 0, fy / zc, -fy * tyz / zc } };
    double G[2][3];    /* J * R_view */
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 3; ++j)
        G[i][j] = J[i][0] * V[0 * 4 + j] + J[i][1] * V[1 * 4 + j] + J[i][2] * V[2 * 4 + j];
    double GS[2][3];
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 3; ++j) {
        double acc = 0; for (int k = 0; k < 3; ++k) acc += G[i][k] * S3[k][j];
        GS[i][j] = acc;
    }
    double a = 0, b = 0, c = 0;
    for (int k = 0; k < 3; ++k) { a += GS[0][k] * G[0][k]; b += GS[0][k] * G[1][k]; c += GS[1][k] * G[1][k]; }
    a += 0.3; c += 0.3;
    double det = a * c - b * b;
    out[0] = fx * xz + cx; out[1] = fy * yz + cy;
    out[2] = a; out[3] = b; out[4] = c;
    out[5] = c / det; out[6] = -2.0 * b / det; out[7] = a / det;
    out[8] = 2.0 * log(255.0 * (double)o);
    *zc_out = zc;
}

/* ---------------------------------------------------------------------------------------
 * N-SCAN: gaussian -> grid-cell row scan ("conservative per-row ellipse-contour
 * scan").  Exact x-extent of the ellipse {q <= tau} inside each row
 * band, rows and columns clipped to the image.  Cell sizes are powers of two.  Emits cell
 * ids r*ncx + m in increasing (r, m).  Returns the number emitted (writes at most `cap`).
 * ------------------------------------------------------------------------------------- */
static inline float clampf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

int orc_scan(const float* g, int W, int H, int cw, int ch, int32_t* out, int cap)
{
    const int ncx = (W + cw - 1) / cw, ncy = (H + ch - 1) / ch;
    const float mux = g[G_MUX], muy = g[G_MUY], a = g[G_A], b = g[G_B], c = g[G_C];
    const float tau = g[G_TAUS], hx = g[G_HX], hy = g[G_HY];   /* the scan runs on tau_s (project_one step 9) */
    const float fcw = (float)cw, fch = (float)ch, fW = (float)W, fH = (float)H;
    const float ytop_e = muy - hy, ybot_e = muy + hy;
    int r0 = (int)clampf(floorf(ytop_e / fch), 0.0f, (float)(ncy - 1));
    int r1 = (int)clampf(floorf(ybot_e / fch), 0.0f, (float)(ncy - 1));
    const float boc = b / c, rc = 1.0f / c;
    const float sdet = fmaxf(0.0f, fmaf(-b, boc, a));      /* a - b^2/c = det/c */
    const float yR = b * sqrtf(tau / a);                   /* dy of the rightmost point */
    const float nyR = -yR;
    int n = 0;
    for (int r = r0; r <= r1; ++r) {
        float y0 = (float)r * fch;
        float y1 = fminf((float)(r + 1) * fch, fH);
        float ylo = fmaxf(y0, ytop_e) - muy;
        float yhi = fminf(y1, ybot_e) - muy;
        if (!(yhi >= ylo)) continue;
        float rlo = sqrtf(fmaxf(0.0f, sdet * fmaf(-(ylo * ylo), rc, tau)));
        float rhi = sqrtf(fmaxf(0.0f, sdet * fmaf(-(yhi * yhi), rc, tau)));
        float xmax = (ylo <= yR && yR <= yhi) ? hx : fmaxf(fmaf(boc, ylo, rlo), fmaf(boc, yhi, rhi));
        float xmin = (ylo <= nyR && nyR <= yhi) ? -hx : fminf(fmaf(boc, ylo, -rlo), fmaf(boc, yhi, -rhi));
        xmin = xmin + mux; xmax = xmax + mux;
        if (!(xmax > 0.0f) || !(xmin < fW)) continue;
        int m0 = (int)clampf(floorf(xmin / fcw), 0.0f, (float)(ncx - 1));
        int m1 = (int)clampf(floorf(xmax / fcw), 0.0f, (float)(ncx - 1));
        for (int m = m0; m <= m1; ++m) { if (n < cap) out[n] = r * ncx + m; ++n; }
    }
    return n;
}

/* ---------------------------------------------------------------------------------------
 * O-LIST: per-macro-tile counts, offsets, (key,id)-sorted pair lists, batch boundaries.
 * mt_count[N_M], mt_offset[N_M+1], batch_offset[N_M+1]; keys/ids have capacity `cap` pairs
 * (pass NULL for keys/ids to only count).  Returns N_pairs.
 * ------------------------------------------------------------------------------------- */
static int cmp_u64(const void* pa, const void* pb)
{
    uint64_t a = *(const uint64_t*)pa, b = *(const uint64_t*)pb;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* Macro-tile of MT_W x MT_H pixels: the paper's is 8 x 4 render tiles of 8 x 8 px = 64 x 32; 128 x 64 in the
 * 16 x 16-tile variant (Table 2); other groupings of 32 render tiles (4 x 8, 16 x 2) for the macro-tile
 * shape sweep.  The lists depend on the macro-tile's extent in pixels only, not on how it is cut into render tiles. */
int64_t orc_bin_grid(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                     int W, int H, int B_r, int MT_W, int MT_H,
                     uint32_t* mt_count, uint32_t* mt_offset, uint32_t* batch_offset,
                     uint32_t* keys, uint32_t* ids, int64_t cap)
{
    const int nmx = (W + MT_W - 1) / MT_W, nmy = (H + MT_H - 1) / MT_H, NM = nmx * nmy;
    int32_t* cells = (int32_t*)malloc(sizeof(int32_t) * (size_t)NM);
    memset(mt_count, 0, sizeof(uint32_t) * (size_t)NM);
    /* (2)-(3): count */
    for (int64_t i = 0; i < N; ++i) {
        if (!valid[i]) continue;
        int n = orc_scan(geo + G_STRIDE * i, W, H, MT_W, MT_H, cells, NM);
        for (int k = 0; k < n; ++k) mt_count[cells[k]]++;
    }
    mt_offset[0] = 0;
    for (int m = 0; m < NM; ++m) mt_offset[m + 1] = mt_offset[m] + mt_count[m];
    int64_t npairs = mt_offset[NM];
    /* (5): batches */
    batch_offset[0] = 0;
    for (int m = 0; m < NM; ++m) batch_offset[m + 1] = batch_offset[m] + (mt_count[m] + (uint32_t)B_r - 1) / (uint32_t)B_r;
    if (keys && ids && npairs <= cap) {
        /* fill in id order, then (4): sort each segment ascending by (key, id) */
        uint64_t* pairs = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)(npairs > 0 ? npairs : 1));
        uint32_t* cursor = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)NM);
        memcpy(cursor, mt_offset, sizeof(uint32_t) * (size_t)NM);
        for (int64_t i = 0; i < N; ++i) {
            if (!valid[i]) continue;
            int n = orc_scan(geo + G_STRIDE * i, W, H, MT_W, MT_H, cells, NM);
            for (int k = 0; k < n; ++k) pairs[cursor[cells[k]]++] = ((uint64_t)key[i] << 32) | (uint64_t)(uint32_t)i;
        }
        for (int m = 0; m < NM; ++m)
            qsort(pairs + mt_offset[m], mt_count[m], sizeof(uint64_t), cmp_u64);
        for (int64_t p = 0; p < npairs; ++p) { keys[p] = (uint32_t)(pairs[p] >> 32); ids[p] = (uint32_t)pairs[p]; }
        free(pairs); free(cursor);
    }
    free(cells);
    return npairs;
}

/* tile = render-tile edge in px (8 or 16), macro-tile = 8 x 4 render tiles */
int64_t orc_bin_tile(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                     int W, int H, int B_r, int tile,
                     uint32_t* mt_count, uint32_t* mt_offset, uint32_t* batch_offset,
                     uint32_t* keys, uint32_t* ids, int64_t cap)
{
    return orc_bin_grid(N, valid, key, geo, W, H, B_r, 8 * tile, 4 * tile, mt_count, mt_offset, batch_offset, keys, ids, cap);
}

int64_t orc_bin(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                int W, int H, int B_r,
                uint32_t* mt_count, uint32_t* mt_offset, uint32_t* batch_offset,
                uint32_t* keys, uint32_t* ids, int64_t cap)
{
    return orc_bin_tile(N, valid, key, geo, W, H, B_r, 8, mt_count, mt_offset, batch_offset, keys, ids, cap);
}

/* ---------------------------------------------------------------------------------------
 * N-Q: the per-pixel quadratic whose comparison with tau decides the 1/255 skip, fp32 pinned
 * (DESIGN.md section 3).  px, py are pixel centres (i + 0.5).
 * ------------------------------------------------------------------------------------- */
float orc_pixel_q(float px, float py, float mux, float muy, float A, float B2, float C)
{
    float dx = px - mux, dy = py - muy;
    float u = A * dx;
    float a0 = u * dx;
    float b0 = B2 * dx;
    float t = fmaf(C, dy, b0);
    return fmaf(t, dy, a0);
}

/* alpha of gaussian g at pixel (i,j), or a negative value if it is skipped.  O-IMG: "q = N-Q(p, g); if
 * q > tau skip; alpha = min(0.99, o exp(-q/2))" - ONE q, the pinned fp32 one, decides the skip and gives alpha; exp and
 * the product are fp64.  (For an elongated gaussian the conic form cancels, and a second, fp64
 * evaluation of q would differ from the pinned one by ~2^-24 a c/det relative: two renderers that agree on every skip
 * decision would then disagree on alpha by that much.) */
static inline double pixel_alpha(int i, int j, const float* geo, const float* conic, float o)
{
    float px = (float)i + 0.5f, py = (float)j + 0.5f;
    float q32 = orc_pixel_q(px, py, geo[G_MUX], geo[G_MUY], conic[0], conic[1], conic[2]);
    if (!(q32 <= geo[G_TAU])) return -1.0;          /* alpha < 1/255: skipped */
    double alpha = (double)o * exp(-0.5 * (double)q32);
    return alpha < ORC_ALPHA_MAX ? alpha : ORC_ALPHA_MAX;   /* min(0.99, alpha) */
}

/* global front-to-back order: valid gaussians ascending by (key, id).  Returns count. */
static int64_t global_order(int64_t N, const uint8_t* valid, const uint32_t* key, uint32_t** order_out)
{
    int64_t nv = 0;
    for (int64_t i = 0; i < N; ++i) nv += valid[i] ? 1 : 0;
    uint64_t* pairs = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)(nv > 0 ? nv : 1));
    int64_t k = 0;
    for (int64_t i = 0; i < N; ++i) if (valid[i]) pairs[k++] = ((uint64_t)key[i] << 32) | (uint64_t)(uint32_t)i;
    qsort(pairs, (size_t)nv, sizeof(uint64_t), cmp_u64);
    uint32_t* order = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(nv > 0 ? nv : 1));
    for (int64_t p = 0; p < nv; ++p) order[p] = (uint32_t)pairs[p];
    free(pairs);
    *order_out = order;
    return nv;
}

typedef struct {
    int64_t nv; const uint32_t* order;
    const float* geo; const float* conic; const float* opac; const double* rgb;
    int x0, y0, x1, y1;       /* window [x0,x1) x [y0,y1) in pixels */
    int ya, yb;               /* this thread's rows */
    int terminate, use_bbox;
    double* out; double* outT; int64_t* ncomp;
} render_job;

/* O-IMG, gaussian-major: walk the gaussians in global order, visit the pixels of the
 * threshold-ellipse bounding box (+1 px), composite with per-pixel (C, T, done). */
static void* render_rows(void* arg)
{
    render_job* jb = (render_job*)arg;
    const int ww = jb->x1 - jb->x0;
    const int rows = jb->yb - jb->ya;
    if (rows <= 0 || ww <= 0) return NULL;
    uint8_t* done = (uint8_t*)calloc((size_t)rows * (size_t)ww, 1);
    int64_t ncomp = 0;
    for (int64_t p = 0; p < jb->nv; ++p) {
        const uint32_t g = jb->order[p];
        const float* geo = jb->geo + G_STRIDE * (int64_t)g;
        const float* cn = jb->conic + 3 * (int64_t)g;
        int ix0 = jb->x0, ix1 = jb->x1 - 1, iy0 = jb->ya, iy1 = jb->yb - 1;
        if (jb->use_bbox) {
            double bx0 = floor((double)geo[G_MUX] - (double)geo[G_HX] - 0.5) - 1.0;
            double bx1 = floor((double)geo[G_MUX] + (double)geo[G_HX] - 0.5) + 1.0;
            double by0 = floor((double)geo[G_MUY] - (double)geo[G_HY] - 0.5) - 1.0;
            double by1 = floor((double)geo[G_MUY] + (double)geo[G_HY] - 0.5) + 1.0;
            if (bx0 > ix0) ix0 = bx0 > 2e9 ? 2000000000 : (int)bx0;
            if (bx1 < ix1) ix1 = bx1 < -2e9 ? -2000000000 : (int)bx1;
            if (by0 > iy0) iy0 = by0 > 2e9 ? 2000000000 : (int)by0;
            if (by1 < iy1) iy1 = by1 < -2e9 ? -2000000000 : (int)by1;
        }
        const float o = jb->opac[g];
        const double* col = jb->rgb + 3 * (int64_t)g;
        for (int j = iy0; j <= iy1; ++j) {
            for (int i = ix0; i <= ix1; ++i) {
                const size_t loc = (size_t)(j - jb->ya) * (size_t)ww + (size_t)(i - jb->x0);
                if (done[loc]) continue;
                double alpha = pixel_alpha(i, j, geo, cn, o);
                if (alpha < 0.0) continue;
                const size_t pix = (size_t)(j - jb->y0) * (size_t)ww + (size_t)(i - jb->x0);
                double T = jb->outT[pix];
                double w = T * alpha;
                jb->out[3 * pix + 0] += w * col[0];
                jb->out[3 * pix + 1] += w * col[1];
                jb->out[3 * pix + 2] += w * col[2];
                T = T * (1.0 - alpha);
                jb->outT[pix] = T;
                ++ncomp;
                if (jb->terminate && T < ORC_EPS_T) done[loc] = 1;
            }
        }
    }
    free(done);
    if (jb->ncomp) *jb->ncomp = ncomp;
    return NULL;
}

static int64_t render_common(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                             const float* conic, const float* opac, const double* rgb,
                             int x0, int y0, int x1, int y1, int terminate, int use_bbox, int nthreads,
                             double* out, double* outT)
{
    const int ww = x1 - x0, hh = y1 - y0;
    if (ww <= 0 || hh <= 0) return 0;
    uint32_t* order = NULL;
    int64_t nv = global_order(N, valid, key, &order);
    double* Tbuf = outT ? outT : (double*)malloc(sizeof(double) * (size_t)ww * (size_t)hh);
    for (size_t i = 0; i < (size_t)ww * (size_t)hh; ++i) { Tbuf[i] = 1.0; out[3 * i] = out[3 * i + 1] = out[3 * i + 2] = 0.0; }
    if (nthreads < 1) nthreads = 1;
    if (nthreads > hh) nthreads = hh;
    render_job* jobs = (render_job*)calloc((size_t)nthreads, sizeof(render_job));
    pthread_t* th = (pthread_t*)calloc((size_t)nthreads, sizeof(pthread_t));
    int64_t* counts = (int64_t*)calloc((size_t)nthreads, sizeof(int64_t));
    for (int t = 0; t < nthreads; ++t) {
        render_job* jb = &jobs[t];
        jb->nv = nv; jb->order = order; jb->geo = geo; jb->conic = conic; jb->opac = opac; jb->rgb = rgb;
        jb->x0 = x0; jb->y0 = y0; jb->x1 = x1; jb->y1 = y1;
        jb->ya = y0 + (int)((int64_t)hh * t / nthreads);
        jb->yb = y0 + (int)((int64_t)hh * (t + 1) / nthreads);
        jb->terminate = terminate; jb->use_bbox = use_bbox;
        jb->out = out; jb->outT = Tbuf; jb->ncomp = &counts[t];
        if (nthreads == 1) render_rows(jb); else pthread_create(&th[t], NULL, render_rows, jb);
    }
    int64_t total = 0;
    for (int t = 0; t < nthreads; ++t) { if (nthreads > 1) pthread_join(th[t], NULL); total += counts[t]; }
    free(jobs); free(th); free(counts); free(order);
    if (!outT) free(Tbuf);
    return total;
}

/* O-IMG over the window [x0,x1) x [y0,y1).  out: hh*ww*3 fp64, outT (may be NULL): hh*ww final
 * transmittance.  terminate=1 applies the T < 1e-4 stop.  Returns the number of composites. */
int64_t orc_render(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                   const float* conic, const float* opac, const double* rgb,
                   int x0, int y0, int x1, int y1, int terminate, int nthreads, double* out, double* outT)
{
    return render_common(N, valid, key, geo, conic, opac, rgb, x0, y0, x1, y1, terminate, 1, nthreads, out, outT);
}

/* The same with no bounding box: every pixel of the window tests every valid gaussian. */
int64_t orc_brute(int64_t N, const uint8_t* valid, const uint32_t* key, const float* geo,
                  const float* conic, const float* opac, const double* rgb,
                  int x0, int y0, int x1, int y1, int terminate, int nthreads, double* out, double* outT)
{
    return render_common(N, valid, key, geo, conic, opac, rgb, x0, y0, x1, y1, terminate, 0, nthreads, out, outT);
}

/* ---------------------------------------------------------------------------------------
 * The method itself, step by step: for every macro-tile, its
 * (key,id)-sorted list is split into consecutive batches of B_r; every batch composites its
 * own gaussians from (C,T) = (0,1); partials are merged front to back with Eq. (1)
 *     C = C_0 + T_0 C_1 + T_0 T_1 C_2 + ...
 * terminate=1 stops a pixel once the running product of transmittances drops below 1e-4.
 * Full image only; pixel-major, slow: small scenes only.  out: H*W*3 fp64.
 * ------------------------------------------------------------------------------------- */
void orc_render_batched_grid(const uint32_t* mt_offset, const uint32_t* ids, const float* geo,
                             const float* conic, const float* opac, const double* rgb,
                             int W, int H, int B_r, int MT_W, int MT_H, int terminate, double* out)
{
    const int nmx = (W + MT_W - 1) / MT_W, nmy = (H + MT_H - 1) / MT_H;
    for (int my = 0; my < nmy; ++my) for (int mx = 0; mx < nmx; ++mx) {
        const int m = my * nmx + mx;
        const uint32_t s = mt_offset[m], e = mt_offset[m + 1];
        for (int j = my * MT_H; j < (my + 1) * MT_H && j < H; ++j)
        for (int i = mx * MT_W; i < (mx + 1) * MT_W && i < W; ++i) {
            double C[3] = { 0, 0, 0 }, Tacc = 1.0;
            int stop = 0;
            for (uint32_t bs = s; bs < e && !stop; bs += (uint32_t)B_r) {
                uint32_t be = bs + (uint32_t)B_r < e ? bs + (uint32_t)B_r : e;
                double Cj[3] = { 0, 0, 0 }, Tj = 1.0;       /* batch partial, starts at (0,1) */
                for (uint32_t p = bs; p < be; ++p) {
                    const uint32_t g = ids[p];
                    double alpha = pixel_alpha(i, j, geo + G_STRIDE * (int64_t)g, conic + 3 * (int64_t)g, opac[g]);
                    if (alpha < 0.0) continue;
                    double w = Tj * alpha;
                    Cj[0] += w * rgb[3 * (int64_t)g]; Cj[1] += w * rgb[3 * (int64_t)g + 1]; Cj[2] += w * rgb[3 * (int64_t)g + 2];
                    Tj *= (1.0 - alpha);
                    if (terminate && Tacc * Tj < ORC_EPS_T) { stop = 1; break; }
                }
                C[0] += Tacc * Cj[0]; C[1] += Tacc * Cj[1]; C[2] += Tacc * Cj[2];   /* Eq. (1) */
                Tacc *= Tj;
            }
            const size_t pix = (size_t)j * (size_t)W + (size_t)i;
            out[3 * pix] = C[0]; out[3 * pix + 1] = C[1]; out[3 * pix + 2] = C[2];
        }
    }
}

void orc_render_batched_tile(const uint32_t* mt_offset, const uint32_t* ids, const float* geo,
                             const float* conic, const float* opac, const double* rgb,
                             int W, int H, int B_r, int tile, int terminate, double* out)
{
    orc_render_batched_grid(mt_offset, ids, geo, conic, opac, rgb, W, H, B_r, 8 * tile, 4 * tile, terminate, out);
}

void orc_render_batched(const uint32_t* mt_offset, const uint32_t* ids, const float* geo,
                        const float* conic, const float* opac, const double* rgb,
                        int W, int H, int B_r, int terminate, double* out)
{
    orc_render_batched_tile(mt_offset, ids, geo, conic, opac, rgb, W, H, B_r, 8, terminate, out);
}

/* ---------------------------------------------------------------------------------------
 * Cholesky form of the inverse covariance (section 3.5):
 *     Sigma^-1 = L L^T,  L = [[l0, 0], [l1, l2]],   q = (l0 dx + l1 dy)^2 + (l2 dy)^2.
 * From the covariance (a, b, c), det = a c - b^2:  l0 = sqrt(c / det), l1 = -b / (det l0),
 * l2 = 1 / sqrt(c)  (so that l0^2 = A, l0 l1 = B2 / 2, l1^2 + l2^2 = C).  fp64.
 * Used by the tests of the fp16 data path (SURVEY.md 8(c) "Cholesky identity"); O-IMG does not use it.
 * ------------------------------------------------------------------------------------- */
void orc_cholesky(double a, double b, double c, double* l)
{
    const double det = a * c - b * b;
    l[0] = sqrt(c / det);
    l[1] = -b / (det * l[0]);
    l[2] = 1.0 / sqrt(c);
}

double orc_q_cholesky(double dx, double dy, const double* l)
{
    const double t1 = l[0] * dx + l[1] * dy, t2 = l[2] * dy;
    return t1 * t1 + t2 * t2;
}


/* ---------------------------------------------------------------------------------------
 * 32-byte SH codec (section 4.2): "YCoCg-R color-space conversion to decorrelate channels,
 * square-root gamma quantization (6 bits luma, 4 bits chroma), and per-basis percentile scaling ... 192 bytes
 * (fp32) to 32 bytes".  The paper gives no bit layout; this is the reading of DESIGN.md section 2 (Q20):
 *   per basis k = 0..15 the coefficient triple (r, g, b) goes to (Y, Co, Cg) by the lifting steps of YCoCg-R
 *       Co = r - b;  t = b + Co/2;  Cg = g - t;  Y = t + Cg/2        (inverse: t = Y - Cg/2; g = Cg + t; b = t - Co/2; r = b + Co)
 *   each value v is scaled by s = the per-(basis, channel) percentile of |v| over the scene (p = 0.999; p = 1 for the DC
 *   basis), clamped to [-1, 1] and quantised on a square-root curve:  code = bias + sign(u) * rint(sqrt(|u|) * L),
 *   u = v / s, with (L, bias) = (31, 32) for 6-bit luma and (7, 8) for 4-bit chroma; decode: w = (code - bias) / L,
 *   v = s * w * |w|.  16 x (6 + 4 + 4) = 224 bits; the remaining 32 bits extend the DC basis, which carries the
 *   base colour, to 16-bit luma (L = 32767) and 15-bit chroma (L = 16383): the 6 / 4-bit fields of k = 0 are the
 *   top bits of those codes.
 *   Layout: bytes 0-11 luma, 6 bits per basis, little-endian bit stream; byte 12 + k = Cg_k << 4 | Co_k;
 *   bytes 28-31 (little-endian word) = DC Y low 10 bits | DC Co low 11 bits << 10 | DC Cg low 11 bits << 21.
 * The encoder's arithmetic is fp32, one rounding per written op (the CUDA encoder produces the same bytes); decoding is fp64.
 * ------------------------------------------------------------------------------------- */
static inline void ycocg_fwd(float r, float g, float b, float* y, float* co, float* cg)
{
    float Co = r - b;
    float t = b + 0.5f * Co;
    float Cg = g - t;
    *y = t + 0.5f * Cg; *co = Co; *cg = Cg;
}

static int cmp_f32(const void* pa, const void* pb)
{
    float a = *(const float*)pa, b = *(const float*)pb;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* scales[k*3 + c], c = 0 Y, 1 Co, 2 Cg: |v| at sorted index min(N-1, floor(p N)), p = 1 for k = 0 else 0.999; 1 if that is 0 */
void orc_sh32_scales(int64_t N, const float* sh, float* scales)
{
    float* col = (float*)malloc(sizeof(float) * (size_t)(N > 0 ? N : 1));
    for (int k = 0; k < 16; ++k) for (int c = 0; c < 3; ++c) {
        for (int64_t i = 0; i < N; ++i) {
            const float* q = sh + (i * 16 + k) * 3;
            float v[3];
            ycocg_fwd(q[0], q[1], q[2], &v[0], &v[1], &v[2]);
            col[i] = fabsf(v[c]);
        }
        qsort(col, (size_t)N, sizeof(float), cmp_f32);
        int64_t idx = k == 0 ? N - 1 : (int64_t)((double)N * 0.999);
        if (idx > N - 1) idx = N - 1;
        float sc = N > 0 ? col[idx] : 1.0f;
        scales[k * 3 + c] = (sc > 0.0f && sc <= FLT_MAX) ? sc : 1.0f;
    }
    free(col);
}

static inline uint32_t sh32_quant(float v, float s, int L)
{
    float u = v / s;
    float a = fminf(fabsf(u), 1.0f);
    float w = sqrtf(a);
    int c = (int)rintf(w * (float)L);
    return (uint32_t)((L + 1) + (u < 0.0f ? -c : c));
}

void orc_sh32_encode(int64_t N, const float* sh, const float* scales, uint8_t* out)
{
    for (int64_t i = 0; i < N; ++i) {
        uint8_t* o = out + 32 * i;
        memset(o, 0, 32);
        uint64_t luma_lo = 0; uint32_t luma_hi = 0;          /* 96-bit little-endian bit stream */
        for (int k = 0; k < 16; ++k) {
            const float* q = sh + (i * 16 + k) * 3;
            float y, co, cg;
            ycocg_fwd(q[0], q[1], q[2], &y, &co, &cg);
            uint32_t cy, cco, ccg;
            if (k == 0) {
                uint32_t y16 = sh32_quant(y, scales[0], 32767), co15 = sh32_quant(co, scales[1], 16383), cg15 = sh32_quant(cg, scales[2], 16383);
                uint32_t ext = (y16 & 0x3ffu) | ((co15 & 0x7ffu) << 10) | ((cg15 & 0x7ffu) << 21);
                o[28] = (uint8_t)ext; o[29] = (uint8_t)(ext >> 8); o[30] = (uint8_t)(ext >> 16); o[31] = (uint8_t)(ext >> 24);
                cy = y16 >> 10; cco = co15 >> 11; ccg = cg15 >> 11;
            } else {
                cy = sh32_quant(y, scales[k * 3], 31); cco = sh32_quant(co, scales[k * 3 + 1], 7); ccg = sh32_quant(cg, scales[k * 3 + 2], 7);
            }
            int bit = 6 * k;
            if (bit < 64) { luma_lo |= (uint64_t)cy << bit; if (bit > 58) luma_hi |= cy >> (64 - bit); }
            else luma_hi |= cy << (bit - 64);
            o[12 + k] = (uint8_t)((ccg << 4) | cco);
        }
        for (int b = 0; b < 8; ++b) o[b] = (uint8_t)(luma_lo >> (8 * b));
        for (int b = 0; b < 4; ++b) o[8 + b] = (uint8_t)(luma_hi >> (8 * b));
    }
}

static inline double sh32_dequant(uint32_t code, double s, int L)
{
    double w = ((double)code - (double)(L + 1)) / (double)L;
    return s * w * fabs(w);
}

/* decoded coefficients, [N][16][3] fp32 (rounded once from the fp64 decode) */
void orc_sh32_decode(int64_t N, const uint8_t* in, const float* scales, float* sh)
{
    for (int64_t i = 0; i < N; ++i) {
        const uint8_t* o = in + 32 * i;
        uint64_t luma_lo = 0; uint32_t luma_hi = 0;
        for (int b = 0; b < 8; ++b) luma_lo |= (uint64_t)o[b] << (8 * b);
        for (int b = 0; b < 4; ++b) luma_hi |= (uint32_t)o[8 + b] << (8 * b);
        uint32_t ext = (uint32_t)o[28] | ((uint32_t)o[29] << 8) | ((uint32_t)o[30] << 16) | ((uint32_t)o[31] << 24);
        for (int k = 0; k < 16; ++k) {
            int bit = 6 * k;
            uint32_t cy = bit < 64 ? (uint32_t)(luma_lo >> bit) : (luma_hi >> (bit - 64));
            if (bit < 64 && bit > 58) cy |= luma_hi << (64 - bit);
            cy &= 63u;
            uint32_t cco = o[12 + k] & 15u, ccg = o[12 + k] >> 4;
            double y, co, cg;
            if (k == 0) {
                y = sh32_dequant((cy << 10) | (ext & 0x3ffu), scales[0], 32767);
                co = sh32_dequant((cco << 11) | ((ext >> 10) & 0x7ffu), scales[1], 16383);
                cg = sh32_dequant((ccg << 11) | (ext >> 21), scales[2], 16383);
            } else {
                y = sh32_dequant(cy, scales[k * 3], 31); co = sh32_dequant(cco, scales[k * 3 + 1], 7); cg = sh32_dequant(ccg, scales[k * 3 + 2], 7);
            }
            double t = y - 0.5 * cg, g = cg + t, b = t - 0.5 * co, r = b + co;
            float* q = sh + (i * 16 + k) * 3;
            q[0] = (float)r; q[1] = (float)g; q[2] = (float)b;
        }
    }
}

int orc_abi_version(void) { return 1; }
