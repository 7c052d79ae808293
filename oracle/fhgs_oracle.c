/*
 * fhgs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU statement of the FHGS hot path (arxiv 2505.19154):
 * EWA projection -> (tile|depth) instances, stable sort, tile ranges -> per-pixel front-to-back
 * compositing of RGB + D feature channels -> weight-aggregated feature fusion.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call
 * this.  It shares NO code, header, table or helper with the CUDA path under
 * paper_2505_19154_b200/csrc/.  Every function cites the passage it follows:
 *   PAPER.md:77-95   primitive, G(u)=exp(-(u^2+v^2)/2), c(x)=sum c_i w_i, w_i = alpha_i T_i,
 *                    alpha_i = op_i G_i, T_i = prod_{j<i}(1-alpha_j)
 *   PAPER.md:302     16x16 tiles, duplication, 64-bit key (tile | depth), radix sort, ranges
 *   PAPER.md:335     front-to-back traversal
 *   SURVEY.md 8(c)   the readings (C1-P, C1-S, C1-R, C1-F, C2) where the paper is silent
 *   DESIGN.md        "Readings of the paper" lists every such reading
 *
 * Parity pins: tests/test_oracle_pins.py (closed forms, invariants, brute force) -- no function in
 * this file is "parity unpinned".
 *
 * Arithmetic rules:
 *   - projection (C1-P): every operation is ONE IEEE binary32 operation in the written order,
 *     no FMA contraction (compile with -ffp-contract=off, no -ffast-math).
 *   - the per-(pixel,Gaussian) decision quantity q uses explicit fmaf (C1-R step 2).
 *   - everything after the decision (exp, alpha, w, sums) is in double.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC fhgs_oracle.c -o libfhgs_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TILE 16

/* params layout (12 floats): z_near, cov_dilation, jac_clamp, q_cutoff, alpha_max, t_min,
 * den_eps, bg[3], rect_mode (0 = scalar radius, 1 = tight per-axis extents; SURVEY 8(f) NEXT-4 i),
 * primitive (0 = 3-axis EWA Gaussian, 1 = 2-D surfel).
 * cam layout (35 floats): view[16], proj[16], cam_pos[3]. */
enum { P_ZNEAR = 0, P_DIL, P_JCLAMP, P_QCUT, P_AMAX, P_TMIN, P_DENEPS, P_BG0, P_BG1, P_BG2, P_RECT, P_PRIM };

int fo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static uint32_t f2u(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* Intrinsics of the pinhole camera from proj[]: computed in double, rounded once. */
static void intrinsics(const float *cam, int W, int H, float *fx, float *fy, float *cx, float *cy,
                       float *tanx, float *tany) {
    const float *proj = cam + 16;
    *fx = (float)((double)proj[0] * (double)W / 2.0);
    *fy = (float)((double)proj[5] * (double)H / 2.0);
    *cx = (float)(((double)proj[2] + 1.0) * (double)W / 2.0 - 0.5);
    *cy = (float)(((double)proj[6] + 1.0) * (double)H / 2.0 - 0.5);
    *tanx = (float)(1.0 / (double)proj[0]);
    *tany = (float)(1.0 / (double)proj[5]);
}

/* Real orthonormal spherical-harmonics basis up to degree 3 (C1-P step 10). d = unit direction. */
static const float SHC0 = 0.28209479177387814f;
static const float SHC1 = 0.4886025119029199f;
static const float SHC2[5] = {1.0925484305920792f, -1.0925484305920792f, 0.31539156525252005f,
                              -1.0925484305920792f, 0.5462742152960396f};
static const float SHC3[7] = {-0.5900435899266435f, 2.890611442640554f, -0.4570457994644658f,
                              0.3731763325901154f, -0.4570457994644658f, 1.445305721320277f,
                              -0.5900435899266435f};

void fo_sh_basis(int degree, float x, float y, float z, float *Y /*[(deg+1)^2]*/) {
    Y[0] = SHC0;
    if (degree < 1) return;
    Y[1] = -(SHC1 * y);
    Y[2] = SHC1 * z;
    Y[3] = -(SHC1 * x);
    if (degree < 2) return;
    float xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
    Y[4] = SHC2[0] * xy;
    Y[5] = SHC2[1] * yz;
    Y[6] = SHC2[2] * ((2.0f * zz - xx) - yy);
    Y[7] = SHC2[3] * xz;
    Y[8] = SHC2[4] * (xx - yy);
    if (degree < 3) return;
    Y[9] = (SHC3[0] * y) * (3.0f * xx - yy);
    Y[10] = (SHC3[1] * xy) * z;
    Y[11] = (SHC3[2] * y) * ((4.0f * zz - xx) - yy);
    Y[12] = (SHC3[3] * z) * ((2.0f * zz - 3.0f * xx) - 3.0f * yy);
    Y[13] = (SHC3[4] * x) * ((4.0f * zz - xx) - yy);
    Y[14] = (SHC3[5] * z) * (xx - yy);
    Y[15] = (SHC3[6] * x) * (xx - 3.0f * yy);
}

/* Quaternion (w,x,y,z), not necessarily unit -> rotation matrix R (row-major), C1-P step 4.
 * Columns of R are t_u, t_v, t_w of PAPER.md:77. */
void fo_quat_to_rot(const float *q, float *R) {
    float w = q[0], x = q[1], y = q[2], z = q[3];
    float n = sqrtf(((w * w + x * x) + y * y) + z * z);
    w = w / n; x = x / n; y = y / n; z = z / n;
    R[0] = 1.0f - 2.0f * (y * y + z * z);
    R[1] = 2.0f * (x * y - w * z);
    R[2] = 2.0f * (x * z + w * y);
    R[3] = 2.0f * (x * y + w * z);
    R[4] = 1.0f - 2.0f * (x * x + z * z);
    R[5] = 2.0f * (y * z - w * x);
    R[6] = 2.0f * (x * z - w * y);
    R[7] = 2.0f * (y * z + w * x);
    R[8] = 1.0f - 2.0f * (x * x + y * y);
}

static float clampf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

/* ------------------------------------------------------------------------------------------
 * Step P (C1-P): PAPER.md:302 CullGaussian, PAPER.md:309-310 2DScreenGaussians, EWA reading D1.
 * Outputs for a culled Gaussian: radius = 0, tiles_touched = 0, rect = 0, floats = 0.
 * ------------------------------------------------------------------------------------------ */
void fo_project(int n, int sh_degree, const float *mean, const float *scale, const float *quat,
                const float *opacity, const float *sh, const float *cam, int W, int H,
                const float *prm, float *xy, float *depth, float *conic_opacity, float *rgb,
                int32_t *radius, uint16_t *rect, uint32_t *tiles_touched) {
    float fx, fy, cx, cy, tanx, tany;
    intrinsics(cam, W, H, &fx, &fy, &cx, &cy, &tanx, &tany);
    const float *V = cam;
    const float *cp = cam + 32;
    const int GW = (W + TILE - 1) / TILE, GH = (H + TILE - 1) / TILE;
    const int K = (sh_degree + 1) * (sh_degree + 1);
    const float z_near = prm[P_ZNEAR], dil = prm[P_DIL];
    const float Lx = prm[P_JCLAMP] * tanx, Ly = prm[P_JCLAMP] * tany;
    const int tight = prm[P_RECT] != 0.0f;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        xy[2 * i] = xy[2 * i + 1] = 0.0f; depth[i] = 0.0f;
        for (int k = 0; k < 4; ++k) conic_opacity[4 * i + k] = 0.0f;
        for (int k = 0; k < 3; ++k) rgb[3 * i + k] = 0.0f;
        radius[i] = 0; tiles_touched[i] = 0;
        for (int k = 0; k < 4; ++k) rect[4 * i + k] = 0;

        const float p0 = mean[3 * i], p1 = mean[3 * i + 1], p2 = mean[3 * i + 2];
        /* 1. camera-space position */
        float t[3];
        for (int k = 0; k < 3; ++k)
            t[k] = ((V[4 * k] * p0 + V[4 * k + 1] * p1) + V[4 * k + 2] * p2) + V[4 * k + 3];
        const float z = t[2];
        if (!(z >= z_near)) continue;
        /* 2. pixel position (integer = pixel centre) */
        const float u = t[0] / z, v = t[1] / z;
        const float px = fx * u + cx, py = fy * v + cy;
        /* 3. clamp for the Jacobian only */
        const float uc = fminf(fmaxf(u, -Lx), Lx), vc = fminf(fmaxf(v, -Ly), Ly);
        const float X = uc * z, Y = vc * z;
        /* 4-5. Sigma3D = R S S^T R^T */
        float R[9];
        fo_quat_to_rot(quat + 4 * i, R);
        float M[9];
        for (int k = 0; k < 3; ++k)
            for (int j = 0; j < 3; ++j) M[3 * k + j] = R[3 * k + j] * scale[3 * i + j];
        float S[9];
        for (int a = 0; a < 3; ++a)
            for (int b = a; b < 3; ++b) {
                float s = (M[3 * a] * M[3 * b] + M[3 * a + 1] * M[3 * b + 1]) + M[3 * a + 2] * M[3 * b + 2];
                S[3 * a + b] = s; S[3 * b + a] = s;
            }
        /* 6. Jacobian of the perspective map times the view rotation */
        const float J00 = fx / z, J02 = -(fx * X) / (z * z), J11 = fy / z, J12 = -(fy * Y) / (z * z);
        float A[6];
        for (int j = 0; j < 3; ++j) {
            A[j] = J00 * V[j] + J02 * V[8 + j];
            A[3 + j] = J11 * V[4 + j] + J12 * V[8 + j];
        }
        /* 7. Sigma2D = A Sigma3D A^T + dil I */
        float U[6];
        for (int a = 0; a < 2; ++a)
            for (int j = 0; j < 3; ++j)
                U[3 * a + j] = (A[3 * a] * S[j] + A[3 * a + 1] * S[3 + j]) + A[3 * a + 2] * S[6 + j];
        const float ca = ((U[0] * A[0] + U[1] * A[1]) + U[2] * A[2]) + dil;
        const float cb = (U[0] * A[3] + U[1] * A[4]) + U[2] * A[5];
        const float cc = ((U[3] * A[3] + U[4] * A[4]) + U[5] * A[5]) + dil;
        const float det = ca * cc - cb * cb;
        if (!(det > 0.0f)) continue;
        const float inv = 1.0f / det;
        const float conA = cc * inv, conB = -(cb * inv), conC = ca * inv;
        /* 8. 3-sigma radius from the larger eigenvalue */
        const float mid = 0.5f * (ca + cc);
        const float disc = fmaxf(mid * mid - det, 0.0f);
        const float lam = mid + sqrtf(disc);
        const float r = ceilf(3.0f * sqrtf(lam));
        /* 9. tile rectangle */
        if (!(isfinite(px) && isfinite(py) && isfinite(r))) continue;
        /* rect_mode 1 (NEXT-4 i): q <= 9 means |dx| <= 3 sqrt(Sigma_xx), |dy| <= 3 sqrt(Sigma_yy) (the exact bounding
         * box of the ellipse d^T Sigma^-1 d <= 9), so the per-axis extents replace the scalar radius */
        const float rx = tight ? ceilf(3.0f * sqrtf(ca)) : r, ry = tight ? ceilf(3.0f * sqrtf(cc)) : r;
        const float x0 = clampf(floorf((px - rx) / 16.0f), 0.0f, (float)GW);
        const float x1 = clampf(floorf((px + rx) / 16.0f) + 1.0f, 0.0f, (float)GW);
        const float y0 = clampf(floorf((py - ry) / 16.0f), 0.0f, (float)GH);
        const float y1 = clampf(floorf((py + ry) / 16.0f) + 1.0f, 0.0f, (float)GH);
        const int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
        const int cnt = (ix1 - ix0) * (iy1 - iy0);
        if (cnt <= 0 || ix1 <= ix0 || iy1 <= iy0) continue;
        /* 10. SH colour */
        float dx = p0 - cp[0], dy = p1 - cp[1], dz = p2 - cp[2];
        const float dn = sqrtf((dx * dx + dy * dy) + dz * dz);
        dx = dx / dn; dy = dy / dn; dz = dz / dn;
        float Yb[16];
        fo_sh_basis(sh_degree, dx, dy, dz, Yb);
        for (int k = 0; k < 3; ++k) {
            float c = 0.5f;
            for (int l = 0; l < K; ++l) c = c + Yb[l] * sh[((size_t)i * K + l) * 3 + k];
            rgb[3 * i + k] = fmaxf(c, 0.0f);
        }
        xy[2 * i] = px; xy[2 * i + 1] = py; depth[i] = z;
        conic_opacity[4 * i] = conA; conic_opacity[4 * i + 1] = conB;
        conic_opacity[4 * i + 2] = conC; conic_opacity[4 * i + 3] = opacity[i];
        radius[i] = (int32_t)r;
        rect[4 * i] = (uint16_t)ix0; rect[4 * i + 1] = (uint16_t)iy0;
        rect[4 * i + 2] = (uint16_t)ix1; rect[4 * i + 3] = (uint16_t)iy1;
        tiles_touched[i] = (uint32_t)cnt;
    }
}

/* ------------------------------------------------------------------------------------------
 * Step P for the paper's own primitive (prm[P_PRIM] = 1): the 2-D surfel of
 * PAPER.md:77-90.  Centre p, tangents t_u, t_v = columns 0, 1 of R(quat), planar scales
 * (s_u, s_v) = scale[0..1] (scale[2] is ignored).  Eq. 2: P(u,v) = p + s_u t_u u + s_v t_v v.
 * Eq. 3: the pixel x = (x, y) sees the point (u,v) with  (x z, y z, z)^T = K W P(u,v), i.e. in
 * homogeneous pixel coordinates  (X, Y, Wc)^T = T (u, v, 1)^T  with the 3x3 matrix
 *     T = [ fx a_x + cx a_z   fx b_x + cx b_z   fx c_x + cx c_z ]     a = R_v (s_u t_u)
 *         [ fy a_y + cy a_z   fy b_y + cy b_z   fy c_y + cy c_z ]     b = R_v (s_v t_v)
 *         [       a_z               b_z               c_z       ]     c = camera-space centre
 * so (u, v, 1) is proportional to T^-1 (x, y, 1)^T = adj(T) (x, y, 1)^T / det T.  The 9 entries of
 * adj(T) (rows: the cross products T_y x T_w, T_w x T_x, T_x x T_y taken as COLUMNS), scaled by an
 * exact power of two, are the per-splat "ray transform" ray_transform[i][0..8] (3 rows padded to
 * float4: [i][4 r + c]); fo_q_surfel evaluates u^2 + v^2 from it.  G = exp(-(u^2+v^2)/2)
 * (PAPER.md:85).  Readings: depth of the key = z of the centre; a splat is culled when
 * its centre or any point of its 3-sigma disc lies in front of z_near (z_min = c_z -
 * 3 sqrt(a_z^2 + b_z^2)); no low-pass filter (the paper states none).
 * Screen bounds (conservative AABB of the pixels with u^2+v^2 <= q_cut): the
 * 3-sigma disc maps to the conic x~^T T^-T diag(1,1,-q) T^-1 x~ <= 0, whose bounding box follows
 * from the dual conic T diag(q,q,-1) T^T:  centre_x = (q T_x0 T_w0 + q T_x1 T_w1 - T_x2 T_w2)/d,
 * half_x^2 = centre_x^2 - (q T_x0^2 + q T_x1^2 - T_x2^2)/d,  d = q T_w0^2 + q T_w1^2 - T_w2^2 < 0;
 * one pixel of margin absorbs the binary32 rounding.  Outputs: xy = box centre, conic_opacity =
 * (half_x, half_y, 0, opacity), radius = max of the two integer half extents, rect from the box.
 * Same arithmetic rule as fo_project: single binary32 operations in the written order.
 * ------------------------------------------------------------------------------------------ */
static void cross3(const float *a, const float *b, float *o) {
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}

void fo_project_surfel(int n, int sh_degree, const float *mean, const float *scale, const float *quat,
                       const float *opacity, const float *sh, const float *cam, int W, int H,
                       const float *prm, float *xy, float *depth, float *conic_opacity, float *rgb,
                       int32_t *radius, uint16_t *rect, uint32_t *tiles_touched, float *ray_transform) {
    float fx, fy, cx, cy, tanx, tany;
    intrinsics(cam, W, H, &fx, &fy, &cx, &cy, &tanx, &tany);
    const float *V = cam;
    const float *cp = cam + 32;
    const int GW = (W + TILE - 1) / TILE, GH = (H + TILE - 1) / TILE;
    const int K = (sh_degree + 1) * (sh_degree + 1);
    const float z_near = prm[P_ZNEAR], qc = prm[P_QCUT];
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        xy[2 * i] = xy[2 * i + 1] = 0.0f; depth[i] = 0.0f;
        for (int k = 0; k < 4; ++k) conic_opacity[4 * i + k] = 0.0f;
        for (int k = 0; k < 3; ++k) rgb[3 * i + k] = 0.0f;
        radius[i] = 0; tiles_touched[i] = 0;
        for (int k = 0; k < 4; ++k) rect[4 * i + k] = 0;
        for (int k = 0; k < 12; ++k) ray_transform[12 * i + k] = 0.0f;

        const float p0 = mean[3 * i], p1 = mean[3 * i + 1], p2 = mean[3 * i + 2];
        /* 1. camera-space centre */
        float c[3];
        for (int k = 0; k < 3; ++k)
            c[k] = ((V[4 * k] * p0 + V[4 * k + 1] * p1) + V[4 * k + 2] * p2) + V[4 * k + 3];
        if (!(c[2] >= z_near)) continue;
        /* 2. scaled tangents in camera space: a = R_v (s_u t_u), b = R_v (s_v t_v) */
        float R[9];
        fo_quat_to_rot(quat + 4 * i, R);
        const float su = scale[3 * i], sv = scale[3 * i + 1];
        const float aw[3] = {R[0] * su, R[3] * su, R[6] * su}, bw[3] = {R[1] * sv, R[4] * sv, R[7] * sv};
        float a[3], b[3];
        for (int k = 0; k < 3; ++k) {
            a[k] = (V[4 * k] * aw[0] + V[4 * k + 1] * aw[1]) + V[4 * k + 2] * aw[2];
            b[k] = (V[4 * k] * bw[0] + V[4 * k + 1] * bw[1]) + V[4 * k + 2] * bw[2];
        }
        /* 3. the whole 3-sigma disc must lie behind the near plane */
        const float zmin = c[2] - 3.0f * sqrtf(a[2] * a[2] + b[2] * b[2]);
        if (!(zmin >= z_near)) continue;
        /* 4. T (rows x, y, w) */
        const float Tx[3] = {fx * a[0] + cx * a[2], fx * b[0] + cx * b[2], fx * c[0] + cx * c[2]};
        const float Ty[3] = {fy * a[1] + cy * a[2], fy * b[1] + cy * b[2], fy * c[1] + cy * c[2]};
        const float Tw[3] = {a[2], b[2], c[2]};
        /* 5. adj(T): columns A0 = Ty x Tw, A1 = Tw x Tx, A2 = Tx x Ty; scaled by 2^-e, e = exponent of max |entry| */
        float A0[3], A1[3], A2[3];
        cross3(Ty, Tw, A0); cross3(Tw, Tx, A1); cross3(Tx, Ty, A2);
        float mx = 0.0f;
        for (int k = 0; k < 3; ++k) mx = fmaxf(mx, fmaxf(fabsf(A0[k]), fmaxf(fabsf(A1[k]), fabsf(A2[k]))));
        if (!(mx > 0.0f) || !isfinite(mx)) continue;
        int e; (void)frexpf(mx, &e);
        const float sc = ldexpf(1.0f, -e);
        /* 6. bounding box of the q <= q_cut footprint from the dual conic */
        const float d = (qc * (Tw[0] * Tw[0]) + qc * (Tw[1] * Tw[1])) - Tw[2] * Tw[2];
        if (!(d < 0.0f)) continue;
        const float ccx = ((qc * (Tx[0] * Tw[0]) + qc * (Tx[1] * Tw[1])) - Tx[2] * Tw[2]) / d;
        const float ccy = ((qc * (Ty[0] * Tw[0]) + qc * (Ty[1] * Tw[1])) - Ty[2] * Tw[2]) / d;
        const float ex = ccx * ccx - ((qc * (Tx[0] * Tx[0]) + qc * (Tx[1] * Tx[1])) - Tx[2] * Tx[2]) / d;
        const float ey = ccy * ccy - ((qc * (Ty[0] * Ty[0]) + qc * (Ty[1] * Ty[1])) - Ty[2] * Ty[2]) / d;
        const float hx = sqrtf(fmaxf(ex, 1e-4f)) + 1.0f, hy = sqrtf(fmaxf(ey, 1e-4f)) + 1.0f;
        if (!(isfinite(ccx) && isfinite(ccy) && isfinite(hx) && isfinite(hy))) continue;
        const float rx = ceilf(hx), ry = ceilf(hy);
        const float x0 = clampf(floorf((ccx - rx) / 16.0f), 0.0f, (float)GW);
        const float x1 = clampf(floorf((ccx + rx) / 16.0f) + 1.0f, 0.0f, (float)GW);
        const float y0 = clampf(floorf((ccy - ry) / 16.0f), 0.0f, (float)GH);
        const float y1 = clampf(floorf((ccy + ry) / 16.0f) + 1.0f, 0.0f, (float)GH);
        const int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
        if (ix1 <= ix0 || iy1 <= iy0) continue;
        /* 7. SH colour (C1-P step 10) */
        float dx = p0 - cp[0], dy = p1 - cp[1], dz = p2 - cp[2];
        const float dn = sqrtf((dx * dx + dy * dy) + dz * dz);
        dx = dx / dn; dy = dy / dn; dz = dz / dn;
        float Yb[16];
        fo_sh_basis(sh_degree, dx, dy, dz, Yb);
        for (int k = 0; k < 3; ++k) {
            float col = 0.5f;
            for (int l = 0; l < K; ++l) col = col + Yb[l] * sh[((size_t)i * K + l) * 3 + k];
            rgb[3 * i + k] = fmaxf(col, 0.0f);
        }
        xy[2 * i] = ccx; xy[2 * i + 1] = ccy; depth[i] = c[2];
        conic_opacity[4 * i] = hx; conic_opacity[4 * i + 1] = hy; conic_opacity[4 * i + 3] = opacity[i];
        radius[i] = (int32_t)fmaxf(rx, ry);
        rect[4 * i] = (uint16_t)ix0; rect[4 * i + 1] = (uint16_t)iy0;
        rect[4 * i + 2] = (uint16_t)ix1; rect[4 * i + 3] = (uint16_t)iy1;
        tiles_touched[i] = (uint32_t)((ix1 - ix0) * (iy1 - iy0));
        float *rt = ray_transform + 12 * i;
        for (int r = 0; r < 3; ++r) { rt[4 * r] = A0[r] * sc; rt[4 * r + 1] = A1[r] * sc; rt[4 * r + 2] = A2[r] * sc; }
    }
}

/* The per-(pixel, surfel) decision quantities in binary32 (both sides evaluate exactly this):
 *   p = adj(T) (x, y, 1)^T,  num = p_x^2 + p_y^2,  den = p_z^2;  (u, v) = (p_x, p_y)/p_z.
 * The surfel contributes iff den > 0 and num <= q_cut * den  (u^2 + v^2 <= q_cut without a division). */
void fo_surfel_terms(const float *rt, int x, int y, float *p /*[3]*/, float *num, float *den) {
    const float fxp = (float)x, fyp = (float)y;
    p[0] = fmaf(fxp, rt[0], fmaf(fyp, rt[1], rt[2]));
    p[1] = fmaf(fxp, rt[4], fmaf(fyp, rt[5], rt[6]));
    p[2] = fmaf(fxp, rt[8], fmaf(fyp, rt[9], rt[10]));
    *num = fmaf(p[0], p[0], p[1] * p[1]);
    *den = p[2] * p[2];
}

/* ------------------------------------------------------------------------------------------
 * Step S (C1-S): PAPER.md:302 DuplicateWithKeys / SortByKeys / IdentifyTileRanges.
 * key = (tile_id << 32) | float_bits(z_cam); stable sort (ties keep ascending Gaussian index,
 * SPEC.md:186); ranges[t] = [first, last+1), (0,0) for an empty tile.
 * ------------------------------------------------------------------------------------------ */
uint64_t fo_count_instances(int n, const uint32_t *tiles_touched) {
    uint64_t m = 0;
    for (int i = 0; i < n; ++i) m += tiles_touched[i];
    return m;
}

typedef struct { uint64_t key; uint32_t val; } fo_pair;

static int cmp_pair(const void *a, const void *b) {
    const fo_pair *x = (const fo_pair *)a, *y = (const fo_pair *)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    /* instances are emitted in ascending Gaussian index, so (key, val) order == stable order */
    if (x->val != y->val) return x->val < y->val ? -1 : 1;
    return 0;
}

/* keys_unsorted/vals_unsorted may be NULL.  Returns M. */
uint64_t fo_bins(int n, const uint32_t *tiles_touched, const uint16_t *rect, const float *depth,
                 int W, int H, uint32_t *offsets, uint64_t *keys_unsorted, uint32_t *vals_unsorted,
                 uint64_t *keys_sorted, uint32_t *vals_sorted, uint32_t *ranges) {
    const int GW = (W + TILE - 1) / TILE, GH = (H + TILE - 1) / TILE;
    uint64_t m = 0;
    for (int i = 0; i < n; ++i) { m += tiles_touched[i]; offsets[i] = (uint32_t)m; }
    fo_pair *pairs = (fo_pair *)malloc((m ? m : 1) * sizeof(fo_pair));
    for (int i = 0; i < n; ++i) {
        if (!tiles_touched[i]) continue;
        uint64_t k = (uint64_t)offsets[i] - tiles_touched[i];
        for (int ty = rect[4 * i + 1]; ty < rect[4 * i + 3]; ++ty)
            for (int tx = rect[4 * i]; tx < rect[4 * i + 2]; ++tx) {
                pairs[k].key = ((uint64_t)((uint32_t)(ty * GW + tx)) << 32) | f2u(depth[i]);
                pairs[k].val = (uint32_t)i;
                ++k;
            }
    }
    if (keys_unsorted) for (uint64_t k = 0; k < m; ++k) keys_unsorted[k] = pairs[k].key;
    if (vals_unsorted) for (uint64_t k = 0; k < m; ++k) vals_unsorted[k] = pairs[k].val;
    qsort(pairs, m, sizeof(fo_pair), cmp_pair);
    for (uint64_t k = 0; k < m; ++k) { keys_sorted[k] = pairs[k].key; vals_sorted[k] = pairs[k].val; }
    memset(ranges, 0, (size_t)GW * GH * 2 * sizeof(uint32_t));
    for (uint64_t k = 0; k < m; ++k) {
        uint32_t t = (uint32_t)(pairs[k].key >> 32);
        if (k == 0 || (uint32_t)(pairs[k - 1].key >> 32) != t) ranges[2 * t] = (uint32_t)k;
        ranges[2 * t + 1] = (uint32_t)(k + 1);
    }
    free(pairs);
    return m;
}

/* Global visit order for the tile-free renderer: visible Gaussians (radius > 0) sorted by
 * (depth bits, index) (C1-R preamble).  Returns the count. */
typedef struct { uint32_t zbits; uint32_t idx; } fo_zi;
static int cmp_zi(const void *a, const void *b) {
    const fo_zi *x = (const fo_zi *)a, *y = (const fo_zi *)b;
    if (x->zbits != y->zbits) return x->zbits < y->zbits ? -1 : 1;
    if (x->idx != y->idx) return x->idx < y->idx ? -1 : 1;
    return 0;
}
int fo_global_order(int n, const int32_t *radius, const float *depth, uint32_t *order) {
    fo_zi *a = (fo_zi *)malloc((n ? n : 1) * sizeof(fo_zi));
    int c = 0;
    for (int i = 0; i < n; ++i)
        if (radius[i] > 0) { a[c].zbits = f2u(depth[i]); a[c].idx = (uint32_t)i; ++c; }
    qsort(a, c, sizeof(fo_zi), cmp_zi);
    for (int i = 0; i < c; ++i) order[i] = a[i].idx;
    free(a);
    return c;
}

/* ------------------------------------------------------------------------------------------
 * The per-(pixel, Gaussian) arithmetic shared by every driver below (C1-R steps 2-3).
 * Returns 0 if the Gaussian does not contribute at this pixel, else 1 and *alpha.
 * PAPER.md:85 G(u)=exp(-(u^2+v^2)/2) == exp(-q/2); PAPER.md:95 alpha = op * G.
 * ------------------------------------------------------------------------------------------ */
float fo_q(float pxg, float pyg, float A, float B, float C, int x, int y) {
    const float dx = pxg - (float)x, dy = pyg - (float)y;
    return fmaf(dx, fmaf(2.0f * B, dy, A * dx), (C * dy) * dy);
}

/* Surfel mode (NEXT-3): g_rt != NULL selects the ray-transform evaluation for every driver below.  It is set by
 * fo_set_surfel() around a call (the drivers' argument lists stay those of the EWA path). */
static const float *g_rt = NULL;
void fo_set_surfel(const float *ray_transform /* [n,12] or NULL */) { g_rt = ray_transform; }

static inline int eval_alpha(const float *xy, const float *co, uint32_t g, int x, int y,
                             float q_cut, float alpha_max, double *alpha) {
    if (g_rt) {
        float p[3], num, den;
        fo_surfel_terms(g_rt + 12 * (size_t)g, x, y, p, &num, &den);
        if (!(den > 0.0f) || !(num <= q_cut * den)) return 0;
        const double G = exp(-0.5 * ((double)num / (double)den));
        *alpha = fmin((double)alpha_max, (double)co[4 * g + 3] * G);
        return 1;
    }
    const float q = fo_q(xy[2 * g], xy[2 * g + 1], co[4 * g], co[4 * g + 1], co[4 * g + 2], x, y);
    if (!(q <= q_cut)) return 0;
    const double G = exp(-0.5 * fmax((double)q, 0.0));
    const double a = (double)co[4 * g + 3] * G;
    *alpha = fmin((double)alpha_max, a);
    return 1;
}

static inline int is_fragile(double T, double t_min) { return fabs(T / t_min - 1.0) < 1e-4; }

/* ------------------------------------------------------------------------------------------
 * Step R, literal form (C1-R): for each requested pixel, walk ALL visible Gaussians in the
 * global order; no tiles, no boxes.  pix == NULL means all W*H pixels in row-major order.
 * Outputs (double, npix rows): rgb[3], feat_img[D] (may be NULL), T_final, n_contrib, fragile.
 * PAPER.md:90-95 (Eq. 4).
 * ------------------------------------------------------------------------------------------ */
void fo_render_literal(int n_order, const uint32_t *order, int D, const float *xy,
                       const float *conic_opacity, const float *rgb_g, const float *feat, int W,
                       int H, const float *prm, int64_t npix, const int32_t *pix, double *out_rgb,
                       double *out_feat, double *out_T, uint32_t *out_n, uint8_t *out_fragile) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    if (!pix) npix = (int64_t)W * H;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t p = 0; p < npix; ++p) {
        const int id = pix ? pix[p] : (int)p;
        const int x = id % W, y = id / W;
        double T = 1.0, C[3] = {0, 0, 0};
        uint32_t cnt = 0; uint8_t frag = 0;
        double *F = out_feat ? out_feat + (size_t)p * D : NULL;
        if (F) for (int c = 0; c < D; ++c) F[c] = 0.0;
        for (int k = 0; k < n_order; ++k) {
            if (is_fragile(T, t_min)) frag = 1;
            if (T < t_min) break;                                   /* step 1 */
            const uint32_t g = order[k];
            double alpha;
            if (!eval_alpha(xy, conic_opacity, g, x, y, q_cut, alpha_max, &alpha)) continue;
            const double w = alpha * T;                             /* w_i = alpha_i T_i */
            for (int c = 0; c < 3; ++c) C[c] += w * (double)rgb_g[3 * g + c];
            if (F) { const float *f = feat + (size_t)g * D; for (int c = 0; c < D; ++c) F[c] += w * (double)f[c]; }
            T = T * (1.0 - alpha);
            ++cnt;
        }
        if (is_fragile(T, t_min)) frag = 1;
        for (int c = 0; c < 3; ++c) out_rgb[3 * p + c] = C[c] + T * (double)prm[P_BG0 + c];
        out_T[p] = T; out_n[p] = cnt; if (out_fragile) out_fragile[p] = frag;
    }
}

/* ------------------------------------------------------------------------------------------
 * Step R, footprint-scatter form: same global order and same arithmetic; each Gaussian visits
 * only the pixels of the box |x-px|<=r, |y-py|<=r, which contains every pixel with q<=9
 * (C1-P step 8).  Threads own horizontal strips of rows, so every pixel sees the same sequence of
 * operations as in the literal form -> the two must agree bitwise (pin C3-17).
 * ------------------------------------------------------------------------------------------ */
void fo_render_scatter(int n_order, const uint32_t *order, int D, const float *xy,
                       const float *conic_opacity, const float *rgb_g, const float *feat,
                       const int32_t *radius, int W, int H, const float *prm, double *out_rgb,
                       double *out_feat, double *out_T, uint32_t *out_n, uint8_t *out_fragile) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    const int strip = 8;
    const int nstrips = (H + strip - 1) / strip;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nstrips; ++s) {
        const int ya = s * strip, yb = (ya + strip < H) ? ya + strip : H;
        for (int y = ya; y < yb; ++y)
            for (int x = 0; x < W; ++x) {
                const size_t p = (size_t)y * W + x;
                out_T[p] = 1.0; out_n[p] = 0; if (out_fragile) out_fragile[p] = 0;
                out_rgb[3 * p] = out_rgb[3 * p + 1] = out_rgb[3 * p + 2] = 0.0;
                if (out_feat) for (int c = 0; c < D; ++c) out_feat[p * D + c] = 0.0;
            }
        for (int k = 0; k < n_order; ++k) {
            const uint32_t g = order[k];
            const float r = (float)radius[g];
            const float pxg = xy[2 * g], pyg = xy[2 * g + 1];
            /* clamp in float first: a huge footprint must not overflow the int conversion */
            const int y0 = (int)fmaxf(ceilf(pyg - r), (float)ya);
            const int y1 = (int)fminf(floorf(pyg + r), (float)(yb - 1));
            if (y0 > y1) continue;
            const int x0 = (int)fmaxf(ceilf(pxg - r), 0.0f);
            const int x1 = (int)fminf(floorf(pxg + r), (float)(W - 1));
            for (int y = y0; y <= y1; ++y)
                for (int x = x0; x <= x1; ++x) {
                    const size_t p = (size_t)y * W + x;
                    const double T = out_T[p];
                    if (out_fragile && is_fragile(T, t_min)) out_fragile[p] = 1;
                    if (T < t_min) continue;
                    double alpha;
                    if (!eval_alpha(xy, conic_opacity, g, x, y, q_cut, alpha_max, &alpha)) continue;
                    const double w = alpha * T;
                    for (int c = 0; c < 3; ++c) out_rgb[3 * p + c] += w * (double)rgb_g[3 * g + c];
                    if (out_feat) {
                        const float *f = feat + (size_t)g * D; double *F = out_feat + p * D;
                        for (int c = 0; c < D; ++c) F[c] += w * (double)f[c];
                    }
                    out_T[p] = T * (1.0 - alpha);
                    out_n[p] += 1;
                }
        }
        for (int y = ya; y < yb; ++y)
            for (int x = 0; x < W; ++x) {
                const size_t p = (size_t)y * W + x;
                const double T = out_T[p];
                if (out_fragile && is_fragile(T, t_min)) out_fragile[p] = 1;
                for (int c = 0; c < 3; ++c) out_rgb[3 * p + c] += T * (double)prm[P_BG0 + c];
            }
    }
}

/* ------------------------------------------------------------------------------------------
 * Step F (C1-F), literal form: for every pixel walk ALL visible Gaussians in the global order with
 * exactly the weights w_i(x) = alpha_i T_i of step R, and accumulate
 *     num_i += w_i(x) * G(x)   (D-vector),   den_i += w_i(x)
 * (north_star's weight-aggregated fusion; reading D3 / C2-2).  num/den are ADDED TO (the caller
 * zeroes them), so several views accumulate (pin C3-19).  gt is [H,W,D] float.
 * ------------------------------------------------------------------------------------------ */
void fo_fuse_literal(int n, int n_order, const uint32_t *order, int D, const float *xy,
                     const float *conic_opacity, const float *gt, int W, int H, const float *prm,
                     double *num, double *den) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
#pragma omp parallel
    {
        double *pn = (double *)calloc((size_t)n * D + 1, sizeof(double));
        double *pd = (double *)calloc((size_t)n + 1, sizeof(double));
#pragma omp for schedule(static)
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                const float *Gx = gt + ((size_t)y * W + x) * D;
                double T = 1.0;
                for (int k = 0; k < n_order; ++k) {
                    if (T < t_min) break;
                    const uint32_t g = order[k];
                    double alpha;
                    if (!eval_alpha(xy, conic_opacity, g, x, y, q_cut, alpha_max, &alpha)) continue;
                    const double w = alpha * T;
                    double *ng = pn + (size_t)g * D;
                    for (int c = 0; c < D; ++c) ng[c] += w * (double)Gx[c];
                    pd[g] += w;
                    T = T * (1.0 - alpha);
                }
            }
#pragma omp critical
        {
            for (size_t j = 0; j < (size_t)n * D; ++j) num[j] += pn[j];
            for (int j = 0; j < n; ++j) den[j] += pd[j];
        }
        free(pn); free(pd);
    }
}

/* Step F, footprint-scatter form: same arithmetic; 8-row strips; each strip accumulates privately
 * for the Gaussians whose box meets it, then merges into num/den. */
void fo_fuse_scatter(int n, int n_order, const uint32_t *order, int D, const float *xy,
                     const float *conic_opacity, const int32_t *radius, const float *gt, int W,
                     int H, const float *prm, double *num, double *den) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    const int strip = 8;
    const int nstrips = (H + strip - 1) / strip;
    (void)n;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nstrips; ++s) {
        const int ya = s * strip, yb = (ya + strip < H) ? ya + strip : H;
        /* Gaussians whose box meets this strip, in global order */
        uint32_t *loc = (uint32_t *)malloc(((size_t)n_order + 1) * sizeof(uint32_t));
        int nl = 0;
        for (int k = 0; k < n_order; ++k) {
            const uint32_t g = order[k];
            const float r = (float)radius[g];
            const float fy0 = ceilf(xy[2 * g + 1] - r), fy1 = floorf(xy[2 * g + 1] + r);
            if (fy1 >= (float)ya && fy0 <= (float)(yb - 1)) loc[nl++] = g;
        }
        double *pn = (double *)calloc((size_t)nl * D + 1, sizeof(double));
        double *pd = (double *)calloc((size_t)nl + 1, sizeof(double));
        double *Tbuf = (double *)malloc((size_t)(yb - ya) * W * sizeof(double));
        for (size_t j = 0; j < (size_t)(yb - ya) * W; ++j) Tbuf[j] = 1.0;
        for (int l = 0; l < nl; ++l) {
            const uint32_t g = loc[l];
            const float r = (float)radius[g];
            const float pxg = xy[2 * g], pyg = xy[2 * g + 1];
            const int y0 = (int)fmaxf(ceilf(pyg - r), (float)ya);
            const int y1 = (int)fminf(floorf(pyg + r), (float)(yb - 1));
            const int x0 = (int)fmaxf(ceilf(pxg - r), 0.0f);
            const int x1 = (int)fminf(floorf(pxg + r), (float)(W - 1));
            double *ng = pn + (size_t)l * D;
            for (int y = y0; y <= y1; ++y)
                for (int x = x0; x <= x1; ++x) {
                    double *Tp = Tbuf + (size_t)(y - ya) * W + x;
                    const double T = *Tp;
                    if (T < t_min) continue;
                    double alpha;
                    if (!eval_alpha(xy, conic_opacity, g, x, y, q_cut, alpha_max, &alpha)) continue;
                    const double w = alpha * T;
                    const float *Gx = gt + ((size_t)y * W + x) * D;
                    for (int c = 0; c < D; ++c) ng[c] += w * (double)Gx[c];
                    pd[l] += w;
                    *Tp = T * (1.0 - alpha);
                }
        }
#pragma omp critical
        {
            for (int l = 0; l < nl; ++l) {
                if (pd[l] == 0.0) continue;
                double *dst = num + (size_t)loc[l] * D; const double *src = pn + (size_t)l * D;
                for (int c = 0; c < D; ++c) dst[c] += src[c];
                den[loc[l]] += pd[l];
            }
        }
        free(loc); free(pn); free(pd); free(Tbuf);
    }
}

/* Finalise (C1-F): f_i = num_i / den_i where den_i > den_eps, else f_i left unchanged;
 * l2norm != 0 additionally divides by ||f_i|| (PAPER.md:136 unit-norm features; off by default). */
void fo_fuse_finalize(int n, int D, const double *num, const double *den, double den_eps,
                      int l2norm, double *feat_inout) {
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        if (!(den[i] > den_eps)) continue;
        double *f = feat_inout + (size_t)i * D;
        double ss = 0.0;
        for (int c = 0; c < D; ++c) { f[c] = num[(size_t)i * D + c] / den[i]; ss += f[c] * f[c]; }
        if (l2norm && ss > 0.0) { const double inv = 1.0 / sqrt(ss); for (int c = 0; c < D; ++c) f[c] *= inv; }
    }
}

/* ------------------------------------------------------------------------------------------
 * NDFD forward (Eq. 5-6, Alg. 2).
 * Per pixel x with ground-truth feature f_gt = gt[x,:], over the fragments of the ray in the
 * front-to-back blend order of C1-R (same q cut-off, alpha clamp, w_i = alpha_i T_i, stop at
 * T < t_min):
 *     phi_i   = f_i . f_gt                      (features are unit-norm, so the
 *                                                cosine is the dot product)
 *     sigma_i = 1 / (1 + exp(k (phi_i - lambda)))
 *     L_gt(x) = sum_i w_i sigma_i                            (Eq. 5)
 *     L_cf(x) = sum_i sigma_i w_i (W_{i-1} - F_{i-1} . f_i)  (Eq. 6)
 * with W_n = sum_{i<=n} w_i and F_n = sum_{i<=n} w_i f_i accumulated
 *   mode 0: in blend order, front to back ("updated one time in each step during the
 *           front-to-back blend") -- the form the CUDA path builds;
 *   mode 1: from far to near ("along the ray from far to near"): the fragment list
 *           of the pixel is collected first and the recurrence runs over it reversed.
 * The two differ (sigma_i multiplies a different partner set); DESIGN.md lists the reading.
 * fo_ndfd_pairwise evaluates the explicit O(N^2) double sum of Eq. 6's first line over the same
 * fragment list (partners j = fragments BEFORE i in the accumulation order) -- the pin of the
 * O(N) recurrence.
 * pix: int32 linear pixel ids (y*W+x) or NULL for all pixels.  Outputs double [npix].
 * ------------------------------------------------------------------------------------------ */
typedef struct { double w; uint32_t g; } fo_frag;

static int collect_fragments(int n_order, const uint32_t *order, const float *xy, const float *co,
                             int x, int y, float q_cut, float alpha_max, double t_min,
                             fo_frag **buf, int *cap) {
    int cnt = 0;
    double T = 1.0;
    for (int k = 0; k < n_order; ++k) {
        if (T < t_min) break;
        const uint32_t g = order[k];
        double alpha;
        if (!eval_alpha(xy, co, g, x, y, q_cut, alpha_max, &alpha)) continue;
        if (cnt == *cap) { *cap = *cap ? 2 * *cap : 256; *buf = (fo_frag *)realloc(*buf, (size_t)*cap * sizeof(fo_frag)); }
        (*buf)[cnt].w = alpha * T; (*buf)[cnt].g = g; ++cnt;
        T = T * (1.0 - alpha);
    }
    return cnt;
}

static double dotf(const float *a, const float *b, int D) {
    double s = 0.0;
    for (int c = 0; c < D; ++c) s += (double)a[c] * (double)b[c];
    return s;
}

void fo_ndfd_literal(int n_order, const uint32_t *order, int D, const float *xy,
                     const float *conic_opacity, const float *feat, const float *gt, int W, int H,
                     const float *prm, double k_sig, double lambda, int mode, int64_t npix,
                     const int32_t *pix, double *out_lgt, double *out_lcf) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    if (!pix) npix = (int64_t)W * H;
#pragma omp parallel
    {
        fo_frag *fr = NULL; int cap = 0;
        double *F = (double *)malloc((size_t)D * sizeof(double));
#pragma omp for schedule(dynamic, 16)
        for (int64_t p = 0; p < npix; ++p) {
            const int id = pix ? pix[p] : (int)p;
            const int x = id % W, y = id / W;
            const float *fgt = gt + (size_t)id * D;
            const int cnt = collect_fragments(n_order, order, xy, conic_opacity, x, y, q_cut, alpha_max, t_min, &fr, &cap);
            double lgt = 0.0, lcf = 0.0, Wc = 0.0;
            for (int c = 0; c < D; ++c) F[c] = 0.0;
            for (int s = 0; s < cnt; ++s) {
                const fo_frag *e = &fr[mode ? cnt - 1 - s : s];
                const float *f = feat + (size_t)e->g * D;
                const double phi = dotf(f, fgt, D);
                const double sigma = 1.0 / (1.0 + exp(k_sig * (phi - lambda)));
                double Ff = 0.0;
                for (int c = 0; c < D; ++c) Ff += F[c] * (double)f[c];
                lgt += e->w * sigma;
                lcf += sigma * e->w * (Wc - Ff);
                Wc += e->w;
                for (int c = 0; c < D; ++c) F[c] += e->w * (double)f[c];
            }
            out_lgt[p] = lgt; out_lcf[p] = lcf;
        }
        free(F); free(fr);
    }
}

void fo_ndfd_pairwise(int n_order, const uint32_t *order, int D, const float *xy,
                      const float *conic_opacity, const float *feat, const float *gt, int W, int H,
                      const float *prm, double k_sig, double lambda, int mode, int64_t npix,
                      const int32_t *pix, double *out_lcf) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    if (!pix) npix = (int64_t)W * H;
#pragma omp parallel
    {
        fo_frag *fr = NULL; int cap = 0;
#pragma omp for schedule(dynamic, 16)
        for (int64_t p = 0; p < npix; ++p) {
            const int id = pix ? pix[p] : (int)p;
            const float *fgt = gt + (size_t)id * D;
            const int cnt = collect_fragments(n_order, order, xy, conic_opacity, id % W, id / W, q_cut, alpha_max, t_min, &fr, &cap);
            double lcf = 0.0;
            for (int s = 0; s < cnt; ++s) {
                const fo_frag *ei = &fr[mode ? cnt - 1 - s : s];
                const float *fi = feat + (size_t)ei->g * D;
                const double sigma = 1.0 / (1.0 + exp(k_sig * (dotf(fi, fgt, D) - lambda)));
                for (int t = 0; t < s; ++t) {
                    const fo_frag *ej = &fr[mode ? cnt - 1 - t : t];
                    lcf += sigma * ei->w * ej->w * (1.0 - dotf(fi, feat + (size_t)ej->g * D, D));
                }
            }
            out_lcf[p] = lcf;
        }
        free(fr);
    }
}

/* ------------------------------------------------------------------------------------------
 * NDFD backward at the w level (PAPER.md:142-146 and appendix A.2,
 * PAPER.md:361-383).  Total loss over the requested pixels
 *     L = sum_x ( lam1 L_gt(x) + lam2 L_cf(x) ),   L_gt, L_cf as in fo_ndfd_literal, mode 0
 * and, per pixel, over its fragment list k = 1..N in blend order:
 *     dL/dw_k     = lam1 sigma_k
 *                 + lam2 [ sigma_k (W_{k-1} - F_{k-1}.f_k) + sum_{i>k} sigma_i w_i (1 - f_i.f_k) ]
 *                                                        (PAPER.md:144 / 365-368)
 *     dL/dalpha_k = T_k dL/dw_k - (1/(1-alpha_k)) sum_{j>k} dL/dw_j w_j      (
 *                   w_j = alpha_j T_j, T_j = prod_{i<j}(1-alpha_i))
 *     dL/dop_g   += dL/dalpha_k G_k   where alpha_k = op_g G_k is not clamped by alpha_max
 * (alpha = min(alpha_max, op G): a clamped fragment passes no gradient to op).  The fragment list is
 * the realised one (cut-off, stopping rule); its dependence on the parameters is not
 * differentiated, exactly as in any alpha-blending rasteriser.  The geometry chain
 * (dG/d mean, scale, rotation) is out of scope.
 * Everything in double.  out_grad_op[n] is ACCUMULATED into (caller zeroes it); returns L.
 * ------------------------------------------------------------------------------------------ */
double fo_ndfd_backward(int n_order, const uint32_t *order, int D, const float *xy,
                        const float *conic_opacity, const float *feat, const float *gt, int W, int H,
                        const float *prm, double k_sig, double lambda, double lam1, double lam2,
                        int64_t npix, const int32_t *pix, double *out_grad_op) {
    const float q_cut = prm[P_QCUT], alpha_max = prm[P_AMAX];
    const double t_min = (double)prm[P_TMIN];
    double L_total = 0.0;
    if (!pix) npix = (int64_t)W * H;
#pragma omp parallel reduction(+ : L_total)
    {
        int cap = 0;
        uint32_t *gid = NULL;
        double *al = NULL, *Gv = NULL, *Tk = NULL, *wk = NULL, *sg = NULL, *gw = NULL;
        double *F = (double *)malloc((size_t)D * sizeof(double));
        double *B = (double *)malloc((size_t)D * sizeof(double));
#pragma omp for schedule(dynamic, 16)
        for (int64_t p = 0; p < npix; ++p) {
            const int id = pix ? pix[p] : (int)p;
            const int x = id % W, y = id / W;
            const float *fgt = gt + (size_t)id * D;
            /* forward: realised fragment list with alpha, G, T, w, sigma */
            int cnt = 0;
            double T = 1.0;
            for (int k = 0; k < n_order; ++k) {
                if (T < t_min) break;
                const uint32_t g = order[k];
                double G;
                if (g_rt) {   /* surfel mode: G = exp(-(u^2+v^2)/2) from the ray transform (same decision as eval_alpha) */
                    float pp[3], num, den;
                    fo_surfel_terms(g_rt + 12 * (size_t)g, x, y, pp, &num, &den);
                    if (!(den > 0.0f) || !(num <= q_cut * den)) continue;
                    G = exp(-0.5 * ((double)num / (double)den));
                } else {
                    const float q = fo_q(xy[2 * g], xy[2 * g + 1], conic_opacity[4 * g], conic_opacity[4 * g + 1], conic_opacity[4 * g + 2], x, y);
                    if (!(q <= q_cut)) continue;
                    G = exp(-0.5 * fmax((double)q, 0.0));
                }
                const double a_raw = (double)conic_opacity[4 * g + 3] * G;
                const double a = fmin((double)alpha_max, a_raw);
                if (cnt == cap) {
                    cap = cap ? 2 * cap : 256;
                    gid = (uint32_t *)realloc(gid, (size_t)cap * sizeof(uint32_t));
                    al = (double *)realloc(al, (size_t)cap * sizeof(double)); Gv = (double *)realloc(Gv, (size_t)cap * sizeof(double));
                    Tk = (double *)realloc(Tk, (size_t)cap * sizeof(double)); wk = (double *)realloc(wk, (size_t)cap * sizeof(double));
                    sg = (double *)realloc(sg, (size_t)cap * sizeof(double)); gw = (double *)realloc(gw, (size_t)cap * sizeof(double));
                }
                gid[cnt] = g; al[cnt] = a; Gv[cnt] = (a_raw < (double)alpha_max) ? G : 0.0;   /* clamped: no gradient to op */
                Tk[cnt] = T; wk[cnt] = a * T;
                sg[cnt] = 1.0 / (1.0 + exp(k_sig * (dotf(feat + (size_t)g * D, fgt, D) - lambda)));
                T = T * (1.0 - a);
                ++cnt;
            }
            /* loss (mode 0 recurrence) and the prefix part of dL/dw_k */
            double Wc = 0.0, lgt = 0.0, lcf = 0.0;
            for (int c = 0; c < D; ++c) F[c] = 0.0;
            for (int s = 0; s < cnt; ++s) {
                const float *f = feat + (size_t)gid[s] * D;
                double Ff = 0.0;
                for (int c = 0; c < D; ++c) Ff += F[c] * (double)f[c];
                lgt += wk[s] * sg[s];
                lcf += sg[s] * wk[s] * (Wc - Ff);
                gw[s] = lam1 * sg[s] + lam2 * sg[s] * (Wc - Ff);
                Wc += wk[s];
                for (int c = 0; c < D; ++c) F[c] += wk[s] * (double)f[c];
            }
            L_total += lam1 * lgt + lam2 * lcf;
            /* suffix part: sum_{i>k} sigma_i w_i (1 - f_i.f_k) = A_k - B_k.f_k, then dL/dalpha */
            double A = 0.0, Csuf = 0.0;
            for (int c = 0; c < D; ++c) B[c] = 0.0;
            for (int s = cnt - 1; s >= 0; --s) {
                const float *f = feat + (size_t)gid[s] * D;
                double Bf = 0.0;
                for (int c = 0; c < D; ++c) Bf += B[c] * (double)f[c];
                gw[s] += lam2 * (A - Bf);
                const double dalpha = Tk[s] * gw[s] - Csuf / (1.0 - al[s]);
                const double contrib = dalpha * Gv[s];
                if (contrib != 0.0) {
#pragma omp atomic
                    out_grad_op[gid[s]] += contrib;
                }
                Csuf += gw[s] * wk[s];
                A += sg[s] * wk[s];
                for (int c = 0; c < D; ++c) B[c] += sg[s] * wk[s] * (double)f[c];
            }
        }
        free(F); free(B); free(gid); free(al); free(Gv); free(Tk); free(wk); free(sg); free(gw);
    }
    return L_total;
}
