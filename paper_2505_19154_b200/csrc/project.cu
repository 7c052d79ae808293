// project.cu -- step P (fhgs_project): EWA projection, culling, tile rectangle, SH colour.
// PAPER.md:302 (CullGaussian), PAPER.md:309-310 (2DScreenGaussians); SURVEY 8(c) C1-P.
//
// Arithmetic rule of this step: every +,-,*,/,sqrt is ONE IEEE binary32 operation, round to
// nearest even, in the written order, never contracted into an FMA.  This file therefore uses
// the __f*_rn intrinsics throughout, which ptxas never fuses, so the result does not depend on
// compiler flags.  236 B read + 56 B written per visible Gaussian at SH degree 3; ~820 instructions per warp
// (18 IEEE divisions, 4 square roots), so the kernel is bound by issue slots and load latency together.
//
// Layout: one thread per Gaussian.  SH degree 3: every Gaussian that can be visible fetches its own 192-byte SH row with
// one bulk async copy while its covariance is computed (project_kernel<3, true>).  Degree 0-2 and the surfel kernel: the SH
// block of a CTA (256 Gaussians x K x 3 floats, one contiguous span of global memory) is staged through shared memory
// with coalesced 16-byte loads; every thread then reads its own row with a conflict-free padded stride.
#include "common.cuh"
#include "ws.cuh"   // mbarrier / bulk-copy wrappers

namespace {

__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float dvd(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float sq(float a) { return __fsqrt_rn(a); }
__device__ __forceinline__ float clampf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }
__device__ __forceinline__ bool finite_dev(float v) { return fabsf(v) <= 3.402823466e38f; }

struct ProjectArgs {
    int n, sh_degree, W, H, GW, GH;
    const float *mean, *scale, *quat, *opacity, *sh;
    float V[16];
    float cam_pos[3];
    float fx, fy, cx, cy, Lx, Ly;
    float z_near, dil;
    int tight;   // FHGS_RECT_TIGHT: per-axis 3-sigma extents instead of the scalar radius
    float *xy, *depth, *conic_opacity, *rgb;
    int32_t* radius;
    uint16_t* rect;
    uint32_t* tiles_touched;
    float q_cutoff;          // surfel mode: the footprint u^2 + v^2 <= q_cutoff
    float* ray_transform;    // surfel mode: [n,12]
};

constexpr int PROJ_THREADS = 256;

// Real orthonormal spherical harmonics up to degree 3 (C1-P step 10).
__device__ __forceinline__ void sh_basis(int degree, float x, float y, float z, float* Y) {
    const float C0 = 0.28209479177387814f, C1 = 0.4886025119029199f;
    Y[0] = C0;
    if (degree < 1) return;
    Y[1] = -mul(C1, y);
    Y[2] = mul(C1, z);
    Y[3] = -mul(C1, x);
    if (degree < 2) return;
    const float xx = mul(x, x), yy = mul(y, y), zz = mul(z, z);
    const float xy = mul(x, y), yz = mul(y, z), xz = mul(x, z);
    Y[4] = mul(1.0925484305920792f, xy);
    Y[5] = mul(-1.0925484305920792f, yz);
    Y[6] = mul(0.31539156525252005f, sub(sub(mul(2.0f, zz), xx), yy));
    Y[7] = mul(-1.0925484305920792f, xz);
    Y[8] = mul(0.5462742152960396f, sub(xx, yy));
    if (degree < 3) return;
    Y[9] = mul(mul(-0.5900435899266435f, y), sub(mul(3.0f, xx), yy));
    Y[10] = mul(mul(2.890611442640554f, xy), z);
    Y[11] = mul(mul(-0.4570457994644658f, y), sub(sub(mul(4.0f, zz), xx), yy));
    Y[12] = mul(mul(0.3731763325901154f, z), sub(sub(mul(2.0f, zz), mul(3.0f, xx)), mul(3.0f, yy)));
    Y[13] = mul(mul(-0.4570457994644658f, x), sub(sub(mul(4.0f, zz), xx), yy));
    Y[14] = mul(mul(1.445305721320277f, z), sub(xx, yy));
    Y[15] = mul(mul(-0.5900435899266435f, x), sub(xx, mul(3.0f, yy)));
}

// Stage the CTA's SH rows: contiguous span [base*ROW, (base+cnt)*ROW), coalesced; row r lands at s_sh[r * PAD].
template <int DEG>
__device__ __forceinline__ void stage_sh_rows(const ProjectArgs& a, float* s_sh, int base, int cnt) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    constexpr int ROW = 3 * K;
    constexpr int PAD = (ROW % 2 == 0) ? ROW + 1 : ROW;
    {
        const float* src = a.sh + (size_t)base * ROW;
        const int total = cnt * ROW;
        if ((((uintptr_t)src) & 15) == 0) {
            const int total4 = total >> 2;
            const float4* src4 = reinterpret_cast<const float4*>(src);
            for (int j = threadIdx.x; j < total4; j += PROJ_THREADS) {
                const float4 v = __ldg(src4 + j);
                const int e = j * 4;
                s_sh[((e + 0) / ROW) * PAD + (e + 0) % ROW] = v.x;
                s_sh[((e + 1) / ROW) * PAD + (e + 1) % ROW] = v.y;
                s_sh[((e + 2) / ROW) * PAD + (e + 2) % ROW] = v.z;
                s_sh[((e + 3) / ROW) * PAD + (e + 3) % ROW] = v.w;
            }
            for (int e = (total4 << 2) + threadIdx.x; e < total; e += PROJ_THREADS)
                s_sh[(e / ROW) * PAD + e % ROW] = __ldg(src + e);
        } else {
            for (int e = threadIdx.x; e < total; e += PROJ_THREADS)
                s_sh[(e / ROW) * PAD + e % ROW] = __ldg(src + e);
        }
    }
}

// C1-P step 10: SH colour of Gaussian at world position (p0,p1,p2) from its staged SH row.
template <int DEG>
__device__ __forceinline__ void sh_colour(const ProjectArgs& a, const float* row, float p0, float p1, float p2, float* o_rgb) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    float dx = sub(p0, a.cam_pos[0]), dy = sub(p1, a.cam_pos[1]), dz = sub(p2, a.cam_pos[2]);
    const float dn = sq(add(add(mul(dx, dx), mul(dy, dy)), mul(dz, dz)));
    dx = dvd(dx, dn); dy = dvd(dy, dn); dz = dvd(dz, dn);
    float Yb[K];
    sh_basis(DEG, dx, dy, dz, Yb);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        float c = 0.5f;
#pragma unroll
        for (int l = 0; l < K; ++l) c = add(c, mul(Yb[l], row[3 * l + k]));
        o_rgb[k] = fmaxf(c, 0.0f);
    }
}

// DIRECT (launched for SH degree 3 with a 16-byte aligned sh array; the rows must be a multiple of 16 bytes): no cooperative
// staging and no CTA-wide barrier.  A thread whose Gaussian passes the z cull and a generous frame test starts ONE bulk
// async copy (cp.async.bulk) of its own row into its own shared-memory slot (stride 208 bytes: conflict-free for the
// 16-byte reads), counted on its warp's mbarrier; the warp does the covariance arithmetic while the rows fly and waits
// for them only before the colour.  Rows of culled Gaussians are not fetched, and the warps of a CTA run their load and
// arithmetic phases out of step with each other.
template <int DEG, bool DIRECT>
__global__ void __launch_bounds__(PROJ_THREADS, DIRECT ? 4 : 1) project_kernel(const ProjectArgs a) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    constexpr int ROW = 3 * K;                 // floats per Gaussian
    constexpr int PAD = (ROW % 2 == 0) ? ROW + 1 : ROW;  // odd stride -> conflict-free rows
    constexpr int DSTRIDE = ROW + 4;           // DIRECT: floats between the row slots of two threads (208 B at degree 3)
    bool staged_row = false;
    uint32_t warp_rows = 0;   // DIRECT: lanes of this warp with a row copy in flight
    extern __shared__ __align__(16) float s_sh[];   // [PROJ_THREADS][PAD], or [PROJ_THREADS][DSTRIDE] in the DIRECT form

    __shared__ uint64_t s_bar[PROJ_THREADS / 32];
    const int base = blockIdx.x * PROJ_THREADS;
    const int i = base + threadIdx.x;
    if (!DIRECT) {
        const int cnt = min(PROJ_THREADS, a.n - base);
        stage_sh_rows<DEG>(a, s_sh, base, cnt);
        __syncthreads();
    } else {
        // per-warp barrier, one phase: lane 0 arrives once with the byte count of the warp's rows
        if ((threadIdx.x & 31) == 0) {
            mbar_init(&s_bar[threadIdx.x >> 5], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncwarp();
        // the frame test (a hint: it decides no result -- a visible Gaussian it misses reads its row from global memory in
        // step 10) is taken by the whole warp before any lane leaves
        bool want = false;
        if (i < a.n) {
            const float p0 = __ldg(a.mean + 3 * (size_t)i), p1 = __ldg(a.mean + 3 * (size_t)i + 1),
                        p2 = __ldg(a.mean + 3 * (size_t)i + 2);
            const float* V = a.V;
            const float tx = V[0] * p0 + V[1] * p1 + V[2] * p2 + V[3], ty = V[4] * p0 + V[5] * p1 + V[6] * p2 + V[7],
                        tz = V[8] * p0 + V[9] * p1 + V[10] * p2 + V[11];
            const float hx = a.fx * tx + (a.cx - 0.5f * (float)a.W) * tz, hy = a.fy * ty + (a.cy - 0.5f * (float)a.H) * tz;
            // |px - W/2| <= W/2 + margin, written without the division; margin ~ the 3-sigma radius of the largest axis
            // (4.2 = 3 sigma x 1.4, the factor covering the clamped perspective stretch) plus the dilation and one tile of slack
            const float smax = fmaxf(fmaxf(__ldg(a.scale + 3 * (size_t)i), __ldg(a.scale + 3 * (size_t)i + 1)), __ldg(a.scale + 3 * (size_t)i + 2));
            const float mz = 4.2f * smax * fmaxf(fabsf(a.fx), fabsf(a.fy)) + 18.f * tz;   // margin * tz
            want = tz >= a.z_near && fabsf(hx) <= 0.5f * (float)a.W * tz + mz && fabsf(hy) <= 0.5f * (float)a.H * tz + mz;
        }
        const uint32_t ballot = __ballot_sync(0xffffffffu, want);
        if (ballot) {
            uint64_t* bar = &s_bar[threadIdx.x >> 5];
            if ((threadIdx.x & 31) == 0) {
                mbar_expect_tx(bar, (uint32_t)(__popc(ballot) * ROW * 4));
                mbar_arrive(bar);
            }
            __syncwarp();
            if (want) bulk_g2s(s_sh + threadIdx.x * DSTRIDE, a.sh + (size_t)i * ROW, ROW * 4, bar);
        }
        staged_row = want;
        warp_rows = ballot;
    }
    if (i >= a.n) return;

    float o_xy0 = 0.f, o_xy1 = 0.f, o_depth = 0.f;
    float4 o_co = make_float4(0.f, 0.f, 0.f, 0.f);
    float o_rgb[3] = {0.f, 0.f, 0.f};
    int o_radius = 0;
    uint32_t o_tt = 0;
    ushort4 o_rect = make_ushort4(0, 0, 0, 0);

    do {
        const float p0 = __ldg(a.mean + 3 * (size_t)i), p1 = __ldg(a.mean + 3 * (size_t)i + 1),
                    p2 = __ldg(a.mean + 3 * (size_t)i + 2);
        // every per-Gaussian input is requested up front (one DRAM round trip instead of three dependent ones; a culled
        // Gaussian wastes 32 bytes)
        const float4 qv = __ldg(reinterpret_cast<const float4*>(a.quat) + i);
        const float s0 = __ldg(a.scale + 3 * (size_t)i), s1 = __ldg(a.scale + 3 * (size_t)i + 1),
                    s2 = __ldg(a.scale + 3 * (size_t)i + 2);
        const float op = __ldg(a.opacity + i);
        const float* V = a.V;
        // 1. camera-space position
        float t[3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
            t[k] = add(add(add(mul(V[4 * k], p0), mul(V[4 * k + 1], p1)), mul(V[4 * k + 2], p2)), V[4 * k + 3]);
        const float z = t[2];
        if (!(z >= a.z_near)) break;
        // 2. pixel position
        const float u = dvd(t[0], z), v = dvd(t[1], z);
        const float px = add(mul(a.fx, u), a.cx), py = add(mul(a.fy, v), a.cy);
        // 3. clamp for the Jacobian only
        const float uc = fminf(fmaxf(u, -a.Lx), a.Lx), vc = fminf(fmaxf(v, -a.Ly), a.Ly);
        const float X = mul(uc, z), Y = mul(vc, z);
        // 4. rotation from the (normalised) quaternion
        float qw = qv.x, qx = qv.y, qy = qv.z, qz = qv.w;
        const float qn = sq(add(add(add(mul(qw, qw), mul(qx, qx)), mul(qy, qy)), mul(qz, qz)));
        qw = dvd(qw, qn); qx = dvd(qx, qn); qy = dvd(qy, qn); qz = dvd(qz, qn);
        float R[9];
        R[0] = sub(1.0f, mul(2.0f, add(mul(qy, qy), mul(qz, qz))));
        R[1] = mul(2.0f, sub(mul(qx, qy), mul(qw, qz)));
        R[2] = mul(2.0f, add(mul(qx, qz), mul(qw, qy)));
        R[3] = mul(2.0f, add(mul(qx, qy), mul(qw, qz)));
        R[4] = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qz, qz))));
        R[5] = mul(2.0f, sub(mul(qy, qz), mul(qw, qx)));
        R[6] = mul(2.0f, sub(mul(qx, qz), mul(qw, qy)));
        R[7] = mul(2.0f, add(mul(qy, qz), mul(qw, qx)));
        R[8] = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qy, qy))));
        // 5. Sigma3D = (R S)(R S)^T
        float M[9];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            M[3 * k] = mul(R[3 * k], s0);
            M[3 * k + 1] = mul(R[3 * k + 1], s1);
            M[3 * k + 2] = mul(R[3 * k + 2], s2);
        }
        float S[9];
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = r; c < 3; ++c) {
                const float s = add(add(mul(M[3 * r], M[3 * c]), mul(M[3 * r + 1], M[3 * c + 1])),
                                    mul(M[3 * r + 2], M[3 * c + 2]));
                S[3 * r + c] = s;
                S[3 * c + r] = s;
            }
        // 6. A = J R_v  (2x3)
        const float J00 = dvd(a.fx, z), J02 = -dvd(mul(a.fx, X), mul(z, z));
        const float J11 = dvd(a.fy, z), J12 = -dvd(mul(a.fy, Y), mul(z, z));
        float A[6];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            A[j] = add(mul(J00, V[j]), mul(J02, V[8 + j]));
            A[3 + j] = add(mul(J11, V[4 + j]), mul(J12, V[8 + j]));
        }
        // 7. Sigma2D = A Sigma3D A^T + dil I
        float U[6];
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int j = 0; j < 3; ++j)
                U[3 * r + j] = add(add(mul(A[3 * r], S[j]), mul(A[3 * r + 1], S[3 + j])), mul(A[3 * r + 2], S[6 + j]));
        const float ca = add(add(add(mul(U[0], A[0]), mul(U[1], A[1])), mul(U[2], A[2])), a.dil);
        const float cb = add(add(mul(U[0], A[3]), mul(U[1], A[4])), mul(U[2], A[5]));
        const float cc = add(add(add(mul(U[3], A[3]), mul(U[4], A[4])), mul(U[5], A[5])), a.dil);
        const float det = sub(mul(ca, cc), mul(cb, cb));
        if (!(det > 0.0f)) break;
        const float inv = dvd(1.0f, det);
        const float conA = mul(cc, inv), conB = -mul(cb, inv), conC = mul(ca, inv);
        // 8. radius
        const float mid = mul(0.5f, add(ca, cc));
        const float disc = fmaxf(sub(mul(mid, mid), det), 0.0f);
        const float lam = add(mid, sq(disc));
        const float r = ceilf(mul(3.0f, sq(lam)));
        // 9. tile rectangle
        if (!(finite_dev(px) && finite_dev(py) && finite_dev(r))) break;
        // tight mode: the q <= 9 ellipse spans exactly +-3 sqrt(Sigma_xx) in x and +-3 sqrt(Sigma_yy) in y
        const float rx = a.tight ? ceilf(mul(3.0f, sq(ca))) : r, ry = a.tight ? ceilf(mul(3.0f, sq(cc))) : r;
        const float x0 = clampf(floorf(dvd(sub(px, rx), 16.0f)), 0.0f, (float)a.GW);
        const float x1 = clampf(add(floorf(dvd(add(px, rx), 16.0f)), 1.0f), 0.0f, (float)a.GW);
        const float y0 = clampf(floorf(dvd(sub(py, ry), 16.0f)), 0.0f, (float)a.GH);
        const float y1 = clampf(add(floorf(dvd(add(py, ry), 16.0f)), 1.0f), 0.0f, (float)a.GH);
        const int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
        if (ix1 <= ix0 || iy1 <= iy0) break;
        // 10. SH colour
        if (DIRECT && staged_row) {
            mbar_wait(&s_bar[threadIdx.x >> 5], 0);   // the rows of this warp have landed
            sh_colour<DEG>(a, s_sh + threadIdx.x * DSTRIDE, p0, p1, p2, o_rgb);
        } else if (DIRECT) {
            sh_colour<DEG>(a, a.sh + (size_t)i * ROW, p0, p1, p2, o_rgb);   // rare: scalar loads from global memory
        } else {
            sh_colour<DEG>(a, s_sh + threadIdx.x * PAD, p0, p1, p2, o_rgb);
        }
        o_xy0 = px; o_xy1 = py; o_depth = z;
        o_co = make_float4(conA, conB, conC, op);
        o_radius = (int)r;
        o_rect = make_ushort4((unsigned short)ix0, (unsigned short)iy0, (unsigned short)ix1, (unsigned short)iy1);
        o_tt = (uint32_t)((ix1 - ix0) * (iy1 - iy0));
    } while (0);

    // no lane leaves while a copy into this CTA's shared memory may still be in flight
    if (DIRECT && warp_rows) mbar_wait(&s_bar[threadIdx.x >> 5], 0);
    reinterpret_cast<float2*>(a.xy)[i] = make_float2(o_xy0, o_xy1);
    a.depth[i] = o_depth;
    reinterpret_cast<float4*>(a.conic_opacity)[i] = o_co;
    a.rgb[3 * (size_t)i] = o_rgb[0];
    a.rgb[3 * (size_t)i + 1] = o_rgb[1];
    a.rgb[3 * (size_t)i + 2] = o_rgb[2];
    a.radius[i] = o_radius;
    reinterpret_cast<ushort4*>(a.rect)[i] = o_rect;
    a.tiles_touched[i] = o_tt;
}

// ---------------------------------------------------------------------------------------------
// Surfel mode (FHGS_PRIM_SURFEL, Eq. 1-3): homography T = K [a b c] of the splat's
// tangent plane, its adjugate as the per-splat ray transform, the footprint's bounding box from the dual conic.
// Same arithmetic rule: single binary32 operations in the written order (bit-identical to the oracle's statement).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void cross3(const float* x, const float* y, float* o) {
    o[0] = sub(mul(x[1], y[2]), mul(x[2], y[1]));
    o[1] = sub(mul(x[2], y[0]), mul(x[0], y[2]));
    o[2] = sub(mul(x[0], y[1]), mul(x[1], y[0]));
}

template <int DEG>
__global__ void __launch_bounds__(PROJ_THREADS) project_surfel_kernel(const ProjectArgs a) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    constexpr int ROW = 3 * K;
    constexpr int PAD = (ROW % 2 == 0) ? ROW + 1 : ROW;
    extern __shared__ float s_sh[];
    const int base = blockIdx.x * PROJ_THREADS;
    const int i = base + threadIdx.x;
    const int cnt = min(PROJ_THREADS, a.n - base);
    stage_sh_rows<DEG>(a, s_sh, base, cnt);
    __syncthreads();
    if (i >= a.n) return;

    float o_xy0 = 0.f, o_xy1 = 0.f, o_depth = 0.f;
    float4 o_co = make_float4(0.f, 0.f, 0.f, 0.f);
    float o_rgb[3] = {0.f, 0.f, 0.f};
    int o_radius = 0;
    uint32_t o_tt = 0;
    ushort4 o_rect = make_ushort4(0, 0, 0, 0);
    float4 o_rt[3] = {make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)};

    do {
        const float p0 = __ldg(a.mean + 3 * (size_t)i), p1 = __ldg(a.mean + 3 * (size_t)i + 1),
                    p2 = __ldg(a.mean + 3 * (size_t)i + 2);
        const float* V = a.V;
        // 1. camera-space centre
        float c[3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
            c[k] = add(add(add(mul(V[4 * k], p0), mul(V[4 * k + 1], p1)), mul(V[4 * k + 2], p2)), V[4 * k + 3]);
        if (!(c[2] >= a.z_near)) break;
        // 2. scaled tangents in camera space
        const float4 qv = __ldg(reinterpret_cast<const float4*>(a.quat) + i);
        float qw = qv.x, qx = qv.y, qy = qv.z, qz = qv.w;
        const float qn = sq(add(add(add(mul(qw, qw), mul(qx, qx)), mul(qy, qy)), mul(qz, qz)));
        qw = dvd(qw, qn); qx = dvd(qx, qn); qy = dvd(qy, qn); qz = dvd(qz, qn);
        float R[9];
        R[0] = sub(1.0f, mul(2.0f, add(mul(qy, qy), mul(qz, qz))));
        R[1] = mul(2.0f, sub(mul(qx, qy), mul(qw, qz)));
        R[3] = mul(2.0f, add(mul(qx, qy), mul(qw, qz)));
        R[4] = sub(1.0f, mul(2.0f, add(mul(qx, qx), mul(qz, qz))));
        R[6] = mul(2.0f, sub(mul(qx, qz), mul(qw, qy)));
        R[7] = mul(2.0f, add(mul(qy, qz), mul(qw, qx)));
        const float su = __ldg(a.scale + 3 * (size_t)i), sv = __ldg(a.scale + 3 * (size_t)i + 1);
        const float aw[3] = {mul(R[0], su), mul(R[3], su), mul(R[6], su)};
        const float bw[3] = {mul(R[1], sv), mul(R[4], sv), mul(R[7], sv)};
        float ta[3], tb[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            ta[k] = add(add(mul(V[4 * k], aw[0]), mul(V[4 * k + 1], aw[1])), mul(V[4 * k + 2], aw[2]));
            tb[k] = add(add(mul(V[4 * k], bw[0]), mul(V[4 * k + 1], bw[1])), mul(V[4 * k + 2], bw[2]));
        }
        // 3. the whole 3-sigma disc behind the near plane
        const float zmin = sub(c[2], mul(3.0f, sq(add(mul(ta[2], ta[2]), mul(tb[2], tb[2])))));
        if (!(zmin >= a.z_near)) break;
        // 4. T rows
        const float Tx[3] = {add(mul(a.fx, ta[0]), mul(a.cx, ta[2])), add(mul(a.fx, tb[0]), mul(a.cx, tb[2])), add(mul(a.fx, c[0]), mul(a.cx, c[2]))};
        const float Ty[3] = {add(mul(a.fy, ta[1]), mul(a.cy, ta[2])), add(mul(a.fy, tb[1]), mul(a.cy, tb[2])), add(mul(a.fy, c[1]), mul(a.cy, c[2]))};
        const float Tw[3] = {ta[2], tb[2], c[2]};
        // 5. adjugate, scaled by an exact power of two
        float A0[3], A1[3], A2[3];
        cross3(Ty, Tw, A0); cross3(Tw, Tx, A1); cross3(Tx, Ty, A2);
        float mx = 0.0f;
#pragma unroll
        for (int k = 0; k < 3; ++k) mx = fmaxf(mx, fmaxf(fabsf(A0[k]), fmaxf(fabsf(A1[k]), fabsf(A2[k]))));
        if (!(mx > 0.0f) || !finite_dev(mx)) break;
        int e;
        (void)frexpf(mx, &e);
        const float sc = ldexpf(1.0f, -e);
        // 6. bounding box of the footprint (dual conic)
        const float qc = a.q_cutoff;
        const float d = sub(add(mul(qc, mul(Tw[0], Tw[0])), mul(qc, mul(Tw[1], Tw[1]))), mul(Tw[2], Tw[2]));
        if (!(d < 0.0f)) break;
        const float ccx = dvd(sub(add(mul(qc, mul(Tx[0], Tw[0])), mul(qc, mul(Tx[1], Tw[1]))), mul(Tx[2], Tw[2])), d);
        const float ccy = dvd(sub(add(mul(qc, mul(Ty[0], Tw[0])), mul(qc, mul(Ty[1], Tw[1]))), mul(Ty[2], Tw[2])), d);
        const float ex = sub(mul(ccx, ccx), dvd(sub(add(mul(qc, mul(Tx[0], Tx[0])), mul(qc, mul(Tx[1], Tx[1]))), mul(Tx[2], Tx[2])), d));
        const float ey = sub(mul(ccy, ccy), dvd(sub(add(mul(qc, mul(Ty[0], Ty[0])), mul(qc, mul(Ty[1], Ty[1]))), mul(Ty[2], Ty[2])), d));
        const float hx = add(sq(fmaxf(ex, 1e-4f)), 1.0f), hy = add(sq(fmaxf(ey, 1e-4f)), 1.0f);
        if (!(finite_dev(ccx) && finite_dev(ccy) && finite_dev(hx) && finite_dev(hy))) break;
        const float rx = ceilf(hx), ry = ceilf(hy);
        const float x0 = clampf(floorf(dvd(sub(ccx, rx), 16.0f)), 0.0f, (float)a.GW);
        const float x1 = clampf(add(floorf(dvd(add(ccx, rx), 16.0f)), 1.0f), 0.0f, (float)a.GW);
        const float y0 = clampf(floorf(dvd(sub(ccy, ry), 16.0f)), 0.0f, (float)a.GH);
        const float y1 = clampf(add(floorf(dvd(add(ccy, ry), 16.0f)), 1.0f), 0.0f, (float)a.GH);
        const int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
        if (ix1 <= ix0 || iy1 <= iy0) break;
        // 7. SH colour
        sh_colour<DEG>(a, s_sh + threadIdx.x * PAD, p0, p1, p2, o_rgb);
        o_xy0 = ccx; o_xy1 = ccy; o_depth = c[2];
        o_co = make_float4(hx, hy, 0.0f, __ldg(a.opacity + i));
        o_radius = (int)fmaxf(rx, ry);
        o_rect = make_ushort4((unsigned short)ix0, (unsigned short)iy0, (unsigned short)ix1, (unsigned short)iy1);
        o_tt = (uint32_t)((ix1 - ix0) * (iy1 - iy0));
#pragma unroll
        for (int r = 0; r < 3; ++r) o_rt[r] = make_float4(mul(A0[r], sc), mul(A1[r], sc), mul(A2[r], sc), 0.0f);
    } while (0);

    reinterpret_cast<float2*>(a.xy)[i] = make_float2(o_xy0, o_xy1);
    a.depth[i] = o_depth;
    reinterpret_cast<float4*>(a.conic_opacity)[i] = o_co;
    a.rgb[3 * (size_t)i] = o_rgb[0];
    a.rgb[3 * (size_t)i + 1] = o_rgb[1];
    a.rgb[3 * (size_t)i + 2] = o_rgb[2];
    a.radius[i] = o_radius;
    reinterpret_cast<ushort4*>(a.rect)[i] = o_rect;
    a.tiles_touched[i] = o_tt;
#pragma unroll
    for (int r = 0; r < 3; ++r) reinterpret_cast<float4*>(a.ray_transform)[3 * (size_t)i + r] = o_rt[r];
}

template <int DEG>
cudaError_t launch_project(const ProjectArgs& a, cudaStream_t st) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    constexpr int ROW = 3 * K;
    constexpr int PAD = (ROW % 2 == 0) ? ROW + 1 : ROW;
    const size_t smem = (size_t)PROJ_THREADS * PAD * sizeof(float);
    const int grid = (a.n + PROJ_THREADS - 1) / PROJ_THREADS;
    // degree 3 (192-byte rows): the per-row bulk-copy form; the shorter rows of degree 0-2 measured faster staged
    if (!a.ray_transform && DEG == 3 && aligned_to(a.sh, 16)) {
        const size_t dsmem = (size_t)PROJ_THREADS * (ROW + 4) * sizeof(float);
        cudaError_t e = cudaFuncSetAttribute(project_kernel<DEG, (DEG == 3)>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsmem);
        if (e != cudaSuccess) return e;
        project_kernel<DEG, (DEG == 3)><<<grid, PROJ_THREADS, dsmem, st>>>(a);
        return cudaGetLastError();
    }
    cudaError_t e = cudaFuncSetAttribute(project_kernel<DEG, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (a.ray_transform) {
        e = cudaFuncSetAttribute(project_surfel_kernel<DEG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        project_surfel_kernel<DEG><<<grid, PROJ_THREADS, smem, st>>>(a);
    } else {
        project_kernel<DEG, false><<<grid, PROJ_THREADS, smem, st>>>(a);
    }
    return cudaGetLastError();
}

}  // namespace

extern "C" fhgs_status fhgs_project(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                                    const fhgs_params* prm, fhgs_view_state* vs, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!g || !cam || !prm || !vs) FHGS_INVALID(ctx, "fhgs_project: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    if (g->n < 0 || g->n != vs->n) FHGS_INVALID(ctx, "fhgs_project: g->n < 0 or != vs->n");
    if (g->sh_degree < 0 || g->sh_degree > 3) FHGS_INVALID(ctx, "fhgs_project: sh_degree not in [0,3]");
    if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    if (g->n == 0) return FHGS_OK;
    if (!g->mean || !g->scale || !g->quat || !g->opacity || !g->sh)
        FHGS_INVALID(ctx, "fhgs_project: NULL Gaussian array");
    if (!aligned_to(g->quat, 16) || !aligned_to(g->mean, 4) || !aligned_to(g->scale, 4) || !aligned_to(g->sh, 4))
        FHGS_INVALID(ctx, "fhgs_project: quat must be 16-byte aligned");

    ProjectArgs a;
    a.n = g->n; a.sh_degree = g->sh_degree; a.W = cam->width; a.H = cam->height;
    a.GW = tiles_x(cam->width); a.GH = tiles_y(cam->height);
    a.mean = g->mean; a.scale = g->scale; a.quat = g->quat; a.opacity = g->opacity; a.sh = g->sh;
    memcpy(a.V, cam->view, sizeof(a.V));
    memcpy(a.cam_pos, cam->cam_pos, sizeof(a.cam_pos));
    const Intrinsics k = make_intrinsics(cam);
    a.fx = k.fx; a.fy = k.fy; a.cx = k.cx; a.cy = k.cy;
    a.Lx = prm->jac_clamp * k.tanx;   // single binary32 multiply, as C1-P step 3
    a.Ly = prm->jac_clamp * k.tany;
    a.z_near = prm->z_near; a.dil = prm->cov_dilation;
    a.tight = prm->rect_mode == FHGS_RECT_TIGHT;
    a.q_cutoff = prm->q_cutoff;
    a.ray_transform = prm->primitive == FHGS_PRIM_SURFEL ? vs->ray_transform : nullptr;
    a.xy = vs->xy; a.depth = vs->depth; a.conic_opacity = vs->conic_opacity; a.rgb = vs->rgb;
    a.radius = vs->radius; a.rect = vs->rect; a.tiles_touched = vs->tiles_touched;

    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    switch (g->sh_degree) {
        case 0: e = launch_project<0>(a, s); break;
        case 1: e = launch_project<1>(a, s); break;
        case 2: e = launch_project<2>(a, s); break;
        default: e = launch_project<3>(a, s); break;
    }
    FHGS_CUDA(ctx, e);
    return FHGS_OK;
}
