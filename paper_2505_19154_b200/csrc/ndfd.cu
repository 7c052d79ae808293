// ndfd.cu -- NDFD forward (fhgs_ndfd_forward): the paper's non-differentiable feature
// driving losses, evaluated in the same front-to-back traversal as step R without rendering a feature image
// (Eq. 5-6; Alg. 2):
//     phi_i = f_i . f_gt(x),  sigma_i = 1 / (1 + exp(k (phi_i - lambda))),  w_i = alpha_i T_i
//     L_gt(x) = sum_i w_i sigma_i
//     L_cf(x) = sum_i sigma_i w_i (W_{i-1} - F_{i-1} . f_i),   W, F accumulated in blend order (DESIGN.md reading)
// MODE 1 (FHGS_NDFD_FAR_TO_NEAR, "along the ray from far to near"): the partners of fragment i are the
// fragments BEHIND it, W_behind = W_tot - W_<=i, F_behind = F_tot - F_<=i.  The totals are only known at the end of the
// front-to-back walk, but the sum splits:
//     L_cf = sum_i sigma_i w_i (W_tot - F_tot . f_i) - sum_i sigma_i w_i (W_<=i - F_<=i . f_i)
//          = W_tot L_gt - F_tot . S - B,      S = sum_i sigma_i w_i f_i  (one more D-vector per pixel),
//                                             B = the blend-order recurrence with INCLUSIVE prefixes
// so the same single traversal serves (no fragment list, no second pass); the oracle's mode 1 walks the collected
// fragment list backwards instead.
//
// First CUDA path of this row (correctness first; not yet the warp-specialised form of render/fuse):
// one CTA of 256 threads per 16 x (16/LPP)-row pixel strip of a tile.  LPP lanes (4 for D <= 128, else 8) share one
// pixel and split the D channels in interleaved float4 groups; each lane keeps its slice of the pixel's
// ground-truth vector f_gt and of the running feature F in registers.  The CTA streams the tile's sorted range
// 256 instances at a time through the traverse.cuh staging (exact ellipse-vs-strip cull) and gathers the
// survivors' feature rows into shared memory with double-buffered cp.async; every warp then walks the survivors
// for its 32/LPP pixels: the normative q / cut-off / alpha / T arithmetic of C1-R, and -- only when one of its
// pixels has a weight -- the two D-length dot products (LPP-lane shuffle reduction) and the update of F.
#include <cuda_fp16.h>

#include "ws.cuh"   // packed fma.rn.f32x2 helpers (and traverse.cuh)

namespace {

struct NdfdArgs {
    TraverseArgs t;
    const void* feat;   // [n,D]
    const void* gt;     // [H,W,D]
    int D;
    float k_sig, lambda;
    float* out_lgt;
    float* out_lcf;
};

template <typename T>
__device__ __forceinline__ float4 ld4(const T* p);
template <>
__device__ __forceinline__ float4 ld4<float>(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
template <>
__device__ __forceinline__ float4 ld4<__half>(const __half* p) {
    const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
}

// LPP lanes share one pixel (LPP = 4 or 8): a warp covers 32/LPP pixels, the CTA (8 warps) a 16 x (16/LPP) strip

template <typename T>
__device__ __forceinline__ float4 lds4(const T* p);
template <>
__device__ __forceinline__ float4 lds4<float>(const float* p) { return *reinterpret_cast<const float4*>(p); }
template <>
__device__ __forceinline__ float4 lds4<__half>(const __half* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// survivors whose feature rows are staged together (one of two 32 KB shared-memory buffers)
template <int D, typename FT>
struct NdSub {
    static constexpr int ROW_BYTES = D * (int)sizeof(FT);
    static constexpr int SB = 32768 / ROW_BYTES > 64 ? 64 : (32768 / ROW_BYTES < 4 ? 4 : 32768 / ROW_BYTES);
};

// CPL = channels per lane = D / LPP
template <int LPP, int CPL, typename FT, typename GT, int MODE, int PRIM>
__global__ void __launch_bounds__(TR_THREADS, MODE ? (CPL <= 16 ? 2 : 1) : (CPL <= 16 ? 3 : (CPL <= 32 ? 2 : 1)))
    ndfd_strip_kernel(const NdfdArgs a) {
    __shared__ TileQueueT<PRIM> q;
    constexpr int PXW = 32 / LPP, ROWS = 8 * PXW / FHGS_TILE, STRIPS = FHGS_TILE / ROWS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x / STRIPS, strip = blockIdx.x % STRIPS;
    const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE + ROWS * strip;
    if (ty0 >= a.t.H) return;
    const int pxl = lane / LPP, cgl = lane % LPP;
    const int pi = warp * PXW + pxl;   // pixel of this lane group inside the strip, row-major
    const int px = tx0 + (pi & 15), py = ty0 + (pi >> 4);
    const bool inside = px < a.t.W && py < a.t.H;
    const float fx = (float)px, fy = (float)py;
    const float bx0 = (float)tx0, by0 = (float)ty0;
    const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + ROWS - 1, a.t.H - 1);
    const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
    const FT* feat = reinterpret_cast<const FT*>(a.feat);
    const GT* gt = reinterpret_cast<const GT*>(a.gt);
    // channel slice of this lane: float4 groups cgl, cgl + LPP, cgl + 2 LPP, ... (interleaved, so that the lanes of a
    // pixel read contiguous bytes per load: coalesced from global, conflict-free from shared memory)
    const int c_lo = cgl * 4;

    // channel pairs packed for fma.rn.f32x2 (two FMAs per issue slot)
    unsigned long long g[CPL / 2], F[CPL / 2], S[MODE ? CPL / 2 : 1];
#pragma unroll
    for (int j = 0; j < (MODE ? CPL / 2 : 1); ++j) S[j] = 0ull;
#pragma unroll
    for (int j = 0; j < CPL / 4; ++j) {
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (inside) v = ld4<GT>(gt + ((size_t)py * a.t.W + px) * a.D + c_lo + 4 * LPP * j);
        g[2 * j] = pack2(v.x, v.y); g[2 * j + 1] = pack2(v.z, v.w);
    }
#pragma unroll
    for (int j = 0; j < CPL / 2; ++j) F[j] = 0ull;
    float T = 1.f, Wc = 0.f, lgt = 0.f, lcf = 0.f;
    bool done = !inside;
    const float k2 = a.k_sig * 1.44269504088896340736f;   // exp(k z) = exp2(k2 z)

    // feature rows of the survivors are gathered into shared memory SB at a time with cp.async, double-buffered,
    // so that the (L2-latency) gather of the next sub-batch overlaps the walk over the current one
    constexpr int SB = NdSub<LPP * CPL, FT>::SB, ROW_BYTES = NdSub<LPP * CPL, FT>::ROW_BYTES;
    extern __shared__ __align__(16) unsigned char rows_raw[];
    auto stage_rows = [&](int sb, int added) {
        unsigned char* dst = rows_raw + (sb & 1) * SB * ROW_BYTES;
        const int nrows = min(SB, added - sb * SB);
        for (int c = tid; c < nrows * (ROW_BYTES / 16); c += TR_THREADS) {
            const int r = c / (ROW_BYTES / 16), o = (c % (ROW_BYTES / 16)) * 16;
            cp_async16(dst + r * ROW_BYTES + o,
                       reinterpret_cast<const unsigned char*>(feat + (size_t)q.id[sb * SB + r] * a.D) + o);
        }
        cp_async_commit();
    };
    uint32_t pos = range.x;
    while (pos < range.y) {
        const int added = stage_chunk(a.t, q, pos, range.y, 0, bx0, by0, bx1, by1);
        pos += TR_THREADS;
        const int nsb = (added + SB - 1) / SB;
        if (nsb > 0) stage_rows(0, added);
        for (int sb = 0; sb < nsb; ++sb) {
            if (sb + 1 < nsb) {
                stage_rows(sb + 1, added);
                cp_async_wait_group<1>();
            } else {
                cp_async_wait_group<0>();
            }
            __syncthreads();
            const FT* rows = reinterpret_cast<const FT*>(rows_raw + (sb & 1) * SB * ROW_BYTES) + c_lo;
            const int k_end = min(added, (sb + 1) * SB);
            // The T-independent part of the weight (normative q, cut-off, alpha = min(alpha_max, op G)) is evaluated for
            // LPP consecutive survivors at once, one per lane of the pixel group, and handed round by shuffles; only
            // w = alpha T, the T update and the stop test run per fragment.
            for (int k0 = sb * SB; k0 < k_end; k0 += LPP) {
              float a_c = 0.f;
              if (PRIM) {   // surfel: u^2 + v^2 from the ray transform (traverse.cuh eval_weight_surfel, same expressions)
                  if (k0 + cgl < k_end) {
                      const float4 m0 = q.m[0][PRIM ? k0 + cgl : 0], m1 = q.m[PRIM ? 1 : 0][PRIM ? k0 + cgl : 0], m2 = q.m[PRIM ? 2 : 0][PRIM ? k0 + cgl : 0];
                      const float p0 = __fmaf_rn(fx, m0.x, __fmaf_rn(fy, m0.y, m0.z));
                      const float p1 = __fmaf_rn(fx, m1.x, __fmaf_rn(fy, m1.y, m1.z));
                      const float p2 = __fmaf_rn(fx, m2.x, __fmaf_rn(fy, m2.y, m2.z));
                      const float num = __fmaf_rn(p0, p0, __fmul_rn(p1, p1)), den = __fmul_rn(p2, p2);
                      if (den > 0.f && num <= __fmul_rn(a.t.q_cutoff, den))
                          a_c = fminf(a.t.alpha_max, q.co[k0 + cgl].w * exp2f(-0.72134752044448170368f * __fdividef(num, den)));
                  }
              } else if (k0 + cgl < k_end) {
                  const float2 gxy = q.xy[k0 + cgl];
                  const float4 co = q.co[k0 + cgl];
                  const float dx = __fsub_rn(gxy.x, fx), dy = __fsub_rn(gxy.y, fy);
                  const float qv = __fmaf_rn(dx, __fmaf_rn(co.y, dy, __fmul_rn(co.x, dx)), __fmul_rn(__fmul_rn(co.z, dy), dy));
                  if (qv <= a.t.q_cutoff) a_c = fminf(a.t.alpha_max, co.w * exp2f(-0.72134752044448170368f * fmaxf(qv, 0.f)));
              }
#pragma unroll
              for (int jj = 0; jj < LPP; ++jj) {
                const int kk = k0 + jj;
                if (kk >= k_end) break;
                const float aj = __shfl_sync(TR_FULL, a_c, (lane & ~(LPP - 1)) + jj);
                float w = 0.f;
                if (!done && aj > 0.f) {
                    w = aj * T;
                    T = fmaf(-aj, T, T);
                    if (T < a.t.t_min) done = true;
                }
                if (!__any_sync(TR_FULL, w != 0.f)) continue;
                const FT* f = rows + (kk - sb * SB) * (CPL * LPP);
                unsigned long long ph[2] = {0ull, 0ull}, ff[2] = {0ull, 0ull};   // 2 packed chains each
                unsigned long long fv[CPL / 2];
#pragma unroll
                for (int j = 0; j < CPL / 4; ++j) {
                    const float4 v = lds4<FT>(f + 4 * LPP * j);
                    fv[2 * j] = pack2(v.x, v.y); fv[2 * j + 1] = pack2(v.z, v.w);
                }
                if (MODE) {   // inclusive prefixes: F_<=i, W_<=i
                    const unsigned long long w2 = pack2(w, w);
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) fma2_acc(F[j], w2, fv[j]);
                    Wc += w;
                }
#pragma unroll
                for (int j = 0; j < CPL / 2; ++j) {
                    fma2_acc(ph[j & 1], fv[j], g[j]);
                    fma2_acc(ff[j & 1], fv[j], F[j]);
                }
                const float2 p0 = unpack2(ph[0]), p1 = unpack2(ph[1]), q0 = unpack2(ff[0]), q1 = unpack2(ff[1]);
                float phi = (p0.x + p0.y) + (p1.x + p1.y), Ff = (q0.x + q0.y) + (q1.x + q1.y);
#pragma unroll
                for (int d = 1; d < LPP; d <<= 1) {
                    phi += __shfl_xor_sync(TR_FULL, phi, d);
                    Ff += __shfl_xor_sync(TR_FULL, Ff, d);
                }
                const float sigma = 1.0f / (1.0f + exp2f(k2 * (phi - a.lambda)));
                const float sw = sigma * w;        // w == 0 for pixels the Gaussian does not reach: nothing changes
                lgt += sw;
                lcf = fmaf(sw, Wc - Ff, lcf);
                if (MODE) {
                    const unsigned long long sw2 = pack2(sw, sw);
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) fma2_acc(S[j], sw2, fv[j]);
                } else {
                    Wc += w;
                    const unsigned long long w2 = pack2(w, w);
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) fma2_acc(F[j], w2, fv[j]);
                }
              }
            }
            __syncthreads();   // the buffer is refilled two sub-batches later; the ring at the next chunk
        }
        if (__syncthreads_and(done)) break;
    }
    if (MODE) {   // L_cf = W_tot L_gt - F_tot . S - B  (B = lcf so far)
        unsigned long long fs[2] = {0ull, 0ull};
#pragma unroll
        for (int j = 0; j < CPL / 2; ++j) fma2_acc(fs[j & 1], F[j], S[j]);
        const float2 s0 = unpack2(fs[0]), s1 = unpack2(fs[1]);
        float FS = (s0.x + s0.y) + (s1.x + s1.y);
#pragma unroll
        for (int d = 1; d < LPP; d <<= 1) FS += __shfl_xor_sync(TR_FULL, FS, d);
        lcf = fmaf(Wc, lgt, -FS) - lcf;
    }
    if (inside && cgl == 0) {
        const size_t o = (size_t)py * a.t.W + px;
        a.out_lgt[o] = lgt;
        a.out_lcf[o] = lcf;
    }
}

template <int LPP, int CPL, typename FT, typename GT, int MODE, int PRIM>
cudaError_t launch(const NdfdArgs& a, int tiles, cudaStream_t st) {
    constexpr int STRIPS = FHGS_TILE / (8 * (32 / LPP) / FHGS_TILE);
    const size_t smem = 2 * (size_t)NdSub<LPP * CPL, FT>::SB * NdSub<LPP * CPL, FT>::ROW_BYTES;
    cudaError_t e = cudaFuncSetAttribute(ndfd_strip_kernel<LPP, CPL, FT, GT, MODE, PRIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ndfd_strip_kernel<LPP, CPL, FT, GT, MODE, PRIM><<<tiles * STRIPS, TR_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename FT, typename GT, int MODE, int PRIM>
cudaError_t dispatch_d(const NdfdArgs& a, int tiles, cudaStream_t st) {
    switch (a.D) {
        case 32: return launch<4, 8, FT, GT, MODE, PRIM>(a, tiles, st);
        case 64: return launch<4, 16, FT, GT, MODE, PRIM>(a, tiles, st);
        // far to near (three running D-vectors per pixel): 8 lanes per pixel keep two CTAs per SM (Mid 9.12 -> 8.24 ms);
        // blend order is faster with 4 lanes per pixel (5.45 ms against 8.38)
        case 128: return MODE ? launch<8, 16, FT, GT, MODE, PRIM>(a, tiles, st) : launch<4, 32, FT, GT, MODE, PRIM>(a, tiles, st);
        case 256: return launch<8, 32, FT, GT, MODE, PRIM>(a, tiles, st);
        case 512: return launch<8, 64, FT, GT, MODE, PRIM>(a, tiles, st);
        default: return cudaErrorInvalidValue;
    }
}
template <typename FT, typename GT>
cudaError_t dispatch(const NdfdArgs& a, int tiles, int mode, cudaStream_t st) {
    return mode ? dispatch_d<FT, GT, 1, 0>(a, tiles, st) : dispatch_d<FT, GT, 0, 0>(a, tiles, st);
}

}  // namespace

extern "C" fhgs_status fhgs_ndfd_forward(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                                         const fhgs_params* prm, const fhgs_view_state* vs, const void* gt,
                                         int32_t gt_dtype, float k_sigmoid, float lambda, int32_t mode, float* out_lgt,
                                         float* out_lcf, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!g || !cam || !prm || !vs || !gt || !out_lgt || !out_lcf) FHGS_INVALID(ctx, "fhgs_ndfd_forward: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    const bool surfel = prm->primitive == FHGS_PRIM_SURFEL;
    if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    if (surfel && (g->feat_dtype != FHGS_F32 || gt_dtype != FHGS_F32))
        FHGS_INVALID(ctx, "fhgs_ndfd_forward: the surfel primitive is built for f32 features and map");
    if (!g->feat) FHGS_INVALID(ctx, "fhgs_ndfd_forward: g->feat is NULL");
    if ((g->feat_dtype != FHGS_F32 && g->feat_dtype != FHGS_F16) || (gt_dtype != FHGS_F32 && gt_dtype != FHGS_F16))
        FHGS_INVALID(ctx, "fhgs_ndfd_forward: unknown dtype");
    const int D = g->feat_dim;
    if (!(D == 32 || D == 64 || D == 128 || D == 256 || D == 512))
        FHGS_INVALID(ctx, "fhgs_ndfd_forward: feat_dim must be 32, 64, 128, 256 or 512");
    if (!aligned_to(g->feat, 16) || !aligned_to(gt, 16)) FHGS_INVALID(ctx, "fhgs_ndfd_forward: feat/gt must be 16-byte aligned");
    if (g->n != vs->n) FHGS_INVALID(ctx, "fhgs_ndfd_forward: g->n != vs->n");
    if (!finite_f(k_sigmoid) || !finite_f(lambda)) FHGS_INVALID(ctx, "fhgs_ndfd_forward: non-finite k / lambda");
    if (mode != FHGS_NDFD_BLEND_ORDER && mode != FHGS_NDFD_FAR_TO_NEAR) FHGS_INVALID(ctx, "fhgs_ndfd_forward: unknown mode");
    NdfdArgs a;
    a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
    a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
    a.t.xy = reinterpret_cast<const float2*>(vs->xy);
    a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
    a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
    a.t.ray_transform = surfel ? reinterpret_cast<const float4*>(vs->ray_transform) : nullptr;
    a.feat = g->feat; a.gt = gt; a.D = D; a.k_sig = k_sigmoid; a.lambda = lambda;
    a.out_lgt = out_lgt; a.out_lcf = out_lcf;
    const int tiles = tiles_x(cam->width) * tiles_y(cam->height);
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    const bool fh = g->feat_dtype == FHGS_F16, gh = gt_dtype == FHGS_F16;
    if (surfel) e = mode ? dispatch_d<float, float, 1, 1>(a, tiles, s) : dispatch_d<float, float, 0, 1>(a, tiles, s);
    else if (fh && gh) e = dispatch<__half, __half>(a, tiles, mode, s);
    else if (fh) e = dispatch<__half, float>(a, tiles, mode, s);
    else if (gh) e = dispatch<float, __half>(a, tiles, mode, s);
    else e = dispatch<float, float>(a, tiles, mode, s);
    FHGS_CUDA(ctx, e);
    return FHGS_OK;
}
