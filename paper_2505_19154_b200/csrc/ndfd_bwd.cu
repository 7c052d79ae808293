// ndfd_bwd.cu -- NDFD backward at the w level (fhgs_ndfd_backward): dL/d opacity of
//     L = sum_x ( lam1 L_gt(x) + lam2 L_cf(x) )            (losses of fhgs_ndfd_forward, Eq. 5-6)
// per pixel, over its fragments k = 1..N in blend order (appendix A.2):
//     g_k         = dL/dw_k = lam1 sigma_k + lam2 [ sigma_k (W_{k-1} - F_{k-1}.f_k) + A_k - B_k.f_k ]
//                   with the suffix sums A_k = sum_{i>k} sigma_i w_i,  B_k = sum_{i>k} sigma_i w_i f_i
//     dL/dalpha_k = T_k g_k - C_k / (1 - alpha_k),   C_k = sum_{j>k} g_j w_j
//     dL/dop_g   += dL/dalpha_k G_k    (0 where alpha is clamped at alpha_max)
//
// First CUDA path of this row: two FORWARD traversals with the strip kernel of ndfd.cu (feature rows staged in
// shared memory with double-buffered cp.async, 4 or 8 lanes per pixel; no reverse walk, no division-recovered
// transmittance).  Pass 1 stores the per-pixel totals A_0 (scalar), B_0 (D-vector) and C_0, where
//     C_0 = sum_j g_j w_j = lam1 L_gt + 2 lam2 L_cf
// because sum_j w_j (A_j - B_j.f_j) = sum_i sigma_i w_i (W_{i-1} - F_{i-1}.f_i) = L_cf (swap the double sum), so the
// forward recurrence suffices.  Pass 2 (MODE 3) turns the totals into running suffixes, evaluates g_k and adds
// dL/dalpha_k G_k into grad_opacity: reduced over the pixels of the warp first, then one atomic per (warp, Gaussian).
#include <cuda_fp16.h>

#include "ws.cuh"   // packed fma.rn.f32x2 helpers (and traverse.cuh)

namespace {

struct BwdArgs {
    TraverseArgs t;
    const void* feat;
    const void* gt;
    int D;
    float k_sig, lambda, lam1, lam2;
    float* A_tot;    // [H*W]
    float* C_tot;    // [H*W]
    float* B_tot;    // [H*W, D]
    float* grad_op;  // [n]
};

template <typename T>
__device__ __forceinline__ float4 ldg4(const T* p);
template <>
__device__ __forceinline__ float4 ldg4<float>(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
template <>
__device__ __forceinline__ float4 ldg4<__half>(const __half* p) {
    const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
}

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

// sum of the four partial sums of a dot product kept in two packed chains
__device__ __forceinline__ float hsum(const unsigned long long (&p)[2]) {
    const float2 a = unpack2(p[0]), b = unpack2(p[1]);
    return (a.x + a.y) + (b.x + b.y);
}

// survivors whose feature rows are staged together (one of two 32 KB shared-memory buffers), as in ndfd.cu
template <int D, typename FT>
struct BwdSub {
    static constexpr int ROW_BYTES = D * (int)sizeof(FT);
    static constexpr int SB = 32768 / ROW_BYTES > 64 ? 64 : (32768 / ROW_BYTES < 4 ? 4 : 32768 / ROW_BYTES);
};

// MODE 1: totals A_0, B_0, C_0.  MODE 3: gradient.
template <int MODE, int LPP, int CPL, typename FT, typename GT, int PRIM>
__global__ void __launch_bounds__(TR_THREADS, CPL <= 16 ? 3 : 2) ndfd_bwd_kernel(const BwdArgs a) {
    __shared__ TileQueueT<PRIM> q;
    constexpr int PXW = 32 / LPP, ROWS = 8 * PXW / FHGS_TILE, STRIPS = FHGS_TILE / ROWS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x / STRIPS, strip = blockIdx.x % STRIPS;
    const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE + ROWS * strip;
    if (ty0 >= a.t.H) return;
    const int pxl = lane / LPP, cgl = lane % LPP;
    const int pi = warp * PXW + pxl;
    const int px = tx0 + (pi & 15), py = ty0 + (pi >> 4);
    const bool inside = px < a.t.W && py < a.t.H;
    const float fx = (float)px, fy = (float)py;
    const float bx0 = (float)tx0, by0 = (float)ty0;
    const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + ROWS - 1, a.t.H - 1);
    const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
    const FT* feat = reinterpret_cast<const FT*>(a.feat);
    const GT* gt = reinterpret_cast<const GT*>(a.gt);
    const int c_lo = cgl * 4;   // interleaved float4 groups cgl, cgl + LPP, ...
    const size_t pix = (size_t)py * a.t.W + px;

    // f_gt slice; prefix sum w f; MODE 1: running sum sigma w f, else suffix B_k -- channel pairs packed for fma.rn.f32x2
    unsigned long long g[CPL / 2], F[CPL / 2], Bs[CPL / 2];
#pragma unroll
    for (int j = 0; j < CPL / 4; ++j) {
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f), b = make_float4(0.f, 0.f, 0.f, 0.f);
        if (inside) {
            v = ldg4<GT>(gt + pix * a.D + c_lo + 4 * LPP * j);
            if (MODE != 1) b = *reinterpret_cast<const float4*>(a.B_tot + pix * a.D + c_lo + 4 * LPP * j);
        }
        g[2 * j] = pack2(v.x, v.y); g[2 * j + 1] = pack2(v.z, v.w);
        Bs[2 * j] = pack2(b.x, b.y); Bs[2 * j + 1] = pack2(b.z, b.w);
        F[2 * j] = F[2 * j + 1] = 0ull;
    }
    float T = 1.f, Wc = 0.f;
    float As = (MODE != 1 && inside) ? a.A_tot[pix] : 0.f;      // MODE 1: running sum; else suffix A_k
    float Cs = (MODE == 3 && inside) ? a.C_tot[pix] : 0.f;      // MODE 1: running sum of C_0; MODE 3: suffix C_k
    bool done = !inside;
    const float k2 = a.k_sig * 1.44269504088896340736f;

    constexpr int SB = BwdSub<LPP * CPL, FT>::SB, ROW_BYTES = BwdSub<LPP * CPL, FT>::ROW_BYTES;
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
            // alpha and G_eff (T-independent) are evaluated for LPP consecutive survivors at once, one per lane of the
            // pixel group, and handed round by shuffles (as in ndfd.cu)
            for (int k0 = sb * SB; k0 < k_end; k0 += LPP) {
              float a_c = 0.f, g_c = 0.f;
              if (PRIM) {   // surfel: G = exp(-(u^2+v^2)/2) from the ray transform (traverse.cuh eval_weight_surfel)
                  if (k0 + cgl < k_end) {
                      const float4 m0 = q.m[0][PRIM ? k0 + cgl : 0], m1 = q.m[PRIM ? 1 : 0][PRIM ? k0 + cgl : 0], m2 = q.m[PRIM ? 2 : 0][PRIM ? k0 + cgl : 0];
                      const float p0 = __fmaf_rn(fx, m0.x, __fmaf_rn(fy, m0.y, m0.z));
                      const float p1 = __fmaf_rn(fx, m1.x, __fmaf_rn(fy, m1.y, m1.z));
                      const float p2 = __fmaf_rn(fx, m2.x, __fmaf_rn(fy, m2.y, m2.z));
                      const float num = __fmaf_rn(p0, p0, __fmul_rn(p1, p1)), den = __fmul_rn(p2, p2);
                      if (den > 0.f && num <= __fmul_rn(a.t.q_cutoff, den)) {
                          const float G = exp2f(-0.72134752044448170368f * __fdividef(num, den));
                          const float a_raw = q.co[k0 + cgl].w * G;
                          a_c = fminf(a.t.alpha_max, a_raw);
                          g_c = a_raw < a.t.alpha_max ? G : 0.f;
                      }
                  }
              } else if (k0 + cgl < k_end) {
                  const float2 gxy = q.xy[k0 + cgl];
                  const float4 co = q.co[k0 + cgl];
                  const float dx = __fsub_rn(gxy.x, fx), dy = __fsub_rn(gxy.y, fy);
                  const float qv = __fmaf_rn(dx, __fmaf_rn(co.y, dy, __fmul_rn(co.x, dx)), __fmul_rn(__fmul_rn(co.z, dy), dy));
                  if (qv <= a.t.q_cutoff) {
                      const float G = exp2f(-0.72134752044448170368f * fmaxf(qv, 0.f));
                      const float a_raw = co.w * G;
                      a_c = fminf(a.t.alpha_max, a_raw);
                      g_c = a_raw < a.t.alpha_max ? G : 0.f;
                  }
              }
#pragma unroll
              for (int jj = 0; jj < LPP; ++jj) {
                const int kk = k0 + jj;
                if (kk >= k_end) break;
                const float alpha = __shfl_sync(TR_FULL, a_c, (lane & ~(LPP - 1)) + jj);
                const float Ge = __shfl_sync(TR_FULL, g_c, (lane & ~(LPP - 1)) + jj);
                const bool hit = !done && alpha > 0.f;
                const float Tb = T;
                if (hit) {
                    T = fmaf(-alpha, T, T);
                    if (T < a.t.t_min) done = true;
                }
                if (!__any_sync(TR_FULL, hit)) continue;
                const float w = hit ? alpha * Tb : 0.f;
                const uint32_t id = q.id[kk];
                const FT* f = rows + (kk - sb * SB) * (CPL * LPP);
                unsigned long long fv[CPL / 2];
#pragma unroll
                for (int j = 0; j < CPL / 4; ++j) {
                    const float4 v = lds4<FT>(f + 4 * LPP * j);
                    fv[2 * j] = pack2(v.x, v.y); fv[2 * j + 1] = pack2(v.z, v.w);
                }
                unsigned long long ph[2] = {0ull, 0ull};   // 2 packed chains per dot product
#pragma unroll
                for (int j = 0; j < CPL / 2; ++j) fma2_acc(ph[j & 1], fv[j], g[j]);
                float phi = hsum(ph);
#pragma unroll
                for (int d = 1; d < LPP; d <<= 1) phi += __shfl_xor_sync(TR_FULL, phi, d);
                const float sigma = 1.0f / (1.0f + exp2f(k2 * (phi - a.lambda)));
                const float sw = sigma * w;
                if (MODE == 1) {
                    // totals A_0, B_0 and the forward losses (prefix recurrence), from which C_0 follows (see the header)
                    unsigned long long fa1[2] = {0ull, 0ull};
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) fma2_acc(fa1[j & 1], fv[j], F[j]);
                    float Ff1 = hsum(fa1);
#pragma unroll
                    for (int d = 1; d < LPP; d <<= 1) Ff1 += __shfl_xor_sync(TR_FULL, Ff1, d);
                    As += sw;
                    Cs += a.lam1 * sw + 2.0f * a.lam2 * sw * (Wc - Ff1);
                    Wc += w;
                    const unsigned long long sw2 = pack2(sw, sw), w2 = pack2(w, w);
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) {
                        fma2_acc(Bs[j], sw2, fv[j]);
                        fma2_acc(F[j], w2, fv[j]);
                    }
                    continue;
                }
                // suffixes exclude k
                As -= sw;
                unsigned long long fa[2] = {0ull, 0ull}, ba[2] = {0ull, 0ull};
                const unsigned long long nsw2 = pack2(-sw, -sw);
#pragma unroll
                for (int j = 0; j < CPL / 2; ++j) {
                    fma2_acc(Bs[j], nsw2, fv[j]);
                    fma2_acc(fa[j & 1], fv[j], F[j]);
                    fma2_acc(ba[j & 1], fv[j], Bs[j]);
                }
                float Ff = hsum(fa), Bf = hsum(ba);
#pragma unroll
                for (int d = 1; d < LPP; d <<= 1) {
                    Ff += __shfl_xor_sync(TR_FULL, Ff, d);
                    Bf += __shfl_xor_sync(TR_FULL, Bf, d);
                }
                const float gk = a.lam1 * sigma + a.lam2 * (sigma * (Wc - Ff) + (As - Bf));
                Wc += w;
                {
                    const unsigned long long w2 = pack2(w, w);
#pragma unroll
                    for (int j = 0; j < CPL / 2; ++j) fma2_acc(F[j], w2, fv[j]);
                }
                {
                    Cs = fmaf(-gk, w, Cs);   // suffix excludes k
                    float contrib = hit ? (Tb * gk - Cs / (1.0f - alpha)) * Ge : 0.f;
                    if (cgl != 0) contrib = 0.f;   // every lane of the pixel group holds the same value
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) contrib += __shfl_xor_sync(TR_FULL, contrib, d);
                    if (lane == 0 && contrib != 0.f) atomicAdd(a.grad_op + id, contrib);
                }
              }
            }
            __syncthreads();
        }
        if (__syncthreads_and(done)) break;
    }
    if (inside) {
        if (MODE == 1) {
            if (cgl == 0) { a.A_tot[pix] = As; a.C_tot[pix] = Cs; }
#pragma unroll
            for (int j = 0; j < CPL / 4; ++j) {
                const float2 b0 = unpack2(Bs[2 * j]), b1 = unpack2(Bs[2 * j + 1]);
                *reinterpret_cast<float4*>(a.B_tot + pix * a.D + c_lo + 4 * LPP * j) = make_float4(b0.x, b0.y, b1.x, b1.y);
            }
        }
    }
}

template <int MODE, int LPP, int CPL, typename FT, typename GT, int PRIM>
cudaError_t launch1(const BwdArgs& a, int tiles, cudaStream_t st) {
    constexpr int STRIPS = FHGS_TILE / (8 * (32 / LPP) / FHGS_TILE);
    const size_t smem = 2 * (size_t)BwdSub<LPP * CPL, FT>::SB * BwdSub<LPP * CPL, FT>::ROW_BYTES;
    cudaError_t e = cudaFuncSetAttribute(ndfd_bwd_kernel<MODE, LPP, CPL, FT, GT, PRIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ndfd_bwd_kernel<MODE, LPP, CPL, FT, GT, PRIM><<<tiles * STRIPS, TR_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <int LPP, int CPL, typename FT, typename GT, int PRIM>
cudaError_t launch3(const BwdArgs& a, int tiles, cudaStream_t st) {
    cudaError_t e;
    if ((e = launch1<1, LPP, CPL, FT, GT, PRIM>(a, tiles, st)) != cudaSuccess) return e;
    return launch1<3, LPP, CPL, FT, GT, PRIM>(a, tiles, st);
}

template <typename FT, typename GT, int PRIM = 0>
cudaError_t dispatch(const BwdArgs& a, int tiles, cudaStream_t st) {
    switch (a.D) {
        case 32: return launch3<4, 8, FT, GT, PRIM>(a, tiles, st);
        case 64: return launch3<4, 16, FT, GT, PRIM>(a, tiles, st);
        case 128: return launch3<4, 32, FT, GT, PRIM>(a, tiles, st);
        case 256: return launch3<8, 32, FT, GT, PRIM>(a, tiles, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

extern "C" size_t fhgs_ndfd_backward_work_bytes(int32_t width, int32_t height, int32_t feat_dim) {
    if (width <= 0 || height <= 0 || feat_dim <= 0) return 0;
    const size_t px = (size_t)width * height;
    return (px * 2 + px * (size_t)feat_dim) * sizeof(float) + 512;
}

extern "C" fhgs_status fhgs_ndfd_backward(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                                          const fhgs_params* prm, const fhgs_view_state* vs, const void* gt,
                                          int32_t gt_dtype, float k_sigmoid, float lambda, float lam1, float lam2,
                                          float* grad_opacity, void* work, size_t work_bytes, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!g || !cam || !prm || !vs || !gt || !grad_opacity || !work) FHGS_INVALID(ctx, "fhgs_ndfd_backward: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    const bool surfel = prm->primitive == FHGS_PRIM_SURFEL;
    if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    if (surfel && (g->feat_dtype != FHGS_F32 || gt_dtype != FHGS_F32))
        FHGS_INVALID(ctx, "fhgs_ndfd_backward: the surfel primitive is built for f32 features and map");
    if (!g->feat) FHGS_INVALID(ctx, "fhgs_ndfd_backward: g->feat is NULL");
    if ((g->feat_dtype != FHGS_F32 && g->feat_dtype != FHGS_F16) || (gt_dtype != FHGS_F32 && gt_dtype != FHGS_F16))
        FHGS_INVALID(ctx, "fhgs_ndfd_backward: unknown dtype");
    const int D = g->feat_dim;
    if (!(D == 32 || D == 64 || D == 128 || D == 256)) FHGS_INVALID(ctx, "fhgs_ndfd_backward: feat_dim must be 32, 64, 128 or 256");
    if (!aligned_to(g->feat, 16) || !aligned_to(gt, 16) || !aligned_to(work, 256))
        FHGS_INVALID(ctx, "fhgs_ndfd_backward: feat/gt must be 16-byte, work 256-byte aligned");
    if (work_bytes < fhgs_ndfd_backward_work_bytes(cam->width, cam->height, D)) FHGS_INVALID(ctx, "fhgs_ndfd_backward: work too small");
    if (g->n != vs->n) FHGS_INVALID(ctx, "fhgs_ndfd_backward: g->n != vs->n");
    if (!finite_f(k_sigmoid) || !finite_f(lambda) || !finite_f(lam1) || !finite_f(lam2)) FHGS_INVALID(ctx, "fhgs_ndfd_backward: non-finite scalar");
    BwdArgs a;
    a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
    a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
    a.t.xy = reinterpret_cast<const float2*>(vs->xy);
    a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
    a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
    a.t.ray_transform = surfel ? reinterpret_cast<const float4*>(vs->ray_transform) : nullptr;
    a.feat = g->feat; a.gt = gt; a.D = D; a.k_sig = k_sigmoid; a.lambda = lambda; a.lam1 = lam1; a.lam2 = lam2;
    const size_t px = (size_t)cam->width * cam->height;
    a.A_tot = reinterpret_cast<float*>(work);
    a.C_tot = a.A_tot + px;
    a.B_tot = reinterpret_cast<float*>((char*)work + ((px * 2 * sizeof(float) + 255) / 256) * 256);
    a.grad_op = grad_opacity;
    const int tiles = tiles_x(cam->width) * tiles_y(cam->height);
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    const bool fh = g->feat_dtype == FHGS_F16, gh = gt_dtype == FHGS_F16;
    if (surfel) e = dispatch<float, float, 1>(a, tiles, s);
    else if (fh && gh) e = dispatch<__half, __half>(a, tiles, s);
    else if (fh) e = dispatch<__half, float>(a, tiles, s);
    else if (gh) e = dispatch<float, __half>(a, tiles, s);
    else e = dispatch<float, float>(a, tiles, s);
    FHGS_CUDA(ctx, e);
    return FHGS_OK;
}
