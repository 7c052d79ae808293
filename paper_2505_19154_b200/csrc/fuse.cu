// fuse.cu -- step F (fhgs_fuse_features): weight-aggregated feature fusion.
//     num[i,:] += sum_x w_i(x) gt[x,:],   den[i] += sum_x w_i(x),   w_i(x) = alpha_i T_i
// (PAPER.md:95 for the weight; the aggregation is north_star's.)
//
// Same per-tile traversal as step R (traverse.cuh).  Per tile the work is the transposed product
//     num[K, D] += W[256 px, K]^T * G[256 px, D]
// TILED variant (D multiple of 64): the GT tile G (256 px x DC channels, fp32) is staged in shared
// memory once per channel pass; per sub-batch of KB staged instances phase B parks the weights
// W[kk][slot]; phase C is a register-tiled product with thread = 4 instances x 8 (DC=128) or 4
// (DC=64) channels reducing over the 256 pixels, so every (tile, Gaussian) segment is reduced
// completely inside the CTA -- across all 8 warps -- before it touches global memory, and leaves
// as D/4 vector reductions `red.global.add.v4.f32` plus one scalar for den (SURVEY 7.2 item 2:
// 6.6x fewer atomics than one per warp segment).
// PIXEL variant (small D): thread = pixel holds its G row in registers; each (warp, Gaussian)
// segment is reduced with shuffles and leaves as one atomic per channel from lane 0.
// The finalise kernel divides (one warp per Gaussian row) and optionally L2-normalises.
#include "traverse.cuh"

namespace {

struct FuseArgs {
    TraverseArgs t;
    const void* gt;   // [H,W,D]
    int D;
    float* num;
    float* den;
};

constexpr int F_KB = 64;

__device__ __forceinline__ void red_add_v4(float* addr, float4 v) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
                 : "memory");
}
__device__ __forceinline__ void red_add(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

template <typename GT>
__device__ __forceinline__ float4 load_gt4(const GT* p);
template <>
__device__ __forceinline__ float4 load_gt4<float>(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
template <>
__device__ __forceinline__ float4 load_gt4<__half>(const __half* p) {
    const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
}

template <int DC>
struct FuseTiledSmem {
    TileQueue q;
    __align__(16) float W[F_KB * TR_THREADS];   // W[kk][slot]
    __align__(16) float G[TR_THREADS * DC];     // G[slot][channel]
    float den[F_KB];
};

// phase C for RT rows per thread (rows kg + 16 i)
template <int DC, int RT>
__device__ __forceinline__ void fuse_gemm(const float* __restrict__ W, const float* __restrict__ G, const float* den_s,
                                          const uint32_t* q_id, int q_head, int nb, int kg, int cg, const FuseArgs& a,
                                          int c0) {
    constexpr int NC = DC / 64;   // float4 channel groups per thread (2 for DC=128, 1 for DC=64)
    float acc[RT][NC * 4];
#pragma unroll
    for (int i = 0; i < RT; ++i)
#pragma unroll
        for (int j = 0; j < NC * 4; ++j) acc[i][j] = 0.f;
#pragma unroll 2
    for (int s = 0; s < TR_THREADS; s += 4) {
        float4 w[RT];
#pragma unroll
        for (int i = 0; i < RT; ++i) w[i] = *reinterpret_cast<const float4*>(&W[(kg + 16 * i) * TR_THREADS + s]);
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            float g[NC * 4];
#pragma unroll
            for (int j = 0; j < NC; ++j) {
                const float4 v = *reinterpret_cast<const float4*>(&G[(s + p) * DC + j * 64 + cg * 4]);
                g[4 * j] = v.x; g[4 * j + 1] = v.y; g[4 * j + 2] = v.z; g[4 * j + 3] = v.w;
            }
#pragma unroll
            for (int i = 0; i < RT; ++i) {
                const float wp = p == 0 ? w[i].x : p == 1 ? w[i].y : p == 2 ? w[i].z : w[i].w;
#pragma unroll
                for (int j = 0; j < NC * 4; ++j) acc[i][j] = fmaf(wp, g[j], acc[i][j]);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < RT; ++i) {
        const int kk = kg + 16 * i;
        if (kk < nb && den_s[kk] != 0.f) {
            const uint32_t id = q_id[(q_head + kk) & (TR_QCAP - 1)];
            float* dst = a.num + (size_t)id * a.D + c0;
#pragma unroll
            for (int j = 0; j < NC; ++j)
                red_add_v4(dst + j * 64 + cg * 4, make_float4(acc[i][4 * j], acc[i][4 * j + 1], acc[i][4 * j + 2], acc[i][4 * j + 3]));
            if (c0 == 0 && cg == 0) red_add(a.den + id, den_s[kk]);
        }
    }
}

template <int DC, typename GT>
__global__ void __launch_bounds__(TR_THREADS, 1) fuse_tiled_kernel(const FuseArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FuseTiledSmem<DC>& sm = *reinterpret_cast<FuseTiledSmem<DC>*>(smem_raw);

    const int tid = threadIdx.x;
    const int tile = blockIdx.x;
    const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE;
    int sx, sy;
    slot_to_xy(tid, sx, sy);
    const int px = tx0 + sx, py = ty0 + sy;
    const bool inside = px < a.t.W && py < a.t.H;
    const float fx = (float)px, fy = (float)py;
    const float bx0 = (float)tx0, by0 = (float)ty0;
    const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + FHGS_TILE - 1, a.t.H - 1);
    const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
    if (range.x >= range.y) return;
    const GT* gt = reinterpret_cast<const GT*>(a.gt);
    const int kg = tid >> 4, cg = tid & 15;

    for (int c0 = 0; c0 < a.D; c0 += DC) {
        // stage the GT tile: G[slot][0..DC) <- gt[py,px,c0..c0+DC); out-of-image slots get zeros
        __syncthreads();
        for (int c = tid; c < TR_THREADS * (DC / 4); c += TR_THREADS) {
            const int slot = c / (DC / 4), ch = (c % (DC / 4)) * 4;
            int qx, qy;
            slot_to_xy(slot, qx, qy);
            const int gx = tx0 + qx, gy = ty0 + qy;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (gx < a.t.W && gy < a.t.H) v = load_gt4<GT>(gt + ((size_t)gy * a.t.W + gx) * a.D + c0 + ch);
            *reinterpret_cast<float4*>(&sm.G[slot * DC + ch]) = v;
        }
        float T = 1.f;
        uint32_t n = 0;
        bool done = !inside;
        uint32_t pos = range.x;
        int q_head = 0, q_count = 0;
        while (true) {
            while (q_count < F_KB && pos < range.y) {
                q_count += stage_chunk(a.t, sm.q, pos, range.y, q_head + q_count, bx0, by0, bx1, by1);
                pos += TR_THREADS;
            }
            const int nb = min(F_KB, q_count);
            if (nb == 0) break;
            __syncthreads();   // G staged; previous phase C finished with W/den
            // phase B
            for (int kk = 0; kk < nb; ++kk) {
                const int s = (q_head + kk) & (TR_QCAP - 1);
                sm.W[kk * TR_THREADS + tid] = eval_weight(sm.q.xy[s], sm.q.co[s], fx, fy, a.t, T, done, n);
            }
            __syncthreads();
            // row sums (den): thread t sums quarter t%4 of row t/4
            {
                const int row = tid >> 2, part = tid & 3;
                float ssum = 0.f;
                if (row < nb) {
#pragma unroll
                    for (int k = 0; k < 16; ++k) {
                        const float4 v = *reinterpret_cast<const float4*>(&sm.W[row * TR_THREADS + part * 64 + k * 4]);
                        ssum += (v.x + v.y) + (v.z + v.w);
                    }
                }
                ssum += __shfl_xor_sync(TR_FULL, ssum, 1);
                ssum += __shfl_xor_sync(TR_FULL, ssum, 2);
                if (part == 0 && row < F_KB) sm.den[row] = ssum;
            }
            __syncthreads();
            // phase C
            const int rt = (nb + 15) >> 4;
            if (rt == 1) fuse_gemm<DC, 1>(sm.W, sm.G, sm.den, sm.q.id, q_head, nb, kg, cg, a, c0);
            else if (rt == 2) fuse_gemm<DC, 2>(sm.W, sm.G, sm.den, sm.q.id, q_head, nb, kg, cg, a, c0);
            else if (rt == 3) fuse_gemm<DC, 3>(sm.W, sm.G, sm.den, sm.q.id, q_head, nb, kg, cg, a, c0);
            else fuse_gemm<DC, 4>(sm.W, sm.G, sm.den, sm.q.id, q_head, nb, kg, cg, a, c0);
            q_head = (q_head + nb) & (TR_QCAP - 1);
            q_count -= nb;
            if (__syncthreads_and(done)) break;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// PIXEL variant: CH channels per pass held by the pixel's thread; warp-segment reduction
// ---------------------------------------------------------------------------------------------
struct FusePixelSmem {
    TileQueue q;
};

template <int CH, typename GT>
__global__ void __launch_bounds__(TR_THREADS) fuse_pixel_kernel(const FuseArgs a) {
    __shared__ FusePixelSmem sm;
    const int tid = threadIdx.x, lane = tid & 31;
    const int tile = blockIdx.x;
    const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE;
    int sx, sy;
    slot_to_xy(tid, sx, sy);
    const int px = tx0 + sx, py = ty0 + sy;
    const bool inside = px < a.t.W && py < a.t.H;
    const float fx = (float)px, fy = (float)py;
    const float bx0 = (float)tx0, by0 = (float)ty0;
    const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + FHGS_TILE - 1, a.t.H - 1);
    const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
    if (range.x >= range.y) return;
    const GT* gt = reinterpret_cast<const GT*>(a.gt);

    for (int c0 = 0; c0 < a.D; c0 += CH) {
        float g[CH];
#pragma unroll
        for (int j = 0; j < CH / 4; ++j) {
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (inside) v = load_gt4<GT>(gt + ((size_t)py * a.t.W + px) * a.D + c0 + 4 * j);
            g[4 * j] = v.x; g[4 * j + 1] = v.y; g[4 * j + 2] = v.z; g[4 * j + 3] = v.w;
        }
        float T = 1.f;
        uint32_t n = 0;
        bool done = !inside;
        uint32_t pos = range.x;
        int q_head = 0, q_count = 0;
        __syncthreads();
        while (true) {
            while (q_count < F_KB && pos < range.y) {
                q_count += stage_chunk(a.t, sm.q, pos, range.y, q_head + q_count, bx0, by0, bx1, by1);
                pos += TR_THREADS;
            }
            const int nb = q_count;
            if (nb == 0) break;
            for (int kk = 0; kk < nb; ++kk) {
                const int s = (q_head + kk) & (TR_QCAP - 1);
                const float w = eval_weight(sm.q.xy[s], sm.q.co[s], fx, fy, a.t, T, done, n);
                if (!__any_sync(TR_FULL, w != 0.f)) continue;
                const uint32_t id = sm.q.id[s];
                float v[CH + 1];
#pragma unroll
                for (int j = 0; j < CH; ++j) v[j] = w * g[j];
                v[CH] = w;
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1)
#pragma unroll
                    for (int j = 0; j < CH + 1; ++j) v[j] += __shfl_xor_sync(TR_FULL, v[j], d);
                if (lane == 0) {
                    float* dst = a.num + (size_t)id * a.D + c0;
#pragma unroll
                    for (int j = 0; j < CH / 4; ++j) red_add_v4(dst + 4 * j, make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]));
                    if (c0 == 0) red_add(a.den + id, v[CH]);
                }
            }
            q_head = (q_head + nb) & (TR_QCAP - 1);
            q_count = 0;
            if (__syncthreads_and(done)) break;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// finalise: one warp per Gaussian row
// ---------------------------------------------------------------------------------------------
template <typename OT>
__global__ void __launch_bounds__(256) finalize_kernel(int n, int D, const float* num, const float* den, float den_eps,
                                                       int l2norm, OT* out) {
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= n) return;
    const float d = __ldg(den + row);
    if (!(d > den_eps)) return;
    const float4* src = reinterpret_cast<const float4*>(num + (size_t)row * D);
    const int n4 = D >> 2;
    float scale = 1.0f;
    if (l2norm) {
        float ss = 0.f;
        for (int j = lane; j < n4; j += 32) {
            const float4 v = __ldg(src + j);
            const float x = v.x / d, y = v.y / d, z = v.z / d, w = v.w / d;
            ss += x * x + y * y + z * z + w * w;
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) ss += __shfl_xor_sync(TR_FULL, ss, o);
        if (ss > 0.f) scale = 1.0f / sqrtf(ss);
    }
    for (int j = lane; j < n4; j += 32) {
        const float4 v = __ldg(src + j);
        const float x = v.x / d * scale, y = v.y / d * scale, z = v.z / d * scale, w = v.w / d * scale;
        if (sizeof(OT) == 4) {
            reinterpret_cast<float4*>(out)[(size_t)row * n4 + j] = make_float4(x, y, z, w);
        } else {
            const __half2 a = __floats2half2_rn(x, y), b = __floats2half2_rn(z, w);
            uint2 r;
            r.x = *reinterpret_cast<const uint32_t*>(&a);
            r.y = *reinterpret_cast<const uint32_t*>(&b);
            reinterpret_cast<uint2*>(out)[(size_t)row * n4 + j] = r;
        }
    }
}

template <typename K>
cudaError_t launch(K kernel, size_t smem, int grid, cudaStream_t st, const FuseArgs& a) {
    if (smem) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kernel<<<grid, TR_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename GT>
cudaError_t dispatch(const FuseArgs& a, int grid, cudaStream_t st) {
    if (a.D % 128 == 0) return launch(fuse_tiled_kernel<128, GT>, sizeof(FuseTiledSmem<128>), grid, st, a);
    if (a.D % 64 == 0) return launch(fuse_tiled_kernel<64, GT>, sizeof(FuseTiledSmem<64>), grid, st, a);
    if (a.D % 16 == 0) return launch(fuse_pixel_kernel<16, GT>, 0, grid, st, a);
    if (a.D % 8 == 0) return launch(fuse_pixel_kernel<8, GT>, 0, grid, st, a);
    return launch(fuse_pixel_kernel<4, GT>, 0, grid, st, a);
}

}  // namespace

extern "C" fhgs_status fhgs_fuse_features(fhgs_ctx* ctx, const fhgs_camera* cam, const fhgs_params* prm,
                                          const fhgs_view_state* vs, const void* gt, int32_t feat_dim,
                                          int32_t gt_dtype, float* num, float* den, void* out_feat,
                                          int32_t out_dtype, uint32_t flags, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!prm || !vs || !num || !den) FHGS_INVALID(ctx, "fhgs_fuse_features: NULL argument");
    if (flags & ~(uint32_t)(FHGS_FUSE_ZERO | FHGS_FUSE_FINALIZE | FHGS_FUSE_L2NORM | FHGS_FUSE_FINALIZE_ONLY | FHGS_FUSE_ZERO_ONLY))
        FHGS_INVALID(ctx, "fhgs_fuse_features: unknown flag");
    const bool zero_only = (flags & FHGS_FUSE_ZERO_ONLY) != 0;
    if (zero_only && (flags & ~(uint32_t)FHGS_FUSE_ZERO_ONLY)) FHGS_INVALID(ctx, "fhgs_fuse_features: ZERO_ONLY excludes other flags");
    const bool accumulate = !(flags & (FHGS_FUSE_FINALIZE_ONLY | FHGS_FUSE_ZERO_ONLY));
    const bool finalize = (flags & (FHGS_FUSE_FINALIZE | FHGS_FUSE_FINALIZE_ONLY)) != 0;
    fhgs_status st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if (gt_dtype != FHGS_F32 && gt_dtype != FHGS_F16) FHGS_INVALID(ctx, "fhgs_fuse_features: unknown gt_dtype");
    if (out_dtype != FHGS_F32 && out_dtype != FHGS_F16) FHGS_INVALID(ctx, "fhgs_fuse_features: unknown out_dtype");
    const int mult = (accumulate && gt_dtype == FHGS_F16) ? 8 : 4;
    if (feat_dim <= 0 || feat_dim % mult) FHGS_INVALID(ctx, "fhgs_fuse_features: feat_dim must be a positive multiple of 4 (f32) / 8 (f16)");
    if (!aligned_to(num, 16) || !aligned_to(den, 4)) FHGS_INVALID(ctx, "fhgs_fuse_features: num must be 16-byte aligned");
    if (vs->n < 0) FHGS_INVALID(ctx, "fhgs_fuse_features: vs->n < 0");
    if (accumulate) {
        if (!cam || !gt) FHGS_INVALID(ctx, "fhgs_fuse_features: cam and gt are required unless FINALIZE_ONLY");
        if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
        if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
        if (!aligned_to(gt, 16)) FHGS_INVALID(ctx, "fhgs_fuse_features: gt must be 16-byte aligned");
    }
    if (finalize) {
        if (!out_feat) FHGS_INVALID(ctx, "fhgs_fuse_features: FINALIZE needs out_feat");
        if (!aligned_to(out_feat, 16)) FHGS_INVALID(ctx, "fhgs_fuse_features: out_feat must be 16-byte aligned");
    }
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = (size_t)vs->n;
    if (flags & (FHGS_FUSE_ZERO | FHGS_FUSE_ZERO_ONLY)) {
        FHGS_CUDA(ctx, cudaMemsetAsync(num, 0, n * feat_dim * sizeof(float), s));
        FHGS_CUDA(ctx, cudaMemsetAsync(den, 0, n * sizeof(float), s));
    }
    if (accumulate && n > 0) {
        FuseArgs a;
        a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
        a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
        a.t.xy = reinterpret_cast<const float2*>(vs->xy);
        a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
        a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
        a.gt = gt; a.D = feat_dim; a.num = num; a.den = den;
        const int grid = tiles_x(cam->width) * tiles_y(cam->height);
        cudaError_t e = gt_dtype == FHGS_F16 ? dispatch<__half>(a, grid, s) : dispatch<float>(a, grid, s);
        FHGS_CUDA(ctx, e);
    }
    if (finalize && n > 0) {
        const int grid = (int)((n + 7) / 8);
        const int l2 = (flags & FHGS_FUSE_L2NORM) ? 1 : 0;
        if (out_dtype == FHGS_F16)
            finalize_kernel<__half><<<grid, 256, 0, s>>>((int)n, feat_dim, num, den, prm->den_eps, l2, (__half*)out_feat);
        else
            finalize_kernel<float><<<grid, 256, 0, s>>>((int)n, feat_dim, num, den, prm->den_eps, l2, (float*)out_feat);
        FHGS_LAUNCH_CHECK(ctx);
    }
    return FHGS_OK;
}
