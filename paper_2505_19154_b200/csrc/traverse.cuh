// traverse.cuh -- the per-tile front-to-back traversal shared by render.cu and fuse.cu
// ("traverse the corresponding range r in front-to-back order"; PAPER.md:90-95
// w_i = alpha_i T_i).  Device code only; not used by oracle/.
//
// One CTA of 256 threads owns one 16x16 tile; thread t owns pixel slot t.  Slots are laid out so
// that a warp covers a compact 8x4 pixel block (fewer (warp, Gaussian) pairs with any weight):
//     slot s: warp = s/32, lane = s%32 -> x = (warp&1)*8 + (lane&7), y = (warp>>1)*4 + (lane>>3).
//
// Stage A (stage_chunk): 256 instances of the tile's sorted range are examined by one thread each:
// the projected Gaussian is fetched and tested against the tile's pixel-centre box with an exact
// convex minimisation of q over the box (centre inside -> 0, else the minimum over the four
// edges).  Instances whose minimum exceeds q_cutoff cannot contribute to any pixel of the tile and
// are dropped; the survivors are appended IN ORDER to a shared-memory ring.  At the Mid workload
// only ~36 % of a tile's instances survive (the 3-sigma bounding square of an anisotropic splat is
// much larger than its ellipse), so the per-pixel phase touches ~3x fewer instances.
// Stage B (per pixel): eval_weight() -- the normative q (bit-identical to the oracle's fmaf
// expression), cut-off, alpha, w = alpha*T, T update, stop flag.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "common.cuh"

constexpr int TR_THREADS = 256;
constexpr int TR_QCAP = 512;           // ring capacity (power of two) >= KB + 256
constexpr uint32_t TR_FULL = 0xffffffffu;

// Four consecutive 16-bit stored values (one 8-byte load) <-> fp32.  Both directions are exact / round-to-nearest-even:
// fp16 and bf16 widen exactly; bf16 is the upper half of the binary32 pattern.
__device__ __forceinline__ float4 cvt16x4(uint2 r, const __half*) {
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ float4 cvt16x4(uint2 r, const __nv_bfloat16*) {
    return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u), __uint_as_float(r.y << 16),
                       __uint_as_float(r.y & 0xffff0000u));
}
__device__ __forceinline__ uint2 pack16x4(float4 v, const __half*) {
    const __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
    return make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&b));
}
__device__ __forceinline__ uint2 pack16x4(float4 v, const __nv_bfloat16*) {
    const __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
    return make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&b));
}

struct TraverseArgs {
    int W, H, GW;
    const uint32_t* ranges;   // [tiles,2]
    const uint32_t* vals;     // sorted Gaussian indices
    const float2* xy;
    const float4* conic_opacity;
    float q_cutoff, alpha_max, t_min;
    const float4* ray_transform;   // [n,3] float4 rows of adj(T): surfel mode (PRIM = 1) only
};

// PRIM = 0: 3-axis Gaussian, EWA conic (north_star).  PRIM = 1: the paper's 2-D surfel, u^2 + v^2 from
// the per-splat ray transform; the staged record then also carries its three rows (m[2].w = opacity).
template <int PRIM>
struct TileQueueT {           // shared-memory ring of staged survivors
    float2 xy[TR_QCAP];
    float4 co[TR_QCAP];       // A, 2B, C, opacity   (surfel: half_x, half_y, 0, opacity)
    uint32_t id[TR_QCAP];
    uint32_t wcount[TR_THREADS / 32];
    float4 m[PRIM ? 3 : 1][PRIM ? TR_QCAP : 1];
};
using TileQueue = TileQueueT<0>;

__device__ __forceinline__ void slot_to_xy(int slot, int& x, int& y) {
    const int warp = slot >> 5, lane = slot & 31;
    x = ((warp & 1) << 3) + (lane & 7);
    y = ((warp >> 1) << 2) + (lane >> 3);
}

// Minimum of q(d) = A dx^2 + 2B dx dy + C dy^2 over the box dx in [dx0,dx1], dy in [dy0,dy1]
// (d = Gaussian centre - pixel), minus a rounding allowance.  Conservative: may keep an instance
// that contributes nowhere, never drops one that does (NaNs compare false -> kept).
__device__ __forceinline__ bool tile_may_contribute(float2 g, float4 co, float bx0, float by0, float bx1, float by1,
                                                    float q_cutoff) {
    const float A = co.x, B2 = co.y, C = co.z;
    const float dx0 = g.x - bx1, dx1 = g.x - bx0;   // range of dx over the box
    const float dy0 = g.y - by1, dy1 = g.y - by0;
    if (dx0 <= 0.f && dx1 >= 0.f && dy0 <= 0.f && dy1 >= 0.f) return true;   // centre inside
    float best = 3.4e38f, best_mag = 0.f;
    // edges dx = const: minimise over dy in [dy0,dy1]; dy* = -B dx / C = -(B2 dx)/(2C)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const float dx = e ? dx1 : dx0;
        const float dy = fminf(fmaxf(-(B2 * dx) / (2.f * C), dy0), dy1);
        const float t0 = A * dx * dx, t1 = B2 * dx * dy, t2 = C * dy * dy;
        const float q = t0 + t1 + t2, m = t0 + fabsf(t1) + t2;
        if (!(q >= best)) { best = q; best_mag = m; }
    }
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const float dy = e ? dy1 : dy0;
        const float dx = fminf(fmaxf(-(B2 * dy) / (2.f * A), dx0), dx1);
        const float t0 = A * dx * dx, t1 = B2 * dx * dy, t2 = C * dy * dy;
        const float q = t0 + t1 + t2, m = t0 + fabsf(t1) + t2;
        if (!(q >= best)) { best = q; best_mag = m; }
    }
    return !(best - 1e-5f * best_mag - 1e-6f > q_cutoff);
}

// Examine instances [pos, min(pos+256, end)) and append the survivors to the ring at q_tail.
// Returns the number appended (same value in every thread).  Contains two __syncthreads().
template <int PRIM>
__device__ __forceinline__ int stage_chunk(const TraverseArgs& a, TileQueueT<PRIM>& q, uint32_t pos, uint32_t end, int q_tail,
                                           float bx0, float by0, float bx1, float by1) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t idx = pos + tid;
    bool keep = false;
    uint32_t id = 0;
    float2 g = make_float2(0.f, 0.f);
    float4 co = make_float4(0.f, 0.f, 0.f, 0.f);
    if (idx < end) {
        id = __ldg(a.vals + idx);
        g = __ldg(a.xy + id);
        co = __ldg(a.conic_opacity + id);
        if (PRIM) {   // footprint bounding box (centre g, half extents co.x, co.y; one pixel of margin is inside) vs the pixel box
            keep = !(g.x + co.x < bx0 || g.x - co.x > bx1 || g.y + co.y < by0 || g.y - co.y > by1);
        } else {
            co.y = 2.0f * co.y;   // exact
            keep = tile_may_contribute(g, co, bx0, by0, bx1, by1, a.q_cutoff);
        }
    }
    const uint32_t ballot = __ballot_sync(TR_FULL, keep);
    if (lane == 0) q.wcount[warp] = __popc(ballot);
    __syncthreads();
    int off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < TR_THREADS / 32; ++w) {
        const int c = (int)q.wcount[w];
        if (w < warp) off += c;
        total += c;
    }
    if (keep) {
        const int s = (q_tail + off + __popc(ballot & ((1u << lane) - 1u))) & (TR_QCAP - 1);
        q.xy[s] = g;
        q.co[s] = co;
        q.id[s] = id;
        if (PRIM) {
#pragma unroll
            for (int r = 0; r < 3; ++r) q.m[PRIM ? r : 0][PRIM ? s : 0] = __ldg(a.ray_transform + 3 * (size_t)id + r);
        }
    }
    __syncthreads();
    return total;
}

// C1-R steps 1-4 for one (pixel, Gaussian): returns w (0 when the Gaussian does not contribute).
// q is the normative expression fmaf(dx, fmaf(2B, dy, A dx), (C dy) dy) in binary32.
__device__ __forceinline__ float eval_weight(float2 g, float4 co, float fx, float fy, const TraverseArgs& a, float& T,
                                             bool& done, uint32_t& n) {
    const float dx = __fsub_rn(g.x, fx), dy = __fsub_rn(g.y, fy);
    const float q = __fmaf_rn(dx, __fmaf_rn(co.y, dy, __fmul_rn(co.x, dx)), __fmul_rn(__fmul_rn(co.z, dy), dy));
    if (done || !(q <= a.q_cutoff)) return 0.f;
    const float G = exp2f(-0.72134752044448170368f * fmaxf(q, 0.f));   // exp(-q/2)
    const float alpha = fminf(a.alpha_max, co.w * G);
    const float w = alpha * T;
    T = fmaf(-alpha, T, T);
    ++n;
    if (T < a.t_min) done = true;
    return w;
}

// Surfel form: p = adj(T) (x, y, 1)^T in binary32 fmaf form, num = p_x^2 + p_y^2, den = p_z^2; the
// splat contributes iff den > 0 and num <= q_cutoff * den (the decision needs no division; both sides evaluate exactly
// this expression); G = exp(-(num/den)/2).
__device__ __forceinline__ float eval_weight_surfel(float4 m0, float4 m1, float4 m2, float op, float fx, float fy,
                                                    const TraverseArgs& a, float& T, bool& done, uint32_t& n) {
    const float p0 = __fmaf_rn(fx, m0.x, __fmaf_rn(fy, m0.y, m0.z));
    const float p1 = __fmaf_rn(fx, m1.x, __fmaf_rn(fy, m1.y, m1.z));
    const float p2 = __fmaf_rn(fx, m2.x, __fmaf_rn(fy, m2.y, m2.z));
    const float num = __fmaf_rn(p0, p0, __fmul_rn(p1, p1)), den = __fmul_rn(p2, p2);
    if (done || !(den > 0.f) || !(num <= __fmul_rn(a.q_cutoff, den))) return 0.f;
    const float G = exp2f(-0.72134752044448170368f * __fdividef(num, den));
    const float alpha = fminf(a.alpha_max, op * G);
    const float w = alpha * T;
    T = fmaf(-alpha, T, T);
    ++n;
    if (T < a.t_min) done = true;
    return w;
}

// weight of staged survivor s of the ring for the pixel (fx, fy)
template <int PRIM>
__device__ __forceinline__ float eval_weight_q(const TileQueueT<PRIM>& q, int s, float fx, float fy, const TraverseArgs& a, float& T,
                                               bool& done, uint32_t& n) {
    if (PRIM) return eval_weight_surfel(q.m[0][PRIM ? s : 0], q.m[PRIM ? 1 : 0][PRIM ? s : 0], q.m[PRIM ? 2 : 0][PRIM ? s : 0], q.co[s].w, fx, fy, a, T, done, n);
    return eval_weight(q.xy[s], q.co[s], fx, fy, a, T, done, n);
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
