// ws.cuh -- the warp-specialised, persistent tile pipeline shared by the tiled render and fuse kernels.
//
// One CTA per SM, 512 threads: warps 0-7 are CONSUMERS (the D-channel product of the step), warps
// 8-15 are PRODUCERS (tile traversal: fetch, tile cull, blend weights w = alpha*T of PAPER.md:95).
// The CTA pulls work items (tile, channel chunk) from an atomic queue until it is empty.
//
// Producer (256 threads, one pixel each; slot s of the 16x16 tile: warp-block = s/32 covers 8x4 px):
//   stage   256 instances of the tile's sorted range are examined by one thread each (one chunk
//           ahead is prefetched into registers): exact ellipse-vs-tile-box test (traverse.cuh),
//           survivors appended in order to a shared-memory ring {xy, conic, opacity, id, rgb}.
//   batch   up to WS_KB ring entries form a batch in pipeline stage s: one bulk async copy
//           (cp.async.bulk, completion counted on the stage's `full` mbarrier) per feature row
//           (render) is issued first; then every producer thread evaluates the normative q, the
//           cut-off, alpha, w, T for its pixel and parks w in W[s][kk][slot]; per warp-block
//           bit masks say which instances gave the block any weight.
//   signal  meta[s] = {nb, tile, chunk, flags}; all 256 producers arrive on full[s].
// Consumer (256 threads): waits full[s], multiplies, arrives on empty[s]; on the LAST batch of an
// item it writes its accumulators out.  Producers run ahead by up to WS_STAGES batches, across
// tile boundaries, so global-load latency, the sequential weight phase and the FFMA-bound product
// overlap instead of alternating.
#pragma once
#include "traverse.cuh"

// Development aid (never defined in the product build): -DFHGS_WS_TIMING makes one consumer and one producer thread
// per CTA accumulate clock64() intervals of their pipeline phases into a device array the TU exports.
#ifdef FHGS_WS_TIMING
static __device__ unsigned long long g_ws_timing[32];
#define WS_TDECL long long ws_t_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}; long long ws_c_ = clock64()
#define WS_TACC(slot) do { const long long t__ = clock64(); ws_t_[slot] += t__ - ws_c_; ws_c_ = t__; } while (0)
#define WS_TCNT(slot) (ws_t_[slot] += 1)
#define WS_TFLUSH(base, pred) do { if (pred) { for (int i__ = 0; i__ < 16; ++i__) atomicAdd(&g_ws_timing[(base) + i__], (unsigned long long)ws_t_[i__]); } } while (0)
#else
#define WS_TDECL do { } while (0)
#define WS_TACC(slot) do { } while (0)
#define WS_TCNT(slot) do { } while (0)
#define WS_TFLUSH(base, pred) do { } while (0)
#endif

constexpr int WS_CONS = 256;
constexpr int WS_PROD = 256;
constexpr int WS_THREADS = WS_CONS + WS_PROD;
constexpr int WS_KB = 32;      // instances per batch (one bit each in the 32-bit block masks)
constexpr int WS_QCAP = 512;   // survivor ring capacity (power of two) >= WS_KB - 1 + WS_PROD

enum { WS_FLAG_LAST = 1, WS_FLAG_EXIT = 2 };
enum { WS_BAR_PROD = 1, WS_BAR_PROD_RED = 2 };   // named barriers (0 = __syncthreads)

struct WsMeta {
    int nb, tile, c0, flags;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// same, with a short sleep between probes (for the side that is normally ahead: it should not
// burn issue slots the other side needs)
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) __nanosleep(100);
}

// Packed FP32 FMA (sm_100+ fma.rn.f32x2): acc.{lo,hi} += w * f.{lo,hi}, each lane an IEEE fma.
// One issue slot for two FMAs -- the consumer loops are issue-bound next to the producer warps.
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float2 unpack2(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// in-place form: the accumulator is tied to one register pair (no copies in loop-carried accumulator tiles)
__device__ __forceinline__ void fma2_acc(unsigned long long& acc, unsigned long long a, unsigned long long b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
// 1-D bulk async copy global -> shared, completion (bytes) counted on `bar`.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// barrier + AND-reduction of a predicate over the participating threads
__device__ __forceinline__ bool named_bar_and(int id, int nthreads, bool pred) {
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %1, 0;\n\tbarrier.red.and.pred q, %2, %3, p;\n\tselp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(r)
        : "r"((uint32_t)pred), "r"(id), "r"(nthreads)
        : "memory");
    return r != 0;
}
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Control block of the pipeline (lives at the front of dynamic shared memory).
// PRIM = 0 (EWA Gaussian): rec0 = gx, gy, A, 2B; rec1 = C, opacity, id, position.
// PRIM = 1 (surfel): the nine entries of the ray transform adj(T): rec0 = m00, m01, m02, m10;
//          rec1 = m11, opacity, id, position; rec2 = m12, m20, m21, m22.
template <int STAGES, int PRIM = 0, int Q = WS_QCAP>
struct WsCtrl {
    // ring capacity: >= WS_KB - 1 + WS_PROD = 287 (a chunk is appended only while fewer than WS_KB survivors are queued).
    // A power of two wraps with a mask; the surfel form of fuse_ws has no shared memory for 512 slots of three records
    // and uses 288 with a modulo.
    static constexpr int QCAP = Q;
    static_assert(Q >= WS_KB - 1 + WS_PROD, "ring too small");
    static __device__ __forceinline__ int slot(int x) { return (Q & (Q - 1)) == 0 ? (x & (Q - 1)) : (int)((unsigned)x % (unsigned)Q); }
    uint64_t full[STAGES];
    uint64_t empty[STAGES];
    WsMeta meta[STAGES];
    uint32_t mask[STAGES][8];     // per warp-block: bit kk set <=> instance kk gave the block a weight
    uint32_t wcount[WS_PROD / 32];
    int item;                     // work item broadcast among the producers
    float4 rec0[Q];
    float4 rec1[Q];               // .y opacity, .z id (bits), .w position in the sorted list (bits)
    float4 rec2[PRIM ? Q : 1];
};

struct WsWork {
    uint32_t* queue;      // [0] next item, [1] finished CTAs (self-resetting; zero between launches)
    int n_items;          // tiles * chunks
    int n_chunks;
    const uint32_t* order;        // tile permutation, longest instance list first (written by fhgs_bin_sort)
    const uint32_t* order_valid;  // device flag: 0 -> identity order
};

// Work item -> tile.  The queue hands out items in increasing order; with the longest-first permutation the heavy
// tiles start early and the tail of the persistent loop is made of short ones.
__device__ __forceinline__ int ws_item_tile(const WsWork& wk, int item) {
    const int t = item / wk.n_chunks;
    return __ldg(wk.order_valid) ? (int)__ldg(wk.order + t) : t;
}

// Per-pixel blend state of a producer thread.
struct WsPixel {
    float fx, fy, T;
    uint32_t n;
    bool done;
};

// C1-R steps 1-4 for one (pixel, Gaussian); q is the normative binary32 expression
// fmaf(dx, fmaf(2B, dy, A dx), (C dy) dy).  Returns w (0 when the Gaussian does not contribute).
__device__ __forceinline__ float ws_weight(const float4 r0, const float C, const float op, WsPixel& p, const float q_cutoff,
                                           const float alpha_max, const float t_min) {
    // branch-free: the only loop-carried chain is w = a*T; T = T - a*T (everything else pipelines)
    const float dx = __fsub_rn(r0.x, p.fx), dy = __fsub_rn(r0.y, p.fy);
    const float q = __fmaf_rn(dx, __fmaf_rn(r0.w, dy, __fmul_rn(r0.z, dx)), __fmul_rn(__fmul_rn(C, dy), dy));
    const float G = ex2_approx(-0.72134752044448170368f * fmaxf(q, 0.f));   // exp(-q/2)
    const float alpha = fminf(alpha_max, op * G);
    const bool c = (q <= q_cutoff) && !p.done;
    const float a = c ? alpha : 0.f;
    const float w = a * p.T;
    p.T = fmaf(-a, p.T, p.T);
    p.n += c ? 1u : 0u;
    p.done = p.done || (p.T < t_min);
    return w;
}

// Surfel form of ws_weight: p = adj(T) (x, y, 1)^T, num = p_x^2 + p_y^2, den = p_z^2 in the normative binary32 fmaf
// expressions (traverse.cuh eval_weight_surfel, oracle fo_surfel_terms); contributes iff den > 0 and num <= q_cut den.
__device__ __forceinline__ float ws_weight_surfel(const float4 r0, const float4 r1, const float4 r2, WsPixel& p, const float q_cutoff,
                                                  const float alpha_max, const float t_min) {
    const float p0 = __fmaf_rn(p.fx, r0.x, __fmaf_rn(p.fy, r0.y, r0.z));
    const float p1 = __fmaf_rn(p.fx, r0.w, __fmaf_rn(p.fy, r1.x, r2.x));
    const float p2 = __fmaf_rn(p.fx, r2.y, __fmaf_rn(p.fy, r2.z, r2.w));
    const float num = __fmaf_rn(p0, p0, __fmul_rn(p1, p1)), den = __fmul_rn(p2, p2);
    const bool c = (den > 0.f) && (num <= __fmul_rn(q_cutoff, den)) && !p.done;
    const float G = ex2_approx(-0.72134752044448170368f * __fdividef(num, c ? den : 1.f));
    const float alpha = fminf(alpha_max, r1.y * G);
    const float a = c ? alpha : 0.f;
    const float w = a * p.T;
    p.T = fmaf(-a, p.T, p.T);
    p.n += c ? 1u : 0u;
    p.done = p.done || (p.T < t_min);
    return w;
}

// Chunk of WS_PROD instances held in registers (one per producer thread), software-pipelined two deep:
// `id_next` (the sorted-list entry of the chunk after this one) is in flight while this chunk's
// projected Gaussian (xy, conic, opacity, colour) is in flight, so neither dependent global load is
// waited for at its issue point.
struct WsChunk {
    uint32_t id;
    float2 g;
    float4 co;
    float r, gr, b;
    bool valid;
    uint32_t id_next;
    bool valid_next;
};

__device__ __forceinline__ void ws_chunk_issue(const TraverseArgs& a, const float* rgb_g, WsChunk& c) {
    // consume id_next -> issue this chunk's gathers
    c.id = c.id_next;
    c.valid = c.valid_next;
    c.g = make_float2(0.f, 0.f);
    c.co = make_float4(0.f, 0.f, 0.f, 0.f);
    c.r = c.gr = c.b = 0.f;
    if (c.valid) {
        c.g = __ldg(a.xy + c.id);
        c.co = __ldg(a.conic_opacity + c.id);
        if (rgb_g) {
            c.r = __ldg(rgb_g + 3 * (size_t)c.id);
            c.gr = __ldg(rgb_g + 3 * (size_t)c.id + 1);
            c.b = __ldg(rgb_g + 3 * (size_t)c.id + 2);
        }
    }
}
__device__ __forceinline__ void ws_chunk_prefetch_id(const TraverseArgs& a, uint32_t pos, uint32_t end, int p, WsChunk& c) {
    const uint32_t idx = pos + (uint32_t)p;
    c.valid_next = idx < end;
    c.id_next = c.valid_next ? __ldg(a.vals + idx) : 0u;
}

// Tile-cull the chunk and append the survivors, in order, to the ring at q_tail.  Returns the number
// appended (same in all producer threads).  Two producer-wide barriers.
template <int PRIM = 0, typename CTRL, typename EXTRA>
__device__ __forceinline__ int ws_chunk_append(CTRL& ct, const WsChunk& c, uint32_t chunk_pos, int q_tail, float bx0, float by0,
                                               float bx1, float by1, float q_cutoff, int p, EXTRA&& extra,
                                               const float4* ray_transform = nullptr) {
    const int lane = p & 31, pw = p >> 5;
    float4 co = c.co;
    bool keep;
    if (PRIM) {   // surfel: footprint bounding box (centre c.g, half extents co.x, co.y) against the tile's pixel box
        keep = c.valid && !(c.g.x + co.x < bx0 || c.g.x - co.x > bx1 || c.g.y + co.y < by0 || c.g.y - co.y > by1);
    } else {
        co.y = 2.0f * co.y;   // exact
        keep = c.valid && tile_may_contribute(c.g, co, bx0, by0, bx1, by1, q_cutoff);
    }
    // surfel: the survivors' ray transforms are fetched here (not prefetched with the chunk: 12 more registers per producer
    // thread would spill; the producers have the slack)
    float4 m0 = make_float4(0.f, 0.f, 0.f, 0.f), m1 = m0, m2 = m0;
    if (PRIM && keep) {
        m0 = __ldg(ray_transform + 3 * (size_t)c.id);
        m1 = __ldg(ray_transform + 3 * (size_t)c.id + 1);
        m2 = __ldg(ray_transform + 3 * (size_t)c.id + 2);
    }
    const uint32_t ballot = __ballot_sync(TR_FULL, keep);
    if (lane == 0) ct.wcount[pw] = __popc(ballot);
    named_bar_sync(WS_BAR_PROD, WS_PROD);
    int off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < WS_PROD / 32; ++w) {
        const int cnt = (int)ct.wcount[w];
        if (w < pw) off += cnt;
        total += cnt;
    }
    if (keep) {
        const int s = CTRL::slot(q_tail + off + __popc(ballot & ((1u << lane) - 1u)));
        if (PRIM) {
            ct.rec0[s] = make_float4(m0.x, m0.y, m0.z, m1.x);
            ct.rec1[s] = make_float4(m1.y, co.w, __uint_as_float(c.id), __uint_as_float(chunk_pos + (uint32_t)p));
            ct.rec2[PRIM ? s : 0] = make_float4(m1.z, m2.x, m2.y, m2.z);
        } else {
            ct.rec0[s] = make_float4(c.g.x, c.g.y, co.x, co.y);
            ct.rec1[s] = make_float4(co.z, co.w, __uint_as_float(c.id), __uint_as_float(chunk_pos + (uint32_t)p));
        }
        extra(s, c);
    }
    named_bar_sync(WS_BAR_PROD, WS_PROD);
    return total;
}

// Work-item queue: thread p == 0 pops; the pop for the NEXT item is issued at the start of the current
// one (ws_pop_begin) and only consumed at its end (ws_pop_end), so its latency is hidden.
__device__ __forceinline__ uint32_t ws_pop_begin(const WsWork& wk, int p) {
    return p == 0 ? atomicAdd(wk.queue, 1u) : 0u;
}
template <typename CTRL>
__device__ __forceinline__ int ws_pop_end(CTRL& ct, uint32_t popped, int p) {
    if (p == 0) ct.item = (int)popped;
    named_bar_sync(WS_BAR_PROD, WS_PROD);
    const int item = ct.item;
    named_bar_sync(WS_BAR_PROD, WS_PROD);
    return item;
}

// Last CTA out resets the queue so that the next launch on this view state starts from zero.
__device__ __forceinline__ void ws_queue_release(const WsWork& wk) {
    __threadfence();
    const uint32_t fin = atomicAdd(wk.queue + 1, 1u);
    if (fin == gridDim.x - 1) {
        wk.queue[0] = 0u;
        wk.queue[1] = 0u;
        __threadfence();
    }
}
