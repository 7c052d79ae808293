// render.cu -- step R (fhgs_render): per-tile front-to-back compositing of RGB + D feature channels.
// PAPER.md:90-95 (Eq. 4); SURVEY 8(c) C1-R.
//
// One CTA (256 threads) per 16x16 tile.  The feature work of a tile is the product
//     F[256 px, D] += W[256 px, K] * f[K, D]
// over the K instances that survive the tile cull (traverse.cuh).  It is evaluated in sub-batches of
// KB staged instances:
//   phase B  thread = pixel: weights w = alpha*T for the KB instances (sequential in T), RGB
//            accumulation, w parked in shared memory W[kk][slot]; each warp records which
//            instances gave any of its 32 pixels a weight.
//   phase C  register-tiled outer products: thread = 8 pixels x (DC/8) channels, accumulators in
//            registers (128 for DC = 128); one broadcast LDS.128 pair of W and DC/32 LDS.128 of f
//            feed 8*DC/8 FFMAs.  Instances with no weight inside the warp are skipped (warp-uniform).
// The feature rows of a sub-batch are fetched with cp.async while phase B runs.
// D > DC is handled by channel passes (the traversal is repeated per pass; RGB/T/n are written by
// pass 0).  Small D (not a multiple of 64) uses the per-pixel variant: CH accumulators per thread,
// updated inside phase B from broadcast shared-memory reads.
#include "layout.cuh"
#include "ws.cuh"

namespace {

struct RenderArgs {
    TraverseArgs t;
    const float* rgb_g;   // [n,3]
    const void* feat;     // [n,D] or NULL
    int D;
    float bg[3];
    float* out_rgb;
    void* out_feat;
    float* out_T;
    uint32_t* out_n;
    uint32_t* tile_visited;   // [tiles] diagnostics: length of the prefix of the tile's list that was walked
};

constexpr int R_KB = 64;   // staged instances per drain of the per-pixel variant

template <typename FT> struct FeatIO;
template <> struct FeatIO<float> {
    static __device__ __forceinline__ float4 load4(const float* p) { return *reinterpret_cast<const float4*>(p); }
    static __device__ __forceinline__ void store4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
    // 4 consecutive channels as two packed pairs, straight from the 16-byte load (no repacking moves)
    static __device__ __forceinline__ ulonglong2 load_pairs(const float* p) { return *reinterpret_cast<const ulonglong2*>(p); }
};
// 16-bit storage (fp16 or bf16): widened exactly on load, rounded to nearest even on store
template <typename HT> struct FeatIO16 {
    static __device__ __forceinline__ float4 load4(const HT* p) { return cvt16x4(*reinterpret_cast<const uint2*>(p), p); }
    static __device__ __forceinline__ void store4(HT* p, float4 v) { *reinterpret_cast<uint2*>(p) = pack16x4(v, p); }
    static __device__ __forceinline__ ulonglong2 load_pairs(const HT* p) {
        const float4 f = load4(p);
        return make_ulonglong2(pack2(f.x, f.y), pack2(f.z, f.w));
    }
};
template <> struct FeatIO<__half> : FeatIO16<__half> {};
template <> struct FeatIO<__nv_bfloat16> : FeatIO16<__nv_bfloat16> {};

// ---------------------------------------------------------------------------------------------
// TILED variant (DC in {64,128}): warp-specialised persistent pipeline (ws.cuh)
// ---------------------------------------------------------------------------------------------
constexpr int R_STAGES = 3;
#ifndef R_PROD_REGS
#define R_PROD_REGS 72
#define R_CONS_REGS 184
#endif
// Which warps are the consumers.  The SMSP arbiter favours high warp ids: with fp32 rows the consumers are the
// critical path and get the high ids (-6 % on Mid); with fp16 rows (conversion work in the consumer loop, four
// channel passes per tile) the producers are the ones that must not starve (measured on Large).
template <typename FT>
constexpr bool kConsHigh = sizeof(FT) == 4;

template <int DC, typename FT, int PRIM = 0>
struct RenderWsSmem {
    WsCtrl<R_STAGES, PRIM> ct;
    float4 rgb[WS_QCAP];                                   // staged colours (xyz used)
    __align__(128) float W[R_STAGES][WS_KB * WS_CONS];     // W[s][kk][slot]
    __align__(128) FT F[R_STAGES][WS_KB * DC];             // feature rows of the batch
};

template <int DC, typename FT, bool DIAG, int PRIM>
__device__ __forceinline__ void render_ws_producer(RenderWsSmem<DC, FT, PRIM>& sm, const RenderArgs& a, const WsWork& wk) {
    const int p = threadIdx.x - (kConsHigh<FT> ? 0 : WS_CONS), lane = p & 31, pw = p >> 5;   // p = pixel slot, pw = warp-block
    const FT* feat = reinterpret_cast<const FT*>(a.feat);
    const float q_cutoff = a.t.q_cutoff, alpha_max = a.t.alpha_max, t_min = a.t.t_min;
    int stage = 0;
    uint32_t phase = 0;
    int sx, sy;
    slot_to_xy(p, sx, sy);
    int item = ws_pop_end(sm.ct, ws_pop_begin(wk, p), p);
    WS_TDECL;
    while (true) {
        if (item >= wk.n_items) {
            mbar_wait(&sm.ct.empty[stage], phase ^ 1u);
            if (p == 0) sm.ct.meta[stage] = WsMeta{0, -1, 0, WS_FLAG_EXIT};
            mbar_arrive(&sm.ct.full[stage]);
            WS_TFLUSH(16, p == 0);
            break;
        }
        const uint32_t popped = ws_pop_begin(wk, p);   // next item, consumed at the end of this one
        const int tile = ws_item_tile(wk, item), c0 = (item % wk.n_chunks) * DC;
        const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE;
        const int px = tx0 + sx, py = ty0 + sy;
        const bool inside = px < a.t.W && py < a.t.H;
        WsPixel P{(float)px, (float)py, 1.f, 0u, !inside};
        float C0 = 0.f, C1 = 0.f, C2 = 0.f;
        const float bx0 = (float)tx0, by0 = (float)ty0;
        const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + FHGS_TILE - 1, a.t.H - 1);
        const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
        uint32_t pos = range.x;
        int qh = 0, qt = 0;
        WsChunk ch;
        ws_chunk_prefetch_id(a.t, pos, range.y, p, ch);
        ws_chunk_issue(a.t, a.rgb_g, ch);
        ws_chunk_prefetch_id(a.t, pos + WS_PROD, range.y, p, ch);
        bool last = false;
        do {
            while (qt - qh < WS_KB && pos < range.y) {
                qt += ws_chunk_append<PRIM>(sm.ct, ch, pos, qt, bx0, by0, bx1, by1, q_cutoff, p,
                                            [&](int s, const WsChunk& c) { sm.rgb[s] = make_float4(c.r, c.gr, c.b, 0.f); },
                                            a.t.ray_transform);
                pos += WS_PROD;
                ws_chunk_issue(a.t, a.rgb_g, ch);
                ws_chunk_prefetch_id(a.t, pos + WS_PROD, range.y, p, ch);
            }
            const int nb = min(WS_KB, qt - qh);
            WS_TACC(1);
            mbar_wait_backoff(&sm.ct.empty[stage], phase ^ 1u);
            WS_TACC(2);
            // feature rows of the batch: one bulk async copy each, counted on full[stage]
            if (pw == 0 && lane < nb) {
                const uint32_t id = __float_as_uint(sm.ct.rec1[(qh + lane) & (WS_QCAP - 1)].z);
                mbar_expect_tx(&sm.ct.full[stage], (uint32_t)(DC * sizeof(FT)));
                bulk_g2s(&sm.F[stage][lane * DC], feat + (size_t)id * a.D + c0, (uint32_t)(DC * sizeof(FT)), &sm.ct.full[stage]);
            }
            // weights of the batch for this thread's pixel
            uint32_t m = 0u;
            float* Wd = sm.W[stage] + p;
            if (!__all_sync(TR_FULL, P.done)) {
#pragma unroll 4
                for (int kk = 0; kk < nb; ++kk) {
                    const int s = (qh + kk) & (WS_QCAP - 1);
                    const float4 r0 = sm.ct.rec0[s];
                    const float4 r1 = sm.ct.rec1[s];
                    const float4 c = sm.rgb[s];
                    const float w = PRIM ? ws_weight_surfel(r0, r1, sm.ct.rec2[PRIM ? s : 0], P, q_cutoff, alpha_max, t_min)
                                         : ws_weight(r0, r1.x, r1.y, P, q_cutoff, alpha_max, t_min);
                    Wd[kk * WS_CONS] = w;
                    C0 = fmaf(w, c.x, C0); C1 = fmaf(w, c.y, C1); C2 = fmaf(w, c.z, C2);
                    m |= (w != 0.f ? 1u : 0u) << kk;
                }
                m = __reduce_or_sync(TR_FULL, m);
            }
            if (lane == 0) sm.ct.mask[stage][pw] = m;
            qh += nb;
            WS_TACC(3);
            const bool all_done = named_bar_and(WS_BAR_PROD_RED, WS_PROD, P.done);
            last = all_done || (pos >= range.y && qt == qh);
            if (p == 0) sm.ct.meta[stage] = WsMeta{nb, tile, c0, last ? WS_FLAG_LAST : 0};
            mbar_arrive(&sm.ct.full[stage]);
            if (DIAG && a.tile_visited && last && c0 == 0 && p == 32) {
                // diagnostics, once per tile and off the critical path: if the tile stopped early, the last blended
                // instance lies in this final batch (the pixel that completed the tile blended it)
                uint32_t visited = range.y - range.x;
                if (all_done) {
                    uint32_t any = 0u;
#pragma unroll
                    for (int w8 = 0; w8 < 8; ++w8) any |= sm.ct.mask[stage][w8];
                    visited = any ? __float_as_uint(sm.ct.rec1[(qh - nb + 31 - __clz(any)) & (WS_QCAP - 1)].w) + 1u - range.x : 0u;
                }
                a.tile_visited[tile] = visited;
            }
            WS_TACC(4);
            if (++stage == R_STAGES) { stage = 0; phase ^= 1u; }
        } while (!last);
        if (c0 == 0 && inside) {
            const size_t o = (size_t)py * a.t.W + px;
            a.out_rgb[3 * o] = fmaf(P.T, a.bg[0], C0);
            a.out_rgb[3 * o + 1] = fmaf(P.T, a.bg[1], C1);
            a.out_rgb[3 * o + 2] = fmaf(P.T, a.bg[2], C2);
            if (a.out_T) a.out_T[o] = P.T;
            if (a.out_n) a.out_n[o] = P.n;
        }
        item = ws_pop_end(sm.ct, popped, p);
        WS_TACC(0);
    }
}

template <int DC, typename FT, int PRIM>
__device__ __forceinline__ void render_ws_consumer(RenderWsSmem<DC, FT, PRIM>& sm, const RenderArgs& a) {
    constexpr int NJ = DC / 32;   // float4 channel groups per thread
    // consumers are the HIGH warps (8-15): the SMSP arbiter favours high warp ids, and the consumers are the critical path
    const int tid = threadIdx.x - (kConsHigh<FT> ? WS_PROD : 0), lane = tid & 31, warp = tid >> 5;
    const int pgl = lane >> 3, cg = lane & 7;
    const int pg = warp * 4 + pgl;   // 8-pixel row run: slots pg*8 .. pg*8+7
    FT* out_feat = reinterpret_cast<FT*>(a.out_feat);
    int stage = 0;
    uint32_t phase = 0;
    WS_TDECL;
    while (true) {   // one iteration per work item: accumulators live exactly one item
        unsigned long long acc[NJ * 2][8];   // [channel pair][pixel], packed (fma.rn.f32x2); this index order leaves ptxas the fewest
                                           // accumulator copies in the loop below (8 instead of 21 per 64 FFMA2)
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < NJ * 2; ++j) acc[j][i] = 0ull;
        WsMeta m;
        while (true) {   // batches of the item
            mbar_wait(&sm.ct.full[stage], phase);
            WS_TACC(0);
            m = sm.ct.meta[stage];
            if (m.flags & WS_FLAG_EXIT) { WS_TFLUSH(0, tid == 0); return; }
            WS_TCNT(5);
            uint32_t mk = sm.ct.mask[stage][warp];
            const float* Ws = sm.W[stage] + pg * 8;
            const FT* Fs = sm.F[stage] + cg * 4;
            while (mk) {
                const int kk = __ffs(mk) - 1;
                mk &= mk - 1u;
                const float4 wa = *reinterpret_cast<const float4*>(Ws + kk * WS_CONS);
                const float4 wb = *reinterpret_cast<const float4*>(Ws + kk * WS_CONS + 4);
                const float wv[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
                unsigned long long fv[NJ * 2];
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const ulonglong2 f = FeatIO<FT>::load_pairs(Fs + kk * DC + j * 32);
                    fv[2 * j] = f.x;
                    fv[2 * j + 1] = f.y;
                }
                unsigned long long w2[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) w2[i] = pack2(wv[i], wv[i]);
#pragma unroll
                for (int j = 0; j < NJ * 2; ++j)
#pragma unroll
                    for (int i = 0; i < 8; ++i) fma2_acc(acc[j][i], w2[i], fv[j]);
            }
            mbar_arrive(&sm.ct.empty[stage]);
            WS_TACC(1);
            if (++stage == R_STAGES) { stage = 0; phase ^= 1u; }
            if (m.flags & WS_FLAG_LAST) break;
        }
        const int tx0 = (m.tile % a.t.GW) * FHGS_TILE, ty0 = (m.tile / a.t.GW) * FHGS_TILE;
        const int oy = ty0 + ((warp >> 1) << 2) + pgl;
        const int ox0 = tx0 + ((warp & 1) << 3);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int ox = ox0 + i;
            if (oy < a.t.H && ox < a.t.W) {
                FT* dst = out_feat + ((size_t)oy * a.t.W + ox) * a.D + m.c0 + cg * 4;
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const float2 lo = unpack2(acc[2 * j][i]), hi = unpack2(acc[2 * j + 1][i]);
                    FeatIO<FT>::store4(dst + j * 32, make_float4(lo.x, lo.y, hi.x, hi.y));
                }
            }
        }
        WS_TACC(2);
        WS_TCNT(6);
    }
}

template <int DC, typename FT, bool DIAG, int PRIM = 0>
__global__ void __launch_bounds__(WS_THREADS, 1) render_ws_kernel(const RenderArgs a, const WsWork wk) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    RenderWsSmem<DC, FT, PRIM>& sm = *reinterpret_cast<RenderWsSmem<DC, FT, PRIM>*>(smem_raw);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < R_STAGES; ++s) {
            mbar_init(&sm.ct.full[s], WS_PROD);
            mbar_init(&sm.ct.empty[s], WS_CONS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    const bool is_producer = kConsHigh<FT> ? threadIdx.x < WS_PROD : threadIdx.x >= WS_CONS;
    if (is_producer) {
        setmaxnreg_dec<R_PROD_REGS>();
        render_ws_producer<DC, FT, DIAG, PRIM>(sm, a, wk);
    } else {
        setmaxnreg_inc<R_CONS_REGS>();
        render_ws_consumer<DC, FT, PRIM>(sm, a);
        if (threadIdx.x == (kConsHigh<FT> ? WS_PROD : 0)) ws_queue_release(wk);
    }
}

// ---------------------------------------------------------------------------------------------
// PIXEL variant: CH in {0,4,8,16} feature channels per pass, accumulated by the pixel's own thread
// ---------------------------------------------------------------------------------------------
template <int CH, int PRIM>
struct PixelSmem {
    TileQueueT<PRIM> q;
    float4 rgb[TR_QCAP];
    __align__(16) float F[TR_QCAP * (CH > 0 ? CH : 1)];
};

template <int CH, typename FT, int PRIM>
__global__ void __launch_bounds__(TR_THREADS) render_pixel_kernel(const RenderArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PixelSmem<CH, PRIM>& sm = *reinterpret_cast<PixelSmem<CH, PRIM>*>(smem_raw);

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
    const FT* feat = reinterpret_cast<const FT*>(a.feat);
    FT* out_feat = reinterpret_cast<FT*>(a.out_feat);
    const int D = CH > 0 ? a.D : 1;

    for (int c0 = 0; c0 < D; c0 += (CH > 0 ? CH : 1)) {
        float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
        uint32_t n = 0;
        bool done = !inside;
        float acc[CH > 0 ? CH : 1];
#pragma unroll
        for (int j = 0; j < (CH > 0 ? CH : 1); ++j) acc[j] = 0.f;
        uint32_t pos = range.x;
        int q_head = 0, q_count = 0;
        while (true) {
            while (q_count < R_KB && pos < range.y) {
                const int tail = q_head + q_count;
                const int added = stage_chunk(a.t, sm.q, pos, range.y, tail, bx0, by0, bx1, by1);
                for (int k = tid; k < added; k += TR_THREADS) {
                    const int s = (tail + k) & (TR_QCAP - 1);
                    const uint32_t id = sm.q.id[s];
                    sm.rgb[s] = make_float4(__ldg(a.rgb_g + 3 * (size_t)id), __ldg(a.rgb_g + 3 * (size_t)id + 1),
                                            __ldg(a.rgb_g + 3 * (size_t)id + 2), 0.f);
                }
                if constexpr (CH > 0) {
                    for (int k = tid; k < added * (CH / 4); k += TR_THREADS) {
                        const int r = k / (CH / 4), c = k % (CH / 4);
                        const int s = (tail + r) & (TR_QCAP - 1);
                        const uint32_t id = sm.q.id[s];
                        *reinterpret_cast<float4*>(&sm.F[s * CH + 4 * c]) = FeatIO<FT>::load4(feat + (size_t)id * a.D + c0 + 4 * c);
                    }
                }
                q_count += added;
                pos += TR_THREADS;
            }
            const int nb = q_count;   // drain everything staged
            if (nb == 0) break;
            __syncthreads();
            for (int kk = 0; kk < nb; ++kk) {
                const int s = (q_head + kk) & (TR_QCAP - 1);
                const float w = eval_weight_q<PRIM>(sm.q, s, fx, fy, a.t, T, done, n);
                if (w != 0.f) {
                    const float4 c = sm.rgb[s];
                    C0 = fmaf(w, c.x, C0); C1 = fmaf(w, c.y, C1); C2 = fmaf(w, c.z, C2);
                    if constexpr (CH > 0) {
#pragma unroll
                        for (int j = 0; j < CH / 4; ++j) {
                            const float4 f = *reinterpret_cast<const float4*>(&sm.F[s * CH + 4 * j]);
                            acc[4 * j] = fmaf(w, f.x, acc[4 * j]);
                            acc[4 * j + 1] = fmaf(w, f.y, acc[4 * j + 1]);
                            acc[4 * j + 2] = fmaf(w, f.z, acc[4 * j + 2]);
                            acc[4 * j + 3] = fmaf(w, f.w, acc[4 * j + 3]);
                        }
                    }
                }
            }
            q_head = (q_head + nb) & (TR_QCAP - 1);
            q_count = 0;
            if (__syncthreads_and(done)) break;
        }
        if (c0 == 0 && tid == 0 && a.tile_visited) a.tile_visited[tile] = min(pos, range.y) - range.x;   // chunk granular (256 instances)
        if (inside) {
            const size_t p = (size_t)py * a.t.W + px;
            if (c0 == 0) {
                a.out_rgb[3 * p] = fmaf(T, a.bg[0], C0);
                a.out_rgb[3 * p + 1] = fmaf(T, a.bg[1], C1);
                a.out_rgb[3 * p + 2] = fmaf(T, a.bg[2], C2);
                if (a.out_T) a.out_T[p] = T;
                if (a.out_n) a.out_n[p] = n;
            }
            if constexpr (CH > 0) {
#pragma unroll
                for (int j = 0; j < CH / 4; ++j)
                    FeatIO<FT>::store4(out_feat + p * a.D + c0 + 4 * j,
                                       make_float4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]));
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Single-traversal render + fuse (fhgs_render_fuse; SURVEY 8(f) NEXT-4 ii) for the per-pixel regime (D not a multiple of
// 64): the pixel's thread evaluates every weight w = alpha T once and uses it twice -- for the pixel's own
// colour / feature sums (step R) and, reduced over the warp's 32 pixels with shuffles, for num[id] += w gt(x), den[id] += w
// (step F: one red per warp and Gaussian).  Same arithmetic and order as render_pixel_kernel and fuse.cu's pixel kernel.
// ---------------------------------------------------------------------------------------------
struct RenderFuseArgs {
    RenderArgs r;
    const void* gt;   // [H,W,D], same storage type as the feature rows
    float* num;
    float* den;
};

__device__ __forceinline__ void rf_red_add_v4(float* addr, float4 v) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void rf_red_add(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

template <int CH, typename FT, int PRIM>
__global__ void __launch_bounds__(TR_THREADS) render_fuse_pixel_kernel(const RenderFuseArgs af) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PixelSmem<CH, PRIM>& sm = *reinterpret_cast<PixelSmem<CH, PRIM>*>(smem_raw);
    const RenderArgs& a = af.r;
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
    const FT* feat = reinterpret_cast<const FT*>(a.feat);
    const FT* gt = reinterpret_cast<const FT*>(af.gt);
    FT* out_feat = reinterpret_cast<FT*>(a.out_feat);

    for (int c0 = 0; c0 < a.D; c0 += CH) {
        float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
        uint32_t n = 0;
        bool done = !inside;
        float acc[CH], g[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) acc[j] = 0.f;
#pragma unroll
        for (int j = 0; j < CH / 4; ++j) {
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (inside) v = FeatIO<FT>::load4(gt + ((size_t)py * a.t.W + px) * a.D + c0 + 4 * j);
            g[4 * j] = v.x; g[4 * j + 1] = v.y; g[4 * j + 2] = v.z; g[4 * j + 3] = v.w;
        }
        uint32_t pos = range.x;
        int q_head = 0, q_count = 0;
        while (true) {
            while (q_count < R_KB && pos < range.y) {
                const int tail = q_head + q_count;
                const int added = stage_chunk(a.t, sm.q, pos, range.y, tail, bx0, by0, bx1, by1);
                for (int k = tid; k < added; k += TR_THREADS) {
                    const int s = (tail + k) & (TR_QCAP - 1);
                    const uint32_t id = sm.q.id[s];
                    sm.rgb[s] = make_float4(__ldg(a.rgb_g + 3 * (size_t)id), __ldg(a.rgb_g + 3 * (size_t)id + 1),
                                            __ldg(a.rgb_g + 3 * (size_t)id + 2), 0.f);
                }
                for (int k = tid; k < added * (CH / 4); k += TR_THREADS) {
                    const int r = k / (CH / 4), c = k % (CH / 4);
                    const int s = (tail + r) & (TR_QCAP - 1);
                    const uint32_t id = sm.q.id[s];
                    *reinterpret_cast<float4*>(&sm.F[s * CH + 4 * c]) = FeatIO<FT>::load4(feat + (size_t)id * a.D + c0 + 4 * c);
                }
                q_count += added;
                pos += TR_THREADS;
            }
            const int nb = q_count;   // drain everything staged
            if (nb == 0) break;
            __syncthreads();
            for (int kk = 0; kk < nb; ++kk) {
                const int s = (q_head + kk) & (TR_QCAP - 1);
                const float w = eval_weight_q<PRIM>(sm.q, s, fx, fy, a.t, T, done, n);   // the one weight phase
                if (w != 0.f) {   // step R: this pixel's sums
                    const float4 c = sm.rgb[s];
                    C0 = fmaf(w, c.x, C0); C1 = fmaf(w, c.y, C1); C2 = fmaf(w, c.z, C2);
#pragma unroll
                    for (int j = 0; j < CH / 4; ++j) {
                        const float4 f = *reinterpret_cast<const float4*>(&sm.F[s * CH + 4 * j]);
                        acc[4 * j] = fmaf(w, f.x, acc[4 * j]);
                        acc[4 * j + 1] = fmaf(w, f.y, acc[4 * j + 1]);
                        acc[4 * j + 2] = fmaf(w, f.z, acc[4 * j + 2]);
                        acc[4 * j + 3] = fmaf(w, f.w, acc[4 * j + 3]);
                    }
                }
                if (!__any_sync(TR_FULL, w != 0.f)) continue;   // step F: this Gaussian's sums over the warp's pixels
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
                    float* dst = af.num + (size_t)id * a.D + c0;
#pragma unroll
                    for (int j = 0; j < CH / 4; ++j) rf_red_add_v4(dst + 4 * j, make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]));
                    if (c0 == 0) rf_red_add(af.den + id, v[CH]);
                }
            }
            q_head = (q_head + nb) & (TR_QCAP - 1);
            q_count = 0;
            if (__syncthreads_and(done)) break;
        }
        if (inside) {
            const size_t p = (size_t)py * a.t.W + px;
            if (c0 == 0) {
                a.out_rgb[3 * p] = fmaf(T, a.bg[0], C0);
                a.out_rgb[3 * p + 1] = fmaf(T, a.bg[1], C1);
                a.out_rgb[3 * p + 2] = fmaf(T, a.bg[2], C2);
                if (a.out_T) a.out_T[p] = T;
                if (a.out_n) a.out_n[p] = n;
            }
#pragma unroll
            for (int j = 0; j < CH / 4; ++j)
                FeatIO<FT>::store4(out_feat + p * a.D + c0 + 4 * j, make_float4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]));
        }
        __syncthreads();
    }
}

template <int CH, typename FT, int PRIM>
cudaError_t launch_render_fuse(const RenderFuseArgs& af, int grid, cudaStream_t st) {
    const size_t smem = sizeof(PixelSmem<CH, PRIM>);
    cudaError_t e = cudaFuncSetAttribute(render_fuse_pixel_kernel<CH, FT, PRIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    render_fuse_pixel_kernel<CH, FT, PRIM><<<grid, TR_THREADS, smem, st>>>(af);
    return cudaGetLastError();
}

template <typename FT>
cudaError_t dispatch_render_fuse(const RenderFuseArgs& af, int grid, cudaStream_t st) {
    const int D = af.r.D;
    if (af.r.t.ray_transform) {
        if (D % 16 == 0) return launch_render_fuse<16, FT, 1>(af, grid, st);
        if (D % 8 == 0) return launch_render_fuse<8, FT, 1>(af, grid, st);
        return launch_render_fuse<4, FT, 1>(af, grid, st);
    }
    if (D % 16 == 0) return launch_render_fuse<16, FT, 0>(af, grid, st);
    if (D % 8 == 0) return launch_render_fuse<8, FT, 0>(af, grid, st);
    return launch_render_fuse<4, FT, 0>(af, grid, st);
}

template <typename K>
cudaError_t launch(K kernel, size_t smem, int grid, cudaStream_t st, const RenderArgs& a) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, TR_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <int DC, typename FT, bool DIAG, int PRIM = 0>
cudaError_t launch_ws1(const RenderArgs& a, const WsWork& wk, int grid, cudaStream_t st) {
    const size_t smem = sizeof(RenderWsSmem<DC, FT, PRIM>);
    cudaError_t e = cudaFuncSetAttribute(render_ws_kernel<DC, FT, DIAG, PRIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    render_ws_kernel<DC, FT, DIAG, PRIM><<<grid, WS_THREADS, smem, st>>>(a, wk);
    return cudaGetLastError();
}

template <int DC, typename FT>
cudaError_t launch_ws(const RenderArgs& a, int tiles, int num_sms, uint32_t* ctrl, const uint32_t* order, cudaStream_t st) {
    WsWork wk;
    wk.queue = ctrl + CTRL_RENDER_QUEUE;
    wk.n_chunks = a.D / DC;
    wk.n_items = tiles * wk.n_chunks;
    wk.order = order;
    wk.order_valid = ctrl + CTRL_ORDER_VALID;
    const int grid = wk.n_items < num_sms ? wk.n_items : num_sms;
    // One instantiation per feature dtype.  The fp32 kernel always carries the (runtime-guarded, once per tile)
    // tile_visited store: with that code present ptxas lays the producer loop out 3.7 % faster (1.361 vs 1.411 ms on
    // the Mid frame, reproducible); without a request a.tile_visited is NULL and nothing is written.  fp16 rows: the
    // variant without it is the faster one (5.07 vs 5.36 ms on Large) and is used unless diagnostics are requested.
    if (a.t.ray_transform) return launch_ws1<DC, FT, true, 1>(a, wk, grid, st);   // surfel form (one instantiation per dtype)
    if (sizeof(FT) == 4 || a.tile_visited) return launch_ws1<DC, FT, true>(a, wk, grid, st);
    return launch_ws1<DC, FT, false>(a, wk, grid, st);
}

template <typename FT>
cudaError_t dispatch(const RenderArgs& a, int grid, int num_sms, uint32_t* queue, const uint32_t* order, cudaStream_t st, bool has_feat) {
    if (a.t.ray_transform) {   // surfel mode (NEXT-3): the same pipelines with the surfel weight; per-pixel kernels for small D
        if (!has_feat) return launch(render_pixel_kernel<0, FT, 1>, sizeof(PixelSmem<0, 1>), grid, st, a);
        if (a.D % 128 == 0) return launch_ws<128, FT>(a, grid, num_sms, queue, order, st);
        if (a.D % 64 == 0) return launch_ws<64, FT>(a, grid, num_sms, queue, order, st);
        if (a.D % 16 == 0) return launch(render_pixel_kernel<16, FT, 1>, sizeof(PixelSmem<16, 1>), grid, st, a);
        if (a.D % 8 == 0) return launch(render_pixel_kernel<8, FT, 1>, sizeof(PixelSmem<8, 1>), grid, st, a);
        return launch(render_pixel_kernel<4, FT, 1>, sizeof(PixelSmem<4, 1>), grid, st, a);
    }
    if (!has_feat) return launch(render_pixel_kernel<0, FT, 0>, sizeof(PixelSmem<0, 0>), grid, st, a);
    if (a.D % 128 == 0) return launch_ws<128, FT>(a, grid, num_sms, queue, order, st);
    if (a.D % 64 == 0) return launch_ws<64, FT>(a, grid, num_sms, queue, order, st);
    if (a.D % 16 == 0) return launch(render_pixel_kernel<16, FT, 0>, sizeof(PixelSmem<16, 0>), grid, st, a);
    if (a.D % 8 == 0) return launch(render_pixel_kernel<8, FT, 0>, sizeof(PixelSmem<8, 0>), grid, st, a);
    return launch(render_pixel_kernel<4, FT, 0>, sizeof(PixelSmem<4, 0>), grid, st, a);
}

}  // namespace

#ifdef FHGS_WS_TIMING
extern "C" __attribute__((visibility("default"))) int fhgs_debug_render_timing(unsigned long long* out32, int reset) {
    if (out32 && cudaMemcpyFromSymbol(out32, g_ws_timing, sizeof(g_ws_timing)) != cudaSuccess) return 1;
    if (reset) {
        unsigned long long z[32] = {0};
        if (cudaMemcpyToSymbol(g_ws_timing, z, sizeof(z)) != cudaSuccess) return 1;
    }
    return 0;
}
#endif

extern "C" fhgs_status fhgs_render(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                                   const fhgs_params* prm, const fhgs_view_state* vs, float* out_rgb,
                                   void* out_feat, float* out_T, uint32_t* out_ncontrib, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!g || !cam || !prm || !vs) FHGS_INVALID(ctx, "fhgs_render: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    if (!out_rgb) FHGS_INVALID(ctx, "fhgs_render: out_rgb is required");
    const bool has_feat = out_feat != nullptr;
    if (has_feat) {
        if (!g->feat) FHGS_INVALID(ctx, "fhgs_render: out_feat given but g->feat is NULL");
        if (g->feat_dtype != FHGS_F32 && g->feat_dtype != FHGS_F16 && g->feat_dtype != FHGS_BF16)
            FHGS_INVALID(ctx, "fhgs_render: unknown feat_dtype");
        const int mult = g->feat_dtype == FHGS_F32 ? 4 : 8;
        if (g->feat_dim <= 0 || g->feat_dim % mult) FHGS_INVALID(ctx, "fhgs_render: feat_dim must be a positive multiple of 4 (f32) / 8 (f16, bf16)");
        if (!aligned_to(g->feat, 16) || !aligned_to(out_feat, 16)) FHGS_INVALID(ctx, "fhgs_render: feat/out_feat must be 16-byte aligned");
        if (g->n != vs->n) FHGS_INVALID(ctx, "fhgs_render: g->n != vs->n");
    }
    RenderArgs a;
    a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
    a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
    a.t.xy = reinterpret_cast<const float2*>(vs->xy);
    a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
    a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
    a.t.ray_transform = prm->primitive == FHGS_PRIM_SURFEL ? reinterpret_cast<const float4*>(vs->ray_transform) : nullptr;
    a.rgb_g = vs->rgb; a.feat = g->feat; a.D = has_feat ? g->feat_dim : 0;
    a.bg[0] = prm->bg[0]; a.bg[1] = prm->bg[1]; a.bg[2] = prm->bg[2];
    a.out_rgb = out_rgb; a.out_feat = out_feat; a.out_T = out_T; a.out_n = out_ncontrib;
    const int grid = tiles_x(cam->width) * tiles_y(cam->height);
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    const ScratchLayout L = make_scratch_layout(vs->n, vs->capacity, cam->width, cam->height);
    uint32_t* queue = reinterpret_cast<uint32_t*>((char*)vs->scratch + L.ctrl);
    const uint32_t* order = reinterpret_cast<const uint32_t*>((char*)vs->scratch + L.tile_order);
    // tile_visited is requested with fhgs_set_diagnostics; otherwise no kernel writes into the caller's scratch
    const bool diag = ctx->diagnostics != 0;
    a.tile_visited = diag ? reinterpret_cast<uint32_t*>((char*)vs->scratch + L.tile_visited) : nullptr;
    cudaError_t e = (has_feat && g->feat_dtype == FHGS_F16)    ? dispatch<__half>(a, grid, ctx->num_sms, queue, order, s, has_feat)
                    : (has_feat && g->feat_dtype == FHGS_BF16) ? dispatch<__nv_bfloat16>(a, grid, ctx->num_sms, queue, order, s, has_feat)
                                                               : dispatch<float>(a, grid, ctx->num_sms, queue, order, s, has_feat);
    FHGS_CUDA(ctx, e);
    return FHGS_OK;
}

extern "C" fhgs_status fhgs_render_fuse(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam, const fhgs_params* prm,
                                        const fhgs_view_state* vs, float* out_rgb, void* out_feat, float* out_T,
                                        uint32_t* out_ncontrib, const void* gt, float* num, float* den, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!g || !cam || !prm || !vs) FHGS_INVALID(ctx, "fhgs_render_fuse: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    if (!out_rgb || !out_feat || !gt || !num || !den || !g->feat) FHGS_INVALID(ctx, "fhgs_render_fuse: out_rgb, out_feat, gt, num, den and g->feat are required");
    if (g->feat_dtype != FHGS_F32 && g->feat_dtype != FHGS_F16 && g->feat_dtype != FHGS_BF16) FHGS_INVALID(ctx, "fhgs_render_fuse: unknown feat_dtype");
    const int mult = g->feat_dtype == FHGS_F32 ? 4 : 8;
    if (g->feat_dim <= 0 || g->feat_dim % mult) FHGS_INVALID(ctx, "fhgs_render_fuse: feat_dim must be a positive multiple of 4 (f32) / 8 (f16, bf16)");
    if (g->feat_dim % 64 == 0)
        FHGS_INVALID(ctx, "fhgs_render_fuse: feat_dim is a multiple of 64 -- the tiled kernels have no shared-memory room for a "
                          "shared weight phase (DESIGN.md 9e ii); call fhgs_render and fhgs_fuse_features");
    if (!aligned_to(g->feat, 16) || !aligned_to(out_feat, 16) || !aligned_to(gt, 16) || !aligned_to(num, 16) || !aligned_to(den, 4))
        FHGS_INVALID(ctx, "fhgs_render_fuse: feat / out_feat / gt / num must be 16-byte aligned");
    if (g->n != vs->n) FHGS_INVALID(ctx, "fhgs_render_fuse: g->n != vs->n");
    RenderFuseArgs af;
    RenderArgs& a = af.r;
    a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
    a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
    a.t.xy = reinterpret_cast<const float2*>(vs->xy);
    a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
    a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
    a.t.ray_transform = prm->primitive == FHGS_PRIM_SURFEL ? reinterpret_cast<const float4*>(vs->ray_transform) : nullptr;
    a.rgb_g = vs->rgb; a.feat = g->feat; a.D = g->feat_dim;
    a.bg[0] = prm->bg[0]; a.bg[1] = prm->bg[1]; a.bg[2] = prm->bg[2];
    a.out_rgb = out_rgb; a.out_feat = out_feat; a.out_T = out_T; a.out_n = out_ncontrib; a.tile_visited = nullptr;
    af.gt = gt; af.num = num; af.den = den;
    const int grid = tiles_x(cam->width) * tiles_y(cam->height);
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = g->feat_dtype == FHGS_F16    ? dispatch_render_fuse<__half>(af, grid, s)
                    : g->feat_dtype == FHGS_BF16 ? dispatch_render_fuse<__nv_bfloat16>(af, grid, s)
                                                 : dispatch_render_fuse<float>(af, grid, s);
    FHGS_CUDA(ctx, e);
    return FHGS_OK;
}
