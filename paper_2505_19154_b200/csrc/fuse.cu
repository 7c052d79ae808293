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
#include "layout.cuh"
#include "ws.cuh"

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
__device__ __forceinline__ float4 load_gt4<__half>(const __half* p) { return cvt16x4(__ldg(reinterpret_cast<const uint2*>(p)), p); }
template <>
__device__ __forceinline__ float4 load_gt4<__nv_bfloat16>(const __nv_bfloat16* p) {
    return cvt16x4(__ldg(reinterpret_cast<const uint2*>(p)), p);
}

template <int DC, int PRIM>
struct FuseTiledSmem {
    TileQueueT<PRIM> q;
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

template <int DC, typename GT, int PRIM>
__global__ void __launch_bounds__(TR_THREADS, 1) fuse_tiled_kernel(const FuseArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FuseTiledSmem<DC, PRIM>& sm = *reinterpret_cast<FuseTiledSmem<DC, PRIM>*>(smem_raw);

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
                sm.W[kk * TR_THREADS + tid] = eval_weight_q<PRIM>(sm.q, s, fx, fy, a.t, T, done, n);
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
// WS variant (fp32 map, D multiple of 128): warp-specialised persistent pipeline (ws.cuh)
//   warps 0-7   consumers: num[32 inst, 128 ch] += W^T G for one batch.  Thread = 8 instances x 4
//               channels over one HALF of the tile's pixels (warps 0-3: pixels 0-127, warps 4-7:
//               128-255); per pixel 1 LDS.128 of G + 2 LDS.128 of W (each one wavefront) feed 16
//               packed FMAs (fma.rn.f32x2, instance pairs packed).  The two halves are combined
//               through shared memory (roles alternate per batch) and leave as one
//               red.global.add.v4.f32 per (tile, Gaussian, 4 channels).
//   warps 8-15  producers: traversal, tile cull, blend weights -> W[stage][pixel][kk] (swizzled
//               float4 quads so that both sides are bank-conflict free).
//   warp 16     scheduler: pops (tile, chunk) items from the global queue, hands them to the
//               producers through a 2-deep ring, and -- once the consumers released the GT tile
//               of the previous item -- issues the bulk async copies of the next GT tile
//               (16 rows x 8 KB when D == 128) onto the g_full mbarrier.
// ---------------------------------------------------------------------------------------------
constexpr int FW_STAGES = 2;
constexpr int FW_DC = 128;
constexpr int FW_THREADS = WS_THREADS + 32;
constexpr int FW_WQ = (WS_CONS + 1) * 4;   // floats per quad row: 256 pixels x float4 + 16 B pad (bank spread over quads)
enum { FW_FLAG_FIRST = 4 };

// GT tile buffers: a 16-bit map leaves room for two (the scheduler loads the next item's tile while the consumers
// multiply the current one); an fp32 tile (128 KB) is single-buffered.
template <typename GT>
constexpr int kGBufs = sizeof(GT) == 2 ? 2 : 1;

// PRIM = 1 (surfel): three records per survivor; the ring shrinks to 288 slots (modulo wrap) to fit beside the fp32 tile
template <typename GT, int PRIM = 0>
struct FuseWsSmem {
    WsCtrl<FW_STAGES, PRIM, PRIM ? 288 : WS_QCAP> ct;
    uint64_t g_full[2][8], g_free[2];                      // g_full: one barrier per pixel half ([0], [4]) or, for a streamed-in
                                                          // tile, per 32 pixels (2 tile rows) of a GT buffer
    uint64_t item_full[2], item_empty[2];
    uint64_t p_full[2];                                   // the writing half's partial sums (and den atomics) of batch b are in place:
                                                          // [b & 1], phase (b >> 1) & 1 (two barriers: a warp may run one batch ahead)
    int items[2];
    __align__(16) uint32_t ids[FW_STAGES][WS_KB];
    __align__(16) float den_s[2][WS_KB];
    __align__(128) float W[FW_STAGES][FW_WQ * WS_KB / 4];  // [quad kk/4][pixel][4], quad stride padded by one float4
    __align__(128) float P[WS_KB * FW_DC];                // partial sums of the writing half
    __align__(128) GT G[kGBufs<GT>][WS_CONS * FW_DC];     // [buffer][pixel][channel], pixel = y*16 + x (storage type of the map)
    GT G_pad[FW_DC];                                      // target of the consumers' one-past-the-end prefetch
};

// 4 consecutive channels of the staged GT tile -> fp32 (exact for fp16 / bf16 storage)
__device__ __forceinline__ float4 ld_g4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 ld_g4(const __half* p) { return cvt16x4(*reinterpret_cast<const uint2*>(p), p); }
__device__ __forceinline__ float4 ld_g4(const __nv_bfloat16* p) { return cvt16x4(*reinterpret_cast<const uint2*>(p), p); }

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

template <typename GT, int PRIM>
__device__ __forceinline__ void fuse_ws_scheduler(FuseWsSmem<GT, PRIM>& sm, const FuseArgs& a, const WsWork& wk) {
    const int lane = threadIdx.x & 31;
    const GT* gt = reinterpret_cast<const GT*>(a.gt);
    int islot = 0, gb = 0;
    uint32_t iphase = 0, gphase = 0;
    while (true) {
        int item = 0;
        if (lane == 0) {
            item = (int)atomicAdd(wk.queue, 1u);
            mbar_wait_backoff(&sm.item_empty[islot], iphase ^ 1u);
            sm.items[islot] = item;
            mbar_arrive(&sm.item_full[islot]);
        }
        item = __shfl_sync(TR_FULL, item, 0);
        if (++islot == 2) { islot = 0; iphase ^= 1u; }
        if (item >= wk.n_items) break;
        const int tile = ws_item_tile(wk, item), c0 = (item % wk.n_chunks) * FW_DC;
        {
            const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
            if (range.x >= range.y) continue;   // empty tile: the producers skip it too
        }
        const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE;
        const int nx = min(FHGS_TILE, a.t.W - tx0), ny = min(FHGS_TILE, a.t.H - ty0);
#ifdef FHGS_NO_STREAM_IN
        const bool split = false;
#else
        const bool split = kGBufs<GT> == 1 && a.D != FW_DC;   // see fuse_ws_consumer
#endif
        if (lane == 0) {
            mbar_wait_backoff(&sm.g_free[gb], gphase ^ 1u);
            if (split) {   // one barrier per pair of tile rows: the consumers start on the first rows while the rest is in flight
#pragma unroll
                for (int b = 0; b < 8; ++b)
                    mbar_arrive_expect_tx(&sm.g_full[gb][b], (uint32_t)(nx * min(max(ny - 2 * b, 0), 2) * FW_DC * sizeof(GT)));
            } else {       // one barrier per pixel half
                mbar_arrive_expect_tx(&sm.g_full[gb][0], (uint32_t)(nx * min(ny, 8) * FW_DC * sizeof(GT)));
                mbar_arrive_expect_tx(&sm.g_full[gb][4], (uint32_t)(nx * max(ny - 8, 0) * FW_DC * sizeof(GT)));
            }
        }
        __syncwarp();
        GT* Gd = sm.G[gb];
        if (a.D == FW_DC) {   // a tile row is one contiguous span
            if (lane < ny)
                bulk_g2s(&Gd[lane * FHGS_TILE * FW_DC], gt + ((size_t)(ty0 + lane) * a.t.W + tx0) * FW_DC,
                         (uint32_t)(nx * FW_DC * sizeof(GT)), &sm.g_full[gb][(lane >> 3) * 4]);
        } else {
            for (int pix = lane; pix < FHGS_TILE_PX; pix += 32) {
                const int x = pix & 15, y = pix >> 4;
                if (x < nx && y < ny)
                    bulk_g2s(&Gd[pix * FW_DC], gt + ((size_t)(ty0 + y) * a.t.W + tx0 + x) * a.D + c0, (uint32_t)(FW_DC * sizeof(GT)),
                             &sm.g_full[gb][split ? pix >> 5 : (pix >> 7) * 4]);
            }
        }
        if (++gb == kGBufs<GT>) { gb = 0; gphase ^= 1u; }
    }
}

template <typename GT, int PRIM>
__device__ __forceinline__ void fuse_ws_producer(FuseWsSmem<GT, PRIM>& sm, const FuseArgs& a, const WsWork& wk) {
    using CT = decltype(sm.ct);
    const int p = threadIdx.x, lane = p & 31;   // producers are warps 0-7
    const float q_cutoff = a.t.q_cutoff, alpha_max = a.t.alpha_max, t_min = a.t.t_min;
    const int sx = p & 15, sy = p >> 4;   // row-major pixel slot (matches the GT tile rows)
    int stage = 0, islot = 0;
    uint32_t phase = 0, iphase = 0;
    WS_TDECL;
    while (true) {
        mbar_wait(&sm.item_full[islot], iphase);
        WS_TACC(0);
        const int item = sm.items[islot];
        mbar_arrive(&sm.item_empty[islot]);
        if (++islot == 2) { islot = 0; iphase ^= 1u; }
        if (item >= wk.n_items) {
            mbar_wait(&sm.ct.empty[stage], phase ^ 1u);
            if (p == 0) sm.ct.meta[stage] = WsMeta{0, -1, 0, WS_FLAG_EXIT};
            mbar_arrive(&sm.ct.full[stage]);
            break;
        }
        WS_TCNT(6);
        const int tile = ws_item_tile(wk, item), c0 = (item % wk.n_chunks) * FW_DC;
        const int tx0 = (tile % a.t.GW) * FHGS_TILE, ty0 = (tile / a.t.GW) * FHGS_TILE;
        const int px = tx0 + sx, py = ty0 + sy;
        const bool inside = px < a.t.W && py < a.t.H;
        WsPixel P{(float)px, (float)py, 1.f, 0u, !inside};
        const float bx0 = (float)tx0, by0 = (float)ty0;
        const float bx1 = (float)min(tx0 + FHGS_TILE - 1, a.t.W - 1), by1 = (float)min(ty0 + FHGS_TILE - 1, a.t.H - 1);
        const uint2 range = __ldg(reinterpret_cast<const uint2*>(a.t.ranges) + tile);
        if (range.x >= range.y) continue;   // empty tile (the scheduler loads no GT tile for it)
        uint32_t pos = range.x;
        int qh = 0, qt = 0;
        WsChunk ch;
        ws_chunk_prefetch_id(a.t, pos, range.y, p, ch);
        ws_chunk_issue(a.t, nullptr, ch);
        ws_chunk_prefetch_id(a.t, pos + WS_PROD, range.y, p, ch);
        bool last = false, first = true;
        do {
            while (qt - qh < WS_KB && pos < range.y) {
                qt += ws_chunk_append<PRIM>(sm.ct, ch, pos, qt, bx0, by0, bx1, by1, q_cutoff, p, [](int, const WsChunk&) {},
                                            a.t.ray_transform);
                pos += WS_PROD;
                ws_chunk_issue(a.t, nullptr, ch);
                ws_chunk_prefetch_id(a.t, pos + WS_PROD, range.y, p, ch);
            }
            const int nb = min(WS_KB, qt - qh);
            WS_TACC(1);
            mbar_wait_backoff(&sm.ct.empty[stage], phase ^ 1u);
            WS_TACC(2);
            WS_TCNT(5);
            if (p < WS_KB) sm.ids[stage][p] = p < nb ? __float_as_uint(sm.ct.rec1[CT::slot(qh + p)].z) : 0u;
            float* Wd = sm.W[stage] + p * 4;
            const bool warp_done = __all_sync(TR_FULL, P.done);
#pragma unroll 2
            for (int kq = 0; kq < WS_KB / 4; ++kq) {
                float w4[4] = {0.f, 0.f, 0.f, 0.f};
                if (!warp_done && kq * 4 < nb) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int kk = kq * 4 + j;
                        const int s = CT::slot(qh + kk);
                        const float4 r0 = sm.ct.rec0[s];
                        const float4 r1 = sm.ct.rec1[s];
                        WsPixel Q = P;
                        const float w = PRIM ? ws_weight_surfel(r0, r1, sm.ct.rec2[PRIM ? s : 0], Q, q_cutoff, alpha_max, t_min)
                                             : ws_weight(r0, r1.x, r1.y, Q, q_cutoff, alpha_max, t_min);
                        if (kk < nb) { P = Q; w4[j] = w; }
                    }
                }
                *reinterpret_cast<float4*>(Wd + kq * FW_WQ) = make_float4(w4[0], w4[1], w4[2], w4[3]);
            }
            qh += nb;
            WS_TACC(3);
            const bool all_done = named_bar_and(WS_BAR_PROD_RED, WS_PROD, P.done);
            last = all_done || (pos >= range.y && qt == qh);
            if (p == 0) sm.ct.meta[stage] = WsMeta{nb, tile, c0, (last ? WS_FLAG_LAST : 0) | (first ? FW_FLAG_FIRST : 0)};
            first = false;
            mbar_arrive(&sm.ct.full[stage]);
            WS_TACC(4);
            if (++stage == FW_STAGES) { stage = 0; phase ^= 1u; }
        } while (!last);
    }
    WS_TFLUSH(16, p == 0);
    (void)lane;
}

template <typename GT, int PRIM>
__device__ __forceinline__ void fuse_ws_consumer(FuseWsSmem<GT, PRIM>& sm, const FuseArgs& a) {
    // consumers are warps 8-15: the SMSP arbiter favours high warp ids and the consumers are the critical path
    const int tid = threadIdx.x - WS_PROD, lane = tid & 31, warp = tid >> 5;
    const int half = warp >> 2, cw = warp & 3;
    const int kg = warp & 3;                  // the warp's 8 instances of the batch (a short batch idles whole warps)
    const int ch = lane * 4;                  // this thread's 4 channels inside the chunk
    int stage = 0, gb = kGBufs<GT> - 1;
    uint32_t phase = 0, gphase = 1u, batch = 0;   // (gb, gphase) advance to buffer 0 / parity 0 at the first item
    const GT* Gs = sm.G[0] + half * 128 * FW_DC + ch;
    WS_TDECL;
    while (true) {
        mbar_wait(&sm.ct.full[stage], phase);
        WS_TACC(0);
        const WsMeta m = sm.ct.meta[stage];
        if (m.flags & WS_FLAG_EXIT) break;
        // A single-buffered tile that arrives as 256 per-pixel copies (fp32 map, D > 128) is consumed block by block as it
        // lands (Multi-view: fuse -3.5 %); where the tile is one copy per row or double-buffered the extra waits only cost
        // (Mid +3 %), so everything is awaited up front there.
        const bool first = (m.flags & FW_FLAG_FIRST) != 0;
#ifdef FHGS_NO_STREAM_IN
        const bool stream_in = false;
#else
        const bool stream_in = first && kGBufs<GT> == 1 && a.D != FW_DC;
#endif
        if (first) {   // next item: its GT tile is in the next buffer
            if (++gb == kGBufs<GT>) { gb = 0; gphase ^= 1u; }
            mbar_wait(&sm.g_full[gb][half * 4], gphase);
            if (stream_in) mbar_wait(&sm.g_full[gb][half * 4 + 1], gphase);
            Gs = sm.G[gb] + half * 128 * FW_DC + ch;
            WS_TACC(1);
        }
        WS_TCNT(5);
        uint32_t id[8];
        {
            const uint4 i0 = *reinterpret_cast<const uint4*>(&sm.ids[stage][kg * 8]);
            const uint4 i1 = *reinterpret_cast<const uint4*>(&sm.ids[stage][kg * 8 + 4]);
            id[0] = i0.x; id[1] = i0.y; id[2] = i0.z; id[3] = i0.w;
            id[4] = i1.x; id[5] = i1.y; id[6] = i1.z; id[7] = i1.w;
        }
        unsigned long long acc[4][4];   // [instance pair][channel], packed (inst 2i, inst 2i+1)
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[i][c] = 0ull;
        // W for pixel s, instances 8 kg .. 8 kg + 7: two float4 at fixed offsets from one base -> no address arithmetic
        const float* Ws = sm.W[stage] + (2 * kg) * FW_WQ + half * 128 * 4;
        // software-pipelined over pixels: the operands of pixel s+1 are in flight while pixel s is multiplied
        ulonglong2 wa = *reinterpret_cast<const ulonglong2*>(Ws);
        ulonglong2 wb = *reinterpret_cast<const ulonglong2*>(Ws + FW_WQ);
        float4 g = ld_g4(Gs);
#pragma unroll 1
        for (int s0 = 0; s0 < (kg * 8 < m.nb ? 128 : 0); s0 += 32) {
            // first batch of an item: the block after this one (its first pixel is prefetched at the end of this block)
            if (stream_in && s0 >= 32 && s0 < 96) mbar_wait(&sm.g_full[gb][half * 4 + (s0 >> 5) + 1], gphase);
            const float* Wb = Ws + s0 * 4;
            const GT* Gb = Gs + s0 * FW_DC;
#pragma unroll
            for (int u = 0; u < 32; ++u) {
                const int un = u + 1;   // the prefetch past the last pixel lands in the row pad / G_pad (never used)
                const ulonglong2 wa_n = *reinterpret_cast<const ulonglong2*>(Wb + un * 4);
                const ulonglong2 wb_n = *reinterpret_cast<const ulonglong2*>(Wb + FW_WQ + un * 4);
                const float4 g_n = ld_g4(Gb + un * FW_DC);
                const unsigned long long g2[4] = {pack2(g.x, g.x), pack2(g.y, g.y), pack2(g.z, g.z), pack2(g.w, g.w)};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    fma2_acc(acc[0][c], wa.x, g2[c]);
                    fma2_acc(acc[1][c], wa.y, g2[c]);
                    fma2_acc(acc[2][c], wb.x, g2[c]);
                    fma2_acc(acc[3][c], wb.y, g2[c]);
                }
                wa = wa_n; wb = wb_n; g = g_n;
            }
        }
        // a warp that had no instances in the first batch skipped the loop and its waits: every warp must have seen the whole
        // tile before it goes on (the later batches of the item do not wait)
        if (stream_in) {
            mbar_wait(&sm.g_full[gb][half * 4 + 2], gphase);
            mbar_wait(&sm.g_full[gb][half * 4 + 3], gphase);
        }
        WS_TACC(2);
        // den partial: warp (half, cw) sums pixels [128 half + 32 cw, +32) for instance kk = lane
        {
            const float* Wp = sm.W[stage] + (lane >> 2) * FW_WQ + (half * 128 + cw * 32) * 4 + (lane & 3);
            float d0 = 0.f, d1 = 0.f;
#pragma unroll
            for (int j = 0; j < 32; j += 2) { d0 += Wp[j * 4]; d1 += Wp[j * 4 + 4]; }
            atomicAdd(&sm.den_s[batch & 1][lane], d0 + d1);
        }
        const bool writer = ((batch & 1u) != 0u) == (half != 0);
        // The reading half releases the W stage at once; the writing half releases it after it has signalled p_full (below):
        // no consumer warp can then be two batches ahead of another one's p_full arrival (the stage it needs is refilled
        // only after every consumer released it), so an arrival never lands in an older phase of the barrier.
        if (!writer) mbar_arrive(&sm.ct.empty[stage]);
        if (m.flags & WS_FLAG_LAST) mbar_arrive(&sm.g_free[gb]);   // done with the GT tile: the scheduler may load the next one
        WS_TACC(3);
        if (writer) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 v0 = unpack2(acc[i][0]), v1 = unpack2(acc[i][1]), v2 = unpack2(acc[i][2]), v3 = unpack2(acc[i][3]);
                *reinterpret_cast<float4*>(&sm.P[(kg * 8 + 2 * i) * FW_DC + ch]) = make_float4(v0.x, v1.x, v2.x, v3.x);
                *reinterpret_cast<float4*>(&sm.P[(kg * 8 + 2 * i + 1) * FW_DC + ch]) = make_float4(v0.y, v1.y, v2.y, v3.y);
            }
        }
        // The halves are not barrier-coupled: the writing half signals p_full and goes on to the next batch, the reading
        // half waits for it (phase = batch parity), so one half's epilogue overlaps the other half's next product.
        // P needs no second buffer: a thread writes exactly the addresses it read one batch earlier, and it cannot get two
        // batches ahead of the other half because as next batch's reader it waits for that half's signal; den_s[b & 1]
        // is cleared by the reader of batch b before that reader signals batch b + 1.
        if (writer) {
            mbar_arrive(&sm.p_full[batch & 1u]);
            mbar_arrive(&sm.ct.empty[stage]);
        } else {
            mbar_wait(&sm.p_full[batch & 1u], (batch >> 1) & 1u);
            asm volatile("bar.sync %0, %1;" ::"r"(4 + half), "r"(128) : "memory");   // this half's own den atomics
            const float4 d0 = *reinterpret_cast<const float4*>(&sm.den_s[batch & 1][kg * 8]);
            const float4 d1 = *reinterpret_cast<const float4*>(&sm.den_s[batch & 1][kg * 8 + 4]);
            const float dv[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 v0 = unpack2(acc[i][0]), v1 = unpack2(acc[i][1]), v2 = unpack2(acc[i][2]), v3 = unpack2(acc[i][3]);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int k8 = 2 * i + e, kk = kg * 8 + k8;
                    if (kk < m.nb && dv[k8] != 0.f) {
                        const float4 pp = *reinterpret_cast<const float4*>(&sm.P[kk * FW_DC + ch]);
                        const float4 mine = e ? make_float4(v0.y, v1.y, v2.y, v3.y) : make_float4(v0.x, v1.x, v2.x, v3.x);
                        red_add_v4(a.num + (size_t)id[k8] * a.D + m.c0 + ch,
                                   make_float4(mine.x + pp.x, mine.y + pp.y, mine.z + pp.z, mine.w + pp.w));
                        if (m.c0 == 0 && ch == 0) red_add(a.den + id[k8], dv[k8]);
                    }
                }
            }
            // all four channel warps of this half must have read den_s before it is cleared
            asm volatile("bar.sync %0, %1;" ::"r"(4 + half), "r"(128) : "memory");
            if (cw == 0) sm.den_s[batch & 1][lane] = 0.f;
        }
        if (++stage == FW_STAGES) { stage = 0; phase ^= 1u; }
        WS_TACC(4);
        ++batch;
    }
    WS_TFLUSH(0, tid == 0);
}


template <typename GT, int PRIM = 0>
__global__ void __launch_bounds__(FW_THREADS, 1) fuse_ws_kernel(const FuseArgs a, const WsWork wk) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FuseWsSmem<GT, PRIM>& sm = *reinterpret_cast<FuseWsSmem<GT, PRIM>*>(smem_raw);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < FW_STAGES; ++s) {
            mbar_init(&sm.ct.full[s], WS_PROD);
            mbar_init(&sm.ct.empty[s], WS_CONS);
        }
        for (int s = 0; s < 2; ++s) {
            for (int b = 0; b < 8; ++b) mbar_init(&sm.g_full[s][b], 1);
            mbar_init(&sm.g_free[s], WS_CONS);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&sm.item_full[s], 1);
            mbar_init(&sm.item_empty[s], WS_PROD);
        }
        mbar_init(&sm.p_full[0], WS_CONS / 2);
        mbar_init(&sm.p_full[1], WS_CONS / 2);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // the GT tile buffer must never hold non-finite garbage (pixels outside the image keep stale data, weight 0)
    for (int i = threadIdx.x; i < (int)((kGBufs<GT> * WS_CONS + 1) * FW_DC * sizeof(GT) / 16); i += FW_THREADS)
        reinterpret_cast<uint4*>(&sm.G[0][0])[i] = make_uint4(0u, 0u, 0u, 0u);
    if (threadIdx.x < 2 * WS_KB) (&sm.den_s[0][0])[threadIdx.x] = 0.f;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (threadIdx.x >= WS_THREADS) {
        fuse_ws_scheduler(sm, a, wk);
    } else if (threadIdx.x < WS_PROD) {
        fuse_ws_producer(sm, a, wk);
    } else {
        fuse_ws_consumer(sm, a);
        if (threadIdx.x == WS_PROD) ws_queue_release(wk);
    }
}

// ---------------------------------------------------------------------------------------------
// PIXEL variant: CH channels per pass held by the pixel's thread; warp-segment reduction
// ---------------------------------------------------------------------------------------------
template <int PRIM>
struct FusePixelSmem {
    TileQueueT<PRIM> q;
};

template <int CH, typename GT, int PRIM>
__global__ void __launch_bounds__(TR_THREADS) fuse_pixel_kernel(const FuseArgs a) {
    __shared__ FusePixelSmem<PRIM> sm;
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
                const float w = eval_weight_q<PRIM>(sm.q, s, fx, fy, a.t, T, done, n);
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
// finalise / sparse clear.  Only a few per cent of the rows carry weight (Mid: 22 188 of 10^6), so a warp first looks at
// 32 consecutive den values at once (one coalesced load) and then walks only the rows that need work.
// ---------------------------------------------------------------------------------------------
constexpr int ROWS_PER_WARP = 32, ROW_WARPS = 8;   // 256 rows per CTA

// one float4 of a finalised row in the storage type of out_feat (16-bit types: round to nearest even)
__device__ __forceinline__ void store_out4(float* out, size_t i4, float4 v) { reinterpret_cast<float4*>(out)[i4] = v; }
__device__ __forceinline__ void store_out4(__half* out, size_t i4, float4 v) { reinterpret_cast<uint2*>(out)[i4] = pack16x4(v, out); }
__device__ __forceinline__ void store_out4(__nv_bfloat16* out, size_t i4, float4 v) { reinterpret_cast<uint2*>(out)[i4] = pack16x4(v, out); }

template <typename OT>
__global__ void __launch_bounds__(256) finalize_kernel(int n, int D, const float* num, const float* den, float den_eps,
                                                       int l2norm, OT* out) {
    const int lane = threadIdx.x & 31;
    const int row0 = (blockIdx.x * ROW_WARPS + (threadIdx.x >> 5)) * ROWS_PER_WARP;
    if (row0 >= n) return;
    const float dl = row0 + lane < n ? __ldg(den + row0 + lane) : 0.f;
    uint32_t live = __ballot_sync(TR_FULL, dl > den_eps);
    const int n4 = D >> 2;
    while (live) {
        const int r = __ffs(live) - 1;
        live &= live - 1u;
        const int row = row0 + r;
        const float d = __shfl_sync(TR_FULL, dl, r);
        const float4* src = reinterpret_cast<const float4*>(num + (size_t)row * D);
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
            store_out4(out, (size_t)row * n4 + j, make_float4(x, y, z, w));
        }
    }
}

// FHGS_FUSE_ZERO_TOUCHED: clear only the rows that carry weight (den != 0).
__global__ void __launch_bounds__(256) zero_touched_kernel(int n, int D, float* num, float* den) {
    const int lane = threadIdx.x & 31;
    const int row0 = (blockIdx.x * ROW_WARPS + (threadIdx.x >> 5)) * ROWS_PER_WARP;
    if (row0 >= n) return;
    const bool mine = row0 + lane < n && den[row0 + lane] != 0.f;
    uint32_t live = __ballot_sync(TR_FULL, mine);
    if (mine) den[row0 + lane] = 0.f;
    while (live) {
        const int r = __ffs(live) - 1;
        live &= live - 1u;
        float4* dst = reinterpret_cast<float4*>(num + (size_t)(row0 + r) * D);
        for (int j = lane; j < (D >> 2); j += 32) dst[j] = make_float4(0.f, 0.f, 0.f, 0.f);
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

template <typename GT, int PRIM = 0>
cudaError_t launch_fuse_ws(const FuseArgs& a, int tiles, int num_sms, uint32_t* ctrl, const uint32_t* order, cudaStream_t st) {
    const size_t smem = sizeof(FuseWsSmem<GT, PRIM>);
    static_assert(sizeof(FuseWsSmem<GT, PRIM>) <= 232448, "fuse_ws shared memory exceeds 227 KB");
    cudaError_t e = cudaFuncSetAttribute(fuse_ws_kernel<GT, PRIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    WsWork wk;
    wk.queue = ctrl + CTRL_FUSE_QUEUE;
    wk.n_chunks = a.D / FW_DC;
    wk.n_items = tiles * wk.n_chunks;
    wk.order = order;
    wk.order_valid = ctrl + CTRL_ORDER_VALID;
    const int grid = wk.n_items < num_sms ? wk.n_items : num_sms;
    fuse_ws_kernel<GT, PRIM><<<grid, FW_THREADS, smem, st>>>(a, wk);
    return cudaGetLastError();
}

template <typename GT>
cudaError_t dispatch(const FuseArgs& a, int grid, int num_sms, uint32_t* queue, const uint32_t* order, cudaStream_t st) {
    if (a.t.ray_transform) {   // surfel mode (NEXT-3): the same pipeline with the surfel weight; tile-per-CTA kernels otherwise
        if (a.D % FW_DC == 0) return launch_fuse_ws<GT, 1>(a, grid, num_sms, queue, order, st);
        if (a.D % 64 == 0) return launch(fuse_tiled_kernel<64, GT, 1>, sizeof(FuseTiledSmem<64, 1>), grid, st, a);
        if (a.D % 16 == 0) return launch(fuse_pixel_kernel<16, GT, 1>, 0, grid, st, a);
        if (a.D % 8 == 0) return launch(fuse_pixel_kernel<8, GT, 1>, 0, grid, st, a);
        return launch(fuse_pixel_kernel<4, GT, 1>, 0, grid, st, a);
    }
    if (a.D % FW_DC == 0) return launch_fuse_ws<GT>(a, grid, num_sms, queue, order, st);
    if (a.D % 64 == 0) return launch(fuse_tiled_kernel<64, GT, 0>, sizeof(FuseTiledSmem<64, 0>), grid, st, a);
    if (a.D % 16 == 0) return launch(fuse_pixel_kernel<16, GT, 0>, 0, grid, st, a);
    if (a.D % 8 == 0) return launch(fuse_pixel_kernel<8, GT, 0>, 0, grid, st, a);
    return launch(fuse_pixel_kernel<4, GT, 0>, 0, grid, st, a);
}

}  // namespace

#ifdef FHGS_WS_TIMING
extern "C" __attribute__((visibility("default"))) int fhgs_debug_fuse_timing(unsigned long long* out32, int reset) {
    if (out32 && cudaMemcpyFromSymbol(out32, g_ws_timing, sizeof(g_ws_timing)) != cudaSuccess) return 1;
    if (reset) {
        unsigned long long z[32] = {0};
        if (cudaMemcpyToSymbol(g_ws_timing, z, sizeof(z)) != cudaSuccess) return 1;
    }
    return 0;
}
#endif

extern "C" fhgs_status fhgs_fuse_features(fhgs_ctx* ctx, const fhgs_camera* cam, const fhgs_params* prm,
                                          const fhgs_view_state* vs, const void* gt, int32_t feat_dim,
                                          int32_t gt_dtype, float* num, float* den, void* out_feat,
                                          int32_t out_dtype, uint32_t flags, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!prm || !vs || !num || !den) FHGS_INVALID(ctx, "fhgs_fuse_features: NULL argument");
    if (flags & ~(uint32_t)(FHGS_FUSE_ZERO | FHGS_FUSE_FINALIZE | FHGS_FUSE_L2NORM | FHGS_FUSE_FINALIZE_ONLY | FHGS_FUSE_ZERO_ONLY |
                            FHGS_FUSE_ZERO_TOUCHED))
        FHGS_INVALID(ctx, "fhgs_fuse_features: unknown flag");
    const bool zero_only = (flags & FHGS_FUSE_ZERO_ONLY) != 0;
    if (zero_only && (flags & ~(uint32_t)(FHGS_FUSE_ZERO_ONLY | FHGS_FUSE_ZERO_TOUCHED)))
        FHGS_INVALID(ctx, "fhgs_fuse_features: ZERO_ONLY excludes other flags (except ZERO_TOUCHED)");
    if ((flags & FHGS_FUSE_ZERO_TOUCHED) && !(flags & (FHGS_FUSE_ZERO | FHGS_FUSE_ZERO_ONLY)))
        FHGS_INVALID(ctx, "fhgs_fuse_features: ZERO_TOUCHED qualifies ZERO / ZERO_ONLY");
    const bool accumulate = !(flags & (FHGS_FUSE_FINALIZE_ONLY | FHGS_FUSE_ZERO_ONLY));
    const bool finalize = (flags & (FHGS_FUSE_FINALIZE | FHGS_FUSE_FINALIZE_ONLY)) != 0;
    fhgs_status st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if (gt_dtype != FHGS_F32 && gt_dtype != FHGS_F16 && gt_dtype != FHGS_BF16) FHGS_INVALID(ctx, "fhgs_fuse_features: unknown gt_dtype");
    if (out_dtype != FHGS_F32 && out_dtype != FHGS_F16 && out_dtype != FHGS_BF16) FHGS_INVALID(ctx, "fhgs_fuse_features: unknown out_dtype");
    const int mult = (accumulate && gt_dtype != FHGS_F32) ? 8 : 4;
    if (feat_dim <= 0 || feat_dim % mult) FHGS_INVALID(ctx, "fhgs_fuse_features: feat_dim must be a positive multiple of 4 (f32) / 8 (f16, bf16)");
    if (!aligned_to(num, 16) || !aligned_to(den, 4)) FHGS_INVALID(ctx, "fhgs_fuse_features: num must be 16-byte aligned");
    if (vs->n < 0) FHGS_INVALID(ctx, "fhgs_fuse_features: vs->n < 0");
    if (accumulate) {
        if (!cam || !gt) FHGS_INVALID(ctx, "fhgs_fuse_features: cam and gt are required unless FINALIZE_ONLY");
        if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
        if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
        if (!aligned_to(gt, 16)) FHGS_INVALID(ctx, "fhgs_fuse_features: gt must be 16-byte aligned");
        if ((st = validate_primitive(ctx, prm, vs)) != FHGS_OK) return st;
    }
    if (finalize) {
        if (!out_feat) FHGS_INVALID(ctx, "fhgs_fuse_features: FINALIZE needs out_feat");
        if (!aligned_to(out_feat, 16)) FHGS_INVALID(ctx, "fhgs_fuse_features: out_feat must be 16-byte aligned");
    }
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = (size_t)vs->n;
    if ((flags & (FHGS_FUSE_ZERO | FHGS_FUSE_ZERO_ONLY)) && n > 0) {
        if (flags & FHGS_FUSE_ZERO_TOUCHED) {
            zero_touched_kernel<<<(int)((n + ROWS_PER_WARP * ROW_WARPS - 1) / (ROWS_PER_WARP * ROW_WARPS)), 256, 0, s>>>((int)n, feat_dim, num, den);
            FHGS_LAUNCH_CHECK(ctx);
        } else {
            FHGS_CUDA(ctx, cudaMemsetAsync(num, 0, n * feat_dim * sizeof(float), s));
            FHGS_CUDA(ctx, cudaMemsetAsync(den, 0, n * sizeof(float), s));
        }
    }
    if (accumulate && n > 0) {
        FuseArgs a;
        a.t.W = cam->width; a.t.H = cam->height; a.t.GW = tiles_x(cam->width);
        a.t.ranges = vs->ranges; a.t.vals = vs->vals[vs->sorted_buf & 1];
        a.t.xy = reinterpret_cast<const float2*>(vs->xy);
        a.t.conic_opacity = reinterpret_cast<const float4*>(vs->conic_opacity);
        a.t.q_cutoff = prm->q_cutoff; a.t.alpha_max = prm->alpha_max; a.t.t_min = prm->t_min;
        a.t.ray_transform = prm->primitive == FHGS_PRIM_SURFEL ? reinterpret_cast<const float4*>(vs->ray_transform) : nullptr;
        a.gt = gt; a.D = feat_dim; a.num = num; a.den = den;
        const int grid = tiles_x(cam->width) * tiles_y(cam->height);
        const ScratchLayout L = make_scratch_layout(vs->n, vs->capacity, cam->width, cam->height);
        uint32_t* queue = reinterpret_cast<uint32_t*>((char*)vs->scratch + L.ctrl);
        const uint32_t* order = reinterpret_cast<const uint32_t*>((char*)vs->scratch + L.tile_order);
        cudaError_t e = gt_dtype == FHGS_F16    ? dispatch<__half>(a, grid, ctx->num_sms, queue, order, s)
                        : gt_dtype == FHGS_BF16 ? dispatch<__nv_bfloat16>(a, grid, ctx->num_sms, queue, order, s)
                                                : dispatch<float>(a, grid, ctx->num_sms, queue, order, s);
        FHGS_CUDA(ctx, e);
    }
    if (finalize && n > 0) {
        const int grid = (int)((n + ROWS_PER_WARP * ROW_WARPS - 1) / (ROWS_PER_WARP * ROW_WARPS));
        const int l2 = (flags & FHGS_FUSE_L2NORM) ? 1 : 0;
        if (out_dtype == FHGS_F16)
            finalize_kernel<__half><<<grid, 256, 0, s>>>((int)n, feat_dim, num, den, prm->den_eps, l2, (__half*)out_feat);
        else if (out_dtype == FHGS_BF16)
            finalize_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>((int)n, feat_dim, num, den, prm->den_eps, l2, (__nv_bfloat16*)out_feat);
        else
            finalize_kernel<float><<<grid, 256, 0, s>>>((int)n, feat_dim, num, den, prm->den_eps, l2, (float*)out_feat);
        FHGS_LAUNCH_CHECK(ctx);
    }
    return FHGS_OK;
}
