// binsort.cu -- step S (fhgs_bin_sort): prefix sum + key duplication, onesweep radix sort, ranges.
// PAPER.md:302, 312-314 (DuplicateWithKeys, SortByKeys, IdentifyTileRanges); SURVEY 8(c) C1-S.
//
// Kernels
//   scan_dup_kernel    single-pass prefix sum of tiles_touched with decoupled look-back (one status
//                      word per CTA), fused with the emission of the (key,val) pairs: the CTA's
//                      instances are produced cooperatively (binary search of the instance index
//                      in the CTA-local prefix sums) so that a Gaussian covering thousands of
//                      tiles does not serialise one thread, and all key/value stores are
//                      coalesced.  The digit histograms of every later sort pass are accumulated
//                      here too (the keys are in registers anyway), saving one full read.
//   onesweep_kernel    one least-significant-digit pass (8-bit digit) of a STABLE radix sort:
//                      warp-synchronous match-any ranking, per-CTA digit counts published to a
//                      status array, chained look-back for the cross-CTA prefix, keys and values
//                      reordered through shared memory so that global stores are coalesced per
//                      digit run.  CTA ids come from an atomic ticket so that a CTA only ever
//                      waits on CTAs that already started.
//   ranges_kernel      tile boundaries of the sorted keys.
//
// Two equivalent schedules (both give the unique sorted list of C1-S step 3):
//   FHGS_SORT_FULL_KEY  LSD passes over all significant bits of the 64-bit keys
//                       (32 + ceil(log2(GW*GH)) bits -> 6 passes at 1080p).
//   default             order the Gaussians by (depth bits, index) first -- 4 passes over N
//                       32-bit keys, ~30x fewer elements than the instance list -- emit the
//                       instances in that order, then run only the tile-id digit passes (2 at
//                       1080p) over the 64-bit keys.  LSD radix sort is stable, so the result is
//                       identical; the instance list is moved 2 times instead of 6.
#include <algorithm>

#include "common.cuh"
#include "layout.cuh"

namespace {

constexpr uint32_t FULL = 0xffffffffu;

__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}
__device__ __forceinline__ uint64_t ld_volatile_u64(const uint64_t* p) { return *reinterpret_cast<const volatile uint64_t*>(p); }
__device__ __forceinline__ void st_volatile_u64(uint64_t* p, uint64_t v) { *reinterpret_cast<volatile uint64_t*>(p) = v; }
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v) { *reinterpret_cast<volatile uint32_t*>(p) = v; }

// ------------------------------------------------------------------------------------------------
// scan + duplicate
// ------------------------------------------------------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = SCAN_TILE / SCAN_THREADS;   // 4
constexpr uint64_t ST_AGG = 1ull << 62, ST_INC = 2ull << 62, ST_VAL = (1ull << 62) - 1;

struct ScanDupArgs {
    int n, GW;
    const uint32_t* tiles_touched;
    const uint16_t* rect;
    const float* depth;
    const uint32_t* perm;        // NULL = index order
    uint32_t* offsets;           // NULL = do not write; indexed by Gaussian
    uint32_t* incl_pos;          // NULL = do not write; indexed by scan position (perm order)
    uint64_t* num_instances;     // NULL = do not write
    uint64_t* status;            // [scan_tiles]
    uint32_t* ticket;
    uint64_t capacity;
    uint64_t* keys;              // NULL = scan only
    uint32_t* vals;
    uint32_t* hist;              // [npass][256]
    int first_bit, npass;
};

__global__ void __launch_bounds__(SCAN_THREADS) scan_dup_kernel(const ScanDupArgs a) {
    __shared__ uint32_t s_incl[SCAN_TILE];     // CTA-local inclusive prefix of tiles_touched
    __shared__ uint32_t s_gid[SCAN_TILE];
    __shared__ uint32_t s_depth[SCAN_TILE];
    __shared__ uint2 s_rect[SCAN_TILE];
    __shared__ uint32_t s_hist[SORT_MAX_PASSES][256];
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_ticket;
    __shared__ uint64_t s_prefix;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_ticket = atomicAdd(a.ticket, 1u);
    if (a.keys)
        for (int j = tid; j < a.npass * 256; j += SCAN_THREADS) (&s_hist[0][0])[j] = 0;
    __syncthreads();
    const uint32_t ticket = s_ticket;
    const int base = (int)ticket * SCAN_TILE;

    // load (blocked: thread t owns items base + 4t .. 4t+3)
    uint32_t tt[SCAN_ITEMS];
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const int j = base + tid * SCAN_ITEMS + k;
        uint32_t g = 0, t = 0;
        if (j < a.n) {
            g = a.perm ? __ldg(a.perm + j) : (uint32_t)j;
            t = __ldg(a.tiles_touched + g);
        }
        tt[k] = t;
        sum += t;
        s_gid[tid * SCAN_ITEMS + k] = g;
    }
    // CTA-wide inclusive scan of the per-thread sums
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t warp_off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        const uint32_t v = s_warp[w];
        if (w < warp) warp_off += v;
        total += v;
    }
    uint32_t run = warp_off + incl - sum;   // exclusive prefix of this thread inside the CTA
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        run += tt[k];
        s_incl[tid * SCAN_ITEMS + k] = run;
    }
    // decoupled look-back for the cross-CTA prefix (one thread; chains are short)
    if (tid == 0) {
        uint64_t excl = 0;
        if (ticket == 0) {
            st_volatile_u64(a.status, ST_INC | (uint64_t)total);
        } else {
            st_volatile_u64(a.status + ticket, ST_AGG | (uint64_t)total);
            int p = (int)ticket - 1;   // nearest predecessor not consumed yet; 8 are fetched per round trip
            while (true) {
                uint64_t v[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) v[j] = p - j >= 0 ? ld_volatile_u64(a.status + p - j) : ST_INC;
                int used = 0;
                bool fin = false;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const uint64_t f = v[j] >> 62;
                    if (!fin && used == j && f != 0) {
                        excl += v[j] & ST_VAL;
                        used = j + 1;
                        fin = f == 2;
                    }
                }
                if (fin) break;
                p -= used;
            }
            st_volatile_u64(a.status + ticket, ST_INC | (excl + total));
        }
        s_prefix = excl;
        if (a.num_instances && base + SCAN_TILE >= a.n) *a.num_instances = excl + total;
    }
    __syncthreads();
    const uint64_t prefix = s_prefix;
    if (a.offsets) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const int j = base + tid * SCAN_ITEMS + k;
            if (j < a.n) a.offsets[s_gid[tid * SCAN_ITEMS + k]] = (uint32_t)(prefix + s_incl[tid * SCAN_ITEMS + k]);
        }
    }
    if (a.incl_pos) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const int j = base + tid * SCAN_ITEMS + k;
            if (j < a.n) a.incl_pos[j] = (uint32_t)(prefix + s_incl[tid * SCAN_ITEMS + k]);
        }
    }
    if (!a.keys) return;

    // stage rect / depth of the Gaussians that emit
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const int li = tid * SCAN_ITEMS + k;
        if (tt[k]) {
            const uint32_t g = s_gid[li];
            s_rect[li] = __ldg(reinterpret_cast<const uint2*>(a.rect) + g);
            const uint32_t zb = __float_as_uint(__ldg(a.depth + g));
            s_depth[li] = zb;
            // depth digits are shared by every instance of the Gaussian: count tt[k] at once
            for (int p = 0; p < a.npass; ++p) {
                const int bit = a.first_bit + 8 * p;
                if (bit < 32) atomicAdd(&s_hist[p][(zb >> bit) & 255u], tt[k]);
            }
        }
    }
    __syncthreads();

    // cooperative emission: instance j of the CTA belongs to the first item with incl > j
    const int first_tile_pass = a.first_bit >= 32 ? 0 : (32 - a.first_bit) / 8;
    const uint32_t rounds = (total + SCAN_THREADS - 1) / SCAN_THREADS;
    for (uint32_t r = 0; r < rounds; ++r) {
        const uint32_t j = r * SCAN_THREADS + tid;
        const bool valid = j < total;
        uint32_t tile_id = 0xffffffffu;
        if (valid) {
            int lo = 0, hi = SCAN_TILE - 1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (s_incl[mid] > j) hi = mid; else lo = mid + 1;
            }
            const uint32_t start = lo ? s_incl[lo - 1] : 0u;
            const uint32_t local = j - start;
            const uint2 rc = s_rect[lo];
            const uint32_t x0 = rc.x & 0xffffu, y0 = rc.x >> 16, x1 = rc.y & 0xffffu;
            const uint32_t w = x1 - x0;
            const uint32_t ty = y0 + local / w, tx = x0 + local % w;
            tile_id = ty * (uint32_t)a.GW + tx;
            const uint64_t pos = prefix + j;
            if (pos < a.capacity) {
                a.keys[pos] = ((uint64_t)tile_id << 32) | (uint64_t)s_depth[lo];
                a.vals[pos] = s_gid[lo];
            }
        }
        // tile-id digits: consecutive instances mostly share the high digits -> aggregate
        // equal digits inside the warp before touching shared memory
        for (int p = first_tile_pass; p < a.npass; ++p) {
            const int bit = a.first_bit + 8 * p - 32;
            const uint32_t d = valid ? ((tile_id >> bit) & 255u) : 256u;
            const uint32_t peers = __match_any_sync(FULL, d);
            if (valid && (peers & lanemask_lt()) == 0) atomicAdd(&s_hist[p][d], (uint32_t)__popc(peers));
        }
    }
    __syncthreads();
    for (int j = tid; j < a.npass * 256; j += SCAN_THREADS) {
        const uint32_t c = (&s_hist[0][0])[j];
        if (c) atomicAdd(a.hist + j, c);
    }
}

// ------------------------------------------------------------------------------------------------
// balanced emission (default schedule).  In depth order the nearest Gaussians -- the ones with the
// largest footprints -- are consecutive, so a CTA-per-1024-Gaussians emission is badly unbalanced
// (one CTA may own millions of instances).  Here the work unit is EMIT_TILE consecutive INSTANCES:
//   emit_partition_kernel  starts[b] = first depth-ordered Gaussian g with incl[g] > min(b*EMIT_TILE, M-1)
//   emit_kernel            persistent CTAs; per unit the covering Gaussians (at most EMIT_TILE + 1,
//                          all visible: culled ones sort last) are staged in shared memory, every
//                          instance finds its owner by binary search; stores are coalesced.
// ------------------------------------------------------------------------------------------------
struct EmitArgs {
    int n, GW;
    const uint32_t* perm;      // [n] depth-ordered Gaussian indices, visible first
    const uint32_t* incl;      // [n] inclusive prefix of tiles_touched in that order
    const uint16_t* rect;
    const float* depth;
    const uint64_t* num_instances;
    uint64_t capacity;
    uint32_t* starts;          // [units + 1]
    int units;                 // ceil(capacity / EMIT_TILE)
    uint64_t* keys;
    uint32_t* vals;
    uint32_t* hist;            // [npass][256] tile-id digit histograms
    int npass;
};

__global__ void __launch_bounds__(256) emit_partition_kernel(const EmitArgs a) {
    const int b = blockIdx.x * 256 + threadIdx.x;
    if (b > a.units) return;
    const uint64_t M = *a.num_instances;
    if (M == 0 || M > a.capacity) return;
    uint64_t j = (uint64_t)b * EMIT_TILE;
    if (j > M - 1) j = M - 1;
    int lo = 0, hi = a.n - 1;   // incl[n-1] = M > j
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if ((uint64_t)__ldg(a.incl + mid) > j) hi = mid; else lo = mid + 1;
    }
    a.starts[b] = (uint32_t)lo;
}

constexpr int EMIT_THREADS = 256;
constexpr int EMIT_ITEMS = EMIT_TILE / EMIT_THREADS;   // 4 consecutive instances per thread

__global__ void __launch_bounds__(EMIT_THREADS) emit_kernel(const EmitArgs a) {
    __shared__ uint32_t s_incl[EMIT_TILE + 1];
    __shared__ uint32_t s_gid[EMIT_TILE + 1];
    __shared__ uint32_t s_depth[EMIT_TILE + 1];
    __shared__ uint2 s_rect[EMIT_TILE + 1];
    __shared__ uint32_t s_hist[SORT_MAX_PASSES][256];
    static_assert(EMIT_ITEMS == 4, "vector stores below assume 4 instances per thread");
    const int tid = threadIdx.x;
    const uint64_t M = *a.num_instances;
    if (M == 0 || M > a.capacity) return;
    for (int j = tid; j < a.npass * 256; j += EMIT_THREADS) (&s_hist[0][0])[j] = 0;
    const uint32_t units = (uint32_t)((M + EMIT_TILE - 1) / EMIT_TILE);
    // The staging of a unit is a chain of three dependent global loads (starts -> perm/incl -> depth/rect).  It is
    // software-pipelined over this CTA's units: while unit u is expanded, the second level of unit u+1 and the first
    // level of unit u+2 are in flight, so only the last gather of a unit is waited for.
    constexpr int EPT = (EMIT_TILE + 1 + EMIT_THREADS - 1) / EMIT_THREADS;   // staged entries per thread (5)
    const uint32_t stride = gridDim.x;
    uint32_t b = blockIdx.x;
    // level 1 of units b and b + stride
    uint32_t lo_c = 0, hi_c = 0, lo_n = 0, hi_n = 0;
    if (b < units) { lo_c = __ldg(a.starts + b); hi_c = __ldg(a.starts + b + 1); }
    if (b + stride < units) { lo_n = __ldg(a.starts + b + stride); hi_n = __ldg(a.starts + b + stride + 1); }
    // level 2 of unit b
    uint32_t r_incl[EPT], r_gid[EPT], r_before = 0;
    if (b < units) {
        const int span0 = (int)(hi_c - lo_c) + 1;
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
            const int i = tid + k * EMIT_THREADS;
            r_incl[k] = i < span0 ? __ldg(a.incl + lo_c + i) : 0u;
            r_gid[k] = i < span0 ? __ldg(a.perm + lo_c + i) : 0u;
        }
        r_before = lo_c ? __ldg(a.incl + lo_c - 1) : 0u;
    }
    for (; b < units; b += stride) {
        const uint32_t j0 = b * EMIT_TILE;
        const uint32_t cnt = (uint32_t)min((uint64_t)EMIT_TILE, M - j0);
        const int span = (int)(hi_c - lo_c) + 1;   // <= EMIT_TILE + 1
        const uint32_t before = r_before;
        // level 3 of this unit
        uint32_t r_depth[EPT];
        uint2 r_rect[EPT];
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
            const int i = tid + k * EMIT_THREADS;
            r_depth[k] = 0u;
            r_rect[k] = make_uint2(0u, 0u);
            if (i < span) {
                r_depth[k] = __float_as_uint(__ldg(a.depth + r_gid[k]));
                r_rect[k] = __ldg(reinterpret_cast<const uint2*>(a.rect) + r_gid[k]);
            }
        }
        __syncthreads();   // previous unit done with the staging arrays (and s_hist zeroed)
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
            const int i = tid + k * EMIT_THREADS;
            if (i < span) { s_incl[i] = r_incl[k]; s_gid[i] = r_gid[k]; }
        }
        // level 2 of the next unit, level 1 of the one after (their registers are free now)
        const uint32_t lo_nn = b + 2 * stride < units ? __ldg(a.starts + b + 2 * stride) : 0u;
        const uint32_t hi_nn = b + 2 * stride < units ? __ldg(a.starts + b + 2 * stride + 1) : 0u;
        if (b + stride < units) {
            const int span1 = (int)(hi_n - lo_n) + 1;
#pragma unroll
            for (int k = 0; k < EPT; ++k) {
                const int i = tid + k * EMIT_THREADS;
                r_incl[k] = i < span1 ? __ldg(a.incl + lo_n + i) : 0u;
                r_gid[k] = i < span1 ? __ldg(a.perm + lo_n + i) : 0u;
            }
            r_before = lo_n ? __ldg(a.incl + lo_n - 1) : 0u;
        }
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
            const int i = tid + k * EMIT_THREADS;
            if (i < span) { s_depth[i] = r_depth[k]; s_rect[i] = r_rect[k]; }
        }
        lo_c = lo_n; hi_c = hi_n; lo_n = lo_nn; hi_n = hi_nn;
        __syncthreads();
        const uint32_t jl = tid * EMIT_ITEMS;
        if (jl < cnt) {
            const uint32_t j = j0 + jl;
            int lo = 0, hi = span - 1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (s_incl[mid] > j) hi = mid; else lo = mid + 1;
            }
            // walk the (up to) 4 consecutive instances: position inside the owner's rect advances in row-major order
            uint32_t end = s_incl[lo];
            uint32_t local = j - (lo ? s_incl[lo - 1] : before);
            uint2 rc = s_rect[lo];
            uint32_t x0 = rc.x & 0xffffu, x1 = rc.y & 0xffffu, w = x1 - x0;
            uint32_t ty = (rc.x >> 16) + local / w, tx = x0 + local % w;
            uint32_t zb = s_depth[lo], gid = s_gid[lo];
            uint64_t k[EMIT_ITEMS];
            uint32_t v[EMIT_ITEMS], tl[EMIT_ITEMS];
#pragma unroll
            for (int e = 0; e < EMIT_ITEMS; ++e) {
                tl[e] = ty * (uint32_t)a.GW + tx;
                k[e] = ((uint64_t)tl[e] << 32) | (uint64_t)zb;
                v[e] = gid;
                if (e + 1 < EMIT_ITEMS && jl + e + 1 < cnt) {
                    if (j + e + 1 == end) {   // next owner (every staged Gaussian has >= 1 instance)
                        ++lo;
                        end = s_incl[lo];
                        rc = s_rect[lo];
                        x0 = rc.x & 0xffffu; x1 = rc.y & 0xffffu;
                        ty = rc.x >> 16; tx = x0;
                        zb = s_depth[lo]; gid = s_gid[lo];
                    } else if (++tx == x1) {
                        tx = x0; ++ty;
                    }
                }
            }
            if (jl + EMIT_ITEMS <= cnt) {
                *reinterpret_cast<ulonglong2*>(a.keys + j) = make_ulonglong2(k[0], k[1]);
                *reinterpret_cast<ulonglong2*>(a.keys + j + 2) = make_ulonglong2(k[2], k[3]);
                *reinterpret_cast<uint4*>(a.vals + j) = make_uint4(v[0], v[1], v[2], v[3]);
            } else {
                for (int e = 0; e < EMIT_ITEMS; ++e)
                    if (jl + e < cnt) { a.keys[j + e] = k[e]; a.vals[j + e] = v[e]; }
            }
            for (int p = 0; p < a.npass; ++p)
                for (int e = 0; e < EMIT_ITEMS; ++e)
                    if (jl + e < cnt) atomicAdd(&s_hist[p][(tl[e] >> (8 * p)) & 255u], 1u);
        }
    }
    __syncthreads();
    for (int j = tid; j < a.npass * 256; j += EMIT_THREADS) {
        const uint32_t c = (&s_hist[0][0])[j];
        if (c) atomicAdd(a.hist + j, c);
    }
}

// exclusive scan of every 256-bin histogram (one CTA of 256 threads per pass)
__global__ void __launch_bounds__(256) hist_scan_kernel(uint32_t* hist) {
    __shared__ uint32_t s_w[8];
    uint32_t* h = hist + blockIdx.x * 256;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t c = h[tid];
    uint32_t incl = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    uint32_t off = 0;
    for (int w = 0; w < warp; ++w) off += s_w[w];
    h[tid] = off + incl - c;
}

// ------------------------------------------------------------------------------------------------
// depth pre-sort input: key = depth bits (0xffffffff for culled Gaussians), val = index;
// accumulates the four digit histograms of the 32-bit keys.
// ------------------------------------------------------------------------------------------------
// When `diff` is given (tile grid small enough for shared memory) the kernel also accumulates the 2-D
// difference array of the per-tile instance counts: +1 at (y0,x0), -1 at (y0,x1), -1 at (y1,x0),
// +1 at (y1,x1) for every visible Gaussian; its 2-D prefix sum (tile_scan_kernel) is the number of
// instances of every tile, from which the tile ranges and the tile-digit histograms follow without
// touching the instance list.
__global__ void __launch_bounds__(256) presort_init_kernel(int n, const float* depth, const uint32_t* tiles_touched,
                                                           uint32_t* keys, uint32_t* vals, uint32_t* hist32,
                                                           const uint16_t* rect, int gw1, int gh1, int* diff) {
    extern __shared__ int s_diff[];
    __shared__ uint32_t s_hist[4][256];
    for (int j = threadIdx.x; j < 1024; j += 256) (&s_hist[0][0])[j] = 0;
    const int cells = diff ? gw1 * gh1 : 0;
    for (int j = threadIdx.x; j < cells; j += 256) s_diff[j] = 0;
    __syncthreads();
    for (int i = blockIdx.x * 256 + threadIdx.x; i < n; i += gridDim.x * 256) {
        const bool vis = __ldg(tiles_touched + i) != 0;
        const uint32_t k = vis ? __float_as_uint(__ldg(depth + i)) : 0xffffffffu;
        keys[i] = k;
        vals[i] = (uint32_t)i;
#pragma unroll
        for (int p = 0; p < 4; ++p) atomicAdd(&s_hist[p][(k >> (8 * p)) & 255u], 1u);
        if (diff && vis) {
            const uint2 rc = __ldg(reinterpret_cast<const uint2*>(rect) + i);
            const int x0 = rc.x & 0xffffu, y0 = rc.x >> 16, x1 = rc.y & 0xffffu, y1 = rc.y >> 16;
            atomicAdd(&s_diff[y0 * gw1 + x0], 1);
            atomicAdd(&s_diff[y0 * gw1 + x1], -1);
            atomicAdd(&s_diff[y1 * gw1 + x0], -1);
            atomicAdd(&s_diff[y1 * gw1 + x1], 1);
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < 1024; j += 256) {
        const uint32_t c = (&s_hist[0][0])[j];
        if (c) atomicAdd(hist32 + j, c);
    }
    for (int j = threadIdx.x; j < cells; j += 256) {
        const int c = s_diff[j];
        if (c) atomicAdd(diff + j, c);
    }
}

// One CTA: 2-D prefix sum of the difference grid -> per-tile instance counts -> tile ranges
// (C1-S step 4: exclusive prefix over tile ids, (0,0) for empty tiles) and the exclusive digit
// histograms of the tile-id sort passes.  Nothing is written when M > capacity.
constexpr int TS_THREADS = 1024;
__global__ void __launch_bounds__(TS_THREADS) tile_scan_kernel(const int* diff, int gw1, int gh1, const uint64_t* num_instances,
                                                               uint64_t capacity, uint32_t* ranges, uint32_t* hist, int npass,
                                                               uint32_t* order, uint32_t* order_valid) {
    extern __shared__ int s_g[];                 // [gh1][gw1]
    __shared__ uint32_t s_bucket[34];            // tiles per log2(count) bucket (descending), then their start offsets
    __shared__ uint32_t s_h[SORT_MAX_PASSES][256];
    __shared__ uint32_t s_part[TS_THREADS / 32];
    __shared__ uint32_t s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint64_t M = *num_instances;
    if (M > capacity) return;
    const int GW = gw1 - 1, GH = gh1 - 1, cells = gw1 * gh1, ntiles = GW * GH;
    for (int j = tid; j < cells; j += TS_THREADS) s_g[j] = diff[j];
    for (int j = tid; j < npass * 256; j += TS_THREADS) (&s_h[0][0])[j] = 0;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int y = tid; y < gh1; y += TS_THREADS) {      // prefix along x
        int run = 0;
        for (int x = 0; x < gw1; ++x) { run += s_g[y * gw1 + x]; s_g[y * gw1 + x] = run; }
    }
    __syncthreads();
    for (int x = tid; x < gw1; x += TS_THREADS) {      // prefix along y
        int run = 0;
        for (int y = 0; y < gh1; ++y) { run += s_g[y * gw1 + x]; s_g[y * gw1 + x] = run; }
    }
    __syncthreads();
    // exclusive scan over tile ids, TS_THREADS tiles per round
    for (int base = 0; base < ntiles; base += TS_THREADS) {
        const int t = base + tid;
        uint32_t c = 0;
        if (t < ntiles) c = (uint32_t)s_g[(t / GW) * gw1 + (t % GW)];
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) s_part[warp] = incl;
        __syncthreads();
        uint32_t off = s_carry;
        for (int w = 0; w < warp; ++w) off += s_part[w];
        const uint32_t excl = off + incl - c;
        if (t < ntiles && c) {
            ranges[2 * (size_t)t] = excl;
            ranges[2 * (size_t)t + 1] = excl + c;
            for (int p = 0; p < npass; ++p) atomicAdd(&s_h[p][((uint32_t)t >> (8 * p)) & 255u], c);
        }
        __syncthreads();
        if (tid == TS_THREADS - 1) s_carry = excl + c;
        __syncthreads();
    }
    // work order of render / fuse: tiles by descending floor(log2(count)) (counting sort; empty tiles last)
    for (int j = tid; j < 34; j += TS_THREADS) s_bucket[j] = 0;
    __syncthreads();
    for (int t = tid; t < ntiles; t += TS_THREADS) {
        const uint32_t c = (uint32_t)s_g[(t / GW) * gw1 + (t % GW)];
        atomicAdd(&s_bucket[c ? __clz(c) : 32], 1u);   // clz small = long list = early bucket
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t run = 0;
        for (int b = 0; b < 33; ++b) { const uint32_t c = s_bucket[b]; s_bucket[b] = run; run += c; }
    }
    __syncthreads();
    for (int t = tid; t < ntiles; t += TS_THREADS) {
        const uint32_t c = (uint32_t)s_g[(t / GW) * gw1 + (t % GW)];
        order[atomicAdd(&s_bucket[c ? __clz(c) : 32], 1u)] = (uint32_t)t;
    }
    if (tid == 0) *order_valid = 1u;
    // exclusive scan of every digit histogram (warp w handles pass w)
    if (warp < npass) {
        uint32_t run = 0;
        for (int b = 0; b < 256; b += 32) {
            const uint32_t c = s_h[warp][b + lane];
            uint32_t incl = c;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t o = __shfl_up_sync(FULL, incl, d);
                if (lane >= d) incl += o;
            }
            hist[warp * 256 + b + lane] = run + incl - c;
            run += __shfl_sync(FULL, incl, 31);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// onesweep pass
// ------------------------------------------------------------------------------------------------
constexpr int OS_THREADS = 256;
constexpr int OS_WARPS = OS_THREADS / 32;
constexpr int OS_LOOKBACK = 8;    // predecessors fetched per look-back round trip
constexpr uint32_t OS_AGG = 1u << 30, OS_INC = 2u << 30, OS_VAL = (1u << 30) - 1;

template <typename KeyT>
struct OneSweepArgs {
    const KeyT* keys_in;
    const uint32_t* vals_in;
    KeyT* keys_out;
    uint32_t* vals_out;
    const uint64_t* count_dev;   // device count (instance sort) or NULL
    uint64_t count_host;         // used when count_dev == NULL
    uint64_t capacity;           // count > capacity -> the pass does nothing
    int shift;
    const uint32_t* hist_excl;   // [256] exclusive digit offsets of this pass
    uint32_t* status;            // [tiles][256]
    uint32_t* ticket;
};

template <typename KeyT, int ITEMS>
__global__ void __launch_bounds__(OS_THREADS, ITEMS >= 16 ? 3 : 5) onesweep_kernel(const OneSweepArgs<KeyT> a) {
    constexpr int TILE = OS_THREADS * ITEMS;
    __shared__ uint32_t s_cnt[OS_WARPS][256];   // per-warp digit counts -> per-warp exclusive offsets
    __shared__ __align__(16) KeyT s_keys[TILE]; // reused for the values
    __shared__ uint32_t s_bin_start[256];       // CTA-local start of each digit run
    __shared__ uint32_t s_goff[256];            // global offset of digit run minus its local start
    __shared__ uint32_t s_w[OS_WARPS];
    __shared__ uint32_t s_ticket;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint64_t count = a.count_dev ? *a.count_dev : a.count_host;
    if (count > a.capacity) return;
    if (tid == 0) s_ticket = atomicAdd(a.ticket, 1u);
#pragma unroll
    for (int w = 0; w < OS_WARPS; ++w) s_cnt[w][tid] = 0;
    __syncthreads();
    const uint32_t ticket = s_ticket;
    const uint64_t tile_base = (uint64_t)ticket * TILE;
    if (tile_base >= count) return;
    const uint32_t tile_valid = (uint32_t)min((uint64_t)TILE, count - tile_base);

    // warp-striped load: warp w, item i, lane l <-> element w*ITEMS*32 + i*32 + l (processing order)
    // (the values are fetched only when they are scattered: 16 fewer live registers during the ranking -> 3 CTAs/SM)
    KeyT key[ITEMS];
    uint32_t rank[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const uint32_t e = warp * ITEMS * 32 + i * 32 + lane;
        key[i] = e < tile_valid ? a.keys_in[tile_base + e] : ~(KeyT)0;   // padding sorts last inside the tile; never written out
    }
    // stable ranking inside the warp: equal digits are ranked by (item, lane).  The 16 match_any are independent
    // of one another and are issued back to back (their latency overlaps); only the shared-memory counter update
    // forms a chain over the items.
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) rank[i] = __match_any_sync(FULL, (uint32_t)(key[i] >> a.shift) & 255u);
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const uint32_t d = (uint32_t)(key[i] >> a.shift) & 255u;
        const uint32_t peers = rank[i];
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader) {
            old = s_cnt[warp][d];
            s_cnt[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(FULL, old, leader);
        rank[i] = old + __popc(peers & lanemask_lt());
        __syncwarp();
    }
    __syncthreads();
    // digit `tid`: per-warp exclusive offsets and the CTA count
    uint32_t cnt = 0;
#pragma unroll
    for (int w = 0; w < OS_WARPS; ++w) {
        const uint32_t c = s_cnt[w][tid];
        s_cnt[w][tid] = cnt;
        cnt += c;
    }
    if (tid == 255) cnt -= (uint32_t)TILE - tile_valid;   // padding keys all carry digit 255
    // publish the CTA's digit counts at once; the look-back itself is deferred until the keys are staged, so that
    // the wait for the predecessors overlaps the local scan and the shared-memory scatter
    uint32_t* my = a.status + (size_t)ticket * 256 + tid;
    st_volatile_u32(my, (ticket == 0 ? OS_INC : OS_AGG) | cnt);
    // CTA-local exclusive scan over digits
    uint32_t incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    uint32_t off = 0;
    for (int w = 0; w < warp; ++w) off += s_w[w];
    const uint32_t bin_start = off + incl - cnt;
    s_bin_start[tid] = bin_start;
    __syncthreads();
    // keys -> shared memory at their CTA-local sorted position
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const uint32_t d = (uint32_t)(key[i] >> a.shift) & 255u;
        rank[i] += s_bin_start[d] + s_cnt[warp][d];
        s_keys[rank[i]] = key[i];
    }
    // look back over the earlier CTAs (digit `tid`)
    // (OS_LOOKBACK predecessors are fetched per round trip: the walk back to the nearest inclusive prefix is a chain of
    // dependent L2 loads, and with ~450 CTAs in flight it is tens of entries long)
    uint32_t excl = 0;
    if (ticket != 0) {
        const uint32_t* p = my - 256;
        int remaining = (int)ticket;   // predecessors not consumed yet; p points at the nearest of them
        while (true) {
            uint32_t v[OS_LOOKBACK];
#pragma unroll
            for (int j = 0; j < OS_LOOKBACK; ++j) v[j] = j < remaining ? ld_volatile_u32(p - 256 * j) : OS_INC;
            int used = 0;
            bool fin = false;
#pragma unroll
            for (int j = 0; j < OS_LOOKBACK; ++j) {
                const uint32_t f = v[j] >> 30;
                if (!fin && used == j && f != 0) {   // consume in order; stop at the first entry that is not published yet
                    excl += v[j] & OS_VAL;
                    used = j + 1;
                    fin = f == 2;
                }
            }
            if (fin) break;
            p -= 256 * used;
            remaining -= used;
        }
        st_volatile_u32(my, OS_INC | (excl + cnt));
    }
    s_goff[tid] = a.hist_excl[tid] + excl - bin_start;
    __syncthreads();
    uint32_t gpos[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const uint32_t j = i * OS_THREADS + tid;
        if (j < tile_valid) {
            const KeyT k = s_keys[j];
            const uint32_t d = (uint32_t)(k >> a.shift) & 255u;
            gpos[i] = s_goff[d] + j;
            a.keys_out[gpos[i]] = k;
        }
    }
    __syncthreads();
    uint32_t* s_vals = reinterpret_cast<uint32_t*>(s_keys);
    {
        uint32_t val[ITEMS];
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const uint32_t e = warp * ITEMS * 32 + i * 32 + lane;
            val[i] = e < tile_valid ? a.vals_in[tile_base + e] : 0u;
        }
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) s_vals[rank[i]] = val[i];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const uint32_t j = i * OS_THREADS + tid;
        if (j < tile_valid) a.vals_out[gpos[i]] = s_vals[j];
    }
}

// ------------------------------------------------------------------------------------------------
// tile ranges (C1-S step 4)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ranges_kernel(const uint64_t* keys, const uint64_t* count_dev, uint64_t capacity,
                                                     uint32_t* ranges) {
    const uint64_t count = *count_dev;
    if (count > capacity) return;
    for (uint64_t k = (uint64_t)blockIdx.x * 256 + threadIdx.x; k < count; k += (uint64_t)gridDim.x * 256) {
        const uint32_t t = (uint32_t)(keys[k] >> 32);
        if (k == 0 || (uint32_t)(keys[k - 1] >> 32) != t) ranges[2 * (size_t)t] = (uint32_t)k;
        if (k + 1 == count || (uint32_t)(keys[k + 1] >> 32) != t) ranges[2 * (size_t)t + 1] = (uint32_t)(k + 1);
    }
}

int ceil_log2(uint64_t v) {
    int b = 0;
    while ((1ull << b) < v) ++b;
    return b;
}

}  // namespace

extern "C" fhgs_status fhgs_bin_sort(fhgs_ctx* ctx, const fhgs_camera* cam, fhgs_view_state* vs,
                                     uint64_t* num_instances_host, uint32_t flags, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!cam || !vs) FHGS_INVALID(ctx, "fhgs_bin_sort: NULL argument");
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    if (flags & ~(uint32_t)FHGS_SORT_FULL_KEY) FHGS_INVALID(ctx, "fhgs_bin_sort: unknown flag");
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    const int GW = tiles_x(cam->width), GH = tiles_y(cam->height);
    const size_t ntiles = (size_t)GW * GH;
    const ScratchLayout L = make_scratch_layout(vs->n, vs->capacity, cam->width, cam->height);
    char* sc = (char*)vs->scratch;
    uint32_t* ctrl = (uint32_t*)(sc + L.ctrl);
    uint32_t* hist = (uint32_t*)(sc + L.hist);
    uint32_t* hist32 = (uint32_t*)(sc + L.hist32);
    uint64_t* scan_status = (uint64_t*)(sc + L.scan_status);
    uint32_t* sort_status = (uint32_t*)(sc + L.sort_status);

    FHGS_CUDA(ctx, cudaMemsetAsync(sc, 0, L.zero_bytes, s));
    FHGS_CUDA(ctx, cudaMemsetAsync(scan_status, 0, 2 * L.scan_tiles * 8, s));
    FHGS_CUDA(ctx, cudaMemsetAsync(vs->ranges, 0, ntiles * 8, s));
    FHGS_CUDA(ctx, cudaMemsetAsync(vs->num_instances, 0, 8, s));

    const int tile_bits = ceil_log2(ntiles);
    const bool full_key = (flags & FHGS_SORT_FULL_KEY) != 0;
    // per-tile counts through the 2-D difference grid (default schedule, grid small enough for shared memory)
    const int gw1 = GW + 1, gh1 = GH + 1;
    const bool grid_counts = !full_key && vs->capacity > 0 && (size_t)gw1 * gh1 <= (size_t)TILE_GRID_MAX;
    int* tile_diff = (int*)(sc + L.tile_diff);
    const size_t diff_bytes = (size_t)gw1 * gh1 * 4;
    if (grid_counts) FHGS_CUDA(ctx, cudaMemsetAsync(tile_diff, 0, diff_bytes, s));
#ifdef FHGS_NO_SIDE
    const bool side_overlap = false;
#else
    const bool side_overlap = grid_counts && vs->n > 0;
#endif
    const int first_bit = full_key ? 0 : 32;
    const int npass = ((32 + tile_bits) - first_bit + 7) / 8;
    vs->sorted_buf = npass & 1;

    if (vs->n > 0) {
        const int scan_grid = (vs->n + SCAN_TILE - 1) / SCAN_TILE;
        const uint32_t* perm = nullptr;
        if (!full_key) {
            // order the Gaussians by (depth bits, index): 4 stable passes over 32-bit keys
            uint32_t* pk[2] = {(uint32_t*)(sc + L.pre_keys[0]), (uint32_t*)(sc + L.pre_keys[1])};
            uint32_t* pv[2] = {(uint32_t*)(sc + L.pre_vals[0]), (uint32_t*)(sc + L.pre_vals[1])};
            const int grid = std::min((vs->n + 255) / 256, ctx->num_sms * (grid_counts ? 4 : 8));
            if (grid_counts)
                FHGS_CUDA(ctx, cudaFuncSetAttribute(presort_init_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)diff_bytes));
            presort_init_kernel<<<grid, 256, grid_counts ? diff_bytes : 0, s>>>(vs->n, vs->depth, vs->tiles_touched, pk[0], pv[0], hist32,
                                                                               vs->rect, gw1, gh1, grid_counts ? tile_diff : nullptr);
            FHGS_LAUNCH_CHECK(ctx);
            if (side_overlap) {
                FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
                FHGS_CUDA(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
            }
            hist_scan_kernel<<<4, 256, 0, s>>>(hist32);
            FHGS_LAUNCH_CHECK(ctx);
            FHGS_CUDA(ctx, cudaFuncSetAttribute(onesweep_kernel<uint32_t, SORT_TILE_K32 / OS_THREADS>,
                                                cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            const int pre_grid = (vs->n + SORT_TILE_K32 - 1) / SORT_TILE_K32;
            for (int p = 0; p < 4; ++p) {
                FHGS_CUDA(ctx, cudaMemsetAsync(sort_status, 0, (size_t)pre_grid * 256 * 4, s));
                OneSweepArgs<uint32_t> oa;
                oa.keys_in = pk[p & 1]; oa.vals_in = pv[p & 1];
                oa.keys_out = pk[(p + 1) & 1]; oa.vals_out = pv[(p + 1) & 1];
                oa.count_dev = nullptr; oa.count_host = (uint64_t)vs->n; oa.capacity = (uint64_t)vs->n;
                oa.shift = 8 * p; oa.hist_excl = hist32 + 256 * p; oa.status = sort_status;
                oa.ticket = ctrl + CTRL_PRESORT_TICKET + p;
                onesweep_kernel<uint32_t, SORT_TILE_K32 / OS_THREADS><<<pre_grid, OS_THREADS, 0, s>>>(oa);
                FHGS_LAUNCH_CHECK(ctx);
            }
            perm = pv[0];   // 4 passes -> back in buffer 0
            // `offsets` is defined in index order (C1-S step 1): a scan-only launch.  With the tile-count path it and the
            // tile scan (ranges, digit offsets of the tile-id passes, tile order) depend only on presort_init: they run on
            // the context's side stream beside the four pre-sort passes and the depth-order scan (forked after
            // presort_init, joined before the emission needs M and before the first tile-id pass needs the offsets).
            ScanDupArgs sa0;
            memset(&sa0, 0, sizeof(sa0));
            sa0.n = vs->n; sa0.GW = GW; sa0.tiles_touched = vs->tiles_touched;
            sa0.offsets = vs->offsets; sa0.num_instances = vs->num_instances;
            sa0.status = scan_status + L.scan_tiles; sa0.ticket = ctrl + CTRL_SCAN2_TICKET;
            cudaStream_t s0 = side_overlap ? ctx->side : s;
            scan_dup_kernel<<<scan_grid, SCAN_THREADS, 0, s0>>>(sa0);
            FHGS_LAUNCH_CHECK(ctx);
            if (side_overlap) FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_offsets, ctx->side));
            if (grid_counts) {   // ranges, digit offsets of the tile-id passes and the tile order from the per-tile counts
                FHGS_CUDA(ctx, cudaFuncSetAttribute(tile_scan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)diff_bytes));
                tile_scan_kernel<<<1, TS_THREADS, diff_bytes, s0>>>(tile_diff, gw1, gh1, vs->num_instances, vs->capacity, vs->ranges,
                                                                 hist, npass, (uint32_t*)(sc + L.tile_order), ctrl + CTRL_ORDER_VALID);
                FHGS_LAUNCH_CHECK(ctx);
            }
            if (side_overlap) FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_tiles, ctx->side));
        }
        if (full_key || vs->capacity == 0) {
            ScanDupArgs sa;
            memset(&sa, 0, sizeof(sa));
            sa.n = vs->n; sa.GW = GW;
            sa.tiles_touched = vs->tiles_touched; sa.rect = vs->rect; sa.depth = vs->depth;
            sa.offsets = vs->offsets; sa.num_instances = vs->num_instances;
            sa.status = scan_status; sa.ticket = ctrl + CTRL_SCAN_TICKET;
            sa.capacity = vs->capacity;
            if (vs->capacity > 0) { sa.keys = vs->keys[0]; sa.vals = vs->vals[0]; }
            sa.hist = hist; sa.first_bit = first_bit; sa.npass = npass;
            if (full_key || perm == nullptr) {
                scan_dup_kernel<<<scan_grid, SCAN_THREADS, 0, s>>>(sa);
                FHGS_LAUNCH_CHECK(ctx);
            }
        } else {
            // prefix sums in depth order, then instance-balanced emission
            uint32_t* incl = (uint32_t*)(sc + L.pre_incl);
            ScanDupArgs sa;
            memset(&sa, 0, sizeof(sa));
            sa.n = vs->n; sa.GW = GW; sa.tiles_touched = vs->tiles_touched; sa.perm = perm;
            sa.incl_pos = incl; sa.status = scan_status; sa.ticket = ctrl + CTRL_SCAN_TICKET;
            scan_dup_kernel<<<scan_grid, SCAN_THREADS, 0, s>>>(sa);
            FHGS_LAUNCH_CHECK(ctx);
            EmitArgs ea;
            ea.n = vs->n; ea.GW = GW; ea.perm = perm; ea.incl = incl; ea.rect = vs->rect; ea.depth = vs->depth;
            ea.num_instances = vs->num_instances; ea.capacity = vs->capacity;
            ea.starts = (uint32_t*)(sc + L.emit_starts); ea.units = (int)L.emit_tiles;
            ea.keys = vs->keys[0]; ea.vals = vs->vals[0]; ea.hist = hist; ea.npass = grid_counts ? 0 : npass;
            // grid_counts: ranges and digit offsets come from the per-tile counts (tile_scan_kernel, on the side stream);
            // the emission needs M from the offsets scan
            if (side_overlap) FHGS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_offsets, 0));
            emit_partition_kernel<<<(ea.units + 1 + 255) / 256, 256, 0, s>>>(ea);
            FHGS_LAUNCH_CHECK(ctx);
            const int egrid = std::min(ea.units, ctx->num_sms * 8);
            emit_kernel<<<egrid, EMIT_THREADS, 0, s>>>(ea);
            FHGS_LAUNCH_CHECK(ctx);
        }

        if (vs->capacity > 0) {
            if (!grid_counts) {
                hist_scan_kernel<<<npass, 256, 0, s>>>(hist);
                FHGS_LAUNCH_CHECK(ctx);
            }
            FHGS_CUDA(ctx, cudaFuncSetAttribute(onesweep_kernel<uint64_t, SORT_TILE_K64 / OS_THREADS>,
                                                cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            const int sort_grid = (int)((vs->capacity + SORT_TILE_K64 - 1) / SORT_TILE_K64);
            if (side_overlap) FHGS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_tiles, 0));
            for (int p = 0; p < npass; ++p) {
                FHGS_CUDA(ctx, cudaMemsetAsync(sort_status, 0, (size_t)sort_grid * 256 * 4, s));
                OneSweepArgs<uint64_t> oa;
                oa.keys_in = vs->keys[p & 1]; oa.vals_in = vs->vals[p & 1];
                oa.keys_out = vs->keys[(p + 1) & 1]; oa.vals_out = vs->vals[(p + 1) & 1];
                oa.count_dev = vs->num_instances; oa.count_host = 0; oa.capacity = vs->capacity;
                oa.shift = first_bit + 8 * p; oa.hist_excl = hist + 256 * p; oa.status = sort_status;
                oa.ticket = ctrl + CTRL_SORT_TICKET + p;
                onesweep_kernel<uint64_t, SORT_TILE_K64 / OS_THREADS><<<sort_grid, OS_THREADS, 0, s>>>(oa);
                FHGS_LAUNCH_CHECK(ctx);
            }
            if (!grid_counts) {
                uint64_t rg = (vs->capacity + 255) / 256;
                if (rg > (uint64_t)ctx->num_sms * 16) rg = (uint64_t)ctx->num_sms * 16;
                const int rgrid = (int)rg;
                ranges_kernel<<<rgrid, 256, 0, s>>>(vs->keys[vs->sorted_buf], vs->num_instances, vs->capacity, vs->ranges);
                FHGS_LAUNCH_CHECK(ctx);
            }
        }
    }
    if (num_instances_host) {
        FHGS_CUDA(ctx, cudaMemcpyAsync(num_instances_host, vs->num_instances, 8, cudaMemcpyDeviceToHost, s));
        FHGS_CUDA(ctx, cudaStreamSynchronize(s));
        if (*num_instances_host > vs->capacity)
            return set_err(ctx, FHGS_ERR_CAPACITY, "fhgs_bin_sort: %s%lld instances exceed capacity", "", (long long)*num_instances_host);
    }
    return FHGS_OK;
}
