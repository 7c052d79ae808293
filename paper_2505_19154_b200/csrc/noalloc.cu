// noalloc.cu -- fhgs_scan_offsets_static: step S1's prefix sum (DuplicateWithKeys needs
// offsets[i] = sum_{j<=i} tiles_touched[j]) with its decoupled look-back status words in a
// file-scope device array instead of caller-supplied scratch.  For callers that cannot provide or allocate
// scratch memory (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the entry point
// allocates nothing.  It is a variant of binsort.cu's scan_dup_kernel (scan part only) and shares no state
// with fhgs_bin_sort; no existing path calls it.
#include <mutex>

#include "common.cuh"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_ITEMS = 4;
constexpr int NA_TILE = NA_THREADS * NA_ITEMS;          // 1024 counts per CTA
constexpr int NA_MAX_N = 1 << 22;                       // 4 194 304 Gaussians (Large-feature is 3e6)
constexpr int NA_MAX_TILES = NA_MAX_N / NA_TILE;        // 4096 status words
constexpr uint64_t NA_AGG = 1ull << 62, NA_INC = 2ull << 62, NA_VAL = (1ull << 62) - 1;
constexpr unsigned NA_FULL = 0xffffffffu;

// 32 KB of look-back status + one ticket word (in its own 256-byte line).  Every GPU that loads libfhgs.so holds
// this array until the process exits.  All calls share it and it keeps the last call's contents: every call
// clears the words it is going to use first, and two calls that overlap on the GPU race on it.
struct NoAllocScratch {
    uint64_t status[NA_MAX_TILES];
    uint32_t ticket;
    uint32_t pad[63];
};
static __device__ __align__(256) NoAllocScratch g_noalloc_scratch;

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the address is looked up once
// per device, with that device current, and handed to the kernels.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
NoAllocScratch* g_na_ptr[NA_MAX_DEVICES] = {};

__global__ void __launch_bounds__(NA_THREADS) noalloc_clear_kernel(NoAllocScratch* sc, int tiles) {
    const int i = blockIdx.x * NA_THREADS + threadIdx.x;
    if (i < tiles) sc->status[i] = 0;
    if (i == 0) sc->ticket = 0;
}

__global__ void __launch_bounds__(NA_THREADS) scan_offsets_static_kernel(const uint32_t* __restrict__ tiles_touched,
                                                                         int n, uint32_t* __restrict__ offsets,
                                                                         uint64_t* num_instances, NoAllocScratch* sc) {
    __shared__ uint32_t s_warp[NA_THREADS / 32];
    __shared__ uint32_t s_ticket;
    __shared__ uint64_t s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // CTAs take their part of the array in the order they start, so a predecessor is always running or done
    if (tid == 0) s_ticket = atomicAdd(&sc->ticket, 1u);
    __syncthreads();
    const uint32_t ticket = s_ticket;
    const int base = (int)ticket * NA_TILE + tid * NA_ITEMS;

    uint32_t tt[NA_ITEMS];
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        tt[k] = base + k < n ? __ldg(tiles_touched + base + k) : 0u;
        sum += tt[k];
    }
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(NA_FULL, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t warp_off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < NA_THREADS / 32; ++w) {
        const uint32_t v = s_warp[w];
        if (w < warp) warp_off += v;
        total += v;
    }
    // decoupled look-back over the predecessors' status words (aggregate | inclusive prefix)
    if (tid == 0) {
        uint64_t excl = 0;
        volatile uint64_t* status = sc->status;
        if (ticket == 0) {
            status[0] = NA_INC | (uint64_t)total;
        } else {
            status[ticket] = NA_AGG | (uint64_t)total;
            for (int p = (int)ticket - 1; p >= 0; --p) {
                uint64_t v;
                do { v = status[p]; } while ((v >> 62) == 0);
                excl += v & NA_VAL;
                if ((v >> 62) == 2) break;
            }
            __threadfence();
            status[ticket] = NA_INC | (excl + total);
        }
        s_prefix = excl;
        if (num_instances && (int)(ticket + 1) * NA_TILE >= n) *num_instances = excl + total;
    }
    __syncthreads();
    uint32_t run = (uint32_t)s_prefix + warp_off + incl - sum;
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        run += tt[k];
        if (base + k < n) offsets[base + k] = run;
    }
}

// once per device, with that device current (the caller holds a DeviceGuard)
cudaError_t noalloc_scratch_ptr(int device, NoAllocScratch** out) {
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_na_ptr[device] = static_cast<NoAllocScratch*>(p);
    }
    *out = g_na_ptr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int32_t fhgs_scan_offsets_static_max_n(void) { return NA_MAX_N; }

extern "C" fhgs_status fhgs_scan_offsets_static(fhgs_ctx* ctx, const uint32_t* tiles_touched, int32_t n,
                                                uint32_t* offsets, uint64_t* num_instances, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (n < 0) FHGS_INVALID(ctx, "scan_offsets_static: n < 0");
    if (n > NA_MAX_N)
        return set_err(ctx, FHGS_ERR_INVALID,
                       "scan_offsets_static: n exceeds the static scratch (%s max n = %lld); use fhgs_bin_sort with "
                       "caller scratch", "", (long long)NA_MAX_N);
    if (n > 0 && (!tiles_touched || !offsets)) FHGS_INVALID(ctx, "scan_offsets_static: NULL tiles_touched / offsets");
    if (!num_instances && n == 0) return FHGS_OK;
    if (ctx->device < 0 || ctx->device >= NA_MAX_DEVICES) FHGS_INVALID(ctx, "scan_offsets_static: device ordinal >= 64");
    DeviceGuard dg(ctx);
    NoAllocScratch* sc = nullptr;
    FHGS_CUDA(ctx, noalloc_scratch_ptr(ctx->device, &sc));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int tiles = n > 0 ? (n + NA_TILE - 1) / NA_TILE : 1;
    noalloc_clear_kernel<<<(tiles + NA_THREADS - 1) / NA_THREADS, NA_THREADS, 0, s>>>(sc, tiles);
    FHGS_LAUNCH_CHECK(ctx);
    scan_offsets_static_kernel<<<tiles, NA_THREADS, 0, s>>>(tiles_touched, n, offsets, num_instances, sc);
    FHGS_LAUNCH_CHECK(ctx);
    return FHGS_OK;
}
