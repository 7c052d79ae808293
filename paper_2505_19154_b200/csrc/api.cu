// api.cu -- context, validation, scratch sizing, the host-buffer frame entry and the FFMA
// micro-benchmark of libfhgs.so (declared in include/fhgs.h).
#include <math.h>
#include <new>

#include "common.cuh"
#include "layout.cuh"

extern "C" const char* fhgs_version(void) { return "fhgs-b200 0.1 sm_100a"; }

extern "C" fhgs_status fhgs_create(fhgs_ctx** out, int device) {
    if (!out) return FHGS_ERR_INVALID;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return FHGS_ERR_INTERNAL;
    fhgs_ctx* c = new (std::nothrow) fhgs_ctx();
    if (!c) return FHGS_ERR_INTERNAL;
    c->device = device;
    c->err[0] = 0;
    c->diagnostics = 0;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete c; return FHGS_ERR_INTERNAL; }
    c->num_sms = prop.multiProcessorCount;
    c->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    if (prop.major < 10) {   // sm_100a only: there is no fallback path
        delete c;
        return FHGS_ERR_INTERNAL;
    }
    if (cudaSetDevice(device) != cudaSuccess) { delete c; return FHGS_ERR_INTERNAL; }
    c->copy_in = c->copy_out = nullptr;
    c->ev_start = c->ev_feat = c->ev_gt = c->ev_render = c->ev_out = nullptr;
    c->side = nullptr;
    c->ev_fork = c->ev_offsets = c->ev_tiles = nullptr;
    bool ok = cudaStreamCreateWithFlags(&c->copy_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->copy_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) == cudaSuccess;
    for (cudaEvent_t* e : {&c->ev_start, &c->ev_feat, &c->ev_gt, &c->ev_render, &c->ev_out, &c->ev_fork, &c->ev_offsets, &c->ev_tiles})
        ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { fhgs_destroy(c); return FHGS_ERR_INTERNAL; }   // releases whatever was created
    *out = c;
    return FHGS_OK;
}

extern "C" void fhgs_destroy(fhgs_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard dg(ctx);
    if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
    if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    for (cudaEvent_t e : {ctx->ev_start, ctx->ev_feat, ctx->ev_gt, ctx->ev_render, ctx->ev_out, ctx->ev_fork, ctx->ev_offsets, ctx->ev_tiles})
        if (e) cudaEventDestroy(e);
    delete ctx;
}

extern "C" void fhgs_set_diagnostics(fhgs_ctx* ctx, int enable) {
    if (ctx) ctx->diagnostics = enable ? 1 : 0;
}

extern "C" const char* fhgs_last_error(const fhgs_ctx* ctx) { return ctx ? ctx->err : "NULL context"; }

extern "C" void fhgs_default_params(fhgs_params* p) {
    if (!p) return;
    p->z_near = 0.2f;
    p->cov_dilation = 0.3f;
    p->jac_clamp = 1.3f;
    p->q_cutoff = 9.0f;
    p->alpha_max = 0.9999f;
    p->t_min = 1e-4f;
    p->den_eps = 1e-8f;
    p->bg[0] = p->bg[1] = p->bg[2] = 0.0f;
    p->rect_mode = FHGS_RECT_RADIUS;
    p->primitive = FHGS_PRIM_EWA;
}

extern "C" size_t fhgs_scratch_bytes(int32_t n, int32_t width, int32_t height, uint64_t capacity) {
    if (n < 0 || width <= 0 || height <= 0) return 0;
    return make_scratch_layout(n, capacity, width, height).total;
}

extern "C" size_t fhgs_scratch_tile_visited(int32_t n, int32_t width, int32_t height, uint64_t capacity) {
    if (n < 0 || width <= 0 || height <= 0) return 0;
    return make_scratch_layout(n, capacity, width, height).tile_visited;
}

fhgs_status validate_camera(fhgs_ctx* ctx, const fhgs_camera* cam) {
    if (cam->width <= 0 || cam->height <= 0) FHGS_INVALID(ctx, "camera: width/height must be > 0");
    const long long tiles = (long long)tiles_x(cam->width) * tiles_y(cam->height);
    if (tiles >= (1LL << 31)) FHGS_INVALID(ctx, "camera: too many tiles for the 32-bit tile id");
    if (tiles_x(cam->width) > 65535 || tiles_y(cam->height) > 65535)
        FHGS_INVALID(ctx, "camera: more than 65535 tiles along one axis (rect is uint16)");
    for (int i = 0; i < 16; ++i)
        if (!finite_f(cam->view[i]) || !finite_f(cam->proj[i])) FHGS_INVALID(ctx, "camera: non-finite matrix entry");
    for (int i = 0; i < 3; ++i)
        if (!finite_f(cam->cam_pos[i])) FHGS_INVALID(ctx, "camera: non-finite cam_pos");
    if (!(cam->proj[0] != 0.0f) || !(cam->proj[5] != 0.0f)) FHGS_INVALID(ctx, "camera: proj[0]/proj[5] must be non-zero");
    return FHGS_OK;
}

fhgs_status validate_params(fhgs_ctx* ctx, const fhgs_params* p) {
    const float v[10] = {p->z_near, p->cov_dilation, p->jac_clamp, p->q_cutoff, p->alpha_max,
                         p->t_min, p->den_eps, p->bg[0], p->bg[1], p->bg[2]};
    for (int i = 0; i < 10; ++i)
        if (!finite_f(v[i])) FHGS_INVALID(ctx, "params: non-finite value");
    if (!(p->z_near > 0.0f)) FHGS_INVALID(ctx, "params: z_near must be > 0 (depth bits must order like depth)");
    if (!(p->q_cutoff >= 0.0f) || !(p->alpha_max > 0.0f && p->alpha_max < 1.0f) || !(p->t_min >= 0.0f))
        FHGS_INVALID(ctx, "params: q_cutoff >= 0, 0 < alpha_max < 1, t_min >= 0 required");   // 1/(1-alpha) in the backward
    if (p->rect_mode != FHGS_RECT_RADIUS && p->rect_mode != FHGS_RECT_TIGHT) FHGS_INVALID(ctx, "params: unknown rect_mode");
    if (p->primitive != FHGS_PRIM_EWA && p->primitive != FHGS_PRIM_SURFEL) FHGS_INVALID(ctx, "params: unknown primitive");
    return FHGS_OK;
}

fhgs_status validate_view_state(fhgs_ctx* ctx, const fhgs_view_state* vs, const fhgs_camera* cam) {
    if (vs->n < 0 || vs->n >= (1 << 30)) FHGS_INVALID(ctx, "view_state: n must be in [0, 2^30)");   // 30-bit packed counts
    if (cam && (vs->width != cam->width || vs->height != cam->height))
        FHGS_INVALID(ctx, "view_state: width/height differ from the camera's");
    if (vs->capacity >= (1ull << 30)) FHGS_INVALID(ctx, "view_state: capacity must be < 2^30");
    if (!vs->xy || !vs->depth || !vs->conic_opacity || !vs->rgb || !vs->radius || !vs->rect ||
        !vs->tiles_touched || !vs->offsets || !vs->num_instances || !vs->ranges || !vs->scratch)
        FHGS_INVALID(ctx, "view_state: NULL buffer");
    if (vs->capacity > 0 && (!vs->keys[0] || !vs->keys[1] || !vs->vals[0] || !vs->vals[1]))
        FHGS_INVALID(ctx, "view_state: NULL key/value buffer");
    if (!aligned_to(vs->conic_opacity, 16) || !aligned_to(vs->xy, 8) || !aligned_to(vs->rect, 8) ||
        !aligned_to(vs->keys[0], 16) || !aligned_to(vs->keys[1], 16) || !aligned_to(vs->vals[0], 16) || !aligned_to(vs->vals[1], 16) || !aligned_to(vs->ranges, 8) ||
        !aligned_to(vs->scratch, 256) || !aligned_to(vs->num_instances, 8))
        FHGS_INVALID(ctx, "view_state: misaligned buffer");
    if (vs->scratch_bytes < fhgs_scratch_bytes(vs->n, vs->width, vs->height, vs->capacity))
        FHGS_INVALID(ctx, "view_state: scratch too small (see fhgs_scratch_bytes)");
    return FHGS_OK;
}

// ------------------------------------------------------------------------------------------------
// Host-buffer frame: copies in, P -> S -> R -> F, copies out.  No arithmetic here.
// ------------------------------------------------------------------------------------------------
extern "C" fhgs_status fhgs_frame_host(fhgs_ctx* ctx, const fhgs_host_frame* host, const fhgs_gaussians* g,
                                       const fhgs_camera* cam, const fhgs_params* prm, fhgs_view_state* vs,
                                       const fhgs_frame_workspace* ws, uint64_t* num_instances_host,
                                       void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (!host || !g || !cam || !prm || !vs || !ws) FHGS_INVALID(ctx, "fhgs_frame_host: NULL argument");
    if (g->n < 0 || g->sh_degree < 0 || g->sh_degree > 3 || !g->feat || g->feat_dim <= 0)
        FHGS_INVALID(ctx, "fhgs_frame_host: bad Gaussian description");
    if (!host->mean || !host->scale || !host->quat || !host->opacity || !host->sh || !host->feat || !host->gt)
        FHGS_INVALID(ctx, "fhgs_frame_host: NULL host input");
    if (!ws->out_rgb || !ws->out_feat || !ws->gt || !ws->num || !ws->den || !ws->fused_feat)
        FHGS_INVALID(ctx, "fhgs_frame_host: NULL workspace buffer");
    // Everything that can be rejected is rejected HERE, before the first event record or copy (fhgs.h: "Nothing is
    // enqueued when FHGS_ERR_INVALID is returned"): the same checks the four steps repeat on entry.
    fhgs_status st;
    if ((st = validate_camera(ctx, cam)) != FHGS_OK) return st;
    if ((st = validate_params(ctx, prm)) != FHGS_OK) return st;
    if ((st = validate_view_state(ctx, vs, cam)) != FHGS_OK) return st;
    if (g->n != vs->n) FHGS_INVALID(ctx, "fhgs_frame_host: g->n != vs->n");
    if (!g->mean || !g->scale || !g->quat || !g->opacity || !g->sh) FHGS_INVALID(ctx, "fhgs_frame_host: NULL device Gaussian array");
    if (g->feat_dtype != FHGS_F32 && g->feat_dtype != FHGS_F16 && g->feat_dtype != FHGS_BF16)
        FHGS_INVALID(ctx, "fhgs_frame_host: unknown feat_dtype");
    if (g->feat_dim % (g->feat_dtype == FHGS_F32 ? 4 : 8)) FHGS_INVALID(ctx, "fhgs_frame_host: feat_dim must be a multiple of 4 (f32) / 8 (f16, bf16)");
    if (!aligned_to(g->feat, 16) || !aligned_to(ws->out_feat, 16) || !aligned_to(ws->gt, 16) || !aligned_to(ws->num, 16) ||
        !aligned_to(ws->den, 4) || !aligned_to(ws->fused_feat, 16))
        FHGS_INVALID(ctx, "fhgs_frame_host: feat / workspace buffers must be 16-byte aligned");
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = (size_t)g->n, K = (size_t)(g->sh_degree + 1) * (g->sh_degree + 1);
    const size_t e = g->feat_dtype == FHGS_F32 ? 4 : 2, D = (size_t)g->feat_dim;
    const size_t px = (size_t)cam->width * cam->height;
    uint64_t m = 0;
    // Schedule (three streams, so that PCIe runs in both directions while the steps execute):
    //   s        : H2D geometry -> P -> S -> [wait feat] R -> [wait gt] F -> D2H fused -> [wait image copies]
    //   copy_in  : H2D feat -> H2D gt                      (behind everything already enqueued on s)
    //   copy_out : [wait R] D2H rgb, feature image         (overlaps H2D gt and F)
    // Once anything is enqueued, every exit -- also an error exit -- first drains s, copy_in and copy_out, so that no
    // DMA is still running against the caller's host buffers or device staging when the call returns.
    st = [&]() -> fhgs_status {
        FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_start, s));
        FHGS_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_in, ctx->ev_start, 0));
        FHGS_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ctx->ev_start, 0));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->mean, host->mean, n * 12, cudaMemcpyHostToDevice, s));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->scale, host->scale, n * 12, cudaMemcpyHostToDevice, s));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->quat, host->quat, n * 16, cudaMemcpyHostToDevice, s));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->opacity, host->opacity, n * 4, cudaMemcpyHostToDevice, s));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->sh, host->sh, n * K * 12, cudaMemcpyHostToDevice, s));
        FHGS_CUDA(ctx, cudaMemcpyAsync((void*)g->feat, host->feat, n * D * e, cudaMemcpyHostToDevice, ctx->copy_in));
        FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_feat, ctx->copy_in));
        FHGS_CUDA(ctx, cudaMemcpyAsync(ws->gt, host->gt, px * D * e, cudaMemcpyHostToDevice, ctx->copy_in));
        FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_gt, ctx->copy_in));
        fhgs_status r;
        if ((r = fhgs_project(ctx, g, cam, prm, vs, stream)) != FHGS_OK) return r;
        if ((r = fhgs_bin_sort(ctx, cam, vs, nullptr, 0, stream)) != FHGS_OK) return r;
        FHGS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_feat, 0));
        if ((r = fhgs_render(ctx, g, cam, prm, vs, ws->out_rgb, ws->out_feat, nullptr, nullptr, stream)) != FHGS_OK) return r;
        FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_render, s));
        FHGS_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ctx->ev_render, 0));
        if (host->out_rgb) FHGS_CUDA(ctx, cudaMemcpyAsync(host->out_rgb, ws->out_rgb, px * 12, cudaMemcpyDeviceToHost, ctx->copy_out));
        if (host->out_feat) FHGS_CUDA(ctx, cudaMemcpyAsync(host->out_feat, ws->out_feat, px * D * e, cudaMemcpyDeviceToHost, ctx->copy_out));
        FHGS_CUDA(ctx, cudaEventRecord(ctx->ev_out, ctx->copy_out));
        FHGS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_gt, 0));
        if ((r = fhgs_fuse_features(ctx, cam, prm, vs, ws->gt, g->feat_dim, g->feat_dtype, ws->num, ws->den,
                                    ws->fused_feat, g->feat_dtype, FHGS_FUSE_ZERO | FHGS_FUSE_FINALIZE, stream)) != FHGS_OK)
            return r;
        if (host->fused_feat) FHGS_CUDA(ctx, cudaMemcpyAsync(host->fused_feat, ws->fused_feat, n * D * e, cudaMemcpyDeviceToHost, s));
        FHGS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_out, 0));
        FHGS_CUDA(ctx, cudaMemcpyAsync(&m, vs->num_instances, 8, cudaMemcpyDeviceToHost, s));
        return FHGS_OK;
    }();
    // drain all three streams (copy_in / copy_out first: on an error path `s` may not be waiting for them)
    const cudaError_t d0 = cudaStreamSynchronize(ctx->copy_in), d1 = cudaStreamSynchronize(ctx->copy_out), d2 = cudaStreamSynchronize(s);
    if (st != FHGS_OK) return st;
    FHGS_CUDA(ctx, d0);
    FHGS_CUDA(ctx, d1);
    FHGS_CUDA(ctx, d2);
    if (num_instances_host) *num_instances_host = m;
    if (m > vs->capacity) return set_err(ctx, FHGS_ERR_CAPACITY, "fhgs_frame_host: %s%lld instances exceed capacity", "", (long long)m);
    return FHGS_OK;
}

// ------------------------------------------------------------------------------------------------
// FP32 micro-benchmark: 8 CTAs of 8 warps per SM, a register-resident outer-product tile per thread.
// The form is the fastest one found on this B200 (probe of scalar FFMA and fma.rn.f32x2 tiles of several shapes and
// operand orders): packed FFMA2, 2 pair operands x 16 broadcast scalars, the 64-bit pair operand
// held over 16 consecutive instructions (operand reuse cache) -- 125 of the nominal 128 FMA/clk/SM.  Scalar 8x8
// tiles reach 108-113, the 4-pair x 4-scalar order of the round-1 kernels 81.
// ------------------------------------------------------------------------------------------------
namespace {
constexpr int FFMA_FMA_PER_ROUND = 64;   // 2 pairs x 16 scalars x 2 lanes
__device__ __forceinline__ unsigned long long peak_pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__global__ void __launch_bounds__(256) ffma_peak_kernel(float* out, int iters, float a0, float b0) {
    unsigned long long acc[2][16], a[2], b[16];
#pragma unroll
    for (int i = 0; i < 2; ++i) a[i] = peak_pack2(a0 * (float)(threadIdx.x + i + 1), a0 * (float)(threadIdx.x + i + 2));
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const float v = b0 * (float)(threadIdx.x + 3 * j + 1);
        b[j] = peak_pack2(v, v);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[i][j] = 0ull;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 16; ++j) asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[i][j]) : "l"(a[i]), "l"(b[j]));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            float lo, hi;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(acc[i][j]));
            s += lo + hi;
        }
    if (s == 123.456f) out[0] = s;   // never true in practice; keeps the chains alive
}
}  // namespace

extern "C" fhgs_status fhgs_ffma_peak(fhgs_ctx* ctx, int32_t iters, double* lane_ops_per_s, double* ms, void* stream) {
    if (!ctx) return FHGS_ERR_INVALID;
    if (iters <= 0 || !lane_ops_per_s) FHGS_INVALID(ctx, "fhgs_ffma_peak: iters <= 0 or NULL output");
    DeviceGuard dg(ctx);
    cudaStream_t s = (cudaStream_t)stream;
    float* d = nullptr;
    FHGS_CUDA(ctx, cudaMalloc(&d, 4));
    const int grid = ctx->num_sms * 8;
    cudaEvent_t e0, e1;
    FHGS_CUDA(ctx, cudaEventCreate(&e0));
    FHGS_CUDA(ctx, cudaEventCreate(&e1));
    ffma_peak_kernel<<<grid, 256, 0, s>>>(d, iters / 4 + 1, 1e-6f, 1e-6f);   // warm-up
    FHGS_CUDA(ctx, cudaEventRecord(e0, s));
    ffma_peak_kernel<<<grid, 256, 0, s>>>(d, iters, 1e-6f, 1e-6f);
    FHGS_CUDA(ctx, cudaEventRecord(e1, s));
    FHGS_CUDA(ctx, cudaStreamSynchronize(s));
    FHGS_LAUNCH_CHECK(ctx);
    float t = 0.f;
    FHGS_CUDA(ctx, cudaEventElapsedTime(&t, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    const double ops = (double)grid * 256.0 * (double)iters * 4.0 * FFMA_FMA_PER_ROUND;
    *lane_ops_per_s = ops / ((double)t * 1e-3);
    if (ms) *ms = (double)t;
    return FHGS_OK;
}
