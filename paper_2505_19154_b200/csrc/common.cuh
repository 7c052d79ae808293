// common.cuh -- shared by the CUDA translation units of libfhgs.so (never by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "fhgs.h"

#define FHGS_TILE 16
#define FHGS_TILE_PX 256

struct fhgs_ctx {
    int device;
    int num_sms;
    int max_smem_optin;
    int diagnostics;   // fhgs_set_diagnostics: fhgs_render also fills the tile_visited array
    // fhgs_frame_host only: copy streams / events that overlap host<->device copies with the steps
    cudaStream_t copy_in, copy_out;
    cudaEvent_t ev_start, ev_feat, ev_gt, ev_render, ev_out;
    // fhgs_bin_sort only: the index-order offsets scan and the tile scan run beside the depth pre-sort on this stream
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_offsets, ev_tiles;
    char err[512];
};

// Every entry point that enqueues work makes the context's device current for the duration of the call and
// restores the caller's device afterwards (a process driving several GPUs may call with any device current).
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const fhgs_ctx* ctx) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// Pinhole intrinsics derived from proj[] (fhgs.h "Conventions"): double, rounded once.
struct Intrinsics {
    float fx, fy, cx, cy, tanx, tany;
};

static inline Intrinsics make_intrinsics(const fhgs_camera* cam) {
    Intrinsics k;
    const double W = (double)cam->width, H = (double)cam->height;
    k.fx = (float)((double)cam->proj[0] * W / 2.0);
    k.fy = (float)((double)cam->proj[5] * H / 2.0);
    k.cx = (float)(((double)cam->proj[2] + 1.0) * W / 2.0 - 0.5);
    k.cy = (float)(((double)cam->proj[6] + 1.0) * H / 2.0 - 0.5);
    k.tanx = (float)(1.0 / (double)cam->proj[0]);
    k.tany = (float)(1.0 / (double)cam->proj[5]);
    return k;
}

static inline fhgs_status set_err(fhgs_ctx* ctx, fhgs_status st, const char* fmt, const char* a = "",
                                  long long b = 0) {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), fmt, a, b);
    return st;
}

#define FHGS_INVALID(ctx, msg) return set_err((ctx), FHGS_ERR_INVALID, "%s", (msg))

#define FHGS_CUDA(ctx, expr)                                                                  \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess) {                                                             \
            snprintf((ctx)->err, sizeof((ctx)->err), "CUDA error %s at %s:%d (%s)",           \
                     cudaGetErrorName(e__), __FILE__, __LINE__, cudaGetErrorString(e__));     \
            return FHGS_ERR_INTERNAL;                                                         \
        }                                                                                     \
    } while (0)

#define FHGS_LAUNCH_CHECK(ctx) FHGS_CUDA(ctx, cudaGetLastError())

static inline bool finite_f(float v) { return v == v && v - v == 0.0f; }
static inline bool aligned_to(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

static inline int tiles_x(int w) { return (w + FHGS_TILE - 1) / FHGS_TILE; }
static inline int tiles_y(int h) { return (h + FHGS_TILE - 1) / FHGS_TILE; }

fhgs_status validate_camera(fhgs_ctx* ctx, const fhgs_camera* cam);
fhgs_status validate_params(fhgs_ctx* ctx, const fhgs_params* prm);
fhgs_status validate_view_state(fhgs_ctx* ctx, const fhgs_view_state* vs, const fhgs_camera* cam);
// FHGS_PRIM_SURFEL needs the per-splat ray transform in the view state
static inline fhgs_status validate_primitive(fhgs_ctx* ctx, const fhgs_params* prm, const fhgs_view_state* vs) {
    if (prm->primitive == FHGS_PRIM_SURFEL && (!vs->ray_transform || !aligned_to(vs->ray_transform, 16)))
        FHGS_INVALID(ctx, "surfel mode needs vs->ray_transform ([n,12] f32, 16-byte aligned)");
    return FHGS_OK;
}
