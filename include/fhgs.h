/*
 * fhgs.h -- C ABI of the FHGS hot path for NVIDIA B200 (sm_100a).
 *
 * FHGS = Feature-Homogenized Gaussian Splatting (arxiv 2505.19154).  The library implements the
 * data-parallel hot path: tile-based Gaussian-splatting rasterisation that carries a D-channel
 * feature per primitive next to RGB, plus weight-aggregated feature fusion.  Citations are
 * "PAPER.md:<line>" / "SPEC.md:<line>" of the reference texts and "SURVEY 8(x)" / "DESIGN.md" for
 * the readings taken where the paper is silent.
 *
 * Conventions shared by every call
 *   - Every pointer inside fhgs_gaussians / fhgs_view_state and every image / accumulator pointer
 *     is a DEVICE pointer owned by the caller.  The library never allocates, frees or keeps them.
 *     fhgs_camera and fhgs_params are HOST structs, read during the call.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every call
 *     only enqueues work on `stream` and returns, except fhgs_bin_sort with a non-NULL
 *     num_instances_host, fhgs_frame_host and fhgs_ffma_peak, which synchronise `stream`.
 *     No entry point other than those three synchronises, allocates device memory or uses the legacy stream on its
 *     own, so a sequence of calls on one stream can be captured into a CUDA graph (fhgs_bin_sort forks onto the
 *     context's side stream and joins back with events inside the call, which capture follows).
 *   - Arrays are row-major.  Images are channel-last [H,W,C].  Tiles are 16x16 px
 *     (PAPER.md:302), tile_id = ty * GW + tx with GW = ceil(W/16), GH = ceil(H/16).
 *   - Camera: view[16] = world->camera, row-major, applied to column vectors; camera frame is
 *     +x right, +y down, +z forward.  proj[16] row-major with w_clip = z_cam; only proj[0], [2],
 *     [5], [6] are used:  fx = proj[0]*W/2, fy = proj[5]*H/2, cx = (proj[2]+1)*W/2 - 1/2,
 *     cy = (proj[6]+1)*H/2 - 1/2 (each evaluated in double, rounded once to float).  Pixel (x,y)
 *     is sampled at continuous coordinate (x,y) (integer = pixel centre).
 *   - Return value: FHGS_OK, or an error; fhgs_last_error(ctx) gives the text.  Nothing is
 *     enqueued when FHGS_ERR_INVALID is returned.
 *   - There is no CPU fallback anywhere: a missing/unsuitable CUDA device is FHGS_ERR_INTERNAL.
 */
#ifndef FHGS_H_
#define FHGS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define FHGS_API __attribute__((visibility("default")))
#else
#define FHGS_API
#endif

typedef enum {
    FHGS_OK = 0,
    FHGS_ERR_INTERNAL = 1, /* CUDA failure (launch, runtime, no device) */
    FHGS_ERR_INVALID = 2,  /* bad argument, shape, dtype or alignment; nothing was enqueued */
    FHGS_ERR_CAPACITY = 3  /* instance buffers too small (only reported by a synchronous bin_sort) */
} fhgs_status;

/* Storage types of feature rows, ground-truth maps and feature outputs; the arithmetic is fp32 throughout.  FHGS_BF16
 * (SURVEY 8(f) NEXT-4 iv) is accepted by fhgs_render, fhgs_fuse_features and fhgs_frame_host; the NDFD entry points take
 * FHGS_F32 / FHGS_F16 only. */
typedef enum { FHGS_F32 = 0, FHGS_F16 = 1, FHGS_BF16 = 2 } fhgs_dtype;

/* Opaque context: device ordinal, SM count, last-error text, two copy streams + events used only by fhgs_frame_host,
 * and one side stream + events on which fhgs_bin_sort runs two small scans beside its depth pre-sort (forked from and
 * joined back into the caller's stream with events inside the call).  Owns no device memory.  A context serves one host
 * thread at a time (use one context per thread / per stream that is driven concurrently). */
typedef struct fhgs_ctx fhgs_ctx;

FHGS_API fhgs_status fhgs_create(fhgs_ctx** out, int device);
FHGS_API void fhgs_destroy(fhgs_ctx* ctx);
/* Valid until the next call on this ctx.  Never NULL. */
FHGS_API const char* fhgs_last_error(const fhgs_ctx* ctx);
/* "fhgs-b200 <version> sm_100a" -- callable without a device. */
FHGS_API const char* fhgs_version(void);

/* The Gaussian primitives theta_i = {p, R, S, op, c, f} of PAPER.md:77-80 (Eq. 1), with the
 * north_star's 3-axis scale and SH colour.  scale and opacity are ACTIVATED
 * values (scale > 0, opacity in [0,1]); quat is (w,x,y,z) and need not be unit. */
typedef struct {
    int32_t n;          /* number of Gaussians, >= 0 */
    int32_t sh_degree;  /* 0..3; K = (sh_degree+1)^2 coefficients per colour channel */
    int32_t feat_dim;   /* D > 0, multiple of 4 (f32) or 8 (f16, bf16); ignored when feat == NULL */
    int32_t feat_dtype; /* fhgs_dtype of `feat` */
    const float* mean;    /* [n,3] */
    const float* scale;   /* [n,3] */
    const float* quat;    /* [n,4] */
    const float* opacity; /* [n]   */
    const float* sh;      /* [n,K,3] coefficient-major, RGB-minor */
    const void* feat;     /* [n,D] f32, f16 or bf16, 16-byte aligned; NULL for RGB-only rendering */
} fhgs_gaussians;

typedef struct {
    float view[16];
    float proj[16];
    float cam_pos[3];
    int32_t width, height; /* > 0; ceil(W/16)*ceil(H/16) must be < 2^31 */
} fhgs_camera;

/* Constants of the method.  Call fhgs_default_params() then override. */
typedef struct {
    float z_near;       /* 0.2     cull z_cam < z_near                                   */
    float cov_dilation; /* 0.3     px^2 added to the 2-D covariance diagonal (EWA low-pass) */
    float jac_clamp;    /* 1.3     clamp of x/z, y/z (in units of tan(fov/2)) for the Jacobian */
    float q_cutoff;     /* 9       a Gaussian contributes to a pixel iff q <= q_cutoff (3 sigma) */
    float alpha_max;    /* 0.9999  alpha = min(alpha_max, op*G)   */
    float t_min;        /* 1e-4    stop a pixel once T < t_min   */
    float den_eps;      /* 1e-8    a Gaussian is fused only if den > den_eps               */
    float bg[3];        /* 0,0,0   background colour, rgb += T_final * bg   */
    int32_t rect_mode;  /* FHGS_RECT_RADIUS (default): tile rectangle from the scalar radius ceil(3 sqrt(lambda_max)), as
                           north_star states it; FHGS_RECT_TIGHT: from the per-axis 3-sigma extents ceil(3 sqrt(Sigma_xx)),
                           ceil(3 sqrt(Sigma_yy)) -- the exact bounding box of the q <= 9 ellipse, so the images and fused
                           vectors are the same while step S handles ~40 % fewer instances (SURVEY 8(f) NEXT-4 i)        */
    int32_t primitive;  /* FHGS_PRIM_EWA (default): 3-axis Gaussian, EWA projection (north_star).  FHGS_PRIM_SURFEL:
                           the paper's own 2-D surfel with exact ray-splat intersection (Eq. 1-3;
                           SURVEY 8(f) NEXT-3): scale[:,0:2] = (s_u, s_v), scale[:,2] is ignored                        */
} fhgs_params;
enum { FHGS_RECT_RADIUS = 0, FHGS_RECT_TIGHT = 1 };
enum { FHGS_PRIM_EWA = 0, FHGS_PRIM_SURFEL = 1 };
FHGS_API void fhgs_default_params(fhgs_params* p);

/* Per-view intermediate state.  All pointers are device pointers owned by the caller.
 * fhgs_project writes xy..tiles_touched; fhgs_bin_sort writes offsets, num_instances,
 * keys/vals (ping-pong), sorted_buf, ranges; fhgs_render / fhgs_fuse_features / fhgs_ndfd_* read them and use
 * per-entry-point work-queue words inside `scratch`: ONE fhgs_render and ONE fhgs_fuse_features on the same
 * view state may run concurrently on two streams; two calls of the same entry point on one view state, and any
 * call concurrent with fhgs_project / fhgs_bin_sort on it, must be stream-ordered.
 * `capacity` = number of (key,val) pairs each of keys[0],keys[1],vals[0],vals[1] can hold; it
 * must be < 2^30.  `scratch` needs fhgs_scratch_bytes(n, width, height, capacity) bytes, 256-byte
 * aligned. */
typedef struct {
    int32_t n, width, height;
    int32_t sorted_buf;      /* 0|1: which of keys[]/vals[] holds the sorted list (set by bin_sort) */
    uint64_t capacity;
    float* xy;               /* [n,2] pixel position of the centre                     */
    float* depth;            /* [n]   z_cam                                            */
    float* conic_opacity;    /* [n,4] inverse 2-D covariance (A,B,C) and opacity; 16-B aligned */
    float* rgb;              /* [n,3] SH colour evaluated for this camera              */
    int32_t* radius;         /* [n]   ceil(3 sqrt(lambda_max)) in px; 0 = culled       */
    uint16_t* rect;          /* [n,4] tile rectangle x0,y0,x1,y1 (x1,y1 exclusive); 8-B aligned */
    uint32_t* tiles_touched; /* [n]   (x1-x0)*(y1-y0); 0 = culled                      */
    uint32_t* offsets;       /* [n]   inclusive prefix sum of tiles_touched            */
    uint64_t* num_instances; /* [1]   M = offsets[n-1]                                 */
    uint64_t* keys[2];       /* [capacity] (tile_id << 32) | float_bits(z_cam)         */
    uint32_t* vals[2];       /* [capacity] Gaussian index                              */
    uint32_t* ranges;        /* [GW*GH,2] [first,last+1) into the sorted list; (0,0) = empty */
    void* scratch;
    size_t scratch_bytes;
    float* ray_transform;    /* [n,12] FHGS_PRIM_SURFEL only (else may be NULL): per splat the 3x3 matrix adj(T) of
                                PAPER.md Eq. 3, rows padded to float4 -- (u,v,1) ~ adj(T) (x,y,1)^T; 16-B aligned.
                                In surfel mode xy holds the centre of the footprint's bounding box and
                                conic_opacity = (half_x, half_y, 0, opacity) of that box */
} fhgs_view_state;

FHGS_API size_t fhgs_scratch_bytes(int32_t n, int32_t width, int32_t height, uint64_t capacity);
/* Diagnostics for the work accounting of SURVEY 8(d) (n_eval), off by default: after
 * fhgs_set_diagnostics(ctx, 1), fhgs_render also fills a uint32_t[GW*GH] array inside `scratch` (byte offset
 * returned by fhgs_scratch_tile_visited) with, per tile, the length of the prefix of the
 * tile's sorted list that was walked before every pixel of the tile had stopped (the whole list if
 * it never stopped; exact -- one past the last instance any pixel blended -- for D % 64 == 0,
 * rounded up to 256-instance chunks otherwise).  Same arguments as fhgs_scratch_bytes.  Not an output of the method. */
FHGS_API size_t fhgs_scratch_tile_visited(int32_t n, int32_t width, int32_t height, uint64_t capacity);
FHGS_API void fhgs_set_diagnostics(fhgs_ctx* ctx, int enable);

/* Step P -- PAPER.md:302 (CullGaussian), PAPER.md:309-310 (2DScreenGaussians); EWA reading
 * per Gaussian, camera-space position, cull (z < z_near, det <= 0, non-finite,
 * zero tiles), Sigma2D = J R_v Sigma3D R_v^T J^T + dilation*I, conic = Sigma2D^-1,
 * radius = ceil(3 sqrt(lambda_max)), tile rectangle, SH -> RGB.  Every floating-point operation
 * is a single IEEE binary32 operation in the order C1-P states (no FMA contraction), so the
 * integer outputs are reproducible bit for bit.  A culled Gaussian gets radius = 0,
 * tiles_touched = 0, rect = 0 and zeros in the float outputs.
 * Reads g->{mean,scale,quat,opacity,sh}; writes vs->{xy,depth,conic_opacity,rgb,radius,rect,
 * tiles_touched}; sets vs->n/width/height must equal g->n / cam->width / cam->height.
 * prm->primitive == FHGS_PRIM_SURFEL: the paper's 2-D surfel: centre p, tangents
 * t_u, t_v = columns 0, 1 of R(quat), scales (s_u, s_v) = scale[:,0:2]; P(u,v) = p + s_u t_u u + s_v t_v v (Eq. 2) and
 * the pixel's (u,v) from the exact ray-splat intersection (Eq. 3) through the homography T = K [R_v s_u t_u, R_v s_v t_v,
 * c]; G = exp(-(u^2+v^2)/2).  Writes vs->ray_transform = adj(T) (scaled by a power of two), the footprint's bounding
 * box (dual conic) into xy / conic_opacity / radius / rect, depth = z of the centre.  Culled: centre or any point of the
 * 3-sigma disc in front of z_near, degenerate transform.  No low-pass filter (the paper states none).  Steps S, R, F
 * run unchanged on the result (R, F evaluate u^2+v^2 from ray_transform when prm->primitive says so). */
FHGS_API fhgs_status fhgs_project(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                         const fhgs_params* prm, fhgs_view_state* vs, void* stream);

/* Step S -- PAPER.md:302, 312-314 (DuplicateWithKeys, SortByKeys, IdentifyTileRanges); SURVEY
 * 8(c) C1-S: inclusive prefix sum of tiles_touched (single pass, decoupled look-back) -> offsets
 * and M; one (key,val) per (Gaussian, tile of its rect), tiles in row-major order,
 * key = (tile_id << 32) | bits(z_cam); STABLE least-significant-digit radix sort (onesweep, 8-bit
 * digits) so that equal keys keep ascending Gaussian index; tile ranges.
 * If M > capacity nothing after the scan is produced: *num_instances = M, ranges all zero.
 * num_instances_host: NULL = fully asynchronous; else the call synchronises `stream`, stores M
 * and returns FHGS_ERR_CAPACITY if M > capacity.  Zero visible Gaussians is not an error
 * (SPEC.md:187): M = 0 and every range is (0,0).
 * `flags`: 0 = default; FHGS_SORT_FULL_KEY forces LSD passes over all significant key bits
 * (the default pre-orders Gaussians by depth bits and then runs only the tile-id digit passes
 * over the 64-bit keys; both give the same, unique, sorted list). */
enum { FHGS_SORT_FULL_KEY = 1 };
FHGS_API fhgs_status fhgs_bin_sort(fhgs_ctx* ctx, const fhgs_camera* cam, fhgs_view_state* vs,
                          uint64_t* num_instances_host, uint32_t flags, void* stream);

/* Step R -- PAPER.md:90-95 (Eq. 4: c(x) = sum_i c_i w_i, w_i = alpha_i T_i, alpha_i = op_i G_i,
 * T_i = prod_{j<i}(1 - alpha_j)), PAPER.md:335 (front-to-back), G = exp(-q/2);
 * per pixel walk its tile's range; stop once T < t_min; skip unless
 * q <= q_cutoff; alpha = min(alpha_max, op*G); C += w*rgb; F += w*f; T *= 1 - alpha.
 * out_rgb  [H,W,3] f32 = C + T*bg                      (required)
 * out_feat [H,W,D] dtype of g->feat = F, unnormalised, no background; NULL = skip
 * out_T    [H,W]   f32 final transmittance; NULL = skip
 * out_ncontrib [H,W] u32 number of blended Gaussians; NULL = skip
 * Uses vs->{xy,conic_opacity,rgb,ranges,vals[sorted_buf]} and g->{feat,feat_dim,feat_dtype}. */
FHGS_API fhgs_status fhgs_render(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                        const fhgs_params* prm, const fhgs_view_state* vs, float* out_rgb,
                        void* out_feat, float* out_T, uint32_t* out_ncontrib, void* stream);

/* Step F -- weight-aggregated feature fusion (north_star; weights w_i(x) = alpha_i T_i of
 * PAPER.md:95, identical to step R's):
 *     num[i,:] += sum_x w_i(x) * gt[x,:],   den[i] += sum_x w_i(x)
 * accumulated over every view passed (caller keeps num/den between calls -- the paper's
 * "cumulative-weight buffers").  Order of the floating-point atomic adds is free.
 * flags: FHGS_FUSE_ZERO clears num,den first; FHGS_FUSE_FINALIZE then writes
 * out_feat[i,:] = num[i,:]/den[i] for every i with den[i] > den_eps and leaves other rows of
 * out_feat untouched; FHGS_FUSE_L2NORM additionally divides finalised rows by their L2 norm
 * (PAPER.md:136 unit-norm features; off by default).  FHGS_FUSE_FINALIZE_ONLY skips the
 * accumulation of a view (gt, cam may then be NULL) and only finalises.  FHGS_FUSE_ZERO_ONLY
 * clears num,den and returns (cam, gt, out_feat may be NULL) -- lets a caller time the three
 * parts of a fused frame separately.  FHGS_FUSE_ZERO_TOUCHED (with ZERO or ZERO_ONLY) clears only the rows with
 * den[i] != 0 instead of the whole accumulator: only valid when every row with den[i] == 0 is already zero in num,
 * which holds for buffers that were last cleared by this call and since then written by it only (a Gaussian gets
 * num without den only from an all-zero weight, i.e. never); at Mid 2 % of the rows carry weight.
 * gt [H,W,D] gt_dtype, 16-byte aligned; num [n,D] f32 16-byte aligned; den [n] f32;
 * out_feat [n,D] out_dtype or NULL. */
enum {
    FHGS_FUSE_ZERO = 1,
    FHGS_FUSE_FINALIZE = 2,
    FHGS_FUSE_L2NORM = 4,
    FHGS_FUSE_FINALIZE_ONLY = 8,
    FHGS_FUSE_ZERO_ONLY = 16,
    FHGS_FUSE_ZERO_TOUCHED = 32
};
FHGS_API fhgs_status fhgs_fuse_features(fhgs_ctx* ctx, const fhgs_camera* cam, const fhgs_params* prm,
                               const fhgs_view_state* vs, const void* gt, int32_t feat_dim,
                               int32_t gt_dtype, float* num, float* den, void* out_feat,
                               int32_t out_dtype, uint32_t flags, void* stream);

/* NDFD forward -- the paper's non-differentiable feature driving losses
 * (Eq. 5-6) and PAPER.md:305-335 (Alg. 2), evaluated per pixel x in the SAME front-to-back traversal as
 * step R (same q cut-off, alpha clamp, w_i = alpha_i T_i, stop once T < t_min), with f_gt = gt[x,:]:
 *     phi_i = f_i . f_gt (features unit-norm),  sigma_i = 1 / (1 + exp(k (phi_i - lambda)))
 *     out_lgt[x] = sum_i w_i sigma_i                                   (Eq. 5)
 *     out_lcf[x] = sum_i sigma_i w_i (W_{i-1} - F_{i-1} . f_i)          (Eq. 6)
 * where W_n = sum_{i<=n} w_i, F_n = sum_{i<=n} w_i f_i are accumulated
 *   mode = FHGS_NDFD_BLEND_ORDER:  in blend order, front to back ("updated one time in each step during the
 *          front-to-back blend");
 *   mode = FHGS_NDFD_FAR_TO_NEAR:  "along the ray from far to near": the partners
 *          of fragment i are the fragments behind it.  Same single traversal (the sum is split around the ray totals).
 * The two readings give different L_cf; out_lgt is the same.  No feature image
 * is rendered.  Paper defaults: k = 20, lambda = 0.5.
 * g->feat [n,D] f32/f16 and gt [H,W,D] f32/f16, both 16-byte aligned; D in {32,64,128,256,512};
 * out_lgt, out_lcf [H,W] f32 (every pixel is written; pixels no Gaussian reaches get 0).
 * Uses vs->{xy,conic_opacity,ranges,vals[sorted_buf]} as fhgs_render does. */
enum { FHGS_NDFD_BLEND_ORDER = 0, FHGS_NDFD_FAR_TO_NEAR = 1 };
FHGS_API fhgs_status fhgs_ndfd_forward(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                              const fhgs_params* prm, const fhgs_view_state* vs, const void* gt,
                              int32_t gt_dtype, float k_sigmoid, float lambda, int32_t mode, float* out_lgt,
                              float* out_lcf, void* stream);

/* NDFD backward at the w level -- PAPER.md:142-146 and appendix A.2.
 * With L = sum_x ( lam1 out_lgt[x] + lam2 out_lcf[x] ) of fhgs_ndfd_forward, per pixel and fragment k in blend order
 *     dL/dw_k     = lam1 sigma_k + lam2 [ sigma_k (W_{k-1} - F_{k-1}.f_k) + sum_{i>k} sigma_i w_i (1 - f_i.f_k) ]
 *     dL/dalpha_k = T_k dL/dw_k - (1/(1 - alpha_k)) sum_{j>k} dL/dw_j w_j
 * and the result is the opacity gradient  grad_opacity[g] += sum_x dL/dalpha_k(x) G_k(x)  over the fragments k of
 * Gaussian g that are not clamped at alpha_max (alpha = min(alpha_max, op G)).  The realised fragment lists
 * (cut-off, stopping rule) are not differentiated; the geometry chain (dG/d mean, scale, rotation) is out of scope.
 * grad_opacity [n] f32 is ACCUMULATED into (the caller zeroes it; atomic order is free).
 * work: device scratch of fhgs_ndfd_backward_work_bytes(width, height, D) bytes, 256-byte aligned (per-pixel
 * totals of the three forward traversals the first path uses).  D in {32,64,128,256}; other arguments as
 * fhgs_ndfd_forward.  Both NDFD calls also run in surfel mode (prm->primitive = FHGS_PRIM_SURFEL; f32 features and map). */
FHGS_API size_t fhgs_ndfd_backward_work_bytes(int32_t width, int32_t height, int32_t feat_dim);
FHGS_API fhgs_status fhgs_ndfd_backward(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam,
                               const fhgs_params* prm, const fhgs_view_state* vs, const void* gt,
                               int32_t gt_dtype, float k_sigmoid, float lambda, float lam1, float lam2,
                               float* grad_opacity, void* work, size_t work_bytes, void* stream);

/* One whole frame (P -> S -> R -> F with ZERO|FINALIZE) from HOST buffers: copies the Gaussian
 * arrays and the GT map host->device into `dev_g` / `dev_gt` (device staging owned by the
 * caller, same shapes), runs the four steps on `stream`, copies out_rgb / out_feat /
 * fused_feat device->host and synchronises.  Every *_host pointer is HOST memory (pinned memory
 * makes the copies asynchronous); dev_* are DEVICE pointers.  NULL host outputs are skipped.
 * The copies run on the context's own copy streams, ordered against `stream` with events, so that
 * host->device, device->host and the steps overlap (feature table behind P/S, GT map and the image
 * read-back behind R/F); on return everything has completed.
 * This is the end-to-end entry bench.py times; it performs no arithmetic of its own. */
typedef struct {
    const float *mean, *scale, *quat, *opacity, *sh; /* HOST, shapes as fhgs_gaussians */
    const void* feat;                                /* HOST [n,D] */
    const void* gt;                                  /* HOST [H,W,D] */
    float* out_rgb;                                  /* HOST [H,W,3] or NULL */
    void* out_feat;                                  /* HOST [H,W,D] or NULL */
    void* fused_feat;                                /* HOST [n,D] or NULL   */
} fhgs_host_frame;
typedef struct {
    float* out_rgb;   /* DEVICE [H,W,3] */
    void* out_feat;   /* DEVICE [H,W,D] */
    void* gt;         /* DEVICE [H,W,D] */
    float* num;       /* DEVICE [n,D]   */
    float* den;       /* DEVICE [n]     */
    void* fused_feat; /* DEVICE [n,D]   */
} fhgs_frame_workspace;
FHGS_API fhgs_status fhgs_frame_host(fhgs_ctx* ctx, const fhgs_host_frame* host, const fhgs_gaussians* dev_g,
                            const fhgs_camera* cam, const fhgs_params* prm, fhgs_view_state* vs,
                            const fhgs_frame_workspace* ws, uint64_t* num_instances_host,
                            void* stream);

/* Steps R and F in ONE traversal with one weight phase (SURVEY 8(f) NEXT-4 ii; the same w = alpha T serves
 * the rendered sums and the fused sums): equivalent to fhgs_render(..., out_feat, ...) followed by
 * fhgs_fuse_features(..., flags = 0) on the same view state -- images bit-identical, num / den equal up to the order of their
 * floating-point atomics.  Available in the per-pixel regime only: feat_dim NOT a multiple of 64 (FHGS_ERR_INVALID otherwise;
 * the tiled kernels cannot hold both working sets).  gt [H,W,D] has the storage type of g->feat; out_rgb,
 * out_feat, gt, num [n,D] f32 and den [n] f32 are required and are NOT cleared (accumulation over views as in step F);
 * out_T / out_ncontrib may be NULL. */
FHGS_API fhgs_status fhgs_render_fuse(fhgs_ctx* ctx, const fhgs_gaussians* g, const fhgs_camera* cam, const fhgs_params* prm,
                             const fhgs_view_state* vs, float* out_rgb, void* out_feat, float* out_T, uint32_t* out_ncontrib,
                             const void* gt, float* num, float* den, void* stream);

/* Allocation-free variant of step S1's prefix sum (DuplicateWithKeys needs, per Gaussian, the
 * inclusive prefix sum of tiles_touched) for callers that cannot provide or allocate scratch memory
 * (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The decoupled look-back status words live in a
 * file-scope device array of the library (32 KB + 256 B, held by every GPU that loads the library until the process
 * exits) instead of fhgs_view_state::scratch; the call makes no cudaMalloc / cudaFree and no allocating library call.
 *   tiles_touched  DEVICE [n] uint32 (as written by fhgs_project);  offsets  DEVICE [n] uint32, offsets[i] =
 *   sum_{j<=i} tiles_touched[j] (mod 2^32, like fhgs_bin_sort's);  num_instances  DEVICE [1] uint64 or NULL, the total M.
 * n must be <= fhgs_scan_offsets_static_max_n() = 4 194 304, else FHGS_ERR_INVALID with nothing enqueued (use
 * fhgs_bin_sort with caller scratch beyond that).  n == 0 writes only *num_instances = 0.  The result is bit-identical to
 * the offsets / num_instances fhgs_bin_sort writes.  Every call shares the one array and clears the words it uses first:
 * calls on one device must be stream-ordered -- two calls that overlap on the GPU race on it.  Enqueues two kernels on
 * `stream` and returns. */
FHGS_API int32_t fhgs_scan_offsets_static_max_n(void);
FHGS_API fhgs_status fhgs_scan_offsets_static(fhgs_ctx* ctx, const uint32_t* tiles_touched, int32_t n, uint32_t* offsets,
                                     uint64_t* num_instances, void* stream);

/* Register-resident FFMA micro-benchmark ("the builder must first run a
 * register-resident FFMA micro-benchmark"): returns the measured FP32 rate in lane-ops/s
 * (one FMA = one lane-op) in *lane_ops_per_s and the kernel time in *ms.  Synchronises. */
FHGS_API fhgs_status fhgs_ffma_peak(fhgs_ctx* ctx, int32_t iters, double* lane_ops_per_s, double* ms,
                           void* stream);

#ifdef __cplusplus
}
#endif
#endif /* FHGS_H_ */
