/* svr.h - C ABI of the B200-native differentiable sparse-voxel tile rasterizer (libsvr.so).
 *
 * The hot path of LiteVoxel's training loop (arXiv 2511.02510; "P:n" = line n of the paper text):
 * "we project, rasterize, measure a photometric objective, and back-propagate", with the
 * per-voxel maximum blending weight w_max gathered during rasterization (eq. 5).
 * The paper states the rasterizer only through eqs. 1-5; everything it is silent on is fixed by
 * the readings R1-R10 and the binning specification B1-B4 in DESIGN.md, which the CPU oracle follows too.
 *
 * Conventions
 *  - Every array pointer is a DEVICE pointer owned by the caller unless the parameter name ends in
 *    `_host`. The library never frees caller memory.
 *  - Every call enqueues its kernels on the context's stream and returns without synchronising, except
 *    svr_preprocess (one 8-byte device->host read of the entry count, which sizes the sort buffers) and
 *    the *_host entry points (they return when the host outputs are valid).
 *  - Calls return an SvrStatus; svr_last_error gives the detail string. On error no output buffer
 *    holds a valid result.
 *  - Workspace (rectangles, keys, sorted lists, per-view colours) comes from a stream-ordered pool owned
 *    by the context; svr_create's `workspace_budget_bytes` (0 = unlimited) bounds it: a request that
 *    would exceed it fails with SVR_ERR_WORKSPACE before anything is launched for that request.
 *  - There is no CPU fallback: with no usable CUDA device svr_create fails with SVR_ERR_CUDA.
 */
#ifndef SVR_H_
#define SVR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct SvrContext SvrContext; /* stream, workspace pool, counters, last error */
typedef struct SvrFrame SvrFrame;     /* one (scene, camera) view: rects, per-view colours, sorted tile lists */

typedef enum {
    SVR_OK = 0,
    SVR_ERR_INVALID_ARG = 1,
    SVR_ERR_CUDA = 2,
    SVR_ERR_WORKSPACE = 3,  /* workspace budget exceeded */
    SVR_ERR_UNSUPPORTED = 4 /* e.g. tile bits + 3 + 3*max_level > 64, K > 4, sh_degree > 3 */
} SvrStatus;

/* Sparse voxel octree leaves. Level-L edge = root_edge / 2^L (R1), lo = root_lo + (ix,iy,iz)*edge.
 * Leaves must be pairwise interior-disjoint. */
typedef struct {
    int64_t n;
    int32_t sh_degree;        /* 0..3 */
    int32_t max_level;        /* Lmax >= every level; Morton codes use 3*Lmax bits */
    float root_lo[3];
    float root_edge;          /* power of two */
    const uint16_t* ijkl;     /* [n,4] ix, iy, iz, level */
    const float* raw_density; /* [n,8] corner c = bx + 2*by + 4*bz; density = exp(trilinear(raw)) (R5) */
    const float* sh;          /* [n,(D+1)^2,3] real SH coefficients, basis index i = l(l+1)+m (R6) */
} SvrVoxels;

/* Pinhole camera, OpenCV axes: p_cam = R p_world + t (R2); ray through pixel centre (x+.5, y+.5) (eq. 1). */
typedef struct {
    int32_t W, H;             /* <= 65535 */
    float fx, fy, cx, cy;
    float R[9];               /* row-major */
    float t[3];
    float z_near;             /* B1 straddle rule; typical 0.01 */
    float bg[3];              /* background colour, composited as T_K * bg (R7) */
} SvrCamera;

typedef struct {
    int32_t K;                /* 1..4 midpoint samples per ray segment (R5) */
    float T_min;              /* a ray stops after the first voxel that leaves T < T_min (R8); 0 = never */
    int32_t record;           /* svr_forward: != 0 records the traversal (per warp and batch: staged list entries, slots
                                 each pixel hit, exp(-tau) per hit) in the frame; a following svr_backward /
                                 svr_backward_heads / svr_backward_normals with the SAME K and T_min replays it and skips its
                                 own cull and test phases (training); with another K or T_min it ignores the record and
                                 walks the lists itself. 0: render only (about 9% faster).
                                 The record's buffers are allocated by the frame's first recording pass (a render-only
                                 frame never holds them); if the workspace budget has no room for them the pass does not
                                 record and svr_backward walks the lists itself (same result, slower).
                                 Ignored by svr_backward: without a record it culls and tests itself. */
    int32_t grad_overwrite;   /* svr_backward / svr_backward_heads: 0 = gradients ACCUMULATE (+=) into grad_raw_density and
                                 grad_sh (several views sum into one buffer; the caller zeroes). != 0: both arrays are
                                 WRITTEN (=) for all n voxels, zeros where this view gives no gradient: a one-view training
                                 step needs no zero fill and the finalize pass reads neither array (C4: 0.35 -> 0.22 ms).
                                 w_max is merged by max in both modes. Ignored by every other call. */
} SvrRenderOpts;

typedef struct {
    float eps;                /* eq. 7, 1e-3 */
    float percentile;         /* q of the percentile-normalised Sobel magnitude (R10), e.g. 0.99 */
    int32_t sobel_source;     /* 0 = target image (default reading), 1 = render */
} SvrLossOpts;

/* Context: device, stream, workspace. Workspace blocks (per-view lists, records, scratch) are cached by the context and
 * reused from view to view; their backing store is
 *   svr_create:                 a PRIVATE stream-ordered memory pool of the context (cudaMemPoolCreate; the device's default
 *                               pool and its release threshold are not touched),
 *   svr_create_with_allocator:  the caller's allocator, e.g. PyTorch's caching allocator ("PyTorch is used only for device
 *                               memory and streams"): alloc_fn(bytes, user) returns device memory usable on `cuda_stream`
 *                               (NULL on failure), free_fn(ptr, user) takes it back; both are called from the thread that
 *                               calls the library, only for blocks the cache does not hold already. Both or neither.
 * `workspace_budget_bytes` (0 = unlimited) bounds the bytes in live + cached blocks. Limits checked by svr_preprocess:
 * root_edge a positive power of two (SVR_ERR_INVALID_ARG otherwise); image up to 65535 pixels a side and
 * (ceil(W/16)+1)(ceil(H/16)+1) <= 51200 tile-grid points, about 14 Mpixel (SVR_ERR_UNSUPPORTED beyond). */
typedef void* (*SvrAllocFn)(size_t bytes, void* user);
typedef void (*SvrFreeFn)(void* ptr, void* user);
SvrStatus svr_create(SvrContext** out, int device, void* cuda_stream, size_t workspace_budget_bytes);
SvrStatus svr_create_with_allocator(SvrContext** out, int device, void* cuda_stream, SvrAllocFn alloc_fn, SvrFreeFn free_fn, void* user,
                                    size_t workspace_budget_bytes);
void svr_destroy(SvrContext* ctx);
const char* svr_last_error(const SvrContext* ctx);
/* High-water mark of the context's workspace pool, bytes (peak VRAM the library itself held). */
size_t svr_workspace_peak_bytes(const SvrContext* ctx);
/* Number of this library's kernels launched on the context so far (bench.py's gpu_launches). */
int64_t svr_kernel_launches(const SvrContext* ctx);

/* (1)+(2) of the path: per-voxel projection to pixel rectangles and (tile, octant) bucket counts (B1), per-view SH
 * colour c_v (R6), key build (tile | direction octant | direction-flipped Morton code, B3), per-bucket device
 * sort, per-(tile,octant) ranges (B4), and a per-voxel view record (geometry relative to the camera,
 * density coefficients, colour) that the compositing kernels gather by voxel id. The frame borrows `vox` pointers: keep them alive and the
 * topology (ijkl) unchanged until svr_frame_release. raw_density / sh VALUES are captured by svr_preprocess;
 * svr_frame_refresh_colors re-captures them (colours + records) after they changed, without redoing the lists. */
SvrStatus svr_preprocess(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cam, SvrFrame** out);
SvrStatus svr_frame_refresh_colors(SvrContext* ctx, SvrFrame* frame);
void svr_frame_release(SvrContext* ctx, SvrFrame* frame);

/* (3) forward compositing, eqs. 2-4: image[H,W,3] = sum_k w_k c_k + T_K bg; depth[H,W] =
 * sum_k w_k t_mid,k (R7); T_final[H,W]; w_max[n] (eq. 5) is MAX-accumulated in place (caller zeroes;
 * never-hit voxels stay 0). depth, T_final, w_max may be NULL. */
SvrStatus svr_forward(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts,
                      float* image, float* depth, float* T_final, float* w_max);

/* (5) LF-weighted photometric loss and its gradient, eqs. 7-10, eq. 18:
 * dL_dimage[H,W,3] = w~(p) sign(R-I) / (3 |P|); *loss (device float) = L_LF. gamma = gamma(t), eq. 9. */
SvrStatus svr_loss_grad(SvrContext* ctx, const float* render, const float* target, int32_t W, int32_t H,
                        float gamma, const SvrLossOpts* opts, float* dL_dimage, float* loss);

/* Optional, before svr_preprocess / svr_forward of the same view: queues the part of eq. 7 that reads only the
 * target (Sobel magnitude and its quantile, R10) on the context's second stream, ordered after the work already
 * queued on the context's stream, so that it runs beside the list build and the forward pass. The next
 * svr_loss_grad with the same target, W, H and percentile (and sobel_source = 0) consumes it; any other
 * svr_loss_grad waits for it and computes everything itself. `target` must stay unchanged in between.
 * No-op when opts->sobel_source != 0. Results are identical with and without this call. */
SvrStatus svr_loss_prepare(SvrContext* ctx, const float* target, int32_t W, int32_t H, const SvrLossOpts* opts);

/* NEXT-3: the structure-aware penalty L_SSIM of eq. 17 and its gradient. The paper names the term
 * only; reading R14: L_SSIM = 1 - mean over pixels and channels of the structural similarity index
 * (Wang et al. 2004) with an 11-tap Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2.
 * render, target, dL_dimage: device [H,W,3] floats. dL_dimage = lambda * dL_SSIM/d render, or += it when
 * accumulate != 0 (so that it adds to svr_loss_grad's output); *loss (device float) = L_SSIM (not scaled by lambda).
 * Errors: null pointers / empty image -> SVR_ERR_INVALID_ARG. */
SvrStatus svr_ssim_loss_grad(SvrContext* ctx, const float* render, const float* target, int32_t W, int32_t H,
                             float lambda, int32_t accumulate, float* dL_dimage, float* loss);

/* svr_ssim_loss_grad for callers that cannot allocate device memory. svr_ssim_loss_grad needs a context (a memory pool and two
 * streams are created with it) and takes 36 bytes of scratch per pixel from that pool. That is not possible everywhere this
 * library is used: inside a host application whose own allocator already holds the GPU's memory, so that an allocation made
 * behind its back may fail or push it over its limit; under a fixed per-process memory reservation that has to be known
 * before the run starts; or in a loop that cannot afford the device-wide stall an allocation or a free can cause. This entry
 * point takes no context and calls no cudaMalloc / cudaFree / pool or other allocating routine, on any call. Its scratch is
 * an array inside the library image, sized for SVR_SSIM_STATIC_MAX_PIXELS pixels (256 + 36 * 2^20 bytes = 36 MiB): every GPU
 * that loads libsvr.so holds it from load until the process exits, whether or not this function is ever called.
 *  - Same result as svr_ssim_loss_grad (the same kernels): dL_dimage[H,W,3] = lambda * dL_SSIM/d render, or += it when
 *    accumulate != 0; *loss (device float) = L_SSIM. render / target / dL_dimage / loss are DEVICE pointers of the caller on
 *    `device`; `cuda_stream` is a cudaStream_t of that device (NULL = the default stream). Asynchronous on that stream.
 *  - W * H > SVR_SSIM_STATIC_MAX_PIXELS (also returned by svr_ssim_static_max_pixels) is refused with SVR_ERR_UNSUPPORTED
 *    before anything is launched; null pointers, an empty image or device outside 0..63 give SVR_ERR_INVALID_ARG; CUDA
 *    failures SVR_ERR_CUDA. svr_static_last_error returns the calling thread's message for the last failed call.
 *  - The FIRST call on each device does a one-time, synchronous set-up (looks up the device address of the scratch array,
 *    uploads the 11 window weights, raises one kernel's shared-memory limit); make that call before any stream capture
 *    begins. Later calls only enqueue a 8-byte memset and two kernels.
 *  - Every call on a device uses the same array, which keeps the previous call's contents; the function clears the one
 *    accumulator that must start at zero. Two calls whose kernels can overlap on the GPU (different streams with no
 *    ordering between them, from one host thread or several) race on the array and both results are garbage: order them. */
#define SVR_SSIM_STATIC_MAX_PIXELS 1048576
SvrStatus svr_ssim_loss_grad_static(int device, void* cuda_stream, const float* render, const float* target, int32_t W,
                                    int32_t H, float lambda, int32_t accumulate, float* dL_dimage, float* loss);
int64_t svr_ssim_static_max_pixels(void);
const char* svr_static_last_error(void);

/* (4) backward compositing: gradients of sum(dL_dimage * image) w.r.t. corner raw densities and SH
 * coefficients. `image` is svr_forward's output for this frame (the suffix colour is image - prefix).
 * grad_raw_density[n,8] and grad_sh[n,(D+1)^2,3] ACCUMULATE (+=; caller zeroes) so several views sum
 * into one buffer, unless opts->grad_overwrite != 0 (then they are written, zeros included); w_max as in svr_forward
 * (may be NULL). */
SvrStatus svr_backward(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts,
                       const float* dL_dimage, const float* image,
                       float* grad_raw_density, float* grad_sh, float* w_max);

/* NEXT-3: the same with gradients arriving through the depth and transmittance heads too (for the depth /
 * transmittance terms of eq. 17): L = sum(dL_dimage * image) + sum(dL_ddepth * depth) + sum(dL_dT * T_final).
 * With D = sum_k w_k t_mid,k and T_K = prod_k exp(-tau_k) (R7; geometry carries no gradient):
 * dD/dtau_k = T_k t_mid,k - sum_{j>k} w_j t_mid,j and dT_K/dtau_k = -T_K. dL_ddepth [H,W] and dL_dT [H,W] may each be NULL;
 * depth / T_final are svr_forward's outputs for this frame (required with the matching gradient). */
SvrStatus svr_backward_heads(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, const float* dL_dimage,
                             const float* dL_ddepth, const float* dL_dT, const float* image, const float* depth,
                             const float* T_final, float* grad_raw_density, float* grad_sh, float* w_max);

/* One whole training-view step with HOST inputs/outputs (bench.py's e2e leg): copies camera + target image
 * host->device, runs preprocess -> forward -> loss_grad -> backward on device-resident voxel parameters and
 * gradient buffers, copies the loss (and, if image_host != NULL, the render) device->host, and returns
 * when they are valid. target_host / image_host: [H,W,3] floats (pinned memory recommended). */
SvrStatus svr_train_view_host(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cam_host,
                              const SvrRenderOpts* ropts, const SvrLossOpts* lopts, float gamma,
                              const float* target_host, float* grad_raw_density, float* grad_sh, float* w_max,
                              float* loss_host, float* image_host);

/* Inspection hooks for the bit-exact binning checks (device pointers valid until svr_frame_release):
 * keys[E] canonical (tile << (3+3Lmax)) | (octant << 3Lmax) | (morton ^ flip), vals[E] voxel ids,
 * ranges[n_tiles,8,2] = [start,end) ((0,0) if empty), rects[n,4] = x0,y0,x1,y1 pixels inclusive
 * (culled: 65535,65535,0,0), tile_masks[n_tiles] octant sets. Any out pointer may be NULL. */
SvrStatus svr_frame_lists(const SvrFrame* frame, const uint64_t** keys, const uint32_t** vals, int64_t* n_entries,
                          const uint32_t** ranges, const uint16_t** rects, const uint8_t** tile_masks);
/* Per-view voxel colours [n,4]: r,g,b and the clamp mask bits (as float bits) - debugging / tests. */
SvrStatus svr_frame_colors(const SvrFrame* frame, const float** rgbm);

/* Measurement hooks (bench.py). svr_forward_stats runs the forward pass with counters compiled in and
 * returns stats_host[4] = ray-voxel hits composited, per-lane slab tests, (warp, voxel) pairs walked after the
 * warp-level rectangle cull, list entries staged. It synchronises. svr_set_stage_timing(1) brackets every
 * stage's kernels with CUDA events on the context's stream; svr_get_stage_times synchronises and returns the
 * accumulated milliseconds and call counts per stage (svr_num_stages() entries, named by svr_stage_name). */
SvrStatus svr_forward_stats(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, float* image,
                            uint64_t* stats_host);
void svr_set_stage_timing(SvrContext* ctx, int enabled);
/* Microbenchmarks of the machine peaks the compositing kernels are set against, run on the context's device and
 * stream, synchronising: out_host[0] = FP32 FMA rate in TFLOP/s (FFMA chains on every SM, FMA = 2 flop), out_host[1] = the
 * same with packed FFMA2 (fma.rn.f32x2), out_host[2] = 1e9 red.global.add.v4.f32 per second into an L2-resident table (the
 * backward pass's gradient reductions), out_host[3] = 1e9 warp instructions issued per second (integer ALU chains). */
SvrStatus svr_measure_peaks(SvrContext* ctx, float* out_host /* [4] */);
int svr_num_stages(void);
/* Experiments / tests only: bit 3 (8) selects the first list-build design (per-voxel scan + global radix sort, the
 * fallback when Morton code + voxel id exceed 64 bits); bit 4 (16): no traversal record (svr_backward walks the lists itself);
 * bit 5 (32): svr_backward ignores the recorded exp(-tau) values and recomputes them; bit 7 (128): the first recording svr_forward of a frame allocates an E
 * record of 64 rows only, so that it overflows and sets the flag that makes the backward pass recompute.
 * Other bits are ignored. */
void svr_set_debug_flags(SvrContext* ctx, int flags);
const char* svr_stage_name(int stage);
SvrStatus svr_get_stage_times(SvrContext* ctx, double* ms, int64_t* calls, int reset);

/* ---- NEXT-3: rendered normals (Fig. 8 shows normal maps; eq. 17 P:212-230 names the depth-normal
 * consistency terms that consume them; the paper gives no formula: DESIGN.md reading R16) ----
 * Per-voxel normal n_v = -g / |g|, g = gradient of the voxel's trilinear raw-density field at the cell centre (0 where g = 0),
 * world space; rendered normal N(p) = sum_k w_k n_{v_k} with the blending weights of eqs. 2-4, zero background, not
 * re-normalised (|N| <= 1 - T_K). svr_render_normals writes normal[H,W,3] (and T_final[H,W] if not NULL) for a frame of
 * svr_preprocess; svr_backward_normals adds d sum(dL_dnormal . N) / d raw to grad_raw_density[n,8] (through the weights and
 * through n_v). Both reuse the compositing kernels with n_v in the colour slot of the view records (restored before they
 * return to the stream), so they cost one forward / backward pass each; svr_backward_normals replays the traversal recorded
 * by svr_forward when there is one. */
SvrStatus svr_render_normals(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, float* normal, float* T_final);
SvrStatus svr_backward_normals(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, const float* dL_dnormal,
                               const float* normal, float* grad_raw_density);

/* ---- NEXT-1: depth-aware quantile pruning, the consumer of w_max (eqs. 11-12) ----
 * One adaptation step over all voxels, statistics gathered over `n_cams` views (reading R11):
 *  1. depth proxy z_v = min over cameras with positive depth of the camera-space depth of the voxel centre
 *     (+inf if none), footprint delta_v = z_v / fx;
 *  2. n_bins depth bins, piecewise-linear in log2 z between the smallest and largest finite depth (integer
 *     arithmetic on the float bit patterns);
 *  3. tau_b = F_b^{-1}(q_b), the nearest-rank q_b-quantile of w_max over the bin (eqs. 11-12),
 *     q_b = q_near + (q_far - q_near) b / (n_bins - 1); inside score x = [w_max > tau_b];
 *  4. guard i: ema = (1 - ema_alpha) ema + ema_alpha x; state = 0 (out) if ema < m_low, 1 (in) if
 *     ema > m_high, else unchanged;
 *  5. guard ii: protected if half-size < kappa * delta_v or w_max >= w_keep;
 *  6. guard iii: at most floor(cap_fraction * n) voxels leave: the unprotected `out` voxels with the
 *     smallest w_max, ties by lower index.
 * w_max[n] in; ema[n] (float) and state[n] (uint8) in/out; keep[n] (uint8, 1 = stays) out. cams_host: HOST array
 * (n_cams <= 64). tau_host[n_bins] (may be NULL) and n_removed_host are HOST outputs: the call synchronises. */
typedef struct {
    int32_t n_bins;           /* 1..64 */
    float q_near, q_far;      /* per-bin quantile at the nearest / farthest bin (annealed by the caller) */
    float ema_alpha, m_low, m_high;
    float kappa, w_keep;
    float cap_fraction;
    int32_t halo;             /* guard ii as a dilation ("keep-halo"): the protected set is the seeds (small footprint or
                                 high w_max) dilated this many times over the face neighbours of the leaves (cells that touch on
                                 one axis and overlap with positive area on the other two, any level difference); 0 = seeds only */
} SvrPruneOpts;
SvrStatus svr_prune_step(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cams_host, int32_t n_cams,
                         const float* w_max, float* ema, uint8_t* state, const SvrPruneOpts* opts, uint8_t* keep,
                         float* tau_host, int64_t* n_removed_host);
/* Stable stream compaction of per-voxel rows: dst[j] = src[i] for the j-th i with keep[i] != 0 (row_bytes a
 * multiple of 4 or 1, 2). Call once per array (ijkl 8 B, raw 32 B, sh 12(D+1)^2 B, ema, state, optimizer moments).
 * src and dst must not overlap. *n_out_host (may be NULL) = number of rows kept (then the call synchronises). */
SvrStatus svr_compact_rows(SvrContext* ctx, const uint8_t* keep, int64_t n, const void* src, void* dst,
                           int64_t row_bytes, int64_t* n_out_host);

/* ---- NEXT-2: priority-driven subdivision (eqs. 13-16; reading R12) ----
 * svr_subdivide_select: depth z_v and footprint delta_v as in svr_prune_step; eligible (eq. 13) iff level <
 * max_level, z_v finite and half-size > kappa * delta_v; z~ = clip((z - z_p5) / (z_p95 - z_p5), 0, 1) (eq. 14) with the
 * 5th / 95th nearest-rank percentile of this step's finite depths (use_current_percentiles != 0) or the running values
 * in the options; priority = usefulness * (1 + beta z~) (eqs. 15-16; usefulness[n] >= 0 is the caller's running score
 * P_v); the max_splits eligible voxels of highest priority are selected, ties by lower index.
 * split[n] (uint8) and priority[n] (may be NULL) are device outputs; z_percentiles_host[2] (may be NULL) and
 * n_split_host are HOST outputs: the call synchronises.
 * svr_subdivide_apply: the new voxel set = the unsplit voxels in their order, then 8 children per split voxel grouped
 * by parent in parent order, child c = bx + 2 by + 4 bz at (2i + bx, 2j + by, 2k + bz, L + 1); child corner raws = the
 * parent's trilinear field at the child's corners (x, then y, then z; a midpoint is 0.5 * (a + b)); SH copied.
 * Output arrays must hold n + 7 * n_split rows; *n_out_host (may be NULL) = that number (then the call synchronises). */
typedef struct {
    float kappa, beta;
    int32_t max_level;              /* voxels at this level or finer never split */
    int64_t max_splits;             /* global growth cap per step */
    int32_t use_current_percentiles;
    float z_p5, z_p95;              /* running percentiles, used when use_current_percentiles == 0 */
} SvrSubdivOpts;
SvrStatus svr_subdivide_select(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cams_host, int32_t n_cams,
                               const float* usefulness, const SvrSubdivOpts* opts, uint8_t* split, float* priority,
                               float* z_percentiles_host, int64_t* n_split_host);
SvrStatus svr_subdivide_apply(SvrContext* ctx, const SvrVoxels* vox, const uint8_t* split, uint16_t* ijkl_out,
                              float* raw_out, float* sh_out, int64_t* n_out_host);

/* Per-voxel side state through a split ("refresh the optimizer/scheduler after topology changes"; reading R17):
 * svr_subdivide_apply writes the new ijkl / raw / sh; every other per-voxel array the trainer keeps (svr_prune_step's ema and
 * state, w_max, the usefulness score, Adam moments) goes through this call with the SAME split mask, once per array, and lands
 * in the same order: dst = the unsplit voxels' rows in their order, then 8 rows per split voxel grouped by parent in parent
 * order, each the parent's row (SVR_ROWS_COPY_PARENT: statistics the children inherit) or zero bytes (SVR_ROWS_ZERO: state that
 * restarts, e.g. the Adam moments of the children's new parameters). src [n] rows, dst [n + 7 * n_split] rows of row_bytes
 * (1, 2 or a multiple of 4) each, device, not overlapping. *n_out_host (may be NULL) = n + 7 * n_split (then the call
 * synchronises). With svr_compact_rows (prune) this lets one adaptation cycle prune -> compact -> subdivide keep its state. */
#define SVR_ROWS_COPY_PARENT 0
#define SVR_ROWS_ZERO 1
SvrStatus svr_subdivide_rows(SvrContext* ctx, const uint8_t* split, int64_t n, const void* src, void* dst, int64_t row_bytes,
                             int32_t mode, int64_t* n_out_host);

/* ---- NEXT-4 (part): fused Adam over a flat float32 parameter array ("Adam state per voxel", ref. [14] P:334) ----
 * m <- b1 m + (1-b1) g; v <- b2 v + (1-b2) g g; theta <- theta - (lr (m / c1)) / (sqrt(v / c2) + eps), c1 = 1 - b1^step,
 * c2 = 1 - b2^step (fp64 on the host, rounded once); float32, each operation rounded in this order. One pass over
 * theta, grad, m, v [n] (device, 16-byte aligned); zero_grad != 0 also clears grad (svr_backward accumulates into it).
 * step >= 1. Asynchronous on the context's stream. */
SvrStatus svr_adam_step(SvrContext* ctx, float* theta, float* grad, float* m, float* v, int64_t n, float lr, float beta1,
                        float beta2, float eps, int32_t step, int32_t zero_grad);

/* NEXT-4 (part): shared grid-point densities. corner_index[n,8] (uint32, corner c = bx + 2 by + 4 bz) names the
 * grid point of every voxel corner; svr_gather_corners fills raw_density[n,8] = grid[corner_index] before svr_preprocess,
 * svr_scatter_add_corners adds grad_raw_density[n,8] into grad_grid[corner_index] (+=, float atomics) after svr_backward.
 * All pointers are device pointers; asynchronous on the context's stream. */
SvrStatus svr_gather_corners(SvrContext* ctx, const float* grid, const uint32_t* corner_index, int64_t n, float* raw_density);
SvrStatus svr_scatter_add_corners(SvrContext* ctx, const float* grad_raw_density, const uint32_t* corner_index, int64_t n,
                                  float* grad_grid);

/* NEXT-4: the total-variation term L_tv of eq. 17 ("total-variation on the sparse density field"). The
 * paper gives no formula; reading R15: L_tv = 1/(12 n) sum_v sum over the 12 edges (a,b) of the cell
 * |raw[v,a] - raw[v,b]| on the raw corner densities. grad_raw_density[n,8] += lambda * dL_tv/draw (sign(0) = 0);
 * *loss (device float) = L_tv (not scaled by lambda). Device pointers, 16-byte aligned; n >= 1. With shared grid points
 * the gradient goes on through svr_scatter_add_corners. */
SvrStatus svr_tv_loss_grad(SvrContext* ctx, const float* raw_density, int64_t n, float lambda, float* grad_raw_density,
                           float* loss);

/* Synchronous device->host copy of `bytes` from a pointer returned by the hooks above (tests). */
SvrStatus svr_copy_to_host(SvrContext* ctx, void* dst_host, const void* src_device, size_t bytes);

/* eq. 9: 0 for t < t0, linear to gamma_max at t1, then gamma_max. Host function. */
float svr_gamma_schedule(float t, float T, float t0_frac, float t1_frac, float gamma_max);

#ifdef __cplusplus
}
#endif
#endif /* SVR_H_ */
