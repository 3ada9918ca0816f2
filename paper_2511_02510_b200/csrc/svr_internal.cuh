// Internal declarations shared by the .cu files of libsvr.so (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <unordered_map>
#include <utility>
#include <vector>
#include <nvtx3/nvToolsExt.h>      // header-only NVTX v3: a no-op function-pointer test unless a profiler has injected itself
#include "svr.h"

// One NVTX range per C-ABI call: ncu --nvtx / a timeline tool shows which call a kernel belongs to.
struct SvrNvtxRange {
    explicit SvrNvtxRange(const char* name) { nvtxRangePushA(name); }
    ~SvrNvtxRange() { nvtxRangePop(); }
    SvrNvtxRange(const SvrNvtxRange&) = delete;
    SvrNvtxRange& operator=(const SvrNvtxRange&) = delete;
};
#define SVR_NVTX() SvrNvtxRange nvtx_range__(__func__)

#define SVR_TILE 16
#define SVR_MAX_K 4
#define SVR_SCAN_SMEM_MAX (200 * 1024)   // dynamic shared memory the one-block bucket scan may use for its tile-grid table
#define SVR_TRAV_WORDS 72     // traversal record: [0..31] hit masks, [32..63] voxel ids, [64] slot count, [65] first E row of the batch, [71] its E row count; [66..70] unused (the record is a multiple of 16 bytes)

enum SvrStage {
    ST_TILE_MASKS = 0, ST_RECTS, ST_SCAN, ST_EMIT, ST_SORT, ST_RANGES, ST_COLORS, ST_FORWARD, ST_LOSS, ST_BACKWARD,
    ST_SH_BACKWARD, ST_PACK, ST_COUNT
};

struct StagePending { int stage; cudaEvent_t e0, e1; };

struct SvrContext {
    bool timing = false;
    int debug_flags = 0;          // measurement experiments only (svr_set_debug_flags)
    std::vector<StagePending> pending;
    std::vector<cudaEvent_t> event_pool;
    double stage_ms[ST_COUNT] = {0};
    int64_t stage_calls[ST_COUNT] = {0};
    int device = 0;
    cudaStream_t stream = nullptr;
    // backing store of the workspace blocks: the caller's allocator (svr_create_with_allocator) or a PRIVATE stream-ordered
    // memory pool of this context (never the device's default pool, which the host application may share)
    SvrAllocFn alloc_fn = nullptr;
    SvrFreeFn free_fn = nullptr;
    void* alloc_user = nullptr;
    cudaMemPool_t pool = nullptr;
    size_t budget = 0;            // 0 = unlimited
    size_t in_use = 0, cached = 0, peak = 0;   // bytes in live blocks, in cached free blocks, and the peak of their sum
    std::vector<std::pair<void*, size_t>> free_blocks;   // cached free workspace blocks (pointer, capacity)
    std::unordered_map<void*, size_t> live;             // live workspace blocks -> capacity
    int64_t launches = 0;
    std::string err;
    // persistent scratch
    // [n_cap,16] per-voxel gradient scratch, one 64-byte row per voxel (one DRAM access): [0,8) density-coefficient gradient,
    // [8,11) colour gradient, [12] max blending weight (float bits); kept all-zero between calls by the finalize kernel
    float* grad_row = nullptr;
    int64_t grad_cap = 0;
    void* loss_ws = nullptr;      // loss workspace (see loss.cu)
    size_t loss_ws_bytes = 0;
    // second stream: work that does not depend on the render (the loss's source phase, the host path's upload)
    cudaStream_t aux = nullptr;
    cudaEvent_t fork_ev = nullptr, loss_ready_ev = nullptr, upload_ev = nullptr, lists_ev = nullptr, sort_ev = nullptr, ectl_ev = nullptr;
    bool loss_prepared = false;   // svr_loss_prepare queued a source phase that the next svr_loss_grad may consume
    const float* loss_prep_target = nullptr;
    int loss_prep_W = 0, loss_prep_H = 0;
    float loss_prep_q = 0.f;
    uint64_t* host_pinned = nullptr;  // 64-byte pinned readback slot (words 4..5: the last forward's E-record cursor / flag)
    double e_units_per_entry = 0.0;   // E-record units (32 floats) used per list entry by the last recorded view: sizes the next one
    int64_t e_last_entries = 0;       // list entries of the frame whose cursor is in flight to host_pinned[4]
    cudaEvent_t readback_ev = nullptr; // marks the readback copy: the host waits for it, not for the work queued behind it
};

// Device-side copy of the camera with everything derived on the host in fp64.
struct CamDev {
    int W, H, tiles_x, tiles_y;
    float fx, fy, cx, cy;
    float R[9], t[3];
    float z_near;
    float bg[3];
    double o[3];                  // camera centre -R^T t (fp64)
};

struct SceneDev {
    int64_t n;
    int sh_degree, n_basis, max_level;
    float root_lo[3];
    float root_edge;
    const uint16_t* ijkl;
    const float* raw;
    const float* sh;
};

// The 80-byte view record of voxel `vid` (5 x 16 B at vrec + 5 vid): centre relative to the camera as hi+lo floats (fp64
// arithmetic), half edge, voxel id, the trilinear raw density as polynomial coefficients * log2(e) (corner c = bx + 2 by +
// 4 bz), the per-view colour. Written by the projection kernel (preprocess.cu) and by voxel_record_kernel (composite.cu).
__device__ __forceinline__ void voxel_record_dev(const SceneDev& s, const CamDev& c, uint2 q, uint32_t vid, float4 col, float4* __restrict__ vrec) {
    const float4* rp = reinterpret_cast<const float4*>(s.raw) + 2 * (size_t)vid;
    const float4 ra = __ldg(rp), rb = __ldg(rp + 1);
    const int L = q.y >> 16;
    const float ef = s.root_edge * __int_as_float((127 - L) << 23);
    const double e = (double)ef;
    const double gx = (double)s.root_lo[0] + ((double)(q.x & 0xFFFF) + 0.5) * e - c.o[0];
    const double gy = (double)s.root_lo[1] + ((double)(q.x >> 16) + 0.5) * e - c.o[1];
    const double gz = (double)s.root_lo[2] + ((double)(q.y & 0xFFFF) + 0.5) * e - c.o[2];
    const float hx = (float)gx, hy = (float)gy, hz = (float)gz;
    const float L2E = 1.4426950408889634f;
    const float c0 = ra.x, cx = ra.y - ra.x, cy = ra.z - ra.x, cz = rb.x - ra.x;
    const float cxy = (ra.w - ra.y) - cy, cxz = (rb.y - ra.y) - cz, cyz = (rb.z - ra.z) - cz;
    const float cxyz = ((rb.w - rb.z) - (rb.y - rb.x)) - ((ra.w - ra.z) - (ra.y - ra.x));
    float4* out = vrec + 5 * (size_t)vid;
    out[0] = make_float4(hx, hy, hz, 0.5f * ef);
    out[1] = make_float4((float)(gx - (double)hx), (float)(gy - (double)hy), (float)(gz - (double)hz), __uint_as_float(vid));
    out[2] = make_float4(c0 * L2E, cx * L2E, cy * L2E, cz * L2E);
    out[3] = make_float4(cxy * L2E, cxz * L2E, cyz * L2E, cxyz * L2E);
    // .w: the half edge dilated by a bound on what the lo parts and the rounding can move (the forward's conservative slab test);
    // the clamp mask of the colour stays in rgbm
    out[4] = make_float4(col.x, col.y, col.z, fmaf(fabsf(hx) + fabsf(hy) + fabsf(hz), 4.8e-7f, (0.5f * ef) * 1.000002f));
}

struct SvrFrame {
    SceneDev scene;
    CamDev cam;
    int n_tiles = 0;
    int tile_bits = 0, key_bits = 0;
    int64_t n_entries = 0;
    // device buffers (pool-allocated)
    uint16_t* rects = nullptr;       // [n,4]
    uint16_t* rects_tight = nullptr; // [n,4] pixels whose centre can see the voxel (visible voxels only; bucketed list build)
    uint8_t* tile_masks = nullptr;   // [n_tiles]
    uint32_t* sat = nullptr;         // [(tiles_y+1)*(tiles_x+1)] summed-area table of popcount(mask)
    uint32_t* offsets = nullptr;     // [n+1] exclusive scan of counts
    float* rgbm = nullptr;           // [n,4]
    uint64_t* keys = nullptr;        // [E] sorted
    uint32_t* vals = nullptr;        // [E] sorted
    uint16_t* rects_sorted = nullptr;// [E,4] pixel rectangle of vals[i] (coalesced reads in the compositing cull)
    uint32_t* ranges = nullptr;      // [n_tiles*8*2]
    float* packed = nullptr;         // [n,20] per-voxel view record, visible voxels only (composite.cu voxel_record_kernel)
    uint32_t* tile_order = nullptr;  // [2*n_tiles]: tile ids by descending list length, then the lengths
    // traversal scratch written by svr_forward, replayed by svr_backward (composite.cu)
    // (trav and trav_E are allocated by the first RECORDING forward pass: a render-only frame never holds them)
    mutable uint32_t* trav = nullptr;        // [trav_cap, SVR_TRAV_WORDS] records
    uint32_t* trav_off = nullptr;    // [n_tiles + 1] first record of each tile
    uint32_t* trav_count = nullptr;  // [n_tiles * 8] records written per warp
    mutable float* trav_E = nullptr;         // [trav_E_cap * 32] exp(-tau) of every queued hit, handed out to warps in chunks
    uint32_t* trav_ectl = nullptr;   // [2] chunk cursor (units of 32 floats), overflow flag
    mutable uint32_t trav_E_cap = 0;         // capacity of trav_E in units of 32 floats
    mutable bool trav_valid = false; // a forward pass has recorded this frame's traversal ...
    mutable float trav_T_min = 0.f;  // ... with this termination threshold
    mutable int trav_K = 0;          // ... and this sample count (the recorded E = exp(-tau) and the termination point depend on it)
    size_t bytes = 0;
};

// ---- error handling -------------------------------------------------------------------------
SvrStatus svr_fail(SvrContext* ctx, SvrStatus st, const char* fmt, ...);
#define SVR_CUDA(ctx, call)                                                                      \
    do {                                                                                         \
        cudaError_t e__ = (call);                                                                \
        if (e__ != cudaSuccess)                                                                  \
            return svr_fail((ctx), SVR_ERR_CUDA, "%s failed: %s (%s:%d)", #call,                 \
                            cudaGetErrorString(e__), __FILE__, __LINE__);                        \
    } while (0)
#define SVR_TRY(call)                          \
    do {                                       \
        SvrStatus s__ = (call);                \
        if (s__ != SVR_OK) return s__;         \
    } while (0)

// Brackets the kernels of one stage with CUDA events on the context's stream when timing is enabled.
struct StageScope {
    SvrContext* ctx; int stage; cudaEvent_t e0 = nullptr, e1 = nullptr;
    static cudaEvent_t get(SvrContext* c) {
        if (!c->event_pool.empty()) { cudaEvent_t e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
        cudaEvent_t e; cudaEventCreate(&e); return e;
    }
    StageScope(SvrContext* c, int st) : ctx(c), stage(st) {
        if (ctx->timing) { e0 = get(ctx); e1 = get(ctx); cudaEventRecord(e0, ctx->stream); }
    }
    ~StageScope() {
        if (e0) { cudaEventRecord(e1, ctx->stream); ctx->pending.push_back({stage, e0, e1}); }
    }
};

// ---- workspace pool --------------------------------------------------------------------------
SvrStatus svr_alloc(SvrContext* ctx, void** p, size_t bytes);
void svr_free(SvrContext* ctx, void* p, size_t bytes);
SvrStatus svr_ensure_grad_rows(SvrContext* ctx, int64_t n);

// ---- stage launchers (each counts its kernel launches into ctx->launches) --------------------
SvrStatus launch_tile_masks(SvrContext* ctx, SvrFrame* f, bool with_sat);
SvrStatus launch_rects_counts(SvrContext* ctx, SvrFrame* f, uint32_t* counts, unsigned long long* totals);
SvrStatus launch_exclusive_scan(SvrContext* ctx, const uint32_t* in, uint32_t* out, int64_t n_plus_1);
SvrStatus launch_emit_keys(SvrContext* ctx, SvrFrame* f, uint64_t* keys, uint32_t* vals, uint32_t* big_list,
                           unsigned int* big_count);
SvrStatus launch_sort_pairs(SvrContext* ctx, uint64_t* keys, uint64_t* keys_alt, uint32_t* vals, uint32_t* vals_alt,
                            int64_t n, int bits, uint64_t** keys_sorted, uint32_t** vals_sorted);
SvrStatus launch_ranges(SvrContext* ctx, SvrFrame* f);
SvrStatus launch_bucket_count(SvrContext* ctx, SvrFrame* f, uint32_t* bcount, int* bigdiff, uint32_t* nonempty,
                              unsigned long long* totals);
SvrStatus launch_bucket_scatter(SvrContext* ctx, SvrFrame* f, uint32_t* cursor, uint64_t* ent, int vb, uint32_t* big_list,
                                unsigned int* big_count);
SvrStatus launch_bucket_sort(SvrContext* ctx, SvrFrame* f, uint64_t* ent, const uint32_t* nonempty, const unsigned long long* totals,
                             unsigned int* work, int vb);
SvrStatus launch_lists_finish(SvrContext* ctx, SvrFrame* f, bool fork);
SvrStatus launch_lists_join(SvrContext* ctx);
SvrStatus launch_voxel_colors(SvrContext* ctx, SvrFrame* f);
SvrStatus launch_voxel_records(SvrContext* ctx, SvrFrame* f);
SvrStatus launch_gather_rects(SvrContext* ctx, SvrFrame* f);
SvrStatus launch_forward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, float* image, float* depth,
                         float* T_final, float* w_max, unsigned long long* stats, bool record);
SvrStatus launch_backward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, const float* dL, const float* image,
                          float* grad_row, bool want_wmax, const float* dL_ddepth, const float* dL_dT,
                          const float* depth, const float* T_final);
SvrStatus launch_sh_backward(SvrContext* ctx, const SvrFrame* f, float* grad_row, float* grad_raw, float* grad_sh, float* w_max,
                             bool overwrite);
SvrStatus launch_loss_prepare(SvrContext* ctx, const float* target, int W, int H, float q);
SvrStatus launch_loss_grad(SvrContext* ctx, const float* render, const float* target, int W, int H, float gamma,
                           float eps, float q, int sobel_source, float* dL, float* loss);

// ---- small device helpers ---------------------------------------------------------------------
#ifdef __CUDACC__
// Real SH basis up to degree 3, no Condon-Shortley phase, i = l(l+1)+m (R6).
__device__ __forceinline__ void sh_basis_dev(int degree, float x, float y, float z, float* Y) {
    Y[0] = 0.28209479177387814f;
    if (degree < 1) return;
    Y[1] = 0.4886025119029199f * y;
    Y[2] = 0.4886025119029199f * z;
    Y[3] = 0.4886025119029199f * x;
    if (degree < 2) return;
    float xx = x * x, yy = y * y, zz = z * z;
    Y[4] = 1.0925484305920792f * x * y;
    Y[5] = 1.0925484305920792f * y * z;
    Y[6] = 0.31539156525252005f * (3.0f * zz - 1.0f);
    Y[7] = 1.0925484305920792f * x * z;
    Y[8] = 0.5462742152960396f * (xx - yy);
    if (degree < 3) return;
    Y[9] = 0.5900435899266435f * y * (3.0f * xx - yy);
    Y[10] = 2.890611442640554f * x * y * z;
    Y[11] = 0.4570457994644658f * y * (5.0f * zz - 1.0f);
    Y[12] = 0.3731763325901154f * z * (5.0f * zz - 3.0f);
    Y[13] = 0.4570457994644658f * x * (5.0f * zz - 1.0f);
    Y[14] = 1.445305721320277f * z * (xx - yy);
    Y[15] = 0.5900435899266435f * x * (xx - 3.0f * yy);
}

__device__ __forceinline__ void voxel_dir_dev(const SceneDev& s, const CamDev& c, uint2 q, float& dx, float& dy, float& dz) {
    int L = q.y >> 16;
    double e = (double)s.root_edge * (double)__int_as_float((127 - L) << 23);
    double gx = (double)s.root_lo[0] + ((double)(q.x & 0xFFFF) + 0.5) * e - c.o[0];
    double gy = (double)s.root_lo[1] + ((double)(q.x >> 16) + 0.5) * e - c.o[1];
    double gz = (double)s.root_lo[2] + ((double)(q.y & 0xFFFF) + 0.5) * e - c.o[2];
    float fx = (float)gx, fy = (float)gy, fz = (float)gz;
    float n2 = fx * fx + fy * fy + fz * fz;
    if (n2 == 0.0f) { dx = 0.f; dy = 0.f; dz = 1.f; return; }
    float inv = rsqrtf(n2);
    dx = fx * inv; dy = fy * inv; dz = fz * inv;
}
#endif

#ifdef __CUDACC__
// Direction-sign octant of a pixel's ray (B2): individually rounded binary32 operations in this
// exact order, so the compositing kernels select the same (tile, octant) list the binning built.
__device__ __forceinline__ int pixel_octant_dev(const CamDev& c, int x, int y) {
    float u = __fdiv_rn(__fsub_rn(__fadd_rn((float)x, 0.5f), c.cx), c.fx);
    float v = __fdiv_rn(__fsub_rn(__fadd_rn((float)y, 0.5f), c.cy), c.fy);
    int s = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float d = __fadd_rn(__fadd_rn(__fmul_rn(c.R[a], u), __fmul_rn(c.R[3 + a], v)), c.R[6 + a]);
        if (d < 0.0f) s |= 1 << a;
    }
    return s;
}
#endif
