// C-ABI entry points of libsvr.so (include/svr.h): context, workspace pool, and the orchestration of
// svr_preprocess / svr_forward / svr_loss_grad / svr_backward. No torch types, no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "svr_internal.cuh"

SvrStatus svr_fail(SvrContext* ctx, SvrStatus st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    return st;
}

// Workspace blocks are cached by the context: a freed block goes to a free list and the next request that fits it
// (capacity within 2x of the need) takes it back without touching the driver. Large blocks are allocated with 12.5%
// slack, so the per-view buffers, whose sizes follow the entry count E, are reused from view to view even though E
// changes; the first time a size is seen costs a cudaMallocAsync (milliseconds when the pool has to grow). Everything
// is ordered on the context's one stream, so reuse needs no extra synchronisation.
static cudaError_t backing_alloc(SvrContext* ctx, void** p, size_t cap) {
    if (ctx->alloc_fn) {
        *p = ctx->alloc_fn(cap, ctx->alloc_user);
        return *p ? cudaSuccess : cudaErrorMemoryAllocation;
    }
    return cudaMallocFromPoolAsync(p, cap, ctx->pool, ctx->stream);
}
static void backing_free(SvrContext* ctx, void* p) {
    if (ctx->free_fn) ctx->free_fn(p, ctx->alloc_user);      // stream-ordered reuse is the caller's allocator's business: it was
    else cudaFreeAsync(p, ctx->stream);                      // told the stream (svr_create_with_allocator's contract)
}

// the per-voxel gradient scratch rows of the backward passes (all-zero between calls)
SvrStatus svr_ensure_grad_rows(SvrContext* ctx, int64_t n) {
    if (ctx->grad_cap >= n) return SVR_OK;
    if (ctx->grad_row) svr_free(ctx, ctx->grad_row, 0);
    ctx->grad_row = nullptr;
    ctx->grad_cap = 0;
    SVR_TRY(svr_alloc(ctx, (void**)&ctx->grad_row, sizeof(float) * 16 * (size_t)n));
    ctx->grad_cap = n;
    SVR_CUDA(ctx, cudaMemsetAsync(ctx->grad_row, 0, sizeof(float) * 16 * (size_t)n, ctx->stream));
    return SVR_OK;
}

SvrStatus svr_alloc(SvrContext* ctx, void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 256;
    const size_t need = (bytes + 255) & ~(size_t)255;
    int best = -1;
    for (int i = 0; i < (int)ctx->free_blocks.size(); ++i) {
        const size_t cap = ctx->free_blocks[i].second;
        if (cap >= need && cap <= 2 * need + ((size_t)1 << 20) && (best < 0 || cap < ctx->free_blocks[best].second)) best = i;
    }
    size_t cap = best >= 0 ? ctx->free_blocks[best].second : (need > ((size_t)1 << 20) ? ((need + need / 8 + 255) & ~(size_t)255) : need);
    if (ctx->budget && ctx->in_use + cap > ctx->budget) {
        if (best < 0 && ctx->in_use + need <= ctx->budget) cap = need;     // no slack when the budget is tight
        else if (ctx->in_use + cap > ctx->budget)
            return svr_fail(ctx, SVR_ERR_WORKSPACE, "workspace budget exceeded: in use %zu + request %zu > budget %zu", ctx->in_use,
                            need, ctx->budget);
    }
    if (best >= 0) {
        *p = ctx->free_blocks[best].first;
        ctx->cached -= cap;
        ctx->free_blocks.erase(ctx->free_blocks.begin() + best);
    } else {
        // make room under the budget by dropping cached blocks first
        while (ctx->budget && ctx->in_use + ctx->cached + cap > ctx->budget && !ctx->free_blocks.empty()) {
            backing_free(ctx, ctx->free_blocks.back().first);
            ctx->cached -= ctx->free_blocks.back().second;
            ctx->free_blocks.pop_back();
        }
        SVR_CUDA(ctx, backing_alloc(ctx, p, cap));
    }
    ctx->live[*p] = cap;
    ctx->in_use += cap;
    if (ctx->in_use + ctx->cached > ctx->peak) ctx->peak = ctx->in_use + ctx->cached;
    return SVR_OK;
}

void svr_free(SvrContext* ctx, void* p, size_t /*bytes*/) {
    if (!p) return;
    auto it = ctx->live.find(p);
    if (it == ctx->live.end()) return;
    const size_t cap = it->second;
    ctx->live.erase(it);
    ctx->in_use -= cap;
    if (ctx->free_blocks.size() >= 48) {         // bounded list: drop the oldest cached block
        backing_free(ctx, ctx->free_blocks.front().first);
        ctx->cached -= ctx->free_blocks.front().second;
        ctx->free_blocks.erase(ctx->free_blocks.begin());
    }
    ctx->free_blocks.emplace_back(p, cap);
    ctx->cached += cap;
}

namespace {

struct FrameAlloc {
    SvrContext* ctx;
    SvrFrame* f;
    SvrStatus get(void** p, size_t bytes) {
        return svr_alloc(ctx, p, bytes);
    }
};

int bits_for(int64_t n) {
    int b = 0;
    while (((int64_t)1 << b) < n) ++b;
    return b;
}

void fill_cam(const SvrCamera* cam, CamDev* c) {
    c->W = cam->W; c->H = cam->H;
    c->tiles_x = (cam->W + SVR_TILE - 1) / SVR_TILE;
    c->tiles_y = (cam->H + SVR_TILE - 1) / SVR_TILE;
    c->fx = cam->fx; c->fy = cam->fy; c->cx = cam->cx; c->cy = cam->cy;
    for (int i = 0; i < 9; ++i) c->R[i] = cam->R[i];
    for (int i = 0; i < 3; ++i) { c->t[i] = cam->t[i]; c->bg[i] = cam->bg[i]; }
    c->z_near = cam->z_near;
    for (int a = 0; a < 3; ++a)   // o = -R^T t in fp64 (R3)
        c->o[a] = -((double)cam->R[a] * cam->t[0] + (double)cam->R[3 + a] * cam->t[1] + (double)cam->R[6 + a] * cam->t[2]);
}

SvrStatus release_frame_buffers(SvrContext* ctx, SvrFrame* f) {
    void* ptrs[] = {f->rects, f->rects_tight, f->tile_masks, f->sat, f->offsets, f->rgbm, f->keys, f->vals, f->ranges, f->rects_sorted, f->tile_order, f->packed,
                    f->trav, f->trav_off, f->trav_count, f->trav_E, f->trav_ectl};
    for (void* p : ptrs)
        if (p) svr_free(ctx, p, 0);
    return SVR_OK;
}

// Traversal scratch (svr_forward records, svr_backward replays): at most E/4 + 80 n_tiles records of SVR_TRAV_WORDS words
// (sum over tiles of 8 warps x (ceil(len / 32) + 9)), plus the E record: exp(-tau) of every queued ray-voxel hit, in units of
// 32 floats handed out by a device-side cursor. Its size follows the recorded views so far (largest number of units per list
// entry, read back asynchronously after each recording forward pass) with 25 % slack; when it is too small, or the budget has
// no room for it, the forward pass sets a flag and the backward pass recomputes E (same result, slower). Debug flag 16 disables
// the traversal record (backward then culls and tests itself).
// The small parts are allocated at preprocess time (the list build fills trav_off):
SvrStatus alloc_traversal(SvrContext* ctx, SvrFrame* f, int64_t /*E*/) {
    if (ctx->debug_flags & 16) return SVR_OK;
    SVR_TRY(svr_alloc(ctx, (void**)&f->trav_off, sizeof(uint32_t) * (size_t)(f->n_tiles + 1)));
    SVR_TRY(svr_alloc(ctx, (void**)&f->trav_count, sizeof(uint32_t) * 8 * (size_t)f->n_tiles));
    SVR_TRY(svr_alloc(ctx, (void**)&f->trav_ectl, 256));
    return SVR_OK;
}

// the records and the E rows, by the first recording forward pass of the frame. Returns false (no record: the backward pass then
// walks the lists itself) when the budget has no room for the records.
bool alloc_traversal_record(SvrContext* ctx, const SvrFrame* f) {
    if (f->trav) return true;
    if ((ctx->debug_flags & 16) || !f->trav_off || f->n_entries <= 0) return false;
    const int64_t E = f->n_entries;
    const size_t cap = (size_t)E / 4 + 80 * (size_t)f->n_tiles + 8;
    if (svr_alloc(ctx, (void**)&f->trav, sizeof(uint32_t) * SVR_TRAV_WORDS * cap) != SVR_OK) {
        f->trav = nullptr;
        ctx->err.clear();
        (void)cudaGetLastError();       // a real out-of-memory leaves the runtime's last error set: the launch check after the
                                        // forward kernel would report it although rendering without a record is fine
        return false;
    }
    if (ctx->e_last_entries > 0 && cudaEventQuery(ctx->ectl_ev) == cudaSuccess) {
        const uint32_t used = reinterpret_cast<const uint32_t*>(ctx->host_pinned + 4)[0];
        // the largest ratio seen, not the last one: the sizes of a camera's buffers then repeat from epoch to epoch and the
        // workspace cache serves them (sizes that follow the previous VIEW made multi-GB blocks miss the cache on C5: 100 ms)
        const double r = (double)used / (double)ctx->e_last_entries;
        if (r > ctx->e_units_per_entry) ctx->e_units_per_entry = r;
        ctx->e_last_entries = 0;
    }
    const double per_entry = ctx->e_units_per_entry > 0.0 ? 1.25 * ctx->e_units_per_entry : 0.5;
    double units = per_entry * (double)E + 64.0 * (double)f->n_tiles + 1024.0;
    if (units > 1.3e8) units = 1.3e8;      // word offsets into the record are 32-bit (rows * 32 < 2^32)
    if (ctx->debug_flags & 128) units = 64.0;       // test hook: an E record that is far too small (exercises the overflow flag)
    f->trav_E_cap = (uint32_t)units;
    if (svr_alloc(ctx, (void**)&f->trav_E, sizeof(float) * 32 * ((size_t)f->trav_E_cap + 64)) != SVR_OK) {   // + 64 rows: read-ahead
        f->trav_E = nullptr;            // no room under the budget: the backward pass recomputes E
        f->trav_E_cap = 0;
        ctx->err.clear();
        (void)cudaGetLastError();       // as above
    }
    return true;
}

}  // namespace

extern "C" {

SvrStatus svr_create(SvrContext** out, int device, void* cuda_stream, size_t workspace_budget_bytes) {
    SVR_NVTX();
    return svr_create_with_allocator(out, device, cuda_stream, nullptr, nullptr, nullptr, workspace_budget_bytes);
}

SvrStatus svr_create_with_allocator(SvrContext** out, int device, void* cuda_stream, SvrAllocFn alloc_fn, SvrFreeFn free_fn, void* user,
                                    size_t workspace_budget_bytes) {
    SVR_NVTX();
    if (!out || ((alloc_fn == nullptr) != (free_fn == nullptr))) return SVR_ERR_INVALID_ARG;
    *out = nullptr;
    SvrContext* ctx = new (std::nothrow) SvrContext();
    if (!ctx) return SVR_ERR_CUDA;
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->budget = workspace_budget_bytes;
    ctx->alloc_fn = alloc_fn;
    ctx->free_fn = free_fn;
    ctx->alloc_user = user;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess && !alloc_fn) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = device;
        e = cudaMemPoolCreate(&ctx->pool, &props);
        if (e == cudaSuccess) {
            uint64_t thr = UINT64_MAX;   // keep freed workspace in THIS pool between frames (the device's default pool is untouched)
            e = cudaMemPoolSetAttribute(ctx->pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
    }
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&ctx->host_pinned), 64);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->readback_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->aux, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->fork_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->loss_ready_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->upload_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->lists_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->sort_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ectl_ev, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        // no usable CUDA device: fail loudly, there is no other path
        fprintf(stderr, "svr_create: CUDA error: %s\n", cudaGetErrorString(e));
        delete ctx;
        return SVR_ERR_CUDA;
    }
    *out = ctx;
    return SVR_OK;
}

void svr_destroy(SvrContext* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    if (ctx->aux) cudaStreamSynchronize(ctx->aux);
    cudaStreamSynchronize(ctx->stream);
    for (auto& b : ctx->free_blocks) backing_free(ctx, b.first);
    for (auto& b : ctx->live) backing_free(ctx, b.first);
    if (ctx->host_pinned) cudaFreeHost(ctx->host_pinned);
    if (ctx->readback_ev) cudaEventDestroy(ctx->readback_ev);
    if (ctx->fork_ev) cudaEventDestroy(ctx->fork_ev);
    if (ctx->loss_ready_ev) cudaEventDestroy(ctx->loss_ready_ev);
    if (ctx->upload_ev) cudaEventDestroy(ctx->upload_ev);
    if (ctx->lists_ev) cudaEventDestroy(ctx->lists_ev);
    if (ctx->sort_ev) cudaEventDestroy(ctx->sort_ev);
    if (ctx->ectl_ev) cudaEventDestroy(ctx->ectl_ev);
    if (ctx->aux) cudaStreamDestroy(ctx->aux);
    cudaStreamSynchronize(ctx->stream);
    for (const StagePending& p : ctx->pending) { cudaEventDestroy(p.e0); cudaEventDestroy(p.e1); }
    for (cudaEvent_t e : ctx->event_pool) cudaEventDestroy(e);
    if (ctx->pool) { cudaStreamSynchronize(ctx->stream); cudaMemPoolDestroy(ctx->pool); }
    delete ctx;
}

const char* svr_last_error(const SvrContext* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
size_t svr_workspace_peak_bytes(const SvrContext* ctx) { return ctx ? ctx->peak : 0; }
int64_t svr_kernel_launches(const SvrContext* ctx) { return ctx ? ctx->launches : 0; }

SvrStatus svr_preprocess(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cam, SvrFrame** out) {
    SVR_NVTX();
    if (!ctx || !vox || !cam || !out) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    if (vox->n < 0 || vox->n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    if (vox->sh_degree < 0 || vox->sh_degree > 3) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "sh_degree must be 0..3");
    if (cam->W <= 0 || cam->H <= 0 || cam->W > 65535 || cam->H > 65535)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "image size must be 1..65535");
    if (vox->max_level < 1 || vox->max_level > 16) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "max_level must be 1..16");
    if (vox->n > 0 && (!vox->ijkl || !vox->raw_density || !vox->sh)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null voxel arrays");
    {
        int ex = 0;      // R1: cell bounds must be exact in fp32, and the kernels form 1/edge by exponent arithmetic
        if (!(vox->root_edge > 0.f) || std::frexp(vox->root_edge, &ex) != 0.5f)
            return svr_fail(ctx, SVR_ERR_INVALID_ARG, "root_edge must be a positive power of two (got %g)", (double)vox->root_edge);
    }
    {
        // the bucket scan keeps a (tiles_x + 1) x (tiles_y + 1) int table in one block's shared memory
        const size_t pts = (size_t)((cam->W + SVR_TILE - 1) / SVR_TILE + 1) * (size_t)((cam->H + SVR_TILE - 1) / SVR_TILE + 1);
        if (pts * sizeof(int) > SVR_SCAN_SMEM_MAX)
            return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "image of %d x %d pixels has %zu tile-grid points (limit %zu: about 14 Mpixel)", cam->W,
                            cam->H, pts, (size_t)SVR_SCAN_SMEM_MAX / sizeof(int));
    }
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));

    SvrFrame* f = new (std::nothrow) SvrFrame();
    if (!f) return svr_fail(ctx, SVR_ERR_CUDA, "out of host memory");
    f->scene.n = vox->n;
    f->scene.sh_degree = vox->sh_degree;
    f->scene.n_basis = (vox->sh_degree + 1) * (vox->sh_degree + 1);
    f->scene.max_level = vox->max_level;
    for (int a = 0; a < 3; ++a) f->scene.root_lo[a] = vox->root_lo[a];
    f->scene.root_edge = vox->root_edge;
    f->scene.ijkl = vox->ijkl;
    f->scene.raw = vox->raw_density;
    f->scene.sh = vox->sh;
    fill_cam(cam, &f->cam);
    f->n_tiles = f->cam.tiles_x * f->cam.tiles_y;
    f->tile_bits = bits_for(f->n_tiles);
    f->key_bits = f->tile_bits + 3 + 3 * vox->max_level;
    if (f->key_bits > 64) {
        const int kb = f->key_bits;
        delete f;
        return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "key needs %d bits (> 64): reduce max_level or image size", kb);
    }

    FrameAlloc A{ctx, f};
    const int64_t n = vox->n;
    const int vb = bits_for(n > 1 ? n : 2);
    // second design of the list build (preprocess.cu "Bucketed list build") whenever code and voxel id fit one word
    const bool bucketed = (3 * vox->max_level + vb <= 64) && (ctx->debug_flags & 8) == 0;
    const size_t n_buckets = (size_t)f->n_tiles * 8;
    uint32_t* counts = nullptr;
    unsigned long long* totals = nullptr;
    uint32_t* big_list = nullptr;
    uint64_t *keys_a = nullptr, *keys_b = nullptr;
    uint32_t *vals_a = nullptr, *vals_b = nullptr;
    uint32_t *bcount = nullptr, *nonempty = nullptr;
    int* bigdiff = nullptr;
    const size_t counts_bytes = sizeof(uint32_t) * (size_t)(n + 1), bucket_bytes = sizeof(uint32_t) * n_buckets;
    const size_t diff_bytes = sizeof(int) * (size_t)(f->cam.tiles_x + 1) * (f->cam.tiles_y + 1);
    size_t big_bytes = 0, ka = 0, va = 0;
    SvrStatus st = SVR_OK;
    auto fail = [&](SvrStatus s) {
        cudaStreamSynchronize(ctx->aux);     // forked list kernels may still read the frame's buffers
        if (counts) svr_free(ctx, counts, counts_bytes);
        if (totals) svr_free(ctx, totals, 128);
        if (big_list) svr_free(ctx, big_list, big_bytes);
        if (keys_a) svr_free(ctx, keys_a, ka);
        if (keys_b) svr_free(ctx, keys_b, ka);
        if (vals_a) svr_free(ctx, vals_a, va);
        if (vals_b) svr_free(ctx, vals_b, va);
        if (bcount) svr_free(ctx, bcount, bucket_bytes);
        if (nonempty) svr_free(ctx, nonempty, bucket_bytes);
        if (bigdiff) svr_free(ctx, bigdiff, diff_bytes);
        f->keys = nullptr; f->vals = nullptr;
        release_frame_buffers(ctx, f);
        delete f;
        return s;
    };
#define TRYF(call) do { st = (call); if (st != SVR_OK) return fail(st); } while (0)
#define CUDAF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail(svr_fail(ctx, SVR_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e__))); } while (0)

    TRYF(A.get((void**)&f->rects, sizeof(uint16_t) * 4 * (size_t)n));
    if (bucketed) TRYF(A.get((void**)&f->rects_tight, sizeof(uint16_t) * 4 * (size_t)n));
    TRYF(A.get((void**)&f->tile_masks, (size_t)f->n_tiles));
    if (!bucketed) TRYF(A.get((void**)&f->sat, sizeof(uint32_t) * (size_t)(f->cam.tiles_x + 1) * (f->cam.tiles_y + 1)));
    TRYF(A.get((void**)&f->rgbm, sizeof(float) * 4 * (size_t)n));
    TRYF(A.get((void**)&f->packed, sizeof(float) * 20 * (size_t)n));
    TRYF(A.get((void**)&f->ranges, sizeof(uint32_t) * 16 * (size_t)f->n_tiles));
    TRYF(A.get((void**)&f->tile_order, sizeof(uint32_t) * 2 * (size_t)f->n_tiles));
    TRYF(svr_alloc(ctx, (void**)&totals, 128));
    CUDAF(cudaMemsetAsync(totals, 0, 128, ctx->stream));
    TRYF(launch_tile_masks(ctx, f, !bucketed));

    if (bucketed) {
        TRYF(svr_alloc(ctx, (void**)&bcount, bucket_bytes));
        TRYF(svr_alloc(ctx, (void**)&nonempty, bucket_bytes));
        TRYF(svr_alloc(ctx, (void**)&bigdiff, diff_bytes));
        CUDAF(cudaMemsetAsync(bcount, 0, bucket_bytes, ctx->stream));
        CUDAF(cudaMemsetAsync(bigdiff, 0, diff_bytes, ctx->stream));
        TRYF(launch_bucket_count(ctx, f, bcount, bigdiff, nonempty, totals));
        // E, the number of many-tile voxels and the number of non-empty buckets: one small readback sizes the lists
        CUDAF(cudaMemcpyAsync(ctx->host_pinned, totals, 32, cudaMemcpyDeviceToHost, ctx->stream));
        CUDAF(cudaStreamSynchronize(ctx->stream));
        const int64_t E = (int64_t)ctx->host_pinned[0];
        const int64_t n_big = (int64_t)ctx->host_pinned[1];
        if (E >= ((int64_t)1 << 31)) return fail(svr_fail(ctx, SVR_ERR_UNSUPPORTED, "%lld list entries (>= 2^31)", (long long)E));
        f->n_entries = E;
        bool forked = false;
        if (E > 0) {
            ka = sizeof(uint64_t) * (size_t)E;
            va = sizeof(uint32_t) * (size_t)E;
            big_bytes = sizeof(uint32_t) * (size_t)(n_big + 1);
            // frame-lifetime buffers first, largest first (the pool then reuses the previous frame's blocks one for one),
            // scratch last
            TRYF(alloc_traversal(ctx, f, E));
            TRYF(svr_alloc(ctx, (void**)&keys_b, ka));   // canonical keys
            TRYF(A.get((void**)&f->rects_sorted, sizeof(uint16_t) * 4 * (size_t)E));
            TRYF(svr_alloc(ctx, (void**)&vals_a, va));
            TRYF(svr_alloc(ctx, (void**)&keys_a, ka));   // packed (code << vb | id) words, scratch
            TRYF(svr_alloc(ctx, (void**)&big_list, big_bytes));
            f->keys = keys_b; f->vals = vals_a;
            TRYF(launch_lists_finish(ctx, f, true));
            forked = true;
            TRYF(launch_bucket_scatter(ctx, f, bcount, keys_a, vb, big_list, reinterpret_cast<unsigned int*>(totals + 2)));
            TRYF(launch_bucket_sort(ctx, f, keys_a, nonempty, totals, reinterpret_cast<unsigned int*>(totals + 8), vb));   // totals[8..9]: the three work-fetch counters
            svr_free(ctx, keys_a, ka);
            svr_free(ctx, big_list, big_bytes);
            keys_a = nullptr; big_list = nullptr;
            keys_b = nullptr; vals_a = nullptr;
        }
        svr_free(ctx, bcount, bucket_bytes);
        svr_free(ctx, nonempty, bucket_bytes);
        svr_free(ctx, bigdiff, diff_bytes);
        bcount = nonempty = nullptr; bigdiff = nullptr;
        svr_free(ctx, totals, 128);
        totals = nullptr;
        if (forked) TRYF(launch_lists_join(ctx));
        else TRYF(launch_lists_finish(ctx, f, false));
        TRYF(launch_gather_rects(ctx, f));
    } else {
        TRYF(A.get((void**)&f->offsets, sizeof(uint32_t) * (size_t)(n + 1)));
        TRYF(svr_alloc(ctx, (void**)&counts, counts_bytes));
        TRYF(launch_rects_counts(ctx, f, counts, totals));
        TRYF(launch_exclusive_scan(ctx, counts, f->offsets, n + 1));
        // E = offsets[n]; number of big voxels = totals[1]: one small readback sizes the sort buffers
        CUDAF(cudaMemcpyAsync(totals, f->offsets + n, sizeof(uint32_t), cudaMemcpyDeviceToDevice, ctx->stream));
        CUDAF(cudaMemcpyAsync(ctx->host_pinned, totals, 16, cudaMemcpyDeviceToHost, ctx->stream));
        // per-view colours do not depend on E: enqueue before the sync so they overlap the readback
        CUDAF(cudaEventRecord(ctx->readback_ev, ctx->stream));
        TRYF(launch_voxel_colors(ctx, f));
        TRYF(launch_voxel_records(ctx, f));
        CUDAF(cudaEventSynchronize(ctx->readback_ev));
        const int64_t E = (int64_t)(ctx->host_pinned[0] & 0xFFFFFFFFull);
        const int64_t n_big = (int64_t)ctx->host_pinned[1];
        svr_free(ctx, counts, counts_bytes);
        counts = nullptr;
        if (E >= ((int64_t)1 << 31)) return fail(svr_fail(ctx, SVR_ERR_UNSUPPORTED, "%lld list entries (>= 2^31)", (long long)E));
        f->n_entries = E;

        if (E > 0) {
            ka = sizeof(uint64_t) * (size_t)E;
            va = sizeof(uint32_t) * (size_t)E;
            big_bytes = sizeof(uint32_t) * (size_t)(n_big + 1);
            TRYF(svr_alloc(ctx, (void**)&keys_a, ka));
            TRYF(svr_alloc(ctx, (void**)&keys_b, ka));
            TRYF(svr_alloc(ctx, (void**)&vals_a, va));
            TRYF(svr_alloc(ctx, (void**)&vals_b, va));
            TRYF(svr_alloc(ctx, (void**)&big_list, big_bytes));
            unsigned int* big_count = reinterpret_cast<unsigned int*>(totals + 2);
            TRYF(launch_emit_keys(ctx, f, keys_a, vals_a, big_list, big_count));
            uint64_t* ks = nullptr;
            uint32_t* vs = nullptr;
            TRYF(launch_sort_pairs(ctx, keys_a, keys_b, vals_a, vals_b, E, f->key_bits, &ks, &vs));
            // keep the buffers holding the sorted result, return the others to the pool
            svr_free(ctx, ks == keys_a ? keys_b : keys_a, ka);
            svr_free(ctx, vs == vals_a ? vals_b : vals_a, va);
            svr_free(ctx, big_list, big_bytes);
            big_list = nullptr;
            f->keys = ks; f->vals = vs;
            TRYF(alloc_traversal(ctx, f, E));
            TRYF(A.get((void**)&f->rects_sorted, sizeof(uint16_t) * 4 * (size_t)E));
            keys_a = keys_b = nullptr;
            vals_a = vals_b = nullptr;
        }
        svr_free(ctx, totals, 128);
        totals = nullptr;
        TRYF(launch_ranges(ctx, f));
        TRYF(launch_gather_rects(ctx, f));
    }
#undef TRYF
#undef CUDAF
    *out = f;
    return SVR_OK;
}

SvrStatus svr_frame_refresh_colors(SvrContext* ctx, SvrFrame* frame) {
    SVR_NVTX();
    if (!ctx || !frame) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    frame->trav_valid = false;      // termination depends on the densities: the next forward pass records again
    SVR_TRY(launch_voxel_colors(ctx, frame));
    return launch_voxel_records(ctx, frame);
}

void svr_frame_release(SvrContext* ctx, SvrFrame* frame) {
    if (!ctx || !frame) return;
    release_frame_buffers(ctx, frame);
    delete frame;
}

SvrStatus svr_forward(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, float* image, float* depth,
                      float* T_final, float* w_max) {
    SVR_NVTX();
    if (!ctx || !frame || !opts || !image) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (opts->K < 1 || opts->K > SVR_MAX_K) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    const bool record = opts->record != 0 && alloc_traversal_record(ctx, frame);
    SvrStatus st = launch_forward(ctx, frame, opts->K, opts->T_min, image, depth, T_final, w_max, nullptr, record);
    if (st == SVR_OK && record) {
        frame->trav_valid = true;
        frame->trav_T_min = opts->T_min;
        frame->trav_K = opts->K;
        if (frame->trav_ectl && frame->n_entries > 0) {
            // how much of the E record this view used: sizes the next frame's (alloc_traversal); never waited for
            SVR_CUDA(ctx, cudaMemcpyAsync(ctx->host_pinned + 4, frame->trav_ectl, 8, cudaMemcpyDeviceToHost, ctx->stream));
            SVR_CUDA(ctx, cudaEventRecord(ctx->ectl_ev, ctx->stream));
            ctx->e_last_entries = frame->n_entries;
        }
    }
    return st;
}

SvrStatus svr_loss_prepare(SvrContext* ctx, const float* target, int32_t W, int32_t H, const SvrLossOpts* opts) {
    SVR_NVTX();
    if (!ctx || !target || !opts) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (W <= 0 || H <= 0) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "empty image");
    if (!(opts->percentile > 0.f && opts->percentile <= 1.f)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "percentile must be in (0,1]");
    if (opts->sobel_source != 0) return SVR_OK;      // the weights read the render: nothing to do ahead of it
    return launch_loss_prepare(ctx, target, W, H, opts->percentile);
}

SvrStatus svr_loss_grad(SvrContext* ctx, const float* render, const float* target, int32_t W, int32_t H, float gamma,
                        const SvrLossOpts* opts, float* dL_dimage, float* loss) {
    SVR_NVTX();
    if (!ctx || !render || !target || !opts || !dL_dimage || !loss) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (W <= 0 || H <= 0) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "empty image");
    if (!(opts->percentile > 0.f && opts->percentile <= 1.f)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "percentile must be in (0,1]");
    return launch_loss_grad(ctx, render, target, W, H, gamma, opts->eps, opts->percentile, opts->sobel_source, dL_dimage, loss);
}

SvrStatus svr_backward_heads(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, const float* dL_dimage,
                             const float* dL_ddepth, const float* dL_dT, const float* image, const float* depth, const float* T_final,
                             float* grad_raw_density, float* grad_sh, float* w_max) {
    SVR_NVTX();
    if (!ctx || !frame || !opts || !dL_dimage || !image || !grad_raw_density || !grad_sh)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if ((dL_ddepth && !depth) || (dL_dT && !T_final))
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "dL_ddepth needs depth and dL_dT needs T_final (svr_forward's outputs)");
    if (opts->K < 1 || opts->K > SVR_MAX_K) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    const int64_t n = frame->scene.n;
    if (n == 0) return SVR_OK;
    SVR_TRY(svr_ensure_grad_rows(ctx, n));
    SVR_TRY(launch_backward(ctx, frame, opts->K, opts->T_min, dL_dimage, image, ctx->grad_row, w_max != nullptr, dL_ddepth, dL_dT,
                            depth, T_final));
    return launch_sh_backward(ctx, frame, ctx->grad_row, grad_raw_density, grad_sh, w_max, opts->grad_overwrite != 0);
}

SvrStatus svr_backward(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, const float* dL_dimage,
                       const float* image, float* grad_raw_density, float* grad_sh, float* w_max) {
    SVR_NVTX();
    return svr_backward_heads(ctx, frame, opts, dL_dimage, nullptr, nullptr, image, nullptr, nullptr, grad_raw_density, grad_sh, w_max);
}

SvrStatus svr_train_view_host(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cam_host, const SvrRenderOpts* ropts,
                              const SvrLossOpts* lopts, float gamma, const float* target_host, float* grad_raw_density,
                              float* grad_sh, float* w_max, float* loss_host, float* image_host) {
    SVR_NVTX();
    if (!ctx || !vox || !cam_host || !ropts || !lopts || !target_host || !loss_host)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    const size_t npix = (size_t)cam_host->W * cam_host->H;
    float* buf = nullptr;   // target | image | dL | loss
    const size_t bytes = sizeof(float) * (npix * 9 + 64);
    SVR_TRY(svr_alloc(ctx, (void**)&buf, bytes));
    float *target = buf, *image = buf + npix * 3, *dL = buf + npix * 6, *loss = buf + npix * 9;
    SvrFrame* f = nullptr;
    SvrStatus st = SVR_OK;
    // the upload and the part of the loss that reads only the target run on the second stream, beside preprocess + forward
    cudaError_t e = cudaEventRecord(ctx->fork_ev, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->aux, ctx->fork_ev, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(target, target_host, sizeof(float) * npix * 3, cudaMemcpyHostToDevice, ctx->aux);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->upload_ev, ctx->aux);
    if (e != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "H2D copy: %s", cudaGetErrorString(e));
    if (st == SVR_OK) st = svr_loss_prepare(ctx, target, cam_host->W, cam_host->H, lopts);
    if (st == SVR_OK) st = svr_preprocess(ctx, vox, cam_host, &f);
    if (st == SVR_OK) st = svr_forward(ctx, f, ropts, image, nullptr, nullptr, nullptr);
    if (st == SVR_OK && cudaStreamWaitEvent(ctx->stream, ctx->upload_ev, 0) != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "stream wait");
    if (st == SVR_OK) st = svr_loss_grad(ctx, image, target, cam_host->W, cam_host->H, gamma, lopts, dL, loss);
    if (st == SVR_OK) st = svr_backward(ctx, f, ropts, dL, image, grad_raw_density, grad_sh, w_max);
    if (st == SVR_OK) {
        e = cudaMemcpyAsync(loss_host, loss, sizeof(float), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess && image_host)
            e = cudaMemcpyAsync(image_host, image, sizeof(float) * npix * 3, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "D2H copy: %s", cudaGetErrorString(e));
    }
    if (f) svr_frame_release(ctx, f);
    if (st != SVR_OK) {                   // the upload and the loss's target phase may still be using buf on the second stream
        cudaStreamSynchronize(ctx->aux);
        ctx->loss_prepared = false;
    }
    svr_free(ctx, buf, bytes);
    return st;
}

SvrStatus svr_frame_lists(const SvrFrame* frame, const uint64_t** keys, const uint32_t** vals, int64_t* n_entries,
                          const uint32_t** ranges, const uint16_t** rects, const uint8_t** tile_masks) {
    SVR_NVTX();
    if (!frame) return SVR_ERR_INVALID_ARG;
    if (keys) *keys = frame->keys;
    if (vals) *vals = frame->vals;
    if (n_entries) *n_entries = frame->n_entries;
    if (ranges) *ranges = frame->ranges;
    if (rects) *rects = frame->rects;
    if (tile_masks) *tile_masks = frame->tile_masks;
    return SVR_OK;
}

SvrStatus svr_frame_colors(const SvrFrame* frame, const float** rgbm) {
    SVR_NVTX();
    if (!frame || !rgbm) return SVR_ERR_INVALID_ARG;
    *rgbm = frame->rgbm;
    return SVR_OK;
}

SvrStatus svr_forward_stats(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, float* image,
                            uint64_t* stats_host) {
    SVR_NVTX();
    if (!ctx || !frame || !opts || !image || !stats_host) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (opts->K < 1 || opts->K > SVR_MAX_K) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    unsigned long long* d = nullptr;
    SVR_TRY(svr_alloc(ctx, (void**)&d, 64));
    cudaMemsetAsync(d, 0, 64, ctx->stream);
    SvrStatus st = launch_forward(ctx, frame, opts->K, opts->T_min, image, nullptr, nullptr, nullptr, d, false);
    if (st == SVR_OK) {
        cudaError_t e = cudaMemcpyAsync(stats_host, d, 32, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "stats readback: %s", cudaGetErrorString(e));
    }
    svr_free(ctx, d, 64);
    return st;
}

void svr_set_stage_timing(SvrContext* ctx, int enabled) {
    if (ctx) ctx->timing = enabled != 0;
}

int svr_num_stages(void) { return ST_COUNT; }

void svr_set_debug_flags(SvrContext* ctx, int flags) {
    if (ctx) ctx->debug_flags = flags;
}

const char* svr_stage_name(int stage) {
    static const char* names[ST_COUNT] = {"tile_masks", "rects_counts", "scan", "emit_keys", "sort", "ranges", "voxel_colors",
                                          "forward_composite", "loss_grad", "backward_composite", "sh_backward", "pack_entries"};
    return (stage >= 0 && stage < ST_COUNT) ? names[stage] : "";
}

SvrStatus svr_get_stage_times(SvrContext* ctx, double* ms, int64_t* calls, int reset) {
    SVR_NVTX();
    if (!ctx) return SVR_ERR_INVALID_ARG;
    SVR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (const StagePending& p : ctx->pending) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, p.e0, p.e1) == cudaSuccess) {
            ctx->stage_ms[p.stage] += (double)t;
            ctx->stage_calls[p.stage] += 1;
        }
        ctx->event_pool.push_back(p.e0);
        ctx->event_pool.push_back(p.e1);
    }
    ctx->pending.clear();
    for (int i = 0; i < ST_COUNT; ++i) {
        if (ms) ms[i] = ctx->stage_ms[i];
        if (calls) calls[i] = ctx->stage_calls[i];
        if (reset) { ctx->stage_ms[i] = 0.0; ctx->stage_calls[i] = 0; }
    }
    return SVR_OK;
}

SvrStatus svr_copy_to_host(SvrContext* ctx, void* dst_host, const void* src_device, size_t bytes) {
    SVR_NVTX();
    if (!ctx || !dst_host || !src_device) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    SVR_CUDA(ctx, cudaMemcpyAsync(dst_host, src_device, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    SVR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SVR_OK;
}

float svr_gamma_schedule(float t, float T, float t0_frac, float t1_frac, float gamma_max) {
    float t0 = t0_frac * T, t1 = t1_frac * T;
    if (t < t0) return 0.0f;
    if (t < t1) return gamma_max * (t - t0) / (t1 - t0);
    return gamma_max;
}

}  // extern "C"
