// NEXT-3: rendered normals and the gradient through them (reading R16; Fig. 8 P:312 shows normal maps, eq. 17
// P:212-230 names the depth-normal consistency terms that consume them; the paper gives no formula).
//   n_v = -g / |g|, g = gradient of the voxel's trilinear raw-density field at the cell centre (the four edge differences along
//   each axis; the positive factor 1 / (4 edge) does not change the direction), n_v = 0 where g = 0;
//   N(p) = sum_k w_k n_{v_k}: the normals compose like a colour over a zero background.
// So nothing new is composited: the per-view records get n_v in the place of the colour for the duration of one forward (or
// backward) launch of the compositing kernels of composite.cu, and a small finalize kernel chains dL/dn_v to the corner raws:
//   dL/draw_c = (A^T dL/dcoef)_c  -  sum_a [(I - n n^T) dL/dn]_a sign_ac / |gs|,   gs = unscaled edge-difference sums.
#include "svr_internal.cuh"

namespace {

__device__ __forceinline__ void edge_sums(const float4& ra, const float4& rb, float* gs) {
    // corner c = bx + 2 by + 4 bz: ra = corners 0..3, rb = corners 4..7
    gs[0] = ((ra.y - ra.x) + (ra.w - ra.z)) + ((rb.y - rb.x) + (rb.w - rb.z));
    gs[1] = ((ra.z - ra.x) + (ra.w - ra.y)) + ((rb.z - rb.x) + (rb.w - rb.y));
    gs[2] = ((rb.x - ra.x) + (rb.y - ra.y)) + ((rb.z - ra.z) + (rb.w - ra.w));
}

// enter != 0: save the record's colour in saved[v] and put n_v there; enter == 0: put the saved colour back. Visible voxels only.
__global__ void __launch_bounds__(256) normal_swap_kernel(SceneDev s, const ushort4* __restrict__ rects, float4* __restrict__ packed,
                                                          float4* __restrict__ saved, int enter) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    const ushort4 r = rects[v];
    if (r.x > r.z) return;
    float4* slot = packed + 5 * (size_t)v + 4;           // (r, g, b, dilated half edge)
    float4 cur = *slot;
    if (enter) {
        saved[v] = cur;
        const float4* rp = reinterpret_cast<const float4*>(s.raw) + 2 * (size_t)v;
        float gs[3];
        edge_sums(__ldg(rp), __ldg(rp + 1), gs);
        const float n2 = gs[0] * gs[0] + gs[1] * gs[1] + gs[2] * gs[2];
        const float inv = n2 > 0.f ? -rsqrtf(n2) : 0.f;
        cur.x = gs[0] * inv; cur.y = gs[1] * inv; cur.z = gs[2] * inv;
    } else {
        const float4 c = saved[v];
        cur.x = c.x; cur.y = c.y; cur.z = c.z;
    }
    *slot = cur;
}

// The voxel's scratch row after a backward launch over normal records: [0,8) dL/dcoef (the weights' path), [8,11) dL/dn_v.
__global__ void __launch_bounds__(256) normal_backward_kernel(SceneDev s, const ushort4* __restrict__ rects, float4* __restrict__ grow,
                                                              float4* __restrict__ grad_raw) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    const ushort4 r = rects[v];
    if (r.x > r.z) return;
    const float4 ga = grow[4 * v], gb = grow[4 * v + 1], gn = grow[4 * v + 2];
    const bool any_c = ga.x != 0.f || ga.y != 0.f || ga.z != 0.f || ga.w != 0.f || gb.x != 0.f || gb.y != 0.f || gb.z != 0.f || gb.w != 0.f;
    const bool any_n = gn.x != 0.f || gn.y != 0.f || gn.z != 0.f;
    if (grow[4 * v + 3].x != 0.f) grow[4 * v + 3] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!any_c && !any_n) return;
    grow[4 * v] = make_float4(0.f, 0.f, 0.f, 0.f);
    grow[4 * v + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    grow[4 * v + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
    float out[8];
    {   // coef = A raw  =>  grad_raw += A^T grad_coef (as in voxel_backward_kernel)
        const float g0 = ga.x, gx = ga.y, gy = ga.z, gz = ga.w, gxy = gb.x, gxz = gb.y, gyz = gb.z, gxyz = gb.w;
        out[0] = ((g0 - gx) - (gy + gz)) + ((gxy + gxz) + (gyz - gxyz));
        out[1] = (gx - gxy) - (gxz - gxyz);
        out[2] = (gy - gxy) - (gyz - gxyz);
        out[3] = gxy - gxyz;
        out[4] = (gz - gxz) - (gyz - gxyz);
        out[5] = gxz - gxyz;
        out[6] = gyz - gxyz;
        out[7] = gxyz;
    }
    if (any_n) {
        const float4* rp = reinterpret_cast<const float4*>(s.raw) + 2 * (size_t)v;
        float gs[3];
        edge_sums(__ldg(rp), __ldg(rp + 1), gs);
        const float n2 = gs[0] * gs[0] + gs[1] * gs[1] + gs[2] * gs[2];
        if (n2 > 0.f) {
            const float inv = rsqrtf(n2);
            const float n[3] = {-gs[0] * inv, -gs[1] * inv, -gs[2] * inv};
            const float dn[3] = {gn.x, gn.y, gn.z};
            const float nd = n[0] * dn[0] + n[1] * dn[1] + n[2] * dn[2];
            float t[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) t[a] = -(dn[a] - n[a] * nd) * inv;      // dL/dgs_a
#pragma unroll
            for (int c = 0; c < 8; ++c)
                out[c] += ((c & 1) ? t[0] : -t[0]) + ((c & 2) ? t[1] : -t[1]) + ((c & 4) ? t[2] : -t[2]);
        }
    }
    float4 a = grad_raw[2 * v], b = grad_raw[2 * v + 1];
    a.x += out[0]; a.y += out[1]; a.z += out[2]; a.w += out[3];
    b.x += out[4]; b.y += out[5]; b.z += out[6]; b.w += out[7];
    grad_raw[2 * v] = a;
    grad_raw[2 * v + 1] = b;
}

SvrStatus swap_normals(SvrContext* ctx, const SvrFrame* f, float4* saved, int enter) {
    normal_swap_kernel<<<(unsigned int)((f->scene.n + 255) / 256), 256, 0, ctx->stream>>>(
        f->scene, reinterpret_cast<const ushort4*>(f->rects), reinterpret_cast<float4*>(f->packed), saved, enter);
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

}  // namespace

extern "C" {

SvrStatus svr_render_normals(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, float* normal, float* T_final) {
    SVR_NVTX();
    if (!ctx || !frame || !opts || !normal) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (opts->K < 1 || opts->K > SVR_MAX_K) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    if (frame->packed == nullptr && frame->scene.n > 0) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "frame has no view records");
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    SvrFrame view = *frame;                                   // same buffers, zero background
    view.cam.bg[0] = view.cam.bg[1] = view.cam.bg[2] = 0.f;
    const int64_t n = frame->scene.n;
    float4* saved = nullptr;
    const size_t sb = sizeof(float4) * (size_t)(n > 0 ? n : 1);
    SVR_TRY(svr_alloc(ctx, (void**)&saved, sb));
    SvrStatus st = n > 0 ? swap_normals(ctx, frame, saved, 1) : SVR_OK;
    if (st == SVR_OK) {
        st = launch_forward(ctx, &view, opts->K, opts->T_min, normal, nullptr, T_final, nullptr, nullptr, false);
        const SvrStatus st2 = n > 0 ? swap_normals(ctx, frame, saved, 0) : SVR_OK;      // always put the colours back
        if (st == SVR_OK) st = st2;
    }
    svr_free(ctx, saved, sb);
    return st;
}

SvrStatus svr_backward_normals(SvrContext* ctx, const SvrFrame* frame, const SvrRenderOpts* opts, const float* dL_dnormal,
                               const float* normal, float* grad_raw_density) {
    SVR_NVTX();
    if (!ctx || !frame || !opts || !dL_dnormal || !normal || !grad_raw_density) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (opts->K < 1 || opts->K > SVR_MAX_K) return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    const int64_t n = frame->scene.n;
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    SVR_TRY(svr_ensure_grad_rows(ctx, n));
    SvrFrame view = *frame;
    view.cam.bg[0] = view.cam.bg[1] = view.cam.bg[2] = 0.f;
    float4* saved = nullptr;
    const size_t sb = sizeof(float4) * (size_t)n;
    SVR_TRY(svr_alloc(ctx, (void**)&saved, sb));
    SvrStatus st = swap_normals(ctx, frame, saved, 1);
    if (st == SVR_OK) {
        st = launch_backward(ctx, &view, opts->K, opts->T_min, dL_dnormal, normal, ctx->grad_row, false, nullptr, nullptr, nullptr, nullptr);
        const SvrStatus st2 = swap_normals(ctx, frame, saved, 0);
        if (st == SVR_OK) st = st2;
    }
    svr_free(ctx, saved, sb);
    if (st != SVR_OK) return st;
    normal_backward_kernel<<<(unsigned int)((n + 255) / 256), 256, 0, ctx->stream>>>(
        frame->scene, reinterpret_cast<const ushort4*>(frame->rects), reinterpret_cast<float4*>(ctx->grad_row),
        reinterpret_cast<float4*>(grad_raw_density));
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

}  // extern "C"
