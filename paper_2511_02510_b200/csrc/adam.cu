// Fused Adam update over a flat float32 parameter array (NEXT-4: "fused Adam over voxel parameters";
// PAPER.md P:62 "Adam state per voxel", ref. [14] P:334). One pass: reads theta, g, m, v, writes theta, m, v and
// (optionally) zeroes g, because svr_backward ACCUMULATES into the gradient buffers: 28 or 32 bytes per parameter, HBM-bound.
// Every operation is individually rounded in the order oracle/adam.py states, so the result is bit-identical to it.
#include <cmath>

#include "svr_internal.cuh"

namespace {

__device__ __forceinline__ void adam_one(float& th, float g, float& m, float& v, float lr, float b1, float b2, float one_b1,
                                         float one_b2, float c1, float c2, float eps) {
    m = __fadd_rn(__fmul_rn(b1, m), __fmul_rn(one_b1, g));
    v = __fadd_rn(__fmul_rn(b2, v), __fmul_rn(one_b2, __fmul_rn(g, g)));
    const float mh = __fdiv_rn(m, c1), vh = __fdiv_rn(v, c2);
    th = __fsub_rn(th, __fdiv_rn(__fmul_rn(lr, mh), __fadd_rn(__fsqrt_rn(vh), eps)));
}

__global__ void __launch_bounds__(256) adam_kernel(float* __restrict__ theta, float* __restrict__ grad, float* __restrict__ m,
                                                   float* __restrict__ v, int64_t n, float lr, float b1, float b2, float one_b1,
                                                   float one_b2, float c1, float c2, float eps, int zero_grad) {
    const int64_t i4 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i4 + 3 < n) {
        float4 t = *reinterpret_cast<float4*>(theta + i4), g = *reinterpret_cast<float4*>(grad + i4);
        float4 mm = *reinterpret_cast<float4*>(m + i4), vv = *reinterpret_cast<float4*>(v + i4);
        adam_one(t.x, g.x, mm.x, vv.x, lr, b1, b2, one_b1, one_b2, c1, c2, eps);
        adam_one(t.y, g.y, mm.y, vv.y, lr, b1, b2, one_b1, one_b2, c1, c2, eps);
        adam_one(t.z, g.z, mm.z, vv.z, lr, b1, b2, one_b1, one_b2, c1, c2, eps);
        adam_one(t.w, g.w, mm.w, vv.w, lr, b1, b2, one_b1, one_b2, c1, c2, eps);
        *reinterpret_cast<float4*>(theta + i4) = t;
        *reinterpret_cast<float4*>(m + i4) = mm;
        *reinterpret_cast<float4*>(v + i4) = vv;
        if (zero_grad) *reinterpret_cast<float4*>(grad + i4) = make_float4(0.f, 0.f, 0.f, 0.f);
    } else {
        for (int64_t i = i4; i < n; ++i) {
            float t = theta[i], mm = m[i], vv = v[i];
            adam_one(t, grad[i], mm, vv, lr, b1, b2, one_b1, one_b2, c1, c2, eps);
            theta[i] = t; m[i] = mm; v[i] = vv;
            if (zero_grad) grad[i] = 0.f;
        }
    }
}

}  // namespace

extern "C" SvrStatus svr_adam_step(SvrContext* ctx, float* theta, float* grad, float* m, float* v, int64_t n, float lr, float beta1,
                                   float beta2, float eps, int32_t step, int32_t zero_grad) {
    SVR_NVTX();
    if (!ctx || !theta || !grad || !m || !v) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 0 || step < 1) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "n must be >= 0 and step >= 1");
    if (((uintptr_t)theta | (uintptr_t)grad | (uintptr_t)m | (uintptr_t)v) & 15)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "arrays must be 16-byte aligned");
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    const float c1 = (float)(1.0 - std::pow((double)beta1, (double)step)), c2 = (float)(1.0 - std::pow((double)beta2, (double)step));
    const float one_b1 = 1.0f - beta1, one_b2 = 1.0f - beta2;
    const int64_t n4 = (n + 3) / 4;
    adam_kernel<<<(unsigned int)((n4 + 255) / 256), 256, 0, ctx->stream>>>(theta, grad, m, v, n, lr, beta1, beta2, one_b1, one_b2, c1, c2,
                                                                          eps, zero_grad);
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// ---- shared grid-point densities (NEXT-4): voxels that share a corner share its raw density ----
// gather: raw[v, c] = grid[idx[v, c]]; scatter: grad_grid[idx[v, c]] += grad_raw[v, c] (float atomics: order-dependent sums).
namespace {

__global__ void __launch_bounds__(256) gather_corners_kernel(const float* __restrict__ grid, const uint32_t* __restrict__ idx, int64_t n8,
                                                             float* __restrict__ raw) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n8) raw[i] = __ldg(grid + idx[i]);
}

__global__ void __launch_bounds__(256) scatter_corners_kernel(const float* __restrict__ grad_raw, const uint32_t* __restrict__ idx, int64_t n8,
                                                              float* __restrict__ grad_grid) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n8) return;
    const float g = grad_raw[i];
    if (g != 0.0f) atomicAdd(grad_grid + idx[i], g);
}

}  // namespace

extern "C" SvrStatus svr_gather_corners(SvrContext* ctx, const float* grid, const uint32_t* corner_index, int64_t n, float* raw_density) {
    SVR_NVTX();
    if (!ctx || !grid || !corner_index || !raw_density) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 0 || n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    gather_corners_kernel<<<(unsigned int)((8 * n + 255) / 256), 256, 0, ctx->stream>>>(grid, corner_index, 8 * n, raw_density);
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

extern "C" SvrStatus svr_scatter_add_corners(SvrContext* ctx, const float* grad_raw_density, const uint32_t* corner_index, int64_t n,
                                             float* grad_grid) {
    SVR_NVTX();
    if (!ctx || !grad_raw_density || !corner_index || !grad_grid) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 0 || n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    scatter_corners_kernel<<<(unsigned int)((8 * n + 255) / 256), 256, 0, ctx->stream>>>(grad_raw_density, corner_index, 8 * n, grad_grid);
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// ---- L_tv (NEXT-4; eq. 17; R15) ----
// L_tv = 1/(12 N) sum_v sum over the 12 cell edges |raw_a - raw_b|; grad_raw += lambda dL/draw. One thread per voxel, 64 B
// read + 64 B read-modify-write; the loss is summed in fp64 (one atomic per block) and written by a second, one-thread kernel.
namespace {

__device__ __forceinline__ float sgnf(float x) { return (float)((x > 0.f) - (x < 0.f)); }

__global__ void __launch_bounds__(256) tv_kernel(const float4* __restrict__ raw, int64_t n, float scale, float4* __restrict__ grad_raw,
                                                 double* __restrict__ acc) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    float local = 0.f;
    if (v < n) {
        const float4 a = raw[2 * v], b = raw[2 * v + 1];
        const float r[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
        float g[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int ax = 0; ax < 3; ++ax)
#pragma unroll
            for (int c = 0; c < 8; ++c)
                if (!((c >> ax) & 1)) {
                    const float d = r[c] - r[c | (1 << ax)];
                    local += fabsf(d);
                    const float sg = sgnf(d);
                    g[c] += sg;
                    g[c | (1 << ax)] -= sg;
                }
        float4 ga = grad_raw[2 * v], gb = grad_raw[2 * v + 1];
        ga.x = fmaf(scale, g[0], ga.x); ga.y = fmaf(scale, g[1], ga.y); ga.z = fmaf(scale, g[2], ga.z); ga.w = fmaf(scale, g[3], ga.w);
        gb.x = fmaf(scale, g[4], gb.x); gb.y = fmaf(scale, g[5], gb.y); gb.z = fmaf(scale, g[6], gb.z); gb.w = fmaf(scale, g[7], gb.w);
        grad_raw[2 * v] = ga;
        grad_raw[2 * v + 1] = gb;
    }
    __shared__ double wsum[8];
    double s = (double)local;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += wsum[w];
        if (t != 0.0) atomicAdd(acc, t);
    }
}

__global__ void tv_finish_kernel(const double* __restrict__ acc, int64_t n, float* __restrict__ loss) {
    *loss = (float)(*acc / (12.0 * (double)n));
}

}  // namespace

extern "C" SvrStatus svr_tv_loss_grad(SvrContext* ctx, const float* raw_density, int64_t n, float lambda, float* grad_raw_density,
                                      float* loss) {
    SVR_NVTX();
    if (!ctx || !raw_density || !grad_raw_density || !loss) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 1 || n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    if (((uintptr_t)raw_density | (uintptr_t)grad_raw_density) & 15) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "arrays must be 16-byte aligned");
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    double* acc = nullptr;
    SVR_TRY(svr_alloc(ctx, (void**)&acc, 64));
    SvrStatus st = SVR_OK;
    cudaError_t e = cudaMemsetAsync(acc, 0, sizeof(double), ctx->stream);
    if (e == cudaSuccess) {
        const float scale = (float)((double)lambda / (12.0 * (double)n));
        tv_kernel<<<(unsigned int)((n + 255) / 256), 256, 0, ctx->stream>>>(reinterpret_cast<const float4*>(raw_density), n, scale,
                                                                           reinterpret_cast<float4*>(grad_raw_density), acc);
        tv_finish_kernel<<<1, 1, 0, ctx->stream>>>(acc, n, loss);
        ctx->launches += 2;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "tv: %s", cudaGetErrorString(e));
    svr_free(ctx, acc, 64);
    return st;
}
