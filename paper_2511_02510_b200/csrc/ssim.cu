// L_SSIM and its gradient (NEXT-3, SURVEY 8f "fused SSIM loss gradient"; eq. 17; R14:
// the index of Wang et al. 2004 with the 11-tap sigma-1.5 Gaussian window, zero padding, C1 = 0.01^2, C2 = 0.03^2).
//
//   L = 1 - mean_{p,ch} S,  S = (2 mu1 mu2 + C1)(2 s12 + C2) / ((mu1^2 + mu2^2 + C1)(s11 + s22 + C2))
//   dL/dR = -(1/(3|P|)) [ g * dS/dm1 + 2 R (g * dS/dq11) + I (g * dS/dq12) ]      (the window is symmetric: adjoint = itself)
//
// Two kernels over 16 x 16 pixel tiles with a 5-pixel halo, all three channels of a tile in one block (rows of the
// interleaved [H,W,3] image are read contiguously), separable window (11 + 11 taps instead of 121):
//   ssim_stats_kernel  the five windowed moments, the index (summed for the loss) and the three derivative maps;
//   ssim_grad_kernel   windows the derivative maps and writes / accumulates lambda * dL/dR.
// The moments are accumulated in fp64: s11 = E[R^2] - mu1^2 cancels against C2 = 9e-4, and fp32 sums would leave a
// relative error of 1e-4 in flat regions. Everything else is fp32. HBM-bound, per pixel: the first kernel reads 24 B (R, I)
// and writes 36 B (three maps), the second reads 36 + 24 B and writes 12 B (+ 12 B read when accumulating): 132 B.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "svr_internal.cuh"

namespace {

constexpr int TS = 16;              // tile edge (pixels)
constexpr int R5 = 5;               // window radius
constexpr int TH = TS + 2 * R5;     // tile edge with halo
constexpr int ROWF = TH * 3;        // floats per staged row (3 channels interleaved)
constexpr int OUTF = TS * 3;        // outputs per row

__constant__ double c_g[11];

struct SsimAcc {
    double sum_s;
};

__device__ __forceinline__ void load_tile(const float* __restrict__ img, int W, int H, int x0, int y0, float* __restrict__ s) {
    // s[TH][ROWF]; zero outside the image (the padding of the "same" correlation)
    for (int i = threadIdx.x; i < TH * ROWF; i += blockDim.x) {
        const int ry = i / ROWF, rc = i - ry * ROWF;
        const int y = y0 - R5 + ry, xc = (x0 - R5) * 3 + rc;
        s[i] = (y >= 0 && y < H && xc >= 0 && xc < W * 3) ? __ldg(img + (size_t)y * W * 3 + xc) : 0.f;
    }
}

__global__ void __launch_bounds__(256) ssim_stats_kernel(const float* __restrict__ render, const float* __restrict__ target, int W, int H,
                                                         float* __restrict__ dm1, float* __restrict__ dq11, float* __restrict__ dq12,
                                                         SsimAcc* __restrict__ acc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* h = reinterpret_cast<double*>(smem_raw);                    // [5][TH][OUTF] horizontal sums
    float* sR = reinterpret_cast<float*>(h + 5 * TH * OUTF);            // [TH][ROWF]
    float* sI = sR + TH * ROWF;
    __shared__ double wsum[8];
    const int x0 = blockIdx.x * TS, y0 = blockIdx.y * TS;
    load_tile(render, W, H, x0, y0, sR);
    load_tile(target, W, H, x0, y0, sI);
    __syncthreads();
    for (int i = threadIdx.x; i < TH * OUTF; i += blockDim.x) {
        const int ry = i / OUTF, oc = i - ry * OUTF;                    // output column oc = 3 * px + ch
        double a = 0, b = 0, aa = 0, bb = 0, ab = 0;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const double g = c_g[k];
            const double r = (double)sR[ry * ROWF + oc + 3 * k], t = (double)sI[ry * ROWF + oc + 3 * k];
            a += g * r; b += g * t; aa += g * (r * r); bb += g * (t * t); ab += g * (r * t);
        }
        h[0 * TH * OUTF + i] = a; h[1 * TH * OUTF + i] = b; h[2 * TH * OUTF + i] = aa; h[3 * TH * OUTF + i] = bb; h[4 * TH * OUTF + i] = ab;
    }
    __syncthreads();
    double local = 0.0;
    for (int i = threadIdx.x; i < TS * OUTF; i += blockDim.x) {
        const int oy = i / OUTF, oc = i - oy * OUTF;
        const int y = y0 + oy, xc = x0 * 3 + oc;
        if (y >= H || xc >= W * 3) continue;
        double m[5] = {0, 0, 0, 0, 0};
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const double g = c_g[k];
#pragma unroll
            for (int q = 0; q < 5; ++q) m[q] += g * h[q * TH * OUTF + (oy + k) * OUTF + oc];
        }
        const double mu1 = m[0], mu2 = m[1];
        const double s11 = m[2] - mu1 * mu1, s22 = m[3] - mu2 * mu2, s12 = m[4] - mu1 * mu2;
        const double C1 = 1e-4, C2 = 9e-4;
        const double A1 = 2.0 * mu1 * mu2 + C1, A2 = 2.0 * s12 + C2, B1 = mu1 * mu1 + mu2 * mu2 + C1, B2 = s11 + s22 + C2;
        const double iB = 1.0 / (B1 * B2);
        local += A1 * A2 * iB;
        const double d11 = -(A1 * A2) * iB / B2;
        const double d12 = 2.0 * A1 * iB;
        const double d1 = 2.0 * mu2 * A2 * iB - 2.0 * mu1 * A1 * A2 * iB / B1 - 2.0 * mu1 * d11 - mu2 * d12;
        const size_t o = (size_t)y * W * 3 + xc;
        dm1[o] = (float)d1; dq11[o] = (float)d11; dq12[o] = (float)d12;
    }
    // block sum of the index -> one double atomic per block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) local += __shfl_down_sync(0xffffffffu, local, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = local;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += wsum[w];
        atomicAdd(&acc->sum_s, t);
    }
}

__global__ void __launch_bounds__(256) ssim_grad_kernel(const float* __restrict__ render, const float* __restrict__ target, int W, int H,
                                                        const float* __restrict__ dm1, const float* __restrict__ dq11,
                                                        const float* __restrict__ dq12, const SsimAcc* __restrict__ acc, float lambda,
                                                        int accumulate, float* __restrict__ dL, float* __restrict__ loss) {
    __shared__ float sD[3][TH * ROWF];          // the three derivative maps with halo
    __shared__ float hD[3][TH * OUTF];          // horizontal sums
    const int x0 = blockIdx.x * TS, y0 = blockIdx.y * TS;
    const double n = 3.0 * (double)W * (double)H;
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *loss = (float)(1.0 - acc->sum_s / n);
    load_tile(dm1, W, H, x0, y0, sD[0]);
    load_tile(dq11, W, H, x0, y0, sD[1]);
    load_tile(dq12, W, H, x0, y0, sD[2]);
    __syncthreads();
    for (int i = threadIdx.x; i < TH * OUTF; i += blockDim.x) {
        const int ry = i / OUTF, oc = i - ry * OUTF;
        float a = 0.f, b = 0.f, c = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float g = (float)c_g[k];
            a = fmaf(g, sD[0][ry * ROWF + oc + 3 * k], a);
            b = fmaf(g, sD[1][ry * ROWF + oc + 3 * k], b);
            c = fmaf(g, sD[2][ry * ROWF + oc + 3 * k], c);
        }
        hD[0][i] = a; hD[1][i] = b; hD[2][i] = c;
    }
    __syncthreads();
    const float scale = (float)(-(double)lambda / n);
    for (int i = threadIdx.x; i < TS * OUTF; i += blockDim.x) {
        const int oy = i / OUTF, oc = i - oy * OUTF;
        const int y = y0 + oy, xc = x0 * 3 + oc;
        if (y >= H || xc >= W * 3) continue;
        float a = 0.f, b = 0.f, c = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float g = (float)c_g[k];
            a = fmaf(g, hD[0][(oy + k) * OUTF + oc], a);
            b = fmaf(g, hD[1][(oy + k) * OUTF + oc], b);
            c = fmaf(g, hD[2][(oy + k) * OUTF + oc], c);
        }
        const size_t o = (size_t)y * W * 3 + xc;
        const float v = scale * (a + 2.f * __ldg(render + o) * b + __ldg(target + o) * c);
        dL[o] = accumulate ? dL[o] + v : v;
    }
}

}  // namespace

extern "C" SvrStatus svr_ssim_loss_grad(SvrContext* ctx, const float* render, const float* target, int32_t W, int32_t H, float lambda,
                                        int32_t accumulate, float* dL_dimage, float* loss) {
    SVR_NVTX();
    if (!ctx || !render || !target || !dL_dimage || !loss) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (W <= 0 || H <= 0) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "empty image");
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    const int smem_stats = 5 * TH * OUTF * (int)sizeof(double) + 2 * TH * ROWF * (int)sizeof(float);
    static double g[11];
    static bool have_g = false;
    if (!have_g) {
        double sum = 0.0;
        for (int k = 0; k < 11; ++k) { g[k] = exp(-(double)((k - 5) * (k - 5)) / (2.0 * 1.5 * 1.5)); sum += g[k]; }
        for (int k = 0; k < 11; ++k) g[k] /= sum;
        have_g = true;
    }
    // per call, on the context's stream: the constant and the attribute belong to the current device
    SVR_CUDA(ctx, cudaMemcpyToSymbolAsync(c_g, g, sizeof(g), 0, cudaMemcpyHostToDevice, ctx->stream));
    SVR_CUDA(ctx, cudaFuncSetAttribute(ssim_stats_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_stats));
    const size_t nf = (size_t)W * H * 3, map_bytes = sizeof(float) * nf, bytes = 3 * map_bytes + 256;
    unsigned char* ws = nullptr;
    SVR_TRY(svr_alloc(ctx, (void**)&ws, bytes));
    SsimAcc* acc = reinterpret_cast<SsimAcc*>(ws);
    float* dm1 = reinterpret_cast<float*>(ws + 256);
    float *dq11 = dm1 + nf, *dq12 = dq11 + nf;
    SvrStatus st = SVR_OK;
    cudaError_t e = cudaMemsetAsync(acc, 0, sizeof(SsimAcc), ctx->stream);
    if (e == cudaSuccess) {
        const dim3 grid((unsigned int)((W + TS - 1) / TS), (unsigned int)((H + TS - 1) / TS));
        ssim_stats_kernel<<<grid, 256, smem_stats, ctx->stream>>>(render, target, W, H, dm1, dq11, dq12, acc);
        ssim_grad_kernel<<<grid, 256, 0, ctx->stream>>>(render, target, W, H, dm1, dq11, dq12, acc, lambda, accumulate, dL_dimage, loss);
        ctx->launches += 2;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) st = svr_fail(ctx, SVR_ERR_CUDA, "ssim: %s", cudaGetErrorString(e));
    svr_free(ctx, ws, bytes);
    return st;
}

// ---- svr_ssim_loss_grad_static: the same two kernels, for callers that must not allocate ----
//
// svr_ssim_loss_grad above takes its three derivative maps (36 B per pixel) from the context's workspace pool, and getting a
// context at all means a memory pool and streams have been created. Some users of this library cannot do either at the point
// where they need L_SSIM: a plug-in running inside a host process whose own allocator has already claimed the device memory
// (a raw allocation from here can fail although that allocator still has room), code under a hard per-process memory
// reservation where every byte has to be accounted for before the run starts, and loops that cannot tolerate the device-wide
// stall an allocation or a free may cause. For them the scratch below is part of the library image: it is reserved on every
// GPU that loads libsvr.so, from load until the process exits, and this entry point makes no allocation call of any kind.
//
// g_ssim_static_scratch is a DEVICE array. In host code its name only stands for the symbol; it is not an address a kernel can
// use. The host side therefore asks the runtime for the device address once per device (cudaGetSymbolAddress, with that device
// current) and hands that pointer to the kernels.
namespace {

constexpr int64_t kStaticMaxPixels = SVR_SSIM_STATIC_MAX_PIXELS;
constexpr size_t kStaticMapFloats = (size_t)kStaticMaxPixels * 3;
constexpr size_t kStaticBytes = 256 + 3 * kStaticMapFloats * sizeof(float);   // accumulator block + dm1, dq11, dq12 at the limit
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) unsigned char g_ssim_static_scratch[kStaticBytes];

std::mutex g_static_mu;                                   // guards the per-device set-up table
unsigned char* g_static_ptr[kStaticMaxDevices] = {};      // device address of the scratch on device d (nullptr: not set up yet)
thread_local char g_static_err[256] = "";

SvrStatus static_fail(SvrStatus st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
    va_end(ap);
    return st;
}

#define SVR_STATIC_CUDA(call)                                                                                              \
    do {                                                                                                                   \
        cudaError_t e__ = (call);                                                                                          \
        if (e__ != cudaSuccess) return static_fail(SVR_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__));         \
    } while (0)

// Once per device, with that device current: resolve the scratch symbol to its device address, upload the window, raise the
// dynamic shared memory limit of the first kernel. Synchronous.
SvrStatus static_setup(int device, unsigned char** out) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (g_static_ptr[device]) { *out = g_static_ptr[device]; return SVR_OK; }
    unsigned char* ptr = nullptr;
    SVR_STATIC_CUDA(cudaGetSymbolAddress((void**)&ptr, g_ssim_static_scratch));
    if (!ptr) return static_fail(SVR_ERR_CUDA, "cudaGetSymbolAddress returned a null scratch address on device %d", device);
    double g[11], sum = 0.0;
    for (int k = 0; k < 11; ++k) { g[k] = exp(-(double)((k - 5) * (k - 5)) / (2.0 * 1.5 * 1.5)); sum += g[k]; }
    for (int k = 0; k < 11; ++k) g[k] /= sum;
    SVR_STATIC_CUDA(cudaMemcpyToSymbol(c_g, g, sizeof(g), 0, cudaMemcpyHostToDevice));
    const int smem_stats = 5 * TH * OUTF * (int)sizeof(double) + 2 * TH * ROWF * (int)sizeof(float);
    SVR_STATIC_CUDA(cudaFuncSetAttribute(ssim_stats_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_stats));
    g_static_ptr[device] = ptr;
    *out = ptr;
    return SVR_OK;
}

}  // namespace

extern "C" int64_t svr_ssim_static_max_pixels(void) { return kStaticMaxPixels; }

extern "C" const char* svr_static_last_error(void) { return g_static_err; }

extern "C" SvrStatus svr_ssim_loss_grad_static(int device, void* cuda_stream, const float* render, const float* target, int32_t W,
                                               int32_t H, float lambda, int32_t accumulate, float* dL_dimage, float* loss) {
    g_static_err[0] = 0;
    if (!render || !target || !dL_dimage || !loss) return static_fail(SVR_ERR_INVALID_ARG, "null argument");
    if (W <= 0 || H <= 0) return static_fail(SVR_ERR_INVALID_ARG, "empty image");
    if (device < 0 || device >= kStaticMaxDevices) return static_fail(SVR_ERR_INVALID_ARG, "device %d outside 0..%d", device, kStaticMaxDevices - 1);
    const int64_t pixels = (int64_t)W * (int64_t)H;
    if (pixels > kStaticMaxPixels)
        return static_fail(SVR_ERR_UNSUPPORTED,
                           "image %d x %d = %lld pixels is over the %lld-pixel limit of the built-in scratch array; use svr_ssim_loss_grad",
                           W, H, (long long)pixels, (long long)kStaticMaxPixels);
    SVR_STATIC_CUDA(cudaSetDevice(device));
    unsigned char* ws = nullptr;
    SVR_TRY(static_setup(device, &ws));
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const size_t nf = (size_t)pixels * 3;
    SsimAcc* acc = reinterpret_cast<SsimAcc*>(ws);
    float* dm1 = reinterpret_cast<float*>(ws + 256);
    float *dq11 = dm1 + nf, *dq12 = dq11 + nf;
    // the array keeps what the previous call left in it: the index sum has to start at zero, the maps are fully rewritten
    // over the W x H pixels the second kernel reads (its halo reads outside the image are zero by construction)
    SVR_STATIC_CUDA(cudaMemsetAsync(acc, 0, sizeof(SsimAcc), stream));
    const int smem_stats = 5 * TH * OUTF * (int)sizeof(double) + 2 * TH * ROWF * (int)sizeof(float);
    const dim3 grid((unsigned int)((W + TS - 1) / TS), (unsigned int)((H + TS - 1) / TS));
    ssim_stats_kernel<<<grid, 256, smem_stats, stream>>>(render, target, W, H, dm1, dq11, dq12, acc);
    ssim_grad_kernel<<<grid, 256, 0, stream>>>(render, target, W, H, dm1, dq11, dq12, acc, lambda, accumulate, dL_dimage, loss);
    SVR_STATIC_CUDA(cudaGetLastError());
    return SVR_OK;
}
