// Stage (5): LF-weighted photometric loss gradient (eqs. 7-10; DESIGN.md row a8, reading R10).
//
//   s(p) = min(1, m(p)/m_q), m = 3x3 Sobel magnitude of the channel-mean grey SOURCE image (target by
//   default), replicate border, m_q = nearest-rank q-quantile;  w = (eps + 1 - s)^gamma  (eq. 7);
//   w~ = w / mean(w)  (eq. 8);  L = 1/|P| sum w~ * mean_ch |R - I|  (eq. 10/18);
//   dL/dR = w~ sign(R - I) / (3 |P|).
//
// Kernels: (1) Sobel magnitude + 2048-bin histogram of the top 11 bits of its float pattern; (2,3) radix
// select refinements (11 + 10 + 10 bits => the exact quantile element, no sort); (4) sum of w and of
// w * sum_ch |r|; (5) gradient write + loss. All HBM-trivial (about 40 B/pixel).
#include "svr_internal.cuh"

namespace {

struct LossWs {
    unsigned int hist[3][2048];
    unsigned int prefix[3];      // selected bucket value after pass 0, 1, 2 (accumulated bit pattern)
    unsigned int rank[3];        // remaining rank inside the selected bucket
    double sum_w;
    double sum_wr;
};

__device__ __forceinline__ float grey_at(const float* __restrict__ img, int W, int H, int x, int y) {
    x = min(max(x, 0), W - 1);
    y = min(max(y, 0), H - 1);
    const float* p = img + ((size_t)y * W + x) * 3;
    return (p[0] + p[1] + p[2]) * (1.0f / 3.0f);
}

__global__ void __launch_bounds__(256) sobel_hist_kernel(const float* __restrict__ src, int W, int H, float* __restrict__ mag,
                                                         LossWs* __restrict__ ws) {
    __shared__ unsigned int h[2048];
    for (int i = threadIdx.x; i < 2048; i += 256) h[i] = 0;
    __syncthreads();
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (p < (int64_t)W * H) {
        int x = (int)(p % W), y = (int)(p / W);
        float a = grey_at(src, W, H, x - 1, y - 1), b = grey_at(src, W, H, x, y - 1), cc = grey_at(src, W, H, x + 1, y - 1);
        float d = grey_at(src, W, H, x - 1, y), f = grey_at(src, W, H, x + 1, y);
        float g = grey_at(src, W, H, x - 1, y + 1), hh = grey_at(src, W, H, x, y + 1), i = grey_at(src, W, H, x + 1, y + 1);
        float gx = (cc - a) + 2.f * (f - d) + (i - g);
        float gy = (g - a) + 2.f * (hh - b) + (i - cc);
        float m = sqrtf(gx * gx + gy * gy);
        mag[p] = m;
        atomicAdd(&h[__float_as_uint(m) >> 20], 1u);       // m >= 0: bits 30..20
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2048; i += 256)
        if (h[i]) atomicAdd(&ws->hist[0][i], h[i]);
}

// One block: find the bucket of pass `pass` that holds the wanted rank.
__global__ void __launch_bounds__(256) select_kernel(LossWs* __restrict__ ws, int pass, unsigned int k0) {
    __shared__ unsigned int part[256];
    const int nb = (pass == 0) ? 2048 : 1024;
    const int per = nb / 256;
    unsigned int k = (pass == 0) ? k0 : ws->rank[pass - 1];
    unsigned int local = 0;
    for (int i = 0; i < per; ++i) local += ws->hist[pass][threadIdx.x * per + i];
    part[threadIdx.x] = local;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int run = 0;
        int t = 0;
        for (; t < 255; ++t) {
            if (run + part[t] > k) break;
            run += part[t];
        }
        int bsel = t * per;
        for (int i = 0; i < per; ++i) {
            unsigned int hv = ws->hist[pass][t * per + i];
            bsel = t * per + i;
            if (run + hv > k) break;
            run += hv;
        }
        unsigned int prev = (pass == 0) ? 0u : ws->prefix[pass - 1];
        int shift = (pass == 0) ? 20 : (pass == 1 ? 10 : 0);
        ws->prefix[pass] = prev | ((unsigned int)bsel << shift);
        ws->rank[pass] = k - run;
    }
}

__global__ void __launch_bounds__(256) refine_hist_kernel(const float* __restrict__ mag, int64_t n, LossWs* __restrict__ ws,
                                                          int pass) {
    __shared__ unsigned int h[1024];
    for (int i = threadIdx.x; i < 1024; i += 256) h[i] = 0;
    __syncthreads();
    const unsigned int prefix = ws->prefix[pass - 1];
    const int hi_shift = (pass == 1) ? 20 : 10, lo_shift = (pass == 1) ? 10 : 0;
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (p < n) {
        unsigned int u = __float_as_uint(mag[p]);
        if ((u >> hi_shift) == (prefix >> hi_shift)) atomicAdd(&h[(u >> lo_shift) & 1023u], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 1024; i += 256)
        if (h[i]) atomicAdd(&ws->hist[pass][i], h[i]);
}

__device__ __forceinline__ float lf_weight(float m, float mq, float eps, float gamma) {
    float s = (mq > 0.f) ? fminf(1.f, m / mq) : 0.f;
    return exp2f(gamma * log2f(eps + 1.f - s));
}

__device__ __forceinline__ double block_sum(double v, double* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < 8; ++i) t += sh[i];
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(256) weight_sum_kernel(const float* __restrict__ mag, const float* __restrict__ render,
                                                         const float* __restrict__ target, int64_t n, float eps, float gamma,
                                                         LossWs* __restrict__ ws) {
    __shared__ double sh[8];
    const float mq = __uint_as_float(ws->prefix[2]);
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    double w = 0.0, wr = 0.0;
    if (p < n) {
        float wf = lf_weight(mag[p], mq, eps, gamma);
        float r0 = fabsf(render[p * 3] - target[p * 3]), r1 = fabsf(render[p * 3 + 1] - target[p * 3 + 1]),
              r2 = fabsf(render[p * 3 + 2] - target[p * 3 + 2]);
        w = (double)wf;
        wr = (double)wf * ((double)r0 + (double)r1 + (double)r2);
    }
    double tw = block_sum(w, sh);
    double twr = block_sum(wr, sh);
    if (threadIdx.x == 0) {
        atomicAdd(&ws->sum_w, tw);
        atomicAdd(&ws->sum_wr, twr);
    }
}

__device__ __forceinline__ float signf(float r) { return (r > 0.f) ? 1.f : ((r < 0.f) ? -1.f : 0.f); }

__global__ void __launch_bounds__(256) grad_kernel(const float* __restrict__ mag, const float* __restrict__ render,
                                                   const float* __restrict__ target, int64_t n, float eps, float gamma,
                                                   const LossWs* __restrict__ ws, float* __restrict__ dL, float* __restrict__ loss) {
    const float mq = __uint_as_float(ws->prefix[2]);
    const double mean_w = ws->sum_w / (double)n;
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (p == 0) *loss = (float)(ws->sum_wr / mean_w / (3.0 * (double)n));
    if (p >= n) return;
    float scale = (float)((double)lf_weight(mag[p], mq, eps, gamma) / mean_w / (3.0 * (double)n));
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) dL[p * 3 + ch] = scale * signf(render[p * 3 + ch] - target[p * 3 + ch]);
}

}  // namespace

static SvrStatus loss_workspace(SvrContext* ctx, int64_t n) {
    size_t need = sizeof(LossWs) + sizeof(float) * (size_t)n + 256;
    if (ctx->loss_ws_bytes < need) {
        if (ctx->loss_ws) svr_free(ctx, ctx->loss_ws, ctx->loss_ws_bytes);
        ctx->loss_ws = nullptr;
        ctx->loss_ws_bytes = 0;
        SVR_TRY(svr_alloc(ctx, &ctx->loss_ws, need));
        ctx->loss_ws_bytes = need;
    }
    return SVR_OK;
}

// The part of eq. 7 that reads only the Sobel source: magnitude and its q-quantile (6 launches) on `stream`.
static SvrStatus loss_source_phase(SvrContext* ctx, cudaStream_t stream, const float* src, int W, int H, float q) {
    const int64_t n = (int64_t)W * H;
    LossWs* ws = reinterpret_cast<LossWs*>(ctx->loss_ws);
    float* mag = reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(ctx->loss_ws) + ((sizeof(LossWs) + 255) & ~(size_t)255));
    SVR_CUDA(ctx, cudaMemsetAsync(ws, 0, sizeof(LossWs), stream));
    // nearest-rank quantile: sorted[ceil(q n) - 1]
    double kq = ceil((double)q * (double)n) - 1.0;
    if (kq < 0) kq = 0;
    if (kq > (double)(n - 1)) kq = (double)(n - 1);
    unsigned int k0 = (unsigned int)kq;
    unsigned int g = (unsigned int)((n + 255) / 256);
    sobel_hist_kernel<<<g, 256, 0, stream>>>(src, W, H, mag, ws);
    select_kernel<<<1, 256, 0, stream>>>(ws, 0, k0);
    refine_hist_kernel<<<g, 256, 0, stream>>>(mag, n, ws, 1);
    select_kernel<<<1, 256, 0, stream>>>(ws, 1, 0);
    refine_hist_kernel<<<g, 256, 0, stream>>>(mag, n, ws, 2);
    select_kernel<<<1, 256, 0, stream>>>(ws, 2, 0);
    ctx->launches += 6;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// svr_loss_prepare: the source phase on the context's second stream, ordered after everything already queued on the main
// stream (the producer of `target`, the previous loss call that still reads the workspace) and after what is queued on the
// second stream (the host path's upload).
SvrStatus launch_loss_prepare(SvrContext* ctx, const float* target, int W, int H, float q) {
    const int64_t n = (int64_t)W * H;
    if (ctx->loss_prepared) SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->loss_ready_ev, 0));   // an unconsumed phase: replaced
    SVR_TRY(loss_workspace(ctx, n));
    SVR_CUDA(ctx, cudaEventRecord(ctx->fork_ev, ctx->stream));
    SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->aux, ctx->fork_ev, 0));
    SVR_TRY(loss_source_phase(ctx, ctx->aux, target, W, H, q));
    SVR_CUDA(ctx, cudaEventRecord(ctx->loss_ready_ev, ctx->aux));
    ctx->loss_prepared = true;
    ctx->loss_prep_target = target;
    ctx->loss_prep_W = W; ctx->loss_prep_H = H; ctx->loss_prep_q = q;
    return SVR_OK;
}

SvrStatus launch_loss_grad(SvrContext* ctx, const float* render, const float* target, int W, int H, float gamma, float eps,
                           float q, int sobel_source, float* dL, float* loss) {
    StageScope scope__(ctx, ST_LOSS);
    const int64_t n = (int64_t)W * H;
    const bool prepared = ctx->loss_prepared && sobel_source == 0 && ctx->loss_prep_target == target && ctx->loss_prep_W == W &&
                          ctx->loss_prep_H == H && ctx->loss_prep_q == q;
    if (ctx->loss_prepared) {        // a prepared phase is consumed (or discarded) by the next loss call; either way wait for it
        SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->loss_ready_ev, 0));
        ctx->loss_prepared = false;
    }
    if (!prepared) {
        SVR_TRY(loss_workspace(ctx, n));
        SVR_TRY(loss_source_phase(ctx, ctx->stream, sobel_source == 0 ? target : render, W, H, q));
    }
    LossWs* ws = reinterpret_cast<LossWs*>(ctx->loss_ws);
    float* mag = reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(ctx->loss_ws) + ((sizeof(LossWs) + 255) & ~(size_t)255));
    unsigned int g = (unsigned int)((n + 255) / 256);
    weight_sum_kernel<<<g, 256, 0, ctx->stream>>>(mag, render, target, n, eps, gamma, ws);
    grad_kernel<<<g, 256, 0, ctx->stream>>>(mag, render, target, n, eps, gamma, ws, dL, loss);
    ctx->launches += 2;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}
