// svr_measure_peaks: the two machine peaks the compositing kernels are set against and that no vendor table gives
// ("The builder measures the FMA peak with a microbenchmark at the clock actually sustained"; "a9 tail: L2 atomic
// throughput ... microbenchmark it"). Measurement hook only: nothing on the hot path calls it.
//   out[0] FP32 FMA rate, TFLOP/s      (FFMA, 8 independent chains per thread, all SMs, FMA = 2 flop)
//   out[1] packed FP32x2 FMA rate, TFLOP/s (FFMA2: two FMAs per lane per instruction; same pipe, half the issue slots)
//   out[2] L2 reduction rate, 1e9 red.global.add.v4.f32 per second (16-byte vector float reductions, one 32-byte sector each,
//          random rows of an L2-resident table: the form the backward kernel's gradient accumulation takes)
//   out[3] warp-instruction issue rate, 1e9 warp instructions per second (integer ALU chain: the bound of a kernel whose
//          instructions are not FP32)
#include "svr_internal.cuh"

namespace {

constexpr int PEAK_ITERS = 4096;

__global__ void __launch_bounds__(256) ffma_peak_kernel(float* out, float a, float b) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 123.456f) out[0] = s;       // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) ffma2_peak_kernel(float* out, float a, float b) {
    unsigned long long x[8], aa, bb;
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    aa = *reinterpret_cast<const unsigned long long*>(&a2);
    bb = *reinterpret_cast<const unsigned long long*>(&b2);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float2 v = make_float2((float)(threadIdx.x + i), (float)i);
        x[i] = *reinterpret_cast<const unsigned long long*>(&v);
    }
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(aa), "l"(bb));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { const float2 v = *reinterpret_cast<const float2*>(&x[i]); s += v.x + v.y; }
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(256) issue_peak_kernel(unsigned int* out, unsigned int a) {
    unsigned int x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x + i;
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = (x[i] ^ a) + (unsigned int)it;      // LOP3 + IADD: two ALU instructions
    }
    unsigned int s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 0x12345u) out[0] = s;
}

// every thread: `reps` vector reductions to pseudo-random 32-byte rows of a table of `rows` rows (L2-resident)
__global__ void __launch_bounds__(256) red_peak_kernel(float* table, unsigned int rows, int reps) {
    unsigned int h = (blockIdx.x * 256u + threadIdx.x) * 2654435761u + 12345u;
    for (int r = 0; r < reps; ++r) {
        h = h * 1664525u + 1013904223u;
        float* p = table + (size_t)((h >> 8) % rows) * 8 + ((h >> 4) & 1u) * 4;
        asm volatile("red.global.add.v4.f32 [%0], {%1, %1, %1, %1};" ::"l"(p), "f"(1.0f) : "memory");
    }
}

}  // namespace

extern "C" SvrStatus svr_measure_peaks(SvrContext* ctx, float* out_host) {
    SVR_NVTX();
    if (!ctx || !out_host) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaDeviceProp prop;
    SVR_CUDA(ctx, cudaGetDeviceProperties(&prop, ctx->device));
    const int n_sm = prop.multiProcessorCount;
    const int blocks = n_sm * 8;                       // 2048 threads per SM: full occupancy
    const unsigned int rows = 1u << 20;                // 32 MB table: resident in the 126 MB L2
    SVR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));          // time on an idle stream: earlier work must not sit inside the first interval
    float* table = nullptr;
    SVR_TRY(svr_alloc(ctx, (void**)&table, sizeof(float) * 8 * (size_t)rows + 256));
    float* sink = table + (size_t)rows * 8;
    cudaEvent_t e[2] = {nullptr, nullptr};
    // every exit below goes through this: the events are destroyed and the table goes back to the workspace
    auto done = [&](cudaError_t err, const char* what) -> SvrStatus {
        for (auto& ev : e) if (ev) cudaEventDestroy(ev);
        svr_free(ctx, table, 0);
        return err == cudaSuccess ? SVR_OK : svr_fail(ctx, SVR_ERR_CUDA, "svr_measure_peaks: %s: %s", what, cudaGetErrorString(err));
    };
    for (auto& ev : e) { const cudaError_t err = cudaEventCreate(&ev); if (err != cudaSuccess) return done(err, "cudaEventCreate"); }
#define PEAK_CUDA(call, what) do { const cudaError_t err__ = (call); if (err__ != cudaSuccess) return done(err__, what); } while (0)
    auto timed = [&](auto launch, float* ms_best) -> cudaError_t {
        *ms_best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {            // first repetition warms up
            cudaEventRecord(e[0], ctx->stream);
            launch();
            cudaEventRecord(e[1], ctx->stream);
            cudaError_t err = cudaEventSynchronize(e[1]);
            if (err != cudaSuccess) return err;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e[0], e[1]);
            if (rep > 0 && ms < *ms_best) *ms_best = ms;
        }
        return cudaGetLastError();
    };
    float ms = 0.f;
    PEAK_CUDA(cudaMemsetAsync(table, 0, sizeof(float) * 8 * (size_t)rows + 256, ctx->stream), "clearing the table");
    PEAK_CUDA(timed([&] { ffma_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(sink, 0.999f, 0.001f); }, &ms), "ffma_peak_kernel");
    const double fma_per_launch = (double)blocks * 256.0 * PEAK_ITERS * 8.0;
    out_host[0] = (float)(2.0 * fma_per_launch / (ms * 1e-3) / 1e12);
    PEAK_CUDA(timed([&] { ffma2_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(sink, 0.999f, 0.001f); }, &ms), "ffma2_peak_kernel");
    out_host[1] = (float)(4.0 * fma_per_launch / (ms * 1e-3) / 1e12);
    const int reps = 256;
    PEAK_CUDA(timed([&] { red_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(table, rows, reps); }, &ms), "red_peak_kernel");
    out_host[2] = (float)((double)blocks * 256.0 * reps / (ms * 1e-3) / 1e9);
    PEAK_CUDA(timed([&] { issue_peak_kernel<<<blocks, 256, 0, ctx->stream>>>(reinterpret_cast<unsigned int*>(sink), 0x5bd1e995u); }, &ms), "issue_peak_kernel");
    out_host[3] = (float)((double)blocks * 8.0 * PEAK_ITERS * 8.0 * 2.0 / (ms * 1e-3) / 1e9);
#undef PEAK_CUDA
    ctx->launches += 16;
    return done(cudaSuccess, "");
}
