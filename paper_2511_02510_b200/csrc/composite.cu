// Stage (3) forward compositing and stage (4) backward compositing (DESIGN.md rows a7, a9).
//
// One CTA per 16x16 tile, 8 warps, each warp owns an 8x4 pixel block. The tile's sorted (tile, octant)
// list is staged CHUNK entries at a time into shared memory (voxel geometry relative to the camera centre
// in double-float form, 8 corner raws, per-view colour, pixel rectangle). Each warp first culls a batch of
// 32 staged voxels against its own 8x4 block (one rectangle test per lane, ballot), then walks only the
// survivors in list order; every lane slab-tests the survivor against its ray, integrates K midpoint
// samples of the trilinear raw density, and composites (eqs. 2-4). w_max (eq. 5) is reduced
// across the warp with one REDUX and one atomicMax per (warp, voxel). A ray stops once T < T_min; a warp
// stops when all its rays have, the CTA when all warps have.
//
// Precision: the ray is set up in fp64 per pixel and kept as hi+lo floats; voxel centres relative to the
// camera are staged as hi+lo floats. The slab test runs in coordinates relative to the ray's closest
// approach to the voxel centre, so the segment length (a difference of two O(1) ray parameters in the
// naive form) keeps ~1e-7 relative accuracy even for 4e-3-wide voxels 2.5 units away.
//
// Backward re-walks the list in the same front-to-back order with the stored final colour: the suffix
// colour S_k = image - prefix_k needs no division by (1 - alpha) (stable for tau >> 1), and
// dL/dtau_k = G . (T_k c_k - S_k). Per (warp, voxel) the 8 corner gradients + 3 colour gradients are
// reduced with a transposing butterfly (16 shuffles for all 11 values), accumulated per CTA in shared
// memory, and flushed once per chunk with coalesced float atomics.
#include "svr_internal.cuh"

namespace {

constexpr int CHUNK = 256;
constexpr unsigned FULL = 0xffffffffu;

struct Staged {
    float4 g0[CHUNK];   // gh.xyz, h (half edge)
    float4 g1[CHUNK];   // gl.xyz, voxel id bits
    float4 r0[CHUNK];   // raw corners 0..3
    float4 r1[CHUNK];   // raw corners 4..7
    float4 col[CHUNK];  // r, g, b, clamp mask
    uint2 rect[CHUNK];  // x0 | y0 << 16, x1 | y1 << 16
};

struct RayF {
    float dh[3], dl[3], inv[3], ainv[3];
};

__device__ __forceinline__ void setup_ray(const CamDev& c, int px, int py, RayF& r) {
    double u = ((double)px + 0.5 - (double)c.cx) / (double)c.fx;
    double v = ((double)py + 0.5 - (double)c.cy) / (double)c.fy;
    double d[3], n2 = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        d[a] = (double)c.R[a] * u + (double)c.R[3 + a] * v + (double)c.R[6 + a];
        n2 += d[a] * d[a];
    }
    double inv = 1.0 / sqrt(n2);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double da = d[a] * inv;
        r.dh[a] = (float)da;
        r.dl[a] = (float)(da - (double)r.dh[a]);
        float dd = (r.dh[a] == 0.0f) ? 1e-30f : r.dh[a];
        r.inv[a] = 1.0f / dd;
        r.ainv[a] = fabsf(r.inv[a]);
    }
}

__device__ __forceinline__ void stage_entry(Staged& S, int j, bool valid, uint32_t vid, const SceneDev& s, const CamDev& c,
                                            const ushort4* __restrict__ rects, const float4* __restrict__ rgbm) {
    if (!valid) {
        S.rect[j] = make_uint2(0xFFFFFFFFu, 0u);
        return;
    }
    uint2 q = __ldg(reinterpret_cast<const uint2*>(s.ijkl) + vid);
    int L = q.y >> 16;
    float ef = s.root_edge * __int_as_float((127 - L) << 23);
    double e = (double)ef;
    double gx = (double)s.root_lo[0] + ((double)(q.x & 0xFFFF) + 0.5) * e - c.o[0];
    double gy = (double)s.root_lo[1] + ((double)(q.x >> 16) + 0.5) * e - c.o[1];
    double gz = (double)s.root_lo[2] + ((double)(q.y & 0xFFFF) + 0.5) * e - c.o[2];
    float hx = (float)gx, hy = (float)gy, hz = (float)gz;
    S.g0[j] = make_float4(hx, hy, hz, 0.5f * ef);
    S.g1[j] = make_float4((float)(gx - (double)hx), (float)(gy - (double)hy), (float)(gz - (double)hz), __uint_as_float(vid));
    const float4* rp = reinterpret_cast<const float4*>(s.raw) + 2 * (size_t)vid;
    S.r0[j] = __ldg(rp);
    S.r1[j] = __ldg(rp + 1);
    S.col[j] = __ldg(rgbm + vid);
    ushort4 r = __ldg(rects + vid);
    S.rect[j] = make_uint2((unsigned)r.x | ((unsigned)r.y << 16), (unsigned)r.z | ((unsigned)r.w << 16));
}

__device__ __forceinline__ float lerpf(float a, float b, float t) { return fmaf(t, b - a, a); }

// Ray/voxel segment in coordinates relative to t_ref (the ray parameter closest to the voxel centre).
// Returns hit; outputs s0, s1 (segment in relative parameter), t_ref, D[3] (centre offset from the ray).
__device__ __forceinline__ bool slab(const RayF& r, const float4& a, const float4& b, float& s0, float& s1, float& t_ref,
                                     float* D) {
    t_ref = fmaf(a.z, r.dh[2], fmaf(a.y, r.dh[1], a.x * r.dh[0]));
    D[0] = fmaf(-t_ref, r.dh[0], a.x) + fmaf(-t_ref, r.dl[0], b.x);
    D[1] = fmaf(-t_ref, r.dh[1], a.y) + fmaf(-t_ref, r.dl[1], b.y);
    D[2] = fmaf(-t_ref, r.dh[2], a.z) + fmaf(-t_ref, r.dl[2], b.z);
    float h = a.w;
    float cx = D[0] * r.inv[0], cy = D[1] * r.inv[1], cz = D[2] * r.inv[2];
    float wx = h * r.ainv[0], wy = h * r.ainv[1], wz = h * r.ainv[2];
    s0 = fmaxf(fmaxf(cx - wx, cy - wy), fmaxf(cz - wz, -t_ref));
    s1 = fminf(fminf(cx + wx, cy + wy), cz + wz);
    return s1 > s0;
}

template <int K, bool BWD>
__device__ __forceinline__ float integrate(const RayF& r, const float* D, float h, float s0, float s1, const float4& ra,
                                           const float4& rb, float* dtau) {
    float inv_e = __int_as_float(0x7E800000 - __float_as_int(h));   // 0.5 / h for h a power of two
    float dt = (s1 - s0) * (1.0f / (float)K);
    float sum = 0.f;
    if (BWD) {
#pragma unroll
        for (int c = 0; c < 8; ++c) dtau[c] = 0.f;
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float s = fmaf((float)j + 0.5f, dt, s0);
        float qx = __saturatef(fmaf(fmaf(s, r.dh[0], -D[0]), inv_e, 0.5f));
        float qy = __saturatef(fmaf(fmaf(s, r.dh[1], -D[1]), inv_e, 0.5f));
        float qz = __saturatef(fmaf(fmaf(s, r.dh[2], -D[2]), inv_e, 0.5f));
        float r00 = lerpf(ra.x, ra.y, qx), r10 = lerpf(ra.z, ra.w, qx);
        float r01 = lerpf(rb.x, rb.y, qx), r11 = lerpf(rb.z, rb.w, qx);
        float rr = lerpf(lerpf(r00, r10, qy), lerpf(r01, r11, qy), qz);
        float sig = __expf(rr);
        sum += sig;
        if (BWD) {
            float sy0 = sig * (1.f - qy), sy1 = sig * qy;
            float a00 = sy0 * (1.f - qx), a10 = sy0 * qx, a01 = sy1 * (1.f - qx), a11 = sy1 * qx;
            float z0 = 1.f - qz;
            dtau[0] = fmaf(a00, z0, dtau[0]); dtau[1] = fmaf(a10, z0, dtau[1]);
            dtau[2] = fmaf(a01, z0, dtau[2]); dtau[3] = fmaf(a11, z0, dtau[3]);
            dtau[4] = fmaf(a00, qz, dtau[4]); dtau[5] = fmaf(a10, qz, dtau[5]);
            dtau[6] = fmaf(a01, qz, dtau[6]); dtau[7] = fmaf(a11, qz, dtau[7]);
        }
    }
    if (BWD) {
#pragma unroll
        for (int c = 0; c < 8; ++c) dtau[c] *= dt;
    }
    return dt * sum;
}

// Sum 11 per-lane values across the warp; after the call lane l (even) holds the total of value
// idx(l) = 8*b4 + 4*b3 + 2*b2 + b1 (bits of l). 16 shuffles instead of 55.
__device__ __forceinline__ float transpose_reduce11(float* v, int lane) {
    bool up = lane & 16;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float hi = (i + 8 < 11) ? v[i + 8] : 0.f;
        float send = up ? v[i] : hi, keep = up ? hi : v[i];
        v[i] = keep + __shfl_xor_sync(FULL, send, 16);
    }
    up = lane & 8;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        float send = up ? v[i] : v[i + 4], keep = up ? v[i + 4] : v[i];
        v[i] = keep + __shfl_xor_sync(FULL, send, 8);
    }
    up = lane & 4;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        float send = up ? v[i] : v[i + 2], keep = up ? v[i + 2] : v[i];
        v[i] = keep + __shfl_xor_sync(FULL, send, 4);
    }
    up = lane & 2;
    {
        float send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
        v[0] = keep + __shfl_xor_sync(FULL, send, 2);
    }
    return v[0] + __shfl_xor_sync(FULL, v[0], 1);
}

template <int K, bool BWD, bool STATS>
__global__ void __launch_bounds__(256) composite_kernel(SceneDev s, CamDev c, const uint32_t* __restrict__ vals,
                                                        const uint32_t* __restrict__ ranges, const ushort4* __restrict__ rects,
                                                        const float4* __restrict__ rgbm, float T_min,
                                                        float* __restrict__ image, float* __restrict__ depth,
                                                        float* __restrict__ T_final, unsigned int* __restrict__ w_max,
                                                        const float* __restrict__ dL, const float* __restrict__ image_in,
                                                        float* __restrict__ grad_raw, float* __restrict__ grad_rgb,
                                                        unsigned long long* __restrict__ stats) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Staged& S = *reinterpret_cast<Staged*>(smem_raw);
    float* acc = reinterpret_cast<float*>(smem_raw + sizeof(Staged));   // [CHUNK*12], BWD only

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x;
    const int tile_x = tile % c.tiles_x, tile_y = tile / c.tiles_x;
    const int wbx0 = tile_x * SVR_TILE + (warp & 1) * 8, wby0 = tile_y * SVR_TILE + (warp >> 1) * 4;
    const int px = wbx0 + (lane & 7), py = wby0 + (lane >> 3);
    const bool inimg = px < c.W && py < c.H;
    const size_t pix = (size_t)py * c.W + px;

    RayF ray;
    int oct = -1;
    if (inimg) {
        setup_ray(c, px, py, ray);
        oct = pixel_octant_dev(c, px, py);
    } else {
#pragma unroll
        for (int a = 0; a < 3; ++a) { ray.dh[a] = 0.f; ray.dl[a] = 0.f; ray.inv[a] = 0.f; ray.ainv[a] = 0.f; }
    }
    float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, Dep = 0.f;
    unsigned int n_hit = 0, n_test = 0, n_surv = 0, n_staged = 0;   // STATS only
    float G0 = 0.f, G1 = 0.f, G2 = 0.f, F0 = 0.f, F1 = 0.f, F2 = 0.f;
    if (BWD) {
        if (inimg) {
            G0 = dL[pix * 3]; G1 = dL[pix * 3 + 1]; G2 = dL[pix * 3 + 2];
            F0 = image_in[pix * 3]; F1 = image_in[pix * 3 + 1]; F2 = image_in[pix * 3 + 2];
        }
        for (int i = tid; i < CHUNK * 12; i += 256) acc[i] = 0.f;
    }

    for (int so = 0; so < 8; ++so) {
        const uint32_t start = ranges[(tile * 8 + so) * 2], end = ranges[(tile * 8 + so) * 2 + 1];
        if (start == end) continue;                                   // CTA-uniform
        bool alive = inimg && (oct == so) && (T >= T_min);
        for (uint32_t base = start; base < end; base += CHUNK) {
            __syncthreads();                                          // previous chunk fully consumed / flushed
            {
                uint32_t idx = base + tid;
                bool valid = idx < end;
                uint32_t vid = valid ? __ldg(vals + idx) : 0u;
                stage_entry(S, tid, valid, vid, s, c, rects, rgbm);
                if (STATS && valid) ++n_staged;
            }
            __syncthreads();
            const int nchunk = min((uint32_t)CHUNK, end - base);
            for (int b = 0; b < nchunk; b += 32) {
                if (!__any_sync(FULL, alive)) break;                  // whole warp terminated
                uint2 rc = S.rect[b + lane];
                bool ov = (int)(rc.x & 0xFFFF) <= wbx0 + 7 && (int)(rc.y & 0xFFFF) >= wbx0 &&
                          (int)(rc.x >> 16) <= wby0 + 3 && (int)(rc.y >> 16) >= wby0;
                unsigned m = __ballot_sync(FULL, ov);
                while (m) {
                    const int jj = __ffs(m) - 1;
                    m &= m - 1;
                    const int j = b + jj;
                    const unsigned rx = __shfl_sync(FULL, rc.x, jj), ry = __shfl_sync(FULL, rc.y, jj);
                    const bool inside = alive && px >= (int)(rx & 0xFFFF) && px <= (int)(ry & 0xFFFF) &&
                                        py >= (int)(rx >> 16) && py <= (int)(ry >> 16);
                    float w = 0.f;
                    float gv[11];
                    if (STATS) { n_surv += (lane == 0); n_test += inside; }
                    if (BWD) {
#pragma unroll
                        for (int i = 0; i < 11; ++i) gv[i] = 0.f;
                    }
                    if (inside) {
                        const float4 a = S.g0[j], bq = S.g1[j];
                        float s0, s1, t_ref, D[3];
                        if (slab(ray, a, bq, s0, s1, t_ref, D)) {
                            const float4 ra = S.r0[j], rb = S.r1[j], col = S.col[j];
                            float dtau[8];
                            float tau = integrate<K, BWD>(ray, D, a.w, s0, s1, ra, rb, dtau);
                            float E = __expf(-tau);
                            if (STATS) ++n_hit;
                            w = T * (1.f - E);
                            T *= E;
                            C0 = fmaf(w, col.x, C0); C1 = fmaf(w, col.y, C1); C2 = fmaf(w, col.z, C2);
                            if (!BWD) Dep = fmaf(w, t_ref + 0.5f * (s0 + s1), Dep);
                            if (BWD) {
                                // suffix colour S_k = final - prefix_k; dL/dtau = G . (T_k c_k - S_k)
                                float dLdtau = G0 * (fmaf(T, col.x, C0) - F0) + G1 * (fmaf(T, col.y, C1) - F1) +
                                               G2 * (fmaf(T, col.z, C2) - F2);
#pragma unroll
                                for (int cc = 0; cc < 8; ++cc) gv[cc] = dLdtau * dtau[cc];
                                gv[8] = w * G0; gv[9] = w * G1; gv[10] = w * G2;
                            }
                            if (T < T_min) alive = false;             // R8: stop after the voxel that crosses T_min
                        }
                    }
                    const unsigned wu = __reduce_max_sync(FULL, __float_as_uint(w));
                    if (wu != 0u) {
                        if (w_max != nullptr && lane == 0) atomicMax(w_max + __float_as_uint(S.g1[j].w), wu);
                        if (BWD) {
                            float tot = transpose_reduce11(gv, lane);
                            int idx = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
                            if (!(lane & 1) && idx < 11 && tot != 0.f) atomicAdd(&acc[j * 12 + idx], tot);
                        }
                    }
                }
            }
            const int any_alive = __syncthreads_or(alive ? 1 : 0);
            if (BWD) {
                // flush the chunk's accumulators: consecutive threads -> consecutive floats of one voxel
                for (int i = tid; i < nchunk * 12; i += 256) {
                    float val = acc[i];
                    if (val != 0.f) {
                        acc[i] = 0.f;
                        int j = i / 12, k = i - j * 12;
                        uint32_t vid = __float_as_uint(S.g1[j].w);
                        if (k < 8) atomicAdd(grad_raw + (size_t)vid * 8 + k, val);
                        else atomicAdd(grad_rgb + (size_t)vid * 4 + (k - 8), val);
                    }
                }
            }
            if (!any_alive) break;
        }
    }
    if (STATS) {
        unsigned int v4[4] = {n_hit, n_test, n_surv, n_staged};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            unsigned int t = __reduce_add_sync(FULL, v4[i]);
            if (lane == 0 && t) atomicAdd(stats + i, (unsigned long long)t);
        }
    }
    if (!BWD && inimg) {
        image[pix * 3] = fmaf(T, c.bg[0], C0);
        image[pix * 3 + 1] = fmaf(T, c.bg[1], C1);
        image[pix * 3 + 2] = fmaf(T, c.bg[2], C2);
        if (depth) depth[pix] = Dep;
        if (T_final) T_final[pix] = T;
    }
}

template <bool BWD>
SvrStatus launch_composite(SvrContext* ctx, const SvrFrame* f, int K, float T_min, float* image, float* depth, float* T_final,
                           float* w_max, const float* dL, const float* image_in, float* grad_raw, float* grad_rgb,
                           unsigned long long* stats) {
    if (f->n_tiles == 0) return SVR_OK;
    StageScope scope__(ctx, BWD ? ST_BACKWARD : ST_FORWARD);
    size_t smem = sizeof(Staged) + (BWD ? CHUNK * 12 * sizeof(float) : 0);
    const ushort4* rects = reinterpret_cast<const ushort4*>(f->rects);
    const float4* rgbm = reinterpret_cast<const float4*>(f->rgbm);
    unsigned int* wm = reinterpret_cast<unsigned int*>(w_max);
#define SVR_ARGS f->scene, f->cam, f->vals, f->ranges, rects, rgbm, T_min, image, depth, T_final, wm, dL, image_in, grad_raw, grad_rgb, stats
#define SVR_LAUNCH(KK)                                                                             \
    do {                                                                                           \
        if (!BWD && stats) composite_kernel<KK, false, true><<<f->n_tiles, 256, smem, ctx->stream>>>(SVR_ARGS); \
        else composite_kernel<KK, BWD, false><<<f->n_tiles, 256, smem, ctx->stream>>>(SVR_ARGS);   \
    } while (0)
    switch (K) {
        case 1: SVR_LAUNCH(1); break;
        case 2: SVR_LAUNCH(2); break;
        case 3: SVR_LAUNCH(3); break;
        case 4: SVR_LAUNCH(4); break;
        default: return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    }
#undef SVR_LAUNCH
#undef SVR_ARGS
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

}  // namespace

SvrStatus launch_forward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, float* image, float* depth, float* T_final,
                         float* w_max, unsigned long long* stats) {
    return launch_composite<false>(ctx, f, K, T_min, image, depth, T_final, w_max, nullptr, nullptr, nullptr, nullptr, stats);
}

SvrStatus launch_backward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, const float* dL, const float* image,
                          float* grad_raw, float* grad_rgb, float* w_max) {
    return launch_composite<true>(ctx, f, K, T_min, nullptr, nullptr, nullptr, w_max, dL, image, grad_raw, grad_rgb, nullptr);
}
