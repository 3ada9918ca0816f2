// Stage (3) forward compositing and stage (4) backward compositing (DESIGN.md rows a7, a9).
//
// One CTA per 16x16 tile; each of its 8 warps owns an 8x4 pixel block and runs independently (no CTA
// barrier anywhere): a barrier per staged chunk cost 37% of the issue slots in the first version
// (profiles/r1a_*), because the 8 blocks of a tile see very different numbers of voxels.
//
// Forward (composite_kernel), per warp, over the tile's sorted (tile, octant) list:
//   1. cull: 32 entries at a time, lane i reads entry i's pixel rectangle (in list order, so the read is
//      coalesced) and computes the 32-bit mask M of this warp's pixels it covers. M == 0 => the entry is
//      skipped by this warp (76% of (warp, entry) pairs on C4).
//   2. stage: surviving lanes copy their voxel's 80-byte view record (voxel_record_dev, svr_internal.cuh: centre
//      relative to the camera as hi+lo floats, half edge, density coefficients, per-view colour, dilated half edge),
//      gathered by the voxel id read beside the rectangle, in list order, into a warp-private shared-memory ring
//      (cp.async, double-buffered).
//   3. test: once >= 32 survivors are staged (or the list ends), the 32x32 bit matrix M[slot][pixel] is
//      transposed across the warp with 5 shuffles, giving every lane the bitmask of slots that cover ITS
//      pixel. Each lane pops its own candidates (ffs) and slab-tests them against a slightly dilated box:
//      lanes work on different voxels in the same instruction.
//   4. hits: each lane pops its own hits: precise slab test, K samples, eqs. 2-4; w_max (eq. 5,
//      P:95) by atomicMax guarded by a plain read (w_max only grows). Front-to-back order per pixel is kept
//      because slots are in list order.
// With REC the forward also writes, per batch, the staged voxel ids and every pixel's hit mask (the traversal record).
// Backward (backward_packed_kernel): replays that record, or runs the same cull / stage / test itself; then the hits
// are compacted into a queue and processed 32 at a time with all lanes busy; see the comment above that kernel.
//
// Density: the trilinear raw density is staged as polynomial coefficients (c0, cx, cy, cz, cxy, cxz, cyz,
// cxyz), pre-multiplied by log2(e), so a sample costs 7 FMA + one EX2 instead of 7 lerps (14 ops) + MUL + EX2.
// Backward accumulates the gradient w.r.t. those coefficients (monomials 1, qx, qy, qz, qxqy, ...) into a
// per-voxel scratch with 16-byte vector reductions (red.global.add.v4.f32; float atomics in shared memory are
// CAS loops on sm_100a, so nothing is accumulated there); the per-voxel finalize kernel (preprocess.cu) maps
// it back to the 8 corners.
//
// Precision: the ray is set up in fp64 per pixel and kept as hi+lo floats; the slab test runs in
// coordinates relative to the ray's closest approach to the voxel centre, so the segment length keeps
// ~1e-7 relative accuracy even for 4e-3-wide voxels 2.5 units away (a plain fp32 t_out - t_in loses 1e-4).
#include "svr_internal.cuh"

namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int RING = 64;          // staging slots per warp
constexpr int TRAV_WORDS = SVR_TRAV_WORDS;   // words of one traversal record (forward -> backward), see composite_kernel
constexpr int WARPS = 8;

struct WarpStage {
    float4 g0[RING];    // gh.xyz, h (half edge)
    float4 g1[RING];    // gl.xyz, voxel id bits
    float4 r0[RING];    // log2(e) * (c0, cx, cy, cz)
    float4 r1[RING];    // log2(e) * (cxy, cxz, cyz, cxyz)
    float4 col[RING];   // r, g, b, clamp mask
    unsigned int M[RING];   // pixels of this warp's 8x4 block covered by the voxel's rectangle
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

// Per visible voxel, once per view: everything the compositing warps need about it (5 x 16 B): centre relative to the
// camera as hi+lo floats (fp64 arithmetic), half edge, voxel id, the trilinear raw density as polynomial coefficients
// * log2(e), and the per-view colour. The compositing warps gather these records by voxel id.
__global__ void __launch_bounds__(256) voxel_record_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                           const float4* __restrict__ rgbm, float4* __restrict__ vrec) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    const ushort4 r = rects[v];
    if (r.x > r.z) return;                                   // not visible in this view: never read
    voxel_record_dev(s, c, __ldg(reinterpret_cast<const uint2*>(s.ijkl) + v), (uint32_t)v, __ldg(rgbm + v), vrec);
}

// rectangle in list order: the compositing cull reads it coalesced
__global__ void __launch_bounds__(256) gather_rects_kernel(const uint32_t* __restrict__ vals, int64_t n, const uint2* __restrict__ rects,
                                                           uint2* __restrict__ rects_sorted) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) rects_sorted[i] = __ldg(rects + __ldg(vals + i));
}

// 32-bit mask of the lanes (pixel = (wbx0 + (lane & 7), wby0 + (lane >> 3))) inside the rectangle.
__device__ __forceinline__ unsigned int block_cover_mask(uint2 rc, int wbx0, int wby0) {
    int cx0 = max((int)(rc.x & 0xFFFF) - wbx0, 0), cx1 = min((int)(rc.y & 0xFFFF) - wbx0, 7);
    int cy0 = max((int)(rc.x >> 16) - wby0, 0), cy1 = min((int)(rc.y >> 16) - wby0, 3);
    if (cx0 > cx1 || cy0 > cy1) return 0u;
    unsigned int colm = ((2u << cx1) - (1u << cx0)) & 0xFFu;
    unsigned int rowb = ((2u << cy1) - (1u << cy0)) & 0xFu;
    unsigned int rows = (rowb & 1u) | ((rowb & 2u) << 7) | ((rowb & 4u) << 14) | ((rowb & 8u) << 21);
    return colm * rows;
}

// Transpose a 32x32 bit matrix held one row per lane (row i in lane i): returns column `lane`.
__device__ __forceinline__ unsigned int transpose32(unsigned int x, int lane) {
#pragma unroll
    for (int j = 16; j >= 1; j >>= 1) {
        const unsigned int m = (j == 16) ? 0x0000FFFFu : (j == 8) ? 0x00FF00FFu : (j == 4) ? 0x0F0F0F0Fu
                             : (j == 2) ? 0x33333333u : 0x55555555u;
        unsigned int t = __shfl_xor_sync(FULL, x, j);
        x = (lane & j) ? (((t >> j) & m) | (x & ~m)) : ((x & m) | ((t & m) << j));
    }
    return x;
}

// Ray/voxel segment in coordinates relative to t_ref (the ray parameter closest to the voxel centre).
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

__device__ __forceinline__ float ex2f(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// K midpoint samples (R5). ca/cb = polynomial coefficients * log2(e). Returns tau; BWD also returns
// dtau[m] = d tau / d coef_m (natural-scale coefficients), m over monomials 1, qx, qy, qz, qxqy, qxqz, qyqz, qxqyqz.
template <int K, bool BWD>
__device__ __forceinline__ float integrate(const RayF& r, const float* D, float h, float s0, float s1, const float4& ca,
                                           const float4& cb, float* dtau) {
    float inv_e = __int_as_float(0x7E800000 - __float_as_int(h));   // 0.5 / h for h a power of two
    float dt = (s1 - s0) * (1.0f / (float)K);
    float sum = 0.f;
    if (BWD) {
#pragma unroll
        for (int c = 1; c < 8; ++c) dtau[c] = 0.f;
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float s = fmaf((float)j + 0.5f, dt, s0);
        float qx = __saturatef(fmaf(fmaf(s, r.dh[0], -D[0]), inv_e, 0.5f));
        float qy = __saturatef(fmaf(fmaf(s, r.dh[1], -D[1]), inv_e, 0.5f));
        float qz = __saturatef(fmaf(fmaf(s, r.dh[2], -D[2]), inv_e, 0.5f));
        float hi = fmaf(fmaf(cb.w, qz, cb.x), qy, fmaf(cb.y, qz, ca.y));     // (cxyz qz + cxy) qy + (cxz qz + cx)
        float lo = fmaf(fmaf(cb.z, qz, ca.z), qy, fmaf(ca.w, qz, ca.x));     // (cyz qz + cy) qy + (cz qz + c0)
        float sig = ex2f(fmaf(hi, qx, lo));
        sum += sig;
        if (BWD) {
            float sx = sig * qx, sy = sig * qy, sz = sig * qz;
            dtau[1] += sx; dtau[2] += sy; dtau[3] += sz;
            float sxy = sx * qy;
            dtau[4] += sxy;
            dtau[5] = fmaf(sx, qz, dtau[5]);
            dtau[6] = fmaf(sy, qz, dtau[6]);
            dtau[7] = fmaf(sxy, qz, dtau[7]);
        }
    }
    if (BWD) {
        dtau[0] = sum * dt;
#pragma unroll
        for (int c = 1; c < 8; ++c) dtau[c] *= dt;
    }
    return dt * sum;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned int d = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
template <int K, bool STATS, bool REC>
__global__ void __launch_bounds__(256, 4) composite_kernel(CamDev c, const float4* __restrict__ packed, const uint32_t* __restrict__ vals,
                                                        const uint2* __restrict__ rects_sorted,
                                                        const uint32_t* __restrict__ ranges,
                                                        const uint32_t* __restrict__ tile_order,
                                                        float T_min,
                                                        float* __restrict__ image, float* __restrict__ depth,
                                                        float* __restrict__ T_final, unsigned int* __restrict__ w_max,
                                                        unsigned long long* __restrict__ stats, uint32_t* __restrict__ trav,
                                                        const uint32_t* __restrict__ trav_off, uint32_t* __restrict__ trav_count) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    WarpStage& S = reinterpret_cast<WarpStage*>(smem_raw)[warp];
    const int tile = (int)tile_order[blockIdx.x];
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
    unsigned int n_hit = 0, n_test = 0, n_surv = 0, n_read = 0;   // STATS only
    // Traversal record for svr_backward (TRAV_WORDS words per batch: 32 hit masks, 32 voxel ids, the slot count): the
    // backward pass replays the batches and skips its own cull and test phases. This warp's records are contiguous.
    uint32_t* rec_out = nullptr;
    uint32_t n_rec = 0;
    if (REC) {
        const uint32_t r0 = trav_off[tile], cap = (trav_off[tile + 1] - r0) >> 3;
        rec_out = trav + ((size_t)r0 + (size_t)warp * cap) * TRAV_WORDS;
    }

    for (int so = 0; so < 8; ++so) {
        const uint32_t start = ranges[(tile * 8 + so) * 2], end = ranges[(tile * 8 + so) * 2 + 1];
        if (start == end) continue;
        bool alive = inimg && (oct == so) && (T >= T_min);
        unsigned int alive_mask = __ballot_sync(FULL, alive);
        if (alive_mask == 0u) continue;                               // no pixel of this warp uses this list
        // Double-buffered staging: the ring is two halves of 32 slots. While one half is walked, the records of the
        // next batch are already on their way into the other half (cp.async: no registers held, no stall on the load).
        uint32_t base = start;
        auto stage = [&](int half) -> int {
            int cnt = 0;
            while (cnt < 32 && base < end) {
                const uint32_t idx = base + lane;
                if (lane < 2) asm volatile("prefetch.global.L1 [%0];" ::"l"(rects_sorted + min(base + 64u + 16u * lane, end - 1u)));   // two chunks ahead
                unsigned int M = 0u;
                uint32_t vid = 0u;
                if (idx < end) { M = block_cover_mask(__ldg(rects_sorted + idx), wbx0, wby0) & alive_mask; vid = __ldg(vals + idx); }
                unsigned int m = __ballot_sync(FULL, M != 0u);
                const int rank = __popc(m & ((1u << lane) - 1u));
                int adv = 32;
                if (__popc(m) > 32 - cnt) {                            // more survivors than free slots: take the first ones
                    if (rank >= 32 - cnt) M = 0u;
                    m = __ballot_sync(FULL, M != 0u);
                    adv = 32 - __clz(m);                               // resume after the last survivor taken
                }
                if (M) {
                    const float4* rec = packed + 5 * (size_t)vid;
                    const int slot = half + cnt + rank;
                    cp_async16(&S.g0[slot], rec); cp_async16(&S.g1[slot], rec + 1); cp_async16(&S.r0[slot], rec + 2);
                    cp_async16(&S.r1[slot], rec + 3); cp_async16(&S.col[slot], rec + 4);
                    S.M[slot] = M;
                }
                if (STATS) { n_read += (idx < end && (int)lane < adv); n_surv += (M != 0u); }
                cnt += __popc(m);
                base += adv;
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            return cnt;
        };
        int head = 0, count = stage(0);
        while (count > 0) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
            const int count_next = stage(head ^ 32);       // in flight during the walk below
            // ---- walk up to 32 staged voxels, every lane through its own candidates ----
            const int n = count;
            unsigned int cand = transpose32(lane < n ? S.M[head + lane] : 0u, lane);
            if (!alive) cand = 0u;
            {
                // two loops: (1) every lane slab-tests its own candidates against a slightly dilated box (centre hi
                // parts only) and records the hits; (2) every lane integrates and composites its own hits. A lane that
                // misses no longer sits idle through another lane's K samples, and the hit loop is as long as the
                // pixel with the most HITS, not the most candidates.
                unsigned int hits = 0u;
                if (STATS) n_test += __popc(cand);
                while (__any_sync(FULL, cand != 0u)) {
                    if (cand) {
                        const int k = __ffs(cand) - 1;
                        cand &= cand - 1;
                        const float4 a = S.g0[(head + k) & (RING - 1)];
                        // dilated half edge (voxel_record_dev): a bound on what the lo parts and the rounding can move, so no
                        // true hit is lost
                        const float hd = S.col[(head + k) & (RING - 1)].w;
                        const float cx = a.x * ray.inv[0], cy = a.y * ray.inv[1], cz = a.z * ray.inv[2];
                        const float wx = hd * ray.ainv[0], wy = hd * ray.ainv[1], wz = hd * ray.ainv[2];
                        const float s0 = fmaxf(fmaxf(cx - wx, cy - wy), fmaxf(cz - wz, 0.f));
                        const float s1 = fminf(fminf(cx + wx, cy + wy), cz + wz);
                        if (s1 > s0) hits |= 1u << k;
                    }
                }
                if (REC) {
                    uint32_t* r = rec_out + (size_t)n_rec * TRAV_WORDS;
                    r[lane] = hits;
                    if (lane < n) r[32 + lane] = __float_as_uint(S.g1[(head + lane) & (RING - 1)].w);    // the staged voxel ids
                    if (lane == 0) r[64] = (uint32_t)n;
                    ++n_rec;
                }
                while (__any_sync(FULL, hits != 0u)) {
                    if (hits) {
                        const int slot = (head + __ffs(hits) - 1) & (RING - 1);
                        hits &= hits - 1;
                        const float4 a = S.g0[slot], bq = S.g1[slot];
                        float s0, s1, t_ref, D[3];
                        if (slab(ray, a, bq, s0, s1, t_ref, D)) {               // the precise test decides
                            const uint32_t vid = __float_as_uint(bq.w);
                            unsigned int wm_old = 0u;
                            if (w_max != nullptr) wm_old = w_max[vid];            // stale read is safe: w_max only grows
                            const float4 ra = S.r0[slot], rb = S.r1[slot], col = S.col[slot];
                            float dtau[8];
                            float tau = integrate<K, false>(ray, D, a.w, s0, s1, ra, rb, dtau);
                            float E = ex2f(-1.4426950408889634f * tau);
                            float w = T * (1.f - E);
                            T *= E;
                            C0 = fmaf(w, col.x, C0); C1 = fmaf(w, col.y, C1); C2 = fmaf(w, col.z, C2);
                            if (STATS) ++n_hit;
                            Dep = fmaf(w, t_ref + 0.5f * (s0 + s1), Dep);
                            if (w_max != nullptr && __float_as_uint(w) > wm_old) atomicMax(w_max + vid, __float_as_uint(w));
                            if (T < T_min) { alive = false; hits = 0u; }          // R8: stop after the voxel that crosses T_min
                        }
                    }
                }
            }
            __syncwarp();
            head ^= 32;
            count = count_next;
            alive_mask = __ballot_sync(FULL, alive);
            if (alive_mask == 0u) break;                              // whole warp terminated
        }
        asm volatile("cp.async.wait_all;" ::: "memory");            // nothing in flight when the ring is reused
        __syncwarp();
    }
    if (STATS) {
        unsigned int v4[4] = {n_hit, n_test, n_surv, n_read};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            unsigned int t = __reduce_add_sync(FULL, v4[i]);
            if (lane == 0 && t) atomicAdd(stats + i, (unsigned long long)t);
        }
    }
    if (REC && lane == 0) trav_count[tile * 8 + warp] = n_rec;
    if (inimg) {
        image[pix * 3] = fmaf(T, c.bg[0], C0);
        image[pix * 3 + 1] = fmaf(T, c.bg[1], C1);
        image[pix * 3 + 2] = fmaf(T, c.bg[2], C2);
        if (depth) depth[pix] = Dep;
        if (T_final) T_final[pix] = T;
    }
}


// ================================================================================================
// Hit-packed backward compositing (row a9). The lane-centric walk above keeps only ~12 of 32 lanes busy
// in the expensive part of the backward pass (K samples + exp + the monomial sums) and needs a quad
// exchange before every reduction. Here only the cheap part stays pixel-centric; the expensive part runs
// on a compacted hit queue:
//   1. cull + stage as above (32 voxel records in list order, warp-private);
//   2. test: every lane pops its own pixel's candidates among the staged voxels and slab-tests them
//      against a slightly dilated box (centre hi parts only, ray in registers), recording a hit bitmask;
//   3. queue: the 32x32 hit matrix is transposed so that lane k knows which pixels hit slot k; a warp scan
//      gives every slot its queue offset; every pixel lane then writes its own hits to their slot-major
//      positions (slot offset + its rank among the slot's pixels);
//   4. hit rounds: 32 hits per round, one per lane, all lanes busy in the precise slab test and the K
//      samples. The sequential per-pixel state (T, P = G . C) lives in shared memory; hits of the same
//      pixel inside a round (match_any) are chained in slot order by a short loop of shuffles, so every
//      pixel composites front to back in exactly the list order:
//          dL/dtau_k = G . (T_k c_k + C_k - C_final) = T_k (G . c_k) + P_k - G . C_final.
//   5. reduce: hits of one voxel are contiguous lanes, so two steps of a segmented shuffle sum give every
//      fragment of up to 4 consecutive hits of a voxel one set of three red.global.add.v4.f32: a voxel that
//      covers 7 of the warp's pixels leaves as 2 reduction sets instead of 7.
// With the traversal record the kernel is bound by the shared-memory pipe (loads of the per-pixel and per-slot data and
// the shuffles): the per-pixel data are 4-byte columns (32 pixels = 32 banks: any set of pixels loads in one
// conflict-free wavefront, 12 per hit round instead of ~24 for four 16-byte rows), and the per-pixel constant of dL/dtau is
// folded into the chained scalar P.
constexpr int QCAP = 512;          // queue entries per warp (a batch is cut so that its hits fit)
#ifndef SVR_RED_STEPS
#define SVR_RED_STEPS 3
#endif
constexpr int RED_STEPS = SVR_RED_STEPS;   // fragments of up to 2^RED_STEPS consecutive hits of one voxel share a reduction set
                                           // (C4 backward: 1 step 2.14 ms, 2 steps 1.66 ms, 3 steps 1.64 ms)
constexpr int NSLOT = 32;          // staged voxels per batch
#ifndef BWD_CTAS
#define BWD_CTAS 4
#endif

struct WarpWork {
    float4 g0[NSLOT];   // gh.xyz, h
    float4 g1[NSLOT];   // gl.xyz, voxel id bits
    float4 r0[NSLOT];   // log2(e) * (c0, cx, cy, cz)
    float4 r1[NSLOT];   // log2(e) * (cxy, cxz, cyz, cxyz)
    float4 col[NSLOT];  // r, g, b, cover mask M of this warp's 8x4 block
    float A[12][32];    // per pixel, 4-byte columns: 32 pixels = 32 banks, so a load of any set of pixels is one
                        // conflict-free wavefront: dh.xyz, dl.xyz, 1/dh.xyz, G.xyz (G = dL/dC)
    float T[32];        //   transmittance
    float Pp[32];       //   P = G . C (+ gD . D with the depth head) - G . C_final (- the heads' constants)
    float PD[32];       //   gD = dL/dDepth (kernels with HEADS only)
    uint2 Hs[32];       // per slot of the batch: pixels that hit it, queue offset
    unsigned short q[QCAP];
};

__device__ __forceinline__ int warp_incl_scan_i(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(FULL, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

template <int K, bool HEADS, bool REPLAY>
__global__ void __launch_bounds__(256, BWD_CTAS) backward_packed_kernel(CamDev c, const float4* __restrict__ packed, const uint32_t* __restrict__ vals,
                                                               const uint2* __restrict__ rects_sorted,
                                                               const uint32_t* __restrict__ ranges,
                                                               const uint32_t* __restrict__ tile_order, float T_min,
                                                               unsigned int* __restrict__ w_max, const float* __restrict__ dL,
                                                               const float* __restrict__ image_in, float* __restrict__ grad_coef,
                                                               float* __restrict__ grad_rgb, const float* __restrict__ dL_ddepth,
                                                               const float* __restrict__ dL_dT, const float* __restrict__ depth_in,
                                                               const float* __restrict__ T_in, const uint32_t* __restrict__ trav,
                                                               const uint32_t* __restrict__ trav_off, const uint32_t* __restrict__ trav_count) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    WarpWork& S = reinterpret_cast<WarpWork*>(smem_raw)[warp];
    const int tile = (int)tile_order[blockIdx.x];
    const int tile_x = tile % c.tiles_x, tile_y = tile / c.tiles_x;
    const int wbx0 = tile_x * SVR_TILE + (warp & 1) * 8, wby0 = tile_y * SVR_TILE + (warp >> 1) * 4;
    const int px = wbx0 + (lane & 7), py = wby0 + (lane >> 3);
    const bool inimg = px < c.W && py < c.H;
    const size_t pix = (size_t)py * c.W + px;
    const unsigned int lt = (1u << lane) - 1u;
    const int swl = lane;                                             // this pixel's row in the tables

    int oct = -1;
    float dh[3], inv[3], ainv[3];
    {
        RayF ray;
        float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
        float gdep = 0.f;
        if (inimg) {
            setup_ray(c, px, py, ray);
            oct = pixel_octant_dev(c, px, py);
            g = make_float4(dL[pix * 3], dL[pix * 3 + 1], dL[pix * 3 + 2], 0.f);
            g.w = g.x * image_in[pix * 3] + g.y * image_in[pix * 3 + 1] + g.z * image_in[pix * 3 + 2];
            if (HEADS) {
                // dL/dtau_k = T_k (G . c_k + gD t_k) + P_k - (G . C_final + gD D_final + gT T_K): the heads only add constants
                gdep = dL_ddepth ? dL_ddepth[pix] : 0.f;
                g.w += gdep * (depth_in ? depth_in[pix] : 0.f) + (dL_dT ? dL_dT[pix] * T_in[pix] : 0.f);
            }
        } else {
#pragma unroll
            for (int a = 0; a < 3; ++a) { ray.dh[a] = 0.f; ray.dl[a] = 0.f; ray.inv[a] = 0.f; ray.ainv[a] = 0.f; }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) { dh[a] = ray.dh[a]; inv[a] = ray.inv[a]; ainv[a] = ray.ainv[a]; }
#pragma unroll
        for (int a = 0; a < 3; ++a) { S.A[a][swl] = ray.dh[a]; S.A[3 + a][swl] = ray.dl[a]; S.A[6 + a][swl] = ray.inv[a]; }
        S.A[9][swl] = g.x; S.A[10][swl] = g.y; S.A[11][swl] = g.z;
        if (HEADS) S.PD[swl] = gdep;
        S.T[swl] = 1.f;
        S.Pp[swl] = -g.w;                        // the per-pixel constant of dL/dtau rides in P
    }
    __syncwarp();
    float Tpix = 1.f;
    // steps 3-5 for the staged slots [head, head + n); returns the number of slots consumed (a batch is cut where the
    // queue is full)
    auto run_batch = [&](const unsigned int hits, int n, const int head) -> int {
        // ---- 3. queue: slot-major positions from the transposed hit matrix ----
        int nh;
        {
            const unsigned int H = transpose32(hits, lane);         // lane k: pixels that hit slot k
            const int cnt = __popc(H);
            const int inc = warp_incl_scan_i(cnt, lane);
            n = min(n, __popc(__ballot_sync(FULL, inc <= QCAP)));  // cut the batch where the queue is full
            nh = __shfl_sync(FULL, inc, n - 1);
            S.Hs[lane] = make_uint2(H, (unsigned int)(inc - cnt));
            __syncwarp();
            unsigned int m = (n < 32) ? (hits & ((1u << n) - 1u)) : hits;
            while (__any_sync(FULL, m != 0u)) {
                if (m) {
                    const int k = __ffs(m) - 1;
                    m &= m - 1;
                    const uint2 hk = S.Hs[k];
                    S.q[hk.y + __popc(hk.x & lt)] = (unsigned short)((k << 5) | swl);
                }
            }
        }
        __syncwarp();
        // ---- 4. hit rounds: one hit per lane ----
        for (int r = 0; r < nh; r += 32) {
            const bool valid = r + lane < nh;
            const unsigned int e = valid ? (unsigned int)S.q[r + lane] : 0xFFFFu;
            const int k = (int)(e >> 5);                         // slot inside the batch (2047 = no entry)
            const int i = (int)(e & 31u);                        // swizzled pixel id
            const int slot = (head + k) & (NSLOT - 1);
            // hits of the same pixel inside this round are chained in slot (= lane) order; issued first so that
            // the match latency hides behind the samples
            const unsigned int peers = __match_any_sync(FULL, valid ? (unsigned int)i : 32u + (unsigned int)lane);
            // hits of one voxel are contiguous lanes (a run): RED_STEPS steps of a segmented sum towards lower lanes,
            // then every lane that starts a fragment of 2^RED_STEPS lanes of its run sends the fragment's sums
            const int kprev = __shfl_up_sync(FULL, k, 1);
            const unsigned int heads = __ballot_sync(FULL, lane == 0 || kprev != k);
            const unsigned int above = (heads >> lane) >> 1;
            const int rem = above ? __ffs(above) - 1 : 31 - lane;     // lanes after this one in its run
            const int run_pos = lane - (31 - __clz(heads & (lt | (1u << lane))));
            const bool frag_head = valid && (run_pos & ((1 << RED_STEPS) - 1)) == 0;
            const uint32_t vid = valid ? __float_as_uint(S.g1[slot].w) : 0u;
            // w_max only grows, so a stale guard read is safe; issued here so that its latency hides behind the samples
            unsigned int wm_old = 0xFFFFFFFFu;
            if (frag_head && w_max != nullptr) wm_old = w_max[vid];
            float tau = 0.f, dtau[8], gc = 0.f;
            float4 G = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int m = 0; m < 8; ++m) dtau[m] = 0.f;
            if (valid) {
                const float4 a = S.g0[slot], bq = S.g1[slot];
                RayF rr;
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                    rr.dh[ax] = S.A[ax][i]; rr.dl[ax] = S.A[3 + ax][i]; rr.inv[ax] = S.A[6 + ax][i];
                    rr.ainv[ax] = fabsf(rr.inv[ax]);
                }
                const float4 col = S.col[slot];
                G = make_float4(S.A[9][i], S.A[10][i], S.A[11][i], 0.f);
                gc = G.x * col.x + G.y * col.y + G.z * col.z;
                float s0, s1, t_ref, D[3];
                if (slab(rr, a, bq, s0, s1, t_ref, D)) {           // the precise test decides
                    const float4 ra = S.r0[slot], rb = S.r1[slot];
                    tau = integrate<K, true>(rr, D, a.w, s0, s1, ra, rb, dtau);
                    if (HEADS) gc = fmaf(S.PD[i], t_ref + 0.5f * (s0 + s1), gc);
                }
            }
            const float E = ex2f(-1.4426950408889634f * tau);
            const unsigned int lower = peers & lt;
            const int level = __popc(lower);
            const int pred = lower ? 31 - __clz(lower) : lane;
            const int maxL = (int)__reduce_max_sync(FULL, (unsigned int)level);
            float2 st = make_float2(0.f, 0.f);
            if (valid && level == 0) st = make_float2(S.T[i], S.Pp[i]);
            float w = 0.f;
            bool live = false;
            for (int L = 0; L <= maxL; ++L) {
                if (L > 0) {
                    const float t0 = __shfl_sync(FULL, st.x, pred), t1 = __shfl_sync(FULL, st.y, pred);
                    if (level == L) st = make_float2(t0, t1);
                }
                if (level == L) {
                    live = valid && st.x >= T_min;                // R8: a ray stops after the voxel that crosses T_min
                    w = live ? st.x * (1.f - E) : 0.f;
                    st.x = live ? st.x * E : st.x;
                    st.y = fmaf(w, gc, st.y);
                }
            }
            if (valid && (peers >> lane) == 1u) { S.T[i] = st.x; S.Pp[i] = st.y; }    // last hit of its pixel in this round
            // ---- 5. reduce ----
            float v[11];
            {
                const float dLdtau = live ? fmaf(st.x, gc, st.y) : 0.f;
#pragma unroll
                for (int m = 0; m < 8; ++m) v[m] = dLdtau * dtau[m];
                v[8] = w * G.x; v[9] = w * G.y; v[10] = w * G.z;
            }
            float wq = w;
#pragma unroll
            for (int s = 0; s < RED_STEPS; ++s) {
                const int step = 1 << s;
                const float take = (step <= rem) ? 1.f : 0.f;
#pragma unroll
                for (int m = 0; m < 11; ++m) v[m] = fmaf(take, __shfl_down_sync(FULL, v[m], step), v[m]);
                wq = fmaxf(wq, take * __shfl_down_sync(FULL, wq, step));
            }
            if (frag_head && wq > 0.f) {
                red_add_v4(grad_coef + (size_t)vid * 8, v[0], v[1], v[2], v[3]);
                red_add_v4(grad_coef + (size_t)vid * 8 + 4, v[4], v[5], v[6], v[7]);
                red_add_v4(grad_rgb + (size_t)vid * 4, v[8], v[9], v[10], 0.f);
                if (__float_as_uint(wq) > wm_old) atomicMax(w_max + vid, __float_as_uint(wq));
            }
            __syncwarp();                                          // pixel state is reused by the next round
        }
        return n;
    };

    if (REPLAY) {
        // The forward pass recorded, per batch, the list entries it staged and the slots every pixel hit: no cull, no test.
        const uint32_t r0 = trav_off[tile], cap = (trav_off[tile + 1] - r0) >> 3;
        const uint32_t* rec = trav + ((size_t)r0 + (size_t)warp * cap) * TRAV_WORDS;
        const uint32_t n_rec = trav_count[tile * 8 + warp];
        for (uint32_t rb = 0; rb < n_rec; ++rb, rec += TRAV_WORDS) {
            const int n = (int)__ldg(rec + 64);
            const unsigned int hits = __ldg(rec + lane);
            if (__ballot_sync(FULL, hits != 0u) == 0u) continue;       // nothing hit in this batch
            if (lane < n) {
                const float4* pr = packed + 5 * (size_t)__ldg(rec + 32 + lane);
                const float4 t0 = __ldg(pr), t1 = __ldg(pr + 1), t2 = __ldg(pr + 2), t3 = __ldg(pr + 3), t4 = __ldg(pr + 4);
                const uint32_t vid = __float_as_uint(t1.w);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(grad_coef + (size_t)vid * 8));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(grad_rgb + (size_t)vid * 4));
                S.g0[lane] = t0; S.g1[lane] = t1; S.r0[lane] = t2; S.r1[lane] = t3; S.col[lane] = t4;
            }
            __syncwarp();
            for (int k0 = 0; k0 < n;) k0 += run_batch(hits >> k0, n - k0, k0);
            __syncwarp();
        }
        return;
    }

    for (int so = 0; so < 8; ++so) {
        const uint32_t start = ranges[(tile * 8 + so) * 2], end = ranges[(tile * 8 + so) * 2 + 1];
        if (start == end) continue;
        bool alive = inimg && (oct == so) && (Tpix >= T_min);
        unsigned int alive_mask = __ballot_sync(FULL, alive);
        if (alive_mask == 0u) continue;                               // no pixel of this warp uses this list
        int head = 0, count = 0;                                      // ring state (warp-uniform)
        uint32_t base = start;
        while (true) {
            // ---- 1. cull + stage until 32 survivors are waiting or the list is exhausted ----
            while (count < NSLOT && base < end) {
                const uint32_t idx = base + lane;
                unsigned int M = 0u;
                uint32_t vid_e = 0u;
                if (idx < end) { M = block_cover_mask(__ldg(rects_sorted + idx), wbx0, wby0) & alive_mask; vid_e = __ldg(vals + idx); }
                unsigned int m = __ballot_sync(FULL, M != 0u);
                const int rank = __popc(m & lt);
                int adv = 32;
                if (__popc(m) > NSLOT - count) {                       // more survivors than free slots: take the first ones
                    if (rank >= NSLOT - count) M = 0u;
                    m = __ballot_sync(FULL, M != 0u);
                    adv = 32 - __clz(m);                               // resume after the last survivor taken
                }
                if (M) {
                    const float4* rec = packed + 5 * (size_t)vid_e;
                    const float4 t0 = __ldg(rec), t1 = __ldg(rec + 1), t2 = __ldg(rec + 2), t3 = __ldg(rec + 3);
                    float4 t4 = __ldg(rec + 4);
                    t4.w = __uint_as_float(M);
                    const int slot = (head + count + rank) & (NSLOT - 1);
                    const uint32_t vid = __float_as_uint(t1.w);
                    // pull the voxel's gradient lines into L2 now: a reduction that misses L2 waits for the DRAM fill
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(grad_coef + (size_t)vid * 8));
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(grad_rgb + (size_t)vid * 4));
                    S.g0[slot] = t0; S.g1[slot] = t1; S.r0[slot] = t2; S.r1[slot] = t3; S.col[slot] = t4;
                }
                count += __popc(m);
                base += adv;
            }
            if (count == 0) break;
            __syncwarp();
            // ---- 2. test: every lane walks its own pixel's candidates (conservative slab test) ----
            int n = count;
            unsigned int hits = 0u;
            {
                unsigned int cand = transpose32(lane < n ? __float_as_uint(S.col[(head + lane) & (NSLOT - 1)].w) : 0u, lane);
                if (!alive) cand = 0u;
                while (__any_sync(FULL, cand != 0u)) {
                    if (cand) {
                        const int k = __ffs(cand) - 1;
                        cand &= cand - 1;
                        const float4 a = S.g0[(head + k) & (NSLOT - 1)];
                        // box dilated by a bound on what the lo parts and the rounding can move: never loses a true hit
                        const float hd = fmaf(fabsf(a.x) + fabsf(a.y) + fabsf(a.z), 4.8e-7f, a.w * 1.000002f);
                        const float cx = a.x * inv[0], cy = a.y * inv[1], cz = a.z * inv[2];
                        const float wx = hd * ainv[0], wy = hd * ainv[1], wz = hd * ainv[2];
                        const float s0 = fmaxf(fmaxf(cx - wx, cy - wy), fmaxf(cz - wz, 0.f));
                        const float s1 = fminf(fminf(cx + wx, cy + wy), cz + wz);
                        if (s1 > s0) hits |= 1u << k;
                    }
                }
            }
            n = run_batch(hits, n, head);
            head = (head + n) & (NSLOT - 1);
            count -= n;
            Tpix = S.T[swl];
            alive = inimg && (oct == so) && (Tpix >= T_min);
            alive_mask = __ballot_sync(FULL, alive);
            if (alive_mask == 0u) break;                              // whole warp terminated
        }
    }
}

template <typename KernelT>
SvrStatus set_smem_once(SvrContext* ctx, KernelT kernel, size_t smem, bool* done) {
    if (!*done) {
        SVR_CUDA(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        *done = true;
    }
    return SVR_OK;
}

}  // namespace

SvrStatus launch_forward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, float* image, float* depth, float* T_final,
                         float* w_max, unsigned long long* stats, bool record) {
    if (f->n_tiles == 0) return SVR_OK;
    StageScope scope__(ctx, ST_FORWARD);
    const size_t smem = sizeof(WarpStage) * WARPS;
    const uint2* rs = reinterpret_cast<const uint2*>(f->rects_sorted);
    const float4* pk = reinterpret_cast<const float4*>(f->packed);
    unsigned int* wm = reinterpret_cast<unsigned int*>(w_max);
    const bool rec = record && f->trav != nullptr;
#define SVR_FWD_GO(KK, SS, RR)                                                                                       \
    do {                                                                                                             \
        static bool done = false;                                                                                    \
        SVR_TRY(set_smem_once(ctx, composite_kernel<KK, SS, RR>, smem, &done));                                      \
        composite_kernel<KK, SS, RR><<<f->n_tiles, 256, smem, ctx->stream>>>(f->cam, pk, f->vals, rs, f->ranges, f->tile_order, T_min, image, depth, \
                                                                             T_final, wm, stats, f->trav, f->trav_off, f->trav_count);       \
    } while (0)
#define SVR_FWD(KK)                                                                                                  \
    do {                                                                                                             \
        if (stats) SVR_FWD_GO(KK, true, false);                                                                      \
        else if (rec) SVR_FWD_GO(KK, false, true);                                                                   \
        else SVR_FWD_GO(KK, false, false);                                                                           \
    } while (0)
    switch (K) {
        case 1: SVR_FWD(1); break;
        case 2: SVR_FWD(2); break;
        case 3: SVR_FWD(3); break;
        case 4: SVR_FWD(4); break;
        default: return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    }
#undef SVR_FWD
#undef SVR_FWD_GO
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_backward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, const float* dL, const float* image,
                          float* grad_coef, float* grad_rgb, float* w_max, const float* dL_ddepth, const float* dL_dT,
                          const float* depth, const float* T_final) {
    if (f->n_tiles == 0) return SVR_OK;
    StageScope scope__(ctx, ST_BACKWARD);
    const size_t smem = sizeof(WarpWork) * WARPS;
    const uint2* rs = reinterpret_cast<const uint2*>(f->rects_sorted);
    const float4* pk = reinterpret_cast<const float4*>(f->packed);
    unsigned int* wm = reinterpret_cast<unsigned int*>(w_max);
    // replay the forward pass's traversal record when there is one for this termination threshold
    const bool replay = f->trav != nullptr && f->trav_valid && f->trav_T_min == T_min && (ctx->debug_flags & 16) == 0;
    const bool heads = dL_ddepth != nullptr || dL_dT != nullptr;
#define SVR_BWD_GO(KK, HH, RR)                                                                                       \
    do {                                                                                                             \
        static bool done = false;                                                                                    \
        SVR_TRY(set_smem_once(ctx, backward_packed_kernel<KK, HH, RR>, smem, &done));                                \
        backward_packed_kernel<KK, HH, RR><<<f->n_tiles, 256, smem, ctx->stream>>>(                                  \
            f->cam, pk, f->vals, rs, f->ranges, f->tile_order, T_min, wm, dL, image, grad_coef, grad_rgb, dL_ddepth, dL_dT, depth, T_final,         \
            f->trav, f->trav_off, f->trav_count);                                                                    \
    } while (0)
#define SVR_BWD(KK)                                                                                                  \
    do {                                                                                                             \
        if (heads && replay) SVR_BWD_GO(KK, true, true);                                                             \
        else if (heads) SVR_BWD_GO(KK, true, false);                                                                 \
        else if (replay) SVR_BWD_GO(KK, false, true);                                                                \
        else SVR_BWD_GO(KK, false, false);                                                                           \
    } while (0)
    switch (K) {
        case 1: SVR_BWD(1); break;
        case 2: SVR_BWD(2); break;
        case 3: SVR_BWD(3); break;
        case 4: SVR_BWD(4); break;
        default: return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "K must be 1..4");
    }
#undef SVR_BWD
#undef SVR_BWD_GO
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// per-voxel view records (needs rects + rgbm; independent of the lists)
SvrStatus launch_voxel_records(SvrContext* ctx, SvrFrame* f) {
    StageScope scope__(ctx, ST_PACK);
    if (f->scene.n > 0) {
        voxel_record_kernel<<<(unsigned int)((f->scene.n + 255) / 256), 256, 0, ctx->stream>>>(
            f->scene, f->cam, reinterpret_cast<const ushort4*>(f->rects), reinterpret_cast<const float4*>(f->rgbm),
            reinterpret_cast<float4*>(f->packed));
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// rectangles in list order (a separate pass: gathering inside the per-bucket sort's output loop cost 0.12 ms, this 0.04)
SvrStatus launch_gather_rects(SvrContext* ctx, SvrFrame* f) {
    StageScope scope__(ctx, ST_PACK);
    if (f->n_entries > 0) {
        gather_rects_kernel<<<(unsigned int)((f->n_entries + 255) / 256), 256, 0, ctx->stream>>>(
            f->vals, f->n_entries, reinterpret_cast<const uint2*>(f->rects), reinterpret_cast<uint2*>(f->rects_sorted));
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}
