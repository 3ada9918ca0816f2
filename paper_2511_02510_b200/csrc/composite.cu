// Stage (3) forward compositing and stage (4) backward compositing (DESIGN.md rows a7, a9).
//
// One CTA per 16x16 tile; each of its 8 warps owns an 8x4 pixel block and runs independently (no CTA
// barrier anywhere): a barrier per staged chunk cost 37% of the issue slots in the first version
// (profiles/r1a_*), because the 8 blocks of a tile see very different numbers of voxels.
//
// Both kernels walk the tile's sorted (tile, octant) lists in BATCHES of up to 32 voxels that survive the
// cull against the warp's pixel block:
//   1. cull: 32 entries at a time, lane i reads entry i's TIGHT pixel rectangle (the pixels whose centre can see the voxel;
//      in list order, so the read is coalesced, two chunks ahead in registers) and computes the 32-bit mask M of this
//      warp's pixels it covers. M == 0 => skipped.
//   2. stage: surviving lanes copy their voxel's 80-byte view record (voxel_record_dev, svr_internal.cuh),
//      gathered by the voxel id read beside the rectangle, in list order, into warp-private shared memory (cp.async,
//      double-buffered).
//   3. test (pixel-major): the 32x32 bit matrix M[slot][pixel] is transposed with 5 shuffles, so every lane holds the
//      slots that cover ITS pixel; it pops them and slab-tests them against a slightly dilated box -> hit bitmask.
// Forward (composite_kernel):
//   4. every lane pops its own hits front to back: precise slab test, K samples, eqs. 2-4, depth, w_max (eq. 5).
//      With REC it writes the traversal record: per batch the staged voxel ids, every pixel's hit mask, and E = exp(-tau)
//      of every hit in pixel-major rows (row i = every pixel's i-th hit of the batch).
// Backward (backward_packed_kernel) replays the record (or culls and tests itself) and splits a batch into a part that is
// sequential per PIXEL but cheap and a part that is parallel over ray-voxel HITS (all 32 lanes busy whatever the shape of
// the voxels):
//   4'. queue layout: the hit matrix is transposed back (lane k: pixels that hit slot k), a warp scan gives every slot its
//      offset: the hits form a slot-major queue of nh entries; entry e is worked on by lane e / C as its (e % C)-th item,
//      C = ceil(nh / 32), per-entry arrays are indexed by st(e) = row e % C, column (e / C + e % C) mod 32: a lane's
//      accesses are conflict-free and its C entries are CONSECUTIVE hits, i.e. mostly hits of one voxel.
//   5'. pixel-major chain: with E from the record (or recomputed by a hit-major sweep), every lane chains its own hits:
//      T_k, P_k = G . C_k and from them dL/dtau_k = T_k (G . c_k) + P_k - G . C_final and w_k, into the queue.
//   6'. hit-major: precise slab + K samples per entry with dL/dtau_k already known, so the gradient of the 8 density
//      coefficients and the colour is accumulated IN REGISTERS over the lane's consecutive entries and leaves as one set of
//      three red.global.add.v4.f32 into the voxel's 64-byte scratch row per (lane, voxel) fragment: no cross-lane reduction.
//      (Round 1 reduced 11 values per hit with a segmented shuffle sum and chained the pixel state through shuffles: 45 % of
//      its instructions, profiles/r1q_*. The same split was tried for the forward pass and lost: profiles/r2b_*.)
//
// Density: the trilinear raw density is staged as polynomial coefficients (c0, cx, cy, cz, cxy, cxz, cyz,
// cxyz), pre-multiplied by log2(e), so a sample costs 7 FMA + one EX2 instead of 7 lerps (14 ops) + MUL + EX2.
// Backward accumulates the gradient w.r.t. those coefficients (monomials 1, qx, qy, qz, qxqy, ...) into a
// per-voxel scratch with 16-byte vector reductions (float atomics in shared memory are CAS loops on sm_100a, so
// nothing is accumulated there); the per-voxel finalize kernel (preprocess.cu) maps it back to the 8 corners.
//
// Precision: the ray is set up in fp64 per pixel and kept as hi+lo floats; the slab test runs in
// coordinates relative to the ray's closest approach to the voxel centre, so the segment length keeps
// ~1e-7 relative accuracy even for 4e-3-wide voxels 2.5 units away (a plain fp32 t_out - t_in loses 1e-4).
#include "svr_internal.cuh"

namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int TRAV_WORDS = SVR_TRAV_WORDS;   // words of one traversal record (forward -> backward), see composite_kernel
constexpr int NSLOT = 32;          // staged voxels per batch
constexpr int QCAP = 256;          // queue entries per warp (a batch is cut into sub-batches whose hits fit)
static_assert(QCAP >= 64 && QCAP <= 512 && QCAP % 32 == 0, "queue entries per lane C = QCAP / 32 <= 16 (QINV); a slot has at most 32 hits");
constexpr int RING = 64;           // forward staging slots per warp (two halves of 32)
// Launch configuration (measured alternatives: DESIGN.md section 6). The eight warps of a tile are independent (no CTA barrier),
// so a tile may span several CTAs.
#define FWD_CTAW 4                                      // forward: warps per CTA
#define FWD_MINB 8                                      // forward: CTAs per SM (63 registers)
#define BWD_CTAW 4                                      // replaying backward: warps per CTA
#define BWD_CW(REPLAY) ((REPLAY) ? BWD_CTAW : 8)        // the self-walking fallback keeps whole tiles (4 is 6 % slower there)
#define BWD_MINB(REPLAY) ((REPLAY) ? 5 : 3)             // replay: 5 x 4 warps, 94 registers (6 x 4 at 80 registers: 3 % slower)
constexpr int BWD_BUFS = 2;        // replaying backward: the gather of the next batch is double-buffered
constexpr int EROWS = 8;           // E rows a backward lane fetches into registers at the start of a sub-batch
constexpr uint32_t ECHUNK = 16;    // the E record is handed out to warps in chunks of (at least) 16 rows of 32 floats

// ceil(65536 / C): (pos * QINV[C]) >> 16 == pos / C for pos < 512, C <= 16
__constant__ unsigned int QINV[17] = {0, 65536, 32768, 21846, 16384, 13108, 10923, 9363, 8192, 7282, 6554, 5958, 5462, 5042, 4682, 4370, 4096};

struct WarpQ {              // hit queue of one sub-batch; per-entry arrays indexed by st(e)
    uint2 Hs[32];           // per slot: pixels that hit it, queue offset
    float2 WD[QCAP];        // x: exp(-tau) from the hit-major sweep, replaced by the blending weight w; y: dL/dtau
    unsigned short q[QCAP]; // (slot << 5) | pixel
};

struct QLayout { int n, nh, C; unsigned int inv; };

// entry e = le * C + c lives at row c, column (le + c) mod 32: the C consecutive entries of a lane sit in different banks
// (the pixel-major passes write runs of consecutive entries), and a row read by the 32 lanes is a permutation of the banks
__device__ __forceinline__ int q_st(int pos, const QLayout& L) {
    const int le = (int)(((unsigned int)pos * L.inv) >> 16);
    const int c = pos - le * L.C;
    return (c << 5) + ((le + c) & 31);
}
__device__ __forceinline__ int q_row(int c, int lane) { return (c << 5) + ((lane + c) & 31); }

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

__device__ __forceinline__ int warp_incl_scan_i(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(FULL, v, o);
        if (lane >= o) v += t;
    }
    return v;
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

// K midpoint samples (R5). ca/cb = polynomial coefficients * log2(e). Returns tau.
template <int K>
__device__ __forceinline__ float integrate(const RayF& r, const float* D, float h, float s0, float s1, const float4& ca,
                                           const float4& cb) {
    float inv_e = __int_as_float(0x7E800000 - __float_as_int(h));   // 0.5 / h for h a power of two
    float dt = (s1 - s0) * (1.0f / (float)K);
    float sum = 0.f;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float s = fmaf((float)j + 0.5f, dt, s0);
        float qx = __saturatef(fmaf(fmaf(s, r.dh[0], -D[0]), inv_e, 0.5f));
        float qy = __saturatef(fmaf(fmaf(s, r.dh[1], -D[1]), inv_e, 0.5f));
        float qz = __saturatef(fmaf(fmaf(s, r.dh[2], -D[2]), inv_e, 0.5f));
        float hi = fmaf(fmaf(cb.w, qz, cb.x), qy, fmaf(cb.y, qz, ca.y));     // (cxyz qz + cxy) qy + (cxz qz + cx)
        float lo = fmaf(fmaf(cb.z, qz, ca.z), qy, fmaf(ca.w, qz, ca.x));     // (cyz qz + cy) qy + (cz qz + c0)
        sum += ex2f(fmaf(hi, qx, lo));
    }
    return dt * sum;
}

// Same samples with dL/dtau known: acc[m] += dL/dtau * d tau / d coef_m (natural-scale coefficients), m over the monomials
// 1, qx, qy, qz, qxqy, qxqz, qyqz, qxqyqz.
template <int K>
__device__ __forceinline__ void integrate_bwd(const RayF& r, const float* D, float h, float s0, float s1, const float4& ca,
                                              const float4& cb, float dLdtau, float* acc) {
    float inv_e = __int_as_float(0x7E800000 - __float_as_int(h));
    float dt = (s1 - s0) * (1.0f / (float)K);
    const float sc = dLdtau * dt;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float s = fmaf((float)j + 0.5f, dt, s0);
        float qx = __saturatef(fmaf(fmaf(s, r.dh[0], -D[0]), inv_e, 0.5f));
        float qy = __saturatef(fmaf(fmaf(s, r.dh[1], -D[1]), inv_e, 0.5f));
        float qz = __saturatef(fmaf(fmaf(s, r.dh[2], -D[2]), inv_e, 0.5f));
        float hi = fmaf(fmaf(cb.w, qz, cb.x), qy, fmaf(cb.y, qz, ca.y));
        float lo = fmaf(fmaf(cb.z, qz, ca.z), qy, fmaf(ca.w, qz, ca.x));
        const float sig = ex2f(fmaf(hi, qx, lo)) * sc;
        const float sx = sig * qx, sy = sig * qy;
        acc[0] += sig;
        acc[1] += sx;
        acc[2] += sy;
        acc[3] = fmaf(sig, qz, acc[3]);
        const float sxy = sx * qy;
        acc[4] += sxy;
        acc[5] = fmaf(sx, qz, acc[5]);
        acc[6] = fmaf(sy, qz, acc[6]);
        acc[7] = fmaf(sxy, qz, acc[7]);
    }
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned int d = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// ---- step 4: queue layout of the sub-batch that starts at the first of `n` slots; hits = this pixel's hit bits over them ----
__device__ __forceinline__ QLayout queue_layout(unsigned int hits, int n, WarpQ& Q, int lane) {
    QLayout L;
    const unsigned int H = transpose32(hits, lane);         // lane k: pixels that hit slot k
    const int cnt = __popc(H);
    const int inc = warp_incl_scan_i(cnt, lane);
    L.n = min(n, __popc(__ballot_sync(FULL, inc <= QCAP)));  // cut where the queue is full (a slot has <= 32 hits: n >= 1)
    L.nh = __shfl_sync(FULL, inc, L.n - 1);
    L.C = (L.nh + 31) >> 5;
    L.inv = QINV[L.C];
    Q.Hs[lane] = make_uint2(H, (unsigned int)(inc - cnt));
    return L;
}

// every pixel lane writes its own hits to their slot-major queue positions
__device__ __forceinline__ void queue_fill(unsigned int m, WarpQ& Q, const QLayout& L, int lane) {
    const unsigned int lt = (1u << lane) - 1u;
    while (__any_sync(FULL, m != 0u)) {
        if (m) {
            const int k = __ffs(m) - 1;
            m &= m - 1;
            const uint2 hk = Q.Hs[k];
            Q.q[q_st((int)hk.y + __popc(hk.x & lt), L)] = (unsigned short)((k << 5) | lane);
        }
    }
}

// ---- hit-major sweep: precise slab + K samples per queue entry -> Q.E = exp(-tau) (1 for a miss), tm_out = t_mid (0 for a miss).
// g0..r1 point at the first slot of the sub-batch; A = per-pixel columns dh.xyz, dl.xyz, 1/dh.xyz. A lane's C entries are
// consecutive hits, mostly of one voxel: its record stays in registers until the slot changes.
template <int K, bool WANT_TM>
__device__ __forceinline__ void sweep_E(const float4* g0, const float4* g1, const float4* r0, const float4* r1,
                                        const float (*A)[32], WarpQ& Q, const QLayout& L, float* tm_out, int lane) {
    int cur = -1;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), bq = a, ra = a, rb = a;
    for (int c = 0; c < L.C; ++c) {
        if (lane * L.C + c < L.nh) {
            const int st = q_row(c, lane);
            const unsigned int u = Q.q[st];
            const int k = (int)(u >> 5), i = (int)(u & 31u);
            if (k != cur) { a = g0[k]; bq = g1[k]; ra = r0[k]; rb = r1[k]; cur = k; }
            RayF rr;
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
                rr.dh[ax] = A[ax][i]; rr.dl[ax] = A[3 + ax][i]; rr.inv[ax] = A[6 + ax][i];
                rr.ainv[ax] = fabsf(rr.inv[ax]);
            }
            float s0, s1, t_ref, D[3], E = 1.f, tm = 0.f;
            if (slab(rr, a, bq, s0, s1, t_ref, D)) {                 // the precise test decides
                const float tau = integrate<K>(rr, D, a.w, s0, s1, ra, rb);
                E = ex2f(-1.4426950408889634f * tau);
                tm = t_ref + 0.5f * (s0 + s1);
            }
            Q.WD[st].x = E;
            if (WANT_TM) tm_out[st] = tm;
        }
    }
}

// conservative slab test of this pixel's candidates among the staged slots (centre hi parts only, dilated half edge hd:
// a bound on what the lo parts and the rounding can move, so no true hit is lost; the precise test decides later)
template <bool HD_IN_COL>
__device__ __forceinline__ unsigned int test_candidates(unsigned int cand, const float4* g0, const float4* col, const float* inv,
                                                        unsigned int& n_test) {
    unsigned int hits = 0u;
    while (__any_sync(FULL, cand != 0u)) {
        if (cand) {
            const int k = __ffs(cand) - 1;
            cand &= cand - 1;
            const float4 a = g0[k];
            const float hd = HD_IN_COL ? col[k].w : fmaf(fabsf(a.x) + fabsf(a.y) + fabsf(a.z), 4.8e-7f, a.w * 1.000002f);
            const float cx = a.x * inv[0], cy = a.y * inv[1], cz = a.z * inv[2];
            const float wx = hd * fabsf(inv[0]), wy = hd * fabsf(inv[1]), wz = hd * fabsf(inv[2]);
            const float s0 = fmaxf(fmaxf(cx - wx, cy - wy), fmaxf(cz - wz, 0.f));
            const float s1 = fminf(fminf(cx + wx, cy + wy), cz + wz);
            if (s1 > s0) hits |= 1u << k;
            ++n_test;
        }
    }
    return hits;
}

// The list entries of one 32-entry chunk, one per lane (rectangle + voxel id); beyond the list: an empty rectangle.
struct Chunk { uint2 rc; uint32_t vid; };
__device__ __forceinline__ Chunk load_chunk(const uint2* __restrict__ rects_sorted, const uint32_t* __restrict__ vals, uint32_t b, uint32_t end,
                                            int lane) {
    Chunk c;
    c.rc = make_uint2(0xFFFFFFFFu, 0u);
    c.vid = 0u;
    const uint32_t idx = b + (uint32_t)lane;
    if (idx < end) { c.rc = __ldg(rects_sorted + idx); c.vid = __ldg(vals + idx); }
    return c;
}

struct FwdWarp {
    float4 g0[RING];    // gh.xyz, h (half edge)
    float4 g1[RING];    // gl.xyz, voxel id bits
    float4 r0[RING];    // log2(e) * (c0, cx, cy, cz)
    float4 r1[RING];    // log2(e) * (cxy, cxz, cyz, cxyz)
    float4 col[RING];   // r, g, b, dilated half edge
    unsigned int M[RING];   // pixels of this warp's 8x4 block covered by the voxel's rectangle
};

// Forward (a7). After the test every lane pops its own HITS front to back: precise slab, K samples, eqs. 2-4, depth,
// w_max (eq. 5) by atomicMax guarded by a plain read. (The hit-major split of the backward pass was tried here too:
// the queue, its fill and the second pixel-major loop cost more instructions than the idle lanes of this loop,
// profiles/r2b_*.) Traversal record of one batch (TRAV_WORDS words, written with REC): [0,32) every pixel's hit mask, [32,64)
// the staged voxel ids, [64] the slot count, [65] the first E row of the batch in the E record, [71] its number of rows; E
// row i holds, for every pixel of the block, exp(-tau) of its i-th hit in the batch (1 where it has none or missed).
template <int K, bool STATS, bool REC, bool WMAX>
__global__ void __launch_bounds__(32 * FWD_CTAW, FWD_MINB) composite_kernel(CamDev c, const float4* __restrict__ packed, const uint32_t* __restrict__ vals,
                                                        const uint2* __restrict__ rects_sorted,
                                                        const uint32_t* __restrict__ ranges,
                                                        const uint32_t* __restrict__ tile_order,
                                                        float T_min,
                                                        float* __restrict__ image, float* __restrict__ depth,
                                                        float* __restrict__ T_final, unsigned int* __restrict__ w_max,
                                                        unsigned long long* __restrict__ stats, uint32_t* __restrict__ trav,
                                                        const uint32_t* __restrict__ trav_off, uint32_t* __restrict__ trav_count,
                                                        float* __restrict__ trav_E, uint32_t* __restrict__ trav_ectl, uint32_t e_cap) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = (int)(blockIdx.x % (8 / FWD_CTAW)) * FWD_CTAW + (tid >> 5);      // warp of the tile: 0..7
    FwdWarp& S = reinterpret_cast<FwdWarp*>(smem_raw)[tid >> 5];
    const int tile = (int)tile_order[blockIdx.x / (8 / FWD_CTAW)];
    const int tile_x = tile % c.tiles_x, tile_y = tile / c.tiles_x;
    const int wbx0 = tile_x * SVR_TILE + (warp & 1) * 8, wby0 = tile_y * SVR_TILE + (warp >> 1) * 4;
    const int px = wbx0 + (lane & 7), py = wby0 + (lane >> 3);
    const bool inimg = px < c.W && py < c.H;
    const size_t pix = (size_t)py * c.W + px;
    const unsigned int lt = (1u << lane) - 1u;

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
    uint32_t* rec_out = nullptr;
    uint32_t n_rec = 0, e_pos = 0, e_left = 0;
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
        // Staging: double-buffered (the ring is two halves of 32 slots: while one half is walked, the records of the next
        // batch are already on their way into the other half; cp.async: no registers held, no stall on the load). The list
        // itself (rectangle + voxel id per entry) is read two chunks of 32 entries ahead into registers, so the cull does not
        // wait for it.
        uint32_t base = start;
        Chunk ca = load_chunk(rects_sorted, vals, base, end, lane), cb = load_chunk(rects_sorted, vals, base + 32u, end, lane);
        auto stage = [&](int half) -> int {
            int cnt = 0;
            while (cnt < 32 && base < end) {
                unsigned int M = block_cover_mask(ca.rc, wbx0, wby0) & alive_mask;
                const uint32_t vid = ca.vid;
                unsigned int m = __ballot_sync(FULL, M != 0u);
                const int rank = __popc(m & lt);
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
                if (STATS) { n_read += (base + lane < end && (int)lane < adv); n_surv += (M != 0u); }
                cnt += __popc(m);
                base += adv;
                if (adv == 32) ca = cb;
                else ca = load_chunk(rects_sorted, vals, base, end, lane);
                cb = load_chunk(rects_sorted, vals, base + 32u, end, lane);
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
            // two loops: (1) every lane slab-tests its own candidates against a slightly dilated box (centre hi parts only)
            // and records the hits; (2) every lane integrates and composites its own hits. A lane that misses does not sit
            // idle through another lane's K samples, and the hit loop is as long as the pixel with the most HITS.
            unsigned int hits = test_candidates<true>(cand, S.g0 + head, S.col + head, ray.inv, n_test);
            uint32_t eoff = 0xFFFFFFFFu;                                  // this lane's word in the E record (none: no room / no hits)
            if (REC && __any_sync(FULL, hits != 0u)) {
                // capacity of this warp's slice of the record (launch_traversal_offsets sizes it as ceil(len / 32) + 9 per list
                // set; re-read here rather than kept in a register). Writing past it would corrupt the next warp's records or
                // the heap, silently: stop the kernel instead (no sanitizer run covers this path on the target machines).
                if (n_rec >= ((trav_off[tile + 1] - trav_off[tile]) >> 3)) __trap();
                uint32_t* r = rec_out + (size_t)n_rec * TRAV_WORDS;
                r[lane] = hits;
                if (lane < n) r[32 + lane] = __float_as_uint(S.g1[head + lane].w);    // the staged voxel ids
                const uint32_t rows = __reduce_max_sync(FULL, (unsigned int)__popc(hits));
                if (e_left < rows) {                                   // next chunk of the E record
                    const uint32_t grab = rows > ECHUNK ? rows : ECHUNK;
                    if (lane == 0) e_pos = atomicAdd(trav_ectl, grab);
                    e_pos = __shfl_sync(FULL, e_pos, 0);
                    e_left = grab;
                }
                if (e_pos + rows <= e_cap) eoff = e_pos * 32u + lane;     // (e_cap < 2^27 rows: the offset fits 32 bits)
                else if (lane == 0) trav_ectl[1] = 1u;                  // E record full: the backward pass recomputes E
                if (lane == 0) { r[64] = (uint32_t)n; r[65] = e_pos; r[71] = rows; }
                e_pos += rows;
                e_left -= rows;
                ++n_rec;
            }
            while (__any_sync(FULL, hits != 0u)) {
                float E = 1.f;
                if (hits) {
                    const int slot = head + __ffs(hits) - 1;
                    hits &= hits - 1;
                    const float4 a = S.g0[slot], bq = S.g1[slot];
                    float s0, s1, t_ref, D[3];
                    if (slab(ray, a, bq, s0, s1, t_ref, D)) {               // the precise test decides
                        const uint32_t vid = __float_as_uint(bq.w);
                        unsigned int wm_old = 0u;
                        if (WMAX) wm_old = w_max[vid];                        // stale read is safe: w_max only grows
                        const float4 ra = S.r0[slot], rb = S.r1[slot], col = S.col[slot];
                        const float tau = integrate<K>(ray, D, a.w, s0, s1, ra, rb);
                        E = ex2f(-1.4426950408889634f * tau);
                        const float w = T * (1.f - E);
                        T *= E;
                        C0 = fmaf(w, col.x, C0); C1 = fmaf(w, col.y, C1); C2 = fmaf(w, col.z, C2);
                        if (STATS) ++n_hit;
                        Dep = fmaf(w, t_ref + 0.5f * (s0 + s1), Dep);
                        if (WMAX && __float_as_uint(w) > wm_old) atomicMax(w_max + vid, __float_as_uint(w));
                        if (T < T_min) { alive = false; hits = 0u; }          // R8: stop after the voxel that crosses T_min
                    }
                }
                if (REC && eoff != 0xFFFFFFFFu) { trav_E[eoff] = E; eoff += 32u; }   // a whole row per step: no partial sectors
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
// Backward compositing (row a9): see the file comment, steps 5'. REPLAY: the forward pass recorded the batches (no cull, no
// test); if it also recorded every hit's E = exp(-tau) (and the kernel has no depth head, whose chain needs t_mid too), the
// hit-major E sweep is skipped as well. The record is a stream known in advance: the header of batch b + 2 is loaded into
// registers and the voxel records of batch b + 1 are gathered (cp.async) into the other half of the staging buffer while
// batch b is worked on.
struct BwdBase {
    float4 g0[BWD_BUFS * NSLOT];   // gh.xyz, h                            (two halves: replay double-buffers the gather)
    float4 g1[BWD_BUFS * NSLOT];   // gl.xyz, voxel id bits
    float4 r0[BWD_BUFS * NSLOT];   // log2(e) * (c0, cx, cy, cz)
    float4 r1[BWD_BUFS * NSLOT];   // log2(e) * (cxy, cxz, cyz, cxyz)
    float4 col[BWD_BUFS * NSLOT];  // r, g, b, cover mask M of this warp's 8x4 block (non-replay) / dilated half edge
    float A[12][32];        // per pixel, 4-byte columns: dh.xyz, dl.xyz, 1/dh.xyz, G.xyz (G = dL/dC)
    WarpQ Q;
};
template <bool HEADS> struct BwdWarp : BwdBase {};
template <> struct BwdWarp<true> : BwdBase { float TM[QCAP]; };   // t_mid per queue entry (depth head)

template <int K, bool HEADS, bool REPLAY>
__global__ void __launch_bounds__(32 * BWD_CW(REPLAY), BWD_MINB(REPLAY)) backward_packed_kernel(CamDev c, const float4* __restrict__ packed, const uint32_t* __restrict__ vals,
                                                               const uint2* __restrict__ rects_sorted,
                                                               const uint32_t* __restrict__ ranges,
                                                               const uint32_t* __restrict__ tile_order, float T_min,
                                                               const bool want_wmax, const float* __restrict__ dL,
                                                               const float* __restrict__ image_in, float* __restrict__ grow,
                                                               const float* __restrict__ dL_ddepth,
                                                               const float* __restrict__ dL_dT, const float* __restrict__ depth_in,
                                                               const float* __restrict__ T_in, const uint32_t* __restrict__ trav,
                                                               const uint32_t* __restrict__ trav_off, const uint32_t* __restrict__ trav_count,
                                                               const float* __restrict__ trav_E, const uint32_t* __restrict__ trav_ectl) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31;
    constexpr int CW = BWD_CW(REPLAY);
    const int warp = (int)(blockIdx.x % (8 / CW)) * CW + (tid >> 5);                  // warp of the tile: 0..7
    BwdWarp<HEADS>& S = reinterpret_cast<BwdWarp<HEADS>*>(smem_raw)[tid >> 5];
    const int tile = (int)tile_order[blockIdx.x / (8 / CW)];
    const int tile_x = tile % c.tiles_x, tile_y = tile / c.tiles_x;
    const int wbx0 = tile_x * SVR_TILE + (warp & 1) * 8, wby0 = tile_y * SVR_TILE + (warp >> 1) * 4;
    const int px = wbx0 + (lane & 7), py = wby0 + (lane >> 3);
    const bool inimg = px < c.W && py < c.H;
    const size_t pix = (size_t)py * c.W + px;
    const unsigned int lt = (1u << lane) - 1u;

    int oct = -1;
    float inv[3];
    float4 G = make_float4(0.f, 0.f, 0.f, 0.f);
    float gdep = 0.f;
    {
        RayF ray;
        if (inimg) {
            setup_ray(c, px, py, ray);
            oct = pixel_octant_dev(c, px, py);
            G = make_float4(dL[pix * 3], dL[pix * 3 + 1], dL[pix * 3 + 2], 0.f);
            G.w = G.x * image_in[pix * 3] + G.y * image_in[pix * 3 + 1] + G.z * image_in[pix * 3 + 2];
            if (HEADS) {
                // dL/dtau_k = T_k (G . c_k + gD t_k) + P_k - (G . C_final + gD D_final + gT T_K): the heads only add constants
                gdep = dL_ddepth ? dL_ddepth[pix] : 0.f;
                G.w += gdep * (depth_in ? depth_in[pix] : 0.f) + (dL_dT ? dL_dT[pix] * T_in[pix] : 0.f);
            }
        } else {
#pragma unroll
            for (int a = 0; a < 3; ++a) { ray.dh[a] = 0.f; ray.dl[a] = 0.f; ray.inv[a] = 0.f; ray.ainv[a] = 0.f; }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) { inv[a] = ray.inv[a]; S.A[a][lane] = ray.dh[a]; S.A[3 + a][lane] = ray.dl[a]; S.A[6 + a][lane] = ray.inv[a]; }
        S.A[9][lane] = G.x; S.A[10][lane] = G.y; S.A[11][lane] = G.z;
    }
    __syncwarp();
    // per-pixel chain state, in this pixel's lane: transmittance and P = G . C (+ gD . D) - the per-pixel constant of dL/dtau
    float T = 1.f, P = -G.w;
    const bool haveE = REPLAY && !HEADS && trav_E != nullptr && trav_ectl[1] == 0u;

    // steps 4-5' for the n slots staged at `buf`; hits = this pixel's hit bits; misc = the record's words 64.. (lane i: word 64 + i)
    auto run_batch = [&](const int buf, const unsigned int hits, const int n, const uint32_t misc) {
        const float4 *g0 = S.g0 + buf, *g1 = S.g1 + buf, *r0 = S.r0 + buf, *r1 = S.r1 + buf, *colp = S.col + buf;
        int j = 0;
        for (int k0 = 0; k0 < n; ++j) {
            const unsigned int hsub = hits >> k0;
            // E rows of this batch: row i = every pixel's i-th hit of the batch; this pixel's hits in this sub-batch start at
            // row popc(its hits in earlier slots). The first EROWS of them are fetched into registers here, in one go (a load
            // inside the chain loop would make every step wait for it: loads share scoreboards); later rows: slow path.
            const float* eg = nullptr;
            float e[EROWS];
            if (haveE) {
                const uint32_t ord = (uint32_t)__popc(hits & ((1u << k0) - 1u)), rows_total = __shfl_sync(FULL, misc, 7);
                eg = trav_E + ((size_t)__shfl_sync(FULL, misc, 1) + ord) * 32u + lane;
#pragma unroll
                for (int u = 0; u < EROWS; ++u) e[u] = (ord + (uint32_t)u < rows_total) ? __ldg(eg + 32 * u) : 1.f;
                eg += 32 * EROWS;
            }
            const QLayout L = queue_layout(hsub, n - k0, S.Q, lane);
            const unsigned int mine = (L.n < 32) ? (hsub & ((1u << L.n) - 1u)) : hsub;
            if (L.nh > 0) {
                __syncwarp();
                if (!haveE) {
                    queue_fill(mine, S.Q, L, lane);
                    __syncwarp();
                    if constexpr (HEADS) sweep_E<K, true>(g0 + k0, g1 + k0, r0 + k0, r1 + k0, S.A, S.Q, L, S.TM, lane);
                    else sweep_E<K, false>(g0 + k0, g1 + k0, r0 + k0, r1 + k0, S.A, S.Q, L, nullptr, lane);
                    __syncwarp();
                }
                // ---- pixel-major chain: eqs. 2-4 front to back, dL/dtau and w of every hit into the queue ----
                {
                    unsigned int m = mine;
                    auto chain = [&](const float e_rec) {
                        const int k = __ffs(m) - 1;
                        m &= m - 1;
                        const uint2 hk = S.Q.Hs[k];
                        const int st = q_st((int)hk.y + __popc(hk.x & lt), L);
                        if (haveE) S.Q.q[st] = (unsigned short)((k << 5) | lane);
                        const float E = haveE ? e_rec : S.Q.WD[st].x;
                        const float4 col = colp[k0 + k];
                        float gc = G.x * col.x + G.y * col.y + G.z * col.z;
                        if constexpr (HEADS) gc = fmaf(gdep, S.TM[st], gc);
                        const bool live = T >= T_min;                // R8: a ray stops after the voxel that crosses T_min
                        const float w = live ? T * (1.f - E) : 0.f;
                        T = live ? T * E : T;
                        P = fmaf(w, gc, P);
                        S.Q.WD[st] = make_float2(w, live ? fmaf(T, gc, P) : 0.f);
                    };
                    bool more = __any_sync(FULL, m != 0u);
#pragma unroll
                    for (int u = 0; u < EROWS; ++u) {
                        if (more) {
                            if (m) chain(e[u]);
                            more = __any_sync(FULL, m != 0u);
                        }
                    }
                    while (more) {                                       // more than EROWS hits of one pixel in a sub-batch
                        float e_rec = 1.f;
                        if (haveE && m) e_rec = __ldg(eg);
                        eg += 32;
                        if (m) chain(e_rec);
                        more = __any_sync(FULL, m != 0u);
                    }
                }
                __syncwarp();
                // the slot headers are not read again in this sub-batch: Hs[k].x now collects slot k's max blending weight
                if (want_wmax) { S.Q.Hs[lane].x = 0u; __syncwarp(); }
                // ---- hit-major: gradients of this lane's C consecutive entries, summed in registers per voxel ----
                {
                    float acc[11];
#pragma unroll
                    for (int m = 0; m < 11; ++m) acc[m] = 0.f;
                    float wq = 0.f;
                    int cur = -1;
                    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), bq = a, ra = a, rb = a;
                    auto flush = [&]() {
                        if (wq > 0.f || acc[0] != 0.f) {
                            const uint32_t vid = __float_as_uint(bq.w);
                            float* row = grow + (size_t)vid * 16;             // the voxel's 64-byte scratch row
                            red_add_v4(row, acc[0], acc[1], acc[2], acc[3]);
                            red_add_v4(row + 4, acc[4], acc[5], acc[6], acc[7]);
                            red_add_v4(row + 8, acc[8], acc[9], acc[10], 0.f);
                            if (want_wmax) atomicMax(&S.Q.Hs[cur].x, __float_as_uint(wq));
                        }
                    };
                    for (int cc = 0; cc < L.C; ++cc) {
                        const bool valid = lane * L.C + cc < L.nh;
                        const int st = q_row(cc, lane);
                        const unsigned int u = valid ? (unsigned int)S.Q.q[st] : 0u;
                        const int k = valid ? (int)(u >> 5) : cur;
                        if (k != cur) {                                  // next voxel: send the finished fragment
                            flush();
#pragma unroll
                            for (int m = 0; m < 11; ++m) acc[m] = 0.f;
                            wq = 0.f;
                            cur = k;
                            a = g0[k0 + k]; bq = g1[k0 + k]; ra = r0[k0 + k]; rb = r1[k0 + k];
                        }
                        if (valid) {
                            const float2 wd = S.Q.WD[st];
                            const float w = wd.x, dLdtau = wd.y;
                            if (w > 0.f || dLdtau != 0.f) {
                                const int i = (int)(u & 31u);
                                RayF rr;
#pragma unroll
                                for (int ax = 0; ax < 3; ++ax) {
                                    rr.dh[ax] = S.A[ax][i]; rr.dl[ax] = S.A[3 + ax][i]; rr.inv[ax] = S.A[6 + ax][i];
                                    rr.ainv[ax] = fabsf(rr.inv[ax]);
                                }
                                float s0, s1, t_ref, D[3];
                                if (slab(rr, a, bq, s0, s1, t_ref, D)) {           // the precise test decides
                                    integrate_bwd<K>(rr, D, a.w, s0, s1, ra, rb, dLdtau, acc);
                                    acc[8] = fmaf(w, S.A[9][i], acc[8]);
                                    acc[9] = fmaf(w, S.A[10][i], acc[9]);
                                    acc[10] = fmaf(w, S.A[11][i], acc[10]);
                                    wq = fmaxf(wq, w);
                                }
                            }
                        }
                    }
                    flush();
                }
                __syncwarp();
                // eq. 5: one atomicMax per voxel of the sub-batch (its hits all lie in this sub-batch); no guard read: a load
                // that is waited for here costs more than the reductions it would save
                if (want_wmax && lane >= k0 && lane < k0 + L.n) {
                    const unsigned int wv = S.Q.Hs[lane - k0].x;
                    if (wv != 0u) {
                        atomicMax(reinterpret_cast<unsigned int*>(grow + (size_t)__float_as_uint(g1[lane].w) * 16 + 12), wv);
                    }
                }
            }
            k0 += L.n;
        }
    };

    if (REPLAY) {
        // The forward pass recorded, per batch, the list entries it staged and the slots every pixel hit: no cull, no test.
        const uint32_t r0 = trav_off[tile], cap = (trav_off[tile + 1] - r0) >> 3;
        const uint32_t* rec = trav + ((size_t)r0 + (size_t)warp * cap) * TRAV_WORDS;
        const uint32_t n_rec = trav_count[tile * 8 + warp];
        if (n_rec == 0u) return;
        struct Hdr { unsigned int hits; uint32_t vid, misc; };
        auto load_hdr = [&](const uint32_t* r) {
            Hdr h;
            h.hits = __ldg(r + lane); h.vid = __ldg(r + 32 + lane); h.misc = __ldg(r + 64 + (lane & 7));
            return h;
        };
        auto gather = [&](const Hdr& h, int buf) {
            const int n = (int)__shfl_sync(FULL, h.misc, 0);
            if (lane < n) {
                const float4* pr = packed + 5 * (size_t)h.vid;
                const int slot = buf + lane;
                cp_async16(&S.g0[slot], pr); cp_async16(&S.g1[slot], pr + 1); cp_async16(&S.r0[slot], pr + 2);
                cp_async16(&S.r1[slot], pr + 3); cp_async16(&S.col[slot], pr + 4);
                // pull the voxel's gradient row into L2 now: a reduction that misses L2 waits for the DRAM fill
                asm volatile("prefetch.global.L2 [%0];" ::"l"(grow + (size_t)h.vid * 16));
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            if (haveE) {                                                // its E rows: into L2
                const uint32_t rows = __shfl_sync(FULL, h.misc, 7), eb = __shfl_sync(FULL, h.misc, 1);
                if ((uint32_t)lane < rows) asm volatile("prefetch.global.L2 [%0];" ::"l"(trav_E + ((size_t)eb + lane) * 32u));
            }
        };
        // header b + 2: into L2 (3 lines); header b + 1: loaded at the top of batch b, its voxel records gathered while batch b
        // is worked on. Only (hits, misc) of two headers live in registers across a batch.
        auto prefetch_hdr = [&](const uint32_t* r) {
            if (lane < 3) asm volatile("prefetch.global.L2 [%0];" ::"l"(r + 32 * lane));
        };
        unsigned int hits_a, hits_b = 0u;
        uint32_t misc_a, misc_b = 0u;
        // three headers deep: header b + 3 into L2, header b + 2 into registers (consumed one batch later, so its round
        // trip to L2 is not waited for), voxel records of batch b + 1 gathered, batch b worked on
        Hdr hn;
        hn.hits = 0u; hn.vid = 0u; hn.misc = 0u;
        {
            const Hdr h0 = load_hdr(rec);
            if (n_rec > 1u) hn = load_hdr(rec + TRAV_WORDS);
            if (n_rec > 2u) prefetch_hdr(rec + 2 * TRAV_WORDS);
            gather(h0, 0);
            hits_a = h0.hits; misc_a = h0.misc;
        }
        for (uint32_t rb = 0; rb < n_rec; ++rb) {
            const int buf = (int)(rb & 1u) * NSLOT;
            if (rb + 1u < n_rec) {
                gather(hn, buf ^ NSLOT);
                hits_b = hn.hits; misc_b = hn.misc;
                if (rb + 2u < n_rec) hn = load_hdr(rec + (size_t)(rb + 2u) * TRAV_WORDS);
                if (rb + 3u < n_rec) prefetch_hdr(rec + (size_t)(rb + 3u) * TRAV_WORDS);
                asm volatile("cp.async.wait_group 1;" ::: "memory");
            } else {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            __syncwarp();
            run_batch(buf, hits_a, (int)__shfl_sync(FULL, misc_a, 0), misc_a);
            __syncwarp();
            hits_a = hits_b; misc_a = misc_b;
        }
        return;
    }

    for (int so = 0; so < 8; ++so) {
        const uint32_t start = ranges[(tile * 8 + so) * 2], end = ranges[(tile * 8 + so) * 2 + 1];
        if (start == end) continue;
        bool alive = inimg && (oct == so) && (T >= T_min);
        unsigned int alive_mask = __ballot_sync(FULL, alive);
        if (alive_mask == 0u) continue;                               // no pixel of this warp uses this list
        uint32_t base = start;
        while (base < end) {
            // ---- 1. cull + stage until 32 survivors are waiting or the list is exhausted ----
            int count = 0;
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
                    const int slot = count + rank;
                    const uint32_t vid = __float_as_uint(t1.w);
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(grow + (size_t)vid * 16));
                    S.g0[slot] = t0; S.g1[slot] = t1; S.r0[slot] = t2; S.r1[slot] = t3; S.col[slot] = t4;
                }
                count += __popc(m);
                base += adv;
            }
            if (count == 0) break;
            __syncwarp();
            // ---- 2. test: every lane walks its own pixel's candidates (conservative slab test) ----
            unsigned int cand = transpose32(lane < count ? __float_as_uint(S.col[lane].w) : 0u, lane);
            if (!alive) cand = 0u;
            unsigned int n_test = 0;
            const unsigned int hits = test_candidates<false>(cand, S.g0, S.col, inv, n_test);
            if (__any_sync(FULL, hits != 0u)) run_batch(0, hits, count, 0u);
            __syncwarp();
            alive = inimg && (oct == so) && (T >= T_min);
            alive_mask = __ballot_sync(FULL, alive);
            if (alive_mask == 0u) break;                              // whole warp terminated
        }
    }
}

}  // namespace

// A cudaFuncAttribute is per device: set it on every launch path once per (kernel, device) (a second context on another GPU
// must get it too); the call is cheap next to a launch, so it is simply repeated.
#define SVR_SET_SMEM(ctx, kernel, smem) SVR_CUDA(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(smem)))

SvrStatus launch_forward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, float* image, float* depth, float* T_final,
                         float* w_max, unsigned long long* stats, bool record) {
    if (f->n_tiles == 0) return SVR_OK;
    const size_t smem = sizeof(FwdWarp) * FWD_CTAW;
    const uint2* rs = reinterpret_cast<const uint2*>(f->rects_sorted);
    const float4* pk = reinterpret_cast<const float4*>(f->packed);
    unsigned int* wm = reinterpret_cast<unsigned int*>(w_max);
    const bool rec = record && f->trav != nullptr;
    if (rec && f->trav_ectl) SVR_CUDA(ctx, cudaMemsetAsync(f->trav_ectl, 0, 2 * sizeof(uint32_t), ctx->stream));
    StageScope scope__(ctx, ST_FORWARD);
#define SVR_FWD_GO2(KK, SS, RR, WW)                                                                                  \
    do {                                                                                                             \
        SVR_SET_SMEM(ctx, (composite_kernel<KK, SS, RR, WW>), smem);                                                 \
        composite_kernel<KK, SS, RR, WW><<<f->n_tiles * (8 / FWD_CTAW), 32 * FWD_CTAW, smem, ctx->stream>>>(f->cam, pk, f->vals, rs, f->ranges, f->tile_order, T_min, image, depth, \
                                                                             T_final, wm, stats, f->trav, f->trav_off, f->trav_count, \
                                                                             f->trav_E, f->trav_ectl, f->trav_E ? f->trav_E_cap : 0u);       \
    } while (0)
#define SVR_FWD_GO(KK, SS, RR)                                                                                       \
    do {                                                                                                             \
        if (wm) SVR_FWD_GO2(KK, SS, RR, true);                                                                       \
        else SVR_FWD_GO2(KK, SS, RR, false);                                                                         \
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
#undef SVR_FWD_GO2
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_backward(SvrContext* ctx, const SvrFrame* f, int K, float T_min, const float* dL, const float* image,
                          float* grad_row, bool want_wmax, const float* dL_ddepth, const float* dL_dT,
                          const float* depth, const float* T_final) {
    if (f->n_tiles == 0) return SVR_OK;
    StageScope scope__(ctx, ST_BACKWARD);
    const uint2* rs = reinterpret_cast<const uint2*>(f->rects_sorted);
    const float4* pk = reinterpret_cast<const float4*>(f->packed);
    // replay the forward pass's traversal record when there is one for this termination threshold and sample count (the
    // recorded E = exp(-tau) values, and through them the slot where a ray stopped, belong to the K they were integrated with)
    const bool replay = f->trav != nullptr && f->trav_valid && f->trav_T_min == T_min && f->trav_K == K && (ctx->debug_flags & 16) == 0;
    const bool heads = dL_ddepth != nullptr || dL_dT != nullptr;
    const float* eg = (ctx->debug_flags & 32) ? nullptr : f->trav_E;       // debug flag 32: ignore the recorded E values
#define SVR_BWD_GO(KK, HH, RR)                                                                                       \
    do {                                                                                                             \
        const size_t smem = sizeof(BwdWarp<HH>) * BWD_CW(RR);                                                             \
        SVR_SET_SMEM(ctx, (backward_packed_kernel<KK, HH, RR>), smem);                                               \
        backward_packed_kernel<KK, HH, RR><<<f->n_tiles * (8 / BWD_CW(RR)), 32 * BWD_CW(RR), smem, ctx->stream>>>(                             \
            f->cam, pk, f->vals, rs, f->ranges, f->tile_order, T_min, want_wmax, dL, image, grad_row, dL_ddepth, dL_dT, depth, T_final,         \
            f->trav, f->trav_off, f->trav_count, eg, f->trav_ectl);                                                  \
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
            f->vals, f->n_entries, reinterpret_cast<const uint2*>(f->rects_tight ? f->rects_tight : f->rects), reinterpret_cast<uint2*>(f->rects_sorted));
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}
