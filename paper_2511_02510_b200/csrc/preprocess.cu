// Stage (1)+(2) kernels: tile octant masks, per-voxel pixel rectangles and entry counts, key emission,
// per-(tile,octant) ranges, per-view SH colours. Integer outputs are bit-exact against the binning
// specification B1-B4 in DESIGN.md: all fp32 arithmetic that decides an integer uses __f*_rn intrinsics
// (never contracted to FMA) in the specified order.
#include "svr_internal.cuh"

namespace {

constexpr int BIG_THRESHOLD = 48;   // voxels with more list entries than this are emitted by a whole CTA

// ---- B2: octant set of every tile ---------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_mask_kernel(CamDev c, uint8_t* __restrict__ masks) {
    __shared__ unsigned int m;
    if (threadIdx.x == 0 && threadIdx.y == 0) m = 0;
    __syncthreads();
    int x = blockIdx.x * SVR_TILE + threadIdx.x, y = blockIdx.y * SVR_TILE + threadIdx.y;
    unsigned int mine = 0;
    if (x < c.W && y < c.H) mine = 1u << pixel_octant_dev(c, x, y);
    mine = __reduce_or_sync(0xffffffffu, mine);
    if (((threadIdx.y * SVR_TILE + threadIdx.x) & 31) == 0) atomicOr(&m, mine);
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) masks[blockIdx.y * c.tiles_x + blockIdx.x] = (uint8_t)m;
}

// Summed-area table of popcount(mask): sat[j*(tx+1)+i] = entries of one voxel covering tiles [0,i) x [0,j).
__global__ void sat_kernel(const uint8_t* __restrict__ masks, uint32_t* __restrict__ sat, int tx, int ty) {
    int sx = tx + 1;
    for (int i = threadIdx.x; i <= tx; i += blockDim.x) sat[i] = 0;
    for (int j = threadIdx.x; j < ty; j += blockDim.x) {      // row prefix sums
        uint32_t run = 0;
        sat[(j + 1) * sx] = 0;
        for (int i = 0; i < tx; ++i) {
            run += __popc((unsigned)masks[j * tx + i]);
            sat[(j + 1) * sx + i + 1] = run;
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= tx; i += blockDim.x) {      // column prefix sums
        uint32_t run = 0;
        for (int j = 1; j <= ty; ++j) {
            run += sat[j * sx + i];
            sat[j * sx + i] = run;
        }
    }
}

__device__ __forceinline__ uint32_t sat_query(const uint32_t* __restrict__ sat, int sx, int i0, int j0, int i1, int j1) {
    // tiles [i0, i1) x [j0, j1)
    return sat[j1 * sx + i1] - sat[j0 * sx + i1] - sat[j1 * sx + i0] + sat[j0 * sx + i0];
}

// ---- B1: pixel rectangle of a voxel ---------------------------------------------------------------
// *tight (optional) = the pixels whose CENTRE lies in the projected bounding box grown by a margin m: only their rays can hit
// the voxel (the projection of a box in front of the camera is inside the bounding box of its projected corners).
// m = max(1/64 px, bound on the fp32 error of the projected corner), per axis. The bound follows the rounding of the chain
// above: each camera-space coordinate is 3 products and 3 sums of magnitude <= Mg = |P|_1 + |t|_inf (|R_ij| <= 1), plus the
// rounding of lo / hi themselves, so |dX|, |dY|, |dZ| <= d = 2^-21 Mg; the quotient, the scaling and the offset add
// 2^-21 (|u| + |cx|); together |du| <= 1.01 (fx + |u - cx|) d / zmin + 2^-21 (|u| + |cx|). Typical views (C4: fx ~ 1000,
// z ~ 2.5, Mg ~ 6) give ~1e-3 px, so the margin stays 1/64 px; it grows for voxels within a few z_near of a camera
// inside the scene and for large fx (4K images: up to a few 0.1 px), where a fixed 1/64 px would drop true hits. The result
// is clamped to the B1 rectangle, whose own margin is at least 0.5 px. The compositing cull uses it; the lists are built from
// the B1 rectangle.
__device__ __forceinline__ ushort4 voxel_rect(const SceneDev& s, const CamDev& c, uint2 q, ushort4* tight = nullptr) {
    const ushort4 culled = make_ushort4(0xFFFF, 0xFFFF, 0, 0);
    if (tight) *tight = culled;
    int L = q.y >> 16;
    float e = __fmul_rn(s.root_edge, __int_as_float((127 - L) << 23));
    float lo[3], hi[3];
    lo[0] = __fadd_rn(s.root_lo[0], __fmul_rn((float)(q.x & 0xFFFF), e));
    lo[1] = __fadd_rn(s.root_lo[1], __fmul_rn((float)(q.x >> 16), e));
    lo[2] = __fadd_rn(s.root_lo[2], __fmul_rn((float)(q.y & 0xFFFF), e));
#pragma unroll
    for (int a = 0; a < 3; ++a) hi[a] = __fadd_rn(lo[a], e);
    float X[8], Y[8], Z[8];
    float zmin = 0.f, zmax = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float Px = (k & 1) ? hi[0] : lo[0], Py = (k & 2) ? hi[1] : lo[1], Pz = (k & 4) ? hi[2] : lo[2];
        X[k] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[0], Px), __fmul_rn(c.R[1], Py)), __fmul_rn(c.R[2], Pz)), c.t[0]);
        Y[k] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[3], Px), __fmul_rn(c.R[4], Py)), __fmul_rn(c.R[5], Pz)), c.t[1]);
        Z[k] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[6], Px), __fmul_rn(c.R[7], Py)), __fmul_rn(c.R[8], Pz)), c.t[2]);
        if (k == 0) { zmin = zmax = Z[k]; }
        else { zmin = fminf(zmin, Z[k]); zmax = fmaxf(zmax, Z[k]); }
    }
    if (!(zmax > 0.0f)) return culled;
    float Wf = (float)c.W, Hf = (float)c.H;
    if (zmin < c.z_near) {
        float cxw = __fsub_rn(c.cx, Wf), cyh = __fsub_rn(c.cy, Hf);
        bool allL = true, allR = true, allT = true, allB = true;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float a0 = __fmul_rn(c.fx, X[k]), b0 = __fmul_rn(c.fy, Y[k]);
            allL = allL && (__fadd_rn(a0, __fmul_rn(c.cx, Z[k])) < 0.0f);
            allR = allR && (__fadd_rn(a0, __fmul_rn(cxw, Z[k])) >= 0.0f);
            allT = allT && (__fadd_rn(b0, __fmul_rn(c.cy, Z[k])) < 0.0f);
            allB = allB && (__fadd_rn(b0, __fmul_rn(cyh, Z[k])) >= 0.0f);
        }
        if (allL || allR || allT || allB) return culled;
        if (tight) *tight = make_ushort4(0, 0, (unsigned short)(c.W - 1), (unsigned short)(c.H - 1));
        return make_ushort4(0, 0, (unsigned short)(c.W - 1), (unsigned short)(c.H - 1));
    }
    float u0 = 0.f, u1 = 0.f, v0 = 0.f, v1 = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float u = __fadd_rn(__fmul_rn(c.fx, __fdiv_rn(X[k], Z[k])), c.cx);
        float w = __fadd_rn(__fmul_rn(c.fy, __fdiv_rn(Y[k], Z[k])), c.cy);
        if (k == 0) { u0 = u1 = u; v0 = v1 = w; }
        else { u0 = fminf(u0, u); u1 = fmaxf(u1, u); v0 = fminf(v0, w); v1 = fmaxf(v1, w); }
    }
    if (u1 < 0.0f || u0 >= Wf || v1 < 0.0f || v0 >= Hf) return culled;
    ushort4 r;
    r.x = (unsigned short)(int)floorf(fmaxf(u0, 0.0f));
    r.z = (unsigned short)(int)floorf(fminf(u1, __fsub_rn(Wf, 1.0f)));
    r.y = (unsigned short)(int)floorf(fmaxf(v0, 0.0f));
    r.w = (unsigned short)(int)floorf(fminf(v1, __fsub_rn(Hf, 1.0f)));
    if (tight) {
        const float Mg = fmaxf(fabsf(lo[0]), fabsf(hi[0])) + fmaxf(fabsf(lo[1]), fabsf(hi[1])) + fmaxf(fabsf(lo[2]), fabsf(hi[2])) +
                         fmaxf(fmaxf(fabsf(c.t[0]), fabsf(c.t[1])), fabsf(c.t[2]));
        const float p21 = 4.76837158e-7f;                                   // 2^-21
        const float dz = 1.01f * p21 * Mg / zmin;                           // zmin >= z_near > 0 here
        const float mu = fmaxf(1.0f / 64.0f, (c.fx + fmaxf(fabsf(u0 - c.cx), fabsf(u1 - c.cx))) * dz + p21 * (fmaxf(fabsf(u0), fabsf(u1)) + fabsf(c.cx)));
        const float mv = fmaxf(1.0f / 64.0f, (c.fy + fmaxf(fabsf(v0 - c.cy), fabsf(v1 - c.cy))) * dz + p21 * (fmaxf(fabsf(v0), fabsf(v1)) + fabsf(c.cy)));
        const int x0 = max((int)ceilf(u0 - (0.5f + mu)), (int)r.x), x1 = min((int)floorf(u1 - (0.5f - mu)), (int)r.z);
        const int y0 = max((int)ceilf(v0 - (0.5f + mv)), (int)r.y), y1 = min((int)floorf(v1 - (0.5f - mv)), (int)r.w);
        if (x0 <= x1 && y0 <= y1) *tight = make_ushort4((unsigned short)x0, (unsigned short)y0, (unsigned short)x1, (unsigned short)y1);
    }
    return r;
}

__global__ void __launch_bounds__(256) rect_count_kernel(SceneDev s, CamDev c, const uint32_t* __restrict__ sat,
                                                         ushort4* __restrict__ rects, uint32_t* __restrict__ counts,
                                                         unsigned long long* __restrict__ totals) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v > s.n) return;
    if (v == s.n) { counts[v] = 0; return; }
    uint2 q = reinterpret_cast<const uint2*>(s.ijkl)[v];
    ushort4 r = voxel_rect(s, c, q);
    rects[v] = r;
    uint32_t cnt = 0;
    if (r.x <= r.z)
        cnt = sat_query(sat, c.tiles_x + 1, r.x >> 4, r.y >> 4, (r.z >> 4) + 1, (r.w >> 4) + 1);
    counts[v] = cnt;
    if (cnt > BIG_THRESHOLD) atomicAdd(&totals[1], 1ULL);
}

// ---- B3: keys ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t part1by2(uint64_t x) {
    x &= 0x1fffffULL;
    x = (x | x << 32) & 0x1f00000000ffffULL;
    x = (x | x << 16) & 0x1f0000ff0000ffULL;
    x = (x | x << 8) & 0x100f00f00f00f00fULL;
    x = (x | x << 4) & 0x10c30c30c30c30c3ULL;
    x = (x | x << 2) & 0x1249249249249249ULL;
    return x;
}

__device__ __forceinline__ uint64_t voxel_code(uint2 q, int Lm) {
    int sh = Lm - (int)(q.y >> 16);
    return part1by2((uint64_t)(q.x & 0xFFFF) << sh) | (part1by2((uint64_t)(q.x >> 16) << sh) << 1) |
           (part1by2((uint64_t)(q.y & 0xFFFF) << sh) << 2);
}

__device__ __forceinline__ uint64_t flip_mask(int o, int Lm) {
    uint64_t xm = 0x1249249249249249ULL & ((Lm >= 21) ? ~0ULL : ((1ULL << (3 * Lm)) - 1ULL));
    return ((o & 1) ? xm : 0ULL) | ((o & 2) ? xm << 1 : 0ULL) | ((o & 4) ? xm << 2 : 0ULL);
}

__device__ __forceinline__ void emit_tile(uint64_t* __restrict__ keys, uint32_t* __restrict__ vals, uint32_t pos,
                                          uint32_t tile, unsigned mask, uint64_t code, int Lm, uint32_t v) {
    while (mask) {
        int o = __ffs(mask) - 1;
        mask &= mask - 1;
        keys[pos] = ((uint64_t)tile << (3 + 3 * Lm)) | ((uint64_t)o << (3 * Lm)) | (code ^ flip_mask(o, Lm));
        vals[pos] = v;
        ++pos;
    }
}

__global__ void __launch_bounds__(256) emit_small_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                         const uint32_t* __restrict__ offsets, const uint8_t* __restrict__ masks,
                                                         uint64_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                         uint32_t* __restrict__ big_list, unsigned int* __restrict__ big_count) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    uint32_t off = offsets[v], cnt = offsets[v + 1] - off;
    if (cnt == 0) return;
    if (cnt > BIG_THRESHOLD) { big_list[atomicAdd(big_count, 1u)] = (uint32_t)v; return; }
    ushort4 r = rects[v];
    uint64_t code = voxel_code(reinterpret_cast<const uint2*>(s.ijkl)[v], s.max_level);
    for (int j = r.y >> 4; j <= (r.w >> 4); ++j)
        for (int i = r.x >> 4; i <= (r.z >> 4); ++i) {
            uint32_t tile = j * c.tiles_x + i;
            unsigned m = masks[tile];
            emit_tile(keys, vals, off, tile, m, code, s.max_level, (uint32_t)v);
            off += __popc(m);
        }
}

__global__ void __launch_bounds__(256) emit_big_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                       const uint32_t* __restrict__ offsets, const uint8_t* __restrict__ masks,
                                                       const uint32_t* __restrict__ sat, uint64_t* __restrict__ keys,
                                                       uint32_t* __restrict__ vals, const uint32_t* __restrict__ big_list,
                                                       const unsigned int* __restrict__ big_count) {
    int sx = c.tiles_x + 1;
    unsigned int nb = *big_count;
    for (unsigned int b = blockIdx.x; b < nb; b += gridDim.x) {
        uint32_t v = big_list[b];
        ushort4 r = rects[v];
        uint32_t off = offsets[v];
        uint64_t code = voxel_code(reinterpret_cast<const uint2*>(s.ijkl)[v], s.max_level);
        int i0 = r.x >> 4, j0 = r.y >> 4, w = (r.z >> 4) - i0 + 1, h = (r.w >> 4) - j0 + 1;
        for (int k = threadIdx.x; k < w * h; k += blockDim.x) {
            int j = k / w, i = k - j * w;
            uint32_t before = sat_query(sat, sx, i0, j0, i0 + w, j0 + j) + sat_query(sat, sx, i0, j0 + j, i0 + i, j0 + j + 1);
            uint32_t tile = (j0 + j) * c.tiles_x + i0 + i;
            emit_tile(keys, vals, off + before, tile, masks[tile], code, s.max_level, v);
        }
    }
}

// ---- B4: ranges -------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ranges_kernel(const uint64_t* __restrict__ keys, int64_t n, int shift,
                                                     uint32_t* __restrict__ ranges) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint64_t p = keys[i] >> shift;
    if (i == 0 || (keys[i - 1] >> shift) != p) ranges[2 * p] = (uint32_t)i;
    if (i + 1 == n || (keys[i + 1] >> shift) != p) ranges[2 * p + 1] = (uint32_t)(i + 1);
}

// ---- tile launch order: longest lists first -----------------------------------------------------------
// List lengths are heavy-tailed (C4: mean 1.3k, max 12k entries per tile). CTAs are dispatched in blockIdx
// order, so handing out the longest tiles first (LPT) keeps a few giants from forming the kernel's tail.
// One block: counting sort of the tiles on their quantised length (1024 bins, longest first). The order
// inside a bin is arbitrary; it only decides which CTA starts first.
__global__ void __launch_bounds__(1024) tile_order_kernel(const uint32_t* __restrict__ ranges, int n_tiles,
                                                          uint32_t* __restrict__ tile_len, uint32_t* __restrict__ tile_order) {
    __shared__ uint32_t hist[1024];
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t max_len;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    hist[tid] = 0;
    if (tid == 0) max_len = 0;
    __syncthreads();
    for (int t = tid; t < n_tiles; t += 1024) {
        uint32_t len = 0;
#pragma unroll
        for (int o = 0; o < 8; ++o) len += ranges[(t * 8 + o) * 2 + 1] - ranges[(t * 8 + o) * 2];
        tile_len[t] = len;
        atomicMax(&max_len, len);
    }
    __syncthreads();
    int shift = 0;
    while ((max_len >> shift) >= 1024u) ++shift;
    for (int t = tid; t < n_tiles; t += 1024) atomicAdd(&hist[1023u - (tile_len[t] >> shift)], 1u);   // bin 0 = longest
    __syncthreads();
    // exclusive scan of the 1024 bins
    uint32_t v = hist[tid], inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = wsum[lane], winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        wsum[lane] = winc - w;
    }
    __syncthreads();
    hist[tid] = wsum[warp] + inc - v;
    __syncthreads();
    for (int t = tid; t < n_tiles; t += 1024) tile_order[atomicAdd(&hist[1023u - (tile_len[t] >> shift)], 1u)] = (uint32_t)t;
}

// Record offsets of the traversal scratch (composite.cu: the forward pass records, per warp and batch, which list entries it
// staged and which of them each pixel hit; the backward pass replays them). Tile t owns 8 * (ceil(len / 32) + 9) records,
// one contiguous eighth per warp. One block of 1024 threads: exclusive scan in tile order.
__global__ void __launch_bounds__(1024) trav_offsets_kernel(const uint32_t* __restrict__ tile_len, int n_tiles, uint32_t* __restrict__ trav_off) {
    __shared__ uint32_t wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (n_tiles + 1023) / 1024, t0 = tid * per, t1 = min(n_tiles, t0 + per);
    uint32_t local = 0;
    for (int t = t0; t < t1; ++t) local += 8u * ((tile_len[t] + 31u) / 32u + 9u);
    uint32_t inc = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = wsum[lane], a = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, a, o);
            if (lane >= o) a += v;
        }
        wsum[lane] = a - w;
    }
    __syncthreads();
    uint32_t run = wsum[warp] + inc - local;
    for (int t = t0; t < t1; ++t) {
        trav_off[t] = run;
        run += 8u * ((tile_len[t] + 31u) / 32u + 9u);
    }
    if (t1 == n_tiles && t0 < n_tiles) trav_off[n_tiles] = run;
    if (n_tiles == 0 && tid == 0) trav_off[0] = 0;
}

// ---- a3: per-view voxel colour (R6) -------------------------------------------------------------------
// c_v = max(0, 0.5 + sum_i Y_i(dir_v) sh[v,i,:]); rgbm[v] = (r, g, b, clamp-mask bits).
template <int DEG>
__device__ __forceinline__ float4 voxel_color_dev(const SceneDev& s, const CamDev& c, uint2 q, int64_t v) {
    constexpr int NB = (DEG + 1) * (DEG + 1);
    float dx, dy, dz, Y[NB];
    voxel_dir_dev(s, c, q, dx, dy, dz);
    sh_basis_dev(DEG, dx, dy, dz, Y);
    const float* p = s.sh + v * (NB * 3);
    float acc[3] = {0.5f, 0.5f, 0.5f};
    if (NB * 3 % 4 == 0) {
        const float4* p4 = reinterpret_cast<const float4*>(p);
#pragma unroll
        for (int k = 0; k < NB * 3 / 4; ++k) {
            float4 t = __ldg(p4 + k);
            float tv[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                int idx = 4 * k + e;
                acc[idx % 3] = fmaf(Y[idx / 3], tv[e], acc[idx % 3]);
            }
        }
    } else {
#pragma unroll
        for (int idx = 0; idx < NB * 3; ++idx) acc[idx % 3] = fmaf(Y[idx / 3], __ldg(p + idx), acc[idx % 3]);
    }
    unsigned mask = (acc[0] > 0.f ? 1u : 0u) | (acc[1] > 0.f ? 2u : 0u) | (acc[2] > 0.f ? 4u : 0u);
    return make_float4(fmaxf(acc[0], 0.f), fmaxf(acc[1], 0.f), fmaxf(acc[2], 0.f), __uint_as_float(mask));
}

template <int DEG>
__global__ void __launch_bounds__(256) voxel_color_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                          float4* __restrict__ rgbm) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    ushort4 r = rects[v];
    if (r.x > r.z) return;                                   // not visible in this view: never read
    rgbm[v] = voxel_color_dev<DEG>(s, c, reinterpret_cast<const uint2*>(s.ijkl)[v], v);
}

// ---- a10: per-voxel backward finalize ---------------------------------------------------------------
// (i) corner gradients from the polynomial-coefficient gradients the compositing kernel accumulated:
//     coef = A raw (see composite.cu) => grad_raw += A^T grad_coef;
// (ii) grad_sh[v,i,ch] += Y_i(dir_v) * grad_rgb[v,ch] * [c_v,ch > 0] (zero sub-gradient at the clamp).
// Consumed scratch entries are re-zeroed, so the scratch buffers stay all-zero between calls.
template <int DEG, bool OVERWRITE>
__global__ void __launch_bounds__(128) voxel_backward_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                             const float4* __restrict__ rgbm, float4* __restrict__ grow,
                                                             float4* __restrict__ grad_raw, float* __restrict__ grad_sh,
                                                             float* __restrict__ w_max) {
    constexpr int NB = (DEG + 1) * (DEG + 1);
    constexpr int ROW = NB * 3;
    __shared__ float Ysm[4][32][NB + 1];
    __shared__ float gsm[4][32][3];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t v0 = ((int64_t)blockIdx.x * 4 + warp) * 32;
    if (v0 >= s.n) return;
    const int64_t v = v0 + lane;
    bool vis = false;
    if (v < s.n) { ushort4 r = rects[v]; vis = r.x <= r.z; }
    bool sh_active = false, raw_done = false;
    if (vis) {
        // the voxel's 64-byte scratch row: coefficient gradient (8), colour gradient (3), -, max blending weight, -
        float4 ga = grow[4 * v], gb = grow[4 * v + 1];
        const float4 g = grow[4 * v + 2];
        const float wv = grow[4 * v + 3].x;
        if (wv != 0.f) {                                              // eq. 5: merge into the caller's w_max
            grow[4 * v + 3] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (w_max != nullptr) w_max[v] = fmaxf(w_max[v], wv);
        }
        if (ga.x != 0.f || ga.y != 0.f || ga.z != 0.f || ga.w != 0.f || gb.x != 0.f || gb.y != 0.f || gb.z != 0.f || gb.w != 0.f) {
            grow[4 * v] = make_float4(0.f, 0.f, 0.f, 0.f);
            grow[4 * v + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
            const float g0 = ga.x, gx = ga.y, gy = ga.z, gz = ga.w, gxy = gb.x, gxz = gb.y, gyz = gb.z, gxyz = gb.w;
            float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = ra;
            if (!OVERWRITE) { ra = grad_raw[2 * v]; rb = grad_raw[2 * v + 1]; }
            ra.x += ((g0 - gx) - (gy + gz)) + ((gxy + gxz) + (gyz - gxyz));
            ra.y += (gx - gxy) - (gxz - gxyz);
            ra.z += (gy - gxy) - (gyz - gxyz);
            ra.w += gxy - gxyz;
            rb.x += (gz - gxz) - (gyz - gxyz);
            rb.y += gxz - gxyz;
            rb.z += gyz - gxyz;
            rb.w += gxyz;
            grad_raw[2 * v] = ra;
            grad_raw[2 * v + 1] = rb;
            raw_done = true;
        }
        if (g.x != 0.f || g.y != 0.f || g.z != 0.f) {
            grow[4 * v + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
            unsigned mask = __float_as_uint(rgbm[v].w);
            float gv0 = (mask & 1u) ? g.x : 0.f, gv1 = (mask & 2u) ? g.y : 0.f, gv2 = (mask & 4u) ? g.z : 0.f;
            sh_active = (gv0 != 0.f || gv1 != 0.f || gv2 != 0.f);
            if (sh_active) {
                float dx, dy, dz, Y[NB];
                voxel_dir_dev(s, c, reinterpret_cast<const uint2*>(s.ijkl)[v], dx, dy, dz);
                sh_basis_dev(DEG, dx, dy, dz, Y);
#pragma unroll
                for (int i = 0; i < NB; ++i) Ysm[warp][lane][i] = Y[i];
                gsm[warp][lane][0] = gv0; gsm[warp][lane][1] = gv1; gsm[warp][lane][2] = gv2;
            }
        }
    }
    if (OVERWRITE && v < s.n && !raw_done) {                          // no gradient from this view: zeros, written not summed
        grad_raw[2 * v] = make_float4(0.f, 0.f, 0.f, 0.f);
        grad_raw[2 * v + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const unsigned amask = __ballot_sync(0xffffffffu, sh_active);
    if (!OVERWRITE && amask == 0u) return;
    __syncwarp();
    // the warp's contiguous grad_sh block, cooperatively: read-modify-write skipping untouched voxels, or (OVERWRITE) plain
    // stores of every voxel's row
    const int nvox = (int)min((int64_t)32, s.n - v0);
    if constexpr (ROW % 4 == 0) {
        float4* p4 = reinterpret_cast<float4*>(grad_sh + v0 * ROW);
        const int total = nvox * (ROW / 4);
        // four independent 16-byte loads in flight per lane before the first use
        for (int e0 = lane; e0 < total; e0 += 128) {
            float4 t[4];
            int vvs[4];
            bool on[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int e = e0 + 32 * u;
                vvs[u] = e / (ROW / 4);
                on[u] = e < total && ((amask >> vvs[u]) & 1u);
                t[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (!OVERWRITE && on[u]) t[u] = p4[e];
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int e = e0 + 32 * u, vv = vvs[u];
                if (!on[u]) {
                    if (OVERWRITE && e < total) p4[e] = make_float4(0.f, 0.f, 0.f, 0.f);
                    continue;
                }
                const int f0 = (e - vv * (ROW / 4)) * 4;
                float tv[4] = {t[u].x, t[u].y, t[u].z, t[u].w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int idx = f0 + k;
                    tv[k] = fmaf(Ysm[warp][vv][idx / 3], gsm[warp][vv][idx % 3], tv[k]);
                }
                p4[e] = make_float4(tv[0], tv[1], tv[2], tv[3]);
            }
        }
    } else {
        float* p = grad_sh + v0 * ROW;
        for (int e = lane; e < nvox * ROW; e += 32) {
            int vv = e / ROW;
            if (!((amask >> vv) & 1u)) {
                if (OVERWRITE) p[e] = 0.f;
                continue;
            }
            int idx = e - vv * ROW;
            p[e] = fmaf(Ysm[warp][vv][idx / 3], gsm[warp][vv][idx % 3], OVERWRITE ? 0.f : p[e]);
        }
    }
}

// ================================================================================================
// Bucketed list build (rows a4-a6, second design). The first design gave every voxel a contiguous block of
// entries (per-voxel counts -> scan over N voxels -> emit) and sorted all E (key, id) pairs on the full
// 51-bit key with 7 radix passes over global memory (21 launches, ~225 B of traffic per entry). The lists are
// (tile, octant) buckets, so here the top key bits are never sorted at all:
//   count    per voxel: atomic count into its (tile, octant) buckets; voxels that cover more than BIG_TILES
//            tiles add a +1/-1 corner pattern to a 2-D difference array instead (4 atomics);
//   scan     one block: 2-D prefix of the difference array -> per-tile cover of big voxels, added to the
//            buckets; exclusive scan of the bucket counts = the ranges (B4) and the write cursors;
//   scatter  per voxel: position = atomicAdd(cursor[bucket]); entry = (flipped Morton code << vb) | voxel id
//            in one 64-bit word (any order inside a bucket);
//   sort     one block per non-empty bucket (dynamic work fetch): radix passes over the code bits only, in shared
//            memory (buckets larger than SORT_CAP: through L2); tiny buckets use a bitonic network.
// Codes are unique within a bucket, so the result is the one sequence the oracle's full sort gives (bit-exact).
// Traffic per entry: 8 B written + 8 B read + 12 B written. Needs 3*Lmax + ceil(log2 N) <= 64 (else: first design).
constexpr int BIG_TILES = 16;
constexpr int SORT_CAP = 6144;        // largest bucket whose radix passes stay in shared memory (two buffers)
constexpr int SORT_CAP_SMALL = 1536;   // size classes: <= 1536 words: 128-thread blocks, <= 6144: 512, <= 12288: 1024
constexpr int SORT_CAP_BIG = 12288;   // same with one 1024-thread block per SM; beyond: passes through L2
constexpr int SMALL_CAP = 256;        // buckets up to this size: bitonic network
constexpr int SORT_THREADS2 = 512;

// The per-view colour (a3) of a visible voxel is computed here too: its 12 (D+1)^2-byte read overlaps the division-heavy
// projection of other warps instead of taking a pass of its own.
template <int DEG>
__global__ void __launch_bounds__(256) rect_bucket_count_kernel(SceneDev s, CamDev c, const uint8_t* __restrict__ masks,
                                                                ushort4* __restrict__ rects, uint32_t* __restrict__ bcount,
                                                                int* __restrict__ bigdiff, unsigned long long* __restrict__ totals,
                                                                float4* __restrict__ rgbm, float4* __restrict__ vrec,
                                                                ushort4* __restrict__ rects_tight) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    ushort4 r = make_ushort4(1, 0, 0, 0);      // "not visible"
    bool vis = false;
    if (v < s.n) {
        const uint2 q = reinterpret_cast<const uint2*>(s.ijkl)[v];
        {
            // the SH row and the corner densities are needed only after the division-heavy projection: start them now (90 % of
            // the voxels are visible), so that their DRAM latency runs beside it
            const char* psh = reinterpret_cast<const char*>(s.sh + v * ((DEG + 1) * (DEG + 1) * 3));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(psh));
            if (DEG >= 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(psh + 12 * (DEG + 1) * (DEG + 1) - 4));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(s.raw + v * 8));
        }
        ushort4 rt;
        r = voxel_rect(s, c, q, &rt);
        rects[v] = r;
        vis = r.x <= r.z;
        if (vis) {
            rects_tight[v] = rt;
            const float4 col = voxel_color_dev<DEG>(s, c, q, v);
            rgbm[v] = col;
            voxel_record_dev(s, c, q, (uint32_t)v, col, vrec);
        }
    }
    const int i0 = r.x >> 4, i1 = r.z >> 4, j0 = r.y >> 4, j1 = r.w >> 4;
    // A voxel inside one tile that has one octant (69 % of the visible ones on C4) has one bucket: the lanes of a warp that
    // share it send ONE atomic. In a scene stored in octree order neighbours share buckets and per-lane atomics serialise on
    // the same address (0.38 instead of 0.28 ms); in a randomly ordered scene the match costs one instruction.
    uint32_t key = 0xFFFFFFFFu - (uint32_t)lane;        // unique: no peers
    bool single = false;
    if (vis && i0 == i1 && j0 == j1) {
        const int tile = j0 * c.tiles_x + i0;
        const unsigned m = masks[tile];
        if ((m & (m - 1u)) == 0u) { single = true; key = (uint32_t)(tile * 8 + __ffs(m) - 1); }
    }
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    if (single) {
        if ((peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&bcount[key], (uint32_t)__popc(peers));
        return;
    }
    if (!vis) return;
    if ((i1 - i0 + 1) * (j1 - j0 + 1) > BIG_TILES) {
        const int sx = c.tiles_x + 1;
        atomicAdd(&totals[1], 1ULL);
        atomicAdd(&bigdiff[j0 * sx + i0], 1);
        atomicAdd(&bigdiff[j0 * sx + i1 + 1], -1);
        atomicAdd(&bigdiff[(j1 + 1) * sx + i0], -1);
        atomicAdd(&bigdiff[(j1 + 1) * sx + i1 + 1], 1);
        return;
    }
    for (int j = j0; j <= j1; ++j)
        for (int i = i0; i <= i1; ++i) {
            const int tile = j * c.tiles_x + i;
            unsigned m = masks[tile];
            while (m) {
                const int o = __ffs(m) - 1;
                m &= m - 1;
                atomicAdd(&bcount[tile * 8 + o], 1u);
            }
        }
}

// One block of 1024 threads. bcount[b] becomes the write cursor (= first entry) of bucket b; ranges[b] = [start, end)
// ((0,0) when empty, B4); nonempty = ids of the non-empty buckets; totals[0] = E, totals[3] = number of non-empty buckets.
// Dynamic shared memory: the (ty+1) x (tx+1) difference array.
__global__ void __launch_bounds__(1024) bucket_scan_kernel(const uint8_t* __restrict__ masks, const int* __restrict__ bigdiff, int tx, int ty,
                                                           uint32_t* __restrict__ bcount, uint32_t* __restrict__ ranges,
                                                           uint32_t* __restrict__ nonempty, unsigned long long* __restrict__ totals) {
    extern __shared__ int sd[];
    __shared__ uint32_t wsum[32], wsum2[32], wsum3[32], wsum4[32], n_big_buckets, n_mid_buckets;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sx = tx + 1, nd = sx * (ty + 1);
    for (int i = tid; i < nd; i += 1024) sd[i] = bigdiff[i];
    __syncthreads();
    for (int j = warp; j <= ty; j += 32) {            // row prefix sums, one warp per row
        int carry = 0;
        for (int i0 = 0; i0 <= tx; i0 += 32) {
            const int i = i0 + lane;
            int v = (i <= tx) ? sd[j * sx + i] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, v, o);
                if (lane >= o) v += t;
            }
            if (i <= tx) sd[j * sx + i] = v + carry;
            carry += __shfl_sync(0xffffffffu, v, 31);
        }
    }
    __syncthreads();
    for (int i = tid; i <= tx; i += 1024) {           // column prefix sums: sd[j][i] = big voxels covering tile (i, j)
        int run = 0;
        for (int j = 0; j <= ty; ++j) { run += sd[j * sx + i]; sd[j * sx + i] = run; }
    }
    __syncthreads();
    const int n_tiles = tx * ty;
    const int tpt = (n_tiles + 1023) / 1024;          // whole tiles per thread: 8 buckets = two 16-byte words each
    const int t0 = tid * tpt, t1 = min(n_tiles, t0 + tpt);
    uint32_t local = 0, local_ne = 0, local_big = 0, local_mid = 0;
    for (int t = t0; t < t1; ++t) {
        const uint4 a = reinterpret_cast<const uint4*>(bcount)[2 * t], b = reinterpret_cast<const uint4*>(bcount)[2 * t + 1];
        const uint32_t c[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
        const uint32_t m = masks[t], cover = (uint32_t)sd[(t / tx) * sx + (t % tx)];
#pragma unroll
        for (int o = 0; o < 8; ++o) {
            const uint32_t cnt = c[o] + (((m >> o) & 1u) ? cover : 0u);
            local += cnt;
            local_big += (cnt > (uint32_t)SORT_CAP);
            local_mid += (cnt > (uint32_t)SORT_CAP_SMALL && cnt <= (uint32_t)SORT_CAP);
            local_ne += (cnt != 0u && cnt <= (uint32_t)SORT_CAP_SMALL);
        }
    }
    atomicAdd(&totals[0], (unsigned long long)local);     // E in 64 bits (the caller zeroed totals): >= 2^31 is refused on the host
    // block-wide exclusive scans of (local, local_ne, local_big, local_mid)
    uint32_t inc = local, inc2 = local_ne, inc3 = local_big, inc4 = local_mid;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o), t2 = __shfl_up_sync(0xffffffffu, inc2, o), t3 = __shfl_up_sync(0xffffffffu, inc3, o),
                 t4 = __shfl_up_sync(0xffffffffu, inc4, o);
        if (lane >= o) { inc += t; inc2 += t2; inc3 += t3; inc4 += t4; }
    }
    if (lane == 31) { wsum[warp] = inc; wsum2[warp] = inc2; wsum3[warp] = inc3; wsum4[warp] = inc4; }
    __syncthreads();
    if (warp == 0) {
        uint32_t w = wsum[lane], w2 = wsum2[lane], w3 = wsum3[lane], w4 = wsum4[lane], a = w, a2 = w2, a3 = w3, a4 = w4;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, a, o), t2 = __shfl_up_sync(0xffffffffu, a2, o), t3 = __shfl_up_sync(0xffffffffu, a3, o),
                     t4 = __shfl_up_sync(0xffffffffu, a4, o);
            if (lane >= o) { a += t; a2 += t2; a3 += t3; a4 += t4; }
        }
        wsum[lane] = a - w; wsum2[lane] = a2 - w2; wsum3[lane] = a3 - w3; wsum4[lane] = a4 - w4;
        if (lane == 31) { totals[3] = a2 + a3 + a4; totals[5] = a3; totals[6] = a3 + a4; n_big_buckets = a3; n_mid_buckets = a4; }
    }
    __syncthreads();
    // work list by size class, largest first: [ > SORT_CAP | > SORT_CAP_SMALL | rest ]
    uint32_t run = wsum[warp] + inc - local, run_big = wsum3[warp] + inc3 - local_big;
    uint32_t run_mid = n_big_buckets + wsum4[warp] + inc4 - local_mid;
    uint32_t run_ne = n_big_buckets + n_mid_buckets + wsum2[warp] + inc2 - local_ne;
    for (int t = t0; t < t1; ++t) {
        const uint4 a = reinterpret_cast<const uint4*>(bcount)[2 * t], b = reinterpret_cast<const uint4*>(bcount)[2 * t + 1];
        const uint32_t c[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
        const uint32_t m = masks[t], cover = (uint32_t)sd[(t / tx) * sx + (t % tx)];
        uint32_t cur[8], rg[16];
#pragma unroll
        for (int o = 0; o < 8; ++o) {
            const uint32_t cnt = c[o] + (((m >> o) & 1u) ? cover : 0u);
            cur[o] = run;
            rg[2 * o] = cnt ? run : 0u;
            rg[2 * o + 1] = cnt ? run + cnt : 0u;
            if (cnt > (uint32_t)SORT_CAP) nonempty[run_big++] = (uint32_t)(t * 8 + o);
            else if (cnt > (uint32_t)SORT_CAP_SMALL) nonempty[run_mid++] = (uint32_t)(t * 8 + o);
            else if (cnt) nonempty[run_ne++] = (uint32_t)(t * 8 + o);
            run += cnt;
        }
        reinterpret_cast<uint4*>(bcount)[2 * t] = make_uint4(cur[0], cur[1], cur[2], cur[3]);
        reinterpret_cast<uint4*>(bcount)[2 * t + 1] = make_uint4(cur[4], cur[5], cur[6], cur[7]);
#pragma unroll
        for (int q = 0; q < 4; ++q)
            reinterpret_cast<uint4*>(ranges)[4 * t + q] = make_uint4(rg[4 * q], rg[4 * q + 1], rg[4 * q + 2], rg[4 * q + 3]);
    }
}

__device__ __forceinline__ void scatter_tile(uint64_t* __restrict__ ent, uint32_t* __restrict__ cursor, int tile, unsigned m,
                                             uint64_t code, int Lm, int vb, uint32_t v) {
    while (m) {
        const int o = __ffs(m) - 1;
        m &= m - 1;
        const uint32_t pos = atomicAdd(&cursor[tile * 8 + o], 1u);
        ent[pos] = ((code ^ flip_mask(o, Lm)) << vb) | (uint64_t)v;
    }
}

__global__ void __launch_bounds__(256) scatter_small_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                            const uint8_t* __restrict__ masks, uint32_t* __restrict__ cursor,
                                                            uint64_t* __restrict__ ent, int vb, uint32_t* __restrict__ big_list,
                                                            unsigned int* __restrict__ big_count) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    ushort4 r = make_ushort4(1, 0, 0, 0);
    if (v < s.n) r = rects[v];
    const bool vis = r.x <= r.z;
    const int i0 = r.x >> 4, i1 = r.z >> 4, j0 = r.y >> 4, j1 = r.w >> 4;
    uint64_t code = 0ull;
    if (vis) code = voxel_code(reinterpret_cast<const uint2*>(s.ijkl)[v], s.max_level);
    // one-bucket voxels: one cursor atomic per distinct bucket of the warp (see rect_bucket_count_kernel)
    uint32_t key = 0xFFFFFFFFu - (uint32_t)lane;
    bool single = false;
    int o1 = 0;
    if (vis && i0 == i1 && j0 == j1) {
        const int tile = j0 * c.tiles_x + i0;
        const unsigned m = masks[tile];
        if ((m & (m - 1u)) == 0u) { single = true; o1 = __ffs(m) - 1; key = (uint32_t)(tile * 8 + o1); }
    }
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    const int leader = __ffs(peers) - 1;
    uint32_t pos0 = 0u;
    if (single && lane == leader) pos0 = atomicAdd(&cursor[key], (uint32_t)__popc(peers));
    pos0 = __shfl_sync(0xffffffffu, pos0, leader);
    if (single) {
        ent[pos0 + __popc(peers & ((1u << lane) - 1u))] = ((code ^ flip_mask(o1, s.max_level)) << vb) | (uint64_t)v;
        return;
    }
    if (!vis) return;
    if ((i1 - i0 + 1) * (j1 - j0 + 1) > BIG_TILES) { big_list[atomicAdd(big_count, 1u)] = (uint32_t)v; return; }
    for (int j = j0; j <= j1; ++j)
        for (int i = i0; i <= i1; ++i) {
            const int tile = j * c.tiles_x + i;
            scatter_tile(ent, cursor, tile, masks[tile], code, s.max_level, vb, (uint32_t)v);
        }
}

__global__ void __launch_bounds__(256) scatter_big_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                          const uint8_t* __restrict__ masks, uint32_t* __restrict__ cursor,
                                                          uint64_t* __restrict__ ent, int vb, const uint32_t* __restrict__ big_list,
                                                          const unsigned int* __restrict__ big_count) {
    const unsigned int nb = *big_count;
    for (unsigned int b = blockIdx.x; b < nb; b += gridDim.x) {
        const uint32_t v = big_list[b];
        const ushort4 r = rects[v];
        const uint64_t code = voxel_code(reinterpret_cast<const uint2*>(s.ijkl)[v], s.max_level);
        const int i0 = r.x >> 4, j0 = r.y >> 4, w = (r.z >> 4) - i0 + 1, h = (r.w >> 4) - j0 + 1;
        for (int k = threadIdx.x; k < w * h; k += blockDim.x) {
            const int j = k / w, i = k - j * w;
            const int tile = (j0 + j) * c.tiles_x + i0 + i;
            scatter_tile(ent, cursor, tile, masks[tile], code, s.max_level, vb, v);
        }
    }
}

// ---- per-bucket sort ----
// Buckets of up to SMALL_CAP words: bitonic network in shared memory (all compare-exchanges ascending, so virtual
// +inf padding never moves). Larger buckets: least-significant-digit radix sort, 8 bits per pass over the code bits
// only, ping-pong between two buffers that live in shared memory (<= CAP words) or in global memory (the
// bucket's own segment and its slice of the key output array, L2-resident). A pass = per-warp digit counts over
// warp-contiguous segments (match_any, no atomics), a scan over (digit, warp), and a stable scatter that repeats
// the walk with the scanned counters. A pass whose digit is the same for the whole bucket is skipped.
template <int THREADS>
__device__ __forceinline__ void smem_merge_steps(uint64_t* sk, int P, int j_first) {
    for (int j = j_first; j > 0; j >>= 1) {
        for (int t = threadIdx.x; t < (P >> 1); t += THREADS) {
            const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
            uint64_t a = sk[i], b = sk[i + j];
            if (b < a) { sk[i] = b; sk[i + j] = a; }
        }
        __syncthreads();
    }
}

template <int THREADS>
__device__ __forceinline__ void smem_sort(uint64_t* sk, int P) {
    for (int k = 2; k <= P; k <<= 1) {
        const int hk = k >> 1;
        for (int t = threadIdx.x; t < (P >> 1); t += THREADS) {      // flip step: (i, i ^ (k - 1))
            const int blk = t / hk, off = t - blk * hk;
            const int i = blk * k + off, l = blk * k + (k - 1 - off);
            uint64_t a = sk[i], b = sk[l];
            if (b < a) { sk[i] = b; sk[l] = a; }
        }
        __syncthreads();
        smem_merge_steps<THREADS>(sk, P, k >> 2);
    }
}

// wh[w][d] (per-warp counts of digit d) -> exclusive offsets over the warps; tot[d] = first position of digit d.
// Returns true (block-uniform) when one digit holds all m words. DPT digits per thread when the block has < 256 threads.
template <int THREADS, typename CT>
__device__ __forceinline__ bool digit_scan(CT* wh, uint32_t* tot, uint32_t* sh8, uint32_t m) {
    constexpr int DPT = (THREADS >= 256) ? 1 : 256 / THREADS;
    constexpr int ACTIVE = 256 / DPT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t sum[DPT], total = 0;
    bool all = false;
    if (tid < ACTIVE) {
#pragma unroll
        for (int j = 0; j < DPT; ++j) {
            const int d = tid * DPT + j;
            uint32_t run = 0;
#pragma unroll
            for (int w = 0; w < (THREADS / 32); ++w) { const uint32_t c = wh[w * 256 + d]; wh[w * 256 + d] = (CT)run; run += c; }
            sum[j] = run;
            total += run;
            all = all || (run == m);
        }
    }
    if (__syncthreads_or(all)) return true;
    uint32_t inc = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (tid < ACTIVE && lane == 31) sh8[warp] = inc;
    __syncthreads();
    if (tid < ACTIVE) {
        uint32_t basev = inc - total;
#pragma unroll
        for (int w = 0; w < ACTIVE / 32; ++w) if (w < warp) basev += sh8[w];
#pragma unroll
        for (int j = 0; j < DPT; ++j) { tot[tid * DPT + j] = basev; basev += sum[j]; }
    }
    __syncthreads();
    return false;
}

// One radix pass over src[0, m) -> dst[0, m) on digit (word >> shift) & mask. wh = [(THREADS / 32)][256] counters, tot = [256].
// Returns false (and writes nothing) when all words share the digit.
template <int THREADS>
__device__ __forceinline__ bool radix_pass(const uint64_t* src, uint64_t* dst, uint32_t m, int shift, uint32_t mask,
                                           uint32_t* wh, uint32_t* tot, uint32_t* sh8) {
    constexpr unsigned FULLM = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    for (int i = tid; i < (THREADS / 32) * 256; i += THREADS) wh[i] = 0;
    __syncthreads();
    const uint32_t rounds = (m + 31) >> 5, rpw = (rounds + (THREADS / 32) - 1) / (THREADS / 32);
    const uint32_t r0 = warp * rpw, r1 = min(rounds, r0 + rpw);
    uint32_t* my = wh + warp * 256;
    for (uint32_t r = r0; r < r1; ++r) {
        const uint32_t i = (r << 5) + lane;
        const uint32_t d = (i < m) ? ((uint32_t)(src[i] >> shift) & mask) : 256u;
        const unsigned peers = __match_any_sync(FULLM, d);
        if ((peers & lt) == 0u && d < 256u) my[d] += __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    if (digit_scan<THREADS>(wh, tot, sh8, m)) return false;
    for (uint32_t r = r0; r < r1; ++r) {
        const uint32_t i = (r << 5) + lane;
        const bool valid = i < m;
        const uint64_t e = valid ? src[i] : 0ull;
        const uint32_t d = valid ? ((uint32_t)(e >> shift) & mask) : 256u;
        const unsigned peers = __match_any_sync(FULLM, d);
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && valid) { old = my[d]; my[d] = old + __popc(peers); }
        old = __shfl_sync(FULLM, old, leader);
        if (valid) dst[tot[d] + old + __popc(peers & lt)] = e;
        __syncwarp();
    }
    __syncthreads();
    return true;
}

// Same pass for buckets of up to CAP words (shared-memory buffers): every warp keeps its (CAP / THREADS) rounds of
// words in registers, ranks them once (match_any + a running per-warp counter) and scatters after the scan without
// walking the data again.
template <int THREADS, int CAP>
__device__ __forceinline__ bool radix_pass_reg(const uint64_t* src, uint64_t* dst, uint32_t m, int shift, uint32_t mask,
                                               uint16_t* wh, uint32_t* tot, uint32_t* sh8) {
    constexpr unsigned FULLM = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t rounds = (m + 31) >> 5, rpw = (rounds + (THREADS / 32) - 1) / (THREADS / 32);     // <= (CAP / THREADS)
    const uint32_t i0 = (warp * rpw << 5) + lane;
    uint64_t e[(CAP / THREADS)];
    uint32_t pre[(CAP / THREADS)];
#pragma unroll
    for (int k = 0; k < (CAP / THREADS); ++k) {
        const uint32_t i = i0 + (k << 5);
        e[k] = ((uint32_t)k < rpw && i < m) ? src[i] : ~0ull;
    }
    for (int i = tid; i < (THREADS / 32) * 256; i += THREADS) wh[i] = 0;
    __syncthreads();
    uint16_t* my = wh + warp * 256;
#pragma unroll
    for (int k = 0; k < (CAP / THREADS); ++k) {
        if ((uint32_t)k < rpw) {
            const uint32_t i = i0 + (k << 5);
            const uint32_t d = (i < m) ? ((uint32_t)(e[k] >> shift) & mask) : 256u;
            const unsigned peers = __match_any_sync(FULLM, d);
            const int leader = __ffs(peers) - 1;
            uint32_t old = 0;
            if (lane == leader && d < 256u) { old = my[d]; my[d] = (uint16_t)(old + __popc(peers)); }
            pre[k] = __shfl_sync(FULLM, old, leader) + __popc(peers & lt);
            __syncwarp();
        }
    }
    __syncthreads();
    if (digit_scan<THREADS>(wh, tot, sh8, m)) return false;
#pragma unroll
    for (int k = 0; k < (CAP / THREADS); ++k) {
        const uint32_t i = i0 + (k << 5);
        if ((uint32_t)k < rpw && i < m) {
            const uint32_t d = (uint32_t)(e[k] >> shift) & mask;
            dst[tot[d] + my[d] + pre[k]] = e[k];
        }
    }
    __syncthreads();
    return true;
}

template <int THREADS, int CAP>
__global__ void __launch_bounds__(THREADS) bucket_sort_kernel(uint64_t* __restrict__ ent, const uint32_t* __restrict__ ranges,
                                                                    const uint32_t* __restrict__ nonempty, const unsigned long long* __restrict__ totals,
                                                                    unsigned int* __restrict__ work, int big_part, int code_bits, int vb,
                                                                    uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* bufA = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* bufB = bufA + CAP;
    uint16_t* wh = reinterpret_cast<uint16_t*>(bufB + CAP);
    __shared__ uint32_t tot[256];
    __shared__ uint32_t sh8[8];
    __shared__ unsigned int next;
    // work list by size class: [0, totals[5]) > SORT_CAP, [totals[5], totals[6]) > SORT_CAP_SMALL, [totals[6], totals[3]) the rest
    const unsigned int w_first = big_part == 0 ? 0u : (unsigned int)totals[big_part == 1 ? 5 : 6];
    const unsigned int n_ne = (unsigned int)totals[big_part == 0 ? 5 : (big_part == 1 ? 6 : 3)];
    const uint64_t vmask = (1ull << vb) - 1ull;
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) next = atomicAdd(work, 1u);
        __syncthreads();
        const unsigned int w = w_first + next;
        if (w >= n_ne) break;
        const uint32_t b = nonempty[w];
        const uint32_t start = ranges[2 * b], m = ranges[2 * b + 1] - start;
        uint64_t* seg = ent + start;
        const uint64_t prefix = (uint64_t)b << code_bits;
        const uint64_t* res;
        if (m <= SMALL_CAP) {
            int P = 2;
            while ((uint32_t)P < m) P <<= 1;
            for (int i = threadIdx.x; i < P; i += THREADS) bufA[i] = ((uint32_t)i < m) ? seg[i] : ~0ull;
            __syncthreads();
            smem_sort<THREADS>(bufA, P);
            res = bufA;
        } else {
            uint64_t *src, *dst;
            if (m <= CAP) {
                for (uint32_t i = threadIdx.x; i < m; i += THREADS) bufA[i] = seg[i];
                src = bufA; dst = bufB;
            } else {
                src = seg; dst = keys_out + start;                     // global ping-pong (both L2-resident)
            }
            __syncthreads();
            for (int shift = 0; shift < code_bits; shift += 8) {
                const uint32_t mask = (code_bits - shift < 8) ? ((1u << (code_bits - shift)) - 1u) : 255u;
                const bool moved = (m <= CAP) ? radix_pass_reg<THREADS, CAP>(src, dst, m, vb + shift, mask, wh, tot, sh8)
                                                   : radix_pass<THREADS>(src, dst, m, vb + shift, mask, reinterpret_cast<uint32_t*>(bufA), tot, sh8);
                if (moved) { uint64_t* t = src; src = dst; dst = t; }
            }
            res = src;
        }
        // res may alias keys_out + start: every thread reads its word before it writes the same index
        for (uint32_t i = threadIdx.x; i < m; i += THREADS) {
            const uint64_t e = res[i];
            keys_out[start + i] = prefix | (e >> vb);
            vals_out[start + i] = (uint32_t)(e & vmask);
        }
    }
}

inline unsigned int blocks_for(int64_t n, int bs) { return (unsigned int)((n + bs - 1) / bs); }

}  // namespace

SvrStatus launch_tile_masks(SvrContext* ctx, SvrFrame* f, bool with_sat) {
    StageScope scope__(ctx, ST_TILE_MASKS);
    dim3 grid(f->cam.tiles_x, f->cam.tiles_y), block(SVR_TILE, SVR_TILE);
    tile_mask_kernel<<<grid, block, 0, ctx->stream>>>(f->cam, f->tile_masks);
    ctx->launches += 1;
    if (with_sat) {      // the summed-area table serves the per-voxel counts of the first list-build design only
        sat_kernel<<<1, 256, 0, ctx->stream>>>(f->tile_masks, f->sat, f->cam.tiles_x, f->cam.tiles_y);
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// totals[1] = number of "big" voxels (caller zeroes); totals[0] is filled by the caller from the scan.
SvrStatus launch_rects_counts(SvrContext* ctx, SvrFrame* f, uint32_t* counts, unsigned long long* totals) {
    StageScope scope__(ctx, ST_RECTS);
    rect_count_kernel<<<blocks_for(f->scene.n + 1, 256), 256, 0, ctx->stream>>>(
        f->scene, f->cam, f->sat, reinterpret_cast<ushort4*>(f->rects), counts, totals);
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_emit_keys(SvrContext* ctx, SvrFrame* f, uint64_t* keys, uint32_t* vals, uint32_t* big_list,
                                unsigned int* big_count) {
    StageScope scope__(ctx, ST_EMIT);
    emit_small_kernel<<<blocks_for(f->scene.n, 256), 256, 0, ctx->stream>>>(
        f->scene, f->cam, reinterpret_cast<const ushort4*>(f->rects), f->offsets, f->tile_masks, keys, vals, big_list, big_count);
    emit_big_kernel<<<148 * 4, 256, 0, ctx->stream>>>(f->scene, f->cam, reinterpret_cast<const ushort4*>(f->rects), f->offsets,
                                                      f->tile_masks, f->sat, keys, vals, big_list, big_count);
    ctx->launches += 2;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_ranges(SvrContext* ctx, SvrFrame* f) {
    StageScope scope__(ctx, ST_RANGES);
    SVR_CUDA(ctx, cudaMemsetAsync(f->ranges, 0, sizeof(uint32_t) * 16 * (size_t)f->n_tiles, ctx->stream));
    if (f->n_entries > 0) {
        ranges_kernel<<<blocks_for(f->n_entries, 256), 256, 0, ctx->stream>>>(
            f->keys, f->n_entries, 3 * f->scene.max_level, f->ranges);
        ctx->launches += 1;
    }
    tile_order_kernel<<<1, 1024, 0, ctx->stream>>>(f->ranges, f->n_tiles, f->tile_order + f->n_tiles, f->tile_order);
    ctx->launches += 1;
    if (f->trav_off) {
        trav_offsets_kernel<<<1, 1024, 0, ctx->stream>>>(f->tile_order + f->n_tiles, f->n_tiles, f->trav_off);
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_voxel_colors(SvrContext* ctx, SvrFrame* f) {
    StageScope scope__(ctx, ST_COLORS);
    if (f->scene.n == 0) return SVR_OK;
    unsigned int g = blocks_for(f->scene.n, 256);
    const ushort4* r = reinterpret_cast<const ushort4*>(f->rects);
    float4* out = reinterpret_cast<float4*>(f->rgbm);
    switch (f->scene.sh_degree) {
        case 0: voxel_color_kernel<0><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, r, out); break;
        case 1: voxel_color_kernel<1><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, r, out); break;
        case 2: voxel_color_kernel<2><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, r, out); break;
        default: voxel_color_kernel<3><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, r, out); break;
    }
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_sh_backward(SvrContext* ctx, const SvrFrame* f, float* grad_row, float* grad_raw, float* grad_sh, float* w_max,
                             bool overwrite) {
    StageScope scope__(ctx, ST_SH_BACKWARD);
    if (f->scene.n == 0) return SVR_OK;
    unsigned int g = blocks_for(f->scene.n, 128);
    const ushort4* r = reinterpret_cast<const ushort4*>(f->rects);
    const float4* rgbm = reinterpret_cast<const float4*>(f->rgbm);
    float4* gc = reinterpret_cast<float4*>(grad_row);
    float4* graw = reinterpret_cast<float4*>(grad_raw);
#define SVR_VB(DD)                                                                                                           \
    do {                                                                                                                     \
        if (overwrite) voxel_backward_kernel<DD, true><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, graw, grad_sh, w_max);  \
        else voxel_backward_kernel<DD, false><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, graw, grad_sh, w_max);           \
    } while (0)
    switch (f->scene.sh_degree) {
        case 0: SVR_VB(0); break;
        case 1: SVR_VB(1); break;
        case 2: SVR_VB(2); break;
        default: SVR_VB(3); break;
    }
#undef SVR_VB
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// ---- launchers of the bucketed list build ----
SvrStatus launch_bucket_count(SvrContext* ctx, SvrFrame* f, uint32_t* bcount, int* bigdiff, uint32_t* nonempty,
                              unsigned long long* totals) {
    if (f->scene.n > 0) {
        StageScope scope__(ctx, ST_RECTS);
        const unsigned int g = blocks_for(f->scene.n, 256);
        ushort4* r = reinterpret_cast<ushort4*>(f->rects);
        float4* col = reinterpret_cast<float4*>(f->rgbm);
        switch (f->scene.sh_degree) {
            case 0: rect_bucket_count_kernel<0><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, f->tile_masks, r, bcount, bigdiff, totals, col, reinterpret_cast<float4*>(f->packed), reinterpret_cast<ushort4*>(f->rects_tight)); break;
            case 1: rect_bucket_count_kernel<1><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, f->tile_masks, r, bcount, bigdiff, totals, col, reinterpret_cast<float4*>(f->packed), reinterpret_cast<ushort4*>(f->rects_tight)); break;
            case 2: rect_bucket_count_kernel<2><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, f->tile_masks, r, bcount, bigdiff, totals, col, reinterpret_cast<float4*>(f->packed), reinterpret_cast<ushort4*>(f->rects_tight)); break;
            default: rect_bucket_count_kernel<3><<<g, 256, 0, ctx->stream>>>(f->scene, f->cam, f->tile_masks, r, bcount, bigdiff, totals, col, reinterpret_cast<float4*>(f->packed), reinterpret_cast<ushort4*>(f->rects_tight)); break;
        }
        ctx->launches += 1;
    }
    {
        StageScope scope__(ctx, ST_SCAN);
        // more than 48 KB of dynamic shared memory above 12 288 grid points (about 3 Mpixel): opt in (per device, every call)
        SVR_CUDA(ctx, cudaFuncSetAttribute(bucket_scan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SVR_SCAN_SMEM_MAX));
        bucket_scan_kernel<<<1, 1024, sizeof(int) * (size_t)(f->cam.tiles_x + 1) * (f->cam.tiles_y + 1), ctx->stream>>>(f->tile_masks, bigdiff, f->cam.tiles_x, f->cam.tiles_y, bcount, f->ranges,
                                                        nonempty, totals);
        ctx->launches += 1;
    }
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_bucket_scatter(SvrContext* ctx, SvrFrame* f, uint32_t* cursor, uint64_t* ent, int vb, uint32_t* big_list,
                                unsigned int* big_count) {
    StageScope scope__(ctx, ST_EMIT);
    const ushort4* r = reinterpret_cast<const ushort4*>(f->rects);
    scatter_small_kernel<<<blocks_for(f->scene.n, 256), 256, 0, ctx->stream>>>(f->scene, f->cam, r, f->tile_masks, cursor, ent, vb,
                                                                              big_list, big_count);
    scatter_big_kernel<<<148 * 4, 256, 0, ctx->stream>>>(f->scene, f->cam, r, f->tile_masks, cursor, ent, vb, big_list, big_count);
    ctx->launches += 2;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_bucket_sort(SvrContext* ctx, SvrFrame* f, uint64_t* ent, const uint32_t* nonempty, const unsigned long long* totals,
                             unsigned int* work, int vb) {
    StageScope scope__(ctx, ST_SORT);
    const int smem_small = 2 * SORT_CAP_SMALL * (int)sizeof(uint64_t) + (128 / 32) * 256 * (int)sizeof(uint16_t);
    const int smem_mid = 2 * SORT_CAP * (int)sizeof(uint64_t) + (SORT_THREADS2 / 32) * 256 * (int)sizeof(uint16_t);
    const int smem_big = 2 * SORT_CAP_BIG * (int)sizeof(uint64_t) + (1024 / 32) * 256 * (int)sizeof(uint16_t);
    // a function attribute is per device: set on every call (cheap), so a second context on another GPU gets it too
    SVR_CUDA(ctx, cudaFuncSetAttribute(bucket_sort_kernel<128, SORT_CAP_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_small));
    SVR_CUDA(ctx, cudaFuncSetAttribute(bucket_sort_kernel<SORT_THREADS2, SORT_CAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_mid));
    SVR_CUDA(ctx, cudaFuncSetAttribute(bucket_sort_kernel<1024, SORT_CAP_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_big));
    // three block shapes so that the fixed cost of a pass (counter reset, scan) scales with the bucket; work[0..2] = fetch counters
    const int cb = 3 * f->scene.max_level;
    // The three classes are independent: the largest and the smallest run on the second stream beside the middle one
    // (each alone leaves SMs idle in its tail).
    SVR_CUDA(ctx, cudaEventRecord(ctx->fork_ev, ctx->stream));
    SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->aux, ctx->fork_ev, 0));
    bucket_sort_kernel<1024, SORT_CAP_BIG><<<148, 1024, smem_big, ctx->aux>>>(ent, f->ranges, nonempty, totals, work, 0, cb, vb, f->keys, f->vals);
    bucket_sort_kernel<SORT_THREADS2, SORT_CAP><<<148 * 2, SORT_THREADS2, smem_mid, ctx->stream>>>(ent, f->ranges, nonempty, totals, work + 1, 1, cb, vb,
                                                                                                    f->keys, f->vals);
    bucket_sort_kernel<128, SORT_CAP_SMALL><<<148 * 8, 128, smem_small, ctx->aux>>>(ent, f->ranges, nonempty, totals, work + 2, 2, cb, vb, f->keys,
                                                                                   f->vals);
    SVR_CUDA(ctx, cudaEventRecord(ctx->sort_ev, ctx->aux));
    SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->sort_ev, 0));
    ctx->launches += 3;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

// rectangles in list order + longest-list-first tile order (the ranges themselves come from the bucket scan)
SvrStatus launch_lists_finish(SvrContext* ctx, SvrFrame* f, bool fork) {
    // Two one-block kernels that read only the ranges: with `fork` they are queued on the second stream (after the
    // allocations queued so far) and run beside the scatter and the sort; launch_lists_join makes the main stream wait.
    cudaStream_t st = ctx->stream;
    if (fork) {
        SVR_CUDA(ctx, cudaEventRecord(ctx->fork_ev, ctx->stream));
        SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->aux, ctx->fork_ev, 0));
        st = ctx->aux;
    }
    tile_order_kernel<<<1, 1024, 0, st>>>(f->ranges, f->n_tiles, f->tile_order + f->n_tiles, f->tile_order);
    ctx->launches += 1;
    if (f->trav_off) {
        trav_offsets_kernel<<<1, 1024, 0, st>>>(f->tile_order + f->n_tiles, f->n_tiles, f->trav_off);
        ctx->launches += 1;
    }
    if (fork) SVR_CUDA(ctx, cudaEventRecord(ctx->lists_ev, ctx->aux));
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}

SvrStatus launch_lists_join(SvrContext* ctx) {
    StageScope scope__(ctx, ST_RANGES);
    SVR_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->lists_ev, 0));
    return SVR_OK;
}
