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
__device__ __forceinline__ ushort4 voxel_rect(const SceneDev& s, const CamDev& c, uint2 q) {
    const ushort4 culled = make_ushort4(0xFFFF, 0xFFFF, 0, 0);
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
                                                     uint32_t* __restrict__ ranges, const uint32_t* __restrict__ vals,
                                                     const uint2* __restrict__ rects, uint2* __restrict__ rects_sorted) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    rects_sorted[i] = __ldg(rects + vals[i]);     // rectangle in list order: the compositing cull reads it coalesced
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

// ---- a3: per-view voxel colour (R6) -------------------------------------------------------------------
// c_v = max(0, 0.5 + sum_i Y_i(dir_v) sh[v,i,:]); rgbm[v] = (r, g, b, clamp-mask bits).
template <int DEG>
__global__ void __launch_bounds__(256) voxel_color_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                          float4* __restrict__ rgbm) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    ushort4 r = rects[v];
    if (r.x > r.z) return;                                   // not visible in this view: never read
    constexpr int NB = (DEG + 1) * (DEG + 1);
    float dx, dy, dz, Y[NB];
    voxel_dir_dev(s, c, reinterpret_cast<const uint2*>(s.ijkl)[v], dx, dy, dz);
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
    rgbm[v] = make_float4(fmaxf(acc[0], 0.f), fmaxf(acc[1], 0.f), fmaxf(acc[2], 0.f), __uint_as_float(mask));
}

// ---- a10: per-voxel backward finalize ---------------------------------------------------------------
// (i) corner gradients from the polynomial-coefficient gradients the compositing kernel accumulated:
//     coef = A raw (see composite.cu) => grad_raw += A^T grad_coef;
// (ii) grad_sh[v,i,ch] += Y_i(dir_v) * grad_rgb[v,ch] * [c_v,ch > 0] (zero sub-gradient at the clamp).
// Consumed scratch entries are re-zeroed, so the scratch buffers stay all-zero between calls.
template <int DEG>
__global__ void __launch_bounds__(128) voxel_backward_kernel(SceneDev s, CamDev c, const ushort4* __restrict__ rects,
                                                             const float4* __restrict__ rgbm, float4* __restrict__ grad_coef,
                                                             float4* __restrict__ grad_rgb, float4* __restrict__ grad_raw,
                                                             float* __restrict__ grad_sh) {
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
    bool sh_active = false;
    if (vis) {
        float4 ga = grad_coef[2 * v], gb = grad_coef[2 * v + 1];
        if (ga.x != 0.f || ga.y != 0.f || ga.z != 0.f || ga.w != 0.f || gb.x != 0.f || gb.y != 0.f || gb.z != 0.f || gb.w != 0.f) {
            grad_coef[2 * v] = make_float4(0.f, 0.f, 0.f, 0.f);
            grad_coef[2 * v + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
            const float g0 = ga.x, gx = ga.y, gy = ga.z, gz = ga.w, gxy = gb.x, gxz = gb.y, gyz = gb.z, gxyz = gb.w;
            float4 ra = grad_raw[2 * v], rb = grad_raw[2 * v + 1];
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
        }
        float4 g = grad_rgb[v];
        if (g.x != 0.f || g.y != 0.f || g.z != 0.f) {
            grad_rgb[v] = make_float4(0.f, 0.f, 0.f, 0.f);
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
    const unsigned amask = __ballot_sync(0xffffffffu, sh_active);
    if (amask == 0u) return;
    __syncwarp();
    // cooperative read-modify-write of the warp's contiguous grad_sh block, skipping untouched voxels
    const int nvox = (int)min((int64_t)32, s.n - v0);
    if (ROW % 4 == 0) {
        float4* p4 = reinterpret_cast<float4*>(grad_sh + v0 * ROW);
        for (int e = lane; e < nvox * (ROW / 4); e += 32) {
            int vv = e / (ROW / 4);
            if (!((amask >> vv) & 1u)) continue;
            int f0 = (e - vv * (ROW / 4)) * 4;
            float4 t = p4[e];
            float tv[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                int idx = f0 + k;
                tv[k] = fmaf(Ysm[warp][vv][idx / 3], gsm[warp][vv][idx % 3], tv[k]);
            }
            p4[e] = make_float4(tv[0], tv[1], tv[2], tv[3]);
        }
    } else {
        float* p = grad_sh + v0 * ROW;
        for (int e = lane; e < nvox * ROW; e += 32) {
            int vv = e / ROW;
            if (!((amask >> vv) & 1u)) continue;
            int idx = e - vv * ROW;
            p[e] = fmaf(Ysm[warp][vv][idx / 3], gsm[warp][vv][idx % 3], p[e]);
        }
    }
}

inline unsigned int blocks_for(int64_t n, int bs) { return (unsigned int)((n + bs - 1) / bs); }

}  // namespace

SvrStatus launch_tile_masks(SvrContext* ctx, SvrFrame* f) {
    StageScope scope__(ctx, ST_TILE_MASKS);
    dim3 grid(f->cam.tiles_x, f->cam.tiles_y), block(SVR_TILE, SVR_TILE);
    tile_mask_kernel<<<grid, block, 0, ctx->stream>>>(f->cam, f->tile_masks);
    sat_kernel<<<1, 256, 0, ctx->stream>>>(f->tile_masks, f->sat, f->cam.tiles_x, f->cam.tiles_y);
    ctx->launches += 2;
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
            f->keys, f->n_entries, 3 * f->scene.max_level, f->ranges, f->vals, reinterpret_cast<const uint2*>(f->rects),
            reinterpret_cast<uint2*>(f->rects_sorted));
        ctx->launches += 1;
    }
    tile_order_kernel<<<1, 1024, 0, ctx->stream>>>(f->ranges, f->n_tiles, f->tile_order + f->n_tiles, f->tile_order);
    ctx->launches += 1;
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

SvrStatus launch_sh_backward(SvrContext* ctx, const SvrFrame* f, float* grad_coef, float* grad_rgb, float* grad_raw, float* grad_sh) {
    StageScope scope__(ctx, ST_SH_BACKWARD);
    if (f->scene.n == 0) return SVR_OK;
    unsigned int g = blocks_for(f->scene.n, 128);
    const ushort4* r = reinterpret_cast<const ushort4*>(f->rects);
    const float4* rgbm = reinterpret_cast<const float4*>(f->rgbm);
    float4* gc = reinterpret_cast<float4*>(grad_coef);
    float4* gr = reinterpret_cast<float4*>(grad_rgb);
    float4* graw = reinterpret_cast<float4*>(grad_raw);
    switch (f->scene.sh_degree) {
        case 0: voxel_backward_kernel<0><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, gr, graw, grad_sh); break;
        case 1: voxel_backward_kernel<1><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, gr, graw, grad_sh); break;
        case 2: voxel_backward_kernel<2><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, gr, graw, grad_sh); break;
        default: voxel_backward_kernel<3><<<g, 128, 0, ctx->stream>>>(f->scene, f->cam, r, rgbm, gc, gr, graw, grad_sh); break;
    }
    ctx->launches += 1;
    SVR_CUDA(ctx, cudaGetLastError());
    return SVR_OK;
}
