// Depth-aware quantile pruning (Sec. IV-C, eqs. 11-12, guards i-iii; R11) and the
// stable compaction of per-voxel rows. All kernels stream over the voxels (HBM-bound, a few bytes per voxel and pass).
// Everything that decides an integer (bin, rank, threshold, cap) is computed with individually rounded float32
// operations in the order the specification states, or in integer arithmetic, so the keep mask is bit-exact against
// the oracle. Quantiles are exact order statistics: 11 + 11 + 10-bit radix select on the float bit pattern of w_max
// (non-negative floats order like their bit patterns), all depth bins at once.
#include <cmath>
#include <cstring>

#include "svr_internal.cuh"

namespace {

constexpr int MAX_CAMS = 64;
constexpr int MAX_BINS = 64;
constexpr int HBINS = 2048;
constexpr unsigned FULL = 0xffffffffu;

struct PruneCams {
    int n;
    float r2[MAX_CAMS][3];    // third row of R
    float t2[MAX_CAMS];
    float fx[MAX_CAMS];
};

// Per-bin selection state (device): rank (1-based, within the current prefix), prefix value, bin size.
struct SelectState {
    uint32_t rank[MAX_BINS + 1];
    uint32_t prefix[MAX_BINS + 1];
    uint32_t size[MAX_BINS + 1];
    uint32_t zlo, zhi;            // smallest / largest finite depth, float bits
    uint32_t n_cand, n_removed;
    uint32_t cap_remaining;       // candidates equal to the cap threshold that still leave
};

__device__ __forceinline__ float voxel_half_and_centre(const SceneDev& s, uint2 q, float* x) {
    const int L = q.y >> 16;
    const float e = __fmul_rn(s.root_edge, __int_as_float((127 - L) << 23));
    x[0] = __fadd_rn(s.root_lo[0], __fmul_rn(__fadd_rn((float)(q.x & 0xFFFF), 0.5f), e));
    x[1] = __fadd_rn(s.root_lo[1], __fmul_rn(__fadd_rn((float)(q.x >> 16), 0.5f), e));
    x[2] = __fadd_rn(s.root_lo[2], __fmul_rn(__fadd_rn((float)(q.y & 0xFFFF), 0.5f), e));
    return __fmul_rn(0.5f, e);
}

// step 1: z_v, delta_v; smallest / largest finite depth
__global__ void __launch_bounds__(256) prune_depth_kernel(SceneDev s, PruneCams cams, float* __restrict__ z_out,
                                                          float* __restrict__ delta_out, SelectState* __restrict__ st) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t lo = 0xFFFFFFFFu, hi = 0u;
    if (v < s.n) {
        float x[3];
        voxel_half_and_centre(s, reinterpret_cast<const uint2*>(s.ijkl)[v], x);
        float z = __int_as_float(0x7f800000), delta = z;
        for (int c = 0; c < cams.n; ++c) {
            const float Z = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(cams.r2[c][0], x[0]), __fmul_rn(cams.r2[c][1], x[1])),
                                                __fmul_rn(cams.r2[c][2], x[2])), cams.t2[c]);
            if (Z > 0.0f && Z < z) { z = Z; delta = __fdiv_rn(Z, cams.fx[c]); }
        }
        z_out[v] = z;
        delta_out[v] = delta;
        if (z < __int_as_float(0x7f800000)) { lo = __float_as_uint(z); hi = lo; }
    }
    // one pair of global atomics per block (per warp they serialise on the two addresses: 0.17 ms for 4 M voxels)
    __shared__ uint32_t blo, bhi;
    if (threadIdx.x == 0) { blo = 0xFFFFFFFFu; bhi = 0u; }
    __syncthreads();
    lo = __reduce_min_sync(FULL, lo);
    hi = __reduce_max_sync(FULL, hi);
    if ((threadIdx.x & 31) == 0) {
        if (lo != 0xFFFFFFFFu) atomicMin(&blo, lo);
        if (hi != 0u) atomicMax(&bhi, hi);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (blo != 0xFFFFFFFFu) atomicMin(&st->zlo, blo);
        if (bhi != 0u) atomicMax(&st->zhi, bhi);
    }
}

// step 2: bin of a depth (integer arithmetic on the bit pattern)
__device__ __forceinline__ int depth_bin(float z, uint32_t zlo, uint32_t zhi, int B) {
    if (!(z < __int_as_float(0x7f800000)) || zlo > zhi) return B - 1;
    const unsigned long long num = (unsigned long long)(min(max(__float_as_uint(z), zlo), zhi) - zlo) * (unsigned long long)B;
    const unsigned long long b = num / ((unsigned long long)(zhi - zlo) + 1ull);
    return (int)min((unsigned long long)(B - 1), b);
}

__global__ void __launch_bounds__(256) prune_bins_kernel(int64_t n, const float* __restrict__ z, const SelectState* __restrict__ st,
                                                         int B, uint8_t* __restrict__ bins) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n) bins[v] = (uint8_t)depth_bin(z[v], st->zlo, st->zhi, B);
}

// One histogram pass of the radix select: digit = (key >> shift) & (HBINS-1 or 1023) of the keys whose higher bits
// equal the bin's prefix. `flags` (may be NULL) restricts the pass to flagged voxels (cap selection: one bin).
__global__ void __launch_bounds__(256) select_hist_kernel(int64_t n, const float* __restrict__ w_max, const uint8_t* __restrict__ bins,
                                                          const uint8_t* __restrict__ flags, const SelectState* __restrict__ st,
                                                          int shift, uint32_t mask, int hi_shift, uint32_t* __restrict__ hist) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t slot = 0xFFFFFFFFu;
    if (v < n && (flags == nullptr || flags[v])) {
        const uint32_t key = __float_as_uint(w_max[v]);
        const int b = bins ? bins[v] : 0;
        if (hi_shift >= 32 || (key >> hi_shift) == st->prefix[b]) slot = (uint32_t)b * HBINS + ((key >> shift) & mask);
    }
    // Equal keys are common (never-seen voxels all have w_max = 0, so one histogram slot receives most of the voxels):
    // aggregate per warp (match_any), then per block in a small tagged shared-memory table (slot mod 64; a warp whose
    // slot loses the tag race goes to global memory directly), and flush the table once per block.
    __shared__ uint32_t tag[64], cnt[64];
    if (threadIdx.x < 64) { tag[threadIdx.x] = 0xFFFFFFFFu; cnt[threadIdx.x] = 0u; }
    __syncthreads();
    const unsigned peers = __match_any_sync(FULL, slot);
    if (slot != 0xFFFFFFFFu && (peers & ((1u << (threadIdx.x & 31)) - 1u)) == 0u) {
        const uint32_t h = slot & 63u, c = (uint32_t)__popc(peers);
        const uint32_t prev = atomicCAS(&tag[h], 0xFFFFFFFFu, slot);
        if (prev == 0xFFFFFFFFu || prev == slot) atomicAdd(&cnt[h], c);
        else atomicAdd(&hist[slot], c);
    }
    __syncthreads();
    if (threadIdx.x < 64 && cnt[threadIdx.x]) atomicAdd(&hist[tag[threadIdx.x]], cnt[threadIdx.x]);
}

// One block per bin: find the digit that holds the bin's rank; refine prefix and rank; clear the histogram row.
// first != 0: the bin size is the row sum and the rank comes from q_b (eq. 12) or, for the cap (q_near < 0), from
// min(cap, size).
__global__ void __launch_bounds__(1024) select_digit_kernel(SelectState* __restrict__ st, uint32_t* __restrict__ hist, int digit_bits, int first,
                                                            int B, float q_near, float q_far, uint32_t cap) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t s_rank, s_total;
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t* row = hist + (size_t)b * HBINS;
    const int nd = 1 << digit_bits;
    const uint32_t c0 = (2 * tid < nd) ? row[2 * tid] : 0u, c1 = (2 * tid + 1 < nd) ? row[2 * tid + 1] : 0u;
    uint32_t inc = c0 + c1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = wsum[lane], a = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(FULL, a, o);
            if (lane >= o) a += t;
        }
        wsum[lane] = a - w;
        if (lane == 31) s_total = a;
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t rank = st->rank[b];
        if (first) {
            const uint32_t size = s_total;
            st->size[b] = size;
            if (q_near < 0.0f) {
                rank = min(cap, size);                                   // cap selection: the cap-th smallest candidate
            } else {
                const float frac = __fdiv_rn((float)b, (float)max(B - 1, 1));
                const float q = __fadd_rn(q_near, __fmul_rn(__fsub_rn(q_far, q_near), frac));
                rank = (uint32_t)max(1.0f, ceilf(__fmul_rn(q, (float)size)));
                rank = min(rank, size);                                  // size == 0 -> rank 0: the bin has no threshold
            }
            st->prefix[b] = 0u;
        }
        s_rank = rank;
    }
    __syncthreads();
    const uint32_t rank = s_rank;
    const uint32_t before = wsum[warp] + inc - (c0 + c1);                // keys with a smaller digit pair
    if (rank > 0u) {
        if (before < rank && rank <= before + c0) {
            st->prefix[b] = (st->prefix[b] << digit_bits) | (uint32_t)(2 * tid);
            st->rank[b] = rank - before;
        } else if (before + c0 < rank && rank <= before + c0 + c1) {
            st->prefix[b] = (st->prefix[b] << digit_bits) | (uint32_t)(2 * tid + 1);
            st->rank[b] = rank - before - c0;
        }
    } else if (tid == 0) {
        st->rank[b] = 0u;
    }
    if (2 * tid < nd) row[2 * tid] = 0u;
    if (2 * tid + 1 < nd) row[2 * tid + 1] = 0u;
}

// steps 3-5: inside score, EMA + hysteresis (guard i), protection (guard ii), candidates
__global__ void __launch_bounds__(256) prune_state_kernel(SceneDev s, const float* __restrict__ w_max, const uint8_t* __restrict__ bins,
                                                          const float* __restrict__ delta, const SelectState* __restrict__ st,
                                                          SvrPruneOpts o, float* __restrict__ ema, uint8_t* __restrict__ state,
                                                          uint8_t* __restrict__ cand, SelectState* __restrict__ st_cap,
                                                          uint8_t* __restrict__ seed) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool c = false;
    if (v < s.n) {
        const float w = w_max[v];
        const int b = bins[v];
        // tau_b: the selected bit pattern; an empty bin never gets here
        const bool inside = __float_as_uint(w) > st->prefix[b];
        const float m = __fadd_rn(__fmul_rn(__fsub_rn(1.0f, o.ema_alpha), ema[v]), __fmul_rn(o.ema_alpha, inside ? 1.0f : 0.0f));
        uint8_t sv = state[v];
        if (m < o.m_low) sv = 0;
        else if (m > o.m_high) sv = 1;
        ema[v] = m;
        state[v] = sv;
        float x[3];
        const float half = voxel_half_and_centre(s, reinterpret_cast<const uint2*>(s.ijkl)[v], x);
        const bool prot = (half < __fmul_rn(o.kappa, delta[v])) || (w >= o.w_keep);
        if (seed != nullptr) {                 // keep-halo: the seeds are dilated first, prune_cand_kernel decides afterwards
            seed[v] = prot ? 1 : 0;
        } else {
            c = (sv == 0) && !prot;
            cand[v] = c ? 1 : 0;
        }
    }
    const unsigned m = __ballot_sync(FULL, c);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&st_cap->n_cand, (uint32_t)__popc(m));
}

// ---- guard ii as a dilation ("keep-halo"): face neighbours through a hash table of the leaves ----
// key of a cell: level, ix, iy, iz (16 bits each); the table maps the key of every leaf to its index (open addressing, linear
// probing, capacity a power of two >= 2 n).
constexpr uint64_t HASH_EMPTY = ~0ull;
__device__ __forceinline__ uint64_t cell_key(uint32_t L, uint32_t x, uint32_t y, uint32_t z) {
    return ((uint64_t)L << 48) | ((uint64_t)x << 32) | ((uint64_t)y << 16) | (uint64_t)z;
}
__device__ __forceinline__ uint32_t hash_slot(uint64_t k, uint32_t mask) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdull; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ull; k ^= k >> 33;
    return (uint32_t)k & mask;
}
__global__ void __launch_bounds__(256) halo_insert_kernel(SceneDev s, unsigned long long* __restrict__ hkeys, uint32_t* __restrict__ hvals,
                                                          uint32_t mask) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    const uint2 q = reinterpret_cast<const uint2*>(s.ijkl)[v];
    const uint64_t k = cell_key(q.y >> 16, q.x & 0xFFFF, q.x >> 16, q.y & 0xFFFF);
    uint32_t i = hash_slot(k, mask);
    while (true) {
        const unsigned long long old = atomicCAS(&hkeys[i], (unsigned long long)HASH_EMPTY, (unsigned long long)k);
        if (old == HASH_EMPTY || old == k) { hvals[i] = (uint32_t)v; return; }
        i = (i + 1) & mask;
    }
}
__device__ __forceinline__ int64_t hash_find(const unsigned long long* __restrict__ hkeys, const uint32_t* __restrict__ hvals, uint32_t mask,
                                             uint64_t k) {
    uint32_t i = hash_slot(k, mask);
    while (true) {
        const unsigned long long cur = hkeys[i];
        if (cur == k) return (int64_t)hvals[i];
        if (cur == HASH_EMPTY) return -1;
        i = (i + 1) & mask;
    }
}
// One dilation step: out (initialised with a copy of in) |= neighbours of in. Every pair of face neighbours is visited from
// the side of its finer (or equal) leaf a: b = the leaf covering the cell of a's size beside one of a's faces, i.e. that cell
// or one of its ancestors (leaves are disjoint: at most one of them is a leaf).
__global__ void __launch_bounds__(256) halo_dilate_kernel(SceneDev s, const unsigned long long* __restrict__ hkeys,
                                                          const uint32_t* __restrict__ hvals, uint32_t mask, const uint8_t* __restrict__ in,
                                                          uint8_t* __restrict__ out) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    const uint2 q = reinterpret_cast<const uint2*>(s.ijkl)[v];
    const int L = (int)(q.y >> 16);
    const int c0[3] = {(int)(q.x & 0xFFFF), (int)(q.x >> 16), (int)(q.y & 0xFFFF)};
    const bool mine = in[v] != 0;
    bool got = false;
    for (int face = 0; face < 6; ++face) {
        int c[3] = {c0[0], c0[1], c0[2]};
        c[face >> 1] += (face & 1) ? 1 : -1;
        if (c[face >> 1] < 0 || c[face >> 1] >= (1 << L)) continue;              // outside the root cube
        for (int up = 0; up <= L; ++up) {
            const int64_t b = hash_find(hkeys, hvals, mask, cell_key((uint32_t)(L - up), (uint32_t)(c[0] >> up), (uint32_t)(c[1] >> up), (uint32_t)(c[2] >> up)));
            if (b >= 0) {
                if (mine) out[b] = 1;
                got = got || in[b] != 0;
                break;
            }
        }
    }
    if (got) out[v] = 1;
}
__global__ void __launch_bounds__(256) prune_cand_kernel(int64_t n, const uint8_t* __restrict__ state, const uint8_t* __restrict__ prot,
                                                         uint8_t* __restrict__ cand, SelectState* __restrict__ st_cap) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool c = false;
    if (v < n) { c = state[v] == 0 && prot[v] == 0; cand[v] = c ? 1 : 0; }
    const unsigned m = __ballot_sync(FULL, c);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&st_cap->n_cand, (uint32_t)__popc(m));
}

// guard iii, part 1: eq[v] = 1 for candidates whose w_max equals the cap threshold (their exclusive prefix count
// decides which of them still leave); also counts the candidates strictly below the threshold.
__global__ void __launch_bounds__(256) prune_cap_flags_kernel(int64_t n, const float* __restrict__ w_max, const uint8_t* __restrict__ cand,
                                                              SelectState* __restrict__ st_cap, uint32_t* __restrict__ eq) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool less = false;
    if (v <= n) {
        uint32_t e = 0;
        if (v < n && cand[v] && st_cap->rank[0] > 0u) {
            const uint32_t key = __float_as_uint(w_max[v]);
            e = (key == st_cap->prefix[0]);
            less = key < st_cap->prefix[0];
        }
        eq[v] = e;
    }
    const unsigned m = __ballot_sync(FULL, less);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&st_cap->n_removed, (uint32_t)__popc(m));   // so far: the ones strictly below
}

// guard iii, part 2: keep mask. A candidate leaves if it is below the threshold, or equal to it and among the first
// (cap - #below) such candidates in index order.
__global__ void __launch_bounds__(256) prune_keep_kernel(int64_t n, const float* __restrict__ w_max, const uint8_t* __restrict__ cand,
                                                         const SelectState* __restrict__ st_cap, const uint32_t* __restrict__ eq_prefix,
                                                         uint32_t cap, uint8_t* __restrict__ keep, uint32_t* __restrict__ n_removed_total) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool rem = false;
    if (v < n) {
        if (cand[v] && st_cap->rank[0] > 0u) {
            const uint32_t key = __float_as_uint(w_max[v]), thr = st_cap->prefix[0];
            const uint32_t below = st_cap->n_removed;                       // candidates strictly below the threshold
            const uint32_t quota = min(cap, st_cap->size[0]) - below;      // equal-valued candidates that still leave
            rem = key < thr || (key == thr && eq_prefix[v] < quota);
        }
        keep[v] = rem ? 0 : 1;
    }
    const unsigned m = __ballot_sync(FULL, rem);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_removed_total, (uint32_t)__popc(m));
}

// ---- stable compaction of rows ----
__global__ void __launch_bounds__(256) keep_to_counts_kernel(int64_t n, const uint8_t* __restrict__ keep, uint32_t* __restrict__ counts) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v <= n) counts[v] = (v < n && keep[v]) ? 1u : 0u;
}

template <typename T>
__global__ void __launch_bounds__(256) compact_rows_kernel(int64_t n, const uint8_t* __restrict__ keep, const uint32_t* __restrict__ offs,
                                                           const T* __restrict__ src, T* __restrict__ dst, int words) {
    // one thread per word of a row: consecutive threads copy consecutive words (coalesced for wide rows)
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t v = i / words;
    if (v >= n || !keep[v]) return;
    const int w = (int)(i - v * words);
    dst[(size_t)offs[v] * words + w] = src[(size_t)v * words + w];
}

// ---- priority-driven subdivision (Sec. IV-D, eqs. 13-16; R12) ----
__global__ void __launch_bounds__(256) subdiv_finite_kernel(int64_t n, const float* __restrict__ z, uint8_t* __restrict__ finite) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n) finite[v] = (z[v] < __int_as_float(0x7f800000)) ? 1 : 0;
}

// eq. 13 eligibility, eq. 14 robust depth normalisation, eqs. 15-16 priority; key = ~bits(priority) so that the
// "smallest keys first" selection of the cap machinery picks the HIGHEST priorities (priority >= 0 required).
__global__ void __launch_bounds__(256) subdiv_priority_kernel(SceneDev s, const float* __restrict__ z, const float* __restrict__ delta,
                                                              const float* __restrict__ P, const SelectState* __restrict__ st5,
                                                              const SelectState* __restrict__ st95, int use_current, float z_p5, float z_p95,
                                                              float kappa, float beta, int max_level, float* __restrict__ priority,
                                                              float* __restrict__ key, uint8_t* __restrict__ cand) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= s.n) return;
    float a = z_p5, b = z_p95;
    if (use_current) {
        a = (st5->size[0] > 0u) ? __uint_as_float(st5->prefix[0]) : 0.0f;
        b = (st95->size[0] > 0u) ? __uint_as_float(st95->prefix[0]) : 0.0f;
    }
    const uint2 q = reinterpret_cast<const uint2*>(s.ijkl)[v];
    float x[3];
    const float half = voxel_half_and_centre(s, q, x);
    const float zv = z[v];
    const bool finite = zv < __int_as_float(0x7f800000);
    const bool elig = finite && ((int)(q.y >> 16) < max_level) && (half > __fmul_rn(kappa, delta[v]));
    const float den = __fsub_rn(b, a);
    float zt = 0.0f;
    if (finite && den > 0.0f) zt = fminf(fmaxf(__fdiv_rn(__fsub_rn(zv, a), den), 0.0f), 1.0f);
    const float pr = __fmul_rn(P[v], __fadd_rn(1.0f, __fmul_rn(beta, zt)));
    if (priority) priority[v] = pr;
    key[v] = __uint_as_float(~__float_as_uint(pr));
    cand[v] = elig ? 1 : 0;
}

__global__ void __launch_bounds__(256) subdiv_invert_kernel(int64_t n, const uint8_t* __restrict__ keep, uint8_t* __restrict__ split) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n) split[v] = keep[v] ? 0 : 1;
}

__global__ void __launch_bounds__(256) split_to_counts_kernel(int64_t n, const uint8_t* __restrict__ split, uint32_t* __restrict__ counts) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v <= n) counts[v] = (v < n && split[v]) ? 1u : 0u;
}

__device__ __forceinline__ float mix_half(float a, float b, int t2) {   // parent coordinate t = t2 / 2 in {0, 1/2, 1}
    return t2 == 0 ? a : (t2 == 2 ? b : __fmul_rn(0.5f, __fadd_rn(a, b)));
}

// cells and corner raws: survivors keep their row (stable), a split voxel writes its 8 children after all survivors,
// grouped by parent in parent order, child order c = bx + 2 by + 4 bz; child raws = the parent's trilinear field at the
// child's corners, interpolated along x, then y, then z.
__global__ void __launch_bounds__(256) subdiv_cells_kernel(int64_t n, const uint8_t* __restrict__ split, const uint32_t* __restrict__ offs,
                                                           const uint2* __restrict__ ijkl, const float4* __restrict__ raw,
                                                           uint2* __restrict__ ijkl_out, float4* __restrict__ raw_out) {
    const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    const uint32_t r = offs[v], n_split = offs[n];
    const uint2 q = ijkl[v];
    const float4 ra = raw[2 * v], rb = raw[2 * v + 1];
    if (!split[v]) {
        const size_t d = (size_t)v - r;
        ijkl_out[d] = q;
        raw_out[2 * d] = ra;
        raw_out[2 * d + 1] = rb;
        return;
    }
    const float p[8] = {ra.x, ra.y, ra.z, ra.w, rb.x, rb.y, rb.z, rb.w};
    const uint32_t ix = q.x & 0xFFFF, iy = q.x >> 16, iz = q.y & 0xFFFF, L = q.y >> 16;
    const size_t base = (size_t)(n - n_split) + 8 * (size_t)r;
#pragma unroll
    for (int o = 0; o < 8; ++o) {
        const int ox = o & 1, oy = (o >> 1) & 1, oz = o >> 2;
        float c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int tx = ox + (k & 1), ty = oy + ((k >> 1) & 1), tz = oz + (k >> 2);
            const float x00 = mix_half(p[0], p[1], tx), x10 = mix_half(p[2], p[3], tx);
            const float x01 = mix_half(p[4], p[5], tx), x11 = mix_half(p[6], p[7], tx);
            c[k] = mix_half(mix_half(x00, x10, ty), mix_half(x01, x11, ty), tz);
        }
        ijkl_out[base + o] = make_uint2((2 * ix + ox) | ((2 * iy + oy) << 16), (2 * iz + oz) | ((L + 1) << 16));
        raw_out[2 * (base + o)] = make_float4(c[0], c[1], c[2], c[3]);
        raw_out[2 * (base + o) + 1] = make_float4(c[4], c[5], c[6], c[7]);
    }
}

// SH rows: one thread per (voxel, 4-byte word); a split voxel's row is copied to its 8 children
__global__ void __launch_bounds__(256) subdiv_sh_kernel(int64_t n, int words, const uint8_t* __restrict__ split, const uint32_t* __restrict__ offs,
                                                        const uint32_t* __restrict__ sh, uint32_t* __restrict__ sh_out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t v = i / words;
    if (v >= n) return;
    const int w = (int)(i - v * words);
    const uint32_t val = sh[i], r = offs[v];
    if (!split[v]) { sh_out[((size_t)v - r) * words + w] = val; return; }
    const size_t base = (size_t)(n - offs[n]) + 8 * (size_t)r;
#pragma unroll
    for (int o = 0; o < 8; ++o) sh_out[(base + o) * words + w] = val;
}

// per-voxel side-state rows through a split (R17): one thread per (voxel, word of type T); an unsplit voxel's row moves
// to its new index, a split voxel's 8 children get the parent's row (zero == 0) or zeros
template <typename T>
__global__ void __launch_bounds__(256) subdiv_rows_kernel(int64_t n, int words, const uint8_t* __restrict__ split, const uint32_t* __restrict__ offs,
                                                          const T* __restrict__ src, T* __restrict__ dst, int zero) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t v = i / words;
    if (v >= n) return;
    const int w = (int)(i - v * words);
    const uint32_t r = offs[v];
    if (!split[v]) { dst[((size_t)v - r) * words + w] = src[i]; return; }
    T val = T();
    if (!zero) val = src[i];
    const size_t base = (size_t)(n - offs[n]) + 8 * (size_t)r;
#pragma unroll
    for (int o = 0; o < 8; ++o) dst[(base + o) * words + w] = val;
}

SceneDev scene_of(const SvrVoxels* vox) {
    SceneDev s{};
    s.n = vox->n; s.sh_degree = vox->sh_degree; s.n_basis = (vox->sh_degree + 1) * (vox->sh_degree + 1); s.max_level = vox->max_level;
    for (int a = 0; a < 3; ++a) s.root_lo[a] = vox->root_lo[a];
    s.root_edge = vox->root_edge; s.ijkl = vox->ijkl; s.raw = vox->raw_density; s.sh = vox->sh;
    return s;
}

PruneCams cams_of(const SvrCamera* cams_host, int n_cams) {
    PruneCams cams{};
    cams.n = n_cams;
    for (int c = 0; c < n_cams; ++c) {
        for (int a = 0; a < 3; ++a) cams.r2[c][a] = cams_host[c].R[6 + a];
        cams.t2[c] = cams_host[c].t[2];
        cams.fx[c] = cams_host[c].fx;
    }
    return cams;
}

inline unsigned int nblocks(int64_t n, int bs) { return (unsigned int)((n + bs - 1) / bs); }

}  // namespace

extern "C" {

SvrStatus svr_prune_step(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cams_host, int32_t n_cams, const float* w_max,
                         float* ema, uint8_t* state, const SvrPruneOpts* opts, uint8_t* keep, float* tau_host,
                         int64_t* n_removed_host) {
    SVR_NVTX();
    if (!ctx || !vox || !cams_host || !w_max || !ema || !state || !opts || !keep || !n_removed_host)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n_cams < 1 || n_cams > MAX_CAMS) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "n_cams must be 1..%d", MAX_CAMS);
    if (opts->n_bins < 1 || opts->n_bins > MAX_BINS) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "n_bins must be 1..%d", MAX_BINS);
    if (opts->halo < 0 || opts->halo > 8) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "halo must be 0..8 dilation steps");
    if (vox->n < 0 || vox->n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    // the keep-halo hash table has 2^k >= 2 n slots addressed with 32-bit masks: 2^31 slots at most
    if (opts->halo > 0 && vox->n > ((int64_t)1 << 30))
        return svr_fail(ctx, SVR_ERR_UNSUPPORTED, "keep-halo (halo > 0) supports at most 2^30 voxels, got %lld", (long long)vox->n);
    { int ex = 0; if (!(vox->root_edge > 0.f) || std::frexp(vox->root_edge, &ex) != 0.5f) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "root_edge must be a positive power of two"); }
    *n_removed_host = 0;
    const int64_t n = vox->n;
    const int B = opts->n_bins;
    if (n == 0) {
        if (tau_host) for (int b = 0; b < B; ++b) tau_host[b] = -1.0f;
        return SVR_OK;
    }
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    const SceneDev s = scene_of(vox);
    const PruneCams cams = cams_of(cams_host, n_cams);
    const uint32_t cap = (uint32_t)floorf(opts->cap_fraction * (float)n);

    // workspace: z, delta [n] f32; bins, cand [n] u8; eq, eq_prefix [n+1] u32; hist [B][2048]; two selection states; a counter
    float *z = nullptr, *delta = nullptr;
    uint8_t *bins = nullptr, *cand = nullptr;
    uint32_t *eq = nullptr, *eqp = nullptr, *hist = nullptr;
    SelectState* st = nullptr;      // st[0]: per-bin quantiles, st[1]: the cap
    unsigned long long* hkeys = nullptr;     // keep-halo (opts->halo > 0): hash table of the leaves, two protection masks
    uint32_t* hvals = nullptr;
    uint8_t *prot_a = nullptr, *prot_b = nullptr;
    size_t hkb = 0, hvb = 0;
    const size_t fb = sizeof(float) * (size_t)n, ub = (size_t)n, eb = sizeof(uint32_t) * (size_t)(n + 1);
    const size_t hb = sizeof(uint32_t) * (size_t)B * HBINS, sb = 2 * sizeof(SelectState) + 64;
    SvrStatus stt = SVR_OK;
    auto cleanup = [&]() {
        svr_free(ctx, z, fb); svr_free(ctx, delta, fb); svr_free(ctx, bins, ub); svr_free(ctx, cand, ub);
        svr_free(ctx, eq, eb); svr_free(ctx, eqp, eb); svr_free(ctx, hist, hb); svr_free(ctx, st, sb);
        svr_free(ctx, hkeys, hkb); svr_free(ctx, hvals, hvb); svr_free(ctx, prot_a, ub); svr_free(ctx, prot_b, ub);
    };
#define PTRY(call) do { stt = (call); if (stt != SVR_OK) { cleanup(); return stt; } } while (0)
#define PCUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cleanup(); return svr_fail(ctx, SVR_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e__)); } } while (0)
    PTRY(svr_alloc(ctx, (void**)&z, fb)); PTRY(svr_alloc(ctx, (void**)&delta, fb));
    PTRY(svr_alloc(ctx, (void**)&bins, ub)); PTRY(svr_alloc(ctx, (void**)&cand, ub));
    PTRY(svr_alloc(ctx, (void**)&eq, eb)); PTRY(svr_alloc(ctx, (void**)&eqp, eb));
    PTRY(svr_alloc(ctx, (void**)&hist, hb)); PTRY(svr_alloc(ctx, (void**)&st, sb));
    SelectState* st_cap = st + 1;
    uint32_t* n_removed_dev = reinterpret_cast<uint32_t*>(st + 2);
    PCUDA(cudaMemsetAsync(st, 0, sb, ctx->stream));
    PCUDA(cudaMemsetAsync(&st->zlo, 0xFF, sizeof(uint32_t), ctx->stream));
    PCUDA(cudaMemsetAsync(hist, 0, hb, ctx->stream));
    const unsigned int g = nblocks(n, 256);
    prune_depth_kernel<<<g, 256, 0, ctx->stream>>>(s, cams, z, delta, st);
    prune_bins_kernel<<<g, 256, 0, ctx->stream>>>(n, z, st, B, bins);
    // eqs. 11-12: per-bin nearest-rank quantile of w_max, 11 + 11 + 10 bits
    const int shifts[3] = {21, 10, 0}, bits[3] = {11, 11, 10}, his[3] = {32, 21, 10};
    for (int p = 0; p < 3; ++p) {
        select_hist_kernel<<<g, 256, 0, ctx->stream>>>(n, w_max, bins, nullptr, st, shifts[p], (1u << bits[p]) - 1u, his[p], hist);
        select_digit_kernel<<<B, 1024, 0, ctx->stream>>>(st, hist, bits[p], p == 0, B, opts->q_near, opts->q_far, 0u);
    }
    if (opts->halo <= 0) {
        prune_state_kernel<<<g, 256, 0, ctx->stream>>>(s, w_max, bins, delta, st, *opts, ema, state, cand, st_cap, nullptr);
    } else {
        // guard ii as a dilation: seeds -> `halo` dilation steps over the face neighbours -> candidates
        uint64_t capn64 = 1024;
        while (capn64 < 2 * (uint64_t)n) capn64 <<= 1;          // <= 2^31: n <= 2^30 was checked above
        const uint32_t capn = (uint32_t)capn64;
        hkb = sizeof(unsigned long long) * (size_t)capn; hvb = sizeof(uint32_t) * (size_t)capn;
        PTRY(svr_alloc(ctx, (void**)&hkeys, hkb)); PTRY(svr_alloc(ctx, (void**)&hvals, hvb));
        PTRY(svr_alloc(ctx, (void**)&prot_a, ub)); PTRY(svr_alloc(ctx, (void**)&prot_b, ub));
        PCUDA(cudaMemsetAsync(hkeys, 0xFF, hkb, ctx->stream));
        prune_state_kernel<<<g, 256, 0, ctx->stream>>>(s, w_max, bins, delta, st, *opts, ema, state, cand, st_cap, prot_a);
        halo_insert_kernel<<<g, 256, 0, ctx->stream>>>(s, hkeys, hvals, capn - 1u);
        for (int it = 0; it < opts->halo; ++it) {
            PCUDA(cudaMemcpyAsync(prot_b, prot_a, ub, cudaMemcpyDeviceToDevice, ctx->stream));
            halo_dilate_kernel<<<g, 256, 0, ctx->stream>>>(s, hkeys, hvals, capn - 1u, prot_a, prot_b);
            uint8_t* t = prot_a; prot_a = prot_b; prot_b = t;
            ctx->launches += 1;
        }
        prune_cand_kernel<<<g, 256, 0, ctx->stream>>>(n, state, prot_a, cand, st_cap);
        ctx->launches += 2;
    }
    // guard iii: the cap-th smallest candidate
    for (int p = 0; p < 3; ++p) {
        select_hist_kernel<<<g, 256, 0, ctx->stream>>>(n, w_max, nullptr, cand, st_cap, shifts[p], (1u << bits[p]) - 1u, his[p], hist);
        select_digit_kernel<<<1, 1024, 0, ctx->stream>>>(st_cap, hist, bits[p], p == 0, 1, -1.0f, -1.0f, cap);
    }
    prune_cap_flags_kernel<<<nblocks(n + 1, 256), 256, 0, ctx->stream>>>(n, w_max, cand, st_cap, eq);
    ctx->launches += 16;
    PCUDA(cudaGetLastError());
    PTRY(launch_exclusive_scan(ctx, eq, eqp, n + 1));
    prune_keep_kernel<<<g, 256, 0, ctx->stream>>>(n, w_max, cand, st_cap, eqp, cap, keep, n_removed_dev);
    ctx->launches += 1;
    PCUDA(cudaGetLastError());
    // host outputs
    SelectState h{};
    uint32_t removed = 0;
    PCUDA(cudaMemcpyAsync(&h, st, sizeof(SelectState), cudaMemcpyDeviceToHost, ctx->stream));
    PCUDA(cudaMemcpyAsync(&removed, n_removed_dev, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
    PCUDA(cudaStreamSynchronize(ctx->stream));
    *n_removed_host = (int64_t)removed;
    if (tau_host)
        for (int b = 0; b < B; ++b) {
            float t = -1.0f;
            if (h.size[b] > 0) memcpy(&t, &h.prefix[b], sizeof(float));
            tau_host[b] = t;
        }
#undef PTRY
#undef PCUDA
    cleanup();
    return SVR_OK;
}

SvrStatus svr_compact_rows(SvrContext* ctx, const uint8_t* keep, int64_t n, const void* src, void* dst, int64_t row_bytes,
                           int64_t* n_out_host) {
    SVR_NVTX();
    if (!ctx || !keep || !src || !dst) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 0 || n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "row count out of range");
    if (row_bytes < 1 || (row_bytes > 2 && row_bytes % 4 != 0)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "row_bytes must be 1, 2 or a multiple of 4");
    if (n_out_host) *n_out_host = 0;
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    uint32_t *counts = nullptr, *offs = nullptr;
    const size_t eb = sizeof(uint32_t) * (size_t)(n + 1);
    SVR_TRY(svr_alloc(ctx, (void**)&counts, eb));
    SvrStatus stt = svr_alloc(ctx, (void**)&offs, eb);
    if (stt != SVR_OK) { svr_free(ctx, counts, eb); return stt; }
    keep_to_counts_kernel<<<nblocks(n + 1, 256), 256, 0, ctx->stream>>>(n, keep, counts);
    stt = launch_exclusive_scan(ctx, counts, offs, n + 1);
    if (stt == SVR_OK) {
        if (row_bytes == 1)
            compact_rows_kernel<uint8_t><<<nblocks(n, 256), 256, 0, ctx->stream>>>(n, keep, offs, (const uint8_t*)src, (uint8_t*)dst, 1);
        else if (row_bytes == 2)
            compact_rows_kernel<uint16_t><<<nblocks(n, 256), 256, 0, ctx->stream>>>(n, keep, offs, (const uint16_t*)src, (uint16_t*)dst, 1);
        else if (row_bytes % 16 == 0 && ((uintptr_t)src % 16) == 0 && ((uintptr_t)dst % 16) == 0) {
            const int words = (int)(row_bytes / 16);
            compact_rows_kernel<uint4><<<nblocks(n * words, 256), 256, 0, ctx->stream>>>(n, keep, offs, (const uint4*)src, (uint4*)dst, words);
        } else {
            const int words = (int)(row_bytes / 4);
            compact_rows_kernel<uint32_t><<<nblocks(n * words, 256), 256, 0, ctx->stream>>>(n, keep, offs, (const uint32_t*)src, (uint32_t*)dst, words);
        }
        ctx->launches += 2;
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess && n_out_host) {
            uint32_t total = 0;
            e = cudaMemcpyAsync(&total, offs + n, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
            *n_out_host = (int64_t)total;
        }
        if (e != cudaSuccess) stt = svr_fail(ctx, SVR_ERR_CUDA, "compact: %s", cudaGetErrorString(e));
    }
    svr_free(ctx, counts, eb);
    svr_free(ctx, offs, eb);
    return stt;
}

SvrStatus svr_subdivide_select(SvrContext* ctx, const SvrVoxels* vox, const SvrCamera* cams_host, int32_t n_cams,
                               const float* usefulness, const SvrSubdivOpts* opts, uint8_t* split, float* priority,
                               float* z_percentiles_host, int64_t* n_split_host) {
    SVR_NVTX();
    if (!ctx || !vox || !cams_host || !usefulness || !opts || !split || !n_split_host)
        return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n_cams < 1 || n_cams > MAX_CAMS) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "n_cams must be 1..%d", MAX_CAMS);
    if (vox->n < 0 || vox->n >= ((int64_t)1 << 31)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    { int ex = 0; if (!(vox->root_edge > 0.f) || std::frexp(vox->root_edge, &ex) != 0.5f) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "root_edge must be a positive power of two"); }
    if (opts->max_splits < 0) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "max_splits must be >= 0");
    *n_split_host = 0;
    if (z_percentiles_host) z_percentiles_host[0] = z_percentiles_host[1] = 0.0f;
    const int64_t n = vox->n;
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    const SceneDev s = scene_of(vox);
    const PruneCams cams = cams_of(cams_host, n_cams);
    const uint32_t cap = (uint32_t)(opts->max_splits < n ? opts->max_splits : n);

    float *z = nullptr, *delta = nullptr, *key = nullptr;
    uint8_t *finite = nullptr, *cand = nullptr, *keep = nullptr;
    uint32_t *eq = nullptr, *eqp = nullptr, *hist = nullptr;
    SelectState* st = nullptr;      // st[0]: 5th percentile, st[1]: 95th, st[2]: the budget
    const size_t fb = sizeof(float) * (size_t)n, ub = (size_t)n, eb = sizeof(uint32_t) * (size_t)(n + 1);
    const size_t hb = sizeof(uint32_t) * HBINS, sb = 3 * sizeof(SelectState) + 64;
    SvrStatus stt = SVR_OK;
    auto cleanup = [&]() {
        svr_free(ctx, z, fb); svr_free(ctx, delta, fb); svr_free(ctx, key, fb); svr_free(ctx, finite, ub); svr_free(ctx, cand, ub);
        svr_free(ctx, keep, ub); svr_free(ctx, eq, eb); svr_free(ctx, eqp, eb); svr_free(ctx, hist, hb); svr_free(ctx, st, sb);
    };
#define PTRY(call) do { stt = (call); if (stt != SVR_OK) { cleanup(); return stt; } } while (0)
#define PCUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cleanup(); return svr_fail(ctx, SVR_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e__)); } } while (0)
    PTRY(svr_alloc(ctx, (void**)&z, fb)); PTRY(svr_alloc(ctx, (void**)&delta, fb)); PTRY(svr_alloc(ctx, (void**)&key, fb));
    PTRY(svr_alloc(ctx, (void**)&finite, ub)); PTRY(svr_alloc(ctx, (void**)&cand, ub)); PTRY(svr_alloc(ctx, (void**)&keep, ub));
    PTRY(svr_alloc(ctx, (void**)&eq, eb)); PTRY(svr_alloc(ctx, (void**)&eqp, eb));
    PTRY(svr_alloc(ctx, (void**)&hist, hb)); PTRY(svr_alloc(ctx, (void**)&st, sb));
    SelectState* st_cap = st + 2;
    uint32_t* n_sel_dev = reinterpret_cast<uint32_t*>(st + 3);
    PCUDA(cudaMemsetAsync(st, 0, sb, ctx->stream));
    PCUDA(cudaMemsetAsync(&st->zlo, 0xFF, sizeof(uint32_t), ctx->stream));
    PCUDA(cudaMemsetAsync(hist, 0, hb, ctx->stream));
    const unsigned int g = nblocks(n, 256);
    const int shifts[3] = {21, 10, 0}, bits[3] = {11, 11, 10}, his[3] = {32, 21, 10};
    prune_depth_kernel<<<g, 256, 0, ctx->stream>>>(s, cams, z, delta, st);
    subdiv_finite_kernel<<<g, 256, 0, ctx->stream>>>(n, z, finite);
    // eq. 14: this step's 5th / 95th percentile of the finite depths (nearest rank): two radix selects on the bits of z
    const float qs[2] = {0.05f, 0.95f};
    for (int k = 0; k < 2; ++k)
        for (int p = 0; p < 3; ++p) {
            select_hist_kernel<<<g, 256, 0, ctx->stream>>>(n, z, nullptr, finite, st + k, shifts[p], (1u << bits[p]) - 1u, his[p], hist);
            select_digit_kernel<<<1, 1024, 0, ctx->stream>>>(st + k, hist, bits[p], p == 0, 1, qs[k], qs[k], 0u);
        }
    subdiv_priority_kernel<<<g, 256, 0, ctx->stream>>>(s, z, delta, usefulness, st, st + 1, opts->use_current_percentiles, opts->z_p5,
                                                       opts->z_p95, opts->kappa, opts->beta, opts->max_level, priority, key, cand);
    // budget: the max_splits eligible voxels of highest priority, ties by lower index
    for (int p = 0; p < 3; ++p) {
        select_hist_kernel<<<g, 256, 0, ctx->stream>>>(n, key, nullptr, cand, st_cap, shifts[p], (1u << bits[p]) - 1u, his[p], hist);
        select_digit_kernel<<<1, 1024, 0, ctx->stream>>>(st_cap, hist, bits[p], p == 0, 1, -1.0f, -1.0f, cap);
    }
    prune_cap_flags_kernel<<<nblocks(n + 1, 256), 256, 0, ctx->stream>>>(n, key, cand, st_cap, eq);
    ctx->launches += 22;
    PCUDA(cudaGetLastError());
    PTRY(launch_exclusive_scan(ctx, eq, eqp, n + 1));
    prune_keep_kernel<<<g, 256, 0, ctx->stream>>>(n, key, cand, st_cap, eqp, cap, keep, n_sel_dev);
    subdiv_invert_kernel<<<g, 256, 0, ctx->stream>>>(n, keep, split);
    ctx->launches += 2;
    PCUDA(cudaGetLastError());
    SelectState h[2];
    uint32_t n_sel = 0;
    PCUDA(cudaMemcpyAsync(h, st, 2 * sizeof(SelectState), cudaMemcpyDeviceToHost, ctx->stream));
    PCUDA(cudaMemcpyAsync(&n_sel, n_sel_dev, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
    PCUDA(cudaStreamSynchronize(ctx->stream));
    *n_split_host = (int64_t)n_sel;
    if (z_percentiles_host)
        for (int k = 0; k < 2; ++k)
            if (h[k].size[0] > 0) memcpy(&z_percentiles_host[k], &h[k].prefix[0], sizeof(float));
#undef PTRY
#undef PCUDA
    cleanup();
    return SVR_OK;
}

SvrStatus svr_subdivide_apply(SvrContext* ctx, const SvrVoxels* vox, const uint8_t* split, uint16_t* ijkl_out, float* raw_out,
                              float* sh_out, int64_t* n_out_host) {
    SVR_NVTX();
    if (!ctx || !vox || !split || !ijkl_out || !raw_out || !sh_out) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (vox->n < 0 || vox->n >= ((int64_t)1 << 28)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "voxel count out of range");
    if (n_out_host) *n_out_host = 0;
    const int64_t n = vox->n;
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    uint32_t *counts = nullptr, *offs = nullptr;
    const size_t eb = sizeof(uint32_t) * (size_t)(n + 1);
    SVR_TRY(svr_alloc(ctx, (void**)&counts, eb));
    SvrStatus stt = svr_alloc(ctx, (void**)&offs, eb);
    if (stt != SVR_OK) { svr_free(ctx, counts, eb); return stt; }
    split_to_counts_kernel<<<nblocks(n + 1, 256), 256, 0, ctx->stream>>>(n, split, counts);
    stt = launch_exclusive_scan(ctx, counts, offs, n + 1);
    if (stt == SVR_OK) {
        const int words = 3 * (vox->sh_degree + 1) * (vox->sh_degree + 1);
        subdiv_cells_kernel<<<nblocks(n, 256), 256, 0, ctx->stream>>>(n, split, offs, reinterpret_cast<const uint2*>(vox->ijkl),
                                                                     reinterpret_cast<const float4*>(vox->raw_density),
                                                                     reinterpret_cast<uint2*>(ijkl_out), reinterpret_cast<float4*>(raw_out));
        subdiv_sh_kernel<<<nblocks(n * words, 256), 256, 0, ctx->stream>>>(n, words, split, offs, reinterpret_cast<const uint32_t*>(vox->sh),
                                                                           reinterpret_cast<uint32_t*>(sh_out));
        ctx->launches += 3;
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess && n_out_host) {
            uint32_t n_split = 0;
            e = cudaMemcpyAsync(&n_split, offs + n, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
            *n_out_host = n + 7 * (int64_t)n_split;
        }
        if (e != cudaSuccess) stt = svr_fail(ctx, SVR_ERR_CUDA, "subdivide: %s", cudaGetErrorString(e));
    }
    svr_free(ctx, counts, eb);
    svr_free(ctx, offs, eb);
    return stt;
}

SvrStatus svr_subdivide_rows(SvrContext* ctx, const uint8_t* split, int64_t n, const void* src, void* dst, int64_t row_bytes,
                             int32_t mode, int64_t* n_out_host) {
    SVR_NVTX();
    if (!ctx || !split || !src || !dst) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "null argument");
    if (n < 0 || n >= ((int64_t)1 << 28)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "row count out of range");
    if (row_bytes < 1 || (row_bytes > 2 && row_bytes % 4 != 0)) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "row_bytes must be 1, 2 or a multiple of 4");
    if (mode != SVR_ROWS_COPY_PARENT && mode != SVR_ROWS_ZERO) return svr_fail(ctx, SVR_ERR_INVALID_ARG, "mode must be SVR_ROWS_COPY_PARENT or SVR_ROWS_ZERO");
    if (n_out_host) *n_out_host = 0;
    if (n == 0) return SVR_OK;
    SVR_CUDA(ctx, cudaSetDevice(ctx->device));
    uint32_t *counts = nullptr, *offs = nullptr;
    const size_t eb = sizeof(uint32_t) * (size_t)(n + 1);
    SVR_TRY(svr_alloc(ctx, (void**)&counts, eb));
    SvrStatus stt = svr_alloc(ctx, (void**)&offs, eb);
    if (stt != SVR_OK) { svr_free(ctx, counts, eb); return stt; }
    split_to_counts_kernel<<<nblocks(n + 1, 256), 256, 0, ctx->stream>>>(n, split, counts);
    stt = launch_exclusive_scan(ctx, counts, offs, n + 1);
    if (stt == SVR_OK) {
        const int zero = mode == SVR_ROWS_ZERO;
        if (row_bytes == 1)
            subdiv_rows_kernel<uint8_t><<<nblocks(n, 256), 256, 0, ctx->stream>>>(n, 1, split, offs, (const uint8_t*)src, (uint8_t*)dst, zero);
        else if (row_bytes == 2)
            subdiv_rows_kernel<uint16_t><<<nblocks(n, 256), 256, 0, ctx->stream>>>(n, 1, split, offs, (const uint16_t*)src, (uint16_t*)dst, zero);
        else {
            const int words = (int)(row_bytes / 4);
            subdiv_rows_kernel<uint32_t><<<nblocks(n * words, 256), 256, 0, ctx->stream>>>(n, words, split, offs, (const uint32_t*)src, (uint32_t*)dst, zero);
        }
        ctx->launches += 2;
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess && n_out_host) {
            uint32_t n_split = 0;
            e = cudaMemcpyAsync(&n_split, offs + n, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
            *n_out_host = n + 7 * (int64_t)n_split;
        }
        if (e != cudaSuccess) stt = svr_fail(ctx, SVR_ERR_CUDA, "subdivide rows: %s", cudaGetErrorString(e));
    }
    svr_free(ctx, counts, eb);
    svr_free(ctx, offs, eb);
    return stt;
}

}  // extern "C"
