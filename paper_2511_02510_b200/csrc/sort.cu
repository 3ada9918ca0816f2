// Hand-written device primitives for stage (2): exclusive scan of the per-voxel entry counts and a
// least-significant-digit radix sort of (key u64, voxel id u32) pairs over the live key bits only
// (tile bits + 3 octant bits + 3*Lmax Morton bits; 51 bits = 7 passes of 8 on C4).
//
// One pass = three kernels over tiles of 2048 pairs:
//   radix_upsweep   per-tile 256-bin digit histogram (shared-memory integer atomics)     reads 8 B/pair
//   radix_scan      one warp per bin: exclusive scan of that bin's counts across tiles, plus the bin total
//   radix_downsweep stable rank inside the tile (match_any per warp round, per-warp counters, digit-major
//                   reorder through shared memory) and a run-coalesced scatter      reads 12, writes 12 B/pair
// => 32 B per pair per pass of HBM traffic. Keys are unique (B3), so stability is only needed between
// passes, which the rank construction guarantees (tile order, then warp segment, then round, then lane).
#include "svr_internal.cuh"

namespace {

constexpr int RADIX = 256;
constexpr int SORT_THREADS = 256;
constexpr int ITEMS = 8;
constexpr int TILE = SORT_THREADS * ITEMS;   // 2048 pairs per tile
constexpr unsigned FULL = 0xffffffffu;

// ---- scan ------------------------------------------------------------------------------------------
constexpr int SCAN_TILE = 2048;

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(FULL, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// inclusive scan of one value per thread across a 256-thread block; returns inclusive prefix, *total = block sum
__device__ __forceinline__ uint32_t block_incl_scan256(uint32_t v, uint32_t* sh /*[8]*/, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = warp_incl_scan(v, lane);
    if (lane == 31) sh[warp] = inc;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        uint32_t s = sh[w];
        if (w < warp) base += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return inc + base;
}

__global__ void __launch_bounds__(256) scan_tile_sums_kernel(const uint32_t* __restrict__ in, int64_t n, uint32_t* __restrict__ sums) {
    __shared__ uint32_t sh[8];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    uint32_t local = 0;
#pragma unroll
    for (int k = 0; k < SCAN_TILE / 256; ++k) {
        int64_t i = base + k * 256 + threadIdx.x;
        if (i < n) local += in[i];
    }
    uint32_t tot;
    block_incl_scan256(local, sh, &tot);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

// single block: exclusive scan of the tile sums in place (n_tiles <= a few thousand)
__global__ void __launch_bounds__(256) scan_sums_kernel(uint32_t* __restrict__ sums, int n_tiles) {
    __shared__ uint32_t sh[8];
    uint32_t carry = 0;
    for (int base = 0; base < n_tiles; base += 256) {
        int i = base + threadIdx.x;
        uint32_t v = (i < n_tiles) ? sums[i] : 0u, tot;
        uint32_t inc = block_incl_scan256(v, sh, &tot);
        if (i < n_tiles) sums[i] = carry + inc - v;
        carry += tot;
    }
}

__global__ void __launch_bounds__(256) scan_apply_kernel(const uint32_t* __restrict__ in, int64_t n, const uint32_t* __restrict__ sums,
                                                         uint32_t* __restrict__ out) {
    __shared__ uint32_t sh[8];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * (SCAN_TILE / 256);
    uint32_t v[SCAN_TILE / 256], local = 0;
#pragma unroll
    for (int k = 0; k < SCAN_TILE / 256; ++k) {
        int64_t i = base + k;
        v[k] = (i < n) ? in[i] : 0u;
        local += v[k];
    }
    uint32_t tot;
    uint32_t run = sums[blockIdx.x] + block_incl_scan256(local, sh, &tot) - local;
#pragma unroll
    for (int k = 0; k < SCAN_TILE / 256; ++k) {
        int64_t i = base + k;
        if (i < n) out[i] = run;
        run += v[k];
    }
}

// ---- radix sort ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t digit_of(uint64_t key, int shift, uint32_t mask) { return (uint32_t)(key >> shift) & mask; }

__global__ void __launch_bounds__(SORT_THREADS) radix_upsweep_kernel(const uint64_t* __restrict__ keys, int64_t n, int shift,
                                                                     uint32_t mask, int n_tiles, uint32_t* __restrict__ tile_hist) {
    __shared__ uint32_t h[RADIX];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * TILE;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        int64_t i = base + k * SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[digit_of(keys[i], shift, mask)], 1u);
    }
    __syncthreads();
    tile_hist[(size_t)threadIdx.x * n_tiles + blockIdx.x] = h[threadIdx.x];   // bin-major: [bin][tile]
}

// one warp per bin: exclusive scan across tiles in place; bin_total[bin] = number of keys with that digit.
// 128 counts per iteration (four coalesced loads in flight) so the row's L2 latency is paid n_tiles/128 times.
__global__ void __launch_bounds__(256) radix_scan_kernel(uint32_t* __restrict__ tile_hist, int n_tiles, uint32_t* __restrict__ bin_total) {
    const int lane = threadIdx.x & 31, bin = blockIdx.x * 8 + (threadIdx.x >> 5);
    uint32_t* row = tile_hist + (size_t)bin * n_tiles;
    uint32_t carry = 0;
    for (int base = 0; base < n_tiles; base += 128) {
        uint32_t v[4], inc[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            int i = base + k * 32 + lane;
            v[k] = (i < n_tiles) ? row[i] : 0u;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) inc[k] = warp_incl_scan(v[k], lane);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            int i = base + k * 32 + lane;
            if (i < n_tiles) row[i] = carry + inc[k] - v[k];
            carry += __shfl_sync(FULL, inc[k], 31);
        }
    }
    if (lane == 0) bin_total[bin] = carry;
}

__global__ void __launch_bounds__(SORT_THREADS) radix_downsweep_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                                                                       uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                                       int64_t n, int shift, uint32_t mask, int n_tiles,
                                                                       const uint32_t* __restrict__ tile_hist,
                                                                       const uint32_t* __restrict__ bin_total) {
    __shared__ uint32_t warp_cnt[8][RADIX];
    __shared__ uint32_t tile_off[RADIX];     // start of each digit inside the tile
    __shared__ uint32_t gofs[RADIX];         // global start of (digit, this tile)
    __shared__ uint32_t sh8[8];
    __shared__ uint64_t skeys[TILE];
    __shared__ uint32_t svals[TILE];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t base = (int64_t)blockIdx.x * TILE;
    const int ntile = (int)min((int64_t)TILE, n - base);

#pragma unroll
    for (int w = 0; w < 8; ++w) warp_cnt[w][tid] = 0;
    {   // global digit bases: exclusive scan of the 256 bin totals, plus this tile's offset inside the bin
        uint32_t t = bin_total[tid], tot;
        uint32_t inc = block_incl_scan256(t, sh8, &tot);
        gofs[tid] = inc - t + tile_hist[(size_t)tid * n_tiles + blockIdx.x];
    }
    uint64_t key[ITEMS];
    uint32_t val[ITEMS], pre[ITEMS];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int li = warp * (32 * ITEMS) + r * 32 + lane;               // warp-contiguous segments keep the rank stable
        key[r] = (li < ntile) ? keys_in[base + li] : ~0ull;
        val[r] = (li < ntile) ? vals_in[base + li] : 0u;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int li = warp * (32 * ITEMS) + r * 32 + lane;
        uint32_t d = (li < ntile) ? digit_of(key[r], shift, mask) : RADIX;   // RADIX = "no key"
        unsigned peers = __match_any_sync(FULL, d);
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && d < RADIX) {
            old = warp_cnt[warp][d];
            warp_cnt[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(FULL, old, leader);
        pre[r] = old + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    {   // per digit: exclusive offsets of the 8 warps, then exclusive scan over digits
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            uint32_t cnt = warp_cnt[w][tid];
            warp_cnt[w][tid] = run;
            run += cnt;
        }
        uint32_t tot;
        uint32_t inc = block_incl_scan256(run, sh8, &tot);
        tile_off[tid] = inc - run;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int li = warp * (32 * ITEMS) + r * 32 + lane;
        if (li < ntile) {
            uint32_t d = digit_of(key[r], shift, mask);
            uint32_t pos = tile_off[d] + warp_cnt[warp][d] + pre[r];
            skeys[pos] = key[r];
            svals[pos] = val[r];
        }
    }
    __syncthreads();
    for (int i = tid; i < ntile; i += SORT_THREADS) {
        uint64_t k = skeys[i];
        uint32_t d = digit_of(k, shift, mask);
        uint32_t dst = gofs[d] + ((uint32_t)i - tile_off[d]);
        keys_out[dst] = k;
        vals_out[dst] = svals[i];
    }
}

}  // namespace

SvrStatus launch_exclusive_scan(SvrContext* ctx, const uint32_t* in, uint32_t* out, int64_t n_plus_1) {
    StageScope scope__(ctx, ST_SCAN);
    const int n_tiles = (int)((n_plus_1 + SCAN_TILE - 1) / SCAN_TILE);
    uint32_t* sums = nullptr;
    SVR_TRY(svr_alloc(ctx, (void**)&sums, sizeof(uint32_t) * (size_t)n_tiles));
    scan_tile_sums_kernel<<<n_tiles, 256, 0, ctx->stream>>>(in, n_plus_1, sums);
    scan_sums_kernel<<<1, 256, 0, ctx->stream>>>(sums, n_tiles);
    scan_apply_kernel<<<n_tiles, 256, 0, ctx->stream>>>(in, n_plus_1, sums, out);
    ctx->launches += 3;
    cudaError_t e = cudaGetLastError();
    svr_free(ctx, sums, sizeof(uint32_t) * (size_t)n_tiles);
    SVR_CUDA(ctx, e);
    return SVR_OK;
}

SvrStatus launch_sort_pairs(SvrContext* ctx, uint64_t* keys, uint64_t* keys_alt, uint32_t* vals, uint32_t* vals_alt,
                            int64_t n, int bits, uint64_t** keys_sorted, uint32_t** vals_sorted) {
    StageScope scope__(ctx, ST_SORT);
    const int n_tiles = (int)((n + TILE - 1) / TILE);
    uint32_t* tile_hist = nullptr;
    const size_t hist_bytes = sizeof(uint32_t) * ((size_t)RADIX * n_tiles + RADIX);
    SVR_TRY(svr_alloc(ctx, (void**)&tile_hist, hist_bytes));
    uint32_t* bin_total = tile_hist + (size_t)RADIX * n_tiles;
    uint64_t *kin = keys, *kout = keys_alt;
    uint32_t *vin = vals, *vout = vals_alt;
    for (int shift = 0; shift < bits; shift += 8) {
        const int nb = (bits - shift < 8) ? bits - shift : 8;
        const uint32_t mask = (1u << nb) - 1u;
        radix_upsweep_kernel<<<n_tiles, SORT_THREADS, 0, ctx->stream>>>(kin, n, shift, mask, n_tiles, tile_hist);
        radix_scan_kernel<<<RADIX / 8, 256, 0, ctx->stream>>>(tile_hist, n_tiles, bin_total);
        radix_downsweep_kernel<<<n_tiles, SORT_THREADS, 0, ctx->stream>>>(kin, vin, kout, vout, n, shift, mask, n_tiles, tile_hist,
                                                                          bin_total);
        ctx->launches += 3;
        uint64_t* tk = kin; kin = kout; kout = tk;
        uint32_t* tv = vin; vin = vout; vout = tv;
    }
    cudaError_t e = cudaGetLastError();
    svr_free(ctx, tile_hist, hist_bytes);
    SVR_CUDA(ctx, e);
    *keys_sorted = kin;
    *vals_sorted = vin;
    return SVR_OK;
}
