// Exclusive scan of the per-voxel entry counts and the (key, voxel id) radix sort over the live key bits.
// Round-1 scaffold: CUB's device scan / onesweep radix sort (library code). DESIGN.md lists the
// hand-written replacement (compressed per-octant rank keys, fewer passes) as the next step for this row.
#include "svr_internal.cuh"
#include <cub/cub.cuh>

SvrStatus launch_exclusive_scan(SvrContext* ctx, const uint32_t* in, uint32_t* out, int64_t n_plus_1) {
    StageScope scope__(ctx, ST_SCAN);
    size_t tmp_bytes = 0;
    SVR_CUDA(ctx, cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, in, out, n_plus_1, ctx->stream));
    void* tmp = nullptr;
    SVR_TRY(svr_alloc(ctx, &tmp, tmp_bytes));
    cudaError_t e = cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, in, out, n_plus_1, ctx->stream);
    ctx->launches += 2;
    svr_free(ctx, tmp, tmp_bytes);
    SVR_CUDA(ctx, e);
    return SVR_OK;
}

SvrStatus launch_sort_pairs(SvrContext* ctx, uint64_t* keys, uint64_t* keys_alt, uint32_t* vals, uint32_t* vals_alt,
                            int64_t n, int bits, uint64_t** keys_sorted, uint32_t** vals_sorted) {
    StageScope scope__(ctx, ST_SORT);
    cub::DoubleBuffer<uint64_t> dk(keys, keys_alt);
    cub::DoubleBuffer<uint32_t> dv(vals, vals_alt);
    size_t tmp_bytes = 0;
    SVR_CUDA(ctx, cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, dk, dv, n, 0, bits, ctx->stream));
    void* tmp = nullptr;
    SVR_TRY(svr_alloc(ctx, &tmp, tmp_bytes));
    cudaError_t e = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, dk, dv, n, 0, bits, ctx->stream);
    ctx->launches += 2 + (bits + 7) / 8;
    svr_free(ctx, tmp, tmp_bytes);
    SVR_CUDA(ctx, e);
    *keys_sorted = dk.Current();
    *vals_sorted = dv.Current();
    return SVR_OK;
}
