// kernels.cuh -- launch interface between the C ABI (api.cu) and the sm_100a kernels (kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "tables.h"

namespace tpcf {

// One pair-count launch: i-points x j-points over the work plan.  All pointers are device pointers.
struct PairParams {
    const float4* xi;           // fp32 unit vectors of the i-side catalog, padded to a multiple of kTileI with (2,2,2,0)
    const float4* xj;           // j-side, padded to a multiple of kTileJ
    const double4* xi64;        // fp64 unit vectors (same padding); the recheck path and the fp64 engine read these
    const double4* xj64;
    uint32_t n_i, n_j;          // real (unpadded) sizes
    int tri;                    // 1: xi == xj and only pairs i<j are enumerated
    uint32_t blocks_i, tiles_j, chunk;
    uint32_t n_items_part;      // items this launch executes (after the partition)
    const uint32_t* row_start;  // tri: first item of i-block I (blocks_i + 1 entries)
    uint32_t part, nparts;      // item w of the full plan is executed iff w % nparts == part
    // fast engine tables
    const float2* lut;          // ncells x (lo, hi)
    const uint16_t* slotmap;    // 2 x ncells: result slot of (cell, d2 < lo) and (cell, d2 >= hi)
    int ncells, shift;
    float sqrt_scale, sqrt_clamp;
    // exact thresholds
    const double* thr;          // nbins + 1
    int nbins;
    unsigned long long* result; // nbins + 3: under, bins, over, discard
    unsigned long long* counters;   // [0] next work item, [1] pairs rechecked in fp64, [2] items done
};

struct LaunchInfo {
    int grid, block, smem_bytes, launches;
};

cudaError_t launch_convert(const void* radec, int is_f64, uint64_t n, uint64_t n_pad, double4* x64, float4* x32,
                           int* bad_flag, cudaStream_t st);
cudaError_t launch_gather(const double4* src64, const float4* src32, const int64_t* rows, uint64_t nrows,
                          uint64_t nrows_pad, uint64_t n_src, double4* dst64, float4* dst32, int* bad_flag,
                          cudaStream_t st);
cudaError_t launch_pairs_fast(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_pairs_exact64(const PairParams& p, int sm_count, cudaStream_t st, LaunchInfo* info);
// result[0 .. nbins+1] -> out (device), subtracting `self_pairs` from the slot that holds theta = 0
cudaError_t launch_finalize(const unsigned long long* result, int nbins, int zero_slot, unsigned long long self_pairs,
                            unsigned long long* out, cudaStream_t st);

}  // namespace tpcf
