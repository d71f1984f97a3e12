// kernels.cuh -- launch interface between the C ABI (api.cu) and the sm_100a kernels (kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "tables.h"

namespace tpcf {

// One pair-count launch: i-points x j-points over the work plan.  All pointers are device pointers.
struct PairParams {
    // i side: rows as fp32 offsets from the centre of their 8-row group ("quad"), and the groups' (centre, radius)
    const float4* xq;
    const float4* cq;
    // j side: rows as (-2 offset, |offset|^2) from the centre of their 64-row subtile, and the subtiles' (centre, radius)
    const float4* xs;
    const float4* cs;
    // j side, tensor engine: the same roles for kTcSubJ = 128-row tiles (rows xt, spheres ct), and per tile a
    // kTcSubJ x kTcK block of TF32 values in the K-major no-swizzle core-matrix layout (8 rows x 16 bytes contiguous;
    // 8-row groups 128 B apart, the four 16-byte K chunks kTcSubJ * 16 B apart).  Row j: m_hi(3) m_lo(3) m_hi(3) 1 1 1
    // w_hi w_mid w_lo 0 with m = -2 offset, w = |offset|^2 split into TF32 parts
    const float4* xt;
    const float4* ct;
    const float* xb;
    const double4* xi64;        // fp64 unit vectors (padded with (2,2,2)); the recheck path and the fp64 engine read these
    const double4* xj64;
    uint32_t n_i, n_j;          // real (unpadded) sizes
    int tri;                    // 1: i and j are the same catalog and only pairs i<j are enumerated
    int window;                 // 1: window loops enabled (tpcf_set_window)
    int prune;                  // 1: pruning mode (tpcf_set_pruning): blocks whose window reaches no band are added wholesale
    uint32_t blocks_i, tiles_j, chunk;
    uint32_t n_items_part;      // items this launch executes (after the partition)
    const uint32_t* row_start;  // tri: first item of i-block I (blocks_i + 1 entries)
    uint32_t part, nparts;      // item w of the full plan is executed iff w % nparts == part
    uint32_t jsplit;            // fast engine: a warp item covers 1/jsplit of its item's (single) j-tile; 1, 2, 4, 8 or 16,
                                // > 1 only when chunk == 1 (small catalogs: more, shorter warp items for the tail)
    // fast engine tables
    const float* lut;           // ncells x threshold of the cell (+inf: none, NaN: several)
    const uint16_t* slotmap;    // 2 x ncells: result slots below the threshold of cell c [c] and at or above it [ncells + c]
    int ncells, shift;
    float sqrt_scale, sqrt_clamp;
    float guard_scale;          // tpcf_set_guard_scale
    int lut_multi;              // 1: some cell sees several thresholds (its lut entry is NaN)
    const float2* band_mh;      // nbands x (mid, half width)
    const float2* band_lh;      // nbands x (lo, hi)
    const uint16_t* band_slot;  // nbands + 1 result slots: below band b; [nbands] = above the last band
    const uint16_t* cell_band;  // ncells: first band whose hi lies above the start of the cell
    int nbands;
    // exact thresholds
    const double* thr;          // nbins + 1
    int nbins;
    unsigned long long* result; // nbins + 3: under, bins, over, discard
    // [0] next work item (fast engine: next warp item), [1] pairs rechecked in fp64, [2] items done,
    // [3..6] (lane-quad x subtile) warp blocks counted by the 1-, 2-, 3-edge window loops and by the cell-lookup loop,
    // [7] lanes of window blocks recounted because a pair came within a guard band, [8] warp blocks sent to the fp64 loop,
    // [9] warp blocks added wholesale in pruning mode
    unsigned long long* counters;
};

struct LaunchInfo {
    int grid, block, smem_bytes, launches;
};

constexpr int kNumCounters = 10;
constexpr int kTcSubJ = 128;           // j-rows per tile of the tensor engine (one bounding sphere, one MMA)
constexpr int kTcK = 16;               // K of the tensor engine's operand tiles (two tcgen05.mma kind::tf32 steps of 8)
constexpr int kSortChunk = 2048;        // elements per block of the radix sort

// RA/Dec rows -> fp64 unit vectors (caller order) + 63-bit Hilbert keys + identity index
// (bounds: 24 words of scratch for the catalog's bounding boxes, which the keys are taken relative to)
cudaError_t launch_convert(const void* radec, int is_f64, uint64_t n, double4* x64_rows, uint64_t* keys, uint32_t* idx,
                           int* bad_flag, uint64_t* bounds, cudaStream_t st);
// 3-D variant: Cartesian rows * scale (a power of two) -> positions inside the unit ball + 63-bit 3-D Hilbert keys
cudaError_t launch_convert_xyz(const void* xyz, int is_f64, uint64_t n, double scale, double max_abs, double4* x64_rows, uint64_t* keys,
                               uint32_t* idx, int* bad_flag, uint64_t* bounds, cudaStream_t st);
// Stable LSD radix sort of (key, idx) pairs on the low `nbits` bits; buffers A hold the input, the sorted
// result ends in A or B (*in_a).  counts: 256 * ceil(n / kSortChunk) words of scratch.
cudaError_t launch_sort_pairs(uint64_t* keys_a, uint64_t* keys_b, uint32_t* idx_a, uint32_t* idx_b, uint32_t* counts,
                              uint32_t n, int nbits, cudaStream_t st, bool* in_a);
// sorted catalog: x64[k] = rows[order[k]], inv[order[k]] = k; rows n..n_pad-1 = padding point
cudaError_t launch_permute(const double4* x64_rows, const uint32_t* order, uint64_t n, uint64_t n_pad, double4* x64,
                           uint32_t* inv, cudaStream_t st);
// i-side role: per kIPerThread-row group ("quad") its (centre, radius) and the rows as fp32 offsets from the centre
cudaError_t launch_quads(const double4* x64, uint64_t n_pad, float4* xq, float4* cq, cudaStream_t st);
// j-side role: per 64-row subtile its (centre, radius) and the rows as (-2 offset, |offset|^2)
cudaError_t launch_subtiles(const double4* x64, uint64_t n_pad, float4* xs, float4* cs, float4* xt, float4* ct, float* xb,
                            cudaStream_t st);
// subset mode: caller rows -> positions in the sorted catalog (keys for the sort) with range check
cudaError_t launch_row_keys(const int64_t* rows, uint64_t nrows, uint64_t n_src, const uint32_t* inv, uint64_t* keys,
                            uint32_t* idx, int* bad_flag, cudaStream_t st);
// dst[k] = src[pos[k]] for k < nrows, padding point after
cudaError_t launch_gather(const double4* src64, const uint64_t* pos, uint64_t nrows, uint64_t nrows_pad, double4* dst64,
                          cudaStream_t st);
// lookup_heavy: almost every block takes the per-pair cell lookup: the variant compiled for 3 CTAs per SM
cudaError_t launch_pairs_fast(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info, bool lookup_heavy);
cudaError_t launch_pairs_tensor(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info);
// out[0] += sampled (8-row group, 128-row tile) blocks the tensor kernel would count pair by pair, out[1] += blocks sampled
cudaError_t launch_sample_modes(const PairParams& p, CellMap map, uint32_t nsamples, unsigned long long* out, cudaStream_t st);
// ntiles x (128 x 128) accumulator tiles of the tensor engine's MMA for given operand rows (device pointers)
cudaError_t launch_tensor_probe(const float4* srows, const float4* brows, float* q, uint32_t ntiles, cudaStream_t st);
cudaError_t launch_pairs_exact64(const PairParams& p, int sm_count, cudaStream_t st, LaunchInfo* info);
// weighted sums: wresult[0 .. nbins+2] += sum of wi[i] * wj[j] per result slot, fp64 (weights in sorted order)
cudaError_t launch_pairs_weighted64(const PairParams& p, const double* wi, const double* wj, double* wresult, int sm_count, cudaStream_t st);
cudaError_t launch_scatter_weights(const double* w, const uint32_t* inv, uint64_t n, uint64_t n_pad, double* out, cudaStream_t st);
// result[0 .. nbins+1] -> out (device), subtracting `self_pairs` from the slot that holds theta = 0
cudaError_t launch_finalize(const unsigned long long* result, int nbins, int zero_slot, unsigned long long self_pairs,
                            unsigned long long* out, cudaStream_t st);

// three-point counts (count3.cu): bytes of the n x n pair-slot matrix, and the two kernels: slots <- slot of every pair (fp64),
// result3[(a * m + b) * m + c] += triples i<j<k whose side slots in ascending order are (a, b, c), m = nbins + 2;
// next_row (one counter) and result3 (m^3) must be zero on entry
size_t count3_slot_bytes(uint64_t n);
cudaError_t launch_count3(const double4* x64, uint32_t n, const double* thr, int nbins, uint8_t* slots, unsigned long long* next_row,
                          unsigned long long* result3, int sm_count, cudaStream_t st);

}  // namespace tpcf
