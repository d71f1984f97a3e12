// count3.cu -- three-point counts (include/tpcf.h tpcf_count3; "higher order
// correlation functions").  Every triple i<j<k of one catalog is counted once in the cell of the ascending
// result slots (0 = under, 1..nbins = bins, nbins+1 = over) of its three sides.
//
// Two kernels.  pair_slots_kernel classifies every pair once, in fp64 exactly as the fp64 engine does (squared chord
// against T_k = 4 sin^2(e_k/2)), into an n x n byte matrix S.  triples_kernel then enumerates the triples as pure byte
// and integer work: a CTA takes row i (work counter in global memory, longest rows first), keeps S[i][*] in shared
// memory, and its warps walk j > i; for one j the lanes read S[i][k] (shared) and S[j][k] (global, coalesced, 4 k per
// lane) for k > j, order the three slots with min/max, and add 1 to the cell of a CTA-private 32-bit histogram in shared
// memory (the paper's scheme for the pair histograms, carried to (nbins+2)^3 cells), which is merged into the
// uint64 result in global memory with integer atomics -- order-independent, hence deterministic.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "kernels.cuh"

namespace tpcf {
namespace {

constexpr int kT3 = 256;             // threads per CTA of both kernels

__device__ __forceinline__ int slot64(const double4& a, const double4& b, const double* __restrict__ thr, int n) {
    const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
    const double d2 = fmin(fma(dz, dz, fma(dy, dy, dx * dx)), 4.0);
    if (d2 < thr[0]) return 0;
    if (d2 > thr[n]) return n + 1;
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (thr[mid] <= d2) lo = mid; else hi = mid;
    }
    return lo + 1;
}

// S[i * pitch + j] = slot of the pair (i, j), all i, j < n (the diagonal and the padding columns are never read)
__global__ void __launch_bounds__(kT3) pair_slots_kernel(const double4* __restrict__ x64, uint32_t n, uint32_t pitch,
                                                         const double* __restrict__ gthr, int nbins, uint8_t* __restrict__ S) {
    extern __shared__ __align__(16) unsigned char smem3[];
    double* thr = reinterpret_cast<double*>(smem3);
    for (int k = threadIdx.x; k <= nbins; k += kT3) thr[k] = gthr[k];
    __syncthreads();
    const uint32_t i = blockIdx.y;
    const double4 a = x64[i];
    for (uint32_t j = blockIdx.x * kT3 + threadIdx.x; j < n; j += gridDim.x * kT3)
        S[(size_t)i * pitch + j] = (uint8_t)slot64(a, x64[j], thr, nbins);
}

__device__ __forceinline__ void add_triple(unsigned* hist, int m, int a, int b, int c) {
    const int lo = min(a, min(b, c)), hi = max(a, max(b, c)), mid = a + b + c - lo - hi;
    atomicAdd(hist + (lo * m + mid) * m + hi, 1u);
}

__global__ void __launch_bounds__(1024) triples_kernel(const uint8_t* __restrict__ S, uint32_t n, uint32_t pitch, int m,
                                                      unsigned long long* __restrict__ next_row, unsigned long long* __restrict__ result) {
    extern __shared__ __align__(16) unsigned char smem3[];
    unsigned* hist = reinterpret_cast<unsigned*>(smem3);                 // m^3 cells
    uint8_t* si = smem3 + (((size_t)m * m * m * sizeof(unsigned) + 15) & ~size_t(15));      // pitch bytes: row i of S
    __shared__ unsigned long long s_row;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, cells = m * m * m;
    const int nthr = blockDim.x;             // 256, or 1024 when the histogram leaves room for one CTA per SM only
    for (int c = tid; c < cells; c += nthr) hist[c] = 0;
    unsigned long long since_flush = 0;          // triples added to the 32-bit partials since they were last merged
    __syncthreads();
    for (;;) {
        if (tid == 0) s_row = atomicAdd(next_row, 1ull);
        __syncthreads();
        const unsigned long long row = s_row;
        __syncthreads();
        if (row + 2 >= n) break;                                        // rows n-2, n-1 hold no triple
        const uint32_t i = (uint32_t)row;
        const unsigned long long r = n - 1 - i, in_row = r * (r - 1) / 2;
        if (since_flush + in_row >= (1ull << 31)) {                     // uniform over the CTA
            for (int c = tid; c < cells; c += nthr) {
                if (hist[c]) atomicAdd(result + c, (unsigned long long)hist[c]);
                hist[c] = 0;
            }
            since_flush = 0;
            __syncthreads();
        }
        since_flush += in_row;
        for (uint32_t k = tid * 16; k < pitch; k += nthr * 16)
            *reinterpret_cast<uint4*>(si + k) = *reinterpret_cast<const uint4*>(S + (size_t)i * pitch + k);
        __syncthreads();
        for (uint32_t j = i + 1 + warp; j + 1 < n; j += nthr / 32) {
            const int a = si[j];
            const uint8_t* sj = S + (size_t)j * pitch;
            for (uint32_t k0 = ((j + 1) & ~127u) + lane * 4; k0 < n; k0 += 128) {
                const uchar4 b = *reinterpret_cast<const uchar4*>(si + k0);
                const uchar4 c = *reinterpret_cast<const uchar4*>(sj + k0);
                if (k0 > j && k0 < n) add_triple(hist, m, a, b.x, c.x);
                if (k0 + 1 > j && k0 + 1 < n) add_triple(hist, m, a, b.y, c.y);
                if (k0 + 2 > j && k0 + 2 < n) add_triple(hist, m, a, b.z, c.z);
                if (k0 + 3 > j && k0 + 3 < n) add_triple(hist, m, a, b.w, c.w);
            }
        }
        __syncthreads();
    }
    for (int c = tid; c < cells; c += nthr)
        if (hist[c]) atomicAdd(result + c, (unsigned long long)hist[c]);
}

}  // namespace

size_t count3_slot_bytes(uint64_t n) {
    const uint64_t pitch = (n + 127) / 128 * 128;
    return (size_t)(pitch * n);
}

cudaError_t launch_count3(const double4* x64, uint32_t n, const double* thr, int nbins, uint8_t* slots, unsigned long long* next_row,
                          unsigned long long* result3, int sm_count, cudaStream_t st) {
    const uint32_t pitch = (n + 127) / 128 * 128;
    const int m = nbins + 2;
    dim3 g1(std::min<uint32_t>((n + kT3 - 1) / kT3, 64), n);
    pair_slots_kernel<<<g1, kT3, (nbins + 1) * sizeof(double), st>>>(x64, n, pitch, thr, nbins, slots);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const size_t smem = (((size_t)m * m * m * sizeof(unsigned) + 15) & ~size_t(15)) + pitch;
    e = cudaFuncSetAttribute(triples_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // a large histogram leaves room for few CTAs per SM: give those CTAs 1024 threads so that the SM still holds 32+ warps
    const int threads = smem > 56 * 1024 ? 1024 : kT3;
    int per_sm = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, triples_kernel, threads, smem);
    if (e != cudaSuccess) return e;
    const int grid = std::max(1, std::min<int>(sm_count * std::max(per_sm, 1), (int)n));
    triples_kernel<<<grid, threads, smem, st>>>(slots, n, pitch, m, next_row, result3);
    return cudaGetLastError();
}

}  // namespace tpcf
