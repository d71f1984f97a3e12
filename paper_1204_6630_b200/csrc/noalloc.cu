// noalloc.cu -- tpcf_count_static (include/tpcf.h): one pair count, RA/Dec rows in, histogram out, that never
// allocates device memory.
//
// Who this is for.  Every other compute entry point of libtpcf reaches cudaMalloc sooner or later (the context's
// accumulators, the catalog arrays, the sort scratch, the plan).  Some hosts cannot afford that: a process whose device
// memory already belongs to one pool allocator (a training framework's caching allocator, RMM) where a raw cudaMalloc
// from a library either fails or fragments the pool; a service with a fixed memory budget per GPU that is checked at
// start-up; a latency-critical loop in which the device-wide synchronisation that cudaMalloc / cudaFree imply would
// stall every other stream.  For those callers this file keeps the scratch the count needs -- the fp64 unit vectors
// made from the rows, the thresholds, the uint64 accumulators, the work counter and the bad-row flag -- in ONE
// file-scope __device__ array of fixed size.  The price: a hard upper limit on the problem size
// (TPCF_STATIC_MAX_ROWS, TPCF_STATIC_MAX_BINS), about 2.07 MiB of device memory held by every GPU that loads this
// library's module until the process exits, and no two calls in flight on one GPU at the same time.
//
// The kernel is a variant of pair_exact64_kernel (kernels.cu): the same fp64 squared chord, the same thresholds
// T_k = 4 sin^2(e_k / 2) (tables.cpp, make_binning), the same slot rule, a work counter in global memory, 32-bit
// partial histograms in shared memory merged into uint64 accumulators; what differs is where the scratch lives and
// that the j-rows of an item are staged in shared memory.  The rows are converted by the arithmetic of convert_kernel.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/tpcf.h"
#include "tables.h"

namespace {

constexpr int kMaxRows = TPCF_STATIC_MAX_ROWS;
constexpr int kMaxBins = TPCF_STATIC_MAX_BINS;
constexpr size_t up256(size_t b) { return (b + 255) & ~size_t(255); }
// layout of the scratch array, every part on a 256-byte boundary
constexpr size_t kOffCtl = 0;                                                    // [0] work counter (u64), [1] bad-row flag (u64)
constexpr size_t kOffResult = kOffCtl + 256;                                     // kMaxBins + 2 accumulators (u64): under, bins, over
constexpr size_t kOffThr = kOffResult + up256((kMaxBins + 2) * sizeof(unsigned long long));   // kMaxBins + 1 thresholds (fp64)
constexpr size_t kOffXyz = kOffThr + up256((kMaxBins + 1) * sizeof(double));     // kMaxRows unit vectors (double4): i-rows, then j-rows
constexpr size_t kScratchBytes = kOffXyz + (size_t)kMaxRows * sizeof(double4);
static_assert(kScratchBytes < (size_t)3 << 20, "the static scratch is meant to stay modest");

// The scratch itself.  In host code this name is only a handle for cudaGetSymbolAddress -- it is NOT a device address.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kT = 256;          // threads per CTA = i-rows per work item (one per thread)
constexpr int kTJ = 256;         // j-rows per work item, staged in shared memory (8 KB)

// RA/Dec (degrees) -> x = cos(dec) cos(ra), y = cos(dec) sin(ra), z = sin(dec), fp64 (reading A8; convert_kernel's arithmetic)
template <typename T>
__global__ void static_convert_kernel(const T* __restrict__ radec, uint32_t n, double4* __restrict__ xyz, unsigned long long* __restrict__ bad) {
    const double kPi = 3.14159265358979323846;
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const double ra = (double)radec[2 * (size_t)k], dec = (double)radec[2 * (size_t)k + 1];
        double4 v = make_double4(1.0, 0.0, 0.0, 0.0);
        if (!(fabs(ra) <= 1.0e6) || !(fabs(dec) <= 90.0)) {      // also NaN and inf
            *bad = 1ull;
        } else {
            const double alpha = ra * kPi / 180.0, delta = dec * kPi / 180.0;
            double sa, ca, sd, cd;
            sincos(alpha, &sa, &ca);
            sincos(delta, &sd, &cd);
            v = make_double4(cd * ca, cd * sa, sd, 0.0);
        }
        xyz[k] = v;
    }
}

// slot: 0 under, 1..n bins, n+1 over; bin k = [T_k, T_{k+1}), last bin closed (reading A5)
__device__ __forceinline__ int static_slot(double d2, const double* __restrict__ thr, int n) {
    d2 = fmin(d2, 4.0);
    if (d2 < thr[0]) return 0;
    if (d2 > thr[n]) return n + 1;
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (thr[mid] <= d2) lo = mid; else hi = mid;
    }
    return lo + 1;
}

// Persistent CTAs take (i-block, j-tile) items off the work counter.  tri: one catalog, pairs i < j only.
__global__ void __launch_bounds__(kT) pair_exact64_static_kernel(unsigned char* __restrict__ scratch, uint32_t n_i, uint32_t n_j, int tri, int nbins) {
    extern __shared__ __align__(16) unsigned char smem[];
    double* thr = reinterpret_cast<double*>(smem);
    double4* tile = reinterpret_cast<double4*>(thr + ((nbins + 1 + 1) & ~1));
    unsigned* hist = reinterpret_cast<unsigned*>(tile + kTJ);
    __shared__ unsigned long long s_item;
    unsigned long long* ctl = reinterpret_cast<unsigned long long*>(scratch + kOffCtl);
    unsigned long long* result = reinterpret_cast<unsigned long long*>(scratch + kOffResult);
    const double* gthr = reinterpret_cast<const double*>(scratch + kOffThr);
    const double4* xi = reinterpret_cast<const double4*>(scratch + kOffXyz);
    const double4* xj = tri ? xi : xi + n_i;
    const int tid = threadIdx.x, nslots = nbins + 2;
    for (int k = tid; k <= nbins; k += kT) thr[k] = gthr[k];
    for (int k = tid; k < nslots; k += kT) hist[k] = 0;
    const uint32_t tiles_j = (n_j + kTJ - 1) / kTJ;
    const unsigned long long n_items = (unsigned long long)((n_i + kT - 1) / kT) * tiles_j;
    unsigned items_done = 0;
    __syncthreads();
    for (;;) {
        if (tid == 0) s_item = atomicAdd(ctl, 1ull);
        __syncthreads();
        const unsigned long long w = s_item;
        __syncthreads();
        if (w >= n_items) break;
        const uint32_t I = (uint32_t)(w / tiles_j), J = (uint32_t)(w % tiles_j);
        const uint32_t j0 = J * kTJ, jn = min((uint32_t)kTJ, n_j - j0);
        if (tri && j0 + jn <= I * kT + 1) continue;        // every j of the tile is <= every i of the block (kT == kTJ)
        if ((uint32_t)tid < jn) tile[tid] = xj[j0 + tid];
        __syncthreads();
        const uint32_t i = I * kT + tid;
        if (i < n_i) {
            const double4 a = xi[i];
            for (uint32_t jj = (tri && j0 <= i) ? i - j0 + 1 : 0; jj < jn; ++jj) {
                const double4 b = tile[jj];
                const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
                atomicAdd(hist + static_slot(fma(dz, dz, fma(dy, dy, dx * dx)), thr, nbins), 1u);
            }
        }
        __syncthreads();
        // at most kT * kTJ = 2^16 pairs per item and slot: a flush every 2^14 items keeps the 32-bit partials below 2^31
        if ((++items_done & 16383u) == 0) {
            for (int k = tid; k < nslots; k += kT) {
                if (hist[k]) atomicAdd(result + k, (unsigned long long)hist[k]);
                hist[k] = 0;
            }
            __syncthreads();
        }
    }
    for (int k = tid; k < nslots; k += kT)
        if (hist[k]) atomicAdd(result + k, (unsigned long long)hist[k]);
}

__global__ void static_finalize_kernel(const unsigned char* __restrict__ scratch, int nslots, unsigned long long* __restrict__ out) {
    const unsigned long long* result = reinterpret_cast<const unsigned long long*>(scratch + kOffResult);
    for (int k = threadIdx.x; k < nslots; k += blockDim.x) out[k] = result[k];
}

// Per-device set-up: the device address of g_static_scratch and the SM count, looked up once per device, with that
// device current.
constexpr int kMaxDevices = 64;
struct DeviceSlot {
    unsigned char* scratch = nullptr;
    int sm_count = 0;
};
std::mutex g_mu;
DeviceSlot g_dev[kMaxDevices];

tpcf_status say(char* err, size_t err_len, tpcf_status s, const std::string& msg) {
    if (err && err_len) std::snprintf(err, err_len, "%s", msg.c_str());
    return s;
}
tpcf_status cuda_say(char* err, size_t err_len, cudaError_t e, const char* what) {
    return say(err, err_len, TPCF_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

}  // namespace

extern "C" tpcf_status tpcf_count_static(int nbins, const double* theta_deg, tpcf_binning mode, const void* radec_i_dev, size_t n_i,
                                         const void* radec_j_dev, size_t n_j, tpcf_dtype dt, uint64_t* hist_dev, void* cuda_stream,
                                         char* err, size_t err_len) {
    if (err && err_len) err[0] = 0;
    if (nbins < 1 || nbins > kMaxBins)
        return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: nbins must be 1.." + std::to_string(kMaxBins) + " (TPCF_STATIC_MAX_BINS)");
    if (!theta_deg || !radec_i_dev || !hist_dev || n_i == 0) return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: NULL argument or empty catalog");
    if (dt != TPCF_F32 && dt != TPCF_F64) return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: dtype must be TPCF_F32 or TPCF_F64");
    const bool tri = radec_j_dev == nullptr;
    if (tri ? n_j != 0 : n_j == 0) return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: n_j must be 0 without a j-catalog and > 0 with one");
    if (n_i > (size_t)kMaxRows || n_j > (size_t)kMaxRows || n_i + n_j > (size_t)kMaxRows)
        return say(err, err_len, TPCF_EINVAL,
                   "tpcf_count_static: " + std::to_string(n_i + n_j) + " rows exceed the static scratch of " + std::to_string(kMaxRows) +
                       " rows (TPCF_STATIC_MAX_ROWS, n_i + n_j); larger catalogs need tpcf_load / tpcf_count, which allocate");
    tpcf::Binning bin;                      // host memory only
    std::string why;
    try {
        why = tpcf::make_binning(nbins, theta_deg, (int)mode, bin);
    } catch (const std::bad_alloc&) {
        return say(err, err_len, TPCF_ENOMEM, "tpcf_count_static: out of host memory");
    }
    if (!why.empty()) return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: " + why);

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cuda_say(err, err_len, e, "no usable CUDA device");      // there is no CPU fallback
    }
    if (dev < 0 || dev >= kMaxDevices) return say(err, err_len, TPCF_ECUDA, "tpcf_count_static: device ordinal beyond 63");
    DeviceSlot slot;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_dev[dev].scratch) {
            // first call on this device: resolve the symbol to the address it has ON THIS DEVICE (the module is loaded here
            // if it was not yet), and check that the device is one this library is built for
            int major = 0, sms = 0;
            e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) return cuda_say(err, err_len, e, "cudaDeviceGetAttribute");
            if (major < 10) return say(err, err_len, TPCF_ECUDA, "libtpcf is built for sm_100a (B200) only");
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p) return cuda_say(err, err_len, e, "cudaGetSymbolAddress(static scratch)");
            g_dev[dev].sm_count = sms;
            g_dev[dev].scratch = static_cast<unsigned char*>(p);
        }
        slot = g_dev[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* S = slot.scratch;
    double4* xyz = reinterpret_cast<double4*>(S + kOffXyz);
    unsigned long long* bad = reinterpret_cast<unsigned long long*>(S + kOffCtl) + 1;
    // the array keeps what the last call left: the work counter, the bad-row flag and the accumulators must start at zero
    e = cudaMemsetAsync(S + kOffCtl, 0, 256, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(S + kOffResult, 0, (size_t)(nbins + 2) * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S + kOffThr, bin.thr.data(), (size_t)(nbins + 1) * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_say(err, err_len, e, "tpcf_count_static: clear scratch");
    const int cgrid_i = (int)((n_i + 255) / 256), cgrid_j = (int)((n_j + 255) / 256);
    if (dt == TPCF_F64) {
        static_convert_kernel<double><<<cgrid_i, 256, 0, st>>>(static_cast<const double*>(radec_i_dev), (uint32_t)n_i, xyz, bad);
        if (!tri) static_convert_kernel<double><<<cgrid_j, 256, 0, st>>>(static_cast<const double*>(radec_j_dev), (uint32_t)n_j, xyz + n_i, bad);
    } else {
        static_convert_kernel<float><<<cgrid_i, 256, 0, st>>>(static_cast<const float*>(radec_i_dev), (uint32_t)n_i, xyz, bad);
        if (!tri) static_convert_kernel<float><<<cgrid_j, 256, 0, st>>>(static_cast<const float*>(radec_j_dev), (uint32_t)n_j, xyz + n_i, bad);
    }
    const uint32_t nj = tri ? (uint32_t)n_i : (uint32_t)n_j;
    const unsigned long long n_items = (unsigned long long)((n_i + kT - 1) / kT) * ((nj + kTJ - 1) / kTJ);
    const int grid = (int)std::min<unsigned long long>(n_items, 4ull * (unsigned long long)slot.sm_count);
    const size_t smem = (size_t)((nbins + 2) & ~1) * sizeof(double) + kTJ * sizeof(double4) + (size_t)(nbins + 2) * sizeof(unsigned);
    static_assert(((kMaxBins + 2) & ~1) * sizeof(double) + kTJ * sizeof(double4) + (kMaxBins + 2) * sizeof(unsigned) <= 48 * 1024 + 16 * 1024,
                  "shared memory of the largest binning");
    if (smem > 48 * 1024) {
        e = cudaFuncSetAttribute(pair_exact64_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return cuda_say(err, err_len, e, "cudaFuncSetAttribute");
    }
    pair_exact64_static_kernel<<<grid, kT, smem, st>>>(S, (uint32_t)n_i, nj, tri ? 1 : 0, nbins);
    static_finalize_kernel<<<1, 256, 0, st>>>(S, nbins + 2, reinterpret_cast<unsigned long long*>(hist_dev));
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_say(err, err_len, e, "tpcf_count_static: kernel launch");
    unsigned long long bad_host = 0;
    e = cudaMemcpyAsync(&bad_host, bad, sizeof(bad_host), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_say(err, err_len, e, "tpcf_count_static");
    if (bad_host) return say(err, err_len, TPCF_EINVAL, "tpcf_count_static: a row has a non-finite value, |RA| > 1e6 or |Dec| > 90");
    return TPCF_OK;
}
