// kernels.cu -- sm_100a kernels of libtpcf.
//
//   convert_kernel      RA/Dec (deg) -> fp64 unit vector + its fp32 rounding          (hot-path step a1)
//   pair_fast_kernel    the all-pairs count: fp32 squared chord, O(1) cell lookup, guard band -> fp64 recheck,
//                       shared-memory partial histogram, uint64 merge                  (steps a3-a7)
//   pair_exact64_kernel plain fp64 count, the device-side cross-check of the fast kernel
//
// What is computed per pair is PAPER.md:37 ("dot product and arc-cosine ... to extract the angle between
// two objects") followed by PAPER.md:38 (histogram fill with shared-memory atomics, partial histograms
// "later combined in a single histogram, in global memory").  How it is computed differs:
// the angle is never formed; |a-b|^2 = 2 - 2 cos(theta) is compared with per-edge thresholds.
#include "kernels.cuh"

namespace tpcf {

namespace {

constexpr int R = kIPerThread;
constexpr int NBUF = 2;                               // j-tile buffers in shared memory
constexpr uint32_t kTileBytes = kTileJ * sizeof(float4);
constexpr uint32_t kSqrtMagic = 0x1FBD1DF5u;
constexpr unsigned long long kFlushPairs = 3500000000ull;   // flush 32-bit partial counters before they can wrap

// ---- small PTX wrappers (mbarrier + bulk async copy, the TMA 1-D path) ---------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}

// ---- exact classification (fp64), shared by the recheck path and the fp64 engine -----------------------
__device__ __forceinline__ double chord2_f64(const double4& a, const double4& b) {
    double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
    return fma(dz, dz, fma(dy, dy, dx * dx));
}
// slot: 0 under, 1..n bins, n+1 over.  Bin k = [T_k, T_{k+1}), last bin closed (reading A5).
__device__ __forceinline__ int exact_slot_dev(double d2, const double* __restrict__ thr, int n) {
    d2 = fmin(d2, 4.0);
    if (d2 < thr[0]) return 0;
    if (d2 > thr[n]) return n + 1;
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (thr[mid] <= d2) lo = mid; else hi = mid;
    }
    return lo + 1;
}

struct SlowCtx {
    const double4* xi64;
    const double4* xj64;
    const double* thr;
    unsigned long long* result;
    unsigned long long* rechecked;
    int nbins;
};

// A pair whose fp32 squared chord fell inside the guard band of a bin edge: classify it from the fp64
// coordinates.  Rare (1e-6 .. 1e-3 of the pairs), so it goes straight to the global histogram.
__device__ __noinline__ void recheck_pair(const SlowCtx* s, uint32_t i, uint32_t j) {
    const double4 a = s->xi64[i], b = s->xj64[j];
    const int slot = exact_slot_dev(chord2_f64(a, b), s->thr, s->nbins);
    atomicAdd(s->result + slot, 1ull);
    atomicAdd(s->rechecked, 1ull);
}

// ---- work items -----------------------------------------------------------------------------------------
struct Item {
    uint32_t I, tile0, ntiles, valid;
};
__device__ __forceinline__ Item decode_item(const PairParams& p, uint32_t w) {
    Item it;
    it.valid = 1;
    if (p.tri) {
        uint32_t lo = 0, hi = p.blocks_i;
        while (hi - lo > 1) {
            uint32_t mid = (lo + hi) >> 1;
            if (p.row_start[mid] <= w) lo = mid; else hi = mid;
        }
        it.I = lo;
        it.tile0 = lo + (w - p.row_start[lo]) * p.chunk;
    } else {
        const uint32_t per_row = (p.tiles_j + p.chunk - 1) / p.chunk;
        it.I = w / per_row;
        it.tile0 = (w % per_row) * p.chunk;
    }
    it.ntiles = min(p.chunk, p.tiles_j - it.tile0);
    return it;
}

template <int MAP>
__device__ __forceinline__ uint32_t cell_byte_offset(float d2, int shift, float scale, float clamp) {
    if (MAP == (int)CellMap::LogBits) {
        return (__float_as_uint(d2) >> (shift - 3)) & ~7u;
    } else {
        const float c = fminf(d2, clamp);
        const float key = __uint_as_float((__float_as_uint(c) >> 1) + kSqrtMagic);
        const float t = fmaf(key, scale, 8388608.0f);
        return (__float_as_uint(t) << 3) & 0x3FFFFF8u;
    }
}

// One 1024-point j-tile against the CTA's 1024 register-resident i-points.
template <int MAP, bool DIAG>
__device__ __forceinline__ void tile_pairs(const float4* __restrict__ jt, const float (&ax)[R], const float (&ay)[R],
                                           const float (&az)[R], const char* lut, char* hist, const SlowCtx* slow,
                                           uint32_t i0 /* global index of this thread's r = 0 point */,
                                           uint32_t j0 /* global index of the tile's first point */, int shift,
                                           float scale, float clamp) {
#pragma unroll 2
    for (int jj = 0; jj < kTileJ; ++jj) {
        const float4 b = jt[jj];                                  // one LDS.128, broadcast to the warp
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float dx = ax[r] - b.x, dy = ay[r] - b.y, dz = az[r] - b.z;
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const uint32_t q8 = cell_byte_offset<MAP>(d2, shift, scale, clamp);
            const float2 lh = *reinterpret_cast<const float2*>(lut + q8);
            const bool above = d2 >= lh.x;
            const bool amb = above && (d2 < lh.y);
            const bool valid = !DIAG || (j0 + jj > i0 + r * kThreads);
            if (amb) {
                if (valid) recheck_pair(slow, i0 + r * kThreads, j0 + jj);
            } else if (valid) {
                atomicAdd(reinterpret_cast<unsigned*>(hist + q8) + (above ? 1 : 0), 1u);
            }
        }
    }
}

// Add the CTA's 32-bit partial counters into the global uint64 result (integer adds: order-independent,
// hence deterministic) and clear them.
__device__ __forceinline__ void flush_hist(unsigned* hist, int nslots, const uint16_t* __restrict__ slotmap,
                                           unsigned long long* result) {
    __syncthreads();
    for (int s = threadIdx.x; s < nslots; s += kThreads) {
        const unsigned v = hist[s];
        if (v) {
            atomicAdd(result + slotmap[s], (unsigned long long)v);
            hist[s] = 0;
        }
    }
    __syncthreads();
}

template <int MAP>
__global__ void __launch_bounds__(kThreads, 3) pair_fast_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    float4* jbuf = reinterpret_cast<float4*>(smem);
    char* lut = reinterpret_cast<char*>(smem + NBUF * kTileBytes);
    unsigned* hist = reinterpret_cast<unsigned*>(lut + (size_t)p.ncells * 8);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(hist) + (size_t)p.ncells * 8);
    Item* s_item = reinterpret_cast<Item*>(bars + NBUF);
    SlowCtx* slow = reinterpret_cast<SlowCtx*>(s_item + 1);

    const int tid = threadIdx.x;
    for (int c = tid; c < p.ncells; c += kThreads) {
        reinterpret_cast<float2*>(lut)[c] = p.lut[c];
        hist[2 * c] = 0;
        hist[2 * c + 1] = 0;
    }
    if (tid == 0) {
        for (int b = 0; b < NBUF; ++b) mbar_init(smem_u32(bars + b), 1);
        fence_barrier_init();
        slow->xi64 = p.xi64;
        slow->xj64 = p.xj64;
        slow->thr = p.thr;
        slow->result = p.result;
        slow->rechecked = p.counters + 1;
        slow->nbins = p.nbins;
    }
    __syncthreads();

    uint32_t tiles_done = 0;                // tiles this CTA consumed so far: selects buffer and mbarrier parity
    unsigned long long pairs_since_flush = 0, items_done = 0;
    for (;;) {
        if (tid == 0) {
            const unsigned long long c = atomicAdd(p.counters, 1ull);
            Item it;
            it.valid = 0;
            if (c < p.n_items_part) it = decode_item(p, (uint32_t)c * p.nparts + p.part);
            *s_item = it;
        }
        __syncthreads();
        const Item it = *s_item;
        if (!it.valid) break;

        // this thread's R i-points (rows past the end of the catalog become (-2,-2,-2): d2 >= 6 against
        // every real point and 48 against a (2,2,2) padding row, i.e. always in the discard range)
        const uint32_t i0 = it.I * kTileI + tid;
        float ax[R], ay[R], az[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const uint32_t i = i0 + r * kThreads;
            float4 a = p.xi[i];
            if (i >= p.n_i) a = make_float4(-kPadCoord, -kPadCoord, -kPadCoord, 0.f);
            ax[r] = a.x;
            ay[r] = a.y;
            az[r] = a.z;
        }
        if (tid == 0) {
            fence_proxy_async();
            for (uint32_t t = 0; t < it.ntiles && t < NBUF; ++t) {
                const uint32_t g = tiles_done + t, bar = smem_u32(bars + g % NBUF);
                mbar_expect_tx(bar, kTileBytes);
                bulk_g2s(smem_u32(jbuf + (size_t)(g % NBUF) * kTileJ), p.xj + (size_t)(it.tile0 + t) * kTileJ, kTileBytes, bar);
            }
        }
        for (uint32_t t = 0; t < it.ntiles; ++t) {
            const uint32_t g = tiles_done + t, buf = g % NBUF;
            mbar_wait(smem_u32(bars + buf), (g / NBUF) & 1);
            const float4* jt = jbuf + (size_t)buf * kTileJ;
            const uint32_t j0 = (it.tile0 + t) * kTileJ;
            if (p.tri && it.tile0 + t == it.I)
                tile_pairs<MAP, true>(jt, ax, ay, az, lut, reinterpret_cast<char*>(hist), slow, i0, j0, p.shift, p.sqrt_scale, p.sqrt_clamp);
            else
                tile_pairs<MAP, false>(jt, ax, ay, az, lut, reinterpret_cast<char*>(hist), slow, i0, j0, p.shift, p.sqrt_scale, p.sqrt_clamp);
            __syncthreads();                // every warp is done reading buffer `buf`
            if (tid == 0 && t + NBUF < it.ntiles) {
                const uint32_t bar = smem_u32(bars + buf);
                mbar_expect_tx(bar, kTileBytes);
                bulk_g2s(smem_u32(jbuf + (size_t)buf * kTileJ), p.xj + (size_t)(it.tile0 + t + NBUF) * kTileJ, kTileBytes, bar);
            }
        }
        tiles_done += it.ntiles;
        ++items_done;
        pairs_since_flush += (unsigned long long)it.ntiles * kTileI * kTileJ;
        if (pairs_since_flush > kFlushPairs) {
            flush_hist(hist, 2 * p.ncells, p.slotmap, p.result);
            pairs_since_flush = 0;
        }
    }
    flush_hist(hist, 2 * p.ncells, p.slotmap, p.result);
    if (tid == 0 && items_done) atomicAdd(p.counters + 2, items_done);
}

// ---- fp64 engine: same plan, no tables, no shared-memory tiles -----------------------------------------
__global__ void __launch_bounds__(kThreads) pair_exact64_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    double* thr = reinterpret_cast<double*>(smem);
    unsigned* hist = reinterpret_cast<unsigned*>(thr + p.nbins + 1);
    __shared__ Item s_item;
    const int tid = threadIdx.x, nslots = p.nbins + 3;
    for (int k = tid; k <= p.nbins; k += kThreads) thr[k] = p.thr[k];
    for (int k = tid; k < nslots; k += kThreads) hist[k] = 0;
    __syncthreads();
    unsigned long long items_done = 0;
    for (;;) {
        if (tid == 0) {
            const unsigned long long c = atomicAdd(p.counters, 1ull);
            Item it;
            it.valid = 0;
            if (c < p.n_items_part) it = decode_item(p, (uint32_t)c * p.nparts + p.part);
            s_item = it;
        }
        __syncthreads();
        const Item it = s_item;
        __syncthreads();
        if (!it.valid) break;
        const uint32_t i0 = it.I * kTileI + tid;
        for (int r = 0; r < R; ++r) {
            const uint32_t i = i0 + r * kThreads;
            if (i >= p.n_i) continue;
            const double4 a = p.xi64[i];
            const uint32_t jbeg = it.tile0 * kTileJ, jend = min(p.n_j, (it.tile0 + it.ntiles) * kTileJ);
            for (uint32_t j = jbeg; j < jend; ++j) {
                if (p.tri && j <= i) continue;
                const int slot = exact_slot_dev(chord2_f64(a, p.xj64[j]), thr, p.nbins);
                atomicAdd(hist + slot, 1u);
            }
        }
        ++items_done;
        // at most kMaxChunk * 2^20 pairs per item and slot; flush well before 2^32
        if ((items_done & 255) == 0) {
            __syncthreads();
            for (int k = tid; k < nslots; k += kThreads) {
                if (hist[k]) atomicAdd(p.result + k, (unsigned long long)hist[k]);
                hist[k] = 0;
            }
            __syncthreads();
        }
    }
    __syncthreads();
    for (int k = tid; k < nslots; k += kThreads)
        if (hist[k]) atomicAdd(p.result + k, (unsigned long long)hist[k]);
    if (tid == 0 && items_done) atomicAdd(p.counters + 2, items_done);
}

// ---- load / convert (step a1) -----------------------------------------------------------------------------
// x = cos(dec) cos(ra), y = cos(dec) sin(ra), z = sin(dec) in fp64 (reading A8); the fp32 copy is that
// vector rounded once (reading A17).  Rows n..n_pad-1 become the padding point (2,2,2).
template <typename T>
__global__ void convert_kernel(const T* __restrict__ radec, uint64_t n, uint64_t n_pad, double4* __restrict__ x64,
                               float4* __restrict__ x32, int* __restrict__ bad) {
    const double kPi = 3.14159265358979323846;
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
        if (k < n) {
            const double ra = (double)radec[2 * k], dec = (double)radec[2 * k + 1];
            if (!(fabs(ra) <= 1.0e6) || !(fabs(dec) <= 90.0)) {      // also catches NaN and inf
                *bad = 1;
            } else {
                const double alpha = ra * kPi / 180.0, delta = dec * kPi / 180.0;
                double sa, ca, sd, cd;
                sincos(alpha, &sa, &ca);
                sincos(delta, &sd, &cd);
                v = make_double4(cd * ca, cd * sa, sd, 0.0);
            }
        }
        x64[k] = v;
        x32[k] = make_float4((float)v.x, (float)v.y, (float)v.z, 0.f);
    }
}

__global__ void gather_kernel(const double4* __restrict__ src64, const float4* __restrict__ src32,
                              const int64_t* __restrict__ rows, uint64_t nrows, uint64_t nrows_pad, uint64_t n_src,
                              double4* __restrict__ dst64, float4* __restrict__ dst32, int* __restrict__ bad) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < nrows_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
        float4 f = make_float4(kPadCoord, kPadCoord, kPadCoord, 0.f);
        if (k < nrows) {
            const int64_t r = rows[k];
            if (r < 0 || (uint64_t)r >= n_src) {
                *bad = 1;
            } else {
                v = src64[r];
                f = src32[r];
            }
        }
        dst64[k] = v;
        dst32[k] = f;
    }
}

__global__ void finalize_kernel(const unsigned long long* __restrict__ result, int nbins, int zero_slot,
                                unsigned long long self_pairs, unsigned long long* __restrict__ out) {
    for (int k = threadIdx.x; k < nbins + 2; k += blockDim.x) out[k] = result[k] - (k == zero_slot ? self_pairs : 0ull);
}

size_t fast_smem_bytes(int ncells) {
    return (size_t)NBUF * kTileBytes + (size_t)ncells * 16 + NBUF * 8 + sizeof(Item) + sizeof(SlowCtx) + 64;
}

}  // namespace

cudaError_t launch_convert(const void* radec, int is_f64, uint64_t n, uint64_t n_pad, double4* x64, float4* x32,
                           int* bad_flag, cudaStream_t st) {
    const int block = 256;
    const int grid = (int)std::min<uint64_t>((n_pad + block - 1) / block, 148ull * 16);
    if (is_f64)
        convert_kernel<double><<<grid, block, 0, st>>>(static_cast<const double*>(radec), n, n_pad, x64, x32, bad_flag);
    else
        convert_kernel<float><<<grid, block, 0, st>>>(static_cast<const float*>(radec), n, n_pad, x64, x32, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_gather(const double4* src64, const float4* src32, const int64_t* rows, uint64_t nrows,
                          uint64_t nrows_pad, uint64_t n_src, double4* dst64, float4* dst32, int* bad_flag,
                          cudaStream_t st) {
    const int block = 256;
    const int grid = (int)std::min<uint64_t>((nrows_pad + block - 1) / block, 148ull * 16);
    gather_kernel<<<grid, block, 0, st>>>(src64, src32, rows, nrows, nrows_pad, n_src, dst64, dst32, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_pairs_fast(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info) {
    const size_t smem = fast_smem_bytes(p.ncells);
    auto kern = (map == CellMap::LogBits) ? pair_fast_kernel<(int)CellMap::LogBits> : pair_fast_kernel<(int)CellMap::SqrtLin>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    // persistent CTAs: a whole number of CTAs per SM, never more than there are work items
    int grid = (int)std::min<uint64_t>((uint64_t)sm_count * per_sm, std::max<uint32_t>(p.n_items_part, 1));
    kern<<<grid, kThreads, smem, st>>>(p);
    if (info) *info = LaunchInfo{grid, kThreads, (int)smem, 1};
    return cudaGetLastError();
}

cudaError_t launch_pairs_exact64(const PairParams& p, int sm_count, cudaStream_t st, LaunchInfo* info) {
    const size_t smem = (size_t)(p.nbins + 1) * 8 + (size_t)(p.nbins + 3) * 4;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pair_exact64_kernel, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    int grid = (int)std::min<uint64_t>((uint64_t)sm_count * per_sm, std::max<uint32_t>(p.n_items_part, 1));
    pair_exact64_kernel<<<grid, kThreads, smem, st>>>(p);
    if (info) *info = LaunchInfo{grid, kThreads, (int)smem, 1};
    return cudaGetLastError();
}

cudaError_t launch_finalize(const unsigned long long* result, int nbins, int zero_slot, unsigned long long self_pairs,
                            unsigned long long* out, cudaStream_t st) {
    finalize_kernel<<<1, 256, 0, st>>>(result, nbins, zero_slot, self_pairs, out);
    return cudaGetLastError();
}

}  // namespace tpcf
