// kernels.cu -- sm_100a kernels of libtpcf.
//
//   convert_kernel      RA/Dec (deg) -> fp64 unit vector + Hilbert key                  (hot-path step a1)
//   radix_* / permute / spheres   spatial sort of the catalog, fp32 copy, subtile bounding spheres (a1)
//   pair_fast_kernel    the all-pairs count: fp32 squared chord; per (lane, 32-row j-subtile) window of
//                       candidate bin edges from bounding spheres -> 1..3 threshold compares per pair with
//                       register counters, else O(1) cell lookup + shared-memory partial histogram;
//                       guard band -> fp64 recheck; uint64 merge                        (steps a3-a7)
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

// ---- per-pair cell-lookup path ("lookup" path) ---------------------------------------------------------------
// One pair: fp32 squared chord -> cell -> (lo, hi) of the cell's guard band -> shared-memory partial histogram,
// or the fp64 recheck when lo <= d2 < hi.
template <int MAP>
__device__ __forceinline__ void lookup_pair(float ax, float ay, float az, const float4& b, const char* lut, char* hist,
                                            const SlowCtx* slow, uint32_t i, uint32_t j, bool valid, int shift,
                                            float scale, float clamp) {
    const float dx = ax - b.x, dy = ay - b.y, dz = az - b.z;
    const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const uint32_t q8 = cell_byte_offset<MAP>(d2, shift, scale, clamp);
    const float2 lh = *reinterpret_cast<const float2*>(lut + q8);
    const bool above = d2 >= lh.x;
    const bool amb = above && (d2 < lh.y);
    if (amb) {
        if (valid) recheck_pair(slow, i, j);
    } else if (valid) {
        atomicAdd(reinterpret_cast<unsigned*>(hist + q8) + (above ? 1 : 0), 1u);
    }
}

// nj consecutive j-points against this thread's R register-resident i-points, every pair by cell lookup.
template <int MAP, bool DIAG>
__device__ __forceinline__ void lookup_block(const float4* __restrict__ jt, int nj, const float (&ax)[R],
                                             const float (&ay)[R], const float (&az)[R], const char* lut, char* hist,
                                             const SlowCtx* slow, uint32_t i0 /* global index of this thread's r = 0 point */,
                                             uint32_t j0 /* global index of jt[0] */, int shift, float scale, float clamp) {
#pragma unroll 2
    for (int jj = 0; jj < nj; ++jj) {
        const float4 b = jt[jj];                                  // one LDS.128, broadcast to the warp
#pragma unroll
        for (int r = 0; r < R; ++r)
            lookup_pair<MAP>(ax[r], ay[r], az[r], b, lut, hist, slow, i0 + r, j0 + jj, !DIAG || (j0 + jj > i0 + r), shift,
                             scale, clamp);
    }
}

// ---- window path ----------------------------------------------------------------------------------------------
// For one lane (R consecutive rows of the spatially sorted i-catalog, bounding sphere (ci, ri)) and one j-subtile
// (kSubJ consecutive rows, bounding sphere sp): every TRUE chord of the block lies in [dc - ri - rj, dc + ri + rj]
// (triangle inequality in R^3).  Returns squared bounds made safe against the fp32 evaluation of the geometry.
__device__ __forceinline__ void chord_bounds(float cx, float cy, float cz, float ri, const float4& sp, float& lo2,
                                             float& hi2) {
    const float dx = cx - sp.x, dy = cy - sp.y, dz = cz - sp.z;
    const float dc2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float dc;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(dc) : "f"(dc2));
    const float rs = ri + sp.w;
    const float lo = fmaf(dc, 1.0f - 4.0e-6f, -rs) - 4.0e-7f;
    const float hi = fmaf(dc, 1.0f + 4.0e-6f, rs) + 4.0e-7f;
    lo2 = lo > 0.f ? __fmul_rd(lo, lo) : 0.f;
    hi2 = __fmul_ru(hi, hi);
}

// The E-edge window loop: counts, for the kSubJ x R pairs of the block, how many have q < mid_e for each of the
// bands k .. k+E-1 (q = fp32 squared chord, accumulated starting from -mid_0 so that the test is a sign bit),
// and tracks the smallest |q - mid_e| seen.  Returns true when some pair came within a band's half width: the
// counters of this lane are then not used and the block is recounted pair by pair.
template <int E>
__device__ __forceinline__ bool window_block(const float4* __restrict__ jt, const float (&ax)[R], const float (&ay)[R],
                                             const float (&az)[R], const float2* __restrict__ band_mh, int k,
                                             unsigned (&c)[E]) {
    const float2 mh0 = band_mh[k];
    const float nm0 = -mh0.x;
    float hmax = mh0.y, dt[E];
    dt[0] = 0.f;
#pragma unroll
    for (int e = 1; e < E; ++e) {
        const float2 mh = band_mh[k + e];
        dt[e] = __fsub_rn(mh0.x, mh.x);
        hmax = fmaxf(hmax, mh.y);
    }
#pragma unroll
    for (int e = 0; e < E; ++e) c[e] = 0;
    float m = 3.0e38f;
#pragma unroll 8
    for (int jj = 0; jj < kSubJ; ++jj) {
        const float4 b = jt[jj];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float dx = __fsub_rn(ax[r], b.x), dy = __fsub_rn(ay[r], b.y), dz = __fsub_rn(az[r], b.z);
            const float q = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, nm0)));
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const float qe = e ? __fadd_rn(q, dt[e]) : q;
                c[e] += __float_as_uint(qe) >> 31;
                m = fminf(m, fabsf(qe));
            }
        }
    }
    return m <= hmax;
}

struct WinTables {
    const float2* band_mh;
    const float2* band_lh;
    const uint16_t* band_slot;
    const uint16_t* cell_band;
    unsigned* whist;            // partial histogram indexed by result slot
    int nbands;
};

// One 1024-point j-tile against the CTA's 1024 register-resident i-points, subtile by subtile.
template <int MAP, bool DIAG>
__device__ __forceinline__ void tile_pairs(const float4* __restrict__ jt, const float4* __restrict__ jsph, bool windows,
                                           const float (&ax)[R], const float (&ay)[R], const float (&az)[R], float cx,
                                           float cy, float cz, float ri, const WinTables& wt, const char* lut, char* hist,
                                           const SlowCtx* slow, uint32_t i0, uint32_t j0, int shift, float scale,
                                           float clamp, unsigned (&npath)[5]) {
    if (DIAG || !windows) {
        lookup_block<MAP, DIAG>(jt, kTileJ, ax, ay, az, lut, hist, slow, i0, j0, shift, scale, clamp);
        npath[3] += kTileJ / kSubJ;
        return;
    }
    const int lane = threadIdx.x & 31;
    for (int sub = 0; sub < kTileJ / kSubJ; ++sub) {
        const float4* js = jt + sub * kSubJ;
        float lo2, hi2;
        chord_bounds(cx, cy, cz, ri, jsph[sub], lo2, hi2);
        // first band that is not wholly below the window, then how many bands the window reaches
        int k = wt.cell_band[cell_byte_offset<MAP>(lo2, shift, scale, clamp) >> 3];
        while (k < wt.nbands && wt.band_lh[k].y <= lo2) ++k;
        int e = 1;
        while (e <= kMaxWinEdges && k + e < wt.nbands && wt.band_lh[k + e].x <= hi2) ++e;
        const int emax = __reduce_max_sync(0xffffffffu, e);
        if (emax > kMaxWinEdges) {
            lookup_block<MAP, false>(js, kSubJ, ax, ay, az, lut, hist, slow, i0, j0 + sub * kSubJ, shift, scale, clamp);
            ++npath[3];
            continue;
        }
        // every lane runs the emax-edge loop on bands k .. k+emax-1; lowering k keeps the window inside them
        k = min(k, wt.nbands - emax);
        unsigned cnt[kMaxWinEdges + 1];
        bool flagged;
        if (emax == 1) {
            unsigned c[1];
            flagged = window_block<1>(js, ax, ay, az, wt.band_mh, k, c);
            cnt[0] = c[0];
            cnt[1] = kSubJ * R - c[0];
            cnt[2] = cnt[3] = 0;
            ++npath[0];
        } else if (emax == 2) {
            unsigned c[2];
            flagged = window_block<2>(js, ax, ay, az, wt.band_mh, k, c);
            cnt[0] = c[0];
            cnt[1] = c[1] - c[0];
            cnt[2] = kSubJ * R - c[1];
            cnt[3] = 0;
            ++npath[1];
        } else {
            unsigned c[3];
            flagged = window_block<3>(js, ax, ay, az, wt.band_mh, k, c);
            cnt[0] = c[0];
            cnt[1] = c[1] - c[0];
            cnt[2] = c[2] - c[1];
            cnt[3] = kSubJ * R - c[2];
            ++npath[2];
        }
        if (!flagged) {
#pragma unroll
            for (int t = 0; t <= kMaxWinEdges; ++t)
                if (cnt[t]) atomicAdd(wt.whist + wt.band_slot[k + t], cnt[t]);      // cnt[t] != 0 only for t <= emax
        }
        // lanes that saw a pair inside a guard band: the warp recounts their kSubJ x R pairs together, lane l
        // taking j-point l, through the cell-lookup path (which sends the ambiguous pairs to the fp64 recheck)
        unsigned todo = __ballot_sync(0xffffffffu, flagged);
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            const float4 b = js[lane];
            const uint32_t isrc = i0 + (uint32_t)(src - lane) * R;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float sx = __shfl_sync(0xffffffffu, ax[r], src), sy = __shfl_sync(0xffffffffu, ay[r], src),
                            sz = __shfl_sync(0xffffffffu, az[r], src);
                lookup_pair<MAP>(sx, sy, sz, b, lut, hist, slow, isrc + r, j0 + sub * kSubJ + lane, true, shift, scale, clamp);
            }
            ++npath[4];
        }
    }
}

// Add the CTA's 32-bit partial counters into the global uint64 result (integer adds: order-independent,
// hence deterministic) and clear them.
__device__ __forceinline__ void flush_hist(unsigned* hist, int nslots, const uint16_t* __restrict__ slotmap,
                                           unsigned* whist, int nres, unsigned long long* result) {
    __syncthreads();
    for (int s = threadIdx.x; s < nslots; s += kThreads) {
        const unsigned v = hist[s];
        if (v) {
            atomicAdd(result + slotmap[s], (unsigned long long)v);
            hist[s] = 0;
        }
    }
    for (int s = threadIdx.x; s < nres; s += kThreads) {
        const unsigned v = whist[s];
        if (v) {
            atomicAdd(result + s, (unsigned long long)v);
            whist[s] = 0;
        }
    }
    __syncthreads();
}

constexpr uint32_t kSphBytes = (kTileJ / kSubJ) * sizeof(float4);
static_assert(kSubJ == 32, "the recount of a flagged lane gives j-point l of the subtile to lane l");
static_assert(kIPerThread == 4, "window_block's pair count assumes R = 4");

// shared-memory layout of pair_fast_kernel (byte offsets; every array 16-byte aligned)
__host__ __device__ inline uint32_t up(uint32_t x) { return (x + 15u) & ~15u; }
struct FastSmem {
    uint32_t jbuf, jsph, lut, hist, band_mh, band_lh, whist, cell_band, band_slot, bars, item, slow, total;
};
__host__ __device__ inline FastSmem fast_smem_layout(int ncells, int nbands, int nbins) {
    FastSmem L;
    uint32_t o = 0;
    L.jbuf = o;       o += NBUF * kTileBytes;
    L.jsph = o;       o += NBUF * kSphBytes;
    L.lut = o;        o = up(o + (uint32_t)ncells * 8);
    L.hist = o;       o = up(o + (uint32_t)ncells * 8);
    L.band_mh = o;    o = up(o + (uint32_t)nbands * 8);
    L.band_lh = o;    o = up(o + (uint32_t)nbands * 8);
    L.whist = o;      o = up(o + (uint32_t)(nbins + 3) * 4);
    L.cell_band = o;  o = up(o + (uint32_t)ncells * 2);
    L.band_slot = o;  o = up(o + (uint32_t)(nbands + 1) * 2);
    L.bars = o;       o += 16 * ((NBUF * 8 + 15) / 16);
    L.item = o;       o += 16;
    L.slow = o;       o = up(o + (uint32_t)sizeof(SlowCtx));
    L.total = o;
    return L;
}

template <int MAP>
__global__ void __launch_bounds__(kThreads, 3) pair_fast_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const FastSmem L = fast_smem_layout(p.ncells, p.nbands, p.nbins);
    float4* jbuf = reinterpret_cast<float4*>(smem + L.jbuf);
    float4* jsph = reinterpret_cast<float4*>(smem + L.jsph);
    char* lut = reinterpret_cast<char*>(smem + L.lut);
    unsigned* hist = reinterpret_cast<unsigned*>(smem + L.hist);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem + L.bars);
    Item* s_item = reinterpret_cast<Item*>(smem + L.item);
    SlowCtx* slow = reinterpret_cast<SlowCtx*>(smem + L.slow);
    WinTables wt;
    wt.band_mh = reinterpret_cast<const float2*>(smem + L.band_mh);
    wt.band_lh = reinterpret_cast<const float2*>(smem + L.band_lh);
    wt.band_slot = reinterpret_cast<const uint16_t*>(smem + L.band_slot);
    wt.cell_band = reinterpret_cast<const uint16_t*>(smem + L.cell_band);
    wt.whist = reinterpret_cast<unsigned*>(smem + L.whist);
    wt.nbands = p.nbands;
    const bool windows = p.sph_j != nullptr;
    const uint32_t tile_tx = kTileBytes + (windows ? kSphBytes : 0u);

    const int tid = threadIdx.x;
    for (int c = tid; c < p.ncells; c += kThreads) {
        reinterpret_cast<float2*>(lut)[c] = p.lut[c];
        hist[2 * c] = 0;
        hist[2 * c + 1] = 0;
        reinterpret_cast<uint16_t*>(smem + L.cell_band)[c] = p.cell_band[c];
    }
    for (int b = tid; b < p.nbands; b += kThreads) {
        reinterpret_cast<float2*>(smem + L.band_mh)[b] = p.band_mh[b];
        reinterpret_cast<float2*>(smem + L.band_lh)[b] = p.band_lh[b];
    }
    for (int b = tid; b <= p.nbands; b += kThreads) reinterpret_cast<uint16_t*>(smem + L.band_slot)[b] = p.band_slot[b];
    for (int b = tid; b < p.nbins + 3; b += kThreads) wt.whist[b] = 0;
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

    auto fetch_tile = [&](uint32_t g, uint32_t tile) {      // one elected thread: TMA bulk copies behind one mbarrier
        const uint32_t buf = g % NBUF, bar = smem_u32(bars + buf);
        mbar_expect_tx(bar, tile_tx);
        bulk_g2s(smem_u32(jbuf + (size_t)buf * kTileJ), p.xj + (size_t)tile * kTileJ, kTileBytes, bar);
        if (windows)
            bulk_g2s(smem_u32(jsph + (size_t)buf * (kTileJ / kSubJ)), p.sph_j + (size_t)tile * (kTileJ / kSubJ), kSphBytes, bar);
    };

    uint32_t tiles_done = 0;                // tiles this CTA consumed so far: selects buffer and mbarrier parity
    unsigned long long pairs_since_flush = 0, items_done = 0;
    unsigned npath[5] = {0, 0, 0, 0, 0};
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

        // this thread's R consecutive i-points (rows past the end of the catalog become (-2,-2,-2): d2 >= 6
        // against every real point and 48 against a (2,2,2) padding row, i.e. always in the discard range)
        const uint32_t i0 = it.I * kTileI + tid * R;
        float ax[R], ay[R], az[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const uint32_t i = i0 + r;
            float4 a = p.xi[i];
            if (i >= p.n_i) a = make_float4(-kPadCoord, -kPadCoord, -kPadCoord, 0.f);
            ax[r] = a.x;
            ay[r] = a.y;
            az[r] = a.z;
        }
        // bounding sphere of the lane's R points around their mean; the radius also covers the distance of the
        // fp64 points from their fp32 roundings (<= 5.2e-8) and the rounding of this evaluation
        const float cx = 0.25f * ((ax[0] + ax[1]) + (ax[2] + ax[3])), cy = 0.25f * ((ay[0] + ay[1]) + (ay[2] + ay[3])),
                    cz = 0.25f * ((az[0] + az[1]) + (az[2] + az[3]));
        float ri2 = 0.f;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float dx = ax[r] - cx, dy = ay[r] - cy, dz = az[r] - cz;
            ri2 = fmaxf(ri2, fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
        }
        const float ri = fmaf(sqrtf(ri2), 1.0f + 4.0e-6f, 2.0e-7f);

        if (tid == 0) {
            fence_proxy_async();
            for (uint32_t t = 0; t < it.ntiles && t < NBUF; ++t) fetch_tile(tiles_done + t, it.tile0 + t);
        }
        for (uint32_t t = 0; t < it.ntiles; ++t) {
            const uint32_t g = tiles_done + t, buf = g % NBUF;
            mbar_wait(smem_u32(bars + buf), (g / NBUF) & 1);
            const float4* jt = jbuf + (size_t)buf * kTileJ;
            const float4* js = jsph + (size_t)buf * (kTileJ / kSubJ);
            const uint32_t j0 = (it.tile0 + t) * kTileJ;
            if (p.tri && it.tile0 + t == it.I)
                tile_pairs<MAP, true>(jt, js, windows, ax, ay, az, cx, cy, cz, ri, wt, lut, reinterpret_cast<char*>(hist), slow,
                                      i0, j0, p.shift, p.sqrt_scale, p.sqrt_clamp, npath);
            else
                tile_pairs<MAP, false>(jt, js, windows, ax, ay, az, cx, cy, cz, ri, wt, lut, reinterpret_cast<char*>(hist), slow,
                                       i0, j0, p.shift, p.sqrt_scale, p.sqrt_clamp, npath);
            __syncthreads();                // every warp is done reading buffer `buf`
            if (tid == 0 && t + NBUF < it.ntiles) fetch_tile(g + NBUF, it.tile0 + t + NBUF);
        }
        tiles_done += it.ntiles;
        ++items_done;
        pairs_since_flush += (unsigned long long)it.ntiles * kTileI * kTileJ;
        if (pairs_since_flush > kFlushPairs) {
            flush_hist(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result);
            pairs_since_flush = 0;
        }
    }
    flush_hist(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result);
    if (tid == 0 && items_done) atomicAdd(p.counters + 2, items_done);
    if ((tid & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 5; ++k)
            if (npath[k]) atomicAdd(p.counters + 3 + k, (unsigned long long)npath[k]);
    }
}

// ---- fp64 engine: same plan, no tables, no shared-memory tiles -----------------------------------------
__global__ void __launch_bounds__(kThreads) pair_exact64_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
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
        const uint32_t i0 = it.I * kTileI + tid * R;
        for (int r = 0; r < R; ++r) {
            const uint32_t i = i0 + r;
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

// ---- load / convert / spatial sort (step a1) -------------------------------------------------------------------
// 63-bit Hilbert-curve index of a point of [-1, 1]^3 quantised to 21 bits per axis (Skilling's transpose
// algorithm).  Only the ORDER it induces is used: consecutive rows of the sorted catalog are close on the sky,
// which is what makes the bounding spheres of the window path small.  Counts do not depend on it.
__device__ inline unsigned long long hilbert_key(double x, double y, double z) {
    constexpr int B = 21;
    uint32_t X[3];
    const double v[3] = {x, y, z};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double t = (v[k] + 1.0) * (double)(1u << (B - 1));
        t = fmin(fmax(t, 0.0), (double)((1u << B) - 1));
        X[k] = (uint32_t)t;
    }
    const uint32_t M = 1u << (B - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {          // inverse undo
        const uint32_t P = Q - 1;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) {
                X[0] ^= P;
            } else {
                const uint32_t t = (X[0] ^ X[i]) & P;
                X[0] ^= t;
                X[i] ^= t;
            }
        }
    }
    X[1] ^= X[0];                                    // Gray encode
    X[2] ^= X[1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t;
    X[1] ^= t;
    X[2] ^= t;
    unsigned long long key = 0;
    for (int b = B - 1; b >= 0; --b) {
#pragma unroll
        for (int k = 0; k < 3; ++k) key = (key << 1) | ((X[k] >> b) & 1u);
    }
    return key;
}

// x = cos(dec) cos(ra), y = cos(dec) sin(ra), z = sin(dec) in fp64 (reading A8), in the caller's row order.
template <typename T>
__global__ void convert_kernel(const T* __restrict__ radec, uint64_t n, double4* __restrict__ x64_rows,
                               unsigned long long* __restrict__ keys, uint32_t* __restrict__ idx, int* __restrict__ bad) {
    const double kPi = 3.14159265358979323846;
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4(1.0, 0.0, 0.0, 0.0);
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
        x64_rows[k] = v;
        keys[k] = hilbert_key(v.x, v.y, v.z);
        idx[k] = (uint32_t)k;
    }
}

// ---- stable LSD radix sort of (key, idx) pairs, 8 bits per pass ----------------------------------------------
// Block b owns elements [b * kSortChunk, (b+1) * kSortChunk).  counts is digit-major: counts[d * nblk + b].
__global__ void radix_hist_kernel(const unsigned long long* __restrict__ keys, uint32_t n, int shift,
                                  uint32_t* __restrict__ counts, uint32_t nblk) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kSortChunk;
    for (uint32_t t = threadIdx.x; t < kSortChunk; t += 256) {
        const uint32_t k = base + t;
        if (k < n) atomicAdd(&h[(uint32_t)(keys[k] >> shift) & 255u], 1u);
    }
    __syncthreads();
    counts[threadIdx.x * nblk + blockIdx.x] = h[threadIdx.x];
}

// exclusive prefix sum of `total` words in place, one block of 1024 threads
__global__ void radix_scan_kernel(uint32_t* __restrict__ counts, uint32_t total) {
    __shared__ uint32_t part[1024];
    const uint32_t per = (total + 1023u) / 1024u, lo = min(total, threadIdx.x * per), hi = min(total, lo + per);
    uint32_t sum = 0;
    for (uint32_t k = lo; k < hi; ++k) sum += counts[k];
    part[threadIdx.x] = sum;
    __syncthreads();
    for (uint32_t off = 1; off < 1024; off <<= 1) {      // Hillis-Steele inclusive scan
        const uint32_t v = (threadIdx.x >= off) ? part[threadIdx.x - off] : 0u;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = part[threadIdx.x] - sum;
    for (uint32_t k = lo; k < hi; ++k) {
        const uint32_t c = counts[k];
        counts[k] = run;
        run += c;
    }
}

// one warp per block walks its chunk in rows of 32: rank within the row by lane order, rows in sequence => stable
__global__ void radix_scatter_kernel(const unsigned long long* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
                                     unsigned long long* __restrict__ keys_out, uint32_t* __restrict__ idx_out, uint32_t n,
                                     int shift, const uint32_t* __restrict__ offsets, uint32_t nblk) {
    __shared__ uint32_t base[256];
    const uint32_t lane = threadIdx.x;
    for (uint32_t d = lane; d < 256; d += 32) base[d] = offsets[d * nblk + blockIdx.x];
    __syncwarp();
    const uint32_t first = blockIdx.x * kSortChunk;
    for (uint32_t row = 0; row < kSortChunk / 32; ++row) {
        const uint32_t k = first + row * 32 + lane;
        if (first + row * 32 >= n) break;
        const bool valid = k < n;
        const unsigned long long key = valid ? keys_in[k] : 0ull;
        const uint32_t d = valid ? ((uint32_t)(key >> shift) & 255u) : 256u;
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u)), cnt = __popc(peers);
        uint32_t pos = 0;
        if (valid) {
            pos = base[d] + rank;
            keys_out[pos] = key;
            idx_out[pos] = idx_in[k];
        }
        __syncwarp();
        if (valid && rank == cnt - 1) base[d] += cnt;
        __syncwarp();
    }
}

// The sorted catalog: fp64 rows in Hilbert order, the fp32 copy (that vector rounded once, reading A17), the
// inverse permutation for row-subset mode; rows n..n_pad-1 become the padding point (2,2,2).
__global__ void permute_kernel(const double4* __restrict__ x64_rows, const uint32_t* __restrict__ order, uint64_t n,
                               uint64_t n_pad, double4* __restrict__ x64, float4* __restrict__ x32, uint32_t* __restrict__ inv) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
        if (k < n) {
            const uint32_t src = order[k];
            v = x64_rows[src];
            inv[src] = (uint32_t)k;
        }
        x64[k] = v;
        x32[k] = make_float4((float)v.x, (float)v.y, (float)v.z, 0.f);
    }
}

// Bounding sphere of each kSubJ = 32 consecutive rows (one warp each): centre = fp32 rounding of the mean,
// radius = max fp64 distance of the fp64 rows from that fp32 centre, rounded up with slack.
__global__ void spheres_kernel(const double4* __restrict__ x64, uint64_t nsub, float4* __restrict__ sph) {
    const uint64_t w = (blockIdx.x * (uint64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= nsub) return;
    const double4 v = x64[w * kSubJ + lane];
    double sx = v.x, sy = v.y, sz = v.z;
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, off);
        sy += __shfl_xor_sync(0xffffffffu, sy, off);
        sz += __shfl_xor_sync(0xffffffffu, sz, off);
    }
    const float cx = (float)(sx / kSubJ), cy = (float)(sy / kSubJ), cz = (float)(sz / kSubJ);
    const double dx = v.x - (double)cx, dy = v.y - (double)cy, dz = v.z - (double)cz;
    double r = sqrt(dx * dx + dy * dy + dz * dz);
#pragma unroll
    for (int off = 16; off; off >>= 1) r = fmax(r, __shfl_xor_sync(0xffffffffu, r, off));
    if (lane == 0) sph[w] = make_float4(cx, cy, cz, __double2float_ru(r * (1.0 + 1.0e-7) + 1.0e-9));
}

// row-subset mode: position of each requested row in the sorted catalog (the key the subset is then sorted by,
// so that consecutive i-rows of the temporary catalog are close on the sky as well)
__global__ void row_keys_kernel(const int64_t* __restrict__ rows, uint64_t nrows, uint64_t n_src, const uint32_t* __restrict__ inv,
                                unsigned long long* __restrict__ keys, uint32_t* __restrict__ idx, int* __restrict__ bad) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < nrows; k += (uint64_t)gridDim.x * blockDim.x) {
        const int64_t r = rows[k];
        unsigned long long key = 0;
        if (r < 0 || (uint64_t)r >= n_src) *bad = 1; else key = inv[r];
        keys[k] = key;
        idx[k] = (uint32_t)k;
    }
}

__global__ void gather_kernel(const double4* __restrict__ src64, const float4* __restrict__ src32,
                              const unsigned long long* __restrict__ pos, uint64_t nrows, uint64_t nrows_pad,
                              double4* __restrict__ dst64, float4* __restrict__ dst32) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < nrows_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
        float4 f = make_float4(kPadCoord, kPadCoord, kPadCoord, 0.f);
        if (k < nrows) {
            v = src64[pos[k]];
            f = src32[pos[k]];
        }
        dst64[k] = v;
        dst32[k] = f;
    }
}

__global__ void finalize_kernel(const unsigned long long* __restrict__ result, int nbins, int zero_slot,
                                unsigned long long self_pairs, unsigned long long* __restrict__ out) {
    for (int k = threadIdx.x; k < nbins + 2; k += blockDim.x) out[k] = result[k] - (k == zero_slot ? self_pairs : 0ull);
}

}  // namespace

static int grid_for(uint64_t n, int block) { return (int)std::max<uint64_t>(1, std::min<uint64_t>((n + block - 1) / block, 148ull * 16)); }

cudaError_t launch_convert(const void* radec, int is_f64, uint64_t n, double4* x64_rows, uint64_t* keys, uint32_t* idx,
                           int* bad_flag, cudaStream_t st) {
    const int block = 256, grid = grid_for(n, block);
    auto* k = reinterpret_cast<unsigned long long*>(keys);
    if (is_f64)
        convert_kernel<double><<<grid, block, 0, st>>>(static_cast<const double*>(radec), n, x64_rows, k, idx, bad_flag);
    else
        convert_kernel<float><<<grid, block, 0, st>>>(static_cast<const float*>(radec), n, x64_rows, k, idx, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_sort_pairs(uint64_t* keys_a, uint64_t* keys_b, uint32_t* idx_a, uint32_t* idx_b, uint32_t* counts,
                              uint32_t n, int nbits, cudaStream_t st, bool* in_a) {
    const uint32_t nblk = (n + kSortChunk - 1) / kSortChunk;
    auto* ka = reinterpret_cast<unsigned long long*>(keys_a);
    auto* kb = reinterpret_cast<unsigned long long*>(keys_b);
    bool a = true;
    for (int shift = 0; shift < nbits; shift += 8) {
        radix_hist_kernel<<<nblk, 256, 0, st>>>(a ? ka : kb, n, shift, counts, nblk);
        radix_scan_kernel<<<1, 1024, 0, st>>>(counts, 256u * nblk);
        radix_scatter_kernel<<<nblk, 32, 0, st>>>(a ? ka : kb, a ? idx_a : idx_b, a ? kb : ka, a ? idx_b : idx_a, n, shift,
                                                  counts, nblk);
        a = !a;
    }
    *in_a = a;
    return cudaGetLastError();
}

cudaError_t launch_permute(const double4* x64_rows, const uint32_t* order, uint64_t n, uint64_t n_pad, double4* x64,
                           float4* x32, uint32_t* inv, cudaStream_t st) {
    const int block = 256;
    permute_kernel<<<grid_for(n_pad, block), block, 0, st>>>(x64_rows, order, n, n_pad, x64, x32, inv);
    return cudaGetLastError();
}

cudaError_t launch_spheres(const double4* x64, uint64_t n_pad, float4* sph, cudaStream_t st) {
    const uint64_t nsub = n_pad / kSubJ;
    const int block = 256;
    spheres_kernel<<<(unsigned)((nsub * 32 + block - 1) / block), block, 0, st>>>(x64, nsub, sph);
    return cudaGetLastError();
}

cudaError_t launch_row_keys(const int64_t* rows, uint64_t nrows, uint64_t n_src, const uint32_t* inv, uint64_t* keys,
                            uint32_t* idx, int* bad_flag, cudaStream_t st) {
    const int block = 256;
    row_keys_kernel<<<grid_for(nrows, block), block, 0, st>>>(rows, nrows, n_src, inv, reinterpret_cast<unsigned long long*>(keys),
                                                              idx, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_gather(const double4* src64, const float4* src32, const uint64_t* pos, uint64_t nrows,
                          uint64_t nrows_pad, double4* dst64, float4* dst32, cudaStream_t st) {
    const int block = 256;
    gather_kernel<<<grid_for(nrows_pad, block), block, 0, st>>>(src64, src32, reinterpret_cast<const unsigned long long*>(pos),
                                                                nrows, nrows_pad, dst64, dst32);
    return cudaGetLastError();
}

cudaError_t launch_pairs_fast(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info) {
    const size_t smem = fast_smem_layout(p.ncells, p.nbands, p.nbins).total;
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
