// kernels.cu -- sm_100a kernels of libtpcf.
//
//   convert_kernel      RA/Dec (deg) -> fp64 unit vector + sort key                     (hot-path step a1)
//   radix_* / permute / spheres   spatial sort of the catalog, fp32 copy, subtile bounding spheres (a1)
//   pair_fast_kernel    the all-pairs count: fp32 squared chord; per (lane, 64-row j-subtile) window of
//                       candidate bin edges from bounding spheres -> 1..3 threshold compares per pair with
//                       register counters, else O(1) cell lookup + shared-memory partial histogram;
//                       guard band -> fp64 recheck; uint64 merge                        (steps a3-a7)
//   pair_tensor_kernel  the same count with the window quantity formed by a 3xTF32 tcgen05.mma into tensor memory
//                       (one i-row per thread, tcgen05.ld read-back), everything else shared with pair_fast_kernel
//   pair_exact64_kernel plain fp64 count, the device-side cross-check of the other two
//
// What is computed per pair is PAPER.md:37 ("dot product and arc-cosine ... to extract the angle between
// two objects") followed by PAPER.md:38 (histogram fill with shared-memory atomics, partial histograms
// "later combined in a single histogram, in global memory").  How it is computed differs:
// the angle is never formed; |a-b|^2 = 2 - 2 cos(theta) is compared with per-edge thresholds.
#include "kernels.cuh"
#include <cstdio>
#include <cstdlib>

namespace tpcf {

namespace {

constexpr int R = kIPerThread;
constexpr uint32_t kSqrtMagic = 0x1FBD1DF5u;
constexpr unsigned long long kFlushPairs = 2000000000ull;   // flush the 32-bit partial counters before they can reach 2^31 (those of the lookup path are signed)

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

// ---- packed fp32 pairs (sm_100 f32x2: one instruction, two IEEE round-to-nearest results) --------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// TF32 split of an fp32 value: hi = x rounded to nearest to TF32's 11-bit significand by Veltkamp's splitting,
// c = fl(x (2^13 + 1)), hi = fl(c - fl(c - x)): three FMA-pipe instructions (that pipe idles in the tensor kernel, while the
// integer form of the rounding would load the ALU pipe, its busiest); the low 13 bits of hi are zero, so it is exactly
// representable whatever the tensor core does with those bits; x - hi is exact in fp32 and |x - hi| <= 2^-11 |x|
__device__ __forceinline__ float tf32_hi(float x) {
    const float c = __fmul_rn(x, 8193.0f);
    return __fsub_rn(c, __fsub_rn(c, x));
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

struct SlowCtx {                     // lives in shared memory
    const double4* xi64;
    const double4* xj64;
    const double* thr;
    unsigned* whist;                 // the CTA's partial histogram indexed by result slot (shared memory)
    unsigned nrecheck;               // pairs classified in fp64 since the last flush
    int nbins;
};

// A pair whose fp32 squared chord fell inside the guard band of a bin edge: classify it from the fp64
// coordinates.  Rare (1e-6 .. 1e-3 of the pairs).
__device__ __noinline__ void recheck_pair(SlowCtx* s, uint32_t i, uint32_t j) {
    const double4 a = s->xi64[i], b = s->xj64[j];
    const int slot = exact_slot_dev(chord2_f64(a, b), s->thr, s->nbins);
    atomicAdd(s->whist + slot, 1u);
    atomicAdd(&s->nrecheck, 1u);
}

// Pairs inside a guard band are rare (1e-5 .. 1e-3) and scattered over the lanes: instead of each lane branching off
// to its own recheck, they are queued per warp in shared memory and rechecked 32 at a time, one per lane.
// rq holds kRecheckQueue entries (i, j); qn (warp-uniform, < 32 between calls) is the fill level.
constexpr int kRecheckQueue = 64;
constexpr int kMaxSlowLanes = 8;          // lookup / fp64 lanes a window block may carry (subtile_pairs)
constexpr float kMaxFlagExpect = 0.35f;   // a lane whose window block expects more ambiguous pairs than this takes the cell lookup
__device__ __forceinline__ void rq_push(uint2* rq, unsigned& qn, bool has, uint32_t i, uint32_t j, SlowCtx* slow) {
    const int lane = threadIdx.x & 31;
    const unsigned bal = __ballot_sync(0xffffffffu, has);
    if (!bal) return;
    if (has) rq[qn + __popc(bal & ((1u << lane) - 1u))] = make_uint2(i, j);
    qn += __popc(bal);
    __syncwarp();
    if (qn >= 32) {
        qn -= 32;
        const uint2 e = rq[qn + lane];
        __syncwarp();
        recheck_pair(slow, e.x, e.y);
    }
}
__device__ __forceinline__ void rq_drain(uint2* rq, unsigned& qn, SlowCtx* slow) {
    const int lane = threadIdx.x & 31;
    if (lane < (int)qn) recheck_pair(slow, rq[lane].x, rq[lane].y);
    qn = 0;
    __syncwarp();
}

// ---- cell-lookup path ("lookup" path) ---------------------------------------------------------------------------
// One pair: fp32 squared chord q (difference form) -> cell -> the one threshold T whose guard band reaches into the
// cell (one LDS.32) -> side of T -> shared-memory partial histogram indexed by (side, cell); a pair with |q - T| <= g is
// not counted here but re-evaluated in fp64.  g = alpha Q + beta_r r sqrt(Q) + beta_0 bounds the fp32 error of every pair
// of the (lane, subtile) block: Q bounds its squared chords, r is the sum of its bounding radii.
struct Lookup {
    const char* lut;        // ncells x fp32 threshold (+inf: none; NaN: several, every pair of the cell is ambiguous)
    char* hist;             // 2 x ncells x u32: [0, ncells) pairs below the cell's threshold, [ncells, 2 ncells) at or above it
    uint32_t lut_s;         // lut as a shared-window address
    uint32_t above_off;     // ncells * 4
    int shift;
    float scale, clamp;
    float alpha, beta_r, beta0;
    int multi;              // some cell holds a NaN: the lazy detection of ambiguous pairs (a minimum) cannot be used
};

__device__ __forceinline__ Lookup make_lookup(const PairParams& p, unsigned char* lut, unsigned char* hist) {
    Lookup lk;
    lk.lut = reinterpret_cast<const char*>(lut);
    lk.hist = reinterpret_cast<char*>(hist);
    lk.lut_s = smem_u32(lut);
    lk.above_off = (uint32_t)p.ncells * 4u;
    lk.shift = p.shift;
    lk.scale = p.sqrt_scale;
    lk.clamp = p.sqrt_clamp;
    lk.alpha = kLookupAlpha * p.guard_scale;
    lk.beta_r = kLookupBetaR * p.guard_scale;
    lk.beta0 = kLookupBeta0 * p.guard_scale;
    lk.multi = p.lut_multi;
    return lk;
}

// byte offset 4 * cell of the lookup cell of q; exactly FastTables::cell_of (tables.cpp)
template <int MAP, bool CLAMP>
__device__ __forceinline__ uint32_t cell_off4(float q, const Lookup& lk) {
    if (MAP == (int)CellMap::LogBits) {
        return (__float_as_uint(q) >> (lk.shift - 2)) & ~3u;
    } else {
        const float c = CLAMP ? fminf(q, lk.clamp) : q;
        const float key = __uint_as_float((__float_as_uint(c) >> 1) + kSqrtMagic);
        const float t = fmaf(key, lk.scale, 8388608.0f);
        return __float_as_uint(t) & 0x7FFFFCu;
    }
}

__device__ __forceinline__ float lookup_guard(const Lookup& lk, float rs, float hi) {
    const float hi2 = __fmul_ru(hi, hi);
    return fmaf(lk.alpha, hi2, fmaf(lk.beta_r * rs, hi * 1.0001f, lk.beta0));
}

// s - b' and its square, two i-rows at a time; b holds (-2 b', .) broadcast to both halves.  Only explicitly rounded
// operations: the rescan of a j-row (lookup_rescan) must reproduce these values bit for bit.
__device__ __forceinline__ f32x2 chord2_diff2(f32x2 sx, f32x2 sy, f32x2 sz, f32x2 bx, f32x2 by, f32x2 bz) {
    const f32x2 half2 = pack2(0.5f, 0.5f);
    const f32x2 dx = fma2(bx, half2, sx), dy = fma2(by, half2, sy), dz = fma2(bz, half2, sz);
    return fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
}

// generic form, one pair at a time (diagonal chunks, recounts of flagged lanes and rows, tables with NaN cells).
// Returns true when the pair is valid and ambiguous (the caller then rechecks it in fp64); every other valid pair is
// counted here.
template <int MAP>
__device__ __forceinline__ bool lookup_pair(float sx, float sy, float sz, const float4& b, const Lookup& lk, float g, bool valid) {
    const float dx = fmaf(b.x, 0.5f, sx), dy = fmaf(b.y, 0.5f, sy), dz = fmaf(b.z, 0.5f, sz);     // s - b', one rounding each
    const float q = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const uint32_t off = cell_off4<MAP, true>(q, lk);
    const float e = __fsub_rn(q, *reinterpret_cast<const float*>(lk.lut + off));
    const bool amb = !(fabsf(e) > g);
    if (valid && !amb) atomicAdd(reinterpret_cast<unsigned*>(lk.hist + off + (e < 0.f ? 0u : lk.above_off)), 1u);
    return valid && amb;
}

// fast form: count the pair on the side of T its fp32 value shows (one shared atomic, no branch); returns |q - T|.
// A pair with |q - T| <= g is taken out again by lookup_rescan, which sees the same bits.
__device__ __forceinline__ float lds_f32(uint32_t addr) {
    float v;
    asm("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
template <int MAP, bool CLAMP>
__device__ __forceinline__ float lookup_count(float q, const Lookup& lk) {
    const uint32_t off = cell_off4<MAP, CLAMP>(q, lk);
    const float e = __fsub_rn(q, lds_f32(lk.lut_s + off));
    atomicAdd(reinterpret_cast<unsigned*>(lk.hist + off + (e < 0.f ? 0u : lk.above_off)), 1u);
    return fabsf(e);
}

// One subtile against this lane's R rows, every pair by cell lookup, generic form.  MASK: only pairs j > i (diagonal
// chunk).  Called by the whole warp; lanes with active == false count nothing.
template <int MAP, bool MASK>
__device__ __forceinline__ void lookup_block(const float4* __restrict__ js, const float (&sx)[R], const float (&sy)[R],
                                             const float (&sz)[R], bool active, const Lookup& lk, float g, SlowCtx* slow,
                                             uint2* rq, unsigned& qn, uint32_t i0, uint32_t j0) {
#pragma unroll 1
    for (int jj = 0; jj < kSubJ; ++jj) {
        const float4 b = js[jj];                                  // one LDS.128, broadcast to the warp
        unsigned amb = 0;
#pragma unroll
        for (int r = 0; r < R; ++r)
            amb |= (lookup_pair<MAP>(sx[r], sy[r], sz[r], b, lk, g, active && (!MASK || (j0 + jj > i0 + r))) ? 1u : 0u) << r;
        while (__any_sync(0xffffffffu, amb != 0)) {               // rare: pairs inside a guard band
            const int r = __ffs(amb) - 1;
            rq_push(rq, qn, amb != 0, i0 + r, j0 + jj, slow);
            amb &= amb - 1;
        }
    }
}

// The ambiguous pairs (|q - T| <= g) of one j-row, which lookup_block_fast counted like every other pair: found again
// (same operations, same bits), taken out of the partial histogram and queued for the fp64 recheck.  The partial
// counters of the lookup path are therefore signed 32-bit values (flush_slots), and a counter may be read as -1 for a
// moment when a flush falls between the two atomics.
template <int MAP, bool CLAMP>
__device__ __forceinline__ void lookup_rescan(const float4 b, float m, const f32x2 (&sx2)[R / 2], const f32x2 (&sy2)[R / 2],
                                              const f32x2 (&sz2)[R / 2], const Lookup& lk, float g, SlowCtx* slow, uint2* rq, unsigned& qn,
                                              uint32_t i0, uint32_t j) {
    unsigned amb = 0;
    if (m <= g) {                                   // only the lanes that saw one walk their R pairs again
        const f32x2 bx = pack2(b.x, b.x), by = pack2(b.y, b.y), bz = pack2(b.z, b.z);
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            float q[2];
            unpack2(chord2_diff2(sx2[r], sy2[r], sz2[r], bx, by, bz), q[0], q[1]);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint32_t off = cell_off4<MAP, CLAMP>(q[h], lk);
                const float e = __fsub_rn(q[h], lds_f32(lk.lut_s + off));
                if (fabsf(e) <= g) {
                    atomicSub(reinterpret_cast<unsigned*>(lk.hist + off + (e < 0.f ? 0u : lk.above_off)), 1u);
                    amb |= 1u << (2 * r + h);
                }
            }
        }
    }
    __syncwarp();
    while (__any_sync(0xffffffffu, amb != 0)) {
        const int r = __ffs(amb) - 1;
        rq_push(rq, qn, amb != 0, i0 + r, j, slow);
        amb &= amb - 1;
    }
}

// One subtile against this lane's R rows, every pair by cell lookup, fast form (every lane active, no mask, no NaN
// cells): per pair 3 packed FMA-pipe instructions for two squared chords, the cell offset, one LDS.32, one subtraction,
// the side select and one shared atomic; ambiguous pairs are detected per j-row from the smallest |q - T|.
template <int MAP, bool CLAMP>
__device__ __forceinline__ void lookup_block_fast(const float4* __restrict__ js, const f32x2 (&sx2)[R / 2], const f32x2 (&sy2)[R / 2],
                                                  const f32x2 (&sz2)[R / 2], const Lookup& lk, float g, SlowCtx* slow, uint2* rq,
                                                  unsigned& qn, uint32_t i0, uint32_t j0) {
#pragma unroll 2
    for (int jj = 0; jj < kSubJ; ++jj) {
        const float4 b = js[jj];
        const f32x2 bx = pack2(b.x, b.x), by = pack2(b.y, b.y), bz = pack2(b.z, b.z);
        float m = 3.0e38f;
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            float q0, q1;
            unpack2(chord2_diff2(sx2[r], sy2[r], sz2[r], bx, by, bz), q0, q1);
            m = fminf(m, fminf(lookup_count<MAP, CLAMP>(q0, lk), lookup_count<MAP, CLAMP>(q1, lk)));
        }
        if (__any_sync(0xffffffffu, m <= g)) lookup_rescan<MAP, CLAMP>(b, m, sx2, sy2, sz2, lk, g, slow, rq, qn, i0, j0 + jj);
    }
}

// Blocks whose bounding radii are too large for the fp32 error bound (sparse or tiny catalogs, quads or subtiles that
// straddle a jump of the sort curve or contain padding rows): every real pair is classified from the fp64
// coordinates.  The warp works together on the lanes in `todo`, one after the other: lane l takes j-row j0 + l.
__device__ __noinline__ void exact_lanes(SlowCtx* s, unsigned todo, uint32_t ibase, uint32_t n_i, uint32_t j0, uint32_t n_j,
                                         bool mask) {
    const int lane = threadIdx.x & 31;
    unsigned cnt = 0;
#pragma unroll 1
    for (int h = 0; h < kSubJ / 32; ++h) {
        const uint32_t j = j0 + h * 32 + lane;
        const double4 b = s->xj64[j];               // rows up to the padded size exist
        unsigned rest = todo;
        while (rest) {
            const int src = __ffs(rest) - 1;
            rest &= rest - 1;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const uint32_t i = ibase + src * R + r;
                if (i >= n_i) break;                // uniform across the warp
                const int slot = exact_slot_dev(chord2_f64(s->xi64[i], b), s->thr, s->nbins);
                if (j < n_j && (!mask || j > i)) {
                    atomicAdd(s->whist + slot, 1u);
                    ++cnt;
                }
            }
        }
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0 && cnt) atomicAdd(&s->nrecheck, cnt);
}

// ---- window path ----------------------------------------------------------------------------------------------
// The E-edge window loop over one subtile.  q = |s|^2 - mid_0 + |b'|^2 - 2 s.b' (4 FMA-pipe instructions); for each
// of the bands k .. k+E-1 the sign bit of q + (mid_0 - mid_e) is accumulated (one LEA.HI) and the smallest
// |q - ...| is tracked (FMNMX3, two values per instruction).  Returns true when some pair came within a band's half
// width: this lane's counters are then not used and its pairs are recounted one by one.
template <int E>
__device__ __forceinline__ bool window_block(const float4* __restrict__ js, const f32x2 (&sx2)[R / 2], const f32x2 (&sy2)[R / 2],
                                             const f32x2 (&sz2)[R / 2], const f32x2 (&nsm2)[R / 2] /* |s|^2 - mid_0 */,
                                             const float (&dt)[kMaxWinEdges], float hmax, unsigned (&c)[kMaxWinEdges]) {
    // two i-rows per f32x2 register; the j-row is broadcast to both halves
    f32x2 dt2[kMaxWinEdges];
#pragma unroll
    for (int e = 0; e < kMaxWinEdges; ++e) {
        c[e] = 0;
        dt2[e] = pack2(dt[e], dt[e]);
    }
    float m = 3.0e38f;
#pragma unroll 4
    for (int jj = 0; jj < kSubJ; ++jj) {
        const float4 b = js[jj];
        const f32x2 bx = pack2(b.x, b.x), by = pack2(b.y, b.y), bz = pack2(b.z, b.z), bw = pack2(b.w, b.w);
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            const f32x2 q = fma2(sx2[r], bx, fma2(sy2[r], by, fma2(sz2[r], bz, add2(nsm2[r], bw))));
#pragma unroll
            for (int e = 0; e < E; ++e) {
                float q0, q1;
                unpack2(e ? add2(q, dt2[e]) : q, q0, q1);
                c[e] += __float_as_uint(q0) >> 31;
                c[e] += __float_as_uint(q1) >> 31;
                m = fminf(m, fminf(fabsf(q0), fabsf(q1)));
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

// One subtile (kSubJ rows at js, bounding sphere sp) against this lane's quad (offsets p*, centre cq*, radius ri).
// Every lane chooses the cheapest loop that is valid for its block; the warp runs the most general of them.
//   1..3  window loop with that many edges      4  cell lookup      5  fp64
template <int MAP>
__device__ __forceinline__ void subtile_pairs(const float4* __restrict__ js, const float4 sp, bool windows, bool prune, bool mask,
                                              const f32x2 (&px2)[R / 2], const f32x2 (&py2)[R / 2], const f32x2 (&pz2)[R / 2], float cqx,
                                              float cqy, float cqz, float ri, const WinTables& wt, const Lookup& lk,
                                              SlowCtx* slow, uint2* rq, unsigned& qn, uint32_t i0, uint32_t n_i,
                                              uint32_t j0, uint32_t n_j, unsigned (&npath)[7]) {
    const int lane = threadIdx.x & 31;
    // bounds on every TRUE chord of the block from the triangle inequality: |cq - cs| -/+ (ri + rj), made safe
    // against the fp32 evaluation (relative 4e-6 on the centre distance, 1e-7 absolute)
    const float tx = __fsub_rn(cqx, sp.x), ty = __fsub_rn(cqy, sp.y), tz = __fsub_rn(cqz, sp.z);
    const float dc2 = fmaf(tz, tz, fmaf(ty, ty, tx * tx));
    float dc;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(dc) : "f"(dc2));
    const float rs = ri + sp.w;
    const float lo = fmaf(dc, 1.0f - 4.0e-6f, -rs) - 1.0e-7f;
    const float hi = fmaf(dc, 1.0f + 4.0e-6f, rs) + 1.0e-7f;
    const float g = lookup_guard(lk, rs, hi);       // guard of the cell-lookup path for this block
    int mode = 4, k = 0;
    if (rs > kRCap) {
        mode = 5;
    } else if (windows && !mask && lo >= kFarKappa * rs) {
        const float lo2 = __fmul_rd(lo, lo), hi2 = __fmul_ru(hi, hi);
        // first band that is not wholly below the window, then how many bands the window reaches
        k = wt.cell_band[cell_off4<MAP, true>(lo2, lk) >> 2];
        while (k < wt.nbands && wt.band_lh[k].y <= lo2) ++k;
        int e = 1;
        while (e <= kMaxWinEdges && k + e < wt.nbands && wt.band_lh[k + e].x <= hi2) ++e;
        mode = e;
        // fine binnings: when the bands fill so much of the window that one of the block's kSubJ x R pairs is likely to
        // fall inside one (chords spread evenly over the window), the window loop would only be followed by a recount
        if (k < wt.nbands && (float)(2 * kSubJ * R) * (float)e * wt.band_mh[k].y > kMaxFlagExpect * (hi2 - lo2)) mode = 4;
    }
    // Pruning mode (tpcf_set_pruning: the dual-tree idea of PAPER.md:29 at block granularity; NOT the
    // brute-force count): when no lane's window reaches a band, every pair of a lane's block lies in one result slot and
    // the kSubJ x R pairs are added wholesale, unevaluated.
    if (prune) {
        const bool empty = mode == 1 && (k >= wt.nbands || wt.band_lh[k].x > __fmul_ru(hi, hi));
        if (__all_sync(0xffffffffu, empty)) {
            atomicAdd(wt.whist + wt.band_slot[min(k, wt.nbands)], (unsigned)(kSubJ * R));
            ++npath[6];
            return;
        }
    }
    // A few lanes that need the cell lookup (or fp64) do not drag the whole warp into lookup_block: the warp runs the
    // window loop of the other lanes, those lanes' counters are dropped and their pairs are recounted by the whole
    // warp together (lookup lanes: the recount of flagged lanes below; fp64 lanes: exact_lanes).
    const unsigned slow_lanes = __ballot_sync(0xffffffffu, mode > kMaxWinEdges);
    const bool hybrid = slow_lanes != 0 && !mask && __popc(slow_lanes) <= kMaxSlowLanes;
    const int wmode = __reduce_max_sync(0xffffffffu, (hybrid && mode > kMaxWinEdges) ? 1 : mode);

    f32x2 sx2[R / 2], sy2[R / 2], sz2[R / 2];
    float sx[R], sy[R], sz[R];                      // the same registers, one row at a time
    {
        const f32x2 tx2 = pack2(tx, tx), ty2 = pack2(ty, ty), tz2 = pack2(tz, tz);
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            sx2[r] = add2(px2[r], tx2);
            sy2[r] = add2(py2[r], ty2);
            sz2[r] = add2(pz2[r], tz2);
            unpack2(sx2[r], sx[2 * r], sx[2 * r + 1]);
            unpack2(sy2[r], sy[2 * r], sy[2 * r + 1]);
            unpack2(sz2[r], sz[2 * r], sz[2 * r + 1]);
        }
    }
    if (wmode > kMaxWinEdges) {
        // lanes with mode 5 are counted below, by the whole warp, in fp64; a quad wholly past the end of the catalog and a
        // subtile of padding rows only (lo > 2.2: no chord between unit vectors exceeds 2) hold no pair at all
        const bool act = mode != 5 && i0 < n_i && lo <= 2.2f;
        if (!act) {
            const f32x2 z2 = pack2(0.f, 0.f);
#pragma unroll
            for (int r = 0; r < R / 2; ++r) sx2[r] = sy2[r] = sz2[r] = z2;      // keeps their (unused) cells inside the table
#pragma unroll
            for (int r = 0; r < R; ++r) sx[r] = sy[r] = sz[r] = 0.f;
        }
        if (mask) {
            lookup_block<MAP, true>(js, sx, sy, sz, act, lk, g, slow, rq, qn, i0, j0);
        } else if (lk.multi || !__all_sync(0xffffffffu, act)) {
            lookup_block<MAP, false>(js, sx, sy, sz, act, lk, g, slow, rq, qn, i0, j0);
        } else if (MAP == (int)CellMap::SqrtLin && __any_sync(0xffffffffu, __fadd_ru(__fmul_ru(hi, hi), g) > lk.clamp)) {      // hi bounds the TRUE chords; the fp32 q may exceed them by g
            lookup_block_fast<MAP, true>(js, sx2, sy2, sz2, lk, g, slow, rq, qn, i0, j0);
        } else {
            lookup_block_fast<MAP, false>(js, sx2, sy2, sz2, lk, g, slow, rq, qn, i0, j0);
        }
        if (wmode == 5) exact_lanes(slow, __ballot_sync(0xffffffffu, mode == 5), i0 - lane * R, n_i, j0, n_j, mask);
        ++npath[wmode == 5 ? 5 : 3];
        return;
    }
    // every lane runs the wmode-edge loop on bands k .. k+wmode-1; lowering k keeps the lane's window inside them
    k = min(k, wt.nbands - wmode);
    const float2 mh0 = wt.band_mh[k];
    float hmax = mh0.y, dt[kMaxWinEdges];
    dt[0] = 0.f;
#pragma unroll
    for (int e = 1; e < kMaxWinEdges; ++e) {
        dt[e] = 0.f;
        if (e < wmode) {
            const float2 mh = wt.band_mh[k + e];
            dt[e] = __fsub_rn(mh0.x, mh.x);
            hmax = fmaxf(hmax, mh.y);
        }
    }
    f32x2 nsm2[R / 2];
    {
        const f32x2 nmid = pack2(-mh0.x, -mh0.x);
#pragma unroll
        for (int r = 0; r < R / 2; ++r) nsm2[r] = add2(fma2(sz2[r], sz2[r], fma2(sy2[r], sy2[r], mul2(sx2[r], sx2[r]))), nmid);
    }
    unsigned c[kMaxWinEdges], cnt[kMaxWinEdges + 1];
    bool flagged;
    if (wmode == 1) {
        flagged = window_block<1>(js, sx2, sy2, sz2, nsm2, dt, hmax, c);
        cnt[0] = c[0];
        cnt[1] = kSubJ * R - c[0];
        cnt[2] = cnt[3] = 0;
        ++npath[0];
    } else if (wmode == 2) {
        flagged = window_block<2>(js, sx2, sy2, sz2, nsm2, dt, hmax, c);
        cnt[0] = c[0];
        cnt[1] = c[1] - c[0];
        cnt[2] = kSubJ * R - c[1];
        cnt[3] = 0;
        ++npath[1];
    } else {
        flagged = window_block<3>(js, sx2, sy2, sz2, nsm2, dt, hmax, c);
        cnt[0] = c[0];
        cnt[1] = c[1] - c[0];
        cnt[2] = c[2] - c[1];
        cnt[3] = kSubJ * R - c[2];
        ++npath[2];
    }
    if (!flagged && mode <= kMaxWinEdges) {
#pragma unroll
        for (int t = 0; t <= kMaxWinEdges; ++t)
            if (cnt[t]) atomicAdd(wt.whist + wt.band_slot[k + t], cnt[t]);      // cnt[t] != 0 only for t <= wmode
    }
    flagged = (flagged && mode <= kMaxWinEdges) || mode == 4;
    // lanes that saw a pair inside a guard band: the warp recounts their kSubJ x R pairs together, lane l taking
    // j-point l, through the cell-lookup path (which sends the ambiguous pairs to the fp64 recheck)
    unsigned todo = __ballot_sync(0xffffffffu, flagged);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t isrc = i0 + (uint32_t)(src - lane) * R;
        const float gsrc = __shfl_sync(0xffffffffu, g, src);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float ux = __shfl_sync(0xffffffffu, sx[r], src), uy = __shfl_sync(0xffffffffu, sy[r], src),
                        uz = __shfl_sync(0xffffffffu, sz[r], src);
#pragma unroll
            for (int h = 0; h < kSubJ / 32; ++h)
                rq_push(rq, qn, lookup_pair<MAP>(ux, uy, uz, js[h * 32 + lane], lk, gsrc, true), isrc + r, j0 + h * 32 + lane, slow);
        }
        ++npath[4];
    }
    if (hybrid) {
        const unsigned ex = __ballot_sync(0xffffffffu, mode == 5);
        if (ex) {
            exact_lanes(slow, ex, i0 - lane * R, n_i, j0, n_j, false);
            ++npath[5];
        }
    }
}

constexpr int NRING = 2;                                               // chunk slots per warp
constexpr int kSubPerChunk = kChunkJ / kSubJ;
constexpr uint32_t kChunkBytes = kChunkJ * sizeof(float4), kChunkSphBytes = kSubPerChunk * sizeof(float4);
constexpr uint32_t kSlotBytes = kChunkBytes + kChunkSphBytes;
static_assert(kSubJ % 32 == 0, "the recount of a flagged lane gives j-points l, l + 32, .. of the subtile to lane l");
static_assert(kIPerThread % 2 == 0, "window_block packs two i-rows per f32x2 register");
static_assert(kWarpI % kChunkJ == 0, "the diagonal chunks of a warp item are the chunks with the warp's own rows");
static_assert(kTileJ % kChunkJ == 0 && kTileI % kWarpI == 0 && kTileI / kWarpI == kWarpsPerCta, "tiling");

// shared-memory layout of pair_fast_kernel (byte offsets; every array 16-byte aligned)
__host__ __device__ inline uint32_t up16(uint32_t x) { return (x + 15u) & ~15u; }
struct FastSmem {
    uint32_t ring, lut, hist, band_mh, band_lh, thr, whist, cell_band, band_slot, bars, slow, rq, total;
};
__host__ __device__ inline FastSmem fast_smem_layout(int ncells, int nbands, int nbins) {
    FastSmem L;
    uint32_t o = 0;
    L.ring = o;       o += kWarpsPerCta * NRING * kSlotBytes;
    L.lut = o;        o = up16(o + (uint32_t)ncells * 4);
    L.hist = o;       o = up16(o + (uint32_t)ncells * 8);
    L.band_mh = o;    o = up16(o + (uint32_t)nbands * 8);
    L.band_lh = o;    o = up16(o + (uint32_t)nbands * 8);
    L.thr = o;        o = up16(o + (uint32_t)(nbins + 1) * 8);
    L.whist = o;      o = up16(o + (uint32_t)(nbins + 3) * 4);
    L.cell_band = o;  o = up16(o + (uint32_t)ncells * 2);
    L.band_slot = o;  o = up16(o + (uint32_t)(nbands + 1) * 2);
    L.bars = o;       o = up16(o + kWarpsPerCta * NRING * 8);
    L.slow = o;       o = up16(o + (uint32_t)sizeof(SlowCtx));
    L.rq = o;         o += kWarpsPerCta * kRecheckQueue * 8;
    L.total = o;
    return L;
}

// i-block of work item w of the triangle plan: the warp probes 32 positions of row_start per round
__device__ __forceinline__ uint32_t tri_row_of(const uint32_t* __restrict__ row_start, uint32_t blocks_i, uint32_t w, int lane) {
    uint32_t lo = 0, hi = blocks_i;                      // row_start[lo] <= w < row_start[hi]
    while (hi - lo > 1) {
        const uint32_t step = (hi - lo + 32) / 33, pos = lo + (lane + 1) * step;
        const bool ok = pos < hi && row_start[pos] <= w;
        const uint32_t cnt = __popc(__ballot_sync(0xffffffffu, ok));      // probes are monotone: the first cnt hold
        hi = min(hi, lo + (cnt + 1) * step);
        lo = lo + cnt * step;
    }
    return lo;
}

// Add partial counters into the global uint64 result and clear them.  Integer adds: order-independent, hence
// deterministic.  atomicExch lets one warp do this while the others keep counting.
__device__ __forceinline__ void flush_slots(unsigned* hist, int nslots, const uint16_t* __restrict__ slotmap, unsigned* whist,
                                            int nres, unsigned long long* result, unsigned* nrecheck,
                                            unsigned long long* rechecked, int first, int stride) {
    for (int s = first; s < nslots; s += stride) {       // signed: lookup_rescan takes ambiguous pairs out again
        const int v = hist[s] ? (int)atomicExch(hist + s, 0u) : 0;
        if (v) atomicAdd(result + slotmap[s], (unsigned long long)(long long)v);
    }
    for (int s = first; s < nres; s += stride) {
        const unsigned v = whist[s] ? atomicExch(whist + s, 0u) : 0u;
        if (v) atomicAdd(result + s, (unsigned long long)v);
    }
    if (first == 0) {
        const unsigned v = *nrecheck ? atomicExch(nrecheck, 0u) : 0u;
        if (v) atomicAdd(rechecked, (unsigned long long)v);
    }
}

// The pair kernel.  Persistent CTAs of 8 independent warps.  A warp item = kWarpI = 256 consecutive i-rows (one 8-row group per lane)
// against the j-rows of one plan item; the warp streams those j-rows through its own 2-slot shared-memory ring in
// 128-row chunks (TMA bulk copies behind mbarriers, issued by lane 0), so no CTA-wide barrier sits in the loop.
// MINB = resident CTAs per SM the register budget is cut for: 2 (128 registers: the window loops need them) or, for launches
// whose blocks almost all take the per-pair cell lookup (fine binnings), 3 (80 registers, the window loops spill, the lookup
// loop gets 24 warps per SM to hide its LDS -> ATOMS chains: config 5 -4 %).
template <int MAP, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) pair_fast_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const FastSmem L = fast_smem_layout(p.ncells, p.nbands, p.nbins);
    unsigned* hist = reinterpret_cast<unsigned*>(smem + L.hist);
    const Lookup lk = make_lookup(p, smem + L.lut, smem + L.hist);
    SlowCtx* slow = reinterpret_cast<SlowCtx*>(smem + L.slow);
    WinTables wt;
    wt.band_mh = reinterpret_cast<const float2*>(smem + L.band_mh);
    wt.band_lh = reinterpret_cast<const float2*>(smem + L.band_lh);
    wt.band_slot = reinterpret_cast<const uint16_t*>(smem + L.band_slot);
    wt.cell_band = reinterpret_cast<const uint16_t*>(smem + L.cell_band);
    wt.whist = reinterpret_cast<unsigned*>(smem + L.whist);
    wt.nbands = p.nbands;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned char* ring = smem + L.ring + (size_t)warp * NRING * kSlotBytes;
    const uint32_t bar0 = smem_u32(smem + L.bars + (size_t)warp * NRING * 8);
    for (int c = tid; c < p.ncells; c += kThreads) {
        reinterpret_cast<float*>(smem + L.lut)[c] = p.lut[c];
        hist[c] = 0;
        hist[p.ncells + c] = 0;
        reinterpret_cast<uint16_t*>(smem + L.cell_band)[c] = p.cell_band[c];
    }
    for (int b = tid; b < p.nbands; b += kThreads) {
        reinterpret_cast<float2*>(smem + L.band_mh)[b] = p.band_mh[b];
        reinterpret_cast<float2*>(smem + L.band_lh)[b] = p.band_lh[b];
    }
    for (int b = tid; b <= p.nbands; b += kThreads) reinterpret_cast<uint16_t*>(smem + L.band_slot)[b] = p.band_slot[b];
    for (int b = tid; b < p.nbins + 3; b += kThreads) wt.whist[b] = 0;
    for (int b = tid; b <= p.nbins; b += kThreads) reinterpret_cast<double*>(smem + L.thr)[b] = p.thr[b];
    if (lane == 0) {
        for (int b = 0; b < NRING; ++b) mbar_init(bar0 + 8 * b, 1);
        fence_barrier_init();
    }
    if (tid == 0) {
        slow->xi64 = p.xi64;
        slow->xj64 = p.xj64;
        slow->thr = reinterpret_cast<const double*>(smem + L.thr);
        slow->whist = wt.whist;
        slow->nrecheck = 0;
        slow->nbins = p.nbins;
    }
    __syncthreads();

    auto fetch_chunk = [&](uint32_t g, uint32_t ch) {      // lane 0: two bulk copies behind the slot's mbarrier
        const uint32_t slot = g % NRING, bar = bar0 + 8 * slot;
        unsigned char* dst = ring + (size_t)slot * kSlotBytes;
        fence_proxy_async();
        mbar_expect_tx(bar, kSlotBytes);
        bulk_g2s(smem_u32(dst), p.xs + (size_t)ch * kChunkJ, kChunkBytes, bar);
        bulk_g2s(smem_u32(dst + kChunkBytes), p.cs + (size_t)ch * kSubPerChunk, kChunkSphBytes, bar);
    };

    const uint32_t per_item = kWarpsPerCta * p.jsplit;      // warp items per plan item
    const unsigned long long n_witems = (unsigned long long)p.n_items_part * per_item;
    const uint32_t per_row = (p.tiles_j + p.chunk - 1) / p.chunk;
    uint2* rq = reinterpret_cast<uint2*>(smem + L.rq) + (size_t)warp * kRecheckQueue;
    unsigned qn = 0;                        // fill level of this warp's recheck queue
    uint32_t g = 0;                         // chunks this warp consumed so far: selects ring slot and mbarrier parity
    unsigned long long pairs_since_flush = 0, witems_done = 0;
    unsigned npath[7] = {0, 0, 0, 0, 0, 0, 0};
    for (;;) {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(p.counters, 1ull);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= n_witems) break;
        const uint32_t w = (uint32_t)(c / per_item) * p.nparts + p.part, ws = (uint32_t)(c % per_item) / p.jsplit,
                       js = (uint32_t)(c % p.jsplit);
        uint32_t I, tile0;
        if (p.tri) {
            I = tri_row_of(p.row_start, p.blocks_i, w, lane);
            tile0 = I + (w - p.row_start[I]) * p.chunk;
        } else {
            I = w / per_row;
            tile0 = (w % per_row) * p.chunk;
        }
        const uint32_t ntiles = min(p.chunk, p.tiles_j - tile0);

        // this lane's quad: R consecutive rows as offsets from the quad centre.  A quad wholly past the end of the
        // catalog is moved to (-2,-2,-2): 6 <= d2 <= 48 against every real or padding j-row, i.e. always discarded.
        const uint32_t ibase = I * kTileI + ws * kWarpI, i0 = ibase + lane * R;
        float4 q4 = p.cq[i0 / R];
        f32x2 px2[R / 2], py2[R / 2], pz2[R / 2];
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            float4 a0 = p.xq[i0 + 2 * r], a1 = p.xq[i0 + 2 * r + 1];
            if (i0 >= p.n_i) a0 = a1 = make_float4(0.f, 0.f, 0.f, 0.f);
            px2[r] = pack2(a0.x, a1.x);
            py2[r] = pack2(a0.y, a1.y);
            pz2[r] = pack2(a0.z, a1.z);
        }
        if (i0 >= p.n_i) q4 = make_float4(-kPadCoord, -kPadCoord, -kPadCoord, 0.f);

        // chunks of kChunkJ rows; in the triangle those wholly below the warp's own rows hold no pair i<j, and the
        // chunks of the warp's own rows are the diagonal ones (masked)
        const uint32_t dch = ibase / kChunkJ, dch_end = (ibase + kWarpI) / kChunkJ;
        uint32_t ch = tile0 * (kTileJ / kChunkJ);
        uint32_t ch_end = (tile0 + ntiles) * (kTileJ / kChunkJ);
        if (p.jsplit > 1) {                                  // chunk == 1: part js of the single tile
            ch += js * ((kTileJ / kChunkJ) / p.jsplit);
            ch_end = ch + (kTileJ / kChunkJ) / p.jsplit;
        }
        if (p.tri) ch = max(ch, dch);
        if (lane == 0 && ch < ch_end) fetch_chunk(g, ch);
        for (; ch < ch_end; ++ch, ++g) {
            if (lane == 0 && ch + 1 < ch_end) fetch_chunk(g + 1, ch + 1);       // the other slot: released by the __syncwarp below
            mbar_wait(bar0 + 8 * (g % NRING), (g / NRING) & 1);
            const float4* jt = reinterpret_cast<const float4*>(ring + (size_t)(g % NRING) * kSlotBytes);
            const float4* jsph = jt + kChunkJ;
            const bool mask = p.tri && ch < dch_end;        // a chunk of the warp's own rows: pairs j > i only
#pragma unroll 1
            for (int sub = 0; sub < kSubPerChunk; ++sub)
                subtile_pairs<MAP>(jt + sub * kSubJ, jsph[sub], p.window != 0, p.prune != 0, mask, px2, py2, pz2, q4.x, q4.y, q4.z, q4.w, wt, lk,
                                   slow, rq, qn, i0, p.n_i, ch * kChunkJ + sub * kSubJ, p.n_j, npath);
            __syncwarp();
            pairs_since_flush += (unsigned long long)kWarpI * kChunkJ;
        }
        if (js == 0) ++witems_done;
        if (pairs_since_flush > kFlushPairs / kWarpsPerCta) {     // 8 warps x this bound < 2^32 per slot
            flush_slots(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result, &slow->nrecheck, p.counters + 1, lane, 32);
            pairs_since_flush = 0;
        }
    }
    rq_drain(rq, qn, slow);
    __syncthreads();
    flush_slots(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result, &slow->nrecheck, p.counters + 1, tid, kThreads);
    if (lane == 0) {
        if (witems_done) atomicAdd(p.counters + 2, witems_done);
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (npath[k]) atomicAdd(p.counters + 3 + k, (unsigned long long)npath[k]);
    }
}

// ---- tensor engine (TPCF_ENGINE_TENSOR) ---------------------------------------------------------------------
// The window quantity q = |s|^2 - mid_0 + |b'|^2 - 2 s.b' of a (128 i-rows) x (128 j-rows) block is one
// 128 x 128 x 16 tcgen05.mma (kind::tf32, two K = 8 steps) whose operands carry the fp32 values split into TF32 parts
// (3xTF32: s_hi m_hi + s_hi m_lo + s_lo m_hi, the two norms as three parts each against columns of ones); the fp32
// accumulators live in tensor memory, one TMEM lane = one i-row = one thread, and come back with tcgen05.ld for the
// same bin decision as the FFMA2 loop (sign count per edge + min |q| against the band half width).  A CTA is 4 warps
// = one 128-row MMA tile; the j side comes in tiles of kTcSubJ = 128 rows (own spheres and offsets: PairParams xt, ct, xb).
// Windows are per (8-row quad, j-tile) as in pair_fast_kernel; rows whose block needs the cell lookup, the diagonal mask or
// fp64 are counted by their warp together, lane l taking j-rows l, l + 32, ..
constexpr int kTcThreads = 128;
constexpr int kTcRing = 3;                                                      // chunk slots per CTA
constexpr uint32_t kTcABytes = kTcThreads * kTcK * 4, kTcBBytes = kTcSubJ * kTcK * 4, kTcRowBytes = kTcSubJ * sizeof(float4);
constexpr uint32_t kTcALbo = kTcThreads * 16, kTcBLbo = kTcSubJ * 16, kTcSbo = 128;
constexpr uint32_t kTcSlotBytes = kTcBBytes + kTcRowBytes + sizeof(float4);     // operand tile, fp32 rows, sphere
constexpr uint32_t kTcCols = kTcSubJ;                                           // one 128 x 128 fp32 accumulator tile
constexpr uint32_t kTcIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kTcSubJ >> 3) << 17) | ((uint32_t)(kTcThreads >> 4) << 24);
static_assert(kTcSubJ == kTcThreads && kTcSubJ == kChunkJ, "the diagonal tile of a tensor-engine CTA is the tile of its own 128 rows");
static_assert(kTcSubJ % 64 == 0, "the accumulators are read back 64 columns at a time");

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}
#define TPCF_TMEM_LD32(r, o, addr)                                                                                            \
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                                                    \
                 "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28," \
                 "%29,%30,%31}, [%32];"                                                                                       \
                 : "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]), "=r"(r[o + 6]),   \
                   "=r"(r[o + 7]), "=r"(r[o + 8]), "=r"(r[o + 9]), "=r"(r[o + 10]), "=r"(r[o + 11]), "=r"(r[o + 12]),            \
                   "=r"(r[o + 13]), "=r"(r[o + 14]), "=r"(r[o + 15]), "=r"(r[o + 16]), "=r"(r[o + 17]), "=r"(r[o + 18]),         \
                   "=r"(r[o + 19]), "=r"(r[o + 20]), "=r"(r[o + 21]), "=r"(r[o + 22]), "=r"(r[o + 23]), "=r"(r[o + 24]),         \
                   "=r"(r[o + 25]), "=r"(r[o + 26]), "=r"(r[o + 27]), "=r"(r[o + 28]), "=r"(r[o + 29]), "=r"(r[o + 30]),         \
                   "=r"(r[o + 31])                                                                                            \
                 : "r"(addr))

// window of one (quad, subtile) block: mode 1..3 = edges of the window loop, 4 = cell lookup, 5 = fp64; k = first band
template <int MAP>
__device__ __forceinline__ void window_of(const float4 cq, const float4 sp, bool windows, const WinTables& wt, const Lookup& lk, int& mode,
                                          int& k, float& g) {
    const float tx = __fsub_rn(cq.x, sp.x), ty = __fsub_rn(cq.y, sp.y), tz = __fsub_rn(cq.z, sp.z);
    const float dc2 = fmaf(tz, tz, fmaf(ty, ty, tx * tx));
    float dc;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(dc) : "f"(dc2));
    const float rs = cq.w + sp.w;
    const float lo = fmaf(dc, 1.0f - 4.0e-6f, -rs) - 1.0e-7f;
    const float hi = fmaf(dc, 1.0f + 4.0e-6f, rs) + 1.0e-7f;
    g = lookup_guard(lk, rs, hi);
    mode = 4;
    k = 0;
    if (rs > kRCap) {
        mode = 5;
    } else if (windows && lo >= kFarKappa * rs) {
        const float lo2 = __fmul_rd(lo, lo), hi2 = __fmul_ru(hi, hi);
        k = wt.cell_band[cell_off4<MAP, true>(lo2, lk) >> 2];
        while (k < wt.nbands && wt.band_lh[k].y <= lo2) ++k;
        int e = 1;
        while (e <= kMaxWinEdges && k + e < wt.nbands && wt.band_lh[k + e].x <= hi2) ++e;
        mode = e;
    }
}

// Which kernel TPCF_ENGINE_TENSOR launches: the modes of nsamples pseudo-random (8-row group of the i side, 128-row tile of
// the j side) blocks; out[0] += blocks that would be counted pair by pair (cell lookup or fp64), out[1] += blocks sampled.
template <int MAP>
__global__ void sample_modes_kernel(const __grid_constant__ PairParams p, uint32_t nsamples, unsigned long long* __restrict__ out) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const Lookup lk = make_lookup(p, nullptr, nullptr);
    WinTables wt;
    wt.band_mh = p.band_mh;
    wt.band_lh = p.band_lh;
    wt.band_slot = p.band_slot;
    wt.cell_band = p.cell_band;
    wt.whist = nullptr;
    wt.nbands = p.nbands;
    const uint32_t nq = (p.n_i + R - 1) / R, nt = (p.n_j + kTcSubJ - 1) / kTcSubJ;
    uint32_t h = t * 2654435761u + 0x9E3779B9u;             // two multiplicative hashes of the sample number
    h ^= h >> 15;
    h *= 2246822519u;
    h ^= h >> 13;
    const uint32_t qi = (uint32_t)(((unsigned long long)h * nq) >> 32);
    h = h * 3266489917u + 0x85EBCA6Bu;
    h ^= h >> 16;
    const uint32_t tj = (uint32_t)(((unsigned long long)h * nt) >> 32);
    int mode = 0, k = 0;
    float g;
    bool slow = false;
    if (t < nsamples) {
        window_of<MAP>(p.cq[qi], p.ct[tj], p.window != 0, wt, lk, mode, k, g);
        slow = mode > kMaxWinEdges;
    }
    const unsigned ns = __popc(__ballot_sync(0xffffffffu, slow)), nn = __popc(__ballot_sync(0xffffffffu, t < nsamples));
    if ((threadIdx.x & 31) == 0 && nn) {
        atomicAdd(out, (unsigned long long)ns);
        atomicAdd(out + 1, (unsigned long long)nn);
    }
}

struct TcSmem {
    uint32_t ring, abuf, lut, hist, band_mh, band_lh, thr, whist, cell_band, band_slot, bars, slow, rq, misc, total;
};
__host__ __device__ inline TcSmem tc_smem_layout(int ncells, int nbands, int nbins) {
    TcSmem L;
    uint32_t o = 0;
    L.ring = o;       o += kTcRing * ((kTcSlotBytes + 127u) & ~127u);
    L.abuf = o;       o += kTcABytes;
    L.lut = o;        o = up16(o + (uint32_t)ncells * 4);
    L.hist = o;       o = up16(o + (uint32_t)ncells * 8);
    L.band_mh = o;    o = up16(o + (uint32_t)nbands * 8);
    L.band_lh = o;    o = up16(o + (uint32_t)nbands * 8);
    L.thr = o;        o = up16(o + (uint32_t)(nbins + 1) * 8);
    L.whist = o;      o = up16(o + (uint32_t)(nbins + 3) * 4);
    L.cell_band = o;  o = up16(o + (uint32_t)ncells * 2);
    L.band_slot = o;  o = up16(o + (uint32_t)(nbands + 1) * 2);
    L.bars = o;       o = up16(o + (kTcRing + 1) * 8);
    L.slow = o;       o = up16(o + (uint32_t)sizeof(SlowCtx));
    L.rq = o;         o += (kTcThreads / 32) * kRecheckQueue * 8;
    L.misc = o;       o += 16;
    L.total = o;
    return L;
}

// rows of `todo` (one bit per lane = i-row) against the kTcSubJ j-rows at xs: every pair through the cell lookup, the warp
// working together on one row at a time (lane l takes j-rows l, l + 32, ..)
template <int MAP>
__device__ __forceinline__ void tc_lookup_rows(unsigned todo, float sx, float sy, float sz, float g, const float4* __restrict__ xs,
                                               const Lookup& lk, SlowCtx* slow, uint2* rq, unsigned& qn, uint32_t iwarp, uint32_t j0,
                                               bool mask) {
    const int lane = threadIdx.x & 31;
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t i = iwarp + src;
        const float ux = __shfl_sync(0xffffffffu, sx, src), uy = __shfl_sync(0xffffffffu, sy, src), uz = __shfl_sync(0xffffffffu, sz, src);
        const float gs = __shfl_sync(0xffffffffu, g, src);
#pragma unroll
        for (int h = 0; h < kTcSubJ / 32; ++h) {
            const uint32_t j = j0 + h * 32 + lane;
            rq_push(rq, qn, lookup_pair<MAP>(ux, uy, uz, xs[h * 32 + lane], lk, gs, !mask || j > i), i, j, slow);
        }
    }
}

// rows of `todo` against the kTcSubJ j-rows from j0 on in fp64 (radii too large for the fp32 bound, padding rows)
__device__ __noinline__ void tc_exact_rows(SlowCtx* s, unsigned todo, uint32_t iwarp, uint32_t n_i, uint32_t j0, uint32_t n_j, bool mask) {
    const int lane = threadIdx.x & 31;
    unsigned cnt = 0;
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t i = iwarp + src;
        if (i >= n_i) continue;
        const double4 a = s->xi64[i];
#pragma unroll 1
        for (int h = 0; h < kTcSubJ / 32; ++h) {
            const uint32_t j = j0 + h * 32 + lane;
            if (j < n_j && (!mask || j > i)) {
                atomicAdd(s->whist + exact_slot_dev(chord2_f64(a, s->xj64[j]), s->thr, s->nbins), 1u);
                ++cnt;
            }
        }
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0 && cnt) atomicAdd(&s->nrecheck, cnt);
}


// per-thread window parameters of one (row, j-tile) block
struct TcRow {
    float sx, sy, sz;           // the row relative to the tile centre (for the lookup recount)
    float dt1, dt2, hmax;       // mid_0 - mid_e of the further edges, largest band half width
    int mode, k, we;            // this row's mode, first band, edges the warp runs
};

// Bin the kTcSubJ accumulators of this thread's row and count or recount the row.
template <int MAP>
__device__ __forceinline__ void tc_bin(const TcRow& pd, uint32_t taddr, const float4* __restrict__ xs, uint32_t j0, bool mask,
                                       const WinTables& wt, const Lookup& lk, SlowCtx* slow, uint2* rq, unsigned& qn,
                                       uint32_t iwarp, uint32_t n_i, uint32_t n_j, float bg, int owner, unsigned (&npath)[7]) {
    const bool win = pd.mode <= kMaxWinEdges;
    bool flagged = false;
    if (pd.we == 1) {                               // warp-uniform; 95 % of the blocks: the leanest path
        unsigned c0 = 0;
        float m = 3.0e38f;
#pragma unroll 1
        for (int half = 0; half < kTcSubJ / 64; ++half) {
            uint32_t v[64];
            TPCF_TMEM_LD32(v, 0, taddr + half * 64);
            TPCF_TMEM_LD32(v, 32, taddr + half * 64 + 32);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            unsigned ca = 0, cb = 0;                // independent chains
            float ma = 3.0e38f, mb = 3.0e38f;
#pragma unroll
            for (int j = 0; j < 64; j += 4) {
                ca += v[j] >> 31;
                cb += v[j + 1] >> 31;
                ca += v[j + 2] >> 31;
                cb += v[j + 3] >> 31;
                ma = fminf(ma, fminf(fabsf(__uint_as_float(v[j])), fabsf(__uint_as_float(v[j + 1]))));
                mb = fminf(mb, fminf(fabsf(__uint_as_float(v[j + 2])), fabsf(__uint_as_float(v[j + 3]))));
            }
            c0 += ca + cb;
            m = fminf(m, fminf(ma, mb));
        }
        flagged = m <= pd.hmax;
        if (win && !flagged) {                      // c0 pairs below the edge, the rest of the kTcSubJ above it
            if (c0) atomicAdd(wt.whist + wt.band_slot[pd.k], c0);
            if (c0 != kTcSubJ) atomicAdd(wt.whist + wt.band_slot[pd.k + 1], kTcSubJ - c0);
        }
    } else if (pd.we <= kMaxWinEdges) {             // warp-uniform
        unsigned c0 = 0, c1 = 0, c2 = 0;
        float m = 3.0e38f;
#pragma unroll 1
        for (int half = 0; half < kTcSubJ / 64; ++half) {
            uint32_t v[64];
            TPCF_TMEM_LD32(v, 0, taddr + half * 64);
            TPCF_TMEM_LD32(v, 32, taddr + half * 64 + 32);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (pd.we == 2) {
#pragma unroll
                for (int j = 0; j < 64; ++j) {
                    const float q = __uint_as_float(v[j]), q1 = __fadd_rn(q, pd.dt1);
                    c0 += __float_as_uint(q) >> 31;
                    c1 += __float_as_uint(q1) >> 31;
                    m = fminf(m, fminf(fabsf(q), fabsf(q1)));
                }
            } else {
#pragma unroll
                for (int j = 0; j < 64; ++j) {
                    const float q = __uint_as_float(v[j]), q1 = __fadd_rn(q, pd.dt1), q2 = __fadd_rn(q, pd.dt2);
                    c0 += __float_as_uint(q) >> 31;
                    c1 += __float_as_uint(q1) >> 31;
                    c2 += __float_as_uint(q2) >> 31;
                    m = fminf(fminf(m, fabsf(q)), fminf(fabsf(q1), fabsf(q2)));
                }
            }
        }
        flagged = m <= pd.hmax;
        if (win && !flagged) {
            // c_e = pairs below edge e (e < we); the rest of the kTcSubJ lies above the last edge
            const unsigned T = kTcSubJ;
            const unsigned n0 = c0, n1 = c1 - c0, n2 = (pd.we >= 3 ? c2 : T) - c1, n3 = pd.we >= 3 ? T - c2 : 0u;
            if (n0) atomicAdd(wt.whist + wt.band_slot[pd.k], n0);
            if (n1) atomicAdd(wt.whist + wt.band_slot[pd.k + 1], n1);
            if (n2) atomicAdd(wt.whist + wt.band_slot[pd.k + 2], n2);
            if (n3) atomicAdd(wt.whist + wt.band_slot[pd.k + 3], n3);
        }
        ++npath[pd.we == 2 ? 1 : 2];
    } else {
        ++npath[3];
    }
    // rows that saw a pair inside a band, rows whose block needs the cell lookup or fp64: rare, one vote in the common case
    if (__any_sync(0xffffffffu, (win && flagged) || pd.mode > kMaxWinEdges)) {
        const unsigned lkrows = __ballot_sync(0xffffffffu, (win && flagged) || pd.mode == 4);
        const unsigned ex = __ballot_sync(0xffffffffu, pd.mode == 5);
        if (lkrows) {
            const float g = __shfl_sync(0xffffffffu, bg, owner);        // the lookup guard of this row's block: only needed here
            tc_lookup_rows<MAP>(lkrows, pd.sx, pd.sy, pd.sz, g, xs, lk, slow, rq, qn, iwarp, j0, mask);
            npath[4] += __popc(lkrows);
        }
        if (ex) {
            tc_exact_rows(slow, ex, iwarp, n_i, j0, n_j, mask);
            ++npath[5];
        }
    }
}

template <int MAP>
__global__ void __launch_bounds__(kTcThreads, 4) pair_tensor_kernel(const __grid_constant__ PairParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const TcSmem L = tc_smem_layout(p.ncells, p.nbands, p.nbins);
    unsigned* hist = reinterpret_cast<unsigned*>(smem + L.hist);
    const Lookup lk = make_lookup(p, smem + L.lut, smem + L.hist);
    SlowCtx* slow = reinterpret_cast<SlowCtx*>(smem + L.slow);
    WinTables wt;
    wt.band_mh = reinterpret_cast<const float2*>(smem + L.band_mh);
    wt.band_lh = reinterpret_cast<const float2*>(smem + L.band_lh);
    wt.band_slot = reinterpret_cast<const uint16_t*>(smem + L.band_slot);
    wt.cell_band = reinterpret_cast<const uint16_t*>(smem + L.cell_band);
    wt.whist = reinterpret_cast<unsigned*>(smem + L.whist);
    wt.nbands = p.nbands;
    volatile uint32_t* misc = reinterpret_cast<volatile uint32_t*>(smem + L.misc);      // [0] TMEM base, [2..3] next work item

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr uint32_t kSlotStride = (kTcSlotBytes + 127u) & ~127u;
    unsigned char* ring = smem + L.ring;
    const uint32_t ring_bar = smem_u32(smem + L.bars), full_bar = ring_bar + 8 * kTcRing;      // kTcRing slot barriers, "accumulators ready"
    for (int c = tid; c < p.ncells; c += kTcThreads) {
        reinterpret_cast<float*>(smem + L.lut)[c] = p.lut[c];
        hist[c] = 0;
        hist[p.ncells + c] = 0;
        reinterpret_cast<uint16_t*>(smem + L.cell_band)[c] = p.cell_band[c];
    }
    for (int b = tid; b < p.nbands; b += kTcThreads) {
        reinterpret_cast<float2*>(smem + L.band_mh)[b] = p.band_mh[b];
        reinterpret_cast<float2*>(smem + L.band_lh)[b] = p.band_lh[b];
    }
    for (int b = tid; b <= p.nbands; b += kTcThreads) reinterpret_cast<uint16_t*>(smem + L.band_slot)[b] = p.band_slot[b];
    for (int b = tid; b < p.nbins + 3; b += kTcThreads) wt.whist[b] = 0;
    for (int b = tid; b <= p.nbins; b += kTcThreads) reinterpret_cast<double*>(smem + L.thr)[b] = p.thr[b];
    // operand row of this thread in the A tile: K chunk 3 = (1, 1, 1, 0) never changes
    unsigned char* arow = smem + L.abuf + (tid / 8) * kTcSbo + (tid % 8) * 16;
    *reinterpret_cast<float4*>(arow + 3 * kTcALbo) = make_float4(1.f, 1.f, 1.f, 0.f);
    if (tid == 0) {
        for (int b = 0; b < kTcRing + 1; ++b) mbar_init(ring_bar + 8 * b, 1);
        fence_barrier_init();
        slow->xi64 = p.xi64;
        slow->xj64 = p.xj64;
        slow->thr = reinterpret_cast<const double*>(smem + L.thr);
        slow->whist = wt.whist;
        slow->nrecheck = 0;
        slow->nbins = p.nbins;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem + L.misc)), "r"(kTcCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    fence_proxy_async();
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = misc[0];
    const uint32_t tlane = tmem + ((uint32_t)warp * 32u << 16);

    auto fetch_tile = [&](uint32_t n, uint32_t t) {       // thread 0: j-tile t into the slot of running tile number n
        const uint32_t slot = n % kTcRing, bar = ring_bar + 8 * slot;
        const uint32_t dst = smem_u32(ring + (size_t)slot * kSlotStride);
        fence_proxy_async();
        mbar_expect_tx(bar, kTcSlotBytes);
        bulk_g2s(dst, p.xb + (size_t)t * kTcSubJ * kTcK, kTcBBytes, bar);
        bulk_g2s(dst + kTcBBytes, p.xt + (size_t)t * kTcSubJ, kTcRowBytes, bar);
        bulk_g2s(dst + kTcBBytes + kTcRowBytes, p.ct + t, sizeof(float4), bar);
    };

    constexpr uint32_t kCtasPerItem = kTileI / kTcThreads;
    const uint32_t per_item = kCtasPerItem * p.jsplit;
    const unsigned long long n_citems = (unsigned long long)p.n_items_part * per_item;
    const uint32_t per_row = (p.tiles_j + p.chunk - 1) / p.chunk;
    uint2* rq = reinterpret_cast<uint2*>(smem + L.rq) + (size_t)warp * kRecheckQueue;
    unsigned qn = 0;
    uint32_t gch = 0, gs = 0;               // j-tiles fetched / multiplied so far: ring slot and mbarrier parities
    unsigned long long pairs_since_flush = 0, items_done = 0;
    unsigned npath[7] = {0, 0, 0, 0, 0, 0, 0};
    for (;;) {
        if (tid == 0) {
            const unsigned long long c = atomicAdd(p.counters, 1ull);
            misc[2] = (uint32_t)c;
            misc[3] = (uint32_t)(c >> 32);
        }
        __syncthreads();
        const unsigned long long c = ((unsigned long long)misc[3] << 32) | misc[2];
        if (c >= n_citems) break;
        const uint32_t w = (uint32_t)(c / per_item) * p.nparts + p.part, ws = (uint32_t)(c % per_item) / p.jsplit, js = (uint32_t)(c % p.jsplit);
        uint32_t I, tile0;
        if (p.tri) {
            I = tri_row_of(p.row_start, p.blocks_i, w, lane);
            tile0 = I + (w - p.row_start[I]) * p.chunk;
        } else {
            I = w / per_row;
            tile0 = (w % per_row) * p.chunk;
        }
        const uint32_t ntiles = min(p.chunk, p.tiles_j - tile0);
        // this thread's row as an offset from the centre of its 8-row quad; a quad wholly past the end of the catalog
        // is moved to (-2,-2,-2) as in pair_fast_kernel
        const uint32_t ibase = I * kTileI + ws * kTcThreads, i = ibase + tid, iq = i & ~(uint32_t)(R - 1);
        float4 a = p.xq[i], cq = p.cq[i / R];
        if (iq >= p.n_i) {
            a = make_float4(0.f, 0.f, 0.f, 0.f);
            cq = make_float4(-kPadCoord, -kPadCoord, -kPadCoord, 0.f);
        }
        const uint32_t dch = ibase / kChunkJ;
        uint32_t ch = tile0 * (kTileJ / kChunkJ), ch_end = (tile0 + ntiles) * (kTileJ / kChunkJ);
        if (p.jsplit > 1) {
            ch += js * ((kTileJ / kChunkJ) / p.jsplit);
            ch_end = ch + (kTileJ / kChunkJ) / p.jsplit;
        }
        if (p.tri) ch = max(ch, dch);
        const uint32_t ntile = ch < ch_end ? ch_end - ch : 0u;      // j-tiles of this item (a tile = a 128-row chunk)
        if (tid == 0)
            for (uint32_t n = 0; n < min(ntile, (uint32_t)kTcRing); ++n) fetch_tile(gch + n, ch + n);

        // window of (this thread's quad, tile (lane & 7) of the current batch of 8), packed: mode | edges the warp runs << 3 |
        // first band << 6; the lookup guard beside it
        int bpack = 4 | (4 << 3);
        float bg = 0.f;
        for (uint32_t t = 0; t < ntile; ++t) {
            const uint32_t n = gch + t, tabs = ch + t;
            unsigned char* slot = ring + (size_t)(n % kTcRing) * kSlotStride;
            mbar_wait(ring_bar + 8 * (n % kTcRing), (n / kTcRing) & 1);
            const bool mask = p.tri && tabs == dch;
            if (t == 0 || (tabs & 7u) == 0) {               // windows of 8 tiles at a time, one per lane of the quad
                const uint32_t su = (tabs & ~7u) + (lane & 7);
                int bmode, bk;
                window_of<MAP>(cq, p.ct[su], p.window != 0, wt, lk, bmode, bk, bg);
                // the warp runs, per tile, the largest window loop one of its four quads needs (none: all rows pair by pair)
                int wm = bmode <= kMaxWinEdges ? bmode : 0;
                wm = max(wm, __shfl_xor_sync(0xffffffffu, wm, 8));
                wm = max(wm, __shfl_xor_sync(0xffffffffu, wm, 16));
                const int bwe = wm ? wm : kMaxWinEdges + 1;
                bpack = bmode | (bwe << 3) | ((bmode > kMaxWinEdges ? 0 : min(bk, p.nbands - bwe)) << 6);
            }
            const int owner = (lane & ~7) | (int)(tabs & 7u);
            const int pk = __shfl_sync(0xffffffffu, bpack, owner);
            TcRow rw;
            rw.mode = pk & 7;
            rw.we = (pk >> 3) & 7;
            rw.k = pk >> 6;
            if (mask) {                                     // the diagonal tile: every row pair by pair (pairs j > i)
                rw.mode = max(rw.mode, 4);
                rw.we = kMaxWinEdges + 1;
                rw.k = 0;
            }
            const float4 sp = *reinterpret_cast<const float4*>(slot + kTcBBytes + kTcRowBytes);
            const float tx = __fsub_rn(cq.x, sp.x), ty = __fsub_rn(cq.y, sp.y), tz = __fsub_rn(cq.z, sp.z);
            rw.sx = __fadd_rn(a.x, tx);
            rw.sy = __fadd_rn(a.y, ty);
            rw.sz = __fadd_rn(a.z, tz);
            const float2 mh0 = wt.band_mh[rw.k];
            rw.hmax = mh0.y;
            rw.dt1 = rw.dt2 = 0.f;
            if (rw.we == 2 || rw.we == 3) {
                const float2 mh = wt.band_mh[rw.k + 1];
                rw.dt1 = __fsub_rn(mh0.x, mh.x);
                rw.hmax = fmaxf(rw.hmax, mh.y);
            }
            if (rw.we == 3) {
                const float2 mh = wt.band_mh[rw.k + 2];
                rw.dt2 = __fsub_rn(mh0.x, mh.x);
                rw.hmax = fmaxf(rw.hmax, mh.y);
            }
            {
                const float nsm = __fadd_rn(fmaf(rw.sz, rw.sz, fmaf(rw.sy, rw.sy, rw.sx * rw.sx)), -mh0.x);
                const float xh = tf32_hi(rw.sx), yh = tf32_hi(rw.sy), zh = tf32_hi(rw.sz);
                const float xl = tf32_hi(rw.sx - xh), yl = tf32_hi(rw.sy - yh), zl = tf32_hi(rw.sz - zh);
                const float nh = tf32_hi(nsm), nm = tf32_hi(nsm - nh), nl = tf32_hi((nsm - nh) - nm);
                *reinterpret_cast<float4*>(arow) = make_float4(xh, yh, zh, xh);
                *reinterpret_cast<float4*>(arow + kTcALbo) = make_float4(yh, zh, xl, yl);
                *reinterpret_cast<float4*>(arow + 2 * kTcALbo) = make_float4(zl, nh, nm, nl);
            }
            fence_proxy_async();
            // operand rows written and the accumulators of the previous tile read by every thread
            asm volatile("tcgen05.fence::before_thread_sync;");
            __syncthreads();
            asm volatile("tcgen05.fence::after_thread_sync;");
            if (tid == 0) {
                const uint32_t sa = smem_u32(smem + L.abuf), sb = smem_u32(slot);
#pragma unroll
                for (int ks = 0; ks < kTcK / 8; ++ks) {
                    const uint64_t da = umma_desc(sa + ks * 2 * kTcALbo, kTcALbo, kTcSbo), db = umma_desc(sb + ks * 2 * kTcBLbo, kTcBLbo, kTcSbo);
                    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}" ::"r"(tmem),
                                 "l"(da), "l"(db), "r"(kTcIdesc), "r"(ks)
                                 : "memory");
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(full_bar) : "memory");
                // every thread is past the bin of tile t - 1: its slot takes tile t + 2
                if (t >= 1 && t + kTcRing - 1 < ntile) fetch_tile(n + kTcRing - 1, tabs + kTcRing - 1);
            }
            mbar_wait(full_bar, gs & 1);
            asm volatile("tcgen05.fence::after_thread_sync;");
            tc_bin<MAP>(rw, tlane, reinterpret_cast<const float4*>(slot + kTcBBytes), tabs * kTcSubJ, mask, wt, lk, slow, rq, qn,
                        ibase + warp * 32, p.n_i, p.n_j, bg, owner, npath);
            ++gs;
        }
        const uint32_t nchunks = ntile;
        gch += nchunks;
        pairs_since_flush += (unsigned long long)nchunks * kChunkJ * kTcThreads;
        if (tid == 0 && ws == 0 && js == 0) ++items_done;
        __syncthreads();
        if (pairs_since_flush > kFlushPairs) {
            flush_slots(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result, &slow->nrecheck, p.counters + 1, tid, kTcThreads);
            pairs_since_flush = 0;
            __syncthreads();
        }
    }
    rq_drain(rq, qn, slow);
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    flush_slots(hist, 2 * p.ncells, p.slotmap, wt.whist, p.nbins + 3, p.result, &slow->nrecheck, p.counters + 1, tid, kTcThreads);
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTcCols));
    if (tid == 0 && items_done) atomicAdd(p.counters + 2, items_done);
    if (lane == 0) {
        npath[0] = gs - npath[1] - npath[2] - npath[3];      // the one-edge blocks are not counted one by one
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (npath[k]) atomicAdd(p.counters + 3 + k, (unsigned long long)npath[k]);
    }
}

// One (128 i-rows) x (128 j-rows) tile through exactly the operand preparation, MMA and read-back of pair_tensor_kernel,
// returning the accumulators instead of binning them: the measurement behind the tensor engine's error bound
// (tpcf_tensor_probe, tests/test_gpu_tensor.py).  srows = (s, |s|^2 - mid_0) per i-row, brows = (-2 b', |b'|^2) per j-row.
__global__ void __launch_bounds__(kTcThreads) tensor_probe_kernel(const float4* __restrict__ srows, const float4* __restrict__ brows,
                                                                  float* __restrict__ q) {
    __shared__ __align__(128) unsigned char sA[kTcABytes];
    __shared__ __align__(128) unsigned char sB[kTcBBytes];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t tbase;
    const int tid = threadIdx.x, warp = tid >> 5;
    const float4 sr = srows[(size_t)blockIdx.x * kTcThreads + tid], br = brows[(size_t)blockIdx.x * kTcSubJ + tid];
    unsigned char* ar = sA + (tid / 8) * kTcSbo + (tid % 8) * 16;
    unsigned char* bp = sB + (tid / 8) * kTcSbo + (tid % 8) * 16;
    {
        const float xh = tf32_hi(sr.x), yh = tf32_hi(sr.y), zh = tf32_hi(sr.z);
        const float xl = tf32_hi(sr.x - xh), yl = tf32_hi(sr.y - yh), zl = tf32_hi(sr.z - zh);
        const float nh = tf32_hi(sr.w), nm = tf32_hi(sr.w - nh), nl = tf32_hi((sr.w - nh) - nm);
        *reinterpret_cast<float4*>(ar) = make_float4(xh, yh, zh, xh);
        *reinterpret_cast<float4*>(ar + kTcALbo) = make_float4(yh, zh, xl, yl);
        *reinterpret_cast<float4*>(ar + 2 * kTcALbo) = make_float4(zl, nh, nm, nl);
        *reinterpret_cast<float4*>(ar + 3 * kTcALbo) = make_float4(1.f, 1.f, 1.f, 0.f);
        const float mh0 = tf32_hi(br.x), mh1 = tf32_hi(br.y), mh2 = tf32_hi(br.z);
        const float ml0 = tf32_hi(br.x - mh0), ml1 = tf32_hi(br.y - mh1), ml2 = tf32_hi(br.z - mh2);
        const float wh = tf32_hi(br.w), wm = tf32_hi(br.w - wh), wl = tf32_hi((br.w - wh) - wm);
        *reinterpret_cast<float4*>(bp) = make_float4(mh0, mh1, mh2, ml0);
        *reinterpret_cast<float4*>(bp + kTcBLbo) = make_float4(ml1, ml2, mh0, mh1);
        *reinterpret_cast<float4*>(bp + 2 * kTcBLbo) = make_float4(mh2, 1.f, 1.f, 1.f);
        *reinterpret_cast<float4*>(bp + 3 * kTcBLbo) = make_float4(wh, wm, wl, 0.f);
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tbase)), "r"(kTcCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid == 0) {
        mbar_init(smem_u32(&bar), 1);
        fence_barrier_init();
    }
    fence_proxy_async();
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = tbase;
    if (tid == 0) {
#pragma unroll
        for (int ks = 0; ks < kTcK / 8; ++ks) {
            const uint64_t da = umma_desc(smem_u32(sA) + ks * 2 * kTcALbo, kTcALbo, kTcSbo), db = umma_desc(smem_u32(sB) + ks * 2 * kTcBLbo, kTcBLbo, kTcSbo);
            asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}" ::"r"(tmem), "l"(da),
                         "l"(db), "r"(kTcIdesc), "r"(ks)
                         : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)) : "memory");
    }
    mbar_wait(smem_u32(&bar), 0);
    asm volatile("tcgen05.fence::after_thread_sync;");
    float* out = q + ((size_t)blockIdx.x * kTcThreads + tid) * kTcSubJ;
#pragma unroll 1
    for (int half = 0; half < kTcSubJ / 64; ++half) {
        uint32_t v[64];
        const uint32_t ta = tmem + ((uint32_t)warp * 32u << 16) + half * 64;
        TPCF_TMEM_LD32(v, 0, ta);
        TPCF_TMEM_LD32(v, 32, ta + 32);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int j = 0; j < 64; ++j) out[half * 64 + j] = __uint_as_float(v[j]);
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTcCols));
}

// ---- fp64 engine: work items per CTA -------------------------------------------------------------------------
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
        // at most kMaxChunk * kTileI * kTileJ = 2^25 pairs per item and slot: 32 items stay below 2^31
        if ((items_done & 31) == 0) {
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

// ---- weighted sums: sum of w_i w_j per bin, fp64 throughout -------------------------
// The same plan and the same fp64 classification as pair_exact64_kernel; the CTA's partial sums are fp64 shared-memory
// atomics, added to the global fp64 sums after every work item (at most 2^25 terms per partial: DESIGN.md section 14).
__global__ void __launch_bounds__(kThreads) pair_weighted64_kernel(const __grid_constant__ PairParams p, const double* __restrict__ wi,
                                                                   const double* __restrict__ wj, double* __restrict__ wresult) {
    extern __shared__ __align__(128) unsigned char smem[];
    double* thr = reinterpret_cast<double*>(smem);
    double* sums = thr + p.nbins + 1;
    __shared__ Item s_item;
    const int tid = threadIdx.x, nslots = p.nbins + 3;
    for (int k = tid; k <= p.nbins; k += kThreads) thr[k] = p.thr[k];
    for (int k = tid; k < nslots; k += kThreads) sums[k] = 0.0;
    __syncthreads();
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
            const double w = wi[i];
            const uint32_t jbeg = it.tile0 * kTileJ, jend = min(p.n_j, (it.tile0 + it.ntiles) * kTileJ);
            for (uint32_t j = jbeg; j < jend; ++j) {
                if (p.tri && j <= i) continue;
                const int slot = exact_slot_dev(chord2_f64(a, p.xj64[j]), thr, p.nbins);
                atomicAdd(sums + slot, w * wj[j]);
            }
        }
        __syncthreads();
        for (int k = tid; k < nslots; k += kThreads) {
            if (sums[k] != 0.0) atomicAdd(wresult + k, sums[k]);
            sums[k] = 0.0;
        }
        __syncthreads();
    }
}

// weights in the caller's row order -> sorted order (inv: caller row -> sorted position), 0 for the padding rows
__global__ void scatter_weights_kernel(const double* __restrict__ w, const uint32_t* __restrict__ inv, uint64_t n, uint64_t n_pad,
                                       double* __restrict__ out) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        if (k < n) out[inv[k]] = w[k];
        else out[k] = 0.0;
    }
}

// ---- load / convert / spatial sort (step a1) -------------------------------------------------------------------
// Bounding boxes of a catalog for the sort keys, as order-preserving 64-bit images of doubles (atomicMin / atomicMax):
// angular: per cube face f the gnomonic coordinates' [4f] u_min, [4f+1] u_max, [4f+2] v_min, [4f+3] v_max; 3-D: [0..5] =
// x_min, x_max, y_min, y_max, z_min, z_max.
constexpr int kBoundWords = 24;
__device__ __forceinline__ unsigned long long ordered_bits(double x) {
    const long long b = __double_as_longlong(x);
    return (unsigned long long)(b ^ ((b >> 63) | (long long)0x8000000000000000ull));
}
__device__ __forceinline__ double from_ordered_bits(unsigned long long o) {
    const long long b = (long long)o;
    return __longlong_as_double(b ^ ((~b >> 63) | (long long)0x8000000000000000ull));
}
__device__ __forceinline__ void face_uv(double x, double y, double z, int& face, double& u, double& v) {
    const double ax = fabs(x), ay = fabs(y), az = fabs(z);
    double m;
    if (ax >= ay && ax >= az) { face = x >= 0 ? 0 : 1; u = y; v = z; m = ax; }
    else if (ay >= az)        { face = y >= 0 ? 2 : 3; u = z; v = x; m = ay; }
    else                      { face = z >= 0 ? 4 : 5; u = x; v = y; m = az; }
    u /= m;
    v /= m;
}
// the warp's minimum / maximum of a value into the bound slots (one atomic pair per warp and slot pair)
__device__ __forceinline__ void bound_update(unsigned long long* b, int slot_min, bool valid, double x) {
    unsigned long long lo = valid ? ordered_bits(x) : ~0ull, hi = valid ? ordered_bits(x) : 0ull;
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, off));
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, off));
    }
    if ((threadIdx.x & 31) == 0 && lo <= hi) {
        atomicMin(b + slot_min, lo);
        atomicMax(b + slot_min + 1, hi);
    }
}
__global__ void bounds_init_kernel(unsigned long long* b) {
    if (threadIdx.x < kBoundWords) b[threadIdx.x] = (threadIdx.x & 1) ? 0ull : ~0ull;
}

// Sort key of a unit vector: the face of the circumscribed cube it projects onto (3 bits) followed by the 56-bit
// index of its projection along a 2-D Hilbert curve (28 bits per axis) of the smallest square of that face, anchored at
// the corner (u_min, v_min), that holds every row of the catalog on the face: the curve then stays inside the populated
// region, so consecutive rows of the sorted catalog are neighbours on the sky (except at the <= 5 face changes), which is
// what keeps the bounding spheres of quads and subtiles small.  Only the ORDER the key induces is used: counts do not
// depend on it.
__device__ inline unsigned long long hilbert_key(double x, double y, double z, const unsigned long long* __restrict__ bounds) {
    constexpr int B = 28;
    int face;
    double u, v;
    face_uv(x, y, z, face, u, v);
    const double u0 = from_ordered_bits(bounds[4 * face]), u1 = from_ordered_bits(bounds[4 * face + 1]);
    const double v0 = from_ordered_bits(bounds[4 * face + 2]), v1 = from_ordered_bits(bounds[4 * face + 3]);
    const double side = fmax(fmax(u1 - u0, v1 - v0), 1.0e-300);
    const double scale = (double)((1u << B) - 1) / side;
    uint32_t X = (uint32_t)fmin(fmax((u - u0) * scale, 0.0), (double)((1u << B) - 1));
    uint32_t Y = (uint32_t)fmin(fmax((v - v0) * scale, 0.0), (double)((1u << B) - 1));
    unsigned long long d = 0;
    for (uint32_t s = 1u << (B - 1); s > 0; s >>= 1) {
        const uint32_t rx = (X & s) ? 1u : 0u, ry = (Y & s) ? 1u : 0u;
        d += (unsigned long long)s * s * ((3u * rx) ^ ry);
        if (ry == 0) {                                  // rotate the quadrant
            if (rx == 1) {
                X = (1u << B) - 1 - X;
                Y = (1u << B) - 1 - Y;
            }
            const uint32_t t = X;
            X = Y;
            Y = t;
        }
    }
    return ((unsigned long long)face << (2 * B)) | d;
}

// x = cos(dec) cos(ra), y = cos(dec) sin(ra), z = sin(dec) in fp64 (reading A8), in the caller's row order.
template <typename T>
__global__ void convert_kernel(const T* __restrict__ radec, uint64_t n, double4* __restrict__ x64_rows,
                               unsigned long long* __restrict__ bounds, uint32_t* __restrict__ idx, int* __restrict__ bad) {
    const double kPi = 3.14159265358979323846;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k0 = blockIdx.x * (uint64_t)blockDim.x; k0 < n; k0 += stride) {      // whole warps walk together (shuffles below)
        const uint64_t k = k0 + threadIdx.x;
        const bool valid = k < n;
        double4 v = make_double4(1.0, 0.0, 0.0, 0.0);
        if (valid) {
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
            idx[k] = (uint32_t)k;
        }
        int face;
        double fu, fv;
        face_uv(v.x, v.y, v.z, face, fu, fv);
        __syncwarp();
        for (int f = 0; f < 6; ++f) {
            bound_update(bounds, 4 * f, valid && face == f, fu);
            bound_update(bounds, 4 * f + 2, valid && face == f, fv);
        }
    }
}

// second pass of the load: the sort keys, once the bounding boxes are known
__global__ void keys_kernel(const double4* __restrict__ x64_rows, uint64_t n, const unsigned long long* __restrict__ bounds, int spatial,
                            unsigned long long* __restrict__ keys);

// 3-D variant: sort key of a position = its index along a 3-D Hilbert curve (21 bits per axis; Skilling's transpose
// algorithm: inverse undo, Gray encode, then the bits of the three axes interleaved) of the smallest cube anchored at
// (x_min, y_min, z_min) that holds the catalog.  As above only the ORDER matters.
__device__ inline unsigned long long hilbert_key3(double x, double y, double z, const unsigned long long* __restrict__ bounds) {
    constexpr int B = 21;
    const double x0 = from_ordered_bits(bounds[0]), y0 = from_ordered_bits(bounds[2]), z0 = from_ordered_bits(bounds[4]);
    const double side = fmax(fmax(fmax(from_ordered_bits(bounds[1]) - x0, from_ordered_bits(bounds[3]) - y0), from_ordered_bits(bounds[5]) - z0), 1.0e-300);
    const double scale = (double)((1u << B) - 1) / side;
    uint32_t X[3];
    X[0] = (uint32_t)fmin(fmax((x - x0) * scale, 0.0), (double)((1u << B) - 1));
    X[1] = (uint32_t)fmin(fmax((y - y0) * scale, 0.0), (double)((1u << B) - 1));
    X[2] = (uint32_t)fmin(fmax((z - z0) * scale, 0.0), (double)((1u << B) - 1));
    const uint32_t M = 1u << (B - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
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
    X[1] ^= X[0];
    X[2] ^= X[1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t;
    X[1] ^= t;
    X[2] ^= t;
    unsigned long long d = 0;
    for (int bit = B - 1; bit >= 0; --bit)
#pragma unroll
        for (int i = 0; i < 3; ++i) d = (d << 1) | ((X[i] >> bit) & 1u);
    return d;
}

// 3-D variant of convert_kernel: rows (x, y, z) in the caller's units -> position * scale (a power of two: exact) inside
// the unit ball, in the caller's row order.  A row with a non-finite coordinate or |coordinate| > max_abs sets *bad.
template <typename T>
__global__ void convert_xyz_kernel(const T* __restrict__ xyz, uint64_t n, double scale, double max_abs, double4* __restrict__ x64_rows,
                                   unsigned long long* __restrict__ bounds, uint32_t* __restrict__ idx, int* __restrict__ bad) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k0 = blockIdx.x * (uint64_t)blockDim.x; k0 < n; k0 += stride) {
        const uint64_t k = k0 + threadIdx.x;
        const bool valid = k < n;
        double4 v = make_double4(0.0, 0.0, 0.0, 0.0);
        bool good = false;
        if (valid) {
            const double x = (double)xyz[3 * k], y = (double)xyz[3 * k + 1], z = (double)xyz[3 * k + 2];
            if (!(fabs(x) <= max_abs) || !(fabs(y) <= max_abs) || !(fabs(z) <= max_abs)) {      // also catches NaN and inf
                *bad = 1;
            } else {
                v = make_double4(x * scale, y * scale, z * scale, 0.0);
                good = true;
            }
            x64_rows[k] = v;
            idx[k] = (uint32_t)k;
        }
        __syncwarp();
        bound_update(bounds, 0, good, v.x);
        bound_update(bounds, 2, good, v.y);
        bound_update(bounds, 4, good, v.z);
    }
}

__global__ void keys_kernel(const double4* __restrict__ x64_rows, uint64_t n, const unsigned long long* __restrict__ bounds, int spatial,
                            unsigned long long* __restrict__ keys) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
        const double4 v = x64_rows[k];
        keys[k] = spatial ? hilbert_key3(v.x, v.y, v.z, bounds) : hilbert_key(v.x, v.y, v.z, bounds);
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

// The sorted catalog: fp64 rows in Hilbert order and the inverse permutation for row-subset mode; rows n..n_pad-1
// become the padding point (2,2,2).
__global__ void permute_kernel(const double4* __restrict__ x64_rows, const uint32_t* __restrict__ order, uint64_t n,
                               uint64_t n_pad, double4* __restrict__ x64, uint32_t* __restrict__ inv) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < n_pad; k += (uint64_t)gridDim.x * blockDim.x) {
        double4 v = make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
        if (k < n) {
            const uint32_t src = order[k];
            v = x64_rows[src];
            inv[src] = (uint32_t)k;
        }
        x64[k] = v;
    }
}

// i-side role of a catalog: every kIPerThread = 8 consecutive rows form a group ("quad" in the names below: one lane
// of the pair kernel).
// cq = (fp32 centre, radius): the centre is the fp32 rounding of the mean, the radius bounds the fp64 distance of
// the fp64 rows from that fp32 point (rounded up, with slack).  xq = fp32 rounding of (row - centre), formed in fp64:
// its error is 2^-24 of the OFFSET, not of the unit vector.
__global__ void quads_kernel(const double4* __restrict__ x64, uint64_t nquads, float4* __restrict__ xq, float4* __restrict__ cq) {
    for (uint64_t q = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; q < nquads; q += (uint64_t)gridDim.x * blockDim.x) {
        double4 v[kIPerThread];
        double sx = 0, sy = 0, sz = 0;
#pragma unroll
        for (int r = 0; r < kIPerThread; ++r) {
            v[r] = x64[q * kIPerThread + r];
            sx += v[r].x; sy += v[r].y; sz += v[r].z;
        }
        const float cx = (float)(sx / kIPerThread), cy = (float)(sy / kIPerThread), cz = (float)(sz / kIPerThread);
        double rad = 0;
#pragma unroll
        for (int r = 0; r < kIPerThread; ++r) {
            const double dx = v[r].x - (double)cx, dy = v[r].y - (double)cy, dz = v[r].z - (double)cz;
            rad = fmax(rad, sqrt(dx * dx + dy * dy + dz * dz));
            xq[q * kIPerThread + r] = make_float4((float)dx, (float)dy, (float)dz, 0.f);
        }
        cq[q] = make_float4(cx, cy, cz, __double2float_ru(rad * (1.0 + 1.0e-7) + 1.0e-12));
    }
}

// j-side role: every kSubJ consecutive rows form a subtile (one warp here).  cs = (fp32 centre, radius) as
// above; xs = (-2 b', |b'|^2) with b' the fp32 rounding of (row - centre) formed in fp64 and |b'|^2 the fp32
// rounding of the fp64 square of that rounded offset (the window loops evaluate |a - b|^2 = |a|^2 + |b|^2 - 2 a.b).
template <int SUBJ>
__global__ void subtiles_kernel(const double4* __restrict__ x64, uint64_t nsub, float4* __restrict__ xs, float4* __restrict__ cs,
                                float* __restrict__ xb) {
    constexpr int H = SUBJ / 32;                   // rows per lane
    const uint64_t w = (blockIdx.x * (uint64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= nsub) return;
    double4 v[H];
    double sx = 0, sy = 0, sz = 0;
#pragma unroll
    for (int h = 0; h < H; ++h) {
        v[h] = x64[w * SUBJ + h * 32 + lane];
        sx += v[h].x; sy += v[h].y; sz += v[h].z;
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, off);
        sy += __shfl_xor_sync(0xffffffffu, sy, off);
        sz += __shfl_xor_sync(0xffffffffu, sz, off);
    }
    const float cx = (float)(sx / SUBJ), cy = (float)(sy / SUBJ), cz = (float)(sz / SUBJ);
    double r = 0;
#pragma unroll
    for (int h = 0; h < H; ++h) {
        const double dx = v[h].x - (double)cx, dy = v[h].y - (double)cy, dz = v[h].z - (double)cz;
        r = fmax(r, sqrt(dx * dx + dy * dy + dz * dz));
        const float bx = (float)dx, by = (float)dy, bz = (float)dz;
        const double nb = (double)bx * bx + (double)by * by + (double)bz * bz;
        xs[w * SUBJ + h * 32 + lane] = make_float4(-2.f * bx, -2.f * by, -2.f * bz, (float)nb);
        if (xb) {   // the same row as a K = 16 TF32 operand row of the tensor engine (layout: kernels.cuh)
            const int j = h * 32 + lane;
            float* t = xb + (size_t)w * SUBJ * kTcK + (j / 8) * 32 + (j % 8) * 4;
            const float m[3] = {-2.f * bx, -2.f * by, -2.f * bz};
            float mh[3], ml[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                mh[d] = tf32_hi(m[d]);
                ml[d] = tf32_hi(m[d] - mh[d]);
            }
            const float wv = (float)nb, wh = tf32_hi(wv), wm = tf32_hi(wv - wh), wl = tf32_hi((wv - wh) - wm);
            *reinterpret_cast<float4*>(t + 0 * SUBJ * 4) = make_float4(mh[0], mh[1], mh[2], ml[0]);
            *reinterpret_cast<float4*>(t + 1 * SUBJ * 4) = make_float4(ml[1], ml[2], mh[0], mh[1]);
            *reinterpret_cast<float4*>(t + 2 * SUBJ * 4) = make_float4(mh[2], 1.f, 1.f, 1.f);
            *reinterpret_cast<float4*>(t + 3 * SUBJ * 4) = make_float4(wh, wm, wl, 0.f);
        }
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) r = fmax(r, __shfl_xor_sync(0xffffffffu, r, off));
    if (lane == 0) cs[w] = make_float4(cx, cy, cz, __double2float_ru(r * (1.0 + 1.0e-7) + 1.0e-12));
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

__global__ void gather_kernel(const double4* __restrict__ src64, const unsigned long long* __restrict__ pos, uint64_t nrows,
                              uint64_t nrows_pad, double4* __restrict__ dst64) {
    for (uint64_t k = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; k < nrows_pad; k += (uint64_t)gridDim.x * blockDim.x)
        dst64[k] = (k < nrows) ? src64[pos[k]] : make_double4((double)kPadCoord, (double)kPadCoord, (double)kPadCoord, 0.0);
}

__global__ void finalize_kernel(const unsigned long long* __restrict__ result, int nbins, int zero_slot,
                                unsigned long long self_pairs, unsigned long long* __restrict__ out) {
    for (int k = threadIdx.x; k < nbins + 2; k += blockDim.x) out[k] = result[k] - (k == zero_slot ? self_pairs : 0ull);
}

}  // namespace

static int grid_for(uint64_t n, int block) { return (int)std::max<uint64_t>(1, std::min<uint64_t>((n + block - 1) / block, 148ull * 16)); }

cudaError_t launch_convert(const void* radec, int is_f64, uint64_t n, double4* x64_rows, uint64_t* keys, uint32_t* idx,
                           int* bad_flag, uint64_t* bounds, cudaStream_t st) {
    const int block = 256, grid = grid_for(n, block);
    auto* k = reinterpret_cast<unsigned long long*>(keys);
    auto* b = reinterpret_cast<unsigned long long*>(bounds);
    bounds_init_kernel<<<1, 32, 0, st>>>(b);
    if (is_f64)
        convert_kernel<double><<<grid, block, 0, st>>>(static_cast<const double*>(radec), n, x64_rows, b, idx, bad_flag);
    else
        convert_kernel<float><<<grid, block, 0, st>>>(static_cast<const float*>(radec), n, x64_rows, b, idx, bad_flag);
    keys_kernel<<<grid, block, 0, st>>>(x64_rows, n, b, 0, k);
    return cudaGetLastError();
}

cudaError_t launch_convert_xyz(const void* xyz, int is_f64, uint64_t n, double scale, double max_abs, double4* x64_rows, uint64_t* keys,
                               uint32_t* idx, int* bad_flag, uint64_t* bounds, cudaStream_t st) {
    const int block = 256, grid = grid_for(n, block);
    auto* k = reinterpret_cast<unsigned long long*>(keys);
    auto* b = reinterpret_cast<unsigned long long*>(bounds);
    bounds_init_kernel<<<1, 32, 0, st>>>(b);
    if (is_f64)
        convert_xyz_kernel<double><<<grid, block, 0, st>>>(static_cast<const double*>(xyz), n, scale, max_abs, x64_rows, b, idx, bad_flag);
    else
        convert_xyz_kernel<float><<<grid, block, 0, st>>>(static_cast<const float*>(xyz), n, scale, max_abs, x64_rows, b, idx, bad_flag);
    keys_kernel<<<grid, block, 0, st>>>(x64_rows, n, b, 1, k);
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
                           uint32_t* inv, cudaStream_t st) {
    const int block = 256;
    permute_kernel<<<grid_for(n_pad, block), block, 0, st>>>(x64_rows, order, n, n_pad, x64, inv);
    return cudaGetLastError();
}

cudaError_t launch_quads(const double4* x64, uint64_t n_pad, float4* xq, float4* cq, cudaStream_t st) {
    const int block = 128;
    quads_kernel<<<grid_for(n_pad / kIPerThread, block), block, 0, st>>>(x64, n_pad / kIPerThread, xq, cq);
    return cudaGetLastError();
}

cudaError_t launch_subtiles(const double4* x64, uint64_t n_pad, float4* xs, float4* cs, float4* xt, float4* ct, float* xb,
                            cudaStream_t st) {
    const int block = 256;
    const uint64_t nsub = n_pad / kSubJ, ntile = n_pad / kTcSubJ;
    subtiles_kernel<kSubJ><<<(unsigned)((nsub * 32 + block - 1) / block), block, 0, st>>>(x64, nsub, xs, cs, nullptr);
    subtiles_kernel<kTcSubJ><<<(unsigned)((ntile * 32 + block - 1) / block), block, 0, st>>>(x64, ntile, xt, ct, xb);
    return cudaGetLastError();
}

cudaError_t launch_row_keys(const int64_t* rows, uint64_t nrows, uint64_t n_src, const uint32_t* inv, uint64_t* keys,
                            uint32_t* idx, int* bad_flag, cudaStream_t st) {
    const int block = 256;
    row_keys_kernel<<<grid_for(nrows, block), block, 0, st>>>(rows, nrows, n_src, inv, reinterpret_cast<unsigned long long*>(keys),
                                                              idx, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_gather(const double4* src64, const uint64_t* pos, uint64_t nrows, uint64_t nrows_pad, double4* dst64,
                          cudaStream_t st) {
    const int block = 256;
    gather_kernel<<<grid_for(nrows_pad, block), block, 0, st>>>(src64, reinterpret_cast<const unsigned long long*>(pos), nrows,
                                                                nrows_pad, dst64);
    return cudaGetLastError();
}

cudaError_t launch_pairs_fast(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info, bool lookup_heavy) {
    const size_t smem = fast_smem_layout(p.ncells, p.nbands, p.nbins).total;
    auto kern = lookup_heavy ? ((map == CellMap::LogBits) ? pair_fast_kernel<(int)CellMap::LogBits, 3> : pair_fast_kernel<(int)CellMap::SqrtLin, 3>)
                             : ((map == CellMap::LogBits) ? pair_fast_kernel<(int)CellMap::LogBits, 2> : pair_fast_kernel<(int)CellMap::SqrtLin, 2>);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    // persistent CTAs: a whole number of CTAs per SM, never more than there are work items
    int grid = (int)std::min<uint64_t>((uint64_t)sm_count * per_sm, std::max<uint64_t>((uint64_t)p.n_items_part * p.jsplit, 1));
    kern<<<grid, kThreads, smem, st>>>(p);
    if (info) *info = LaunchInfo{grid, kThreads, (int)smem, 1};
    return cudaGetLastError();
}

cudaError_t launch_pairs_tensor(const PairParams& p, CellMap map, int sm_count, cudaStream_t st, LaunchInfo* info) {
    const size_t smem = tc_smem_layout(p.ncells, p.nbands, p.nbins).total;
    auto kern = (map == CellMap::LogBits) ? pair_tensor_kernel<(int)CellMap::LogBits> : pair_tensor_kernel<(int)CellMap::SqrtLin>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    // cudaOccupancyMaxActiveBlocksPerMultiprocessor answers 1 for a kernel that allocates tensor memory, whatever it
    // allocates; the SM does co-schedule CTAs whose allocations fit (measured: 1, 2, 4 CTAs/SM -> 80, 44, 27 ms).  So
    // the resident CTAs per SM are worked out here from shared memory, registers and the 512 TMEM columns.
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    int dev = 0, smem_sm = 0, regs_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev);
    const int regs_cta = ((fa.numRegs + 7) / 8 * 8) * kTcThreads;
    int per_sm = std::min<int>(smem_sm / (int)(smem + fa.sharedSizeBytes + 1024), regs_sm / std::max(regs_cta, 1));
    per_sm = std::min(per_sm, (int)(512 / kTcCols));
    // fine binnings (thousands of lookup cells: config 5) leave room for fewer than 3 such CTAs per SM, i.e. too few
    // warps to hide the step-by-step MMA pipeline: those run the FFMA2 kernel
    if (per_sm < 3) return launch_pairs_fast(p, map, sm_count, st, info, false);
    const uint64_t citems = (uint64_t)p.n_items_part * (kTileI / kTcThreads) * p.jsplit;
    int grid = (int)std::min<uint64_t>((uint64_t)sm_count * per_sm, std::max<uint64_t>(citems, 1));
    kern<<<grid, kTcThreads, smem, st>>>(p);
    if (info) *info = LaunchInfo{grid, kTcThreads, (int)smem, 1};
    return cudaGetLastError();
}

cudaError_t launch_sample_modes(const PairParams& p, CellMap map, uint32_t nsamples, unsigned long long* out, cudaStream_t st) {
    const int block = 256, grid = (int)((nsamples + block - 1) / block);
    if (map == CellMap::LogBits)
        sample_modes_kernel<(int)CellMap::LogBits><<<grid, block, 0, st>>>(p, nsamples, out);
    else
        sample_modes_kernel<(int)CellMap::SqrtLin><<<grid, block, 0, st>>>(p, nsamples, out);
    return cudaGetLastError();
}

cudaError_t launch_tensor_probe(const float4* srows, const float4* brows, float* q, uint32_t ntiles, cudaStream_t st) {
    tensor_probe_kernel<<<ntiles, kTcThreads, 0, st>>>(srows, brows, q);
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

cudaError_t launch_pairs_weighted64(const PairParams& p, const double* wi, const double* wj, double* wresult, int sm_count, cudaStream_t st) {
    const size_t smem = (size_t)(p.nbins + 1) * 8 + (size_t)(p.nbins + 3) * 8;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pair_weighted64_kernel, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    const int grid = (int)std::min<uint64_t>((uint64_t)sm_count * per_sm, std::max<uint32_t>(p.n_items_part, 1));
    pair_weighted64_kernel<<<grid, kThreads, smem, st>>>(p, wi, wj, wresult);
    return cudaGetLastError();
}

cudaError_t launch_scatter_weights(const double* w, const uint32_t* inv, uint64_t n, uint64_t n_pad, double* out, cudaStream_t st) {
    const int block = 256;
    scatter_weights_kernel<<<grid_for(n_pad, block), block, 0, st>>>(w, inv, n, n_pad, out);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const unsigned long long* result, int nbins, int zero_slot, unsigned long long self_pairs,
                            unsigned long long* out, cudaStream_t st) {
    finalize_kernel<<<1, 256, 0, st>>>(result, nbins, zero_slot, self_pairs, out);
    return cudaGetLastError();
}

}  // namespace tpcf
