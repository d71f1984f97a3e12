// api.cu -- the C ABI of libtpcf (include/tpcf.h): context, argument checking, device memory, launches.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/tpcf.h"
#include "kernels.cuh"
#include "tables.h"

using namespace tpcf;

namespace {
struct Catalog {                 // rows in Hilbert order (counts are order-invariant, reading A16)
    uint64_t n = 0, n_pad = 0;
    double4* x64 = nullptr;
    uint32_t* inv = nullptr;     // caller row -> position in the sorted catalog (row-subset mode)
    float4 *xq = nullptr, *cq = nullptr;   // i-side role: rows as offsets from their 8-row group ("quad") centre; (centre, radius)
    float4 *xs = nullptr, *cs = nullptr;   // j-side role: rows as (-2 offset, |offset|^2) from their 64-row subtile centre
    float4 *xt = nullptr, *ct = nullptr;   // j-side role of the tensor engine: the same for 128-row tiles
    float* xb = nullptr;                   // ... and per tile a 128 x 16 TF32 operand block (kernels.cuh)
    double* w64 = nullptr;                 // per-object weights in sorted order, n_pad entries, 0 for padding (tpcf_set_weights)
};
// scratch of one spatial sort: (key, idx) ping-pong buffers and the digit counts
struct SortScratch {
    uint64_t *ka = nullptr, *kb = nullptr;
    uint32_t *ia = nullptr, *ib = nullptr, *counts = nullptr;
    void release() {
        cudaFree(ka); cudaFree(kb); cudaFree(ia); cudaFree(ib); cudaFree(counts);
        *this = SortScratch();
    }
};
constexpr int kNumKinds = 5;                    // DD, DR, RR, D1D2, D2R
constexpr float kTensorMaxSlowShare = 0.025f;   // above this share of pair-by-pair blocks TPCF_ENGINE_TENSOR launches pair_fast_kernel
struct PlanCache {
    bool valid = false;
    float share = -1.f;          // sampled share of (group, tile) blocks the tensor kernel would count pair by pair; < 0: not sampled yet
    Plan plan;
    uint32_t* d_row_start = nullptr;
};
}  // namespace

struct tpcf_ctx {
    Binning bin;
    FastTables ft;
    double guard_scale = 1.0;
    bool tables_dirty = true;
    tpcf_engine engine = TPCF_ENGINE_TENSOR;
    bool window = true;
    bool prune = false;
    float tensor_share_limit = kTensorMaxSlowShare;
    cudaStream_t stream = nullptr;
    int part = 0, nparts = 1;
    Catalog cat[3];              // D, R, D2
    PlanCache plans[kNumKinds];
    // device side
    bool cuda_ready = false;
    int sm_count = kPlanSMs;    // replaced by cudaDevAttrMultiProcessorCount of the context's device at its first GPU call
    int device = -1;            // the device the context is bound to (ensure_cuda)
    float* d_lut = nullptr;
    int lut_multi = 0;
    uint16_t* d_slotmap = nullptr;
    float2 *d_band_mh = nullptr, *d_band_lh = nullptr;
    uint16_t *d_band_slot = nullptr, *d_cell_band = nullptr;
    double* d_thr = nullptr;
    // one set per kind: tpcf_count_all_async has the three pair kernels in flight together
    unsigned long long* d_result3 = nullptr;    // kNumKinds x (nbins + 3)
    unsigned long long* d_counters3 = nullptr;  // kNumKinds x kNumCounters
    unsigned long long* d_out3 = nullptr;       // kNumKinds x (nbins + 2)
    double* d_wresult = nullptr;                // nbins + 3 weighted sums (tpcf_count_weighted)
    cudaStream_t side[2] = {nullptr, nullptr};  // streams of the second and third count of tpcf_count_all_async
    cudaEvent_t fork = nullptr, join[2] = {nullptr, nullptr};
    int* d_bad = nullptr;
    void* arena = nullptr;                      // scratch of tpcf_load, grown on demand, kept until destroy
    size_t arena_bytes = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool time_kernels = false;
    int warp_items_per_item = 1;                // how the pair kernel that ran counts work items (pair_fast_kernel: per warp)
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> kev_pool, kev_used;
    // stored full counts for tpcf_estimate
    std::vector<uint64_t> counts[kNumKinds];
    bool have[kNumKinds] = {false, false, false, false, false};
    tpcf_stats stats{};
    std::string err;
};

namespace {

tpcf_status fail(tpcf_ctx* c, tpcf_status s, const std::string& msg) {
    if (c) c->err = msg;
    return s;
}
tpcf_status cuda_fail(tpcf_ctx* c, cudaError_t e, const char* what) {
    return fail(c, e == cudaErrorMemoryAllocation ? TPCF_ENOMEM : TPCF_ECUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call, what)                                       \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, what); \
    } while (0)

// No CPU fallback: without a usable GPU every compute entry point fails with TPCF_ECUDA.
tpcf_status ensure_cuda(tpcf_ctx* ctx) {
    if (ctx->cuda_ready) {
        // the context lives on the device that was current at its first GPU call: make it current again for this call
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess || cur != ctx->device) CU(cudaSetDevice(ctx->device), "cudaSetDevice");
        return TPCF_OK;
    }
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n < 1) {
        cudaGetLastError();
        return fail(ctx, TPCF_ECUDA, std::string("no usable CUDA device: ") + (e != cudaSuccess ? cudaGetErrorString(e) : "device count is 0"));
    }
    int dev = 0;
    CU(cudaGetDevice(&dev), "cudaGetDevice");
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, dev), "cudaGetDeviceProperties");
    if (prop.major < 10) return fail(ctx, TPCF_ECUDA, "libtpcf is built for sm_100a (B200) only");
    ctx->sm_count = prop.multiProcessorCount;
    ctx->device = dev;
    const int nb = ctx->bin.nbins;
    CU(cudaMalloc(&ctx->d_thr, (nb + 1) * sizeof(double)), "cudaMalloc thresholds");
    CU(cudaMalloc(&ctx->d_result3, kNumKinds * (nb + 3) * sizeof(unsigned long long)), "cudaMalloc result");
    CU(cudaMalloc(&ctx->d_out3, kNumKinds * (nb + 2) * sizeof(unsigned long long)), "cudaMalloc out");
    CU(cudaMalloc(&ctx->d_counters3, kNumKinds * kNumCounters * sizeof(unsigned long long)), "cudaMalloc counters");
    for (int k = 0; k < 2; ++k) {
        CU(cudaStreamCreateWithFlags(&ctx->side[k], cudaStreamNonBlocking), "cudaStreamCreate");
        CU(cudaEventCreateWithFlags(&ctx->join[k], cudaEventDisableTiming), "cudaEventCreate");
    }
    CU(cudaEventCreateWithFlags(&ctx->fork, cudaEventDisableTiming), "cudaEventCreate");
    CU(cudaMalloc(&ctx->d_bad, sizeof(int)), "cudaMalloc flag");
    CU(cudaMalloc(&ctx->d_wresult, (nb + 3) * sizeof(double)), "cudaMalloc weighted result");
    CU(cudaMemcpy(ctx->d_thr, ctx->bin.thr.data(), (nb + 1) * sizeof(double), cudaMemcpyHostToDevice), "upload thresholds");
    CU(cudaEventCreate(&ctx->ev0), "cudaEventCreate");
    CU(cudaEventCreate(&ctx->ev1), "cudaEventCreate");
    ctx->cuda_ready = true;
    return TPCF_OK;
}

void rebuild_tables(tpcf_ctx* ctx) {
    for (auto& pc : ctx->plans) pc.share = -1.f;
    build_fast_tables(ctx->bin, ctx->guard_scale, ctx->engine == TPCF_ENGINE_TENSOR, ctx->ft);
    ctx->tables_dirty = true;
}

tpcf_status upload_tables(tpcf_ctx* ctx) {
    if (!ctx->tables_dirty && ctx->d_lut) return TPCF_OK;
    const FastTables& t = ctx->ft;
    cudaFree(ctx->d_lut);
    cudaFree(ctx->d_slotmap);
    cudaFree(ctx->d_band_mh);
    cudaFree(ctx->d_band_lh);
    cudaFree(ctx->d_band_slot);
    cudaFree(ctx->d_cell_band);
    ctx->d_lut = nullptr;
    ctx->d_band_mh = ctx->d_band_lh = nullptr;
    ctx->d_slotmap = ctx->d_band_slot = ctx->d_cell_band = nullptr;
    std::vector<uint16_t> sm(2 * (size_t)t.ncells);
    ctx->lut_multi = 0;
    for (int c = 0; c < t.ncells; ++c) {
        if (t.tcell[c] != t.tcell[c]) ctx->lut_multi = 1;
        sm[c] = t.slot0[c];
        sm[(size_t)t.ncells + c] = t.slot1[c];
    }
    CU(cudaMalloc(&ctx->d_lut, t.tcell.size() * sizeof(float)), "cudaMalloc lut");
    CU(cudaMalloc(&ctx->d_slotmap, sm.size() * sizeof(uint16_t)), "cudaMalloc slotmap");
    CU(cudaMemcpy(ctx->d_lut, t.tcell.data(), t.tcell.size() * sizeof(float), cudaMemcpyHostToDevice), "upload lut");
    CU(cudaMemcpy(ctx->d_slotmap, sm.data(), sm.size() * sizeof(uint16_t), cudaMemcpyHostToDevice), "upload slotmap");
    std::vector<float2> mh(t.nbands), lh(t.nbands);
    for (int b = 0; b < t.nbands; ++b) {
        mh[b] = make_float2(t.band_mid[b], t.band_half[b]);
        lh[b] = make_float2(t.band_lo[b], t.band_hi[b]);
    }
    CU(cudaMalloc(&ctx->d_band_mh, mh.size() * sizeof(float2)), "cudaMalloc bands");
    CU(cudaMalloc(&ctx->d_band_lh, lh.size() * sizeof(float2)), "cudaMalloc bands");
    CU(cudaMalloc(&ctx->d_band_slot, t.band_slot.size() * sizeof(uint16_t)), "cudaMalloc bands");
    CU(cudaMalloc(&ctx->d_cell_band, t.cell_band.size() * sizeof(uint16_t)), "cudaMalloc bands");
    CU(cudaMemcpy(ctx->d_band_mh, mh.data(), mh.size() * sizeof(float2), cudaMemcpyHostToDevice), "upload bands");
    CU(cudaMemcpy(ctx->d_band_lh, lh.data(), lh.size() * sizeof(float2), cudaMemcpyHostToDevice), "upload bands");
    CU(cudaMemcpy(ctx->d_band_slot, t.band_slot.data(), t.band_slot.size() * sizeof(uint16_t), cudaMemcpyHostToDevice), "upload bands");
    CU(cudaMemcpy(ctx->d_cell_band, t.cell_band.data(), t.cell_band.size() * sizeof(uint16_t), cudaMemcpyHostToDevice), "upload bands");
    ctx->tables_dirty = false;
    return TPCF_OK;
}

void free_catalog(Catalog& c) {
    cudaFree(c.x64);
    cudaFree(c.inv);
    cudaFree(c.xq);
    cudaFree(c.cq);
    cudaFree(c.xs);
    cudaFree(c.cs);
    cudaFree(c.xb);
    cudaFree(c.xt);
    cudaFree(c.ct);
    cudaFree(c.w64);
    c = Catalog();
}

tpcf_status alloc_sort_scratch(tpcf_ctx* ctx, SortScratch& sc, uint64_t n) {
    const uint64_t nblk = (n + kSortChunk - 1) / kSortChunk;
    CU(cudaMalloc(&sc.ka, n * sizeof(uint64_t)), "cudaMalloc sort keys");
    CU(cudaMalloc(&sc.kb, n * sizeof(uint64_t)), "cudaMalloc sort keys");
    CU(cudaMalloc(&sc.ia, n * sizeof(uint32_t)), "cudaMalloc sort index");
    CU(cudaMalloc(&sc.ib, n * sizeof(uint32_t)), "cudaMalloc sort index");
    CU(cudaMalloc(&sc.counts, 256 * nblk * sizeof(uint32_t)), "cudaMalloc sort counts");
    return TPCF_OK;
}

// One device block for the scratch of a load, reused by later loads (a load ends with a stream synchronize, so no
// work is in flight on it when the next one starts): no cudaMalloc / cudaFree on the steady-state path.
tpcf_status arena_reserve(tpcf_ctx* ctx, size_t bytes) {
    if (ctx->arena_bytes >= bytes) return TPCF_OK;
    cudaFree(ctx->arena);
    ctx->arena = nullptr;
    ctx->arena_bytes = 0;
    CU(cudaMalloc(&ctx->arena, bytes), "cudaMalloc load scratch");
    ctx->arena_bytes = bytes;
    return TPCF_OK;
}
struct Carver {
    char* base;
    size_t off = 0;
    template <typename T>
    T* take(size_t count) {
        T* p = reinterpret_cast<T*>(base + off);
        off += (count * sizeof(T) + 255) & ~size_t(255);
        return p;
    }
};

uint64_t pad_to(uint64_t n, uint64_t m) { return (n + m - 1) / m * m; }

struct Sides {
    int ci, cj;      // catalog indices of the i-side and the j-side
    bool tri;
};
Sides sides_of(tpcf_kind k) {
    switch (k) {
        case TPCF_DD: return {0, 0, true};
        case TPCF_RR: return {1, 1, true};
        case TPCF_D1D2: return {0, 2, false};
        case TPCF_D2R: return {2, 1, false};
        default: return {0, 1, false};
    }
}

// SM count the plan's chunking balances for.  Under a partition (tpcf_set_partition) every rank must number the
// same items, whatever GPU it runs on: the chunking then uses the constant kPlanSMs; the device's own SM count only
// sizes the grid and the j-split of a launch.
int plan_sms(const tpcf_ctx* ctx) { return ctx->nparts > 1 ? kPlanSMs : ctx->sm_count; }

uint32_t items_of_part(uint64_t n_items, int part, int nparts) {
    if ((uint64_t)part >= n_items) return 0;
    return (uint32_t)((n_items - part + nparts - 1) / nparts);
}

// Enqueue one count on stream st (nullptr entry: ctx->stream); the nbins+2 result lands in out_dev.  rows_host == nullptr: full count.
tpcf_status enqueue_count(tpcf_ctx* ctx, tpcf_kind kind, const int64_t* rows_host, size_t nrows, unsigned long long* out_dev,
                          Catalog* tmp, int64_t** tmp_rows, uint64_t* pairs_out, cudaStream_t* on_stream = nullptr) {
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    if ((int)kind < 0 || (int)kind >= kNumKinds) return fail(ctx, TPCF_EINVAL, "unknown kind");
    const Sides sd = sides_of(kind);
    const Catalog& ci = ctx->cat[sd.ci];
    const Catalog& cj = ctx->cat[sd.cj];
    if (!ci.n || !cj.n) return fail(ctx, TPCF_ESTATE, "count before the needed catalog(s) were loaded");
    if (ctx->engine != TPCF_ENGINE_EXACT64) {
        s = upload_tables(ctx);
        if (s) return s;
    }
    cudaStream_t st = on_stream ? *on_stream : ctx->stream;
    const int nb = ctx->bin.nbins;
    unsigned long long* d_result = ctx->d_result3 + (size_t)kind * (nb + 3);
    unsigned long long* d_counters = ctx->d_counters3 + (size_t)kind * kNumCounters;

    PairParams p{};
    Plan subset_plan;
    const Plan* plan = nullptr;
    const uint32_t* d_row_start = nullptr;
    unsigned long long self_pairs = 0;
    if (rows_host) {
        // row-subset mode: gather the rows into a temporary i-side catalog, count the rectangle against all j
        if (nrows == 0) return fail(ctx, TPCF_EINVAL, "nrows == 0 with rows != NULL");
        if (nrows > 0x7FFFFFFFull) return fail(ctx, TPCF_EINVAL, "more than 2^31-1 rows");
        const uint64_t np = pad_to(nrows, kTileI);
        CU(cudaMalloc(tmp_rows, nrows * sizeof(int64_t)), "cudaMalloc rows");
        CU(cudaMalloc(&tmp->x64, np * sizeof(double4)), "cudaMalloc subset");
        CU(cudaMalloc(&tmp->xq, np * sizeof(float4)), "cudaMalloc subset");
        CU(cudaMalloc(&tmp->cq, np / kIPerThread * sizeof(float4)), "cudaMalloc subset");
        SortScratch sc;
        tpcf_status ss = alloc_sort_scratch(ctx, sc, nrows);
        if (ss) { sc.release(); return ss; }
        // the listed rows, ordered by their position in the sorted catalog (the order of the i-rows does not
        // change a sum over them; it keeps consecutive i-rows close on the sky for the window path)
        cudaError_t e = cudaMemcpyAsync(*tmp_rows, rows_host, nrows * sizeof(int64_t), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(ctx->d_bad, 0, sizeof(int), st);
        if (e == cudaSuccess) e = launch_row_keys(*tmp_rows, nrows, ci.n, ci.inv, sc.ka, sc.ia, ctx->d_bad, st);
        bool in_a = true;
        if (e == cudaSuccess) e = launch_sort_pairs(sc.ka, sc.kb, sc.ia, sc.ib, sc.counts, (uint32_t)nrows, 32, st, &in_a);
        if (e == cudaSuccess) e = launch_gather(ci.x64, in_a ? sc.ka : sc.kb, nrows, np, tmp->x64, st);
        if (e == cudaSuccess) e = launch_quads(tmp->x64, np, tmp->xq, tmp->cq, st);
        int bad = 0;
        if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, ctx->d_bad, sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        sc.release();
        if (e != cudaSuccess) return cuda_fail(ctx, e, "gather subset rows");
        if (bad) return fail(ctx, TPCF_EINVAL, "row index out of range");
        make_plan(false, nrows, cj.n, plan_sms(ctx), subset_plan);
        plan = &subset_plan;
        p.xq = tmp->xq;
        p.cq = tmp->cq;
        p.xi64 = tmp->x64;
        p.n_i = (uint32_t)nrows;
        p.tri = 0;
        if (sd.tri) self_pairs = nrows;      // each listed row meets itself once at theta = 0: remove it
        ctx->stats.launches = 1;
    } else {
        PlanCache& pc = ctx->plans[kind];
        if (!pc.valid) {
            make_plan(sd.tri, ci.n, cj.n, plan_sms(ctx), pc.plan);
            if (pc.d_row_start) cudaFree(pc.d_row_start);
            pc.d_row_start = nullptr;
            if (sd.tri) {
                CU(cudaMalloc(&pc.d_row_start, pc.plan.row_start.size() * sizeof(uint32_t)), "cudaMalloc plan");
                CU(cudaMemcpy(pc.d_row_start, pc.plan.row_start.data(), pc.plan.row_start.size() * sizeof(uint32_t),
                              cudaMemcpyHostToDevice), "upload plan");
            }
            pc.valid = true;
        }
        plan = &pc.plan;
        d_row_start = pc.d_row_start;
        p.xq = ci.xq;
        p.cq = ci.cq;
        p.xi64 = ci.x64;
        p.n_i = (uint32_t)ci.n;
        p.tri = sd.tri ? 1 : 0;
        ctx->stats.launches = 0;
    }
    p.xs = cj.xs;
    p.cs = cj.cs;
    p.xb = cj.xb;
    p.xt = cj.xt;
    p.ct = cj.ct;
    p.xj64 = cj.x64;
    p.n_j = (uint32_t)cj.n;
    p.blocks_i = plan->blocks_i;
    p.tiles_j = plan->tiles_j;
    p.chunk = plan->chunk;
    if (plan->n_items > 0xFFFFFFFFull) return fail(ctx, TPCF_EINVAL, "catalogs too large for the 32-bit work-item index");
    p.n_items_part = items_of_part(plan->n_items, ctx->part, ctx->nparts);
    p.row_start = d_row_start;
    // small catalogs: split the j-tile of every warp item until each resident warp gets ~32 of them
    p.jsplit = 1;
    while (p.chunk == 1 && p.jsplit < (uint32_t)(kTileJ / kChunkJ) &&
           (uint64_t)p.n_items_part * kWarpsPerCta * p.jsplit < 32ull * (uint64_t)ctx->sm_count * 2 * kWarpsPerCta)
        p.jsplit *= 2;
    p.part = (uint32_t)ctx->part;
    p.nparts = (uint32_t)ctx->nparts;
    p.lut = ctx->d_lut;
    p.slotmap = ctx->d_slotmap;
    p.window = (ctx->window && ctx->ft.nbands >= 1) ? 1 : 0;
    p.prune = (ctx->prune && p.window) ? 1 : 0;
    p.band_mh = ctx->d_band_mh;
    p.band_lh = ctx->d_band_lh;
    p.band_slot = ctx->d_band_slot;
    p.cell_band = ctx->d_cell_band;
    p.nbands = ctx->ft.nbands;
    p.ncells = ctx->ft.ncells;
    p.shift = ctx->ft.shift;
    p.sqrt_scale = ctx->ft.sqrt_scale;
    p.sqrt_clamp = ctx->ft.sqrt_clamp;
    p.guard_scale = (float)ctx->guard_scale;
    p.lut_multi = ctx->lut_multi;
    p.thr = ctx->d_thr;
    p.nbins = nb;
    p.result = d_result;
    p.counters = d_counters;

    CU(cudaMemsetAsync(d_result, 0, (nb + 3) * sizeof(unsigned long long), st), "memset result");
    CU(cudaMemsetAsync(d_counters, 0, kNumCounters * sizeof(unsigned long long), st), "memset counters");
    LaunchInfo li{};
    std::pair<cudaEvent_t, cudaEvent_t> kev{nullptr, nullptr};
    if (ctx->time_kernels && ctx->kev_used.size() < 64) {
        if (ctx->kev_pool.empty()) {
            CU(cudaEventCreate(&kev.first), "cudaEventCreate");
            CU(cudaEventCreate(&kev.second), "cudaEventCreate");
        } else {
            kev = ctx->kev_pool.back();
            ctx->kev_pool.pop_back();
        }
        CU(cudaEventRecord(kev.first, st), "cudaEventRecord");
    }
    {
        // TPCF_ENGINE_TENSOR runs the FFMA2 kernel where too many pairs would take the tensor kernel's pair-by-pair rows
        // (fine binnings, catalogs whose tiles are large against the scales binned): the share of such (8-row group, 128-row
        // tile) blocks is SAMPLED once per (kind, catalogs, tables) and kept with the plan
        bool tensor_kernel = ctx->engine == TPCF_ENGINE_TENSOR && !p.prune;      // pruning lives in the FFMA2 kernel
        bool lookup_heavy = false;
        if (ctx->engine != TPCF_ENGINE_EXACT64) {
            float share = -1.f;
            PlanCache* pc = rows_host ? nullptr : &ctx->plans[kind];
            if (pc && pc->share >= 0.f) share = pc->share;
            if (share < 0.f) {
                unsigned long long h[2] = {0, 0};
                CU(cudaMemsetAsync(d_counters, 0, 2 * sizeof(unsigned long long), st), "memset counters");
                CU(launch_sample_modes(p, ctx->ft.map, 1u << 16, d_counters, st), "sample_modes_kernel launch");
                CU(cudaMemcpyAsync(h, d_counters, sizeof(h), cudaMemcpyDeviceToHost, st), "copy sample");
                CU(cudaStreamSynchronize(st), "sample block modes");
                CU(cudaMemsetAsync(d_counters, 0, kNumCounters * sizeof(unsigned long long), st), "memset counters");
                share = h[1] ? (float)((double)h[0] / (double)h[1]) : 0.f;
                if (pc) pc->share = share;
            }
            ctx->stats.lookup_share = share;
            // ... unless the catalogs are so small that pair_fast_kernel's 2048-row plan items cannot fill the GPU: the
            // tensor kernel's CTAs take 128 rows each (config 1: 48 CTAs against 512)
            const bool tiny = (uint64_t)p.n_items_part * p.jsplit < 2ull * (uint64_t)ctx->sm_count && ctx->tensor_share_limit > 0.f;
            tensor_kernel = tensor_kernel && (share <= ctx->tensor_share_limit || tiny);
            lookup_heavy = share >= 0.8f && !p.prune;       // the FFMA2 kernel's variant for 3 CTAs per SM (kernels.cu)
        }
        if (ctx->engine == TPCF_ENGINE_EXACT64) p.prune = 0;
        const cudaError_t le = ctx->engine == TPCF_ENGINE_FAST || (ctx->engine == TPCF_ENGINE_TENSOR && !tensor_kernel)
                                   ? launch_pairs_fast(p, ctx->ft.map, ctx->sm_count, st, &li, lookup_heavy)
                               : ctx->engine == TPCF_ENGINE_TENSOR ? launch_pairs_tensor(p, ctx->ft.map, ctx->sm_count, st, &li)
                                                                   : launch_pairs_exact64(p, ctx->sm_count, st, &li);
        if (le != cudaSuccess) {
            if (kev.first) ctx->kev_pool.push_back(kev);        // the event pair goes back to the pool
            return cuda_fail(ctx, le, "pair kernel launch");
        }
    }
    if (kev.first) {
        CU(cudaEventRecord(kev.second, st), "cudaEventRecord");
        ctx->kev_used.push_back(kev);
    }
    const int zero_slot = (ctx->bin.thr[0] > 0.0) ? 0 : 1;
    CU(launch_finalize(d_result, nb, zero_slot, self_pairs, out_dev, st), "finalize launch");
    ctx->stats.launches += 2;
    ctx->stats.grid = li.grid;
    ctx->stats.block = li.block;
    ctx->warp_items_per_item = (li.block == kThreads && ctx->engine != TPCF_ENGINE_EXACT64) ? kWarpsPerCta : 1;
    ctx->stats.smem_bytes = li.smem_bytes;
    ctx->stats.cells = ctx->ft.ncells;
    ctx->stats.cell_bits = (ctx->ft.map == CellMap::LogBits) ? 23 - ctx->ft.shift : -1;
    if (pairs_out) {
        uint64_t pairs = 0;
        if (ctx->nparts == 1) {
            pairs = plan->tri ? plan->n_i * (plan->n_i - 1) / 2 : plan->n_i * plan->n_j;
        } else {
            for (uint64_t w = ctx->part; w < plan->n_items; w += ctx->nparts) pairs += plan->item_pairs(w);
        }
        *pairs_out = pairs - self_pairs;
    }
    return TPCF_OK;
}

}  // namespace

extern "C" {

tpcf_status tpcf_create(tpcf_ctx** out, int nbins, const double* theta_deg, tpcf_binning mode) {
    if (!out) return TPCF_EINVAL;
    *out = nullptr;
    tpcf_ctx* ctx = new (std::nothrow) tpcf_ctx();
    if (!ctx) return TPCF_ENOMEM;
    std::string why;
    try {
        why = make_binning(nbins, theta_deg, (int)mode, ctx->bin);
        if (why.empty()) rebuild_tables(ctx);
    } catch (const std::bad_alloc&) {
        delete ctx;
        return TPCF_ENOMEM;
    }
    if (!why.empty()) {
        delete ctx;
        return TPCF_EINVAL;
    }
    *out = ctx;
    return TPCF_OK;
}

tpcf_status tpcf_create_r(tpcf_ctx** out, int nbins, const double* r_edges, tpcf_binning mode, double max_abs_coord) {
    if (!out) return TPCF_EINVAL;
    *out = nullptr;
    tpcf_ctx* ctx = new (std::nothrow) tpcf_ctx();
    if (!ctx) return TPCF_ENOMEM;
    std::string why;
    try {
        why = make_binning_r(nbins, r_edges, (int)mode, max_abs_coord, ctx->bin);
        if (why.empty()) rebuild_tables(ctx);
    } catch (const std::bad_alloc&) {
        delete ctx;
        return TPCF_ENOMEM;
    }
    if (!why.empty()) {
        delete ctx;
        return TPCF_EINVAL;
    }
    *out = ctx;
    return TPCF_OK;
}

tpcf_status tpcf_get_edges(const tpcf_ctx* ctx, double* edges_out) {
    if (!ctx || !edges_out) return TPCF_EINVAL;
    std::memcpy(edges_out, ctx->bin.edges.data(), ctx->bin.edges.size() * sizeof(double));
    return TPCF_OK;
}

tpcf_status tpcf_get_thresholds(const tpcf_ctx* ctx, double* t_out) {
    if (!ctx || !t_out) return TPCF_EINVAL;
    std::memcpy(t_out, ctx->bin.thr.data(), ctx->bin.thr.size() * sizeof(double));
    return TPCF_OK;
}

static tpcf_status load_catalog(tpcf_ctx* ctx, tpcf_cat which, const void* radec_deg, tpcf_dtype dt, size_t n, int on_device,
                                void* cuda_stream, bool spatial) {
    if (!ctx) return TPCF_EINVAL;
    if (ctx->bin.spatial != spatial)
        return fail(ctx, TPCF_ESTATE, spatial ? "tpcf_load_xyz needs a context made by tpcf_create_r" : "tpcf_load needs a context made by tpcf_create");
    const int cols = spatial ? 3 : 2;       // values per row
    if (which != TPCF_D && which != TPCF_R && which != TPCF_D2) return fail(ctx, TPCF_EINVAL, "which must be TPCF_D, TPCF_R or TPCF_D2");
    if (dt != TPCF_F32 && dt != TPCF_F64) return fail(ctx, TPCF_EINVAL, "dtype must be TPCF_F32 or TPCF_F64");
    if (!radec_deg || n == 0) return fail(ctx, TPCF_EINVAL, "empty catalog");
    if (n > 0x7FFFFFFFull) return fail(ctx, TPCF_EINVAL, "more than 2^31-1 rows");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    cudaStream_t st = cuda_stream ? static_cast<cudaStream_t>(cuda_stream) : ctx->stream;
    Catalog& c = ctx->cat[which];
    // the arrays of the catalog being replaced may still be read by counts enqueued on the context's stream
    if (st != ctx->stream) CU(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    for (int k = 0; k < kNumKinds; ++k) {   // DR depends on both catalogs
        const Sides sd = sides_of((tpcf_kind)k);
        if (sd.ci == (int)which || sd.cj == (int)which) {
            ctx->have[k] = false;
            ctx->plans[k].valid = false;
            ctx->plans[k].share = -1.f;
        }
    }
    const uint64_t n_pad = pad_to(n, kTileI);
    const size_t esz = (dt == TPCF_F64) ? 8 : 4;
    if (c.w64) {                                // weights belong to the rows they were set for
        cudaFree(c.w64);
        c.w64 = nullptr;
    }
    if (c.x64 && c.n_pad == n_pad && c.n == n) {
        c.n = 0;                                // same shape as the catalog it replaces: keep the device arrays
    } else {
        free_catalog(c);
        CU(cudaMalloc(&c.x64, n_pad * sizeof(double4)), "cudaMalloc catalog (fp64)");
        CU(cudaMalloc(&c.inv, n * sizeof(uint32_t)), "cudaMalloc catalog (row map)");
        CU(cudaMalloc(&c.xq, n_pad * sizeof(float4)), "cudaMalloc catalog (quad offsets)");
        CU(cudaMalloc(&c.cq, n_pad / kIPerThread * sizeof(float4)), "cudaMalloc catalog (quad centres)");
        CU(cudaMalloc(&c.xs, n_pad * sizeof(float4)), "cudaMalloc catalog (subtile offsets)");
        CU(cudaMalloc(&c.cs, n_pad / kSubJ * sizeof(float4)), "cudaMalloc catalog (subtile centres)");
        CU(cudaMalloc(&c.xb, n_pad * kTcK * sizeof(float)), "cudaMalloc catalog (TF32 tiles)");
        CU(cudaMalloc(&c.xt, n_pad * sizeof(float4)), "cudaMalloc catalog (tile offsets)");
        CU(cudaMalloc(&c.ct, n_pad / kTcSubJ * sizeof(float4)), "cudaMalloc catalog (tile centres)");
    }
    const uint64_t nblk = (n + kSortChunk - 1) / kSortChunk;
    const size_t need = n * sizeof(double4) + 2 * n * sizeof(uint64_t) + 2 * n * sizeof(uint32_t) + 256 * nblk * sizeof(uint32_t) +
                        (on_device ? 0 : n * cols * esz) + 10 * 256;
    s = arena_reserve(ctx, need);
    if (s) { free_catalog(c); return s; }
    Carver cv{static_cast<char*>(ctx->arena)};
    double4* rows64 = cv.take<double4>(n);
    SortScratch sc;
    sc.ka = cv.take<uint64_t>(n);
    sc.kb = cv.take<uint64_t>(n);
    sc.ia = cv.take<uint32_t>(n);
    sc.ib = cv.take<uint32_t>(n);
    sc.counts = cv.take<uint32_t>(256 * nblk);
    uint64_t* bounds = cv.take<uint64_t>(32);
    cudaError_t e = cudaSuccess;
    const void* src = radec_deg;
    if (!on_device) {
        void* staged = cv.take<char>(n * cols * esz);
        e = cudaMemcpyAsync(staged, radec_deg, n * cols * esz, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { free_catalog(c); return cuda_fail(ctx, e, "copy catalog to device"); }
        src = staged;
    }
    // convert (fp64 unit vectors + sort keys) -> sort -> sorted fp64 rows + row map -> quad and subtile roles
    e = cudaMemsetAsync(ctx->d_bad, 0, sizeof(int), st);
    if (e == cudaSuccess)
        e = spatial ? launch_convert_xyz(src, dt == TPCF_F64, n, ctx->bin.scale, ctx->bin.max_abs, rows64, sc.ka, sc.ia, ctx->d_bad, bounds, st)
                    : launch_convert(src, dt == TPCF_F64, n, rows64, sc.ka, sc.ia, ctx->d_bad, bounds, st);
    bool in_a = true;
    if (e == cudaSuccess) e = launch_sort_pairs(sc.ka, sc.kb, sc.ia, sc.ib, sc.counts, (uint32_t)n, 63, st, &in_a);
    if (e == cudaSuccess) e = launch_permute(rows64, in_a ? sc.ia : sc.ib, n, n_pad, c.x64, c.inv, st);
    if (e == cudaSuccess) e = launch_quads(c.x64, n_pad, c.xq, c.cq, st);
    if (e == cudaSuccess) e = launch_subtiles(c.x64, n_pad, c.xs, c.cs, c.xt, c.ct, c.xb, st);
    int bad = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, ctx->d_bad, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        free_catalog(c);
        return cuda_fail(ctx, e, "convert catalog");
    }
    if (bad) {
        free_catalog(c);
        return fail(ctx, TPCF_EINVAL, spatial ? "catalog has a non-finite coordinate or one beyond max_abs_coord"
                                              : "catalog has a non-finite value, |RA| > 1e6 or |Dec| > 90");
    }
    c.n = n;
    c.n_pad = n_pad;
    return TPCF_OK;
}

tpcf_status tpcf_load(tpcf_ctx* ctx, tpcf_cat which, const void* radec_deg, tpcf_dtype dt, size_t n, int on_device,
                      void* cuda_stream) {
    return load_catalog(ctx, which, radec_deg, dt, n, on_device, cuda_stream, false);
}

tpcf_status tpcf_load_xyz(tpcf_ctx* ctx, tpcf_cat which, const void* xyz, tpcf_dtype dt, size_t n, int on_device, void* cuda_stream) {
    return load_catalog(ctx, which, xyz, dt, n, on_device, cuda_stream, true);
}

tpcf_status tpcf_count(tpcf_ctx* ctx, tpcf_kind kind, uint64_t* hist_out, uint64_t* under_over_out, const int64_t* rows,
                       size_t nrows) {
    if (!ctx) return TPCF_EINVAL;
    if (!hist_out) return fail(ctx, TPCF_EINVAL, "hist_out is NULL");
    if (!rows && nrows) return fail(ctx, TPCF_EINVAL, "nrows != 0 with rows == NULL");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    Catalog tmp;                 // row-subset mode: the listed rows as a temporary i-side catalog
    int64_t* tmp_rows = nullptr;
    uint64_t pairs = 0;
    cudaStream_t st = ctx->stream;
    const int nb = ctx->bin.nbins;
    std::vector<unsigned long long> host(nb + 2), ctr(kNumCounters);
    cudaError_t e = cudaEventRecord(ctx->ev0, st);
    unsigned long long* d_out = ctx->d_out3 + (size_t)kind * (nb + 2);
    s = (e == cudaSuccess) ? enqueue_count(ctx, kind, rows, nrows, d_out, &tmp, &tmp_rows, &pairs)
                           : cuda_fail(ctx, e, "cudaEventRecord");
    if (s == TPCF_OK) {
        e = cudaEventRecord(ctx->ev1, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), d_out, (nb + 2) * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(ctr.data(), ctx->d_counters3 + (size_t)kind * kNumCounters, kNumCounters * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) s = cuda_fail(ctx, e, "pair count");
    }
    free_catalog(tmp);
    if (tmp_rows) cudaFree(tmp_rows);
    if (s) return s;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
    ctx->stats.kernel_ms = ms;
    ctx->stats.pairs = pairs;
    ctx->stats.rechecked = ctr[1];
    // pair_fast_kernel (also when the tensor engine falls back to it) executes every plan item as kWarpsPerCta warp items
    ctx->stats.work_items = ctr[2] / ctx->warp_items_per_item;
    for (int k = 0; k < 6; ++k) ctx->stats.win_blocks[k] = ctr[3 + k];
    ctx->stats.pruned_blocks = ctr[9];
    for (int k = 0; k < nb; ++k) hist_out[k] = host[k + 1];
    if (under_over_out) {
        under_over_out[0] = host[0];
        under_over_out[1] = host[nb + 1];
    }
    if (!rows && ctx->nparts == 1) {
        ctx->counts[kind].assign(hist_out, hist_out + nb);
        ctx->have[kind] = true;
    }
    return TPCF_OK;
}

tpcf_status tpcf_count_async(tpcf_ctx* ctx, tpcf_kind kind, uint64_t* hist_dev) {
    if (!ctx) return TPCF_EINVAL;
    if (!hist_dev) return fail(ctx, TPCF_EINVAL, "hist_dev is NULL");
    return enqueue_count(ctx, kind, nullptr, 0, reinterpret_cast<unsigned long long*>(hist_dev), nullptr, nullptr, nullptr);
}

// DD, DR and RR of one w(theta) in flight together: DR (twice the pairs) on the context's stream, DD and RR on two side
// streams forked from it and joined back, so that the persistent grids of the three pair kernels fill each other's ramps
// and tails.  Results land in hist_dev[kind].
static tpcf_status enqueue_count_all(tpcf_ctx* ctx, unsigned long long* hist_dev, uint64_t* pairs_out /* 3, nullable */) {
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    const int nb = ctx->bin.nbins;
    cudaStream_t st = ctx->stream;
    const bool timing = ctx->time_kernels;
    std::pair<cudaEvent_t, cudaEvent_t> kev{nullptr, nullptr};
    if (timing && ctx->kev_used.size() < 64) {      // one event pair around the whole group, on the context's stream
        if (ctx->kev_pool.empty()) {
            CU(cudaEventCreate(&kev.first), "cudaEventCreate");
            CU(cudaEventCreate(&kev.second), "cudaEventCreate");
        } else {
            kev = ctx->kev_pool.back();
            ctx->kev_pool.pop_back();
        }
        CU(cudaEventRecord(kev.first, st), "cudaEventRecord");
    }
    ctx->time_kernels = false;              // restored below on every path
    {
        const cudaError_t e = cudaEventRecord(ctx->fork, st);
        if (e != cudaSuccess) s = cuda_fail(ctx, e, "cudaEventRecord");
    }
    const tpcf_kind order[3] = {TPCF_DR, TPCF_DD, TPCF_RR};
    for (int k = 0; k < 3 && s == TPCF_OK; ++k) {
        cudaStream_t on = k == 0 ? st : ctx->side[k - 1];
        if (k > 0) {
            cudaError_t e = cudaStreamWaitEvent(on, ctx->fork, 0);
            if (e != cudaSuccess) { s = cuda_fail(ctx, e, "cudaStreamWaitEvent"); break; }
        }
        s = enqueue_count(ctx, order[k], nullptr, 0, hist_dev + (size_t)order[k] * (nb + 2), nullptr, nullptr,
                          pairs_out ? pairs_out + order[k] : nullptr, &on);
        if (k > 0) {
            // a side stream that was forked is joined back whether or not its count could be enqueued: the context's stream
            // must never run ahead of work that reads the catalogs
            cudaError_t e = cudaEventRecord(ctx->join[k - 1], on);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ctx->join[k - 1], 0);
            if (e != cudaSuccess && s == TPCF_OK) s = cuda_fail(ctx, e, "join side stream");
        }
    }
    ctx->time_kernels = timing;
    if (kev.first) {
        if (s == TPCF_OK && cudaEventRecord(kev.second, st) == cudaSuccess)
            ctx->kev_used.push_back(kev);
        else
            ctx->kev_pool.push_back(kev);
    }
    return s;
}

tpcf_status tpcf_count_all_async(tpcf_ctx* ctx, uint64_t* hist_dev) {
    if (!ctx) return TPCF_EINVAL;
    if (!hist_dev) return fail(ctx, TPCF_EINVAL, "hist_dev is NULL");
    return enqueue_count_all(ctx, reinterpret_cast<unsigned long long*>(hist_dev), nullptr);
}

tpcf_status tpcf_count_all(tpcf_ctx* ctx, uint64_t* hist_out, uint64_t* under_over_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!hist_out) return fail(ctx, TPCF_EINVAL, "hist_out is NULL");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    const int nb = ctx->bin.nbins;
    std::vector<unsigned long long> host(3 * (size_t)(nb + 2));
    uint64_t pairs[3] = {0, 0, 0};
    cudaError_t e = cudaEventRecord(ctx->ev0, ctx->stream);
    s = (e == cudaSuccess) ? enqueue_count_all(ctx, ctx->d_out3, pairs) : cuda_fail(ctx, e, "cudaEventRecord");
    if (s) return s;
    e = cudaEventRecord(ctx->ev1, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), ctx->d_out3, host.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pair counts");
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
    ctx->stats.kernel_ms = ms;
    ctx->stats.pairs = pairs[0] + pairs[1] + pairs[2];
    for (int k = 0; k < 3; ++k) {
        const unsigned long long* h = host.data() + (size_t)k * (nb + 2);
        for (int b = 0; b < nb; ++b) hist_out[(size_t)k * nb + b] = h[b + 1];
        if (under_over_out) {
            under_over_out[2 * k] = h[0];
            under_over_out[2 * k + 1] = h[nb + 1];
        }
        if (ctx->nparts == 1) {
            ctx->counts[k].assign(hist_out + (size_t)k * nb, hist_out + (size_t)(k + 1) * nb);
            ctx->have[k] = true;
        }
    }
    return TPCF_OK;
}

tpcf_status tpcf_set_weights(tpcf_ctx* ctx, tpcf_cat which, const double* w, size_t n) {
    if (!ctx) return TPCF_EINVAL;
    if (which != TPCF_D && which != TPCF_R && which != TPCF_D2) return fail(ctx, TPCF_EINVAL, "which must be TPCF_D, TPCF_R or TPCF_D2");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    Catalog& c = ctx->cat[which];
    if (!c.n) return fail(ctx, TPCF_ESTATE, "tpcf_set_weights before the catalog was loaded");
    if (!w || n != c.n) return fail(ctx, TPCF_EINVAL, "weights must hold one value per row of the loaded catalog");
    for (size_t k = 0; k < n; ++k)
        if (!(std::fabs(w[k]) <= 1.0e150)) return fail(ctx, TPCF_EINVAL, "non-finite weight");
    cudaStream_t st = ctx->stream;
    // a failure below must not leave a weights array that tpcf_count_weighted would accept: the old one is dropped first
    // and the new one is attached to the catalog only when it is complete
    cudaFree(c.w64);
    c.w64 = nullptr;
    s = arena_reserve(ctx, n * sizeof(double));
    if (s) return s;
    double* w64 = nullptr;
    CU(cudaMalloc(&w64, c.n_pad * sizeof(double)), "cudaMalloc weights");
    double* staged = static_cast<double*>(ctx->arena);
    cudaError_t e = cudaMemcpyAsync(staged, w, n * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = launch_scatter_weights(staged, c.inv, n, c.n_pad, w64, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        cudaFree(w64);
        return cuda_fail(ctx, e, "set weights");
    }
    c.w64 = w64;
    return TPCF_OK;
}

tpcf_status tpcf_count_weighted(tpcf_ctx* ctx, tpcf_kind kind, double* wsum_out, double* under_over_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!wsum_out) return fail(ctx, TPCF_EINVAL, "wsum_out is NULL");
    if ((int)kind < 0 || (int)kind >= kNumKinds) return fail(ctx, TPCF_EINVAL, "unknown kind");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    const Sides sd = sides_of(kind);
    const Catalog& ci = ctx->cat[sd.ci];
    const Catalog& cj = ctx->cat[sd.cj];
    if (!ci.n || !cj.n) return fail(ctx, TPCF_ESTATE, "count before the needed catalog(s) were loaded");
    if (!ci.w64 || !cj.w64) return fail(ctx, TPCF_ESTATE, "tpcf_count_weighted needs tpcf_set_weights on the catalog(s) it pairs");
    cudaStream_t st = ctx->stream;
    const int nb = ctx->bin.nbins;
    Plan plan;
    make_plan(sd.tri, ci.n, cj.n, plan_sms(ctx), plan);
    if (plan.n_items > 0xFFFFFFFFull) return fail(ctx, TPCF_EINVAL, "catalogs too large for the 32-bit work-item index");
    uint32_t* d_row_start = nullptr;
    if (sd.tri) {
        CU(cudaMalloc(&d_row_start, plan.row_start.size() * sizeof(uint32_t)), "cudaMalloc plan");
        cudaError_t e = cudaMemcpy(d_row_start, plan.row_start.data(), plan.row_start.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { cudaFree(d_row_start); return cuda_fail(ctx, e, "upload plan"); }
    }
    PairParams p{};
    p.xi64 = ci.x64;
    p.xj64 = cj.x64;
    p.n_i = (uint32_t)ci.n;
    p.n_j = (uint32_t)cj.n;
    p.tri = sd.tri ? 1 : 0;
    p.blocks_i = plan.blocks_i;
    p.tiles_j = plan.tiles_j;
    p.chunk = plan.chunk;
    p.n_items_part = items_of_part(plan.n_items, ctx->part, ctx->nparts);
    p.row_start = d_row_start;
    p.part = (uint32_t)ctx->part;
    p.nparts = (uint32_t)ctx->nparts;
    p.thr = ctx->d_thr;
    p.nbins = nb;
    p.counters = ctx->d_counters3 + (size_t)kind * kNumCounters;
    std::vector<double> host(nb + 3);
    cudaError_t e = cudaMemsetAsync(ctx->d_wresult, 0, (nb + 3) * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(p.counters, 0, kNumCounters * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev0, st);
    if (e == cudaSuccess) e = launch_pairs_weighted64(p, ci.w64, cj.w64, ctx->d_wresult, ctx->sm_count, st);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev1, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), ctx->d_wresult, (nb + 3) * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_row_start);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "weighted pair sums");
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
    ctx->stats.kernel_ms = ms;
    for (int k = 0; k < nb; ++k) wsum_out[k] = host[k + 1];
    if (under_over_out) {
        under_over_out[0] = host[0];
        under_over_out[1] = host[nb + 1];
    }
    return TPCF_OK;
}

tpcf_status tpcf_count3(tpcf_ctx* ctx, tpcf_cat which, uint64_t* hist3_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!hist3_out) return fail(ctx, TPCF_EINVAL, "hist3_out is NULL");
    if (which != TPCF_D && which != TPCF_R && which != TPCF_D2) return fail(ctx, TPCF_EINVAL, "which must be TPCF_D, TPCF_R or TPCF_D2");
    const int nb = ctx->bin.nbins;
    if (nb > TPCF_COUNT3_MAX_BINS) return fail(ctx, TPCF_EINVAL, "tpcf_count3: more than TPCF_COUNT3_MAX_BINS (30) bins");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    const Catalog& c = ctx->cat[which];
    if (!c.n) return fail(ctx, TPCF_ESTATE, "tpcf_count3 before the catalog was loaded");
    if (c.n > (uint64_t)TPCF_COUNT3_MAX_ROWS) return fail(ctx, TPCF_EINVAL, "tpcf_count3: more than TPCF_COUNT3_MAX_ROWS (16384) rows");
    const size_t m = (size_t)nb + 2, cells = m * m * m;
    cudaStream_t st = ctx->stream;
    // scratch: the pair-slot matrix, the result cells and the row counter, carved from the context's arena (tpcf_load's scratch)
    const size_t sbytes = count3_slot_bytes(c.n);
    s = arena_reserve(ctx, sbytes + cells * sizeof(unsigned long long) + 3 * 256);
    if (s) return s;
    Carver cv{static_cast<char*>(ctx->arena)};
    uint8_t* slots = cv.take<uint8_t>(sbytes);
    unsigned long long* result3 = cv.take<unsigned long long>(cells);
    unsigned long long* next_row = cv.take<unsigned long long>(1);
    cudaError_t e = cudaMemsetAsync(result3, 0, cells * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(next_row, 0, sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev0, st);
    if (e == cudaSuccess) e = launch_count3(c.x64, (uint32_t)c.n, ctx->d_thr, nb, slots, next_row, result3, ctx->sm_count, st);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev1, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hist3_out, result3, cells * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "three-point counts");
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
    ctx->stats.kernel_ms = ms;
    ctx->stats.pairs = c.n * (c.n - 1) * (c.n - 2) / 6;      // triples, here
    ctx->stats.launches = 2;
    return TPCF_OK;
}

tpcf_status tpcf_estimate_cross(tpcf_ctx* ctx, double* w_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!w_out) return fail(ctx, TPCF_EINVAL, "w_out is NULL");
    if (!ctx->have[TPCF_D1D2] || !ctx->have[TPCF_DR] || !ctx->have[TPCF_D2R] || !ctx->have[TPCF_RR])
        return fail(ctx, TPCF_ESTATE, "the cross estimate needs full D1D2, DR, D2R and RR counts on the current catalogs");
    const double n1 = (double)ctx->cat[0].n, n2 = (double)ctx->cat[2].n, nr = (double)ctx->cat[1].n;
    const double n12 = n1 * n2, n1r = n1 * nr, n2r = n2 * nr, nrr = 0.5 * nr * (nr - 1.0);
    for (int k = 0; k < ctx->bin.nbins; ++k) {
        const double rr = (double)ctx->counts[TPCF_RR][k];
        if (rr == 0.0) { w_out[k] = std::nan(""); continue; }
        const double frr = rr / nrr;
        w_out[k] = ((double)ctx->counts[TPCF_D1D2][k] / n12 - (double)ctx->counts[TPCF_DR][k] / n1r -
                    (double)ctx->counts[TPCF_D2R][k] / n2r + frr) / frr;
    }
    return TPCF_OK;
}

tpcf_status tpcf_estimate_from(const uint64_t* dd, const uint64_t* dr, const uint64_t* rr, int nbins, uint64_t n_d,
                               uint64_t n_r, double* w_out) {
    if (!dd || !dr || !rr || !w_out || nbins < 1) return TPCF_EINVAL;
    estimate(dd, dr, rr, nbins, n_d, n_r, w_out);
    return TPCF_OK;
}

tpcf_status tpcf_estimate(tpcf_ctx* ctx, double* w_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!w_out) return fail(ctx, TPCF_EINVAL, "w_out is NULL");
    if (!ctx->have[TPCF_DD] || !ctx->have[TPCF_DR] || !ctx->have[TPCF_RR])
        return fail(ctx, TPCF_ESTATE, "estimate needs full DD, DR and RR counts on the current catalogs");
    estimate(ctx->counts[TPCF_DD].data(), ctx->counts[TPCF_DR].data(), ctx->counts[TPCF_RR].data(), ctx->bin.nbins,
             ctx->cat[0].n, ctx->cat[1].n, w_out);
    return TPCF_OK;
}

void tpcf_destroy(tpcf_ctx* ctx) {
    if (!ctx) return;
    if (ctx->cuda_ready) {
        cudaSetDevice(ctx->device);
        for (auto& c : ctx->cat) free_catalog(c);
        for (auto& pc : ctx->plans)
            if (pc.d_row_start) cudaFree(pc.d_row_start);
        cudaFree(ctx->d_lut);
        cudaFree(ctx->d_slotmap);
        cudaFree(ctx->d_band_mh);
        cudaFree(ctx->d_band_lh);
        cudaFree(ctx->d_band_slot);
        cudaFree(ctx->d_cell_band);
        cudaFree(ctx->d_thr);
        cudaFree(ctx->d_result3);
        cudaFree(ctx->d_out3);
        cudaFree(ctx->d_counters3);
        cudaFree(ctx->d_wresult);
        for (int k = 0; k < 2; ++k) {
            if (ctx->side[k]) cudaStreamDestroy(ctx->side[k]);
            if (ctx->join[k]) cudaEventDestroy(ctx->join[k]);
        }
        if (ctx->fork) cudaEventDestroy(ctx->fork);
        cudaFree(ctx->d_bad);
        cudaFree(ctx->arena);
        if (ctx->ev0) cudaEventDestroy(ctx->ev0);
        if (ctx->ev1) cudaEventDestroy(ctx->ev1);
        for (auto* v : {&ctx->kev_pool, &ctx->kev_used})
            for (auto& kv : *v) {
                cudaEventDestroy(kv.first);
                cudaEventDestroy(kv.second);
            }
    }
    delete ctx;
}

const char* tpcf_last_error(const tpcf_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

tpcf_status tpcf_set_stream(tpcf_ctx* ctx, void* cuda_stream) {
    if (!ctx) return TPCF_EINVAL;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return TPCF_OK;
}

tpcf_status tpcf_set_engine(tpcf_ctx* ctx, tpcf_engine e) {
    if (!ctx) return TPCF_EINVAL;
    if (e != TPCF_ENGINE_FAST && e != TPCF_ENGINE_EXACT64 && e != TPCF_ENGINE_TENSOR) return fail(ctx, TPCF_EINVAL, "unknown engine");
    const bool rebuild = (ctx->engine == TPCF_ENGINE_TENSOR) != (e == TPCF_ENGINE_TENSOR);
    ctx->engine = e;
    if (rebuild) rebuild_tables(ctx);       // the tensor engine's window bands are wider
    return TPCF_OK;
}

tpcf_status tpcf_set_window(tpcf_ctx* ctx, int enabled) {
    if (!ctx) return TPCF_EINVAL;
    ctx->window = enabled != 0;
    return TPCF_OK;
}

tpcf_status tpcf_set_tensor_share_limit(tpcf_ctx* ctx, double limit) {
    if (!ctx) return TPCF_EINVAL;
    if (!(limit >= 0.0) || !(limit <= 1.0)) return fail(ctx, TPCF_EINVAL, "the share limit must be in [0, 1]");
    ctx->tensor_share_limit = (float)limit;
    return TPCF_OK;
}

tpcf_status tpcf_set_pruning(tpcf_ctx* ctx, int enabled) {
    if (!ctx) return TPCF_EINVAL;
    ctx->prune = enabled != 0;
    return TPCF_OK;
}

tpcf_status tpcf_set_guard_scale(tpcf_ctx* ctx, double scale) {
    if (!ctx) return TPCF_EINVAL;
    if (!(scale > 0.0) || !(scale <= 1.0e6)) return fail(ctx, TPCF_EINVAL, "guard scale must be in (0, 1e6]");
    ctx->guard_scale = scale;
    rebuild_tables(ctx);
    return TPCF_OK;
}

tpcf_status tpcf_set_partition(tpcf_ctx* ctx, int part, int nparts) {
    if (!ctx) return TPCF_EINVAL;
    if (nparts < 1 || part < 0 || part >= nparts) return fail(ctx, TPCF_EINVAL, "need 0 <= part < nparts");
    if ((ctx->nparts > 1) != (nparts > 1))
        for (auto& pc : ctx->plans) pc.valid = false;       // the chunking differs between the two (plan_sms)
    ctx->part = part;
    ctx->nparts = nparts;
    return TPCF_OK;
}

tpcf_status tpcf_set_kernel_timing(tpcf_ctx* ctx, int enabled) {
    if (!ctx) return TPCF_EINVAL;
    ctx->time_kernels = enabled != 0;
    return TPCF_OK;
}

tpcf_status tpcf_get_kernel_times(tpcf_ctx* ctx, float* ms_out, int capacity, int* n_out) {
    if (!ctx || !n_out || (capacity > 0 && !ms_out)) return TPCF_EINVAL;
    int n = 0;
    for (auto& kv : ctx->kev_used) {
        CU(cudaEventSynchronize(kv.second), "cudaEventSynchronize");
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, kv.first, kv.second), "cudaEventElapsedTime");
        if (n < capacity) ms_out[n++] = ms;
        ctx->kev_pool.push_back(kv);
    }
    ctx->kev_used.clear();
    *n_out = n;
    return TPCF_OK;
}

tpcf_status tpcf_get_stats(const tpcf_ctx* ctx, tpcf_stats* out) {
    if (!ctx || !out) return TPCF_EINVAL;
    *out = ctx->stats;
    out->cells = ctx->ft.ncells;
    out->cell_bits = (ctx->ft.map == CellMap::LogBits) ? 23 - ctx->ft.shift : -1;
    return TPCF_OK;
}

tpcf_status tpcf_classify_fast(const tpcf_ctx* ctx, float d2, int* slot_out) {
    if (!ctx || !slot_out) return TPCF_EINVAL;
    if (!(d2 >= 0.0f) || !(d2 < 64.0f)) return TPCF_EINVAL;
    *slot_out = ctx->ft.classify(d2);
    return TPCF_OK;
}

tpcf_status tpcf_tensor_probe(tpcf_ctx* ctx, const float* s_rows, const float* b_rows, size_t ntiles, float* q_out) {
    if (!ctx) return TPCF_EINVAL;
    if (!s_rows || !b_rows || !q_out || ntiles == 0 || ntiles > 65535) return fail(ctx, TPCF_EINVAL, "tpcf_tensor_probe: bad argument");
    tpcf_status s = ensure_cuda(ctx);
    if (s) return s;
    const size_t rows = ntiles * 128;
    float4 *ds = nullptr, *db = nullptr;
    float* dq = nullptr;
    cudaError_t e = cudaMalloc(&ds, rows * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&db, rows * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&dq, rows * 128 * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpyAsync(ds, s_rows, rows * sizeof(float4), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(db, b_rows, rows * sizeof(float4), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = launch_tensor_probe(ds, db, dq, (uint32_t)ntiles, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(q_out, dq, rows * 128 * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(ds);
    cudaFree(db);
    cudaFree(dq);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "tpcf_tensor_probe");
    return TPCF_OK;
}

tpcf_status tpcf_window_host(const tpcf_ctx* ctx, float lo2, float hi2, int* first_band_out, int* n_edges_out) {
    if (!ctx || !first_band_out || !n_edges_out) return TPCF_EINVAL;
    if (!(lo2 >= 0.0f) || !(hi2 >= lo2) || !(hi2 < 64.0f)) return TPCF_EINVAL;
    ctx->ft.window(lo2, hi2, *first_band_out, *n_edges_out);
    return TPCF_OK;
}

tpcf_status tpcf_get_bands(const tpcf_ctx* ctx, int capacity, float* lo_out, float* hi_out, int* slot_below_out, int* n_out) {
    if (!ctx || !n_out) return TPCF_EINVAL;
    const FastTables& t = ctx->ft;
    *n_out = t.nbands;
    if (capacity < t.nbands) return (lo_out || hi_out || slot_below_out) ? TPCF_EINVAL : TPCF_OK;
    for (int b = 0; b < t.nbands; ++b) {
        if (lo_out) lo_out[b] = t.band_lo[b];
        if (hi_out) hi_out[b] = t.band_hi[b];
        if (slot_below_out) slot_below_out[b] = t.band_slot[b];
    }
    return TPCF_OK;
}

tpcf_status tpcf_plan(const tpcf_ctx* ctx, tpcf_kind kind, uint64_t n_d, uint64_t n_r, uint64_t* n_items_out) {
    if (!ctx || !n_items_out || n_d == 0 || n_r == 0) return TPCF_EINVAL;
    if ((int)kind < 0 || (int)kind > (int)TPCF_RR) return TPCF_EINVAL;      // the D2 kinds have a third size
    Plan p;
    const Sides sd = sides_of(kind);
    make_plan(sd.tri, sd.ci == 0 ? n_d : n_r, sd.cj == 0 ? n_d : n_r, plan_sms(ctx), p);
    *n_items_out = p.n_items;
    return TPCF_OK;
}

tpcf_status tpcf_plan_item_pairs(const tpcf_ctx* ctx, tpcf_kind kind, uint64_t n_d, uint64_t n_r, uint64_t w,
                                 uint64_t* pairs_out) {
    if (!ctx || !pairs_out || n_d == 0 || n_r == 0) return TPCF_EINVAL;
    if ((int)kind < 0 || (int)kind > (int)TPCF_RR) return TPCF_EINVAL;
    Plan p;
    const Sides sd = sides_of(kind);
    make_plan(sd.tri, sd.ci == 0 ? n_d : n_r, sd.cj == 0 ? n_d : n_r, plan_sms(ctx), p);
    if (w >= p.n_items) return TPCF_EINVAL;
    *pairs_out = p.item_pairs(w);
    return TPCF_OK;
}

}  // extern "C"
