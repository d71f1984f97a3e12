/*
 * tpcf.h -- C ABI of the B200-native pair-counting library (libtpcf.so).
 *
 * The library computes the hot path of the Landy-Szalay angular two-point correlation function of
 * arXiv:1204.6630: brute-force all-pairs angular pair counting of a data catalog D and a
 * random catalog R into the three theta-binned histograms DD, DR, RR (the definitions
 * under Eq. 1; Section 3 bullets 1-2: per pair a dot product and an arc-cosine, then a
 * histogram update with shared-memory atomics, partial histograms merged in global memory), and the
 * estimator of Eq. 1.  Every step runs in hand-written CUDA kernels for sm_100a; there
 * is no CPU fallback: every entry point that needs the GPU returns TPCF_ECUDA when none is usable.
 *
 * Conventions
 *   - All pointers are HOST pointers unless the argument says "device".  The caller owns every buffer
 *     it passes in; the library copies what it needs before returning and owns all of its own device
 *     memory through the opaque context.  No torch / C++ types cross this boundary.
 *   - Every function returns a tpcf_status and never throws or aborts; tpcf_last_error() gives a
 *     human-readable message for the last failure on that context.
 *   - Calls on one context must not be concurrent.  All calls are synchronous on return except the
 *     explicitly *_async one.
 *   - Bins (reading A5 in DESIGN.md; the paper does not state a convention): bin k = [e_k, e_{k+1}) in
 *     theta, the LAST bin closed at e_n (numpy.histogram's convention); under = theta < e_0,
 *     over = theta > e_n; always under + sum(bins) + over = number of pairs enumerated.
 *   - Pairs (reading A3): DD / RR enumerate the unordered pairs i<j of one catalog, N(N-1)/2 of them;
 *     DR enumerates all N_D*N_R ordered pairs (BASELINE.json north_star).
 */
#ifndef TPCF_H
#define TPCF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpcf_ctx tpcf_ctx;

typedef enum { TPCF_OK = 0, TPCF_EINVAL = 1, TPCF_ENOMEM = 2, TPCF_ECUDA = 3, TPCF_ESTATE = 4 } tpcf_status;
typedef enum { TPCF_LINEAR = 0, TPCF_LOG = 1, TPCF_EXPLICIT = 2 } tpcf_binning;
typedef enum { TPCF_D = 0, TPCF_R = 1, TPCF_D2 = 2 } tpcf_cat;     /* D2: a second data catalog (cross-correlations) */
typedef enum { TPCF_F32 = 0, TPCF_F64 = 1 } tpcf_dtype;
typedef enum { TPCF_DD = 0, TPCF_DR = 1, TPCF_RR = 2, TPCF_D1D2 = 3, TPCF_D2R = 4 } tpcf_kind;

/* Which kernel family tpcf_count uses (tpcf_set_engine).
 *   TPCF_ENGINE_TENSOR  (default) blocks of 128 i-rows x 128 j-rows; for every (8-row group, j-tile) block whose bounding
 *                       spheres leave at most 3 bin edges in reach, the window quantity q = |a-b|^2 - mid is formed by a
 *                       3xTF32 tcgen05.mma (fp32 accumulators in tensor memory, one i-row per thread) and every pair is
 *                       classified by 1..3 sign tests; a pair within the guard band of an edge (4.0e-6 T: 1.5 times the
 *                       proven bound 43.7 x 2^-24 T of DESIGN.md section 4, which rests on the measured, bit-exactly
 *                       reproduced accumulation model of tests/tc_model.py), near blocks and fine binnings go through the
 *                       fp32 cell lookup of TPCF_ENGINE_FAST and, inside its guard band, the fp64 recheck: the
 *                       histograms equal those of TPCF_ENGINE_EXACT64.  Launches in which more than a small share of the
 *                       blocks would take that pair-by-pair path (fine binnings such as config 5; the share is sampled,
 *                       see tpcf_set_tensor_share_limit) run TPCF_ENGINE_FAST's kernel instead.
 *   TPCF_ENGINE_FAST    the same windows with q formed by packed FP32 FMAs (FFMA2) on the CUDA cores, 8 i-rows per lane
 *                       against 64-row j-subtiles (guard band 3.0e-6 T, proven bound 29.1 x 2^-24 T); otherwise an O(1)
 *                       cell lookup against chord-space thresholds with privatised shared-memory histograms; every pair
 *                       inside a guard band is re-evaluated in fp64.  Same histograms.
 *   TPCF_ENGINE_EXACT64 plain fp64 kernel: fp64 squared chord against fp64 thresholds 4 sin^2(e_k/2) by
 *                       binary search.  Slow; kept as the device-side cross-check of the other two.
 */
typedef enum { TPCF_ENGINE_FAST = 0, TPCF_ENGINE_EXACT64 = 1, TPCF_ENGINE_TENSOR = 2 } tpcf_engine;

/*
 * tpcf_create -- fix the theta binning (the paper gives none; BASELINE.json configs do).
 *   nbins      >= 1 (and <= 4096).
 *   theta_deg  LINEAR / LOG: two doubles {min, max} in degrees, 0 <= min < max <= 180 (LOG: min > 0).
 *                LINEAR: e_k = min + k (max-min)/nbins.  LOG: e_k = min * (max/min)^(k/nbins).
 *                e_0 = min and e_n = max exactly.
 *              EXPLICIT: nbins+1 strictly increasing edges in [0, 180].
 *   Does not touch the GPU (thresholds and lookup tables are built on the host here and uploaded at the
 *   first count).  Errors: TPCF_EINVAL on any violated condition above or a NaN edge.
 */
tpcf_status tpcf_create(tpcf_ctx** out, int nbins, const double* theta_deg, tpcf_binning mode);

/* Copies the nbins+1 edges (degrees) the context uses, so a checker can bin with the very same values. */
tpcf_status tpcf_get_edges(const tpcf_ctx* ctx, double* edges_out /* nbins+1 */);

/*
 * tpcf_load -- load catalog D or R: n rows of (RA, Dec) in degrees, row-major n x 2, dtype F32 or F64
 *   ("input file lines").  The rows are copied to the device (or read in place
 *   when on_device != 0, in which case radec_deg is a device pointer) and converted ON THE DEVICE to unit
 *   vectors x = cos(dec)cos(ra), y = cos(dec)sin(ra), z = sin(dec) in fp64 (reading A8), sorted along a space-
 *   filling curve (counts do not depend on the order; `rows` of tpcf_count always index the caller's order) and
 *   stored a second time as fp32 offsets from the centres of small groups of consecutive rows (what the fast
 *   engine reads).  Replaces any previous catalog in that slot and invalidates stored
 *   counts that used it; device arrays are reused when the size is unchanged, so do not call it while a
 *   tpcf_count_async on another stream than cuda_stream / the context's stream is still reading them.
 *   cuda_stream: a cudaStream_t (or NULL for the context's stream) the copy and conversion are ordered on;
 *   the call returns after they completed.
 *   Errors: TPCF_EINVAL for n == 0, n > 2^31-1, |Dec| > 90, |RA| > 1e6 or a non-finite value in any row
 *   (checked on the device; RA is periodic, any value up to 1e6 degrees in magnitude is accepted); TPCF_ENOMEM; TPCF_ECUDA.
 *   The context is bound to the CUDA device that is current at its first GPU call; later calls make that device current.
 */
tpcf_status tpcf_load(tpcf_ctx* ctx, tpcf_cat which, const void* radec_deg, tpcf_dtype dt, size_t n, int on_device,
                      void* cuda_stream);

/*
 * tpcf_count -- one histogram.
 *   kind       TPCF_DD (pairs i<j of D), TPCF_RR (pairs i<j of R), TPCF_DR (all pairs D x R).
 *   hist_out   nbins uint64 counts (host).
 *   under_over_out  NULL, or 2 uint64: {pairs with theta < e_0, pairs with theta > e_n}.
 *   rows/nrows NULL/0 for the full count.  Otherwise ROW-SUBSET mode (validation of catalogs too large for
 *              a CPU oracle, BASELINE.json): rows are indices into D (for DD, DR) or R (for RR), and the
 *              call counts sum over i in rows of all j != i of the same catalog (DD, RR: nrows*(N-1) pairs,
 *              both sides of the diagonal) or of all j of R (DR: nrows*N_R pairs).  A subset count is not
 *              stored for tpcf_estimate.
 *   Errors: TPCF_ESTATE if a needed catalog is not loaded; TPCF_EINVAL for a row index out of range;
 *   TPCF_ECUDA.
 */
tpcf_status tpcf_count(tpcf_ctx* ctx, tpcf_kind kind, uint64_t* hist_out, uint64_t* under_over_out,
                       const int64_t* rows, size_t nrows);

/*
 * tpcf_count_async -- the same full count, without host synchronisation: enqueues the kernels on the
 *   context's stream (tpcf_set_stream) and writes nbins+2 uint64 {under, bin_0..bin_{n-1}, over} to the
 *   DEVICE buffer hist_dev when they complete.  The count is not stored for tpcf_estimate.  This is the
 *   entry point timed with CUDA events when the catalogs are already resident.
 *   One exception to "without host synchronisation": the FIRST count of a kind after tpcf_load, tpcf_set_engine or
 *   tpcf_set_guard_scale (engines other than EXACT64) samples the block mix that picks the kernel variant, reads two
 *   words back and waits for the stream once; it may also allocate (plan, tables).  Later calls on the same catalogs
 *   neither wait nor allocate.  The same holds for tpcf_count_all_async.
 */
tpcf_status tpcf_count_async(tpcf_ctx* ctx, tpcf_kind kind, uint64_t* hist_dev /* device, nbins+2 */);

/*
 * tpcf_count_all / tpcf_count_all_async -- the three full histograms of one w(theta) in one call: DD, DR and RR are put
 *   in flight together (DR on the context's stream, DD and RR on two internal streams forked from it and joined back), so
 *   that the persistent grids of the three pair kernels fill each other's ramp and tail instead of running back to back;
 *   the results are those of three tpcf_count calls.
 *   tpcf_count_all: hist_out = 3 x nbins uint64 (host) in the order DD, DR, RR; under_over_out = NULL or 3 x 2 uint64; the
 *   counts are stored for tpcf_estimate (unless a partition is set).  tpcf_count_all_async: hist_dev = 3 x (nbins+2)
 *   uint64 on the DEVICE, {under, bins, over} per kind in the same order, valid once the context's stream has passed the
 *   call; nothing is stored.  Errors as tpcf_count.
 */
tpcf_status tpcf_count_all(tpcf_ctx* ctx, uint64_t* hist_out /* 3 x nbins */, uint64_t* under_over_out /* 3 x 2, nullable */);
tpcf_status tpcf_count_all_async(tpcf_ctx* ctx, uint64_t* hist_dev /* device, 3 x (nbins+2) */);

/*
 * tpcf_estimate -- Landy-Szalay w(theta) in the pair-count-normalised form (Eq. 1, whose
 *   extraction lost the square on N_random/N_real; form fixed by BASELINE.json north_star, reading A1):
 *     w_k = (DD_k/nDD - 2 DR_k/nDR + RR_k/nRR) / (RR_k/nRR),
 *     nDD = N_D(N_D-1)/2, nDR = N_D N_R, nRR = N_R(N_R-1)/2;   RR_k = 0 gives NaN.
 *   Needs full (non-subset, non-partitioned) DD, DR and RR counted by tpcf_count on the current catalogs,
 *   else TPCF_ESTATE.
 */
tpcf_status tpcf_estimate(tpcf_ctx* ctx, double* w_out /* nbins */);

/* The same arithmetic on caller-supplied histograms (used after a multi-process reduction). */
tpcf_status tpcf_estimate_from(const uint64_t* dd, const uint64_t* dr, const uint64_t* rr, int nbins, uint64_t n_d,
                               uint64_t n_r, double* w_out /* nbins */);

/*
 * 3-D variant (Section 2: "our results are extendible to the 3-dimensional variant as well"): the same three
 * histograms DD, DR, RR over the Euclidean separation r = |a - b| of Cartesian positions, and the same estimator on
 * them (the spatial two-point function xi(r)).  Everything else -- tpcf_count, tpcf_count_async, tpcf_estimate, the
 * controls, row-subset mode -- is shared with the angular contexts.
 *
 * tpcf_create_r -- fix the separation binning: r_edges as theta_deg in tpcf_create (LINEAR / LOG: {min, max}, min >= 0,
 *   LOG: min > 0; EXPLICIT: nbins+1 strictly increasing values >= 0), in the units of the coordinates.  Bin k =
 *   [e_k, e_{k+1}) in r, last bin closed, under = r < e_0, over = r > e_n.
 *   max_abs_coord: a bound the caller guarantees for |x|, |y|, |z| of every row of both catalogs (> 0).  Positions are
 *   multiplied by the power of two that brings them inside the unit ball (exact in binary floating point) and bins are
 *   compared in squared separation, (e_k * scale)^2, so the fp64 engine's decision differs from sqrt(dx^2+dy^2+dz^2)
 *   against e_k only for pairs within fp64 rounding of an edge.  e_n may not exceed the largest separation the bound
 *   allows (2 / scale >= 2 sqrt(3) max_abs_coord): TPCF_EINVAL, as for any other violated condition.
 * tpcf_load_xyz -- load catalog D or R: n rows of (x, y, z), row-major n x 3, dtype F32 or F64, host or device memory
 *   as in tpcf_load.  The rows are sorted along a 3-D Hilbert curve and stored as fp32 offsets from group centres
 *   exactly as the angular rows are (DESIGN.md section 4 uses nothing of the unit sphere but d^2 <= 4).
 *   Errors: TPCF_ESTATE on a context made by tpcf_create (and tpcf_load on one made by tpcf_create_r); TPCF_EINVAL for
 *   n == 0, n > 2^31-1, a non-finite coordinate or one beyond max_abs_coord; TPCF_ENOMEM; TPCF_ECUDA.
 */
tpcf_status tpcf_create_r(tpcf_ctx** out, int nbins, const double* r_edges, tpcf_binning mode, double max_abs_coord);
tpcf_status tpcf_load_xyz(tpcf_ctx* ctx, tpcf_cat which, const void* xyz, tpcf_dtype dt, size_t n, int on_device,
                          void* cuda_stream);

/*
 * Cross-catalog and weighted counts (PAPER.md:16 cross-correlations of galaxy positions with other
 * quantities, PAPER.md:83, 89 extensions named as future work).
 *
 * A third catalog slot TPCF_D2 (tpcf_load / tpcf_load_xyz with which = TPCF_D2) and two more kinds for tpcf_count and
 * tpcf_count_async: TPCF_D1D2 = all N_D x N_D2 pairs of D with D2, TPCF_D2R = all N_D2 x N_R pairs (row subsets index
 * D for D1D2 and D2 for D2R).  The same kernels count them.
 * tpcf_estimate_cross -- the Landy-Szalay cross-correlation of D and D2 in the pair-count-normalised form,
 *     w12_k = (D1D2_k/(N_D N_D2) - DR_k/(N_D N_R) - D2R_k/(N_D2 N_R) + RR_k/nRR) / (RR_k/nRR);
 *   needs full D1D2, DR, D2R and RR counts by tpcf_count on the current catalogs, else TPCF_ESTATE.
 *
 * tpcf_set_weights -- one fp64 weight per row of a loaded catalog, in the caller's row order (n must equal the
 *   catalog's size; a later tpcf_load of that slot drops them).  Errors: TPCF_ESTATE before the load, TPCF_EINVAL for a
 *   wrong n or a non-finite weight.
 * tpcf_count_weighted -- per bin the sum over the pairs of `kind` of w_i * w_j (under_over_out: the two out-of-range
 *   sums), in fp64 throughout: fp64 separations against the fp64 thresholds (the bins are those of
 *   TPCF_ENGINE_EXACT64) and fp64 sums.  The order of the additions is not fixed (fp64 atomics), so a sum of m terms is
 *   reproducible only up to (m - 1) 2^-53 sum |w_i w_j|; partial sums hold at most 2^25 terms.
 *   A first, correct path on the fp64 kernel's plan: about 50 times slower than the unweighted counts.
 *   Errors: TPCF_ESTATE without catalogs or weights; TPCF_ECUDA.
 */
tpcf_status tpcf_estimate_cross(tpcf_ctx* ctx, double* w_out /* nbins */);
tpcf_status tpcf_set_weights(tpcf_ctx* ctx, tpcf_cat which, const double* w, size_t n);
tpcf_status tpcf_count_weighted(tpcf_ctx* ctx, tpcf_kind kind, double* wsum_out /* nbins */, double* under_over_out /* 2, nullable */);

void tpcf_destroy(tpcf_ctx* ctx);
const char* tpcf_last_error(const tpcf_ctx* ctx);

/* ---- controls ------------------------------------------------------------------------------------- */

/* Stream (a cudaStream_t) all later kernels of this context are launched on; NULL = legacy default. */
tpcf_status tpcf_set_stream(tpcf_ctx* ctx, void* cuda_stream);
tpcf_status tpcf_set_engine(tpcf_ctx* ctx, tpcf_engine e);
/* Multiplies the width of the fp32 guard band around each bin edge (default 1.0).  Any value >= 1 must
 * give identical histograms; the tests use 2.0 and 8.0 to demonstrate that the band is wide enough.
 * scale <= 0 is TPCF_EINVAL. */
tpcf_status tpcf_set_guard_scale(tpcf_ctx* ctx, double scale);
/* Window path on (default) / off.  On: catalogs are held in Hilbert-curve order with a bounding sphere per 8-row group
 * (i side) and per 64-row subtile / 128-row tile (j side); for every (group, subtile) block the kernel bounds the chord
 * lengths by the triangle inequality, and when at most 3 bin edges can be reached it classifies each pair with that many
 * sign tests against the band midpoints (register counters, no shared-memory traffic per pair); otherwise, and always
 * when off, each pair goes through the cell lookup.  Every pair is evaluated either way; the histograms are identical
 * (tests). */
tpcf_status tpcf_set_window(tpcf_ctx* ctx, int enabled);
/* TPCF_ENGINE_TENSOR launches the tensor kernel when the sampled share of pair-by-pair blocks (tpcf_stats.lookup_share) is at
 * most `limit` (default 0.025), else the FFMA2 kernel.  0 = always the FFMA2 kernel; 1 = always the tensor kernel (what the
 * tests use to exercise it on small catalogs).  The histograms do not depend on it. */
tpcf_status tpcf_set_tensor_share_limit(tpcf_ctx* ctx, double limit);
/* Pruning mode, off by default (PAPER.md:29-31 k-trees, "coding the k-trees" as future
 * work).  On: a (256 i-rows, 64 j-rows) block none of whose 32 (8-row group, subtile) windows reaches a bin edge is added
 * to the histogram wholesale -- its pairs are NOT evaluated.  The histograms are the same integers (the windows bound
 * every true separation, tests), but this is the dual-tree idea at block granularity, not the brute-force count the
 * paper and BASELINE.json's metric are about: "pair evaluations per second" loses its meaning, so bench.py reports it as
 * a separate line (--pruning) and never as the headline.  Runs the FFMA2 kernel whatever the engine. */
tpcf_status tpcf_set_pruning(tpcf_ctx* ctx, int enabled);
/* Work partition for multi-process runs (one process per GPU): this context enumerates only the tile
 * work items w with w % nparts == part; summing the histograms of all parts gives the full count
 * (integer, order-independent).  Default (0, 1).  Every part must number the same items: with nparts > 1 the plan's
 * chunking is fixed (balanced for 148 SMs) and does not depend on the GPU a rank runs on; all ranks must load the same
 * catalogs (same sizes) and use the same nparts. */
tpcf_status tpcf_set_partition(tpcf_ctx* ctx, int part, int nparts);

/* Per-kernel device timing: when enabled, every later count records a CUDA event pair around its pair
 * kernel on the context's stream (up to 64 outstanding).  tpcf_get_kernel_times waits for them, writes the
 * durations in milliseconds, oldest first, and clears the list.  tpcf_count_all(_async) records ONE pair around its three
 * kernels (they overlap).  Used by bench.py for the roofline line. */
tpcf_status tpcf_set_kernel_timing(tpcf_ctx* ctx, int enabled);
tpcf_status tpcf_get_kernel_times(tpcf_ctx* ctx, float* ms_out, int capacity, int* n_out);

typedef struct {
    uint64_t pairs;          /* pairs enumerated by the last count (after the partition) */
    uint64_t rechecked;      /* pairs the fast engine re-evaluated in fp64 (inside a guard band) */
    uint64_t work_items;     /* tile work items executed */
    int launches;            /* kernels launched by the last count */
    int grid, block, smem_bytes;   /* geometry of the pair kernel */
    int cells, cell_bits;    /* lookup cells of the fast engine and mantissa bits per octave */
    float kernel_ms;         /* device time of the last synchronous count (CUDA events) */
    uint64_t win_blocks[6];  /* (warp of 256 i-rows, 64-row j-subtile) blocks -- tensor engine: (warp of 32 i-rows, 128-row j-tile) -- of the last synchronous count by path:
                                counted by the 1-, 2-, 3-edge window loops, by the per-pair cell lookup; [4] = lanes of
                                window blocks recounted pair by pair because a pair came within a guard band;
                                [5] = blocks classified wholly in fp64 (bounding radii too large for the fp32 bound) */
    uint64_t pruned_blocks;  /* pruning mode: (warp, subtile) blocks added wholesale by the last synchronous count */
    float lookup_share;      /* TPCF_ENGINE_TENSOR: share of the (8-row group, 128-row tile) blocks the tensor kernel would count pair
                                by pair (near blocks, more than 3 edges in reach, radii beyond the cap), sampled on 65536 blocks once per
                                catalog pair; above 0.025 the engine launches the FFMA2 kernel (the histograms are the same) */
} tpcf_stats;
tpcf_status tpcf_get_stats(const tpcf_ctx* ctx, tpcf_stats* out);

/* ---- host-only helpers (no GPU needed) ------------------------------------------------------------- */

/* fp64 thresholds T_k = 4 sin^2(e_k/2) in squared-chord space the engines compare against (nbins+1). */
tpcf_status tpcf_get_thresholds(const tpcf_ctx* ctx, double* t_out /* nbins+1 */);

/*
 * The fast engine's classification of one fp32 squared chord d2, evaluated on the host with the very
 * tables the kernel uses: returns in *slot_out the result slot (0 = under, 1..nbins = bins, nbins+1 = over,
 * nbins+2 = discarded padding lane) or -1 when d2 falls in a guard band (the kernel then re-evaluates the
 * pair in fp64).  Lets CPU tests check the table builder against the thresholds without a GPU.
 */
tpcf_status tpcf_classify_fast(const tpcf_ctx* ctx, float d2, int* slot_out);

/* The guard bands of the fast engine (ascending, disjoint; the last is the zero-width "discard" band that separates
 * real pairs from padding lanes): *n_out = number of bands; if capacity >= that, lo/hi (fp32 squared chord) and the
 * result slot just below each band are written (any of the three may be NULL). */
tpcf_status tpcf_get_bands(const tpcf_ctx* ctx, int capacity, float* lo_out, float* hi_out, int* slot_below_out, int* n_out);
/* Host mirror of the kernel's window selection: for a block whose fp32 squared chords all lie in [lo2, hi2], the first
 * band that is not wholly below lo2 and the number of consecutive bands the block can reach (1..3, or 4 = too many,
 * cell-lookup path).  0 <= lo2 <= hi2 < 64. */
tpcf_status tpcf_window_host(const tpcf_ctx* ctx, float lo2, float hi2, int* first_band_out, int* n_edges_out);

/* Number of tile work items of a full count of `kind` (TPCF_DD, TPCF_DR or TPCF_RR; the D2 kinds have a third size and
 * are refused with TPCF_EINVAL) for catalog sizes (n_d, n_r), and the number of pairs in item w: the partition arithmetic
 * of tpcf_set_partition, testable without a GPU.  With nparts > 1 set on the context the numbering is the fixed one every
 * rank uses; with nparts == 1 it is the one this context's own counts use (balanced for its device once it has seen one). */
tpcf_status tpcf_plan(const tpcf_ctx* ctx, tpcf_kind kind, uint64_t n_d, uint64_t n_r, uint64_t* n_items_out);
tpcf_status tpcf_plan_item_pairs(const tpcf_ctx* ctx, tpcf_kind kind, uint64_t n_d, uint64_t n_r, uint64_t w,
                                 uint64_t* pairs_out);

/* ---- diagnostics (not part of the counting path; needs the GPU) ------------------------------------------ */

/* The tensor engine's arithmetic on its own: ntiles tiles of 128 i-rows x 128 j-rows.  s_rows: ntiles x
 * 128 x 4 floats (s_x, s_y, s_z, |s|^2 - mid) and b_rows: ntiles x 128 x 4 floats (-2 b'_x, -2 b'_y, -2 b'_z, |b'|^2), host
 * memory; q_out: ntiles x 128 x 128 floats, row-major per tile, host memory: q[i][j] = s_w[i] + b_w[j] + s[i] . b[j] as the
 * 3xTF32 tcgen05.mma of pair_tensor_kernel forms it (same operand split, same instruction, same read-back).  What the tests
 * measure the tensor core's accumulation error with.  TPCF_EINVAL for NULL pointers or ntiles == 0 or > 65535. */
tpcf_status tpcf_tensor_probe(tpcf_ctx* ctx, const float* s_rows, const float* b_rows, size_t ntiles, float* q_out);

/* ---- three-point counts ------------------------------------------------------------------------------------ */

/*
 * tpcf_count3 -- three-point counts of one loaded catalog ("extending the work to higher
 *   order correlation functions"; the paper names the extension and gives no formula -- the definition is
 *   DESIGN.md section 15's).  Every unordered triple i<j<k of the catalog is a triangle with three sides; each side gets
 *   the result slot a pair gets (0 = under, 1..nbins = bin_0..bin_{n-1}, nbins+1 = over; same edges, same conventions as
 *   tpcf_count), and the triple is counted once in the cell of its three slots in ascending order a <= b <= c:
 *     hist3_out[(a * m + b) * m + c],  m = nbins + 2,  host memory, m^3 uint64 (cells that are not ascending stay 0).
 *   sum(hist3_out) = N(N-1)(N-2)/6 exactly.  Brute force: every triple is enumerated (O(N^3) byte operations after one
 *   O(N^2) fp64 classification of the pairs).  Angular and 3-D contexts alike.  Not part of the w(theta) headline.
 *   Limits: N <= TPCF_COUNT3_MAX_ROWS (the N x N byte matrix of pair slots is scratch), nbins <= TPCF_COUNT3_MAX_BINS
 *   (the m^3 partial histogram lives in shared memory); beyond them TPCF_EINVAL.  TPCF_ESTATE before the catalog is loaded.
 *   tpcf_get_stats afterwards: kernel_ms of the two kernels, pairs = number of triples.
 */
#define TPCF_COUNT3_MAX_ROWS 16384
#define TPCF_COUNT3_MAX_BINS 30
tpcf_status tpcf_count3(tpcf_ctx* ctx, tpcf_cat which, uint64_t* hist3_out /* (nbins+2)^3 */);

/* ---- a count that allocates nothing ---------------------------------------------------------------------- */

/*
 * tpcf_count_static -- one pair count (the histogram over theta of the separations of all pairs;
 *   PAPER.md:37-38), from RA/Dec rows to histogram, WITHOUT any allocation of device memory: no cudaMalloc, no cudaFree,
 *   no allocating library routine, on the first call or any later one.  It needs no context.
 *
 *   Who needs it.  tpcf_load and tpcf_count allocate (catalog arrays, sort scratch, accumulators, the plan).  A caller
 *   cannot always let a library do that: all device memory may already sit in the host application's own pool (a
 *   framework's caching allocator), so that a raw cudaMalloc fails or eats into what the pool believes it owns; a
 *   service may have to prove its per-GPU memory use at start-up; and cudaMalloc / cudaFree synchronise the whole
 *   device, which a loop with other streams in flight cannot tolerate.  Such a caller hands in device pointers it
 *   already owns and gets the result in a device buffer it already owns.
 *
 *   How.  The scratch of the count (the fp64 unit vectors made from the rows, the thresholds, the uint64 accumulators,
 *   the work counter, the bad-row flag) lives in one fixed array inside the library's device image, about 2.07 MiB,
 *   which every GPU that loads the image holds until the process exits.  Hence the limits:
 *     rows:  n_i + n_j <= TPCF_STATIC_MAX_ROWS;   bins:  nbins <= TPCF_STATIC_MAX_BINS;
 *   anything larger is refused with TPCF_EINVAL and a message that names the limit.  The pairs are counted by a variant
 *   of the TPCF_ENGINE_EXACT64 kernel (fp64 squared chord against 4 sin^2(e_k/2)), so the histogram is the one
 *   tpcf_count gives with any engine, up to fp64 ties; at these sizes the fp64 count takes milliseconds.
 *
 *   nbins, theta_deg, mode   the binning, as for tpcf_create (host memory).
 *   radec_i_dev, n_i         DEVICE pointer to n_i rows of (RA, Dec) in degrees, row-major, dtype dt.
 *   radec_j_dev, n_j         DEVICE pointer to a second catalog: all n_i * n_j pairs are counted (DR).
 *                            NULL with n_j = 0: the n_i (n_i - 1) / 2 pairs i < j of the first catalog (DD, RR).
 *   hist_dev                 DEVICE buffer of nbins + 2 uint64: {under, bin_0 .. bin_{n-1}, over} (tpcf_count_async's layout).
 *   cuda_stream              the cudaStream_t to work on (NULL: the default stream).  The call returns after that stream
 *                            has drained (it reads the bad-row flag back), so hist_dev is complete on return.
 *   err, err_len             optional host buffer for a message when the status is not TPCF_OK (there is no context
 *                            to ask).
 *
 *   One array serves every call.  It keeps whatever the last call left there; the call clears the parts that must
 *   start at zero itself.  Two calls that overlap in time on one GPU (two host threads, two streams) corrupt each other:
 *   serialise them.  Calls on different GPUs do not interact.
 *   The first call on each device looks up where the array lives on that device (the device current at the call is the
 *   one used) and may load the library's device image; make that first call before starting any stream capture.
 *   Errors: TPCF_EINVAL (limits, NULL pointers, bad edges, a non-finite value, |RA| > 1e6 or |Dec| > 90 in a row);
 *   TPCF_ECUDA (no usable sm_100 device -- there is no CPU fallback -- or a CUDA failure).
 */
#define TPCF_STATIC_MAX_ROWS 65536
#define TPCF_STATIC_MAX_BINS 4096
tpcf_status tpcf_count_static(int nbins, const double* theta_deg, tpcf_binning mode, const void* radec_i_dev, size_t n_i,
                              const void* radec_j_dev, size_t n_j, tpcf_dtype dt, uint64_t* hist_dev /* device, nbins+2 */,
                              void* cuda_stream, char* err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* TPCF_H */
