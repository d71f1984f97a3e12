// tables.h -- host-side (no CUDA) logic of libtpcf: theta edges, chord-space thresholds, the fast engine's
// guard bands and cell lookup table, the tile work plan and the estimator.  See DESIGN.md sections 3-5.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace tpcf {

// Geometry shared by the host plan and the kernels.
constexpr int kThreads = 256;          // threads per CTA
constexpr int kIPerThread = 8;         // i-points held in registers per thread (one "group": they share a bounding sphere)
constexpr int kTileI = kThreads * kIPerThread;   // 2048 i-points per plan item
constexpr int kTileJ = kTileI;         // j-points per plan tile (the triangle plan needs kTileJ == kTileI)
constexpr int kMaxChunk = 8;           // j-tiles per work item, at most
constexpr int kPlanSMs = 148;          // SM count the plan balances for until the context has seen its device (B200: 148)
constexpr float kPadCoord = 2.0f;      // padding rows are (2,2,2): 6.07 <= d2 <= 19.9 against any unit vector
constexpr float kDiscardFrom = 5.0f;   // d2 >= 5 can only involve a padding row
constexpr int kMaxCells = 8192;
// guard of the cell-lookup path around the threshold of a cell: a pair with fp32 squared chord q is
// decided in fp32 iff |q - T| > scale * (kLookupAlpha * Q + kLookupBetaR * r * sqrt(Q) + kLookupBeta0), Q >= q a bound on the
// squared chords of the (lane, subtile) block and r the sum of its bounding radii; true error <= (9 q + 10 sqrt(q) r) 2^-24
constexpr float kLookupAlpha = 7.5e-7f, kLookupBetaR = 8.0e-7f, kLookupBeta0 = 1.0e-13f;
constexpr int kSubJ = 64;              // j-points per window subtile (one bounding sphere each)
constexpr int kChunkJ = 128;           // j-points per bulk copy into a warp's shared-memory ring (= i-points per warp)
constexpr int kWarpsPerCta = kThreads / 32;
constexpr int kWarpI = 32 * kIPerThread;   // i-points per warp work item
constexpr float kRCap = 0.25f;         // blocks whose bounding radii sum to more go to the fp64 path (guard_width_lookup assumes it)
constexpr float kFarKappa = 2.5f;      // the expanded-form window loops need  min chord >= kFarKappa * (ri + rj)
constexpr int kMaxWinEdges = 3;        // a (lane, subtile) window that sees more guard bands goes to the cell-lookup path

enum class CellMap : int { LogBits = 0, SqrtLin = 1 };

// Result-slot numbering used everywhere: 0 = under, 1..nbins = bins, nbins+1 = over, nbins+2 = discard.
struct FastTables {
    CellMap map = CellMap::LogBits;
    int shift = 21;                 // LogBits: cell = bits(d2) >> shift
    float sqrt_scale = 0.f;         // SqrtLin: 4 * cell + 2 noise bits = low 23 bits of fmaf(approx_sqrt(min(d2, sqrt_clamp)), sqrt_scale, 2^23)
    float sqrt_clamp = 0.f;
    int ncells = 0;
    int merged_bands = 0;           // guard bands that had to be merged because they shared a cell (0 normally)
    double guard_scale = 1.0;       // tpcf_set_guard_scale: multiplies every guard width, in the tables and in the kernels
    // per cell: the one threshold T (fp32 rounding of 4 sin^2(e_k/2)) whose guard band reaches into the cell:
    //   d2 < T -> slot0, d2 >= T -> slot1, |d2 - T| <= guard -> ambiguous (fp64 recheck);
    // +inf: no band reaches the cell (slot0 == slot1); NaN: several do, every pair of the cell is ambiguous
    std::vector<float> tcell;
    std::vector<uint16_t> slot0, slot1;
    // The guard bands themselves, ascending and disjoint (the last one is the zero-width "discard" band at
    // kDiscardFrom).  The window path of the kernel compares against these directly: a pair whose fp32 squared chord
    // q satisfies |q - band_mid| > band_half is on the side of the edge its sign shows.
    int nbands = 0;
    std::vector<float> band_lo, band_hi, band_mid, band_half;
    std::vector<uint16_t> band_slot;    // nbands + 1: result slot below band b; [nbands] = slot above the last band
    std::vector<uint16_t> cell_band;    // per cell: first band whose hi lies above the start of the cell
    int cell_of(float d2) const;    // exactly the kernel's integer arithmetic
    int classify(float d2) const;   // result slot, or -1 when ambiguous
    // Host mirror of the kernel's window selection: given bounds lo2 <= q <= hi2 on every squared chord of a
    // (lane, subtile) block, the first band that can matter and how many consecutive bands can (1..kMaxWinEdges,
    // or kMaxWinEdges + 1 = "too many": cell-lookup path).
    void window(float lo2, float hi2, int& first_band, int& n_edges) const;
};

struct Binning {
    int nbins = 0;
    std::vector<double> edges;      // degrees (angular contexts) or lengths (3-D contexts), nbins+1
    std::vector<double> thr;        // angular: T_k = 4 sin^2(e_k/2); 3-D: T_k = (e_k * scale)^2; nbins+1
    bool spatial = false;           // 3-D context (tpcf_create_r): rows are Cartesian positions, bins are in |a - b|
    double scale = 1.0;             // 3-D: positions are multiplied by this power of two (exact) so that |p * scale| <= 1
    double max_abs = 0.0;           // 3-D: the largest |coordinate| the caller promised
    bool drop_first = false;        // e_0 == 0: nothing can be "under"
    bool drop_last = false;         // e_n == 180: nothing can be "over"
};

// Returns "" on success, else the reason (-> TPCF_EINVAL).
std::string make_binning(int nbins, const double* theta_deg, int mode, Binning& out);
// 3-D variant: edges are separations r >= 0 in the units of the coordinates; every coordinate of every row
// will satisfy |x| <= max_abs_coord.
std::string make_binning_r(int nbins, const double* r_edges, int mode, double max_abs_coord, Binning& out);

// fp32 rounding bound of the fast engine's squared chord around the true value t.
double guard_width(double t, double scale);
// ... of the tensor engine's: the 3xTF32 split and the tensor core's truncating accumulation come on top
double guard_width_tensor(double t, double scale);
// ... and of the difference form alone (the bands of the cell-lookup tables)
double guard_width_lookup(double t, double scale);

// tensor: the window bands are those of the tensor engine (guard_width_tensor)
void build_fast_tables(const Binning& b, double guard_scale, bool tensor, FastTables& out);

// Exact classification used by the fp64 engine and the recheck path (host mirror of the device code).
int exact_slot(double d2, const Binning& b);

// ---- tile work plan --------------------------------------------------------------------------------
struct Plan {
    bool tri = false;               // true: one catalog, pairs i<j; false: rectangle n_i x n_j
    uint64_t n_i = 0, n_j = 0;
    uint32_t blocks_i = 0, tiles_j = 0, chunk = 1;
    uint64_t n_items = 0;
    std::vector<uint32_t> row_start;   // tri only: first item of i-block I (blocks_i + 1 entries)
    // item w -> i-block, first j-tile, number of j-tiles
    void item(uint64_t w, uint32_t& I, uint32_t& tile0, uint32_t& ntiles) const;
    uint64_t item_pairs(uint64_t w) const;
};
void make_plan(bool tri, uint64_t n_i, uint64_t n_j, int sm_count, Plan& out);

void estimate(const uint64_t* dd, const uint64_t* dr, const uint64_t* rr, int nbins, uint64_t n_d, uint64_t n_r,
              double* w);

}  // namespace tpcf
