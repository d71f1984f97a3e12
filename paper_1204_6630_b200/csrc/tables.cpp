// tables.cpp -- host-side logic of libtpcf (no CUDA calls): binning, thresholds, guard bands, cell lookup
// table, work plan, estimator.  DESIGN.md sections 3-5 derive everything here.
#include "tables.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>

namespace tpcf {

static const double kPi = 3.14159265358979323846;

static inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
static inline float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }
static float float_down(double x) {
    float f = (float)x;
    if ((double)f > x) f = std::nextafterf(f, -std::numeric_limits<float>::infinity());
    return f;
}
static float float_up(double x) {
    float f = (float)x;
    if ((double)f < x) f = std::nextafterf(f, std::numeric_limits<float>::infinity());
    return f;
}

// --------------------------------------------------------------------------------------------------
// Binning.  The paper fixes no bins (reading A4); edges in degrees, chord-space thresholds
// T_k = |a-b|^2 at separation e_k = 2 - 2 cos(e_k) = 4 sin^2(e_k/2): a monotone function of the dot
// product of PAPER.md:37, so comparing against T_k is "binning in cos(theta) space" without an acos and
// without the cancellation of 1 - cos at small angles.
// --------------------------------------------------------------------------------------------------
std::string make_binning(int nbins, const double* theta, int mode, Binning& out) {
    if (nbins < 1 || nbins > 4096) return "nbins must be in [1, 4096]";
    if (!theta) return "theta_deg is NULL";
    std::vector<double> e((size_t)nbins + 1);
    if (mode == 0 || mode == 1) {
        double lo = theta[0], hi = theta[1];
        if (!(lo == lo) || !(hi == hi)) return "NaN edge";
        if (!(lo >= 0.0 && hi <= 180.0 && lo < hi)) return "need 0 <= min < max <= 180";
        if (mode == 1 && !(lo > 0.0)) return "LOG binning needs min > 0";
        for (int k = 0; k <= nbins; ++k)
            e[k] = (mode == 0) ? lo + k * ((hi - lo) / nbins) : lo * std::pow(hi / lo, (double)k / nbins);
        e[0] = lo;
        e[nbins] = hi;
    } else if (mode == 2) {
        for (int k = 0; k <= nbins; ++k) {
            if (!(theta[k] == theta[k])) return "NaN edge";
            e[k] = theta[k];
        }
    } else {
        return "unknown binning mode";
    }
    if (!(e[0] >= 0.0 && e[nbins] <= 180.0)) return "edges must lie in [0, 180]";
    for (int k = 0; k < nbins; ++k)
        if (!(e[k] < e[k + 1])) return "edges must be strictly increasing";
    out.nbins = nbins;
    out.edges = e;
    out.thr.resize((size_t)nbins + 1);
    for (int k = 0; k <= nbins; ++k) {
        double s = std::sin(e[k] * kPi / 360.0);
        out.thr[k] = 4.0 * s * s;
    }
    out.drop_first = (e[0] == 0.0);
    out.drop_last = (e[nbins] == 180.0);
    if (out.drop_first) out.thr[0] = 0.0;
    if (out.drop_last) out.thr[nbins] = 4.0;
    for (int k = 0; k < nbins; ++k)
        if (!(out.thr[k] < out.thr[k + 1])) return "edges closer than fp64 can separate in chord space";
    return "";
}

// 3-D variant ("results are extendible to the 3-dimensional variant as well"): the same histograms over the
// Euclidean separation r = |a - b| of Cartesian positions.  Positions are scaled by a power of two (exact in binary
// floating point) into the unit ball, so that everything the kernels assume about squared chords of unit vectors holds
// (d^2 <= 4, padding rows at (2,2,2) are farther than 6 from every row); thresholds T_k = (e_k * scale)^2.
std::string make_binning_r(int nbins, const double* r, int mode, double max_abs, Binning& out) {
    if (nbins < 1 || nbins > 4096) return "nbins must be in [1, 4096]";
    if (!r) return "r_edges is NULL";
    if (!(max_abs > 0.0) || !(max_abs < 1.0e300)) return "max_abs_coord must be positive and finite";
    int ex = 0;
    std::frexp(max_abs * 1.7320508075688774, &ex);          // 2^ex > sqrt(3) max_abs >= |p|
    const double scale = std::ldexp(1.0, -ex);
    std::vector<double> e((size_t)nbins + 1);
    if (mode == 0 || mode == 1) {
        const double lo = r[0], hi = r[1];
        if (!(lo == lo) || !(hi == hi)) return "NaN edge";
        if (!(lo >= 0.0 && lo < hi) || !(hi < 1.0e300)) return "need 0 <= min < max";
        if (mode == 1 && !(lo > 0.0)) return "LOG binning needs min > 0";
        for (int k = 0; k <= nbins; ++k)
            e[k] = (mode == 0) ? lo + k * ((hi - lo) / nbins) : lo * std::pow(hi / lo, (double)k / nbins);
        e[0] = lo;
        e[nbins] = hi;
    } else if (mode == 2) {
        for (int k = 0; k <= nbins; ++k) {
            if (!(r[k] == r[k])) return "NaN edge";
            e[k] = r[k];
        }
    } else {
        return "unknown binning mode";
    }
    if (!(e[0] >= 0.0)) return "edges must be >= 0";
    for (int k = 0; k < nbins; ++k)
        if (!(e[k] < e[k + 1])) return "edges must be strictly increasing";
    out = Binning();
    out.nbins = nbins;
    out.edges = e;
    out.spatial = true;
    out.scale = scale;
    out.max_abs = max_abs;
    out.thr.resize((size_t)nbins + 1);
    for (int k = 0; k <= nbins; ++k) {
        const double es = e[k] * scale;                     // exact
        out.thr[k] = std::min(es * es, 4.5);                // no two scaled rows are farther apart than 2
    }
    out.drop_first = (e[0] == 0.0);
    out.drop_last = false;
    for (int k = 0; k < nbins; ++k)
        if (!(out.thr[k] < out.thr[k + 1]) || out.thr[k + 1] > 4.0) return "edges beyond the largest possible separation, or closer than fp64 can separate";
    return "";
}

int exact_slot(double d2, const Binning& b) {
    const int n = b.nbins;
    if (d2 > 4.0) d2 = 4.0;                 // the oracle clamps the dot product to [-1, 1] (reading A7)
    if (d2 < b.thr[0]) return 0;
    if (d2 > b.thr[n]) return n + 1;
    int lo = 0, hi = n;                     // thr[lo] <= d2, (hi == n or d2 < thr[hi])
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (b.thr[mid] <= d2) lo = mid; else hi = mid;
    }
    return lo + 1;
}

// Bound on |q_fp32 - q| of the fast engine around a threshold t, u = 2^-24.  Coordinates are
// held relative to the centre of their kIPerThread-row group (i side) and kSubJ-row subtile (j side), so every error is
// relative to the chord d or to the radii r = ri + rj <= kRCap:
//   difference form (cell-lookup path):                   (9 d^2 + 10 d r) u   <= 5.4e-7 t + 6.0e-8 sqrt(t)
//   expanded form (window path, d >= kFarKappa r = 2.5 r): 29.1 d^2 u          <= 1.74e-6 t
// The constants below add margin (x1.67 on the sqrt term, x1.72 on the linear one).
double guard_width(double t, double scale) { return scale * (1.0e-7 * std::sqrt(t) + 3.0e-6 * t + 1.0e-13); }
// The tensor engine forms the same expanded form from 3xTF32 operands on the tensor core: inputs and norms 15.2 u, 3xTF32
// split residual 13.4 u, the tensor core's truncating accumulation 13.1 u, further edges 2 u = 43.7 u max(d^2, mid) =
// 2.61e-6 t (lemma T; the accumulation model is checked bit for bit on the GPU); margin x1.53.
double guard_width_tensor(double t, double scale) { return scale * (1.0e-7 * std::sqrt(t) + 4.0e-6 * t + 1.0e-13); }
// The cell-lookup path only ever evaluates the difference form: (9 d^2 + 10 d r) u with r <= kRCap = 0.25, i.e.
// 5.4e-7 t + 1.5e-7 sqrt(t); margins x1.85 and x1.67.  This width decides which cells SEE a threshold (tables.h
// FastTables::tcell); whether a pair is ambiguous is decided in the kernel from the radii of its own block.
double guard_width_lookup(double t, double scale) { return scale * (2.5e-7 * std::sqrt(t) + 1.0e-6 * t + 1.0e-13); }

// --------------------------------------------------------------------------------------------------
// Cell maps.  Both are integer/IEEE arithmetic on the float's bit pattern, reproduced exactly on the device.
// --------------------------------------------------------------------------------------------------
static const uint32_t kSqrtMagic = 0x1FBD1DF5u;   // bits(sqrt(x)) ~ (bits(x) >> 1) + magic (within ~4 %)
static const uint32_t kTopBits = 0x42800000u;     // bits(64.0f): no squared chord, padded or not, reaches it

int FastTables::cell_of(float d2) const {
    if (map == CellMap::LogBits) return (int)(f2u(d2) >> shift);
    float c = std::fmin(d2, sqrt_clamp);
    float key = u2f((f2u(c) >> 1) + kSqrtMagic);
    float t = std::fmaf(key, sqrt_scale, 8388608.0f);
    return (int)((f2u(t) & 0x7FFFFFu) >> 2);
}

int FastTables::classify(float d2) const {
    int c = cell_of(d2);
    if (c < 0 || c >= ncells) return -2;
    const float T = tcell[c];
    if (T != T) return -1;
    // the kernel's test with the widest block it admits (r = kRCap) and the tightest bound on the block's chords (q itself)
    const float e = d2 - T;
    const double g = guard_scale * ((double)kLookupAlpha * d2 + (double)kLookupBetaR * kRCap * std::sqrt((double)d2) + (double)kLookupBeta0);
    if (!(std::fabs((double)e) > g)) return -1;
    return e < 0.0f ? slot0[c] : slot1[c];
}

void FastTables::window(float lo2, float hi2, int& first_band, int& n_edges) const {
    int c = cell_of(lo2);
    if (c < 0) c = 0;
    if (c >= ncells) c = ncells - 1;
    int k = cell_band[c];
    while (k < nbands && band_hi[k] <= lo2) ++k;
    int e = 1;
    while (e <= kMaxWinEdges && k + e < nbands && band_lo[k + e] <= hi2) ++e;
    first_band = k;
    n_edges = e;
}

namespace {
struct Band {
    float lo, hi;
    int below, above;
    float t = 0.f;          // fp32 rounding of the threshold the band surrounds
    bool merged = false;    // several overlapping bands in one: no single threshold
};

// first float (as bits) whose cell index is >= c; cell_of is monotone non-decreasing in d2 >= 0
uint32_t first_bits_of_cell(const FastTables& t, int c) {
    uint32_t a = 0, b = kTopBits;           // answer in [a, b]
    if (t.cell_of(u2f(b)) < c) return b + 1;
    while (a < b) {
        uint32_t m = a + (b - a) / 2;
        if (t.cell_of(u2f(m)) >= c) b = m; else a = m + 1;
    }
    return a;
}

// Fill lo/hi/slot tables for the current map; returns the number of cells that see more than one band.
int fill(FastTables& t, const std::vector<Band>& bands, int lowest_slot) {
    const float inf = std::numeric_limits<float>::infinity();
    t.ncells = t.cell_of(u2f(kTopBits)) + 1;
    t.tcell.assign(t.ncells, inf);
    t.slot0.assign(t.ncells, 0);
    t.slot1.assign(t.ncells, 0);
    t.cell_band.assign(t.ncells, 0);
    int bad = 0;
    size_t first = 0;                       // first band with hi > start of this cell
    for (int c = 0; c < t.ncells; ++c) {
        uint32_t b0 = first_bits_of_cell(t, c), b1 = first_bits_of_cell(t, c + 1);
        if (b1 == b0) {                     // empty cell (SqrtLin can skip indices): never addressed
            t.slot0[c] = t.slot1[c] = (uint16_t)lowest_slot;
            t.cell_band[c] = (uint16_t)first;
            continue;
        }
        float f0 = (c == 0) ? 0.0f : u2f(b0);
        float f1 = (b1 > kTopBits) ? inf : u2f(b1);
        while (first < bands.size() && bands[first].hi <= f0) ++first;   // bands wholly below this cell
        t.cell_band[c] = (uint16_t)first;
        // bands [first, last) intersect [f0, f1)
        size_t last = first;
        while (last < bands.size() && bands[last].lo < f1) ++last;
        int region = (first == 0) ? lowest_slot : bands[first - 1].above;
        if (last == first) {
            t.slot0[c] = t.slot1[c] = (uint16_t)region;
        } else {
            // More than one band reaches into the cell (or one that stands for several merged ones): every pair of the
            // cell is treated as ambiguous (classified by the fp64 path), which is always correct, only slower.
            const bool multi = last - first > 1 || bands[first].merged;
            if (last - first > 1) ++bad;
            t.tcell[c] = multi ? std::numeric_limits<float>::quiet_NaN() : bands[first].t;
            t.slot0[c] = (uint16_t)bands[first].below;
            t.slot1[c] = (uint16_t)bands[last - 1].above;
        }
    }
    return bad;
}
}  // namespace

static void export_bands(const std::vector<Band>& bands, FastTables& t) {
    t.nbands = (int)bands.size();
    t.band_lo.resize(t.nbands);
    t.band_hi.resize(t.nbands);
    t.band_mid.resize(t.nbands);
    t.band_half.resize(t.nbands);
    t.band_slot.resize((size_t)t.nbands + 1);
    for (int k = 0; k < t.nbands; ++k) {
        const float lo = bands[k].lo, hi = bands[k].hi;
        const float mid = (float)(0.5 * ((double)lo + (double)hi));
        // [mid - half, mid + half] covers [lo, hi] whatever the rounding of mid
        const float half = float_up(std::max((double)hi - (double)mid, (double)mid - (double)lo));
        t.band_lo[k] = lo;
        t.band_hi[k] = hi;
        t.band_mid[k] = mid;
        t.band_half[k] = half;
        t.band_slot[k] = (uint16_t)bands[k].below;   // == bands[k-1].above: the bands chain
    }
    t.band_slot[t.nbands] = (uint16_t)bands.back().above;
}

// Guard bands around the droppable edges (ascending, overlapping ones merged) + the zero-width discard band.
// Returns the number of merges.
static int make_bands(const Binning& b, double gs, int form /* 0 window, 1 lookup, 2 tensor window */, std::vector<Band>& bands) {
    const int n = b.nbins;
    int overlapping = 0;
    bands.clear();
    for (int k = 0; k <= n; ++k) {
        if ((k == 0 && b.drop_first) || (k == n && b.drop_last)) continue;
        double T = b.thr[k], g = form == 1 ? guard_width_lookup(T, gs) : form == 2 ? guard_width_tensor(T, gs) : guard_width(T, gs);
        Band bd;
        bd.lo = (T - g <= 0.0 || T < 1e-12) ? 0.0f : float_down(T - g);
        bd.hi = float_up(T + g);
        bd.below = k;
        bd.above = k + 1;
        bd.t = (float)T;
        if (!bands.empty() && bd.lo < bands.back().hi) {      // overlapping guard bands: one wider ambiguous band
            bands.back().hi = std::max(bands.back().hi, bd.hi);
            bands.back().above = bd.above;
            bands.back().merged = true;
            ++overlapping;
        } else {
            bands.push_back(bd);
        }
    }
    const int lowest = b.drop_first ? 1 : 0;
    {   // everything at or above kDiscardFrom involves a padding row: zero-width band, never ambiguous
        Band d;
        d.lo = d.hi = d.t = kDiscardFrom;
        d.below = bands.empty() ? lowest : bands.back().above;
        d.above = n + 2;
        if (!bands.empty() && bands.back().hi > kDiscardFrom) bands.back().hi = kDiscardFrom;
        bands.push_back(d);
    }
    return overlapping;
}

// per cell: first window band whose hi lies above the start of the cell (the kernel's window search starts there)
static void fill_cell_band(FastTables& t, const std::vector<Band>& bands) {
    t.cell_band.assign(t.ncells, 0);
    size_t first = 0;
    for (int c = 0; c < t.ncells; ++c) {
        const uint32_t b0 = first_bits_of_cell(t, c), b1 = first_bits_of_cell(t, c + 1);
        if (b1 != b0) {
            const float f0 = (c == 0) ? 0.0f : u2f(b0);
            while (first < bands.size() && bands[first].hi <= f0) ++first;
        }
        t.cell_band[c] = (uint16_t)first;
    }
}

static void build_fast_tables_impl(const Binning& b, const std::vector<Band>& bands, int overlapping, FastTables& out);

void build_fast_tables(const Binning& b, double gs, bool tensor, FastTables& out) {
    std::vector<Band> lookup_bands, window_bands;
    const int ov = make_bands(b, gs, 1, lookup_bands);
    make_bands(b, gs, tensor ? 2 : 0, window_bands);
    build_fast_tables_impl(b, lookup_bands, ov, out);      // cell map + (threshold, slots) per cell: the lookup path
    out.guard_scale = gs;
    export_bands(window_bands, out);                       // the bands the window loops compare against
    fill_cell_band(out, window_bands);
}

static void build_fast_tables_impl(const Binning& b, const std::vector<Band>& bands, int overlapping, FastTables& out) {
    const int lowest = b.drop_first ? 1 : 0;

    // 1. LogBits with 2, 4, ... cells per octave
    FastTables t;
    t.merged_bands = overlapping;
    for (int shift = 22; shift >= 19; --shift) {
        t.map = CellMap::LogBits;
        t.shift = shift;
        if ((int)(kTopBits >> shift) + 1 > kMaxCells) break;
        if (fill(t, bands, lowest) == 0) { out = t; return; }
    }
    // 2. SqrtLin (bins of near-constant width in theta)
    {
        double top = 0.0;
        for (size_t m = 0; m + 1 < bands.size(); ++m) top = std::max(top, (double)bands[m].hi);
        float clamp = std::min(kDiscardFrom * 0.999f, (float)(top * 1.25 + 1e-9));
        float keymax = u2f((f2u(clamp) >> 1) + kSqrtMagic);
        for (int target = 512; target <= kMaxCells; target *= 2) {
            t.map = CellMap::SqrtLin;
            t.sqrt_clamp = clamp;
            t.sqrt_scale = (float)(4.0 * (target - 2) / (double)keymax);
            if (fill(t, bands, lowest) == 0 && t.ncells <= kMaxCells) { out = t; return; }
        }
    }
    // 3. Fallback, always correct: finest LogBits map; a cell that sees several guard bands treats the whole
    //    span between them as ambiguous, so those pairs are classified by the fp64 path.
    t.map = CellMap::LogBits;
    t.shift = 19;
    t.merged_bands += fill(t, bands, lowest);
    out = t;
}

// --------------------------------------------------------------------------------------------------
// Work plan: the N_D x N_R rectangle (DR) or the i<j triangle (DD, RR) cut into items of one kTileI-row
// i-block times up to `chunk` kTileJ-column j-tiles (north_star "triangular tiles").
// --------------------------------------------------------------------------------------------------
void make_plan(bool tri, uint64_t n_i, uint64_t n_j, int sm_count, Plan& p) {
    p = Plan();
    p.tri = tri;
    p.n_i = n_i;
    p.n_j = tri ? n_i : n_j;
    p.blocks_i = (uint32_t)((n_i + kTileI - 1) / kTileI);
    p.tiles_j = (uint32_t)((p.n_j + kTileJ - 1) / kTileJ);
    uint64_t tiles = tri ? (uint64_t)p.blocks_i * (p.blocks_i + 1) / 2 : (uint64_t)p.blocks_i * p.tiles_j;
    uint64_t c = tiles / (160ull * (uint64_t)std::max(sm_count, 1));
    p.chunk = (uint32_t)std::min<uint64_t>(std::max<uint64_t>(c, 1), kMaxChunk);
    if (tri) {
        p.row_start.resize((size_t)p.blocks_i + 1);
        uint64_t acc = 0;
        for (uint32_t I = 0; I < p.blocks_i; ++I) {
            p.row_start[I] = (uint32_t)acc;
            acc += (p.tiles_j - I + p.chunk - 1) / p.chunk;
        }
        p.row_start[p.blocks_i] = (uint32_t)acc;
        p.n_items = acc;
    } else {
        p.n_items = (uint64_t)p.blocks_i * ((p.tiles_j + p.chunk - 1) / p.chunk);
    }
}

void Plan::item(uint64_t w, uint32_t& I, uint32_t& tile0, uint32_t& ntiles) const {
    if (tri) {
        uint32_t lo = 0, hi = blocks_i;     // row_start[lo] <= w < row_start[hi]
        while (hi - lo > 1) {
            uint32_t mid = (lo + hi) >> 1;
            if (row_start[mid] <= w) lo = mid; else hi = mid;
        }
        I = lo;
        uint32_t c = (uint32_t)(w - row_start[lo]);
        tile0 = I + c * chunk;
        ntiles = std::min(chunk, tiles_j - tile0);
    } else {
        uint32_t per_row = (tiles_j + chunk - 1) / chunk;
        I = (uint32_t)(w / per_row);
        uint32_t c = (uint32_t)(w % per_row);
        tile0 = c * chunk;
        ntiles = std::min(chunk, tiles_j - tile0);
    }
}

uint64_t Plan::item_pairs(uint64_t w) const {
    uint32_t I, t0, nt;
    item(w, I, t0, nt);
    uint64_t rows = std::min<uint64_t>(kTileI, n_i - (uint64_t)I * kTileI), total = 0;
    for (uint32_t t = t0; t < t0 + nt; ++t) {
        uint64_t cols = std::min<uint64_t>(kTileJ, n_j - (uint64_t)t * kTileJ);
        total += (tri && t == I) ? rows * (rows - 1) / 2 : rows * cols;
    }
    return total;
}

// PAPER.md:20-25 Eq. 1 in the pair-count-normalised reading A1 (BASELINE.json north_star).
void estimate(const uint64_t* dd, const uint64_t* dr, const uint64_t* rr, int nbins, uint64_t n_d, uint64_t n_r,
              double* w) {
    const double ndd = 0.5 * (double)n_d * ((double)n_d - 1.0);
    const double ndr = (double)n_d * (double)n_r;
    const double nrr = 0.5 * (double)n_r * ((double)n_r - 1.0);
    for (int k = 0; k < nbins; ++k) {
        if (rr[k] == 0) { w[k] = std::numeric_limits<double>::quiet_NaN(); continue; }
        const double frr = (double)rr[k] / nrr;
        w[k] = ((double)dd[k] / ndd - 2.0 * ((double)dr[k] / ndr) + frr) / frr;
    }
}

}  // namespace tpcf
