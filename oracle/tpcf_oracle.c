/*
 * tpcf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision brute-force oracle for the angular pair counts DD, DR, RR and the
 * Landy-Szalay estimator of arXiv:1204.6630 (reference text: PAPER.md).  It is the *definition*
 * of the result written out: for every pair, dot product -> arc-cosine -> theta -> bin, exactly the
 * two operations the paper names for its kernels (Section 3, first bullet), filling
 * the three histograms of PAPER.md:25/38 (Eq. 1 and Section 3, second bullet).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or constant with paper_1204_6630_b200/.
 *
 * Readings of the paper where it is silent (restated in DESIGN.md):
 *   A3  DD/RR count unordered pairs i<j; DR counts all N_D*N_R ordered pairs.
 *   A5  bin k = [e_k, e_{k+1}) in theta, last bin closed at e_n (numpy.histogram convention).
 *   A7  the dot product is clamped to [-1, 1] before acos.
 *   A8  RA/Dec in degrees; x = cos(dec)cos(ra), y = cos(dec)sin(ra), z = sin(dec).
 *   A1  estimator in pair-normalised form (BASELINE.json north_star), see orc_estimate.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): hand catalogs P1, totals P2,
 * numpy.histogram of arccos of a Gram matrix P3, great-circle ring closed form P4, integer
 * identities P5, uniform-sphere closed form P6, null test P7, Eq. 1 hand case P8 (cross estimator: hand case 3/4,
 * w12 = 1/N identity and null test, P8x), acos-vs-asin P9;
 * 3-D variant (orc_count_*_xyz): cubic-lattice multiplicities X1, totals X2, unit-cube distance
 * distribution X3, unit vectors with chord edges reproduce the angular histogram X4.
 * Three-point counts (orc_count_triples): octahedron and equator hand triples, total C(N,3), row permutation,
 * side-marginal identity against orc_count_auto, brute-force numpy on 40 points (T1-T5).
 * Unpinned: absolute w(theta) values on the MICE catalogs / Fig. 1 (data not available).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared tpcf_oracle.c -o libtpcf_oracle.so -lm
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* O2 (A8): RA, Dec in degrees -> unit vector.  radec is n rows x 2, xyz is n rows x 3. */
void orc_radec_to_xyz(const double *radec, size_t n, double *xyz)
{
    for (size_t i = 0; i < n; ++i) {
        double alpha = radec[2 * i] * M_PI / 180.0;
        double delta = radec[2 * i + 1] * M_PI / 180.0;
        xyz[3 * i + 0] = cos(delta) * cos(alpha);
        xyz[3 * i + 1] = cos(delta) * sin(alpha);
        xyz[3 * i + 2] = sin(delta);
    }
}

/* O5 (A5): slot 0 = under (theta < e_0), slots 1..n = bins, slot n+1 = over (theta > e_n). */
static int bin_slot(double theta, const double *e, int n)
{
    if (theta < e[0]) return 0;
    if (theta > e[n]) return n + 1;
    int lo = 0, hi = n; /* invariant: e[lo] <= theta, and (hi == n or theta < e[hi]) */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (e[mid] <= theta) lo = mid; else hi = mid;
    }
    return lo + 1; /* largest k with e_k <= theta, capped at n-1 */
}

/* One pair: O4 (dot, clamp A7, acos), O5 (bin), optional O6 (near-edge counters), optional O8. */
static inline void one_pair(const double *a, const double *b, const double *e, const double *cose, int n,
                            uint64_t *hist, uint64_t *near, uint64_t *mismatch)
{
    double s = a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
    if (s > 1.0) s = 1.0;
    if (s < -1.0) s = -1.0;
    double theta = acos(s) * 180.0 / M_PI;
    int slot = bin_slot(theta, e, n);
    ++hist[slot];
    if (near) {
        /* O6: ++near[k] for every edge k with |s - cos(e_k)| <= 1e-6 (BASELINE.json tolerance).
         * cos(e_k) decreases with k, so the edges that qualify are one contiguous run: find its
         * start by bisection and walk it (same set as testing every k). */
        int lo = 0, hi = n + 1; /* first k with cose[k] <= s + 1e-6 */
        while (lo < hi) {
            int mid = (lo + hi) / 2;
            if (cose[mid] <= s + 1e-6) hi = mid; else lo = mid + 1;
        }
        for (int k = (lo > 0 ? lo - 1 : 0); k <= n && cose[k] >= s - 2e-6; ++k) /* generous window */
            if (fabs(s - cose[k]) <= 1e-6) ++near[k];                          /* the defining test */
    }
    if (mismatch) {
        /* O8 / P9: theta' = 2 asin(|a-b|/2), well conditioned at small theta; must bin identically. */
        double dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
        double h = 0.5 * sqrt(dx * dx + dy * dy + dz * dz);
        if (h > 1.0) h = 1.0;
        double theta2 = 2.0 * asin(h) * 180.0 / M_PI;
        if (bin_slot(theta2, e, n) != slot) ++*mismatch;
    }
}

#define MAX_EDGES 4100

static int prep(const double *e, int n, double *cose)
{
    if (n < 1 || n + 1 > MAX_EDGES) return -1;
    for (int k = 0; k <= n; ++k) cose[k] = cos(e[k] * M_PI / 180.0);
    return 0;
}

/*
 * Auto-pairs (DD, RR): all i<j with i in [i_begin, i_end) (A3).  hist has n+2 slots and is
 * ACCUMULATED into (caller zeroes it); near has n+1 slots or is NULL; mismatch is one counter or NULL.
 */
int orc_count_auto(const double *xyz, size_t npts, size_t i_begin, size_t i_end, const double *edges, int nbins,
                   uint64_t *hist, uint64_t *near, uint64_t *mismatch)
{
    double cose[MAX_EDGES];
    if (prep(edges, nbins, cose)) return -1;
    for (size_t i = i_begin; i < i_end && i < npts; ++i)
        for (size_t j = i + 1; j < npts; ++j)
            one_pair(xyz + 3 * i, xyz + 3 * j, edges, cose, nbins, hist, near, mismatch);
    return 0;
}

/* Cross-pairs (DR): all (i, j), i in [i_begin, i_end) of a, every j of b. */
int orc_count_cross(const double *a, size_t na, size_t i_begin, size_t i_end, const double *b, size_t nb,
                    const double *edges, int nbins, uint64_t *hist, uint64_t *near, uint64_t *mismatch)
{
    double cose[MAX_EDGES];
    if (prep(edges, nbins, cose)) return -1;
    for (size_t i = i_begin; i < i_end && i < na; ++i)
        for (size_t j = 0; j < nb; ++j)
            one_pair(a + 3 * i, b + 3 * j, edges, cose, nbins, hist, near, mismatch);
    return 0;
}

/*
 * Row-subset mode: sum over i in rows[r_begin..r_end) of all j in b; with
 * exclude_self != 0 (a and b are the same catalog) the pair j == rows[r] is skipped, so the total is
 * nrows*(N-1) and both sides of the diagonal are counted.
 */
int orc_count_rows(const double *a, const int64_t *rows, size_t r_begin, size_t r_end, const double *b, size_t nb,
                   int exclude_self, const double *edges, int nbins, uint64_t *hist, uint64_t *near,
                   uint64_t *mismatch)
{
    double cose[MAX_EDGES];
    if (prep(edges, nbins, cose)) return -1;
    for (size_t r = r_begin; r < r_end; ++r) {
        size_t i = (size_t)rows[r];
        for (size_t j = 0; j < nb; ++j) {
            if (exclude_self && j == i) continue;
            one_pair(a + 3 * i, b + 3 * j, edges, cose, nbins, hist, near, mismatch);
        }
    }
    return 0;
}

/*
 * Three-point counts ("extending the work to higher order correlation functions",
 * PAPER.md:89).  The paper names the extension and gives no formula; the plain definition used here (DESIGN.md
 * section 15): every unordered triple i<j<k of one catalog is a spherical triangle with the three side angles
 * theta_ij, theta_ik, theta_jk, each computed exactly as a pair is (O4: dot, clamp, acos) and put in a slot exactly as a
 * pair is (O5: slot 0 = under, 1..n = bins, n+1 = over).  The triple is counted once, in cell (a, b, c) of a dense
 * (n+2)^3 array, a <= b <= c the three slots in ascending order: hist3[(a*(n+2) + b)*(n+2) + c].  Hence
 *   sum(hist3) = N(N-1)(N-2)/6 exactly, and
 *   for every slot s:  sum over cells of hist3[a,b,c] * ([a==s] + [b==s] + [c==s]) = (N-2) * (pairs in slot s),
 * because every pair is a side of exactly N-2 triples.  i runs over [i_begin, i_end) so that callers can split the work;
 * hist3 is ACCUMULATED into.  No blocking, no pair-slot table: each side is recomputed from its two points.
 */
int orc_count_triples(const double *xyz, size_t npts, size_t i_begin, size_t i_end, const double *edges, int nbins,
                      uint64_t *hist3)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    const size_t m = (size_t)nbins + 2;
    for (size_t i = i_begin; i < i_end && i < npts; ++i)
        for (size_t j = i + 1; j < npts; ++j)
            for (size_t k = j + 1; k < npts; ++k) {
                const double *p[3] = {xyz + 3 * i, xyz + 3 * j, xyz + 3 * k};
                int slot[3];
                for (int side = 0; side < 3; ++side) {          /* sides ij, ik, jk */
                    const double *a = p[side == 2 ? 1 : 0], *b = p[side == 0 ? 1 : 2];
                    double s = a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
                    if (s > 1.0) s = 1.0;
                    if (s < -1.0) s = -1.0;
                    slot[side] = bin_slot(acos(s) * 180.0 / M_PI, edges, nbins);
                }
                /* ascending order of the three slots */
                if (slot[0] > slot[1]) { int t = slot[0]; slot[0] = slot[1]; slot[1] = t; }
                if (slot[1] > slot[2]) { int t = slot[1]; slot[1] = slot[2]; slot[2] = t; }
                if (slot[0] > slot[1]) { int t = slot[0]; slot[0] = slot[1]; slot[1] = t; }
                ++hist3[((size_t)slot[0] * m + (size_t)slot[1]) * m + (size_t)slot[2]];
            }
    return 0;
}

/*
 * O7: Landy-Szalay in pair-count-normalised form (Eq. 1, whose extraction lost the
 * square on N_random/N_real -- reading A1; form fixed by BASELINE.json north_star):
 *   w_k = (DD_k/nDD - 2 DR_k/nDR + RR_k/nRR) / (RR_k/nRR),
 *   nDD = N_D(N_D-1)/2, nDR = N_D N_R, nRR = N_R(N_R-1)/2;  RR_k = 0 -> NaN (A14).
 * dd, dr, rr point at the nbins in-range counts (no under/over slots).
 */
void orc_estimate(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, int nbins, uint64_t n_d, uint64_t n_r,
                  double *w)
{
    double ndd = 0.5 * (double)n_d * ((double)n_d - 1.0);
    double ndr = (double)n_d * (double)n_r;
    double nrr = 0.5 * (double)n_r * ((double)n_r - 1.0);
    for (int k = 0; k < nbins; ++k) {
        if (rr[k] == 0) { w[k] = NAN; continue; }
        double fdd = (double)dd[k] / ndd, fdr = (double)dr[k] / ndr, frr = (double)rr[k] / nrr;
        w[k] = (fdd - 2.0 * fdr + frr) / frr;
    }
}

/*
 * Cross-correlation of two data catalogs D1, D2 against one random catalog R (PAPER.md:16
 * "cross-correlation"; the form of Eq. 1, with the data-data term split over the two catalogs):
 *   w12_k = (D1D2_k/n12 - D1R_k/n1r - D2R_k/n2r + RR_k/nrr) / (RR_k/nrr),
 *   n12 = N_1 N_2, n1r = N_1 N_R, n2r = N_2 N_R (all ordered pairs), nrr = N_R(N_R-1)/2;  RR_k = 0 -> NaN (A14).
 * With D2 = D1 = D this is NOT orc_estimate (D1D2 would count ordered pairs and self-pairs); it is its own definition.
 * Pins: hand case 3/4, null test, sign test of each cross term (tests/test_oracle_pins.py).
 */
void orc_estimate_cross(const uint64_t *d1d2, const uint64_t *d1r, const uint64_t *d2r, const uint64_t *rr, int nbins,
                        uint64_t n_1, uint64_t n_2, uint64_t n_r, double *w)
{
    double n12 = (double)n_1 * (double)n_2;
    double n1r = (double)n_1 * (double)n_r;
    double n2r = (double)n_2 * (double)n_r;
    double nrr = 0.5 * (double)n_r * ((double)n_r - 1.0);
    for (int k = 0; k < nbins; ++k) {
        if (rr[k] == 0) { w[k] = NAN; continue; }
        double f12 = (double)d1d2[k] / n12, f1r = (double)d1r[k] / n1r, f2r = (double)d2r[k] / n2r;
        double frr = (double)rr[k] / nrr;
        w[k] = (f12 - f1r - f2r + frr) / frr;
    }
}

/*
 * ---- 3-D variant ("results are extendible to the 3-dimensional variant as well") ----
 * The spatial two-point function xi(r) needs the same three histograms with the Euclidean separation
 * r = |a - b| of Cartesian positions in place of the angle.  Definition written out: r in fp64 by
 * sqrt(dx^2 + dy^2 + dz^2), bins [e_k, e_{k+1}) in r, last bin closed (A5), under = r < e_0,
 * over = r > e_n.  near[k] counts the pairs with |r - e_k| <= near_tol (the checker's tolerance for
 * pairs a different rounding order may put on the other side of an edge).
 */
static inline void one_pair_xyz(const double *a, const double *b, const double *e, int n, double near_tol,
                                uint64_t *hist, uint64_t *near)
{
    double dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
    double r = sqrt(dx * dx + dy * dy + dz * dz);
    ++hist[bin_slot(r, e, n)];
    if (near)
        for (int k = 0; k <= n; ++k)
            if (fabs(r - e[k]) <= near_tol) ++near[k];
}

int orc_count_auto_xyz(const double *xyz, size_t npts, size_t i_begin, size_t i_end, const double *edges, int nbins,
                       double near_tol, uint64_t *hist, uint64_t *near)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    for (size_t i = i_begin; i < i_end && i < npts; ++i)
        for (size_t j = i + 1; j < npts; ++j)
            one_pair_xyz(xyz + 3 * i, xyz + 3 * j, edges, nbins, near_tol, hist, near);
    return 0;
}

int orc_count_cross_xyz(const double *a, size_t na, size_t i_begin, size_t i_end, const double *b, size_t nb,
                        const double *edges, int nbins, double near_tol, uint64_t *hist, uint64_t *near)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    for (size_t i = i_begin; i < i_end && i < na; ++i)
        for (size_t j = 0; j < nb; ++j)
            one_pair_xyz(a + 3 * i, b + 3 * j, edges, nbins, near_tol, hist, near);
    return 0;
}

int orc_count_rows_xyz(const double *a, const int64_t *rows, size_t r_begin, size_t r_end, const double *b, size_t nb,
                       int exclude_self, const double *edges, int nbins, double near_tol, uint64_t *hist,
                       uint64_t *near)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    for (size_t r = r_begin; r < r_end; ++r) {
        size_t i = (size_t)rows[r];
        for (size_t j = 0; j < nb; ++j) {
            if (exclude_self && j == i) continue;
            one_pair_xyz(a + 3 * i, b + 3 * j, edges, nbins, near_tol, hist, near);
        }
    }
    return 0;
}

/*
 * ---- weighted counts (cross-correlations of galaxy positions with weighted quantities such as shear;
 * extensions named as future work) ----
 * Every object carries a weight; the histogram holds, per theta bin, the sum over the pairs of w_i * w_j instead of the
 * number of pairs.  Definition written out: the pair's bin exactly as in one_pair (dot -> clamp -> acos -> degrees ->
 * bin_slot), the product w_i * w_j in fp64, added to the bin's fp64 sum in the loop's order (i ascending, j ascending).
 * wsum has n+2 slots {under, bins, over} and is ACCUMULATED into; asum, if not NULL, accumulates |w_i * w_j| the same way
 * (the scale of the checker's tolerance: a different summation order changes a sum of m terms by at most
 * (m - 1) 2^-53 sum |terms|).
 */
int orc_wsum_auto(const double *xyz, const double *w, size_t npts, size_t i_begin, size_t i_end, const double *edges,
                  int nbins, double *wsum, double *asum)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    for (size_t i = i_begin; i < i_end && i < npts; ++i)
        for (size_t j = i + 1; j < npts; ++j) {
            const double *a = xyz + 3 * i, *b = xyz + 3 * j;
            double s = a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
            if (s > 1.0) s = 1.0;
            if (s < -1.0) s = -1.0;
            int slot = bin_slot(acos(s) * 180.0 / M_PI, edges, nbins);
            double t = w[i] * w[j];
            wsum[slot] += t;
            if (asum) asum[slot] += fabs(t);
        }
    return 0;
}

int orc_wsum_cross(const double *a, const double *wa, size_t na, size_t i_begin, size_t i_end, const double *b,
                   const double *wb, size_t nb, const double *edges, int nbins, double *wsum, double *asum)
{
    if (nbins < 1 || nbins + 1 > MAX_EDGES) return -1;
    for (size_t i = i_begin; i < i_end && i < na; ++i)
        for (size_t j = 0; j < nb; ++j) {
            const double *p = a + 3 * i, *q = b + 3 * j;
            double s = p[0] * q[0] + p[1] * q[1] + p[2] * q[2];
            if (s > 1.0) s = 1.0;
            if (s < -1.0) s = -1.0;
            int slot = bin_slot(acos(s) * 180.0 / M_PI, edges, nbins);
            double t = wa[i] * wb[j];
            wsum[slot] += t;
            if (asum) asum[slot] += fabs(t);
        }
    return 0;
}
