/*
 * smre_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU statement of what the hot path of
 * arXiv 1503.03492 computes: Dykstra's projection of a residual image onto the
 * intersection of the window balls  ||x_S||^2 <= c_S  (Eq. 5),
 * in the standard form (Alg. 2) and in the paper's
 * "incomplete" form (Sec. 3.2 + Listing 2/3).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may call this file.  It shares no code, header, table
 * or helper with the CUDA path under paper_1503_03492_b200/csrc/.
 *
 * Notation: thresholds c_S = 1 / c_s(alpha) of the paper;
 * increment sign  v = x + q  (q here = -q of Alg. 2; negation is exact).
 *
 * Every loop below is window-serial and in the order the paper / DESIGN.md
 * readings state; no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py): closed-form single ball (Eq. 14), identity on
 * feasible input, one-family == one projection, side-1 == clip, conservation
 * x + sum_f q_f == y, feasibility in the limit, variational inequality, KKT
 * structure, SLSQP brute force on tiny images, box-cap-ball closed form,
 * symmetries, ICD == composition of restricted standard runs == explicit
 * tile-by-tile solve, counts, the all-windows checker against a strided-view
 * sum, the stop rules of the tolerance modes against fixed-count runs and an
 * independent tile-wise solve; the PSF operator against scipy and the 2-D
 * definition, the ADMM against the problem it solves (projection limit, KKT
 * system, SLSQP).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------------------
 * One window step.  Eq. 14 with c_S = 1/c_s:
 *     p_s(v) = v * sqrt(c_S / ||v||^2)  if ||v||^2 > c_S   (strict, A5)
 *              v                         else
 * applied to v = x + q (Listing 3: s1 = e - q, paper sign), then
 * q' = v - p_s(v)   (Listing 3, PAPER.md:502 + 510: q = -s1; q += s1_scaled).
 * The sum of squares runs row-major over the window.
 * Returns 1 when the window was scaled (constraint active), else 0.
 * ------------------------------------------------------------------------- */
static int window_step(double *x, double *q, int W, int wy, int wx, int s, double c)
{
    double n2 = 0.0;
    for (int r = wy; r < wy + s; ++r)
        for (int col = wx; col < wx + s; ++col) {
            double v = x[(size_t)r * W + col] + q[(size_t)r * W + col];
            n2 += v * v;
        }
    double alpha = 1.0;
    int active = 0;
    if (n2 > c) {
        alpha = sqrt(c / n2);
        active = 1;
    }
    for (int r = wy; r < wy + s; ++r)
        for (int col = wx; col < wx + s; ++col) {
            size_t i = (size_t)r * W + col;
            double v = x[i] + q[i];
            double xn = alpha * v;
            q[i] = v - xn;
            x[i] = xn;
        }
    return active;
}

/* One family pass: every window of side s with origin == (oy, ox) mod s that
 * lies fully inside the H x W image (reading A6).  The windows of a family are
 * disjoint, so their order is irrelevant; row-major here. */
static long long family_pass(double *x, double *q, int H, int W,
                             int s, int oy, int ox, double c)
{
    long long n_active = 0;
    for (int wy = oy; wy + s <= H; wy += s)
        for (int wx = ox; wx + s <= W; wx += s)
            n_active += window_step(x, q, W, wy, wx, s, c);
    return n_active;
}

/* ---------------------------------------------------------------------------
 * Cyclic Dykstra over an explicit ordered family list (Alg. 2, PAPER.md:178,
 * read as A1/A2: one step per set, sets visited cyclically, one sweep = one
 * pass over the list).  q_f = 0 initially for every f.
 *   y      : H*W row-major input
 *   fam_*  : F entries: side, row offset, column offset, threshold
 *   x_out  : H*W result
 *   q_out  : NULL, or F*H*W increments after the last sweep (plane f = family f)
 *   n_active_last : NULL, or number of scaled windows during the last sweep
 * Returns 0, or -1 on allocation failure / bad arguments.
 * ------------------------------------------------------------------------- */
int smre_oracle_dykstra_families(const double *y, int H, int W,
                                 const int *fam_side, const int *fam_oy,
                                 const int *fam_ox, const double *fam_c, int F,
                                 int n_sweeps, double *x_out, double *q_out,
                                 long long *n_active_last)
{
    if (!y || !x_out || H <= 0 || W <= 0 || F < 0 || n_sweeps < 0) return -1;
    size_t N = (size_t)H * W;
    double *q = q_out;
    if (!q) {
        q = (double *)malloc(sizeof(double) * N * (size_t)(F > 0 ? F : 1));
        if (!q) return -1;
    }
    memset(q, 0, sizeof(double) * N * (size_t)F);
    if (x_out != y) memcpy(x_out, y, sizeof(double) * N);
    long long act = 0;
    for (int sweep = 0; sweep < n_sweeps; ++sweep) {
        act = 0;
        for (int f = 0; f < F; ++f)
            act += family_pass(x_out, q + (size_t)f * N, H, W,
                               fam_side[f], fam_oy[f], fam_ox[f], fam_c[f]);
    }
    if (n_active_last) *n_active_last = act;
    if (!q_out) free(q);
    return 0;
}

/* Number of families of the standard ("exact") method: sum of s^2. */
int smre_oracle_std_family_count(const int *sides, int n_sides)
{
    int F = 0;
    for (int a = 0; a < n_sides; ++a) F += sides[a] * sides[a];
    return F;
}

/* Canonical family order, reading A3: sides[] as given, then oy ascending,
 * then ox ascending.  Arrays must hold smre_oracle_std_family_count entries. */
void smre_oracle_std_family_list(const int *sides, const double *c, int n_sides,
                                 int *fam_side, int *fam_oy, int *fam_ox, double *fam_c)
{
    int f = 0;
    for (int a = 0; a < n_sides; ++a)
        for (int oy = 0; oy < sides[a]; ++oy)
            for (int ox = 0; ox < sides[a]; ++ox) {
                fam_side[f] = sides[a];
                fam_oy[f] = oy;
                fam_ox[f] = ox;
                fam_c[f] = c[a];
                ++f;
            }
}

/* ---------------------------------------------------------------------------
 * Algorithm O-STD: the "exact method" window set, all square
 * windows of every side in sides[] at every shift, n_sweeps
 * sweeps in the canonical order.  q_out: NULL or F*H*W.
 * ------------------------------------------------------------------------- */
int smre_oracle_std(const double *y, int H, int W, const int *sides, const double *c,
                    int n_sides, int n_sweeps, double *x_out, double *q_out,
                    long long *n_active_last)
{
    if (!sides || !c || n_sides <= 0) return -1;
    int F = smre_oracle_std_family_count(sides, n_sides);
    int *fs = (int *)malloc(sizeof(int) * 3 * (size_t)F);
    double *fc = (double *)malloc(sizeof(double) * (size_t)F);
    if (!fs || !fc) { free(fs); free(fc); return -1; }
    smre_oracle_std_family_list(sides, c, n_sides, fs, fs + F, fs + 2 * F, fc);
    int rc = smre_oracle_dykstra_families(y, H, W, fs, fs + F, fs + 2 * F, fc, F,
                                          n_sweeps, x_out, q_out, n_active_last);
    free(fs);
    free(fc);
    return rc;
}

/* ---------------------------------------------------------------------------
 * Algorithm O-ICD, the paper's incomplete Dykstra:
 *   window collection: squares of edge 2^k, k <= K, shifted by
 *   2^i "in each direction" (diagonal, Listing 2 PAPER.md:393,
 *   reading A-ICD-4/5);  Omega^i = all levels k >= i at shift 2^i
 *   (union of collections, reading A-ICD-1);
 *   P_incomplete = product over i = 0..K of P_{Omega^i} (PAPER.md:377,
 *   A-ICD-2), applied i ascending (Listing 2, A-ICD-3).
 * Each P_{Omega^i} is a Dykstra run from q = 0 (Listing 3 PAPER.md:431-433,
 * A-ICD-9) over the levels K, K-1, ..., i in that order (PAPER.md:453,
 * A-ICD-10), repeated n_sweeps times (reading A-ICD-8: the paper's
 * "while delta > tol*1024" loop is replaced by a fixed count).
 * Borders (A-ICD-13): a level is the tiling of the whole plane with origin
 * (2^i mod 2^k) on the diagonal, restricted to windows fully inside the image.
 *
 *   level_c[k] : threshold of side 2^k, k = 0..K
 * ------------------------------------------------------------------------- */
int smre_oracle_icd_levels(const double *y, int H, int W, int K, const double *level_c,
                           int n_sweeps, double *x_out)
{
    if (!y || !x_out || !level_c || H <= 0 || W <= 0 || K < 0 || K > 30 || n_sweeps < 0)
        return -1;
    size_t N = (size_t)H * W;
    double *q = (double *)malloc(sizeof(double) * N * (size_t)(K + 1));
    if (!q) return -1;
    if (x_out != y) memcpy(x_out, y, sizeof(double) * N);
    for (int i = 0; i <= K; ++i) {                    /* shift loop, Listing 2 */
        int shift = 1 << i;
        memset(q, 0, sizeof(double) * N * (size_t)(K + 1));   /* "Set q = 0" */
        for (int cyc = 0; cyc < n_sweeps; ++cyc)
            for (int k = K; k >= i; --k) {            /* for (s = 5; s >= smin; s--) */
                int side = 1 << k;
                int o = shift % side;                  /* offset (o, o) */
                family_pass(x_out, q + (size_t)k * N, H, W, side, o, o, level_c[k]);
            }
    }
    free(q);
    return 0;
}

/* Front end taking the same (sides, c) table as the standard variant:
 * K = floor(log2(max side)) (Eq. 21, reading A-ICD-6); every 2^k,
 * k <= K, must be present in sides[] (else -2); other sides are ignored
 * (reading A-ICD-7). */
int smre_oracle_icd(const double *y, int H, int W, const int *sides, const double *c,
                    int n_sides, int n_sweeps, double *x_out)
{
    if (!sides || !c || n_sides <= 0) return -1;
    int smax = 0;
    for (int a = 0; a < n_sides; ++a) if (sides[a] > smax) smax = sides[a];
    if (smax < 1) return -1;
    int K = 0;
    while ((2 << K) <= smax) ++K;
    double level_c[32];
    for (int k = 0; k <= K; ++k) {
        int found = 0;
        for (int a = 0; a < n_sides; ++a)
            if (sides[a] == (1 << k)) { level_c[k] = c[a]; found = 1; break; }
        if (!found) return -2;
    }
    return smre_oracle_icd_levels(y, H, W, K, level_c, n_sweeps, x_out);
}

/* ---------------------------------------------------------------------------
 * Sum of squares of EVERY s x s window fully inside the image (all shifts),
 * by direct summation: out[(H-s+1)*(W-s+1)], out[wy*(W-s+1)+wx] = t_s of the
 * window with origin (wy, wx)  (t_s).  Used by the tests to form
 * the violated-window sets of the parity protocol.
 * ------------------------------------------------------------------------- */
int smre_oracle_window_sums(const double *x, int H, int W, int s, double *out)
{
    if (!x || !out || s < 1 || s > H || s > W) return -1;
    int nwy = H - s + 1, nwx = W - s + 1;
    for (int wy = 0; wy < nwy; ++wy)
        for (int wx = 0; wx < nwx; ++wx) {
            double n2 = 0.0;
            for (int r = wy; r < wy + s; ++r)
                for (int col = wx; col < wx + s; ++col) {
                    double v = x[(size_t)r * W + col];
                    n2 += v * v;
                }
            out[(size_t)wy * nwx + wx] = n2;
        }
    return 0;
}

/* ===========================================================================
 * Convergence-controlled runs: the paper never runs a
 * fixed sweep count.
 *
 * Standard variant, Alg. 2: "while ||x_r - x_{r-1}||_2^2 >
 * delta".  Reading A4': r counts SWEEPS (one pass over all families, reading
 * A2), x_r is the image after sweep r, x_0 = y; the run stops after the first
 * sweep r >= 1 with ||x_r - x_{r-1}||^2 <= delta, or after max_sweeps.
 * *sweeps_done receives r.  The square sum runs row-major over the image.
 * ------------------------------------------------------------------------- */
int smre_oracle_std_tol(const double *y, int H, int W, const int *sides, const double *c,
                        int n_sides, int max_sweeps, double delta, double *x_out,
                        int *sweeps_done)
{
    if (!y || !x_out || !sides || !c || n_sides <= 0 || H <= 0 || W <= 0 || max_sweeps < 1)
        return -1;
    int F = smre_oracle_std_family_count(sides, n_sides);
    size_t N = (size_t)H * W;
    int *fs = (int *)malloc(sizeof(int) * 3 * (size_t)F);
    double *fc = (double *)malloc(sizeof(double) * (size_t)F);
    double *q = (double *)calloc(N * (size_t)F, sizeof(double));
    double *prev = (double *)malloc(sizeof(double) * N);
    if (!fs || !fc || !q || !prev) { free(fs); free(fc); free(q); free(prev); return -1; }
    smre_oracle_std_family_list(sides, c, n_sides, fs, fs + F, fs + 2 * F, fc);
    if (x_out != y) memcpy(x_out, y, sizeof(double) * N);
    int r = 0;
    for (;;) {
        memcpy(prev, x_out, sizeof(double) * N);                 /* x_{r-1} */
        for (int f = 0; f < F; ++f)
            family_pass(x_out, q + (size_t)f * N, H, W, fs[f], fs[F + f], fs[2 * F + f], fc[f]);
        ++r;
        double d2 = 0.0;
        for (size_t i = 0; i < N; ++i) {
            double d = x_out[i] - prev[i];
            d2 += d * d;
        }
        if (!(d2 > delta) || r >= max_sweeps) break;             /* while ||x_r - x_{r-1}||^2 > delta */
    }
    if (sweeps_done) *sweeps_done = r;
    free(fs); free(fc); free(q); free(prev);
    return 0;
}

/* ---------------------------------------------------------------------------
 * Incomplete variant with the stop rule of Listing 3:
 * every thread block iterates ITS tile "while (delta > tol*1024)", where delta
 * collects mabs(e_old - e_new) of the block's pixels over all levels of one
 * cycle and 1024 is the number of pixels of the paper's 32 x 32 tile.
 * Readings (DESIGN.md A-ICD-16): the tile is the L x L square, L = 2^K, of the
 * tiling with origin (2^i mod L) on the diagonal (virtual tiles overhang the
 * border, A-ICD-13); delta = sum over the levels K..i of one cycle and over the
 * tile's pixels inside the image of |x_old - x_new| (the block-wide reduction
 * the listing elides, A-ICD-11); a tile stops after the first cycle with
 * delta <= tol * L^2, or after max_cycles.  Tiles are independent (all windows
 * of a shift nest inside its tiles), so this is tile-serial.
 *   cycles_total : NULL or sum over shifts and tiles of the cycles run
 *   cycles_max   : NULL or the largest cycle count of any tile
 * ------------------------------------------------------------------------- */
static int icd_levels_tol_impl(const double *y, int H, int W, int K, const double *level_c,
                               int max_cycles, double tol, double *x_out,
                               long long *cycles_total, int *cycles_max,
                               int *tile_cycles_out, const int *tile_cycles_in, double band,
                               long long *n_bad);

int smre_oracle_icd_levels_tol(const double *y, int H, int W, int K, const double *level_c,
                               int max_cycles, double tol, double *x_out,
                               long long *cycles_total, int *cycles_max)
{
    return icd_levels_tol_impl(y, H, W, K, level_c, max_cycles, tol, x_out, cycles_total, cycles_max,
                               NULL, NULL, 0.0, NULL);
}

/* Number of tiles along an axis of extent N for shift i (tile edge L): origins o - L, o, o + L, ...
 * with o = 2^i mod L, those with origin + L <= 0 left out. */
int smre_oracle_icd_tiles_along(int N, int K, int i)
{
    const int L = 1 << K, o = (1 << i) % L;
    int n = 0;
    for (int t = o - L; t < N; t += L)
        if (t + L > 0) ++n;
    return n;
}

/* Same run, additionally writing the cycles every tile ran: tile_cycles_out, shift-major, per shift
 * [tiles along y][tiles along x] (smre_oracle_icd_tiles_along). */
int smre_oracle_icd_levels_tol_counts(const double *y, int H, int W, int K, const double *level_c,
                                      int max_cycles, double tol, double *x_out, int *tile_cycles_out)
{
    return icd_levels_tol_impl(y, H, W, K, level_c, max_cycles, tol, x_out, NULL, NULL,
                               tile_cycles_out, NULL, 0.0, NULL);
}

/* REPLAY of somebody else's stop decisions (the fp32 kernel's): every tile runs exactly the cycles
 * tile_cycles_in prescribes (same layout), and the fp64 deltas are checked against those decisions
 * within a relative band: a tile that ran c cycles must have had delta > tol L^2 (1 - band) after
 * every cycle before c, and delta <= tol L^2 (1 + band) after cycle c unless c == max_cycles.
 * *n_bad counts the tiles whose count the band does not allow. */
int smre_oracle_icd_levels_replay(const double *y, int H, int W, int K, const double *level_c,
                                  int max_cycles, double tol, const int *tile_cycles_in, double band,
                                  double *x_out, long long *n_bad)
{
    if (!tile_cycles_in || !n_bad) return -1;
    return icd_levels_tol_impl(y, H, W, K, level_c, max_cycles, tol, x_out, NULL, NULL,
                               NULL, tile_cycles_in, band, n_bad);
}

static int icd_levels_tol_impl(const double *y, int H, int W, int K, const double *level_c,
                               int max_cycles, double tol, double *x_out,
                               long long *cycles_total, int *cycles_max,
                               int *tile_cycles_out, const int *tile_cycles_in, double band,
                               long long *n_bad)
{
    if (!y || !x_out || !level_c || H <= 0 || W <= 0 || K < 0 || K > 12 || max_cycles < 1)
        return -1;
    const int L = 1 << K;
    size_t N = (size_t)H * W;
    double *q = (double *)malloc(sizeof(double) * N * (size_t)(K + 1));
    double *tmp = (double *)malloc(sizeof(double) * (size_t)L * L);
    if (!q || !tmp) { free(q); free(tmp); return -1; }
    if (x_out != y) memcpy(x_out, y, sizeof(double) * N);
    long long total = 0, bad = 0;
    size_t tile_idx = 0;
    int cmax = 0;
    const double thresh = tol * (double)L * (double)L;
    for (int i = 0; i <= K; ++i) {                                /* shift loop, Listing 2 */
        const int shift = 1 << i, o = shift % L;
        memset(q, 0, sizeof(double) * N * (size_t)(K + 1));       /* "Set q = 0" */
        for (int ty = o - L; ty < H; ty += L)                     /* tiles of this shift, incl. overhanging ones */
            for (int tx = o - L; tx < W; tx += L) {
                if (ty + L <= 0 || tx + L <= 0) continue;
                const int prescribed = tile_cycles_in ? tile_cycles_in[tile_idx] : 0;
                int cyc = 0, tile_bad = 0;
                if (tile_cycles_in && (prescribed < 1 || prescribed > max_cycles)) { ++bad; ++tile_idx; continue; }
                for (;;) {
                    double delta = 0.0;
                    for (int k = K; k >= i; --k) {                /* for (s = 5; s >= smin; s--) */
                        const int side = 1 << k;
                        double *qk = q + (size_t)k * N;
                        for (int wy = ty; wy < ty + L; wy += side)
                            for (int wx = tx; wx < tx + L; wx += side) {
                                if (wy < 0 || wx < 0 || wy + side > H || wx + side > W) continue;
                                /* keep the old values, take the step, add |e_old - e_new| */
                                for (int r = 0; r < side; ++r)
                                    for (int cc = 0; cc < side; ++cc)
                                        tmp[r * side + cc] = x_out[(size_t)(wy + r) * W + wx + cc];
                                window_step(x_out, qk, W, wy, wx, side, level_c[k]);
                                for (int r = 0; r < side; ++r)
                                    for (int cc = 0; cc < side; ++cc)
                                        delta += fabs(tmp[r * side + cc] - x_out[(size_t)(wy + r) * W + wx + cc]);
                            }
                    }
                    ++cyc;
                    if (tile_cycles_in) {                         /* replay: the count is given, the deltas are checked */
                        if (cyc < prescribed) { if (!(delta > thresh * (1.0 - band))) tile_bad = 1; }
                        else {
                            if (cyc < max_cycles && delta > thresh * (1.0 + band)) tile_bad = 1;
                            break;
                        }
                    } else if (!(delta > thresh) || cyc >= max_cycles) break;
                }
                total += cyc;
                bad += tile_bad;
                if (cyc > cmax) cmax = cyc;
                if (tile_cycles_out) tile_cycles_out[tile_idx] = cyc;
                ++tile_idx;
            }
    }
    if (n_bad) *n_bad = bad;
    if (cycles_total) *cycles_total = total;
    if (cycles_max) *cycles_max = cmax;
    free(q);
    free(tmp);
    return 0;
}

int smre_oracle_icd_tol(const double *y, int H, int W, const int *sides, const double *c,
                        int n_sides, int max_cycles, double tol, double *x_out,
                        long long *cycles_total, int *cycles_max)
{
    if (!sides || !c || n_sides <= 0) return -1;
    int smax = 0;
    for (int a = 0; a < n_sides; ++a) if (sides[a] > smax) smax = sides[a];
    if (smax < 1) return -1;
    int K = 0;
    while ((2 << K) <= smax) ++K;
    double level_c[32];
    for (int k = 0; k <= K; ++k) {
        int found = 0;
        for (int a = 0; a < n_sides; ++a)
            if (sides[a] == (1 << k)) { level_c[k] = c[a]; found = 1; break; }
        if (!found) return -2;
    }
    return smre_oracle_icd_levels_tol(y, H, W, K, level_c, max_cycles, tol, x_out, cycles_total, cycles_max);
}

/* ===========================================================================
 * Threshold calibration (sec. 2.1, lines 89-113).
 *
 *   t_s(eps) = sum_{i in s} eps_i^2
 *   (t_s)^(1/4) ~ N(mu_s = (|s| - 0.5)^(1/4), sigma_s^2 = 1 / (8 sqrt|s|))
 *   Q_Omega = max_{s in Omega} ((t_s)^(1/4) - mu_s) / sigma_s
 *   c_s(alpha) = 1 / (q_alpha sigma_s + mu_s)^4,  q_alpha the alpha quantile of Q_Omega
 * Omega = the exact method's window set: every square window of every side in
 * sides[] at every shift, fully inside the image (reading A6);
 * |s| = side^2.  In this library's threshold convention c_S = 1 / c_s(alpha)
 * = (q_alpha sigma_s + mu_s)^4.
 * Readings (DESIGN.md A-CAL): the noise images are INPUTS (unit variance); the
 * alpha quantile of the n simulated values is the order statistic of rank
 * ceil(alpha n) (1-based, clamped to [1, n]).
 * ------------------------------------------------------------------------- */
double smre_oracle_cal_mu(int side)    { double n = (double)side * side; return pow(n - 0.5, 0.25); }
double smre_oracle_cal_sigma(int side) { double n = (double)side * side; return sqrt(1.0 / (8.0 * sqrt(n))); }

/* Q_Omega of one image. */
int smre_oracle_q_stat(const double *eps, int H, int W, const int *sides, int n_sides, double *q_out)
{
    if (!eps || !sides || !q_out || H <= 0 || W <= 0 || n_sides <= 0) return -1;
    double best = -HUGE_VAL;
    for (int a = 0; a < n_sides; ++a) {
        const int s = sides[a];
        if (s < 1 || s > H || s > W) return -1;
        const double mu = smre_oracle_cal_mu(s), sg = smre_oracle_cal_sigma(s);
        for (int wy = 0; wy + s <= H; ++wy)
            for (int wx = 0; wx + s <= W; ++wx) {
                double t = 0.0;
                for (int r = wy; r < wy + s; ++r)
                    for (int col = wx; col < wx + s; ++col) {
                        double v = eps[(size_t)r * W + col];
                        t += v * v;
                    }
                double z = (pow(t, 0.25) - mu) / sg;
                if (z > best) best = z;
            }
    }
    *q_out = best;
    return 0;
}

static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* q_alpha = order statistic of rank ceil(alpha n) of q[0..n), then c_out[a] = (q_alpha sigma + mu)^4. */
int smre_oracle_thresholds_from_q(const double *q, int n, double alpha, const int *sides, int n_sides,
                                  double *q_alpha_out, double *c_out)
{
    if (!q || n <= 0 || !sides || n_sides <= 0 || !c_out || !(alpha > 0.0) || !(alpha <= 1.0)) return -1;
    double *tmp = (double *)malloc(sizeof(double) * (size_t)n);
    if (!tmp) return -1;
    memcpy(tmp, q, sizeof(double) * (size_t)n);
    qsort(tmp, (size_t)n, sizeof(double), cmp_double);
    int k = (int)ceil(alpha * (double)n);
    if (k < 1) k = 1;
    if (k > n) k = n;
    const double qa = tmp[k - 1];
    free(tmp);
    if (q_alpha_out) *q_alpha_out = qa;
    for (int a = 0; a < n_sides; ++a) {
        double base = qa * smre_oracle_cal_sigma(sides[a]) + smre_oracle_cal_mu(sides[a]);
        c_out[a] = base * base * base * base;
    }
    return 0;
}

/* ===========================================================================
 * Second-order SOFI cumulant at zero time lag (Eq. 19):
 *     C_2(r, 0) = <F^2(r, t)>_t - <F(r, t)>_t^2
 * per pixel over the n frames of a stack F[n][H][W] (population variance: both means divide by n).
 * The plain definition, two passes per pixel.
 * ------------------------------------------------------------------------- */
int smre_oracle_cumulant2(const double *stack, int n, int H, int W, double *c2_out)
{
    if (!stack || !c2_out || n <= 0 || H <= 0 || W <= 0) return -1;
    size_t N = (size_t)H * W;
    for (size_t i = 0; i < N; ++i) {
        double m1 = 0.0, m2 = 0.0;
        for (int t = 0; t < n; ++t) {
            double v = stack[(size_t)t * N + i];
            m1 += v;
            m2 += v * v;
        }
        m1 /= (double)n;
        m2 /= (double)n;
        c2_out[i] = m2 - m1 * m1;
    }
    return 0;
}

/* ===========================================================================
 * The ADMM around the projection (Alg. 1, Eq. 9-13; parameters App. B,
 * PAPER.md:697-753).  DESIGN.md readings A-ADMM-1..9.
 *
 * Problem (Eq. 10):   min  G(eps) + R(z)   s.t.  I = A * x + eps,  z = x,
 * G = indicator of the multi-resolution constraint set (Eq. 5), R(z) = (lambda / 2) ||z||^2 ("we use the generic L2
 * norm as regularization"; lambda = `regularization` of App. B).
 *
 * A ("approximated as Gaussian kernel with the standard deviation sigma_PSF"): separable, taps
 * g[t] = exp(-t^2 / (2 sigma^2)), |t| <= radius = ceil(3 sigma), normalised to sum 1; the image is continued by
 * zero outside (A-ADMM-2), so A is a symmetric matrix and A^T * = A *.  sigma = 0: A = identity.
 * ------------------------------------------------------------------------- */
int smre_oracle_gauss_taps(double sigma, double *taps, int max_taps)
{
    if (sigma < 0.0 || !taps) return -1;
    int radius = (int)ceil(3.0 * sigma);
    if (2 * radius + 1 > max_taps) return -1;
    double sum = 0.0;
    for (int t = -radius; t <= radius; ++t) {
        taps[t + radius] = sigma > 0.0 ? exp(-(double)t * t / (2.0 * sigma * sigma)) : 1.0;
        sum += taps[t + radius];
    }
    for (int t = 0; t <= 2 * radius; ++t) taps[t] /= sum;
    return radius;
}

/* out = A * x: rows first, then columns (two plain passes, zero outside the image). */
int smre_oracle_gauss_conv(const double *x, int H, int W, double sigma, double *out)
{
    double taps[257];
    int radius = smre_oracle_gauss_taps(sigma, taps, 257);
    if (radius < 0 || !x || !out || H <= 0 || W <= 0) return -1;
    double *tmp = (double *)malloc((size_t)H * W * sizeof(double));
    if (!tmp) return -2;
    for (int y = 0; y < H; ++y)
        for (int c = 0; c < W; ++c) {
            double a = 0.0;
            for (int t = -radius; t <= radius; ++t) {
                int cc = c + t;
                if (cc >= 0 && cc < W) a += taps[t + radius] * x[(size_t)y * W + cc];
            }
            tmp[(size_t)y * W + c] = a;
        }
    for (int y = 0; y < H; ++y)
        for (int c = 0; c < W; ++c) {
            double a = 0.0;
            for (int t = -radius; t <= radius; ++t) {
                int yy = y + t;
                if (yy >= 0 && yy < H) a += taps[t + radius] * tmp[(size_t)yy * W + c];
            }
            out[(size_t)y * W + c] = a;
        }
    free(tmp);
    return 0;
}

/* Alg. 1 with the z = x splitting of Eq. 10, in the order of the algorithm box:
 *
 *   x_{r+1}   = x_r - (1 / (2 gamma)) grad_x L(x_r)                                  (Eq. 11, reading A-ADMM-3)
 *               grad_x L = -A^T * (rho1 (I - A * x_r - eps_r) + Y1) + rho2 (x_r - z_r) + Y2
 *   eps_{r+1} = P_G(I - A * x_{r+1} + Y1 / rho1)                                     (Eq. 12; Dykstra, variant 0 / 1,
 *                                                                                     n_sweeps from q = 0, A13)
 *   z_{r+1}   = (rho2 x_{r+1} + Y2) / (lambda + rho2)                                (argmin_z of L; A-ADMM-4)
 *   Y1       += alpha1 (I - A * x_{r+1} - eps_{r+1})                                  (Alg. 1, steepest ascent)
 *   Y2       += alpha2 (x_{r+1} - z_{r+1})
 *
 * from x_0 = z_0 = 0, eps_0 = 0, Y = 0 (A-ADMM-5: with x_0 = I the first x-update is the identity and the `while`
 * would end at once), while r < max_iter and
 * ( ||x_r - x_{r-1}||_2 > delta  or  ||I - (A * x_r + eps_r)||_2 > delta ): the loop ends when BOTH are small
 * (A-ADMM-6: Alg. 1 prints `and`, which would end the loop in the first iteration whose projection absorbs the
 * residual completely -- the residual is exactly 0 whenever the argument of P_G is feasible -- long before x has
 * settled; App. B states "Finish when |x_r - x_{r-1}| < tolerance").
 *
 * Outputs: x, eps, z, Y1, Y2 [H*W] (any may be null), *iters = iterations done, hist[2 * max_iter] (may be null) =
 * the two norms after each iteration.
 */
int smre_oracle_admm(const double *I, int H, int W, const int *sides, const double *c, int n_sides, int variant,
                     int n_sweeps, double sigma, double rho1, double rho2, double alpha1, double alpha2,
                     double lambda, double gamma, double delta, int max_iter,
                     double *x_out, double *eps_out, double *z_out, double *y1_out, double *y2_out,
                     int *iters, double *hist)
{
    if (!I || H <= 0 || W <= 0 || !sides || !c || n_sides <= 0 || n_sweeps <= 0 || max_iter <= 0) return -1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(gamma > 0.0) || lambda < 0.0 || sigma < 0.0) return -1;
    size_t N = (size_t)H * W;
    double *buf = (double *)calloc(9 * N, sizeof(double));
    if (!buf) return -2;
    double *x = buf, *eps = buf + N, *z = buf + 2 * N, *Y1 = buf + 3 * N, *Y2 = buf + 4 * N;
    double *Ax = buf + 5 * N, *w = buf + 6 * N, *Aw = buf + 7 * N, *X = buf + 8 * N;
    int rc = 0, r = 0;
    while (r < max_iter) {
        /* x-update */
        if ((rc = smre_oracle_gauss_conv(x, H, W, sigma, Ax)) != 0) break;
        for (size_t i = 0; i < N; ++i) w[i] = rho1 * (I[i] - Ax[i] - eps[i]) + Y1[i];
        if ((rc = smre_oracle_gauss_conv(w, H, W, sigma, Aw)) != 0) break;          /* A^T * = A * */
        double dx2 = 0.0;
        for (size_t i = 0; i < N; ++i) {
            double g = -Aw[i] + rho2 * (x[i] - z[i]) + Y2[i];
            double xn = x[i] - g / (2.0 * gamma);
            dx2 += (xn - x[i]) * (xn - x[i]);
            x[i] = xn;
        }
        /* eps-update: the projection */
        if ((rc = smre_oracle_gauss_conv(x, H, W, sigma, Ax)) != 0) break;
        for (size_t i = 0; i < N; ++i) X[i] = I[i] - Ax[i] + Y1[i] / rho1;
        if (variant == 0) rc = smre_oracle_std(X, H, W, sides, c, n_sides, n_sweeps, eps, NULL, NULL);
        else rc = smre_oracle_icd(X, H, W, sides, c, n_sides, n_sweeps, eps);
        if (rc != 0) break;
        /* z-update, dual ascent */
        double res2 = 0.0;
        for (size_t i = 0; i < N; ++i) {
            z[i] = (rho2 * x[i] + Y2[i]) / (lambda + rho2);
            double r1 = I[i] - Ax[i] - eps[i];
            Y1[i] += alpha1 * r1;
            Y2[i] += alpha2 * (x[i] - z[i]);
            res2 += r1 * r1;
        }
        ++r;
        if (hist) { hist[2 * (r - 1)] = sqrt(dx2); hist[2 * (r - 1) + 1] = sqrt(res2); }
        if (!(sqrt(dx2) > delta || sqrt(res2) > delta)) break;
    }
    if (rc == 0) {
        if (x_out) memcpy(x_out, x, N * sizeof(double));
        if (eps_out) memcpy(eps_out, eps, N * sizeof(double));
        if (z_out) memcpy(z_out, z, N * sizeof(double));
        if (y1_out) memcpy(y1_out, Y1, N * sizeof(double));
        if (y2_out) memcpy(y2_out, Y2, N * sizeof(double));
        if (iters) *iters = r;
    }
    free(buf);
    return rc;
}
