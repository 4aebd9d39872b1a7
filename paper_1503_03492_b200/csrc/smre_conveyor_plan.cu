// Host planner of the conveyor sweep scheduler: tile-boundary trajectories and their invariants.
// Pure host code (no kernels, no device calls): the CPU tests exercise it through smre_plan_check.
//
// Along one axis, at step g the family has window edge s and offset o, i.e. the window grid lines
// are { o + m*s }.  Boundary k of the tiling sits at
//         E_k(g) = smallest grid line of step g that is >= a(g) + k*T          (k any integer)
// with T the nominal tile extent and a(g) a non-decreasing anchor chosen as the smallest value for
// which no boundary moves backwards: E_k(g) >= E_k(g-1) wherever that matters (inside the image).
// Tile k owns [E_k, E_k+1) clipped to the image.  Consequences the kernel relies on:
//   * every window of the step's family lies inside exactly one tile (boundaries are grid lines);
//   * boundaries only move towards higher coordinates, so a pixel only ever changes owner from
//     tile k to tile k-1: data flows in ONE direction and tile k-1 may lag behind tile k;
//   * extents stay within T +- (s-1) because all boundaries share one anchor.
// Tiles are born at coordinate 0 and die at coordinate N; tile k runs on slot (k mod slots).
#include "smre_conveyor.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>

namespace smre {

static inline int floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }
static inline int ceil_grid(int p, int o, int s) { return o - floordiv(o - p, s) * s; }
static inline int clipN(int v, int N) { return v < 0 ? 0 : (v > N ? N : v); }

static void set_why(char *why, size_t n, const char *fmt, int a = 0, int b = 0, int c = 0)
{
    if (why && n) snprintf(why, n, fmt, a, b, c);
}

// extra per-axis numbers the kernel would otherwise derive every step
static void fill_extras(AxisEntry &e, bool y_axis, int s, int N)
{
    if (y_axis) {
        const int kr = cv_kr(s);
        e.e0 = (short)((e.nw + kr - 1) / kr);
        e.e1 = (short)(e.nw * s);
    } else {
        const int pitch = (N + 3) & ~3;                       // row pitch of the q planes
        const int c0 = e.w0 & ~3, c1 = std::min((e.w0 + e.nw * s + 3) & ~3, pitch);
        e.e0 = (short)c0;
        e.e1 = (short)(e.nw > 0 ? (c1 - c0) >> 2 : 0);
    }
}

static void window_range(int L, int R, int s, int o, int N, short &w0, short &nw)
{
    const int n_total = (N - o) / s;                       // windows fully inside (reading A6)
    int i0 = (L <= o) ? 0 : (L - o + s - 1) / s;
    int i1 = std::min(n_total - 1, floordiv(R - 1 - o, s));
    if (R <= L || i1 < i0) { w0 = 0; nw = 0; return; }
    w0 = (short)(o + i0 * s);
    nw = (short)(i1 - i0 + 1);
}

bool plan_axis(int N, const std::vector<Family> &fams, bool y_axis, int n_sweeps, int T,
               AxisPlan &out, char *why, size_t why_len)
{
    const int F = (int)fams.size();
    const long long total_ll = (long long)F * n_sweeps;
    if (total_ll <= 0 || total_ll > (1ll << 26)) { set_why(why, why_len, "step count out of range"); return false; }
    const int total = (int)total_ll;
    out = AxisPlan{};
    out.N = N; out.T = T;
    auto side = [&](int g) { return fams[g % F].side; };
    auto off = [&](int g) { return y_axis ? fams[g % F].oy : fams[g % F].ox; };

    if (T == 0) {                                          // one static tile: nothing ever moves
        if (N > CV_PW) { set_why(why, why_len, "static tile needs extent <= %d", CV_PW); return false; }
        out.slots = 1; out.max_extent = N;
        out.tab.resize(total);
        for (int g = 0; g < total; ++g) {
            AxisEntry e{};
            e.L = 0; e.R = (short)N; e.A = (short)(g == 0 ? 0 : N); e.D = 0;
            window_range(0, N, side(g), off(g), N, e.w0, e.nw);
            fill_extras(e, y_axis, side(g), N);
            out.tab[g] = e;
        }
        return true;
    }

    int smax = 1;
    for (const Family &f : fams) smax = std::max(smax, f.side);
    if (T < 2 * smax || T > CV_PW) { set_why(why, why_len, "nominal tile %d unusable", T); return false; }

    // ---- pass 1: anchors a(g) ------------------------------------------------------------------
    std::vector<int> anchor(total);
    int a = 0, max_live = 0;
    for (int g = 0; g < total; ++g) {
        const int s = side(g), o = off(g);
        if (g > 0) {
            const int sp = side(g - 1), op = off(g - 1), ap = anchor[g - 1];
            const int klo = floordiv(-ap - smax, T) - 1, khi = floordiv(N + smax - ap, T) + 1;
            for (;; ++a) {
                bool ok = true;
                for (int k = klo; k <= khi && ok; ++k)
                    ok = clipN(ceil_grid(a + k * T, o, s), N) >= clipN(ceil_grid(ap + k * T, op, sp), N);
                if (ok) break;
            }
        }
        anchor[g] = a;
        const int klo = floordiv(-a - s, T) - 1, khi = floordiv(N - a, T) + 1;
        int live = 0;
        for (int k = klo; k <= khi; ++k)
            live += clipN(ceil_grid(a + (k + 1) * T, o, s), N) > clipN(ceil_grid(a + k * T, o, s), N);
        max_live = std::max(max_live, live);
    }
    out.drift = anchor[total - 1];

    // ---- pass 2: the table ----------------------------------------------------------------------
    // A slot must stay EMPTY for at least one step between the death of its tile at the far edge and the
    // birth of its next tile at the near edge.  A CTA walks through the steps in order; if it were the last
    // tile of the chain at step g and the first one at step g+1, the hand-off of step g would close a cycle
    // (every tile finishes step g only after it has received what its neighbour produced in step g).
    // One spare slot breaks the cycle.
    for (int S = max_live; S <= max_live + 1; ++S) {
    out.slots = S;
    out.max_extent = 0; out.max_move = 0;
    out.tab.assign((size_t)total * S, AxisEntry{});
    for (int g = 0; g < total; ++g) {
        const int s = side(g), o = off(g), ag = anchor[g];
        const int klo = floordiv(-ag - s, T) - 1, khi = floordiv(N - ag, T) + 1;
        for (int k = klo; k <= khi; ++k) {
            const int L = clipN(ceil_grid(ag + k * T, o, s), N);
            const int R = clipN(ceil_grid(ag + (k + 1) * T, o, s), N);
            if (R <= L) continue;
            AxisEntry e{};
            e.L = (short)L; e.R = (short)R;
            int A = L, D = L;
            if (g > 0) {
                const int Rp = clipN(ceil_grid(anchor[g - 1] + (k + 1) * T, off(g - 1), side(g - 1)), N);
                A = std::max(L, std::min(R, Rp));
                out.max_move = std::max(out.max_move, R - A);
            }
            if (g + 1 < total) {
                const int Ln = clipN(ceil_grid(anchor[g + 1] + k * T, off(g + 1), side(g + 1)), N);
                D = std::min(R, std::max(L, Ln));
            }
            e.A = (short)A; e.D = (short)D;
            window_range(L, R, s, o, N, e.w0, e.nw);
            fill_extras(e, y_axis, s, N);
            const int slot = ((k % S) + S) % S;
            AxisEntry &dst = out.tab[(size_t)g * S + slot];
            if (dst.R > dst.L) { set_why(why, why_len, "two live tiles in slot %d at step %d", slot, g); return false; }
            dst = e;
            out.max_extent = std::max(out.max_extent, R - L);
        }
    }
    bool switched = false;                                 // a slot alive in two consecutive steps with different tiles
    for (int g = 0; g + 1 < total && !switched; ++g)
        for (int c = 0; c < S; ++c) {
            const AxisEntry &e = out.tab[(size_t)g * S + c], &n = out.tab[(size_t)(g + 1) * S + c];
            if (e.R > e.L && n.R > n.L && n.A == n.L) { switched = true; break; }
        }
    if (!switched) break;
    }
    // How far (in slots, cyclically to the right / down) the slot that wrote the increment of a pixel in one
    // sweep is from the slot that reads it in the next: the owner of a pixel moves to lower tile numbers only,
    // and the owner number is monotone in the pixel, so the last pixel of a tile has the farthest writer.
    out.reach = 0;
    {
        const int S = out.slots, F = (int)fams.size();
        for (int g = F; g < total; ++g)
            for (int c = 0; c < S; ++c) {
                const AxisEntry &e = out.tab[(size_t)g * S + c];
                if (e.R <= e.L) continue;
                for (int d = out.reach + 1; d < S; ++d) {
                    const AxisEntry &w = out.tab[(size_t)(g - F) * S + (c + d) % S];
                    if (w.R > w.L && w.L < e.R && w.R > e.L) out.reach = d;
                }
            }
    }
    return verify_axis(out, why, why_len);
}

bool verify_axis(const AxisPlan &ap, char *why, size_t why_len)
{
    const int S = ap.slots, N = ap.N;
    const int total = (int)(ap.tab.size() / (size_t)S);
    auto E = [&](int g, int c) -> const AxisEntry & { return ap.tab[(size_t)g * S + c]; };
    for (int g = 0; g < total; ++g) {
        // (1) the live tiles partition [0, N)
        int covered = 0, pos = 0;
        for (int n = 0; n < S; ++n) {                      // walk tiles in order of position
            int best = -1;
            for (int c = 0; c < S; ++c)
                if (E(g, c).R > E(g, c).L && E(g, c).L == pos) best = c;
            if (best < 0) break;
            covered += E(g, best).R - E(g, best).L;
            pos = E(g, best).R;
        }
        int live_sum = 0;
        for (int c = 0; c < S; ++c) live_sum += E(g, c).R - E(g, c).L;
        if (pos != N || covered != N || live_sum != N) { set_why(why, why_len, "step %d: tiles do not partition the axis", g); return false; }
        for (int c = 0; c < S; ++c) {
            const AxisEntry &e = E(g, c);
            if (e.R <= e.L) continue;
            if (!(e.L <= e.A && e.A <= e.R && e.L <= e.D && e.D <= e.R)) { set_why(why, why_len, "step %d slot %d: A/D outside the tile", g, c); return false; }
            if (g == 0 && e.A != e.L) { set_why(why, why_len, "step 0 slot %d: everything must arrive", c); return false; }
            if (g > 0 && e.R - e.A > CV_SD) { set_why(why, why_len, "step %d slot %d: arrival strip deeper than %d", g, c, CV_SD); return false; }
            if (e.D - e.L > CV_SD) { set_why(why, why_len, "step %d slot %d: departure strip deeper than %d", g, c, CV_SD); return false; }
            if (e.R - e.L > CV_PW) { set_why(why, why_len, "step %d slot %d: tile wider than the torus", g, c); return false; }
            if (e.nw > 0 && (e.w0 < e.L || e.w0 + 0 >= e.R)) { set_why(why, why_len, "step %d slot %d: window range outside the tile", g, c); return false; }
            if (S == 1 && (e.D != e.L || (g > 0 && e.A != e.R))) { set_why(why, why_len, "step %d: a single tile must not hand off", g); return false; }
        }
        if (g + 1 == total) {
            for (int c = 0; c < S; ++c)
                if (E(g, c).D != E(g, c).L) { set_why(why, why_len, "last step: slot %d still departs", c); return false; }
            break;
        }
        for (int c = 0; c < S; ++c) {
            const AxisEntry &e = E(g, c), &n = E(g + 1, c);
            const bool live = e.R > e.L, nlive = n.R > n.L;
            if (live && nlive && n.A == n.L && S > 1) { set_why(why, why_len, "step %d slot %d: a new tile right after the old one (no empty step)", g, c); return false; }
            // (2) what the tile keeps is exactly what it holds, un-arrived, at the next step
            if (live && e.D < e.R) {
                if (!nlive || n.L != e.D || n.A != e.R) { set_why(why, why_len, "step %d slot %d: kept part does not continue", g, c); return false; }
            } else if (nlive && n.A != n.L) { set_why(why, why_len, "step %d slot %d: new tile must receive everything", g + 1, c); return false; }
            // (3) departures of slot c are exactly the arrivals of slot c-1 (the tile to the left)
            const AxisEntry &r = E(g + 1, (c + S - 1) % S);
            const int dep = live ? e.D - e.L : 0;
            const int arr = (r.R > r.L) ? r.R - r.A : 0;
            if (S > 1) {
                if (dep != arr || (dep > 0 && (r.A != e.L || r.R != e.D))) { set_why(why, why_len, "step %d slot %d: departures do not match the neighbour's arrivals", g, c); return false; }
            } else if (dep != 0) { set_why(why, why_len, "step %d: single tile departs", g); return false; }
        }
        // (4) torus injectivity: what a CTA touches in iteration g+1 -- sends of step g, the tile of
        //     step g+1, deposits for step g+2 -- must not alias modulo CV_PW
        if (g + 2 < total)
            for (int c = 0; c < S; ++c) {
                unsigned long long seen = 0;
                const int lo[3] = {E(g, c).L, E(g + 1, c).L, E(g + 2, c).L};
                const int hi[3] = {E(g, c).R, E(g + 1, c).R, E(g + 2, c).R};
                for (int i = 0; i < 3; ++i)
                    for (int p = lo[i]; p < hi[i]; ++p) {
                        bool counted = false;
                        for (int j = 0; j < i; ++j) counted = counted || (p >= lo[j] && p < hi[j]);
                        if (counted) continue;
                        const unsigned long long bit = 1ull << (p & (CV_PW - 1));
                        if (seen & bit) { set_why(why, why_len, "step %d slot %d: torus aliasing", g, c); return false; }
                        seen |= bit;
                    }
            }
    }
    return true;
}

// Nominal tile extents to try, best first: few, large tiles keep all slots on one wave of CTAs.
static std::vector<int> candidates(int N, int smax)
{
    std::vector<int> t;
    if (N <= CV_PW) { t.push_back(0); return t; }
    for (int T = CV_PW - CV_SD; T >= std::max(2 * smax, 16); --T) t.push_back(T);
    return t;
}

bool conveyor_summary(int H, int W, const std::vector<Family> &fams, int n_sweeps, int max_ctas,
                      ConveyorSummary *out, char *why, size_t why_len)
{
    int smax = 1;
    for (const Family &f : fams) smax = std::max(smax, f.side);
    if ((int)fams.size() > CV_MAX_F) { set_why(why, why_len, "more than %d families", CV_MAX_F); return false; }
    struct Cand { int T, slots, ext, move, reach; long long drift; };
    std::vector<Cand> cy, cx;
    char w2[160];
    for (int axis = 0; axis < 2; ++axis) {
        const int N = axis == 0 ? H : W;
        for (int T : candidates(N, smax)) {
            AxisPlan ap;
            if (!plan_axis(N, fams, axis == 0, n_sweeps, T, ap, w2, sizeof w2)) continue;
            (axis == 0 ? cy : cx).push_back(Cand{T, ap.slots, ap.max_extent, ap.max_move, ap.reach, ap.drift});
        }
    }
    if (cy.empty() || cx.empty()) { set_why(why, why_len, "no admissible tiling of an axis (last reason: %d)", 0); if (why && why_len) snprintf(why, why_len, "no admissible tiling: %s", w2); return false; }
    double best = 1e30;
    int by = -1, bx = -1;
    for (size_t i = 0; i < cy.size(); ++i)
        for (size_t j = 0; j < cx.size(); ++j) {
            if (cy[i].slots * cx[j].slots > max_ctas) continue;
            // cost of a step ~ fixed part + tile area; prefer the smallest largest tile
            const double cost = 600.0 + 1.0 * cy[i].ext * cx[j].ext;
            if (cost < best) { best = cost; by = (int)i; bx = (int)j; }
        }
    if (by < 0) { set_why(why, why_len, "tiling needs more than %d CTAs", max_ctas); return false; }
    if (out) {
        const int F = (int)fams.size();
        *out = ConveyorSummary{cy[by].slots, cx[bx].slots, cy[by].T, cx[bx].T, cy[by].ext, cx[bx].ext,
                               cy[by].move, cx[bx].move, cy[by].reach, cx[bx].reach, cy[by].drift, cx[bx].drift,
                               (long long)F * n_sweeps * (cy[by].slots + cx[bx].slots) * (long long)sizeof(AxisEntry)};
    }
    return true;
}

}  // namespace smre
