// Conveyor sweep scheduler: ONE cooperative kernel runs all
// n_sweeps * F strictly ordered family passes of the standard variant.
//
// Why not a barrier (or a kernel boundary) per family: a family pass of the 512^2 config moves
// 2 MiB of q -- 0.33 us of HBM time -- while a grid-wide barrier or a neighbour round trip through
// L2 costs 0.5-2 us.  A static tiling needs such a round trip per step, because windows straddle
// the tile boundaries in both directions.  Here the boundaries MOVE (smre_conveyor_plan.cu): at
// every step they lie on the window grid of that step's family, so
//   * each window is inside exactly one tile: a CTA projects the windows of its tile from shared
//     memory with no halo and no duplicated work;
//   * boundaries only move right / down, so a pixel changes owner only towards the left / upper
//     neighbour: dependencies point ONE way, the left / upper tiles simply run a few steps behind
//     the right / lower ones, and the hand-off latency is off the critical path;
//   * x lives in shared memory (torus-addressed 64 x 64 tile per CTA) from the first to the last
//     step; q streams HBM -> shared memory (16-byte cp.async.cg, CV_PF steps ahead; its addresses
//     do not depend on x) -> registers -> HBM (streaming stores).  That is the only HBM traffic.
// Hand-off: the previous owner writes each departing pixel as ONE 8-byte word {step tag, value} into
// the new owner's mailbox (global memory, L2 resident, ring of CV_D steps); the new owner loads the
// words one step before it needs them and deposits them into its tile.  No fences, no flags: the tag
// makes a word self-validating.  A per-CTA progress counter keeps a writer from lapping the ring.
//
// The per-window arithmetic and its summation order are those of family_pass_kernel, so this
// scheduler and the graph scheduler return identical bits.
#include "smre_conveyor.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace smre {

struct CFamily {
    int side, G;                  // window edge; lanes per window (power of two >= side)
    float c, sqrt_c;
};

struct CParams {
    const float *y;               // [B_total][H][W]
    float *x_out;                 // [B_total][H][W]
    float *q;                     // [F][B_total][H][Wq]
    const CFamily *fams;          // [F]
    const AxisEntry *taby;        // [total][NR]
    const AxisEntry *tabx;        // [total][NC]
    unsigned long long *mbox;     // [n_cta][CV_D][CV_MBW] words {tag:32 | value:32}
    unsigned *prog;               // [n_cta][CV_PROG_STRIDE] "mailbox read up to and including step" (one line each)
    int *status;                  // != 0: a poll timed out somewhere (protocol bug) -> everybody leaves
    unsigned long long *trace;    // debug (SMRE_CV_TRACE): [n_cta][total][8] globaltimer stamps, or null
    int F, total;
    int H, W, Wq, B_total, frame0;   // Wq: row pitch of the q planes (W rounded up to 4)
    int NR, NC;
};

// ---- small PTX helpers ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_u64_gpu(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_u64_gpu(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_u32_gpu(const unsigned *p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_u32_gpu(unsigned *p, unsigned v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async16(unsigned smem_addr, const void *gptr) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Spin until the mailbox word carries `tag`.  A poll that outlives ~1 s (or sees another CTA's failure)
// raises *status and gives up, so a protocol bug cannot hang the GPU.
__device__ __noinline__ unsigned long long poll_tag(const unsigned long long *p, unsigned tag, int *status) {
    const long long t0 = clock64();
    unsigned long long v;
    for (unsigned spins = 1;; ++spins) {
        v = ld_u64_gpu(p);
        if ((unsigned)(v >> 32) == tag) break;
        __nanosleep(64);                                   // polling a line bounces it between the L2 halves
        if ((spins & 63u) == 0) {
            if (*(volatile int *)status != 0) break;
            if (clock64() - t0 > 2000000000LL) { atomicExch(status, 1); break; }
        }
    }
    return v;
}
__device__ __noinline__ unsigned poll_prog(const unsigned *p, unsigned need, int *status) {
    const long long t0 = clock64();
    unsigned v;
    for (unsigned spins = 1;; ++spins) {
        v = ld_u32_gpu(p);
        if (v >= need) break;
        __nanosleep(200);
        if ((spins & 63u) == 0) {
            if (*(volatile int *)status != 0) return need;
            if (clock64() - t0 > 2000000000LL) { atomicExch(status, 1); return need; }
        }
    }
    return v;
}

__device__ __forceinline__ int tidx(int r, int c) { return ((r & (CV_PW - 1)) << 6) | (c & (CV_PW - 1)); }
static_assert(CV_PW == 64, "tidx assumes a 64 x 64 torus");

// mailbox word of pixel (r, c): column strips are column-major so that the usual one-column strip is
// contiguous; row strips row-major.  Unique inside a strip because strips are <= CV_SD deep.
__device__ __forceinline__ int mbox_col_word(int r, int c) { return ((c & (CV_SD - 1)) << 6) | (r & 63); }
__device__ __forceinline__ int mbox_row_word(int r, int c) { return CV_SD * 64 + (((r & (CV_SD - 1)) << 6) | (c & 63)); }

struct Smem {
    float xs[CV_PW * CV_PW];                 // the x tile, torus addressed by image (row, column)
    float qs[CV_NST][CV_PW * CV_PW];         // q stages: [(row - first window row) * 64 + (column - c0)]
    AxisEntry tab[CV_TR][2];                 // [step % CV_TR][0 = y, 1 = x]
    CFamily fams[CV_MAX_F];
};

// The windows of one step inside this CTA's tile, for a compile-time window edge S.
// G = lanes per window (power of two >= S): lane j of a window owns column j.  A lane handles KR
// vertically stacked windows (S * KR rows of its column) so that the per-item index arithmetic is
// paid once per ~8 pixels whatever the window size.  Summation order per window = family_pass_kernel's:
// rows top to bottom inside the lane (fma), then an xor-shuffle tree over the G lanes.
template <int S, int KR>
__device__ __forceinline__ void project_tile(Smem &sm, const float *qst, float *__restrict__ qplane,
                                             const AxisEntry &ey, const AxisEntry &ex, float c, float sqrt_c,
                                             int Wq, bool first_sweep, int cw, int lane)
{
    constexpr int G = S <= 1 ? 1 : S <= 2 ? 2 : S <= 4 ? 4 : 8;
    constexpr int R = S * KR;
    const int nwy = ey.nw, nwx = ex.nw;
    const int nby = (nwy + KR - 1) / KR;                 // blocks of KR window rows
    const int n_items = nby * nwx * G;
    const int c0 = ex.w0 & ~3;
    for (int base = cw * 32; base < n_items; base += CV_NCW * 32) {
        const int item = base + lane;
        const int grp = item / G, j = item % G;
        const int by = (int)(((unsigned)grp * ex.magic) >> 20), wix = grp - by * nwx;
        const bool on = item < n_items && j < S;
        const int nwin = on ? min(KR, nwy - by * KR) : 0;    // valid windows of this block
        const int rr0 = by * R;
        const int r0 = ey.w0 + rr0, cc = ex.w0 + wix * S + j;
        const int xi0 = tidx(r0, cc);
        const float *qs0 = qst + rr0 * CV_PW + (cc - c0);
        float *qg = qplane + (size_t)r0 * Wq + cc;
        float v[R], part[KR];
#pragma unroll
        for (int k = 0; k < KR; ++k) {
            part[k] = 0.0f;
#pragma unroll
            for (int r = 0; r < S; ++r) {
                const int rr = k * S + r;
                v[rr] = 0.0f;
                if (k < nwin) {
                    const float xv = sm.xs[(xi0 + rr * CV_PW) & (CV_PW * CV_PW - 1)];
                    v[rr] = first_sweep ? xv : xv + qs0[rr * CV_PW];
                }
                part[k] = fmaf(v[rr], v[rr], part[k]);
            }
        }
#pragma unroll
        for (int m = G / 2; m > 0; m >>= 1)
#pragma unroll
            for (int k = 0; k < KR; ++k) part[k] += __shfl_xor_sync(0xffffffffu, part[k], m);
#pragma unroll
        for (int k = 0; k < KR; ++k) {
            const float alpha = ball_scale(part[k], c, sqrt_c);
#pragma unroll
            for (int r = 0; r < S; ++r) {
                const int rr = k * S + r;
                if (k < nwin) {
                    const float xn = alpha * v[rr];
                    sm.xs[(xi0 + rr * CV_PW) & (CV_PW * CV_PW - 1)] = xn;
                    __stcs(qg + (size_t)rr * Wq, v[rr] - xn);
                }
            }
        }
    }
}

// Window edges above 8: G = 16 or 32 lanes per window, run-time edge s, one window per lane group.
template <int G>
__device__ __forceinline__ void project_tile_big(Smem &sm, const float *qst, float *__restrict__ qplane,
                                                 const AxisEntry &ey, const AxisEntry &ex, int s, float c,
                                                 float sqrt_c, int Wq, bool first_sweep, int cw, int lane)
{
    const int nwx = ex.nw;
    const int n_items = ey.nw * nwx * G;
    const int c0 = ex.w0 & ~3;
    for (int base = cw * 32; base < n_items; base += CV_NCW * 32) {
        const int item = base + lane;
        const int win = item / G, j = item % G;
        const int wiy = (int)(((unsigned)win * ex.magic) >> 20), wix = win - wiy * nwx;
        const bool on = item < n_items && j < s;
        const int rr0 = wiy * s;
        const int r0 = ey.w0 + rr0, cc = ex.w0 + wix * s + j;
        const int xi0 = tidx(r0, cc);
        const float *qs0 = qst + rr0 * CV_PW + (cc - c0);
        float *qg = qplane + (size_t)r0 * Wq + cc;
        float v[G];
        float part = 0.0f;
#pragma unroll
        for (int r = 0; r < G; ++r) {
            v[r] = 0.0f;
            if (r < s && on) {
                const float xv = sm.xs[(xi0 + r * CV_PW) & (CV_PW * CV_PW - 1)];
                v[r] = first_sweep ? xv : xv + qs0[r * CV_PW];
            }
            part = fmaf(v[r], v[r], part);
        }
#pragma unroll
        for (int m = G / 2; m > 0; m >>= 1) part += __shfl_xor_sync(0xffffffffu, part, m);
        const float alpha = ball_scale(part, c, sqrt_c);
#pragma unroll
        for (int r = 0; r < G; ++r) {
            if (r < s && on) {
                const float xn = alpha * v[r];
                sm.xs[(xi0 + r * CV_PW) & (CV_PW * CV_PW - 1)] = xn;
                __stcs(qg + (size_t)r * Wq, v[r] - xn);
            }
        }
    }
}

__global__ void __launch_bounds__(CV_NT, 1)
conveyor_kernel(const __grid_constant__ CParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x;
    const int bl = cta / (p.NR * p.NC);
    const int t2 = cta - bl * p.NR * p.NC;
    const int ci = t2 / p.NC, cj = t2 - ci * p.NC;
    const size_t frame_off = (size_t)(p.frame0 + bl) * p.H * p.W;
    const size_t frame_off_q = (size_t)(p.frame0 + bl) * p.H * p.Wq;
    const size_t plane = (size_t)p.B_total * p.H * p.Wq;
    // receivers of departing pixels: bit 0 = left neighbour, bit 1 = upper neighbour (3 = up-left)
    const int cjl = (cj + p.NC - 1) % p.NC, ciu = (ci + p.NR - 1) % p.NR;
    auto nbr_cta = [&](int which) {
        return (bl * p.NR + ((which & 2) ? ciu : ci)) * p.NC + ((which & 1) ? cjl : cj);
    };
    unsigned long long *my_box = p.mbox + (size_t)cta * CV_D * CV_MBW;
    const int total = p.total;

    // ---- prologue: families and the first table entries into shared memory; x <- y on the tile ----
    for (int i = tid; i < p.F; i += CV_NT) sm.fams[i] = p.fams[i];
    for (int i = tid; i < 2 * min(total, CV_LA + 1); i += CV_NT) {
        const int g = i >> 1, ax = i & 1;
        sm.tab[g % CV_TR][ax] = ax ? p.tabx[(size_t)g * p.NC + cj] : p.taby[(size_t)g * p.NR + ci];
    }
    __syncthreads();
    {
        const AxisEntry ey = sm.tab[0][0], ex = sm.tab[0][1];
        const int h = ey.R - ey.L, w = ex.R - ex.L;
        for (int i = tid; i < h * w; i += CV_NT) {
            const int r = ey.L + i / w, c = ex.L + i % w;
            sm.xs[tidx(r, c)] = p.y[frame_off + (size_t)r * p.W + c];
        }
    }
    __syncthreads();

    // role state (each used by one warp only)
    unsigned long long pend0 = 0, pend1 = 0;   // receiver: mailbox words loaded one step ahead
    unsigned prog_pend = 0, prog_seen = 0;     // sender lanes 1..3: progress of the receiving CTAs
    int prog_iter = -1;                        // step at which prog_pend was requested (-1: none in flight)
    int status_pend = 0;                       // receiver lane 0: the failure flag, loaded one step ahead
    int f = 0;                                 // family of step g
    int fp = CV_PF % p.F;                      // family of step g + CV_PF

    for (int g = 0; g < total; ++g) {
        int bad = 0;
        if (warp < CV_NCW) {
            // ---- compute warps: the windows of step g ---------------------------------------------------
            const AxisEntry ey = sm.tab[g % CV_TR][0], ex = sm.tab[g % CV_TR][1];
            if (ey.nw > 0 && ex.nw > 0) {
                const CFamily fam = sm.fams[f];
                float *qplane = p.q + (size_t)f * plane + frame_off_q;
                const float *qst = sm.qs[g % CV_NST];
                const bool first = g < p.F;
                switch (fam.side) {
                    case 1: project_tile<1, 8>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 2: project_tile<2, 4>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 3: project_tile<3, 3>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 4: project_tile<4, 2>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 5: project_tile<5, 2>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 6: project_tile<6, 1>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 7: project_tile<7, 1>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    case 8: project_tile<8, 1>(sm, qst, qplane, ey, ex, fam.c, fam.sqrt_c, p.Wq, first, warp, lane); break;
                    default:
                        if (fam.G <= 16) project_tile_big<16>(sm, qst, qplane, ey, ex, fam.side, fam.c, fam.sqrt_c, p.Wq, first, warp, lane);
                        else project_tile_big<32>(sm, qst, qplane, ey, ex, fam.side, fam.c, fam.sqrt_c, p.Wq, first, warp, lane);
                }
            }
        } else if (warp == CV_NCW) {
            // ---- loader warp: q of step g + CV_PF and the table entry of step g + CV_LA + 1 ---------------
            const int gp = g + CV_PF;
            if (gp < total && gp >= p.F) {                           // the first sweep reads no q (q = 0)
                const AxisEntry qy = sm.tab[gp % CV_TR][0], qx = sm.tab[gp % CV_TR][1];
                if (qy.nw > 0 && qx.nw > 0) {
                    const int s = sm.fams[fp].side;
                    const int rows = qy.nw * s;
                    const int c0 = qx.w0 & ~3, c1 = (qx.w0 + qx.nw * s + 3) & ~3;
                    const int half = lane >> 4, ch = lane & 15;      // 16 chunks of 4 columns cover a row
                    const int c = c0 + 4 * ch;
                    if (c < c1 && c < p.Wq) {
                        const float *src = p.q + (size_t)fp * plane + frame_off_q + (size_t)(qy.w0 + half) * p.Wq + c;
                        unsigned dst = (unsigned)__cvta_generic_to_shared(sm.qs[gp % CV_NST]) + 4u * (unsigned)(half * CV_PW + 4 * ch);
                        for (int rr = half; rr < rows; rr += 2) {
                            cp_async16(dst, src);
                            dst += 2 * CV_PW * 4;
                            src += 2 * (size_t)p.Wq;
                        }
                    }
                }
            }
            const int gt = g + CV_LA + 1;
            if (gt < total && lane < 2) {
                const AxisEntry *src = lane ? p.tabx + (size_t)gt * p.NC + cj : p.taby + (size_t)gt * p.NR + ci;
                cp_async16((unsigned)__cvta_generic_to_shared(&sm.tab[gt % CV_TR][lane]), src);
            }
            cp_async_commit();
            cp_async_wait<CV_PF - 1>();                              // q of step g+1 has landed
        } else if (warp == CV_NCW + 1) {
            // ---- sender warp: departures of step g-1 -> the neighbours' mailboxes, tagged g --------------
            if (g > 0) {
                if (lane >= 1 && lane <= 3) {                        // the ring slot must have been read
                    // the neighbour's counter is re-read only when the ring is half used, and the value is
                    // picked up a few steps later: the load must never sit on this warp's critical path
                    if (prog_iter >= 0 && g >= prog_iter + 3) { prog_seen = max(prog_seen, prog_pend); prog_iter = -1; }
                    if ((int)prog_seen + CV_D < g) {
                        prog_seen = poll_prog(p.prog + (size_t)nbr_cta(lane) * CV_PROG_STRIDE, (unsigned)(g - CV_D), p.status);
                        prog_iter = -1;
                    } else if (prog_iter < 0 && (int)prog_seen + CV_D / 2 < g) {
                        prog_pend = ld_u32_gpu(p.prog + (size_t)nbr_cta(lane) * CV_PROG_STRIDE);
                        prog_iter = g;
                    }
                }
                __syncwarp();
                if (p.trace && lane == 0) {
                    unsigned long long t;
                    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
                    p.trace[((size_t)cta * total + g) * 8 + 6] = t;
                }
                const AxisEntry py = sm.tab[(g - 1) % CV_TR][0], px = sm.tab[(g - 1) % CV_TR][1];
                const size_t slot = (size_t)(g % CV_D) * CV_MBW;
                const unsigned long long tag = (unsigned long long)(unsigned)g << 32;
                for (int c = px.L; c < px.D; ++c)                    // column strip: columns [L, D), all rows
                    for (int r = py.L + lane; r < py.R; r += 32) {
                        const int which = 1 | (r < py.D ? 2 : 0);
                        st_u64_gpu(p.mbox + (size_t)nbr_cta(which) * CV_D * CV_MBW + slot + mbox_col_word(r, c),
                                   tag | __float_as_uint(sm.xs[tidx(r, c)]));
                    }
                for (int r = py.L; r < py.D; ++r)                    // row strip: rows [L, D), columns [D, R)
                    for (int c = px.D + lane; c < px.R; c += 32)
                        st_u64_gpu(p.mbox + (size_t)nbr_cta(2) * CV_D * CV_MBW + slot + mbox_row_word(r, c),
                                   tag | __float_as_uint(sm.xs[tidx(r, c)]));
            }
        } else {
            // ---- receiver warp: arrivals of step g+1 into the tile; preload the first line of step g+2 ----
            if (g + 1 < total) {
                const AxisEntry ny = sm.tab[(g + 1) % CV_TR][0], nx = sm.tab[(g + 1) % CV_TR][1];
                const unsigned long long *box = my_box + (size_t)((g + 1) % CV_D) * CV_MBW;
                const unsigned tag = (unsigned)(g + 1);
                bool first_line = true;
                for (int c = nx.A; c < nx.R; ++c) {                  // column strip: columns [A, R), all rows
                    for (int r = ny.L + lane, t = 0; r < ny.R; r += 32, ++t) {
                        unsigned long long wv = (first_line && t < 2) ? (t ? pend1 : pend0) : 0ull;
                        if ((unsigned)(wv >> 32) != tag) wv = poll_tag(box + mbox_col_word(r, c), tag, p.status);
                        sm.xs[tidx(r, c)] = __uint_as_float((unsigned)wv);
                    }
                    first_line = false;
                }
                for (int r = ny.A; r < ny.R; ++r) {                  // row strip: rows [A, R), columns [L, A)
                    for (int c = nx.L + lane, t = 0; c < nx.A; c += 32, ++t) {
                        unsigned long long wv = (first_line && t < 2) ? (t ? pend1 : pend0) : 0ull;
                        if ((unsigned)(wv >> 32) != tag) wv = poll_tag(box + mbox_row_word(r, c), tag, p.status);
                        sm.xs[tidx(r, c)] = __uint_as_float((unsigned)wv);
                    }
                    first_line = false;
                }
                __syncwarp();
                if (lane == 0) st_u32_gpu(p.prog + (size_t)cta * CV_PROG_STRIDE, (unsigned)(g + 1));   // mailbox of step g+1 has been read
                pend0 = pend1 = 0;
                if (g + 2 < total) {
                    const AxisEntry my = sm.tab[(g + 2) % CV_TR][0], mx = sm.tab[(g + 2) % CV_TR][1];
                    const unsigned long long *box2 = my_box + (size_t)((g + 2) % CV_D) * CV_MBW;
                    if (mx.A < mx.R) {                               // first line = first arriving column
                        const int r = my.L + lane;
                        if (r < my.R) pend0 = ld_u64_gpu(box2 + mbox_col_word(r, mx.A));
                        if (r + 32 < my.R) pend1 = ld_u64_gpu(box2 + mbox_col_word(r + 32, mx.A));
                    } else if (my.A < my.R) {                        // ... or the first arriving row
                        const int c = mx.L + lane;
                        if (c < mx.A) pend0 = ld_u64_gpu(box2 + mbox_row_word(my.A, c));
                        if (c + 32 < mx.A) pend1 = ld_u64_gpu(box2 + mbox_row_word(my.A, c + 32));
                    }
                }
            }
            if (lane == 0) { bad = status_pend; status_pend = *(volatile int *)p.status; }
        }

        // ---- one barrier per step ----------------------------------------------------------------------
        if (p.trace && lane == 0 && (warp == 0 || warp >= CV_NCW - 1)) {      // debug: when each role finished
            unsigned long long t;
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
            p.trace[((size_t)cta * total + g) * 8 + 1 + (warp == 0 ? 0 : warp - (CV_NCW - 2))] = t;
        }
        if (__syncthreads_or(bad)) return;
        if (p.trace && tid == 0) {
            unsigned long long t;
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
            p.trace[((size_t)cta * total + g) * 8] = t;
        }
        if (++f == p.F) f = 0;
        if (++fp == p.F) fp = 0;
    }

    // ---- a9: x_out <- the tile of the last step -----------------------------------------------------
    {
        const AxisEntry ey = sm.tab[(total - 1) % CV_TR][0], ex = sm.tab[(total - 1) % CV_TR][1];
        const int h = ey.R - ey.L, w = ex.R - ex.L;
        for (int i = tid; i < h * w; i += CV_NT) {
            const int r = ey.L + i / w, c = ex.L + i % w;
            p.x_out[frame_off + (size_t)r * p.W + c] = sm.xs[tidx(r, c)];
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------

struct DeviceTables {             // boundary tables of one n_sweeps value, resident on the device
    int n_sweeps = 0;
    AxisEntry *d_y = nullptr, *d_x = nullptr;
};

struct ConveyorPlan {
    int H, W, Wq, B, F;
    int T_y, T_x, NR, NC;
    int frames_per_launch;
    std::vector<Family> fams;
    float *q, *xwork;
    CFamily *d_fams = nullptr;
    unsigned long long *d_mbox = nullptr;
    size_t mbox_bytes = 0;
    unsigned *d_prog = nullptr;
    int *d_status = nullptr;
    std::vector<DeviceTables> tables;
};

static void free_tables(DeviceTables &t)
{
    if (t.d_y) cudaFree(t.d_y);
    if (t.d_x) cudaFree(t.d_x);
    t = DeviceTables{};
}

// Boundary tables for n_sweeps sweeps with the plan's tile extents; cached per n_sweeps.
static const DeviceTables *tables_for(ConveyorPlan *pl, int n_sweeps, cudaStream_t st)
{
    for (const DeviceTables &t : pl->tables)
        if (t.n_sweeps == n_sweeps) return &t;
    AxisPlan ay, ax;
    char why[160];
    if (!plan_axis(pl->H, pl->fams, true, n_sweeps, pl->T_y, ay, why, sizeof why)) return nullptr;
    if (!plan_axis(pl->W, pl->fams, false, n_sweeps, pl->T_x, ax, why, sizeof why)) return nullptr;
    // slot numbering (tile k -> slot k mod slots) depends on the slot count the plan was sized for
    if (ay.slots != pl->NR || ax.slots != pl->NC) return nullptr;
    const std::vector<AxisEntry> &ty = ay.tab, &tx = ax.tab;
    if (pl->tables.size() >= 4) { free_tables(pl->tables.front()); pl->tables.erase(pl->tables.begin()); }
    DeviceTables t;
    t.n_sweeps = n_sweeps;
    bool ok = cudaMalloc(&t.d_y, ty.size() * sizeof(AxisEntry)) == cudaSuccess &&
              cudaMalloc(&t.d_x, tx.size() * sizeof(AxisEntry)) == cudaSuccess &&
              cudaMemcpyAsync(t.d_y, ty.data(), ty.size() * sizeof(AxisEntry), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(t.d_x, tx.data(), tx.size() * sizeof(AxisEntry), cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaStreamSynchronize(st) == cudaSuccess;       // the host vectors die at return (first call only)
    if (!ok) { cudaGetLastError(); free_tables(t); return nullptr; }
    pl->tables.push_back(t);
    return &pl->tables.back();
}

ConveyorPlan *conveyor_plan_create(int H, int W, int B, const std::vector<Family> &fams, float *q,
                                   float *xwork)
{
    if (fams.empty() || (int)fams.size() > CV_MAX_F || H > 32000 || W > 32000) return nullptr;
    int dev = 0, n_sm = 0, smem_optin = 0, coop = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop || (size_t)smem_optin < sizeof(Smem)) return nullptr;
    if (cudaFuncSetAttribute(conveyor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, conveyor_kernel, CV_NT, sizeof(Smem)) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return nullptr;
    }
    const int capacity = per_sm * n_sm;
    ConveyorSummary cs;
    char why[160];
    // the tiling is chosen on a short run; tables_for() re-plans (and re-verifies) each real length
    if (!conveyor_summary(H, W, fams, 3, capacity, &cs, why, sizeof why)) return nullptr;

    ConveyorPlan *pl = new ConveyorPlan;
    pl->H = H; pl->W = W; pl->Wq = (W + 3) & ~3; pl->B = B; pl->F = (int)fams.size();
    pl->T_y = cs.T_y; pl->T_x = cs.T_x; pl->NR = cs.tiles_y; pl->NC = cs.tiles_x;
    pl->fams = fams; pl->q = q; pl->xwork = xwork;
    const int tiles = pl->NR * pl->NC;
    pl->frames_per_launch = std::max(1, std::min(B, capacity / tiles));
    std::vector<CFamily> cf(fams.size());
    for (size_t i = 0; i < fams.size(); ++i) {
        int G = 1;
        while (G < fams[i].side) G <<= 1;
        cf[i] = CFamily{fams[i].side, G, fams[i].c, fams[i].sqrt_c};
    }
    const size_t n_cta = (size_t)pl->frames_per_launch * tiles;
    pl->mbox_bytes = n_cta * CV_D * CV_MBW * sizeof(unsigned long long);
    const bool good =
        cudaMalloc(&pl->d_fams, cf.size() * sizeof(CFamily)) == cudaSuccess &&
        cudaMalloc(&pl->d_mbox, pl->mbox_bytes) == cudaSuccess &&
        cudaMalloc(&pl->d_prog, n_cta * CV_PROG_STRIDE * sizeof(unsigned)) == cudaSuccess &&
        cudaMalloc(&pl->d_status, sizeof(int)) == cudaSuccess &&
        cudaMemcpy(pl->d_fams, cf.data(), cf.size() * sizeof(CFamily), cudaMemcpyHostToDevice) == cudaSuccess &&
        cudaMemset(pl->d_status, 0, sizeof(int)) == cudaSuccess;
    if (!good) {
        cudaGetLastError();
        conveyor_plan_destroy(pl);
        return nullptr;
    }
    return pl;
}

void conveyor_plan_destroy(ConveyorPlan *p)
{
    if (!p) return;
    for (DeviceTables &t : p->tables) free_tables(t);
    if (p->d_fams) cudaFree(p->d_fams);
    if (p->d_mbox) cudaFree(p->d_mbox);
    if (p->d_prog) cudaFree(p->d_prog);
    if (p->d_status) cudaFree(p->d_status);
    delete p;
}

void conveyor_plan_tiles(const ConveyorPlan *p, int *tiles_y, int *tiles_x)
{
    *tiles_y = p->NR;
    *tiles_x = p->NC;
}

int conveyor_plan_status(const ConveyorPlan *p)
{
    int s = -1;
    if (cudaMemcpy(&s, p->d_status, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return s;
}

cudaError_t conveyor_run(ConveyorPlan *pl, const float *y, float *x_out, int n_sweeps,
                         cudaStream_t st, long long *launches)
{
    cudaError_t e;
    const DeviceTables *tabs = tables_for(pl, n_sweeps, st);
    if (!tabs) return cudaErrorNotSupported;               // caller falls back to the graph schedule
    const size_t img_bytes = (size_t)pl->B * pl->H * pl->W * sizeof(float);
    if (y == x_out) {      // in place: a tile's first and last regions differ, so read from a copy
        if ((e = cudaMemcpyAsync(pl->xwork, y, img_bytes, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
        y = pl->xwork;
    }
    CParams p{};
    p.y = y; p.x_out = x_out; p.q = pl->q; p.fams = pl->d_fams; p.taby = tabs->d_y; p.tabx = tabs->d_x;
    p.mbox = pl->d_mbox; p.prog = pl->d_prog; p.status = pl->d_status;
    p.F = pl->F; p.total = pl->F * n_sweeps; p.H = pl->H; p.W = pl->W; p.Wq = pl->Wq; p.B_total = pl->B;
    p.NR = pl->NR; p.NC = pl->NC;
    const int tiles = pl->NR * pl->NC;
    const char *trace_path = getenv("SMRE_CV_TRACE");        // debug only: synchronises and writes a file
    if (trace_path && cudaMalloc(&p.trace, (size_t)tiles * p.total * 64) != cudaSuccess) p.trace = nullptr;
    for (int f0 = 0; f0 < pl->B; f0 += pl->frames_per_launch) {
        p.frame0 = f0;
        const int nb = std::min(pl->frames_per_launch, pl->B - f0);
        // tags and progress counters restart in every launch
        if ((e = cudaMemsetAsync(pl->d_mbox, 0, (size_t)nb * tiles * CV_D * CV_MBW * 8, st)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(pl->d_prog, 0, (size_t)nb * tiles * CV_PROG_STRIDE * sizeof(unsigned), st)) != cudaSuccess) return e;
        void *args[] = {&p};
        e = cudaLaunchCooperativeKernel((const void *)conveyor_kernel, dim3((unsigned)(nb * tiles)),
                                        dim3(CV_NT), args, sizeof(Smem), st);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
    if (p.trace) {
        std::vector<unsigned long long> t((size_t)tiles * p.total * 8);
        cudaStreamSynchronize(st);
        cudaMemcpy(t.data(), p.trace, t.size() * 8, cudaMemcpyDeviceToHost);
        cudaFree(p.trace);
        if (FILE *fh = fopen(trace_path, "wb")) {
            const int hdr[4] = {pl->NR, pl->NC, p.total, pl->F};
            fwrite(hdr, sizeof hdr, 1, fh);
            fwrite(t.data(), 8, t.size(), fh);
            fclose(fh);
        }
    }
    return cudaSuccess;
}

}  // namespace smre
