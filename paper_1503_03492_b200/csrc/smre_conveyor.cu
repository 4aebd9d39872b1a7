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
//     step; q streams HBM -> shared memory (one TMA box per step, CV_PF steps ahead: its addresses
//     do not depend on x) -> registers -> HBM (streaming stores).  That is the only HBM traffic.
// Warp roles per CTA: CV_NCW compute warps (one lane = one column of cv_kr(side) stacked windows; one
// template instantiation per window edge, entered once per run of equal edges), a control warp (plans
// CV_BATCH steps at a time, one per lane, into a descriptor ring; per step it orders the TMA box of step
// g + CV_PF and waits for the box of step g + 1), a sender warp and a receiver warp (first two lines of
// every hand-off, located by the planner; the compute warps share the rest at changes of window edge).
// One bar.sync per step.
// Hand-off: the previous owner writes each departing pixel as ONE 8-byte word {step tag, value} into
// the new owner's mailbox (global memory, L2 resident, ring of CV_D steps); the new owner loads the
// words one step before it needs them and deposits them into its tile.  No fences, no flags: the tag
// makes a word self-validating.  A per-CTA progress counter keeps a writer from lapping the ring.
//
// The per-window arithmetic and its summation order are those of family_pass_kernel, so this
// scheduler and the graph scheduler return identical bits.
#include "smre_conveyor.cuh"

#include <cuda.h>          // CUtensorMap (types only; the encoder is fetched with cudaGetDriverEntryPoint)
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace smre {

struct CFamily {                  // 32 bytes
    int side, lgG;                // window edge; log2 of the lanes per window (power of two >= side)
    int run_left;                 // families from this one to the end of its run of equal edges (within a sweep)
    int pad0;
    float c, sqrt_c;
    int pad1[2];
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
    unsigned *gmin;               // per frame of the launch: a lower bound of all its progress counters (control warp)
    int gmin_mask;                // gmin is recomputed every gmin_mask + 1 steps (4 .. 16)
    int fence_mask;               // the fenced counters it is computed from are refreshed every fence_mask + 1 steps (4 .. 64)
    int qp;                       // row pitch (floats) of a q stage in shared memory = columns of a TMA box
    CUtensorMap qmap[8];          // q as a 2-D tensor [F*B*H rows][Wq]; box = qp columns x 8*(k+1) rows
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
__device__ __forceinline__ unsigned ld_acquire_u32_gpu(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
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

// ---- mbarrier + TMA (the q boxes) ----------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long *bar, unsigned parity) {
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_2d_hint(void *smem_dst, const CUtensorMap *map, int c0, int c1, unsigned long long *bar, unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(map), "r"(c0), "r"(c1),
                   "r"((unsigned)__cvta_generic_to_shared(bar)), "l"(pol) : "memory");
}

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
// A slot held back by gmin: the published value is refreshed only every few steps of the slot that keeps it, and
// that slot may be waiting (through hand-offs) for this one.  So the lane recomputes the minimum itself, and
// publishes it, until it suffices: a slot is held back only while some slot really is that far behind.
__device__ __noinline__ unsigned poll_gmin(const unsigned *counters, int n, unsigned *gmin, unsigned need, int *status) {
    const long long t0 = clock64();
    for (unsigned spins = 1;; ++spins) {
        unsigned m = 0xffffffffu;
#pragma unroll 8
        for (int i = 0; i < n; ++i) m = min(m, ld_u32_gpu(counters + (size_t)i * CV_PROG_STRIDE + 1));
        __threadfence();
        atomicMax(gmin, m);                                // never lower a published bound (see publish_min)
        if (m >= need) return m;
        __nanosleep(400);
        if ((spins & 63u) == 0) {
            if (*(volatile int *)status != 0) return need;
            if (clock64() - t0 > 2000000000LL) { atomicExch(status, 1); return need; }
        }
    }
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

// Per-step descriptor (80 bytes; the compute warps read the first 32), written one step ahead by the control
// warp so that the compute warps do almost no index arithmetic of their own.
struct StepDesc {
    // v0
    int geom;                     // changes whenever (side, window counts) change: lanes re-derive their item then
    int n_items;                  // lanes of work (blocks of window rows * windows per row * G); 0: nothing
    int w0yx;                     // origin of the first window: row | column << 16
    unsigned qbase;               // float offset in Smem::qs of (first window row, first window column) of this step's box;
                                  // bit 31: first sweep (q is zero and is not read)
    // v1
    unsigned goff_lo, goff_hi;    // element offset in q of (family plane, frame, first window row, first window column)
    int f;                        // family index of this step
    int run_left;                 // steps left in this run of equal window edges, this one included
    // v2: the TMA box that brings this step's q (issued CV_PF steps before the step, awaited just before it)
    int tma_col, tma_row;         // tensor coordinates: 4-aligned column, row of (family, frame, first window row)
    int tma_k;                    // box height / 8 (1..8); 0: this step reads no q
    unsigned send_x;              // sender, per line (A: bits 0-15, B: bits 16-31): pixels that go to the up-left CTA | all-up flag << 8
    // v3, v4: the first two lines (two 32-lane chunks each) of the hand-off, enough for every step except the
    //     changes of window edge.  For lane position pos: v = (var0 + pos) & 63, mailbox word = wbase | v,
    //     tile index = xbase | v << sh.   a = wbase | xbase << 16,  b = var0 | len << 8 | sh << 16 | chunks of
    //     the whole step << 24 (line A only)
    unsigned recv_a[2], recv_b[2];   // arrivals OF this step          (stored a0, a1, b0, b1)
    unsigned send_a[2], send_b[2];   // departures AFTER this step
};
static_assert(sizeof(StepDesc) == 80, "StepDesc must be 80 bytes");

struct GeomDesc { int nwx, nwy, n_items, pad; };   // read by the lanes only when StepDesc::geom changes

struct Smem {
    float xs[CV_PW * CV_PW];                 // the x tile, torus addressed by image (row, column)
    float qs[CV_NST * CV_PW * CV_PW];        // q stages, filled by TMA: [(row - first window row) * qp + (column - c0)], c0 = first window column rounded down to 4
    AxisEntry tab[CV_TR][2];                 // [step % CV_TR][0 = y, 1 = x]
    StepDesc desc[CV_DR];                    // [step % CV_DR]
    GeomDesc geo[CV_DR];                     // [geom % CV_DR]: at most CV_AHEAD + CV_BATCH ids are planned ahead
    unsigned long long qbar[CV_NST];         // mbarriers: the TMA box of a stage has landed
    CFamily fams[CV_MAX_F];
    int abort;                               // set by the receiver warp when the failure flag is up
    int cur_step;                            // control warp -> planner warp: the step the CTA is in
    int planned;                             // planner warp -> control warp: steps [0, planned) have descriptors
};

// One barrier per step.  Every 8th step all warps also look at Smem::abort (set only at steps = 3 mod 8,
// so that every warp reads the same value) and leave together if a hand-off has timed out somewhere.
#define CV_STEP_BARRIER()                                                         \
    do {                                                                          \
        asm volatile("bar.sync 1, %0;" ::"n"(CV_NST_T) : "memory");              \
        if ((g & 7) == 7 && *(volatile int *)&sm.abort) return;                   \
    } while (0)

#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 2
#define CV_CLK(k) do { if (clk) clk[k] = clock64(); } while (0)
#else
#define CV_CLK(k) ((void)0)
#endif

#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 4
#define CV_RCLK(k) do { if (p.trace && lane == 0) rclk[k] = clock64(); } while (0)
#else
#define CV_RCLK(k) ((void)0)
#endif

#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD != 4
#define CV_STAMP(slot)                                                            \
    do {                                                                          \
        if (p.trace) {                                                            \
            unsigned long long t_;                                                \
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_));                 \
            p.trace[((size_t)cta * total + g) * 8 + (slot)] = t_;                 \
        }                                                                         \
    } while (0)
#else
#define CV_STAMP(slot) ((void)0)
#endif

// One item = one lane's column of KR vertically stacked windows of edge S (rows masked onto the torus).
// Summation order per window = family_pass_kernel's: rows top to bottom inside the lane (fma), then an
// xor-shuffle tree over the G lanes of the window.
template <int S, int KR, int G, int WQ>
__device__ __forceinline__ void project_item(float *xs, const float *qs0, float *__restrict__ qg, int xi0,
                                             int nwin, float c, float sqrt_c, int Wq_rt, int qp_rt, bool first_sweep,
                                             long long *clk = nullptr)
{
    constexpr int R = S * KR;
    const int Wq = WQ ? WQ : Wq_rt;
    const int qp = WQ ? CV_PW : qp_rt;                     // q stage pitch: 64 whenever the pitch of q is templated
    float v[R], part[KR];
#pragma unroll
    for (int k = 0; k < KR; ++k) {
        part[k] = 0.0f;
#pragma unroll
        for (int r = 0; r < S; ++r) {
            const int rr = k * S + r;
            v[rr] = 0.0f;
            if (k < nwin) {
                const float xv = xs[(xi0 + rr * CV_PW) & (CV_PW * CV_PW - 1)];
                v[rr] = first_sweep ? xv : __fadd_rn(xv, qs0[rr * qp]);
            }
            part[k] = fmaf(v[rr], v[rr], part[k]);
        }
    }
    if (part[0] >= 0.0f) CV_CLK(3);
#pragma unroll
    for (int m = 1; m < G; m <<= 1)                           // neighbouring columns first, as in family_pass_kernel
#pragma unroll
        for (int k = 0; k < KR; ++k) part[k] += __shfl_xor_sync(0xffffffffu, part[k], m);
    if (part[0] >= 0.0f) CV_CLK(4);
#pragma unroll
    for (int k = 0; k < KR; ++k) {
        const float alpha = ball_scale(part[k], c, sqrt_c);
        if (alpha >= 0.0f) CV_CLK(5);
#pragma unroll
        for (int r = 0; r < S; ++r) {
            const int rr = k * S + r;
            if (k < nwin) {
                float xn, qn;
                ball_update(v[rr], alpha, xn, qn);
                xs[(xi0 + rr * CV_PW) & (CV_PW * CV_PW - 1)] = xn;
                __stcs(qg + rr * Wq, qn);
            }
        }
    }
}

// Window edges above 8 (G = 16 or 32 lanes per window, run-time edge s, one window per lane group) and any
// item beyond the first CV_NCW * 32 of a step: the generic, un-cached path.
template <int G>
__device__ __forceinline__ void project_generic(Smem &sm, const GeomDesc &ge, int s, int kr, int w0y, int w0x,
                                                const float *qst, float *__restrict__ qplane, float c,
                                                float sqrt_c, int Wq, int qp, bool first_sweep, int base0, int cw, int lane)
{
    for (int base = base0 + cw * 32; base < ge.n_items; base += CV_NCW * 32) {
        const int item = base + lane;
        const int grp = item / G, j = item % G;
        const int by = grp / ge.nwx, wix = grp - by * ge.nwx;
        const bool on = item < ge.n_items && j < s;
#pragma unroll 1
        for (int k = 0; k < kr; ++k) {                       // stacked windows, one at a time
            const bool act = on && by * kr + k < ge.nwy;
            const int rr0 = (by * kr + k) * s;
            const int r0 = w0y + rr0, cc = w0x + wix * s + j;
            const int xi0 = tidx(r0, cc);
            const float *qs0 = qst + rr0 * qp + (wix * s + j);
            float *qg = qplane + (rr0 * Wq + wix * s + j);
            float v[G];
            float part = 0.0f;
#pragma unroll
            for (int r = 0; r < G; ++r) {
                v[r] = 0.0f;
                if (r < s && act) {
                    const float xv = sm.xs[(xi0 + r * CV_PW) & (CV_PW * CV_PW - 1)];
                    v[r] = first_sweep ? xv : __fadd_rn(xv, qs0[r * qp]);
                }
                part = fmaf(v[r], v[r], part);
            }
#pragma unroll
            for (int m = 1; m < G; m <<= 1) part += __shfl_xor_sync(0xffffffffu, part, m);
            const float alpha = ball_scale(part, c, sqrt_c);
#pragma unroll
            for (int r = 0; r < G; ++r) {
                if (r < s && act) {
                    float xn, qn;
                    ball_update(v[r], alpha, xn, qn);
                    sm.xs[(xi0 + r * CV_PW) & (CV_PW * CV_PW - 1)] = xn;
                    __stcs(qg + r * Wq, qn);
                }
            }
        }
    }
}

// State of one compute lane that survives from step to step.
struct LaneCache {
    int geom;                     // geometry id the fields below were derived for
    int nwin;                     // valid stacked windows of this lane's first item (0: lane idle)
    int busy;                     // warp-uniform: this warp has an item at all
    int rr0, colofs;              // row / column of the item relative to the first window's origin
    int lq, lg;                   // rr0 * qp + colofs,  rr0 * Wq + colofs
};

__device__ void help_handoff(Smem &sm, const CParams &p, int g, unsigned help, int warp, int lane);

// A run of steps [g, g_end) that share the window edge S, for one compute warp.
template <int S, int KR, int WQ>
__device__ __forceinline__ void run_steps(Smem &sm, const CParams &p, LaneCache &lc, int &g, int g_end, float c,
                                          float sqrt_c, int warp, int lane, int cta, int total)
{
    constexpr int G = S <= 1 ? 1 : S <= 2 ? 2 : S <= 4 ? 4 : 8;
    constexpr int LG = S <= 1 ? 0 : S <= 2 ? 1 : S <= 4 ? 2 : 3;
    const int Wq = WQ ? WQ : p.Wq;
    const int qp = WQ ? CV_PW : p.qp;
    // Items go to compute warps 15, 0, 1, 2, ...: with four schedulers (warp % 4) the usual 9-13 busy warps
    // then spread 3-3-3-x over them together with the control, sender and receiver warps (16, 17, 18).
    const int cwi = (warp + 1) % CV_NCW;
    for (; g < g_end; ++g) {
#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 2
        long long clkbuf[8];
        long long *clk = (warp == 0 && lane == 0 && p.trace) ? clkbuf : nullptr;
        if (clk) for (int i = 0; i < 8; ++i) clk[i] = 0;
        CV_CLK(0);
#else
        long long *clk = nullptr;
#endif
        const uint4 v0 = *reinterpret_cast<const uint4 *>(&sm.desc[g % CV_DR].geom);
        const uint2 v1 = *reinterpret_cast<const uint2 *>(&sm.desc[g % CV_DR].goff_lo);
        if ((int)v0.y >= 0) CV_CLK(1);
        if (warp == 0 && lane == 0) CV_STAMP(6);
        if ((int)v0.x != lc.geom) {                            // rare: the tile's window counts changed
            const GeomDesc ge = sm.geo[v0.x % CV_DR];
            const int n_items = (int)v0.y;
            lc.geom = (int)v0.x;
            const int item = cwi * 32 + lane;
            const int grp = item >> LG, j = item & (G - 1);
            const int by = ge.nwx > 0 ? grp / ge.nwx : 0, wix = grp - by * ge.nwx;
            const bool on = item < n_items && j < S;
            lc.nwin = on ? min(KR, ge.nwy - by * KR) : 0;
            lc.busy = cwi * 32 < n_items;
            lc.rr0 = by * KR * S;
            lc.colofs = wix * S + j;
            lc.lq = lc.rr0 * qp + lc.colofs;
            lc.lg = lc.rr0 * Wq + lc.colofs;
        }
        if (lc.busy) {
            const int r0 = (int)(v0.z & 0xffffu) + lc.rr0, cc = (int)(v0.z >> 16) + lc.colofs;
            const float *qs0 = sm.qs + (v0.w & 0x1fffffffu) + lc.lq;
            float *qg = p.q + (((unsigned long long)v1.y << 32) | v1.x) + lc.lg;
            if (r0 + cc >= 0) CV_CLK(2);
            project_item<S, KR, G, WQ>(sm.xs, qs0, qg, tidx(r0, cc), lc.nwin, c, sqrt_c, p.Wq, p.qp, (v0.w >> 31) != 0, clk);
            CV_CLK(6);
            if ((int)v0.y > CV_NCW * 32)
                project_generic<G>(sm, sm.geo[v0.x % CV_DR], S, KR, (int)(v0.z & 0xffffu), (int)(v0.z >> 16),
                                   sm.qs + (v0.w & 0x1fffffffu), p.q + (((unsigned long long)v1.y << 32) | v1.x),
                                   c, sqrt_c, Wq, qp, (v0.w >> 31) != 0, CV_NCW * 32, cwi, lane);
        }
        if (v0.w & 0x60000000u) help_handoff(sm, p, g, (v0.w >> 13) & 0x30000u, warp, lane);
        if (warp == 0 && lane == 0) CV_STAMP(1);
        CV_CLK(7);
        CV_STEP_BARRIER();
        if (warp == 0 && lane == 0) CV_STAMP(0);
#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 2
        if (clk) {
            const long long t_end = clock64();
            for (int i = 1; i < 8; ++i) p.trace[((size_t)cta * total + g) * 8 + i] = (unsigned long long)(clk[i] - clk[0]);
            p.trace[((size_t)cta * total + g) * 8] = (unsigned long long)(t_end - clk[0]);
        }
#endif
    }
}

// Window edges above 8: same loop, generic arithmetic only.
template <int G, int WQ>
__device__ __forceinline__ void run_steps_big(Smem &sm, const CParams &p, int s, int &g, int g_end, float c,
                                              float sqrt_c, int warp, int lane, int cta, int total)
{
    const int Wq = WQ ? WQ : p.Wq;
    const int qp = WQ ? CV_PW : p.qp;
    for (; g < g_end; ++g) {
        const uint4 v0 = *reinterpret_cast<const uint4 *>(&sm.desc[g % CV_DR].geom);
        const uint2 v1 = *reinterpret_cast<const uint2 *>(&sm.desc[g % CV_DR].goff_lo);
        if ((int)v0.y > 0)
            project_generic<G>(sm, sm.geo[v0.x % CV_DR], s, 1, (int)(v0.z & 0xffffu), (int)(v0.z >> 16),
                               sm.qs + (v0.w & 0x1fffffffu), p.q + (((unsigned long long)v1.y << 32) | v1.x),
                               c, sqrt_c, Wq, qp, (v0.w >> 31) != 0, 0, (warp + 1) % CV_NCW, lane);
        if (v0.w & 0x60000000u) help_handoff(sm, p, g, (v0.w >> 13) & 0x30000u, warp, lane);
        CV_STEP_BARRIER();
    }
}

// Control warp, all lanes: lane i plans step first + i (i < count <= 32) into the descriptor ring.
// geom / key: geometry id and key of the last step planned before `first` (warp-uniform, updated).
__device__ __forceinline__ void plan_steps(Smem &sm, const CParams &p, int first, int count, int lane, int total,
                                           unsigned long long frame_off_q, unsigned long long plane, int frame,
                                           int &geom, int &key)
{
    const int g = first + lane;
    const bool on = lane < count && g < total;
    int my_key = key, n_items = 0;
    AxisEntry ey{}, ex{};
    CFamily fam{};
    int f = 0;
    if (on) {
        ey = sm.tab[g % CV_TR][0]; ex = sm.tab[g % CV_TR][1];
        f = g % p.F;
        fam = sm.fams[f];
        n_items = (ey.nw > 0 && ex.nw > 0) ? (ey.e0 * ex.nw) << fam.lgG : 0;
        my_key = (fam.side << 16) | (ey.nw << 8) | ex.nw;
    }
    // geometry ids: a new id wherever the key differs from the previous step's
    int prev_key = __shfl_up_sync(0xffffffffu, my_key, 1);
    if (lane == 0) prev_key = key;
    const bool changed = on && my_key != prev_key;
    const unsigned chg = __ballot_sync(0xffffffffu, changed);
    const int my_geom = geom + __popc(chg & (0xffffffffu >> (31 - lane)));
    if (changed) {
        GeomDesc ge; ge.nwx = ex.nw; ge.nwy = ey.nw; ge.n_items = n_items; ge.pad = 0;
        sm.geo[my_geom % CV_DR] = ge;
    }
    if (on) {
        StepDesc d;
        d.geom = my_geom; d.n_items = n_items;
        d.w0yx = ey.w0 | (ex.w0 << 16);
        d.qbase = (unsigned)((g % CV_NST) * (CV_PW * CV_PW) + (ex.w0 - ex.e0)) | (g < p.F ? 0x80000000u : 0u);   // bits 29, 30: help flags, below
        const unsigned long long goff = frame_off_q + (unsigned long long)f * plane + (unsigned)(ey.w0 * p.Wq + ex.w0);
        d.goff_lo = (unsigned)goff; d.goff_hi = (unsigned)(goff >> 32);
        // bit 16: the departures of step g-1 have more than two lines, bit 17: so have the arrivals of step g+1:
        // then the compute warps share those lines during step g (changes of window edge move boundaries far)
        unsigned help = 0;
        if (g > 0) {
            const AxisEntry py = sm.tab[(g - 1) % CV_TR][0], px = sm.tab[(g - 1) % CV_TR][1];
            if (py.R > py.L && px.R > px.L && (px.D - px.L) + (px.R > px.D ? py.D - py.L : 0) > 2) help |= 1u << 16;
        }
        if (g + 1 < total) {
            const AxisEntry ny = sm.tab[(g + 1) % CV_TR][0], nx = sm.tab[(g + 1) % CV_TR][1];
            if (ny.R > ny.L && nx.R > nx.L && (nx.R - nx.A) + (nx.A > nx.L ? ny.R - ny.A : 0) > 2) help |= 1u << 17;
        }
        d.f = f; d.run_left = min(fam.run_left, total - g);
        d.qbase |= help << 13;                                        // bits 29 (send), 30 (receive)
        d.tma_col = ex.e0;
        d.tma_row = (f * p.B_total + frame) * p.H + ey.w0;
        d.tma_k = (g >= p.F && n_items > 0) ? (ey.e1 + 7) >> 3 : 0;          // the first sweep reads no q (q = 0)
        {
            // Lines of a hand-off in order: the columns of the column strip (all tile rows), then the rows of
            // the row strip.  line(k) describes line k (k = 0, 1) of the arrivals (arr) or departures of this step.
            const int h = ey.R - ey.L, live = (h > 0 && ex.R > ex.L);
            auto line = [&](bool arr, int k, unsigned &a, unsigned &b, unsigned &x) {
                const int c_lo = arr ? ex.A : ex.L, c_hi = arr ? ex.R : ex.D;          // column strip [c_lo, c_hi)
                const int r_lo = arr ? ey.A : ey.L, r_hi = arr ? ey.R : ey.D;          // row strip rows [r_lo, r_hi)
                const int rc_lo = arr ? ex.L : ex.D, rc_hi = arr ? ex.A : ex.R;        // ... and its columns
                const int ncl = c_hi - c_lo, nrl = (rc_hi > rc_lo) ? r_hi - r_lo : 0;
                const int chunks = live ? 2 * (ncl + nrl) : 0;
                unsigned wbase = 0, xbase = 0, var0 = 0, len = 0, sh = 0;
                x = 0;
                if (live && k < ncl) {
                    const int c = c_lo + k;
                    wbase = (c & (CV_SD - 1)) << 6; xbase = c & 63; var0 = ey.L & 63; len = h; sh = 6;
                    x = arr ? 0u : (unsigned)(ey.D - ey.L);                             // these go up-left
                } else if (live && k < ncl + nrl) {
                    const int r = r_lo + (k - ncl);
                    wbase = CV_SD * 64 + ((r & (CV_SD - 1)) << 6); xbase = (r & 63) << 6; var0 = rc_lo & 63;
                    len = rc_hi - rc_lo; sh = 0;
                    x = 1u << 8;                                                        // everything goes up
                }
                a = wbase | (xbase << 16);
                b = var0 | (len << 8) | (sh << 16) | (k == 0 ? (unsigned)chunks << 24 : 0u);
            };
            unsigned x0, x1;
            line(true, 0, d.recv_a[0], d.recv_b[0], x0);
            line(true, 1, d.recv_a[1], d.recv_b[1], x1);
            line(false, 0, d.send_a[0], d.send_b[0], x0);
            line(false, 1, d.send_a[1], d.send_b[1], x1);
            d.send_x = x0 | (x1 << 16);
        }
        sm.desc[g % CV_DR] = d;
    }
    const int last = min(count, total - first) - 1;              // last planned lane (>= 0 when anything was planned)
    if (last >= 0) {
        geom = __shfl_sync(0xffffffffu, my_geom, last);
        key = __shfl_sync(0xffffffffu, my_key, last);
    }
}

// Control warp: table entries of steps [first, first + 16) into the ring, one 16-byte cp.async per lane.
__device__ __forceinline__ void fetch_table(Smem &sm, const CParams &p, int first, int lane, int ci, int cj, int total)
{
    const int g = first + (lane >> 1), ax = lane & 1;
    if (g < total) {
        const AxisEntry *src = ax ? p.tabx + (size_t)g * p.NC + cj : p.taby + (size_t)g * p.NR + ci;
        cp_async16((unsigned)__cvta_generic_to_shared(&sm.tab[g % CV_TR][ax]), src);
    }
    cp_async_commit();
}

// Arrival chunk k of the step described by (Y, X): 32 consecutive positions of one line.  Lines: the
// columns [X.A, X.R) of the column strip (all tile rows), then the rows [Y.A, Y.R) of the row strip
// (columns [X.L, X.A)); two chunks per line (tiles are at most 64 wide / tall).
__device__ __forceinline__ bool arrival_chunk(const AxisEntry &Y, const AxisEntry &X, int k, int lane,
                                              int &r, int &c, int &word)
{
    const int ncl = X.R - X.A;
    const int line = k >> 1, pos = ((k & 1) << 5) + lane;
    if (line < ncl) {
        c = X.A + line; r = Y.L + pos;
        word = mbox_col_word(r, c);
        return r < Y.R;
    }
    r = Y.A + (line - ncl); c = X.L + pos;
    word = mbox_row_word(r, c);
    return r < Y.R && c < X.A;
}
__device__ __forceinline__ int arrival_chunks(const AxisEntry &Y, const AxisEntry &X)
{
    if (Y.R <= Y.L || X.R <= X.L) return 0;
    return 2 * ((X.R - X.A) + (X.A > X.L ? Y.R - Y.A : 0));
}

// Changes of window edge move the boundaries by up to CV_SD pixels: many lines change owner in one step.  The
// sender / receiver warps handle the first two lines of every step; the compute warps share the others
// (line 2 + warp, + CV_NCW, ...) during the step in which they are due.
__device__ __noinline__ void help_handoff(Smem &sm, const CParams &p, int g, unsigned help, int warp, int lane)
{
    const int cta = blockIdx.x;
    const int bl = cta / (p.NR * p.NC);
    const int t2 = cta - bl * p.NR * p.NC;
    const int ci = t2 / p.NC, cj = t2 - ci * p.NC;
    if (help & (1u << 16)) {                                         // departures of step g-1, tagged g
        const int cjl = (cj + p.NC - 1) % p.NC, ciu = (ci + p.NR - 1) % p.NR;
        unsigned long long *const box_l = p.mbox + (size_t)((bl * p.NR + ci) * p.NC + cjl) * CV_D * CV_MBW;
        unsigned long long *const box_u = p.mbox + (size_t)((bl * p.NR + ciu) * p.NC + cj) * CV_D * CV_MBW;
        unsigned long long *const box_ul = p.mbox + (size_t)((bl * p.NR + ciu) * p.NC + cjl) * CV_D * CV_MBW;
        const AxisEntry py = sm.tab[(g - 1) % CV_TR][0], px = sm.tab[(g - 1) % CV_TR][1];
        const int slot = (g % CV_D) * CV_MBW;
        const unsigned long long tag = (unsigned long long)(unsigned)g << 32;
        const int ncl = px.D - px.L, nlines = ncl + (px.R > px.D ? py.D - py.L : 0);
        for (int line = 2 + warp; line < nlines; line += CV_NCW) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int pos = (u << 5) + lane;
                int r, c, word;
                bool ok;
                unsigned long long *box;
                if (line < ncl) {
                    c = px.L + line; r = py.L + pos;
                    ok = r < py.R;
                    word = mbox_col_word(r, c);
                    box = (r < py.D) ? box_ul : box_l;
                } else {
                    r = py.L + (line - ncl); c = px.D + pos;
                    ok = c < px.R;
                    word = mbox_row_word(r, c);
                    box = box_u;
                }
                if (ok) st_u64_gpu(box + slot + word, tag | __float_as_uint(sm.xs[tidx(r, c)]));
            }
        }
    }
    if (help & (1u << 17)) {                                         // arrivals of step g+1
        const AxisEntry ny = sm.tab[(g + 1) % CV_TR][0], nx = sm.tab[(g + 1) % CV_TR][1];
        const unsigned long long *box = p.mbox + ((size_t)cta * CV_D + (size_t)((g + 1) % CV_D)) * CV_MBW;
        const unsigned tag = (unsigned)(g + 1);
        const int nchunks = arrival_chunks(ny, nx);
        for (int k0 = 4 + 2 * warp; k0 < nchunks; k0 += 2 * CV_NCW) {
            unsigned long long w[2];
            int xi[2], wd[2];
            bool ok[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                int r, c;
                ok[u] = arrival_chunk(ny, nx, k0 + u, lane, r, c, wd[u]);
                xi[u] = tidx(r, c);
                w[u] = ok[u] ? ld_u64_gpu(box + wd[u]) : 0ull;
            }
#pragma unroll
            for (int u = 0; u < 2; ++u)
                if (ok[u]) {
                    if ((unsigned)(w[u] >> 32) != tag) w[u] = poll_tag(box + wd[u], tag, p.status);
                    sm.xs[xi[u]] = __uint_as_float((unsigned)w[u]);
                }
        }
    }
}

template <int WQ>
__global__ void __launch_bounds__(CV_NT, 1)
conveyor_kernel(const __grid_constant__ CParams p)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x;
    const int bl = cta / (p.NR * p.NC);
    const int t2 = cta - bl * p.NR * p.NC;
    const int ci = t2 / p.NC, cj = t2 - ci * p.NC;
    const size_t frame_off = (size_t)(p.frame0 + bl) * p.H * p.W;
    const int total = p.total;

    // ---- prologue: families and the first table entries into shared memory; x <- y on the tile ----
    for (int i = tid; i < p.F; i += CV_NT) sm.fams[i] = p.fams[i];
    for (int i = tid; i < 2 * min(total, 3 * CV_BATCH); i += CV_NT) {
        const int g = i >> 1, ax = i & 1;
        sm.tab[g % CV_TR][ax] = ax ? p.tabx[(size_t)g * p.NC + cj] : p.taby[(size_t)g * p.NR + ci];
    }
    if (tid == 0) { sm.abort = 0; sm.cur_step = 0; sm.planned = CV_AHEAD; }
    __syncthreads();
    {
        const AxisEntry ey = sm.tab[0][0], ex = sm.tab[0][1];
        const int h = ey.R - ey.L, w = ex.R - ex.L;
        for (int i = tid; i < h * w; i += CV_NT) {
            const int r = ey.L + i / w, c = ex.L + i % w;
            sm.xs[tidx(r, c)] = p.y[frame_off + (size_t)r * p.W + c];
        }
    }
    const unsigned long long frame_off_q = (unsigned long long)(p.frame0 + bl) * p.H * p.Wq;
    const unsigned long long plane = (unsigned long long)p.B_total * p.H * p.Wq;
    int geom = 0, key = -1;                     // control warp: geometry id / key of the last planned step
    if (warp == CV_NCW) {
        if (lane == 0) {
            for (int i = 0; i < CV_NST; ++i) mbar_init(&sm.qbar[i], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    if (warp == CV_NCW + 3) plan_steps(sm, p, 0, CV_AHEAD, lane, total, frame_off_q, plane, p.frame0 + bl, geom, key);
    __syncthreads();

    if (warp < CV_NCW) {
        // =============== compute warps: runs of steps with one window edge ===============================
        LaneCache lc;
        lc.geom = -1; lc.nwin = 0; lc.rr0 = lc.colofs = lc.lq = lc.lg = 0;
        int g = 0;
        while (g < total) {
            const int f = sm.desc[g % CV_DR].f;
            const int g_end = g + sm.desc[g % CV_DR].run_left;
            const CFamily fam = sm.fams[f];
            switch (fam.side) {
                case 1: run_steps<1, cv_kr(1), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 2: run_steps<2, cv_kr(2), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 3: run_steps<3, cv_kr(3), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 4: run_steps<4, cv_kr(4), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 5: run_steps<5, cv_kr(5), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 6: run_steps<6, cv_kr(6), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 7: run_steps<7, cv_kr(7), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                case 8: run_steps<8, cv_kr(8), WQ>(sm, p, lc, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total); break;
                default:
                    if (fam.side <= 16) run_steps_big<16, WQ>(sm, p, fam.side, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total);
                    else run_steps_big<32, WQ>(sm, p, fam.side, g, g_end, fam.c, fam.sqrt_c, warp, lane, cta, total);
            }
            if (g < g_end) return;                                   // a run was cut short: abort
        }
    } else if (warp == CV_NCW) {
        // =============== control warp: plans steps in batches; per step only the TMA order and its wait ====
        int st1 = 1 % CV_NST;                  // q stage of step g + 1
        int stp = CV_PF % CV_NST;              // q stage of step g + CV_PF
        unsigned phase = 0;                    // bit s: parity the next wait on q stage s has to use
        // Ordering of q across sweeps.  The q of a pixel is written by one slot and read, a sweep (F steps) later,
        // by a slot up / left of it, which orders the box CV_PF steps ahead of its use.  Hand-offs alone do not
        // order the two: a boundary that does not move for some steps carries no message, and a slot without a
        // tile waits for nothing.  So the box of step s is ordered only when gmin, a lower bound of every progress
        // (fenced) counter of the frame, has reached s - F + 2: a value v is stored after the barrier of step v - 2
        // and a fence, so every slot's q writes of step s - F are visible.  The natural lag of the pipeline (tail to
        // head) is far smaller than a sweep of the usual configurations, and gmin is re-read, a step before the
        // value is needed, only when the last value seen gets old: the check is almost free.
        const unsigned *const gmin_ptr = p.gmin + (size_t)bl * CV_PROG_STRIDE;
        unsigned long long q_policy = 0;       // q is read once per sweep: its lines should leave L2 first
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(q_policy));
        unsigned gm_seen = 0, gm_pend = 0;     // lane 0
        bool gm_inflight = false;
        const bool ordered = p.NR * p.NC > 1;
        for (int g = 0; g < total; ++g) {
            if (lane == 0) {
                // (release at CTA scope: the services warp fences the q writes of the steps before this one)
                __threadfence_block();
                *(volatile int *)&sm.cur_step = g;                   // paces the services warp
                constexpr int CK = CV_BATCH - 1 - CV_PF < CV_BATCH / 2 ? CV_BATCH - 1 - CV_PF : CV_BATCH / 2;
                static_assert(CK >= 2, "the services warp needs a few steps for a batch of descriptors");
                if ((g & (CV_BATCH - 1)) == CK) {
                    // The descriptors of steps [g - CK + 16, g - CK + 32) were released to the services warp at step
                    // g - CK; nobody has looked beyond step g - 1 + CV_PF < g - CK + 16 so far.  Normally they are long done.
                    const int need = min(total, g - CK + CV_AHEAD + CV_BATCH);
                    const long long t0 = clock64();
                    while (*(volatile int *)&sm.planned < need) {
                        if (*(volatile int *)&sm.abort) break;
                        if (clock64() - t0 > 2000000000LL) { atomicExch(p.status, 1); break; }
                    }
                    __threadfence_block();
                }
                if (g + CV_PF < total) {                             // order the q box of step g + CV_PF
                    const StepDesc &d = sm.desc[(g + CV_PF) % CV_DR];
                    const int k = d.tma_k;
                    if (ordered) {
                        const int need = g + CV_PF - p.F + 2;
                        bool fresh = false;
                        if (gm_inflight) {
                            gm_seen = max(gm_seen, gm_pend); gm_inflight = false;
                            asm volatile("fence.proxy.async.global;" ::: "memory");     // generic -> async proxy (the TMA reads)
                        }
                        else if ((int)gm_seen < need + 8) { gm_pend = ld_acquire_u32_gpu(gmin_ptr); gm_inflight = true; }
                        if (k > 0 && (int)gm_seen < need) {        // held back: work out the minimum itself, it may be stale
                            gm_seen = poll_gmin(p.prog + (size_t)bl * p.NR * p.NC * CV_PROG_STRIDE, p.NR * p.NC,
                                                p.gmin + (size_t)bl * CV_PROG_STRIDE, (unsigned)need, p.status);
                            fresh = true;
                        }
                        if (fresh) {                               // (rare) acquire side, and generic -> async proxy
                            __threadfence();
                            asm volatile("fence.proxy.async.global;" ::: "memory");
                        }
                    }
                    if (k > 0) {
                        // single tile: the q rows of this box were written by this CTA's compute warps with generic-proxy
                        // stores one sweep ago; the step barriers order them before this point at CTA scope, the fence
                        // orders the async-proxy read of the TMA behind them (the multi-tile path fences above)
                        if (!ordered) asm volatile("fence.proxy.async.global;" ::: "memory");
                        mbar_expect_tx(&sm.qbar[stp], (unsigned)(k * 8 * p.qp * 4));
                        tma_load_2d_hint(sm.qs + (size_t)stp * (CV_PW * CV_PW), &p.qmap[k - 1], d.tma_col, d.tma_row, &sm.qbar[stp], q_policy);
                    }
                }
                CV_STAMP(7);
                if (g + 1 < total && sm.desc[(g + 1) % CV_DR].tma_k > 0) {   // q of step g+1 has landed
                    const unsigned parity = (phase >> st1) & 1u;
                    const long long t0 = clock64();
                    while (!mbar_try_wait(&sm.qbar[st1], parity))
                        if (clock64() - t0 > 2000000000LL) { atomicExch(p.status, 1); break; }
                    phase ^= 1u << st1;
                }
                CV_STAMP(3);
            }
            CV_STEP_BARRIER();
            if (++st1 == CV_NST) st1 = 0;
            if (++stp == CV_NST) stp = 0;
        }
        if (lane == 0) { __threadfence_block(); *(volatile int *)&sm.cur_step = total; }   // all steps done
    } else if (warp == CV_NCW + 1) {
        // =============== sender warp: departures of step g-1 -> the neighbours' mailboxes, tagged g ======
        // receivers of departing pixels: bit 0 = left neighbour, bit 1 = upper neighbour (3 = up-left)
        const int cjl = (cj + p.NC - 1) % p.NC, ciu = (ci + p.NR - 1) % p.NR;
        auto nbr_cta = [&](int which) {
            return (bl * p.NR + ((which & 2) ? ciu : ci)) * p.NC + ((which & 1) ? cjl : cj);
        };
        unsigned long long *const box_l = p.mbox + (size_t)nbr_cta(1) * CV_D * CV_MBW;
        unsigned long long *const box_u = p.mbox + (size_t)nbr_cta(2) * CV_D * CV_MBW;
        unsigned long long *const box_ul = p.mbox + (size_t)nbr_cta(3) * CV_D * CV_MBW;
        const unsigned *my_nbr_prog = p.prog + (size_t)nbr_cta(lane >= 1 && lane <= 3 ? lane : 1) * CV_PROG_STRIDE;
        unsigned prog_pend = 0, prog_seen = 0;  // lanes 1..3: progress of the receiving CTAs
        int prog_iter = -1;                     // step at which prog_pend was requested (-1: none in flight)
        for (int g = 0; g < total; ++g) {
            if (g > 0) {
                if ((g & 3) == 1 && lane >= 1 && lane <= 3) {
                    // Ring slots g .. g+4 (through the next check, so that helpers may send right away) must have
                    // been read by the receiver: its counter must have reached g + 4 - CV_D.  The counter is re-read only when the ring is half used, and the value is
                    // picked up 4 steps later: the load never sits on this warp's critical path.
                    if (prog_iter >= 0) { prog_seen = max(prog_seen, prog_pend); prog_iter = -1; }
                    if ((int)prog_seen + CV_D < g + 4) {
                        prog_seen = poll_prog(my_nbr_prog, (unsigned)(g + 4 - CV_D), p.status);
                    } else if ((int)prog_seen + CV_D / 2 < g + 4) {
                        prog_pend = ld_u32_gpu(my_nbr_prog);
                        prog_iter = g;
                    }
                }
                __syncwarp();
                const int slot = (g % CV_D) * CV_MBW;
                const unsigned long long tag = (unsigned long long)(unsigned)g << 32;
                // the first two departing lines of step g-1 (all there is except at changes of window edge)
                const uint4 ln = *reinterpret_cast<const uint4 *>(&sm.desc[(g - 1) % CV_DR].send_a[0]);   // {a0, a1, b0, b1}
                const unsigned sx = sm.desc[(g - 1) % CV_DR].send_x;
                const int nchunks = (int)(ln.z >> 24);
                if (nchunks > 0) {
                    float val[4];
                    unsigned wd[4];
                    bool ok[4];
#pragma unroll
                    for (int l = 0; l < 2; ++l) {
                        const unsigned a = l ? ln.y : ln.x, b = l ? ln.w : ln.z;
                        const unsigned var0 = b & 63u, len = (b >> 8) & 0xffu, sh = (b >> 16) & 0xffu;
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            const unsigned pos = (u << 5) + lane, v = (var0 + pos) & 63u;
                            ok[2 * l + u] = pos < len;
                            wd[2 * l + u] = (a & 0xffffu) | v;
                            val[2 * l + u] = pos < len ? sm.xs[(a >> 16) | (v << sh)] : 0.0f;
                        }
                    }
#pragma unroll
                    for (int l = 0; l < 2; ++l) {
                        const unsigned x = l ? sx >> 16 : sx & 0xffffu;
                        unsigned long long *const box_lo = (x >> 8) ? box_u : box_l;    // row line: everything goes up
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            const unsigned pos = (u << 5) + lane;
                            if (ok[2 * l + u])
                                st_u64_gpu((pos < (x & 0xffu) ? box_ul : box_lo) + slot + wd[2 * l + u],
                                           tag | __float_as_uint(val[2 * l + u]));
                        }
                    }
                }
                // (lines beyond the second are sent by the compute warps: help_handoff)
            }
            if (lane == 0) CV_STAMP(4);
            CV_STEP_BARRIER();
        }
    } else if (warp == CV_NCW + 3) {
        // =============== services warp: everything that is slow and that nobody has to wait for ===================
        // Paced by Smem::cur_step only; it never joins the step barrier.  (a) Descriptors of steps [16 b + 16,
        // 16 b + 32) as soon as step 16 b runs (~2-3 us per batch; rings: a batch overwrites descriptors of steps
        // < 16 b - 32 and table entries of steps < 16 b - 64, all retired by then).  (b) The mailbox progress counter
        // (word 0): when the CTA is in step c, its receiver has read the arrivals of step c.  (c) The fenced counter
        // (word 1; gmin is the minimum of these): the barrier of step c - 1 lies behind the CTA, so the q writes of all
        // steps <= c - 1 have been issued; control's CTA-scope release of cur_step and this warp's fence make them
        // visible before the value c + 1 is.  Every fence_mask + 1 steps (a fence takes 1-4 us).  (d) The first slot
        // of a frame keeps that frame's gmin.
        const int tiles = p.NR * p.NC;
        const bool ordered = tiles > 1;
        const bool keeper = ordered && ci == 0 && cj == 0;
        const unsigned *const frame_prog = p.prog + (size_t)bl * tiles * CV_PROG_STRIDE;
        unsigned *const gmin_out = p.gmin + (size_t)bl * CV_PROG_STRIDE;
        unsigned cnt[5] = {0, 0, 0, 0, 0};
        auto read_counters = [&]() {
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const int i = lane + 32 * k;
                cnt[k] = i < tiles ? ld_u32_gpu(frame_prog + (size_t)i * CV_PROG_STRIDE + 1) : 0xffffffffu;
            }
        };
        auto publish_min = [&]() {
            unsigned m = min(min(min(cnt[0], cnt[1]), min(cnt[2], cnt[3])), cnt[4]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
            // atomicMax: this minimum may be older than one the receiver lane of this CTA has published while it
            // was held back; a bound that drops could hold back the very slot this one is waiting for
            if (lane == 0) { __threadfence(); atomicMax(gmin_out, m); }
            return m;
        };
        int next_b = 0, seen = -1, last_fence = -1000000, last_keep = -1000000;
        long long t_last = clock64();
        bool dead = false;
        for (;;) {
            int c = 0;
            if (lane == 0) c = *(volatile int *)&sm.cur_step;
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c == seen) {
                int bad = 0;
                if (lane == 0) bad = *(volatile int *)&sm.abort || clock64() - t_last > 4000000000LL;
                if (__shfl_sync(0xffffffffu, bad, 0)) { dead = true; break; }
                __nanosleep(40);
                continue;
            }
            seen = c;
            t_last = clock64();
            const bool fin = c >= total;
            if (lane == 0) {
                __threadfence_block();                               // acquire side of cur_step (CTA scope)
                st_u32_gpu(p.prog + (size_t)cta * CV_PROG_STRIDE, (unsigned)min(c, total - 1));
            }
            if (ordered && (fin || c - last_fence > p.fence_mask)) {
                last_fence = c;
                if (lane == 0) {
                    __threadfence();
                    st_u32_gpu(p.prog + (size_t)cta * CV_PROG_STRIDE + 1, (unsigned)(c + 1));
                }
            }
            if (keeper && (fin || c - last_keep > p.gmin_mask)) { last_keep = c; read_counters(); publish_min(); }
            if (fin) break;
            if (CV_BATCH * next_b + CV_AHEAD < total && c >= CV_BATCH * next_b) {
                cp_async_wait<0>();                                  // table entries fetched a batch ago
                __syncwarp();
                fetch_table(sm, p, CV_BATCH * next_b + 3 * CV_BATCH, lane, ci, cj, total);
                plan_steps(sm, p, CV_BATCH * next_b + CV_AHEAD, CV_BATCH, lane, total, frame_off_q, plane, p.frame0 + bl, geom, key);
                __threadfence_block();
                __syncwarp();
                if (lane == 0) *(volatile int *)&sm.planned = CV_BATCH * next_b + CV_AHEAD + CV_BATCH;
                ++next_b;
            }
        }
        cp_async_wait<0>();
        if (keeper && !dead) {
            // slower slots still need gmin: keep it until every counter has its final value (total + 1)
            const long long t0 = clock64();
            for (;;) {
                read_counters();
                if (publish_min() + 1 >= (unsigned)total || *(volatile int *)p.status != 0) break;
                if (clock64() - t0 > 4000000000LL) { atomicExch(p.status, 1); break; }
                __nanosleep(500);
            }
        }
    } else {
        // =============== receiver warp: arrivals of step g+1 into the tile ================================
        // The first two lines (two chunks each) of every step -- all there is in the usual step -- are located and
        // requested one step ahead, right after the deposit of the previous set; their geometry is kept in
        // registers.  (Requesting them earlier -- at the start of that step -- was measured: 42.5 ms against 38.8 ms
        // on C1.  The feeding tile is usually only just ahead, an early request misses its tag and pays a poll.)
        unsigned long long *const my_box = p.mbox + (size_t)cta * CV_D * CV_MBW;
        struct Pending { unsigned long long w[4]; int xi[4], wd[4]; bool ok[4]; };
        Pending pc{};
        int status_pend = 0;                         // lane 0: the failure flag, loaded a step ahead
        auto locate = [&](int step, Pending &q) {    // chunks 0..3 of `step` from the planner; requests their words
            const uint4 ln = *reinterpret_cast<const uint4 *>(&sm.desc[step % CV_DR].recv_a[0]);   // {a0, a1, b0, b1}
            const unsigned long long *box2 = my_box + (size_t)(step % CV_D) * CV_MBW;
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                const unsigned a = l ? ln.y : ln.x, b = l ? ln.w : ln.z;
                const unsigned var0 = b & 63u, len = (b >> 8) & 0xffu, sh = (b >> 16) & 0xffu;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const unsigned pos = (u << 5) + lane, v = (var0 + pos) & 63u;
                    q.ok[2 * l + u] = pos < len;
                    q.wd[2 * l + u] = (int)((a & 0xffffu) | v);
                    q.xi[2 * l + u] = (int)((a >> 16) | (v << sh));
                    q.w[2 * l + u] = ld_u64_gpu(box2 + q.wd[2 * l + u]);       // unconditional: nothing waits on it
                }
            }
        };
        if (total > 1) locate(1, pc);
#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 4
        long long rclk[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
        for (int g = 0; g < total; ++g) {
            CV_RCLK(0);
            if (g + 1 < total) {
                const unsigned long long *box = my_box + (size_t)((g + 1) % CV_D) * CV_MBW;
                const unsigned tag = (unsigned)(g + 1);
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (pc.ok[u]) {
                        unsigned long long w = pc.w[u];
                        if ((unsigned)(w >> 32) != tag) w = poll_tag(box + pc.wd[u], tag, p.status);
                        sm.xs[pc.xi[u]] = __uint_as_float((unsigned)w);
                    }
                // (lines beyond the second are received by the compute warps: help_handoff)
                CV_RCLK(1);
                __syncwarp();
                CV_RCLK(2);
                if (lane == 0) CV_STAMP(2);
                CV_RCLK(3);
                // (the services warp publishes "step g+1 has been read" when it sees the CTA in step g+1)
                CV_RCLK(4);
                if (g + 2 < total) locate(g + 2, pc);
            }
            if (lane == 0 && (g & 7) == 3) {
                if (status_pend) sm.abort = 1;
                status_pend = *(volatile int *)p.status;             // consumed 8 steps later
            }
            if (lane == 0) CV_STAMP(5);
            CV_RCLK(5);
            CV_STEP_BARRIER();
#if defined(SMRE_CV_TRACE_BUILD) && SMRE_CV_TRACE_BUILD == 4
            if (p.trace && lane == 0) {
                const long long t_end = clock64();
                for (int i = 1; i < 6; ++i) p.trace[((size_t)cta * total + g) * 8 + i] = (unsigned long long)(rclk[i] - rclk[0]);
                p.trace[((size_t)cta * total + g) * 8] = (unsigned long long)(t_end - rclk[0]);
            }
#endif
        }
    }

    // ---- a9: x_out <- the tile of the last step -----------------------------------------------------
    __syncthreads();                                             // the planner warp joins the others here
    {
        const AxisEntry ey = sm.tab[(total - 1) % CV_TR][0], ex = sm.tab[(total - 1) % CV_TR][1];
        const int h = ey.R - ey.L, w = ex.R - ex.L;
        for (int i = tid; i < h * w; i += CV_NT) {
            const int r = ey.L + i / w, c = ex.L + i % w;
            p.x_out[frame_off + (size_t)r * p.W + c] = sm.xs[tidx(r, c)];
        }
    }
}

using ConveyorKernel = void (*)(const CParams);
// q row pitches with their own instantiation (immediate row offsets in the q stores); 0 = run-time pitch
static ConveyorKernel kernel_for(int Wq)
{
    switch (Wq) {
        case 512: return conveyor_kernel<512>;
        case 256: return conveyor_kernel<256>;
        default: return conveyor_kernel<0>;
    }
}

// ---- host side ----------------------------------------------------------------------------------

// The fenced counters are refreshed every fence_mask + 1 steps (a fence costs ~1 us): at most a third of the lead
// a sweep allows.  gmin is recomputed from them every gmin_mask + 1 steps.
constexpr int CV_SVC_LAG = 4;      // steps the services warp may be late with a counter (it also plans: 2-3 us per batch)
static int fence_mask_for(int F)
{
    int m = 63;
    while (m > 3 && m + 2 + CV_SVC_LAG > (F - CV_PF - 2) / 3) m >>= 1;
    return m;
}

struct DeviceTables {             // boundary tables of one n_sweeps value, resident on the device
    int n_sweeps = 0;
    AxisEntry *d_y = nullptr, *d_x = nullptr;
};

struct ConveyorPlan {
    int H, W, Wq, B, F;
    int T_y, T_x, NR, NC;
    int frames_per_launch;
    ConveyorKernel kernel;
    int qp = 0;                         // columns of a TMA box = row pitch of a q stage
    CUtensorMap qmap[8];
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
    // q of a step is fetched CV_PF steps ahead of its use and was written one sweep (F steps) earlier
    if ((int)fams.size() < CV_PF + 3) return nullptr;
    int smax_f = 1;
    for (const Family &f : fams) smax_f = std::max(smax_f, f.side);
    if ((long long)fams.size() * B * H >= (1ll << 31)) return nullptr;          // tensor rows are 32-bit coordinates
    int dev = 0, n_sm = 0, smem_optin = 0, coop = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop || (size_t)smem_optin < sizeof(Smem)) return nullptr;
    const ConveyorKernel kernel = kernel_for((W + 3) & ~3);
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, CV_NT, sizeof(Smem)) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return nullptr;
    }
    const int capacity = per_sm * n_sm;
    ConveyorSummary cs;
    char why[160];
    // the tiling is chosen on a short run; tables_for() re-plans (and re-verifies) each real length
    if (!conveyor_summary(H, W, fams, 3, capacity, &cs, why, sizeof why)) return nullptr;
    // With several tiles a slot may lead the slowest slot by F - CV_PF - 2 steps minus the age of the fenced
    // counters (q ordering, see the control warp).  The tile that feeds another is at least one step ahead of it,
    // so the last tile leads the first by the length of the chain between them; a lead with no slack beyond that
    // would run, but in lock step.
    if (cs.tiles_y * cs.tiles_x > 1 &&
        (int)fams.size() - CV_PF - 2 - (fence_mask_for((int)fams.size()) + 2 + CV_SVC_LAG) < cs.tiles_y + cs.tiles_x + 4) return nullptr;

    ConveyorPlan *pl = new ConveyorPlan;
    pl->H = H; pl->W = W; pl->Wq = (W + 3) & ~3; pl->B = B; pl->F = (int)fams.size();
    pl->T_y = cs.T_y; pl->T_x = cs.T_x; pl->NR = cs.tiles_y; pl->NC = cs.tiles_x;
    pl->fams = fams; pl->q = q; pl->xwork = xwork; pl->kernel = kernel;
    {   // q as a 2-D fp32 tensor [F*B*H][Wq]; one map per box height 8, 16, .., 64 (plain layout, zero fill)
        typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                     const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                     CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
            cudaGetLastError();
            delete pl;
            return nullptr;
        }
        pl->qp = std::min(CV_PW, pl->Wq);
        const cuuint64_t gdim[2] = {(cuuint64_t)pl->Wq, (cuuint64_t)fams.size() * B * H};
        const cuuint64_t gstride[1] = {(cuuint64_t)pl->Wq * sizeof(float)};
        const cuuint32_t estr[2] = {1, 1};
        for (int k = 0; k < 8; ++k) {
            const cuuint32_t box[2] = {(cuuint32_t)pl->qp, (cuuint32_t)(8 * (k + 1))};
            if (((EncodeFn)fn)(&pl->qmap[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, q, gdim, gstride, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                               CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
                delete pl;
                return nullptr;
            }
        }
    }
    const int tiles = pl->NR * pl->NC;
    pl->frames_per_launch = std::max(1, std::min(B, capacity / tiles));
    std::vector<CFamily> cf(fams.size());
    for (size_t i = 0; i < fams.size(); ++i) {
        int lg = 0;
        while ((1 << lg) < fams[i].side) ++lg;
        size_t e = i;
        while (e + 1 < fams.size() && fams[e + 1].side == fams[i].side) ++e;
        cf[i] = CFamily{fams[i].side, lg, (int)(e - i + 1), 0, fams[i].c, fams[i].sqrt_c, {0, 0}};
    }
    const size_t n_cta = (size_t)pl->frames_per_launch * tiles;
    pl->mbox_bytes = n_cta * CV_D * CV_MBW * sizeof(unsigned long long);
    const bool good =
        cudaMalloc(&pl->d_fams, cf.size() * sizeof(CFamily)) == cudaSuccess &&
        cudaMalloc(&pl->d_mbox, pl->mbox_bytes) == cudaSuccess &&
        cudaMalloc(&pl->d_prog, (n_cta + pl->frames_per_launch) * CV_PROG_STRIDE * sizeof(unsigned)) == cudaSuccess &&
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
    p.NR = pl->NR; p.NC = pl->NC; p.qp = pl->qp; p.fence_mask = fence_mask_for(pl->F);
    p.gmin_mask = std::min(p.fence_mask, 15);
    p.gmin = pl->d_prog + (size_t)pl->frames_per_launch * pl->NR * pl->NC * CV_PROG_STRIDE;
    memcpy(p.qmap, pl->qmap, sizeof p.qmap);
    const int tiles = pl->NR * pl->NC;
    if ((e = cudaMemsetAsync(pl->d_status, 0, sizeof(int), st)) != cudaSuccess) return e;   // health flag of THIS run
#ifdef SMRE_CV_TRACE_BUILD                                  // debug builds only: synchronises and writes a file
    const char *trace_path = getenv("SMRE_CV_TRACE");
    if (trace_path && cudaMalloc(&p.trace, (size_t)tiles * p.total * 64) != cudaSuccess) p.trace = nullptr;
#endif
    for (int f0 = 0; f0 < pl->B; f0 += pl->frames_per_launch) {
        p.frame0 = f0;
        const int nb = std::min(pl->frames_per_launch, pl->B - f0);
        // tags and progress counters restart in every launch
        if ((e = cudaMemsetAsync(pl->d_mbox, 0, (size_t)nb * tiles * CV_D * CV_MBW * 8, st)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(pl->d_prog, 0, (size_t)pl->frames_per_launch * (tiles + 1) * CV_PROG_STRIDE * sizeof(unsigned), st)) != cudaSuccess) return e;
        void *args[] = {&p};
        e = cudaLaunchCooperativeKernel((const void *)pl->kernel, dim3((unsigned)(nb * tiles)),
                                        dim3(CV_NT), args, sizeof(Smem), st);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
#ifdef SMRE_CV_TRACE_BUILD
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
#endif
    return cudaSuccess;
}

}  // namespace smre
