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
    unsigned *prog;               // [n_cta] "mailbox read up to and including step"
    int *status;                  // != 0: a poll timed out somewhere (protocol bug) -> everybody leaves
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
    float xs[CV_PW * CV_PW];                 // the x tile, torus addressed
    float qs[CV_NST][CV_PW * CV_PW];         // q stages, same addressing
    AxisEntry tab[CV_TR][2];                 // [step % CV_TR][0 = y, 1 = x]
    CFamily fams[CV_MAX_F];
    unsigned nbr_prog[4];                    // cached progress of the left / up / up-left CTAs
};

// Arrival i of the step described by (ey, ex): pixel and mailbox word.  Column strip first
// (all tile rows x columns [ex.A, ex.R)), then the row strip (rows [ey.A, ey.R) x columns [ex.L, ex.A)).
__device__ __forceinline__ void arrival(const AxisEntry &ey, const AxisEntry &ex, int i, int n_col,
                                        int &r, int &c, int &word) {
    const int h = ey.R - ey.L;
    if (i < n_col) {
        const int k = i / h;
        c = ex.A + k; r = ey.L + (i - k * h);
        word = mbox_col_word(r, c);
    } else {
        const int w = ex.A - ex.L, j = i - n_col;
        const int k = j / w;
        r = ey.A + k; c = ex.L + (j - k * w);
        word = mbox_row_word(r, c);
    }
}

// The windows of one step inside this CTA's tile.  G = lanes per window (power of two >= side); lane j
// of a window owns column j and keeps the `side` values of that column in registers.
template <int G>
__device__ __forceinline__ void project_tile(Smem &sm, const float *qst, float *__restrict__ qplane,
                                             const AxisEntry &ey, const AxisEntry &ex, const CFamily &fam,
                                             int W, bool first_sweep)
{
    const int s = fam.side;
    const int nwx = ex.nw;
    const int n_items = ey.nw * nwx * G;
    for (int base = 0; base < n_items; base += CV_NT) {
        if (base + (int)(threadIdx.x & ~31u) >= n_items) break;        // warp-uniform: nothing left
        const int item = base + threadIdx.x;
        const int win = item / G, j = item % G;
        const int wiy = (int)(((unsigned)win * ex.magic) >> 20), wix = win - wiy * nwx;
        const bool on = item < n_items && j < s;
        const int r0 = ey.w0 + wiy * s, c = ex.w0 + wix * s + j;
        const int i0 = tidx(r0, c);
        float *qg = qplane + (size_t)r0 * W + c;
        float v[G];
        float part = 0.0f;
#pragma unroll
        for (int r = 0; r < G; ++r) {
            v[r] = 0.0f;
            if (r < s && on) {
                const int i = (i0 + (r << 6)) & (CV_PW * CV_PW - 1);
                v[r] = sm.xs[i] + (first_sweep ? 0.0f : qst[i]);
            }
            part = fmaf(v[r], v[r], part);
        }
#pragma unroll
        for (int m = G / 2; m > 0; m >>= 1) part += __shfl_xor_sync(0xffffffffu, part, m);
        const float alpha = ball_scale(part, fam.c, fam.sqrt_c);
#pragma unroll
        for (int r = 0; r < G; ++r) {
            if (r < s && on) {
                const int i = (i0 + (r << 6)) & (CV_PW * CV_PW - 1);
                const float xn = alpha * v[r];
                sm.xs[i] = xn;
                __stcs(qg + (size_t)r * W, v[r] - xn);
            }
        }
    }
}

__global__ void __launch_bounds__(CV_NT, 1)
conveyor_kernel(const __grid_constant__ CParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);
    const int tid = threadIdx.x;
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
    if (tid < 4) sm.nbr_prog[tid] = 0;
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

    unsigned long long pend = 0;      // mailbox word loaded ahead of time (arrival index NT-1-tid)
    unsigned prog_pend = 0;           // neighbour progress loaded ahead of time (tid 1..3)
    int status_pend = 0;              // status flag loaded ahead of time (tid 0)
    int f = 0;                        // family of step g
    int fp = CV_PF % p.F;             // family of step g + CV_PF
    const int hi = CV_NT - 1 - tid;   // hand-off duties go to the highest threads first

    for (int g = 0; g < total; ++g) {
        const AxisEntry ey = sm.tab[g % CV_TR][0], ex = sm.tab[g % CV_TR][1];
        const CFamily fam = sm.fams[f];

        // ---- (f) departures of step g-1 -> the neighbours' mailboxes, tagged g -----------------------
        if (g > 0) {
            const AxisEntry py = sm.tab[(g - 1) % CV_TR][0], px = sm.tab[(g - 1) % CV_TR][1];
            const int h = py.R - py.L, w = px.R - px.L;
            const int n_col = h * (px.D - px.L);                    // columns [L, D), all rows
            const int n_row = (py.D - py.L) * (px.R - px.D);         // rows [L, D), columns [D, R)
            const int n_dep = n_col + n_row;
            (void)w;
            for (int i = hi; i < n_dep; i += CV_NT) {
                int r, c, word;
                if (i < n_col) {
                    const int k = i / h;
                    c = px.L + k; r = py.L + (i - k * h);
                    word = mbox_col_word(r, c);
                } else {
                    const int ww = px.R - px.D, j = i - n_col;
                    const int k = j / ww;
                    r = py.L + k; c = px.D + (j - k * ww);
                    word = mbox_row_word(r, c);
                }
                const int which = (c < px.D ? 1 : 0) | (r < py.D ? 2 : 0);    // 1 left, 2 up, 3 up-left
                if ((int)sm.nbr_prog[which] + CV_D < g)              // ring slot still unread by the receiver?
                    poll_prog(p.prog + nbr_cta(which), (unsigned)(g - CV_D), p.status);
                const unsigned long long wv = ((unsigned long long)(unsigned)g << 32) | __float_as_uint(sm.xs[tidx(r, c)]);
                st_u64_gpu(p.mbox + ((size_t)nbr_cta(which) * CV_D + (g % CV_D)) * CV_MBW + word, wv);
            }
        }

        // ---- (a) prefetch q of step g + CV_PF and the table entry of step g + CV_LA ---------------------
        {
            const int gp = g + CV_PF;
            if (gp < total && gp >= p.F) {                           // the first sweep reads no q (q = 0)
                const AxisEntry qy = sm.tab[gp % CV_TR][0], qx = sm.tab[gp % CV_TR][1];
                const CFamily qf = sm.fams[fp];
                if (qy.nw > 0 && qx.nw > 0) {
                    const int rows = qy.nw * qf.side;
                    const int c0 = qx.w0 & ~3, c1 = (qx.w0 + qx.nw * qf.side + 3) & ~3;
                    const int nch = (c1 - c0) >> 2;
                    const float *src = p.q + (size_t)fp * plane + frame_off_q;
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(sm.qs[gp % CV_NST]);
                    for (int i = tid; i < rows * nch; i += CV_NT) {
                        const int rr = i / nch, ch = i - rr * nch;
                        const int r = qy.w0 + rr, c = c0 + 4 * ch;
                        if (c < p.Wq)
                            cp_async16(dst + 4u * (unsigned)tidx(r, c), src + (size_t)r * p.Wq + c);
                    }
                }
            }
            const int gt = g + CV_LA + 1;
            if (gt < total && tid < 2) {
                const AxisEntry *src = tid ? p.tabx + (size_t)gt * p.NC + cj : p.taby + (size_t)gt * p.NR + ci;
                cp_async16((unsigned)__cvta_generic_to_shared(&sm.tab[gt % CV_TR][tid]), src);
            }
            cp_async_commit();
        }

        // ---- (c) the windows of step g ----------------------------------------------------------------
        if (ey.nw > 0 && ex.nw > 0) {
            float *qplane = p.q + (size_t)f * plane + frame_off_q;
            const float *qst = sm.qs[g % CV_NST];
            const bool first = g < p.F;
            switch (fam.G) {
                case 1: project_tile<1>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
                case 2: project_tile<2>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
                case 4: project_tile<4>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
                case 8: project_tile<8>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
                case 16: project_tile<16>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
                default: project_tile<32>(sm, qst, qplane, ey, ex, fam, p.Wq, first); break;
            }
        }

        // ---- (d) arrivals of step g+1 into the tile; start loading the arrivals of step g+2 ------------
        if (g + 1 < total) {
            const AxisEntry ny = sm.tab[(g + 1) % CV_TR][0], nx = sm.tab[(g + 1) % CV_TR][1];
            const int n_col = (ny.R - ny.L) * (nx.R - nx.A);
            const int n_arr = n_col + (ny.R - ny.A) * (nx.A - nx.L);
            const unsigned long long *box = my_box + (size_t)((g + 1) % CV_D) * CV_MBW;
            for (int i = hi; i < n_arr; i += CV_NT) {
                int r, c, word;
                arrival(ny, nx, i, n_col, r, c, word);
                unsigned long long wv = (i == hi) ? pend : 0ull;
                if ((unsigned)(wv >> 32) != (unsigned)(g + 1)) wv = poll_tag(box + word, (unsigned)(g + 1), p.status);
                sm.xs[tidx(r, c)] = __uint_as_float((unsigned)wv);
            }
            pend = 0;
            if (g + 2 < total) {
                const AxisEntry my = sm.tab[(g + 2) % CV_TR][0], mx = sm.tab[(g + 2) % CV_TR][1];
                const int m_col = (my.R - my.L) * (mx.R - mx.A);
                const int m_arr = m_col + (my.R - my.A) * (mx.A - mx.L);
                if (hi < m_arr) {
                    int r, c, word;
                    arrival(my, mx, hi, m_col, r, c, word);
                    pend = ld_u64_gpu(my_box + (size_t)((g + 2) % CV_D) * CV_MBW + word);
                }
            }
        }

        // ---- bookkeeping loads, consumed one iteration later ------------------------------------------
        int bad = 0;
        if (tid == 0) { bad = status_pend; status_pend = *(volatile int *)p.status; }
        if (tid >= 1 && tid <= 3) {
            sm.nbr_prog[tid] = prog_pend;
            prog_pend = ld_u32_gpu(p.prog + nbr_cta(tid));
        }

        // ---- (e) one barrier per step; q of step g+1 has landed -----------------------------------------
        cp_async_wait<CV_PF - 1>();
        if (__syncthreads_or(bad)) return;
        if (tid == 0) st_u32_gpu(p.prog + cta, (unsigned)(g + 1));   // mailbox of step g+1 has been read

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
        cudaMalloc(&pl->d_prog, n_cta * sizeof(unsigned)) == cudaSuccess &&
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
    for (int f0 = 0; f0 < pl->B; f0 += pl->frames_per_launch) {
        p.frame0 = f0;
        const int nb = std::min(pl->frames_per_launch, pl->B - f0);
        // tags and progress counters restart in every launch
        if ((e = cudaMemsetAsync(pl->d_mbox, 0, (size_t)nb * tiles * CV_D * CV_MBW * 8, st)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(pl->d_prog, 0, (size_t)nb * tiles * sizeof(unsigned), st)) != cudaSuccess) return e;
        void *args[] = {&p};
        e = cudaLaunchCooperativeKernel((const void *)conveyor_kernel, dim3((unsigned)(nb * tiles)),
                                        dim3(CV_NT), args, sizeof(Smem), st);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
    return cudaSuccess;
}

}  // namespace smre
