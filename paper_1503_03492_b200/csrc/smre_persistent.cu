// Persistent sweep scheduler: ONE cooperative kernel runs all
// n_sweeps * F strictly ordered family passes of the standard variant.
//
// Why: a family pass of the 512^2 config moves 2 MiB of q -- 0.32 us of HBM time -- so a kernel
// boundary or a grid-wide barrier per family (1-2.5 us) caps the path near 10-25 % of the HBM
// roofline.  The dependency between consecutive families is LOCAL (a window overlaps only windows
// within side-1 pixels), so the grid barrier is replaced by neighbour hand-off:
//
//  * the image is cut into a grid of tiles, one CTA per tile, all co-resident (cooperative launch);
//    a CTA keeps its tile of x, extended by a halo of h = max_side-1 pixels to the right and below,
//    in SHARED MEMORY for the whole call; x never touches HBM between the first and last step;
//  * a window belongs to the CTA whose tile contains its origin (top-left pixel), so every window
//    is computed exactly once and its q is read and written by one fixed thread: q streams
//    HBM -> registers -> HBM, prefetched into L2 a few families ahead (its addresses do not depend
//    on x);
//  * a pixel is "held" by its home CTA and by the left / upper / upper-left neighbours whose halo
//    covers it.  Whoever computes a pixel sends the new value to the other holders through a
//    mailbox in global memory (L2): one 8-byte word {value, step tag} per pixel, written with a
//    single store and polled by the receiver (no separate flag, no fence: one L2 round trip).
//    The receiver knows from the family geometry exactly which words to wait for;
//  * one __syncthreads per family step; a one-word heartbeat per neighbour and step keeps
//    neighbours within one step of each other, which makes a 4-deep mailbox ring sufficient.
//
// The per-window arithmetic and its summation order are those of family_pass_kernel, so both
// schedulers return identical bits.
#include "smre_persistent.cuh"

#include <cooperative_groups.h>
#include <cassert>
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#ifdef SMRE_DEBUG
#define SMRE_CHECK(cond) assert(cond)
#else
#define SMRE_CHECK(cond) ((void)0)
#endif

namespace smre {

constexpr int NSLOT = 4;          // mailbox ring depth (>= 2 needed, see header comment)
constexpr int MAX_TILES_1D = 160;
constexpr int PF_STEPS = 6;       // L2 prefetch distance for q, in family steps

struct PFamily {                  // device copy of a family, plus a division magic
    int side, oy, ox, ny, nx;
    float c, sqrt_c;
    unsigned magic;               // floor(n / side) == (n * magic) >> 20 for n < 2^15
    int G;                        // lanes per window: next power of two >= side
};

struct PParams {
    const float *y;               // [B][H][W] input
    float *x_out;                 // [B][H][W] result
    float *q;                     // [F][B][H][W] increment planes
    const PFamily *fams;
    unsigned long long *mbox;     // [n_cta][NSLOT][mbox_stride] words {tag:32 | value:32}
    int *status;                  // device flag: != 0 -> a poll timed out (protocol bug)
    int F, n_sweeps;
    int H, W, B;                  // B = frames in this launch
    int frame0;                   // first frame of this launch inside the full batch
    int B_total;
    int gy, gx;                   // tile grid
    int h;                        // halo = max side - 1
    int pitch;                    // shared-memory row pitch of the x tile (same for every CTA)
    int eh_max;                   // max extended tile height
    int mbox_stride;              // eh_max * pitch + 8 heartbeat words
    short yb[MAX_TILES_1D + 1];   // tile row boundaries
    short xb[MAX_TILES_1D + 1];   // tile column boundaries
};

struct PersistentPlan {
    int H, W, B, F;
    int gy, gx, h, pitch, eh_max, mbox_stride, threads;
    int frames_per_launch;
    size_t smem_bytes;
    std::vector<short> yb, xb;
    float *q, *xwork;
    PFamily *d_fams = nullptr;
    unsigned long long *d_mbox = nullptr;
    size_t mbox_bytes = 0;
    int *d_status = nullptr;
};


// ---- mailbox words: one 64-bit store / load, relaxed, gpu scope (served by L2) -----------------
__device__ __forceinline__ unsigned long long ld_mbox(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_mbox(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void *p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// Spin until the word carries `tag`; returns its payload.  A poll that outlives ~1 s of SM clocks
// (or sees another CTA's failure) raises *status and gives up, so a protocol bug cannot hang the GPU.
__device__ __noinline__ float poll_word(const unsigned long long *p, unsigned tag, int *status) {
    unsigned long long v = ld_mbox(p);
    if ((unsigned)(v >> 32) == tag) return __uint_as_float((unsigned)v);
    const long long t0 = clock64();
    for (unsigned spins = 1;; ++spins) {
        v = ld_mbox(p);
        if ((unsigned)(v >> 32) == tag) break;
        if ((spins & 255u) == 0) {
            if (*(volatile int *)status != 0) return 0.0f;
            if (clock64() - t0 > 2000000000LL) { atomicExch(status, 1); return 0.0f; }
        }
    }
    return __uint_as_float((unsigned)v);
}

struct TileCtx {
    int ty, tx, bl;               // tile coordinates, frame index inside this launch
    int y0, y1, x0, x1;           // home region
    int th, tw, eh, ew;           // home and extended (home + right/bottom halo) sizes
    int cta;                      // linear CTA id = (bl*gy + ty)*gx + tx
    size_t frame_off;             // element offset of this frame inside a [B_total][H][W] plane set
    float *xs;                    // shared: x tile, pitch p.pitch
    unsigned char *hold;          // shared: per pixel, which of the 8 neighbours also hold it
    unsigned *shared_list;        // shared: (ly << 16 | lx) of every pixel with hold != 0
    int n_shared;
};

// direction d in 0..7 <-> (dy, dx) in {-1,0,1}^2 \ {(0,0)}: d9 = (dy+1)*3 + (dx+1), d = d9 - (d9 > 4)
__device__ __forceinline__ int dir_dy(int d) { int d9 = d + (d >= 4); return d9 / 3 - 1; }
__device__ __forceinline__ int dir_dx(int d) { int d9 = d + (d >= 4); return d9 % 3 - 1; }

__device__ __forceinline__ int div_magic(int n, unsigned magic) { return (int)(((unsigned)n * magic) >> 20); }

// Windows of family `fam` whose origin lies in [lo, hi) along one axis (o = offset, n = number of
// windows of the family along the axis): first origin and count.
__device__ __forceinline__ void owned_range(int lo, int hi, int o, int n, int s, unsigned magic,
                                            int &first, int &count) {
    first = (lo <= o) ? o : o + div_magic(lo - o + s - 1, magic) * s;
    const int last = min(hi - 1, o + (n - 1) * s);
    count = (n > 0 && first <= last) ? div_magic(last - first, magic) + 1 : 0;
}

// Receive phase: apply every value that another CTA computed in step (g-1) (family fam, tag g) to
// the shared-memory tile, and wait for the neighbours' heartbeats of that step.
__device__ __forceinline__ void receive_step(const PParams &p, const TileCtx &c, const PFamily &fam,
                                             unsigned tag, int slot, bool heartbeats) {
    const unsigned long long *box = p.mbox + ((size_t)c.cta * NSLOT + slot) * p.mbox_stride;
    for (int i = threadIdx.x; i < c.n_shared; i += blockDim.x) {
        const unsigned e = c.shared_list[i];
        const int ly = (int)(e >> 16), lx = (int)(e & 0xffffu);
        const int py = c.y0 + ly, px = c.x0 + lx;
        if (py < fam.oy || px < fam.ox) continue;
        const int iy = div_magic(py - fam.oy, fam.magic), ix = div_magic(px - fam.ox, fam.magic);
        if (iy >= fam.ny || ix >= fam.nx) continue;                  // not covered: unchanged
        const int wy = fam.oy + iy * fam.side, wx = fam.ox + ix * fam.side;
        const int hy = c.ty + (ly >= c.th), hx = c.tx + (lx >= c.tw);  // home tile of the pixel
        const int oty = hy - (wy < p.yb[hy]), otx = hx - (wx < p.xb[hx]);   // owner of its window
        if (oty == c.ty && otx == c.tx) continue;                    // computed here
        SMRE_CHECK(ly < c.eh && lx < c.ew && ly * p.pitch + lx < p.eh_max * p.pitch);
        c.xs[ly * p.pitch + lx] = poll_word(box + ly * p.pitch + lx, tag, p.status);
    }
    if (heartbeats && threadIdx.x < 8) {
        const int d = threadIdx.x;
        const int nty = c.ty + dir_dy(d), ntx = c.tx + dir_dx(d);
        if (nty >= 0 && nty < p.gy && ntx >= 0 && ntx < p.gx)
            poll_word(box + p.eh_max * p.pitch + (7 - d), tag, p.status);
    }
}

__device__ __forceinline__ void send_heartbeats(const PParams &p, const TileCtx &c, unsigned tag, int slot) {
    if (threadIdx.x < 8) {
        const int d = threadIdx.x;
        const int nty = c.ty + dir_dy(d), ntx = c.tx + dir_dx(d);
        if (nty >= 0 && nty < p.gy && ntx >= 0 && ntx < p.gx) {
            const int nb = (c.bl * p.gy + nty) * p.gx + ntx;
            st_mbox(p.mbox + ((size_t)nb * NSLOT + slot) * p.mbox_stride + p.eh_max * p.pitch + d,
                    (unsigned long long)tag << 32);
        }
    }
}

// Pull the q rectangle this CTA will need PF_STEPS families from now towards L2 (one warp).
__device__ __forceinline__ void prefetch_family(const PParams &p, const TileCtx &c, const PFamily &fam,
                                                int f) {
    int wy0, nwy, wx0, nwx;
    owned_range(c.y0, c.y1, fam.oy, fam.ny, fam.side, fam.magic, wy0, nwy);
    owned_range(c.x0, c.x1, fam.ox, fam.nx, fam.side, fam.magic, wx0, nwx);
    if (nwy == 0 || nwx == 0) return;
    const int rows = nwy * fam.side, cols = nwx * fam.side;
    const float *base = p.q + ((size_t)f * p.B_total) * p.H * p.W + c.frame_off + (size_t)wy0 * p.W + wx0;
    const int lane = threadIdx.x & 31;
    for (int r = lane; r < rows; r += 32) {
        const char *a = (const char *)(base + (size_t)r * p.W);
        const char *end = a + cols * 4;
        for (const char *l = (const char *)((uintptr_t)a & ~(uintptr_t)127); l < end; l += 128) prefetch_l2(l);
    }
}

// Send the new value of pixel (ly, lx) of this tile to every other CTA that holds it.
__device__ __forceinline__ void send_pixel(const PParams &p, const TileCtx &c, int ly, int lx, float val,
                                           unsigned mask, unsigned tag, int slot) {
    const int py = c.y0 + ly, px = c.x0 + lx;
    const unsigned long long word = ((unsigned long long)tag << 32) | __float_as_uint(val);
    while (mask) {
        const int d = __ffs(mask) - 1;
        mask &= mask - 1;
        const int nty = c.ty + dir_dy(d), ntx = c.tx + dir_dx(d);
        const int nb = (c.bl * p.gy + nty) * p.gx + ntx;
        const int idx = (py - p.yb[nty]) * p.pitch + (px - p.xb[ntx]);
        SMRE_CHECK(nty >= 0 && nty < p.gy && ntx >= 0 && ntx < p.gx);
        SMRE_CHECK(py - p.yb[nty] >= 0 && py - p.yb[nty] < p.eh_max && px - p.xb[ntx] >= 0 && px - p.xb[ntx] < p.pitch);
        st_mbox(p.mbox + ((size_t)nb * NSLOT + slot) * p.mbox_stride + idx, word);
    }
}

// One family step g of one CTA.  G = lanes per window (power of two >= side); lane j of a window
// owns column j and keeps the `side` values of that column in registers -- the mapping and the
// summation order of family_pass_kernel.
template <int G>
__device__ __forceinline__ bool family_step(const PParams &p, const TileCtx &c, const PFamily &fam,
                                            const PFamily &prev, int f, int g, bool first_sweep)
{
    const int s = fam.side;
    int wy0, nwy, wx0, nwx;
    owned_range(c.y0, c.y1, fam.oy, fam.ny, s, fam.magic, wy0, nwy);
    owned_range(c.x0, c.x1, fam.ox, fam.nx, s, fam.magic, wx0, nwx);
    const int n_items = nwy * nwx * G;
    const int nwx_div = max(nwx, 1);   // never divide by zero: it is UB, and lets the compiler assume nwx != 0
    float *qplane = p.q + ((size_t)f * p.B_total) * p.H * p.W + c.frame_off;
    const unsigned tag = (unsigned)g + 1u;
    const int slot = g & (NSLOT - 1);
    const int nt = blockDim.x;

    // item -> (smem index of the column's first pixel, global q index, predicate)
    auto locate = [&](int item, int &e0, size_t &gq, int &ly0, int &lx) -> bool {
        const int win = item / G, j = item % G;
        const int wiy = win / nwx_div, wix = win - wiy * nwx;
        const bool on = item < n_items && j < s;
        ly0 = wy0 + wiy * s - c.y0;
        lx = wx0 + wix * s + j - c.x0;
        e0 = ly0 * p.pitch + lx;
        gq = (size_t)(c.y0 + ly0) * p.W + (size_t)(c.x0 + lx);
        return on;
    };
    auto load_q = [&](bool on, size_t gq, float (&qv)[G]) {
#pragma unroll
        for (int r = 0; r < G; ++r)
        {
            SMRE_CHECK(!(r < s && on) || gq + (size_t)r * p.W < (size_t)p.H * p.W);
            qv[r] = (r < s && on && !first_sweep) ? __ldcs(qplane + gq + (size_t)r * p.W) : 0.0f;
        }
    };

    // (1) issue this step's first q loads before waiting on the neighbours: q does not depend on x
    int e0, ly0, lx;
    size_t gq;
    float qv[G];
    bool on = locate(threadIdx.x, e0, gq, ly0, lx);
    load_q(on, gq, qv);

    // (2) values computed elsewhere in step g-1, then one barrier for the whole step
    if (g > 0) receive_step(p, c, prev, (unsigned)g, (g - 1) & (NSLOT - 1), true);
    const int bad = *(volatile int *)p.status;
    if (__syncthreads_or(bad)) return false;
    send_heartbeats(p, c, tag, slot);

    // (3) the windows this CTA owns
    for (int base = 0; base < n_items; base += nt) {
        if (base > 0) {
            on = locate(base + threadIdx.x, e0, gq, ly0, lx);
            load_q(on, gq, qv);
        }
        if (base + (int)(threadIdx.x & ~31u) >= n_items) break;      // warp-uniform: nothing left
        float v[G];
        float part = 0.0f;
#pragma unroll
        for (int r = 0; r < G; ++r) {
            v[r] = 0.0f;
            if (r < s && on) {
                SMRE_CHECK(ly0 >= 0 && ly0 + r < c.eh && lx >= 0 && lx < c.ew);
                v[r] = c.xs[e0 + r * p.pitch] + qv[r];
            }
            part = fmaf(v[r], v[r], part);
        }
#pragma unroll
        for (int m = G / 2; m > 0; m >>= 1) part += __shfl_xor_sync(0xffffffffu, part, m);
        const float alpha = ball_scale(part, fam.c, fam.sqrt_c);
#pragma unroll
        for (int r = 0; r < G; ++r) {
            if (r < s && on) {
                const float xn = alpha * v[r];
                const int e = e0 + r * p.pitch;
                c.xs[e] = xn;
                __stcs(qplane + gq + (size_t)r * p.W, v[r] - xn);
                const unsigned mask = c.hold[e];
                if (mask) send_pixel(p, c, ly0 + r, lx, xn, mask, tag, slot);
            }
        }
    }
    return true;
}

__global__ void __launch_bounds__(512, 1)
persistent_sweep_kernel(const __grid_constant__ PParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int n_shared_s;
    const int tile_px = p.eh_max * p.pitch;

    TileCtx c;
    c.xs = reinterpret_cast<float *>(smem_raw);
    c.shared_list = reinterpret_cast<unsigned *>(smem_raw + (size_t)tile_px * 4);
    c.hold = smem_raw + (size_t)tile_px * 8;
    c.cta = blockIdx.x;
    c.bl = c.cta / (p.gy * p.gx);
    const int t2 = c.cta - c.bl * p.gy * p.gx;
    c.ty = t2 / p.gx;
    c.tx = t2 - c.ty * p.gx;
    c.y0 = p.yb[c.ty]; c.y1 = p.yb[c.ty + 1];
    c.x0 = p.xb[c.tx]; c.x1 = p.xb[c.tx + 1];
    c.th = c.y1 - c.y0; c.tw = c.x1 - c.x0;
    c.eh = min(c.y1 + p.h, p.H) - c.y0;
    c.ew = min(c.x1 + p.h, p.W) - c.x0;
    c.frame_off = (size_t)(p.frame0 + c.bl) * p.H * p.W;

    // ---- a1: x <- y for this tile (home + halo); who else holds each pixel ----------------------
    if (threadIdx.x == 0) n_shared_s = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < c.eh * c.ew; i += blockDim.x) {
        const int ly = i / c.ew, lx = i - ly * c.ew;
        c.xs[ly * p.pitch + lx] = p.y[c.frame_off + (size_t)(c.y0 + ly) * p.W + (c.x0 + lx)];
        const int hy = c.ty + (ly >= c.th), hx = c.tx + (lx >= c.tw);
        const int ry = c.y0 + ly - p.yb[hy], rx = c.x0 + lx - p.xb[hx];
        unsigned mask = 0;
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                const bool holds = (a == 0 || (ry < p.h && hy > 0)) && (b == 0 || (rx < p.h && hx > 0));
                const int dy = hy - a - c.ty, dx = hx - b - c.tx;
                if (holds && (dy != 0 || dx != 0)) {
                    const int d9 = (dy + 1) * 3 + (dx + 1);
                    mask |= 1u << (d9 - (d9 > 4));
                }
            }
        c.hold[ly * p.pitch + lx] = (unsigned char)mask;
        if (mask) c.shared_list[atomicAdd(&n_shared_s, 1)] = ((unsigned)ly << 16) | (unsigned)lx;
    }
    __syncthreads();
    c.n_shared = n_shared_s;

    // ---- a3: the ordered family sequence, n_sweeps times, no host round trip ---------------------
    const int total = p.n_sweeps * p.F;
    const bool pf_warp = (threadIdx.x >> 5) == (blockDim.x >> 5) - 1;
    PFamily prev = p.fams[0];
    int f = 0;
    bool ok = true;
    for (int g = 0; g < total && ok; ++g) {
        const PFamily fam = p.fams[f];
        if (pf_warp && g + PF_STEPS < total && g + PF_STEPS >= p.F) {
            int fp = f + PF_STEPS;
            while (fp >= p.F) fp -= p.F;
            prefetch_family(p, c, p.fams[fp], fp);
        }
        const bool first = g < p.F;
        switch (fam.G) {
            case 1: ok = family_step<1>(p, c, fam, prev, f, g, first); break;
            case 2: ok = family_step<2>(p, c, fam, prev, f, g, first); break;
            case 4: ok = family_step<4>(p, c, fam, prev, f, g, first); break;
            case 8: ok = family_step<8>(p, c, fam, prev, f, g, first); break;
            case 16: ok = family_step<16>(p, c, fam, prev, f, g, first); break;
            default: ok = family_step<32>(p, c, fam, prev, f, g, first); break;
        }
        prev = fam;
        if (++f == p.F) f = 0;
    }

    // ---- a9: values the neighbours computed in the last step, then x_out <- home region ---------
    if (ok) receive_step(p, c, prev, (unsigned)total, (total - 1) & (NSLOT - 1), false);
    __syncthreads();
    for (int i = threadIdx.x; i < c.th * c.tw; i += blockDim.x) {
        const int ly = i / c.tw, lx = i - ly * c.tw;
        p.x_out[c.frame_off + (size_t)(c.y0 + ly) * p.W + (c.x0 + lx)] = c.xs[ly * p.pitch + lx];
    }
}

// ---- host side ----------------------------------------------------------------------------------

static size_t tile_smem_bytes(int eh, int pitch) { return (size_t)eh * pitch * 9 + 16; }

static std::vector<short> split(int n, int parts) {
    std::vector<short> b(parts + 1);
    for (int i = 0; i <= parts; ++i) b[i] = (short)(((long long)i * n + parts / 2) / parts);
    return b;
}

PersistentPlan *persistent_plan_create(int H, int W, int B, const std::vector<Family> &fams,
                                       float *q, float *xwork)
{
    if (fams.empty() || H > 32000 || W > 32000) return nullptr;
    int dev = 0, n_sm = 0, smem_optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) return nullptr;

    int smax = 1;
    for (const Family &f : fams) smax = std::max(smax, f.side);
    const int h = smax - 1;
    const int min_dim = std::max(h, 1);
    int threads = 512;
    if (const char *e = getenv("SMRE_THREADS")) threads = std::max(64, std::min(512, atoi(e) / 32 * 32));

    // Tile grid: minimise a per-step cost model  t = t_fixed + px(extended tile) * t_px (+ t_sync if
    // more than one tile), over the grids that fit one CTA per SM (all frames of a launch resident).
    int best_gy = 0, best_gx = 0;
    double best_cost = 1e30;
    const size_t smem_limit = (size_t)smem_optin - 1024;
    int force_gy = 0, force_gx = 0;
    if (const char *e = getenv("SMRE_TILES")) sscanf(e, "%d,%d", &force_gy, &force_gx);
    for (int gy = 1; gy <= std::min(H / min_dim, MAX_TILES_1D); ++gy)
        for (int gx = 1; gx <= std::min(W / min_dim, MAX_TILES_1D); ++gx) {
            if (gy * gx > n_sm) continue;
            if (force_gy && (gy != force_gy || gx != force_gx)) continue;
            const std::vector<short> yb = split(H, gy), xb = split(W, gx);
            int th = 0, tw = 0, thmin = 1 << 30, twmin = 1 << 30;
            for (int i = 0; i < gy; ++i) { th = std::max(th, yb[i + 1] - yb[i]); thmin = std::min(thmin, yb[i + 1] - yb[i]); }
            for (int i = 0; i < gx; ++i) { tw = std::max(tw, xb[i + 1] - xb[i]); twmin = std::min(twmin, xb[i + 1] - xb[i]); }
            if (thmin < min_dim || twmin < min_dim) continue;
            const int eh = std::min(th + h, H), ew = std::min(tw + h, W);
            if (eh > 65535 || ew > 65535 || tile_smem_bytes(eh, ew | 1) > smem_limit) continue;
            double cost = 250.0 + 0.30 * eh * ew * (512.0 / threads) + (gy * gx > 1 ? 600.0 : 0.0);
            if (tw % 8) cost += 10.0;                       // prefer sector-aligned tile columns
            if (cost < best_cost) { best_cost = cost; best_gy = gy; best_gx = gx; }
        }
    if (!best_gy) return nullptr;

    PersistentPlan *pl = new PersistentPlan;
    pl->H = H; pl->W = W; pl->B = B; pl->F = (int)fams.size();
    pl->gy = best_gy; pl->gx = best_gx; pl->h = h; pl->threads = threads;
    pl->yb = split(H, best_gy); pl->xb = split(W, best_gx);
    int th = 0, tw = 0;
    for (int i = 0; i < best_gy; ++i) th = std::max(th, pl->yb[i + 1] - pl->yb[i]);
    for (int i = 0; i < best_gx; ++i) tw = std::max(tw, pl->xb[i + 1] - pl->xb[i]);
    pl->eh_max = std::min(th + h, H);
    pl->pitch = std::min(tw + h, W) | 1;                    // odd pitch: rows fall on different banks
    pl->mbox_stride = pl->eh_max * pl->pitch + 8;
    pl->smem_bytes = tile_smem_bytes(pl->eh_max, pl->pitch);
    pl->q = q; pl->xwork = xwork;

    bool good = cudaFuncSetAttribute(persistent_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)pl->smem_bytes) == cudaSuccess;
    int per_sm = 0;
    good = good && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, persistent_sweep_kernel, threads,
                                                                 pl->smem_bytes) == cudaSuccess;
    const int tiles = best_gy * best_gx;
    const int capacity = per_sm * n_sm;
    good = good && capacity >= tiles;
    if (good) {
        pl->frames_per_launch = std::max(1, std::min(B, capacity / tiles));
        std::vector<PFamily> pf(fams.size());
        for (size_t i = 0; i < fams.size(); ++i) {
            const Family &f = fams[i];
            int G = 1;
            while (G < f.side) G <<= 1;
            pf[i] = PFamily{f.side, f.oy, f.ox, f.ny, f.nx, f.c, f.sqrt_c,
                            (unsigned)(((1u << 20) + f.side - 1) / f.side), G};
        }
        pl->mbox_bytes = (size_t)pl->frames_per_launch * tiles * NSLOT * pl->mbox_stride * 8;
        good = cudaMalloc(&pl->d_fams, pf.size() * sizeof(PFamily)) == cudaSuccess &&
               cudaMalloc(&pl->d_mbox, pl->mbox_bytes) == cudaSuccess &&
               cudaMalloc(&pl->d_status, sizeof(int)) == cudaSuccess &&
               cudaMemcpy(pl->d_fams, pf.data(), pf.size() * sizeof(PFamily), cudaMemcpyHostToDevice) == cudaSuccess &&
               cudaMemset(pl->d_status, 0, sizeof(int)) == cudaSuccess;
    }
    if (!good) {
        cudaGetLastError();
        persistent_plan_destroy(pl);
        return nullptr;
    }
    return pl;
}

void persistent_plan_destroy(PersistentPlan *p)
{
    if (!p) return;
    if (p->d_fams) cudaFree(p->d_fams);
    if (p->d_mbox) cudaFree(p->d_mbox);
    if (p->d_status) cudaFree(p->d_status);
    delete p;
}

void persistent_plan_tiles(const PersistentPlan *p, int *tiles_y, int *tiles_x)
{
    *tiles_y = p->gy;
    *tiles_x = p->gx;
}

int persistent_plan_status(const PersistentPlan *p)
{
    int s = -1;
    if (cudaMemcpy(&s, p->d_status, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return s;
}

cudaError_t persistent_run(PersistentPlan *pl, const float *y, float *x_out, int n_sweeps,
                           cudaStream_t st, long long *launches)
{
    cudaError_t e;
    const size_t img_bytes = (size_t)pl->B * pl->H * pl->W * sizeof(float);
    if (y == x_out) {      // in place: tiles read their halo from y while neighbours may already write x_out
        if ((e = cudaMemcpyAsync(pl->xwork, y, img_bytes, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
        y = pl->xwork;
    }
    PParams p{};
    p.y = y; p.x_out = x_out; p.q = pl->q; p.fams = pl->d_fams; p.mbox = pl->d_mbox; p.status = pl->d_status;
    p.F = pl->F; p.n_sweeps = n_sweeps; p.H = pl->H; p.W = pl->W; p.B_total = pl->B;
    p.gy = pl->gy; p.gx = pl->gx; p.h = pl->h; p.pitch = pl->pitch; p.eh_max = pl->eh_max;
    p.mbox_stride = pl->mbox_stride;
    memcpy(p.yb, pl->yb.data(), pl->yb.size() * sizeof(short));
    memcpy(p.xb, pl->xb.data(), pl->xb.size() * sizeof(short));
    for (int f0 = 0; f0 < pl->B; f0 += pl->frames_per_launch) {
        p.frame0 = f0;
        p.B = std::min(pl->frames_per_launch, pl->B - f0);
        // tags restart at 1 in every launch: clear the mailboxes (a few MB, L2-resident)
        if ((e = cudaMemsetAsync(pl->d_mbox, 0, pl->mbox_bytes, st)) != cudaSuccess) return e;
        void *args[] = {&p};
        e = cudaLaunchCooperativeKernel((const void *)persistent_sweep_kernel,
                                        dim3((unsigned)(p.B * pl->gy * pl->gx)), dim3((unsigned)pl->threads),
                                        args, pl->smem_bytes, st);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
    return cudaSuccess;
}

}  // namespace smre
