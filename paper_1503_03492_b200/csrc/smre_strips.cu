// "Strips" sweep scheduler of the standard variant: ONE persistent cooperative
// kernel runs all n_sweeps * F strictly ordered family steps (Alg. 2; order matters only for
// overlapping sets).  Geometry: smre_strips.cuh.  Per CTA = one strip of one frame:
//
//   * x rows of the strip live in shared memory for the whole call (tile row = image row - j*T + 7);
//   * compute warp k owns chunk k of every band: floor(32/s) windows, lane = image column; per family step it
//     reads x (+ q), reduces per window (column-serial fma chain, then a fixed shuffle tree over the s lanes of
//     the window -- the summation order of family_pass_kernel, so both schedulers agree bit for bit), scales
//     (Eq. 14), writes x back to the tile and q to HBM; one named barrier per family step;
//   * a loader warp streams the q rows of the strip for the coming steps from HBM into a shared-memory ring with
//     bulk async copies (cp.async.bulk + mbarrier transaction counts), as deep as the ring allows.  The q of a
//     pixel is always written and read by the SAME CTA (the geometry does not depend on the sweep), so there is
//     no cross-CTA ordering of q at all; inside the CTA the loader orders a row behind its writer through
//     `written` (release / acquire at CTA scope) and a generic->async proxy fence;
//   * when the strip boundaries move (every macro step) the rows that change owner travel through per-CTA
//     mailboxes in global memory as self-validating 8-byte words {tag, value}: no fence, no flag.
//
// Nothing here depends on n_sweeps except the loop bound.
#include "smre_strips.cuh"

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace smre {

struct StripArgs {
    const float *y;
    float *x_out;
    float *q;                       // [F][Btot][H][Wq]
    unsigned long long *mail_up;    // [cta][ST_RU][max_up][Wq]   written by the strip below
    unsigned long long *mail_down;  // [cta][ST_RD][max_down][Wq] written by the strip above
    unsigned *done;                 // [cta][32]: tag of the last transition this CTA has fully received
    unsigned *status;               // device word: 0 healthy, else code of the first wait that timed out
    unsigned *status_host;          // pinned host copy, written by the last CTA to finish
    unsigned *finished;             // CTAs that have finished (for status_host)
    int H, W, Wq, Btot, frame0;
    int NS, NWC, n_sides, F, n_sweeps, NR, max_up, max_down;
    int side[ST_MAX_SIDES], fam_base[ST_MAX_SIDES];
    float c[ST_MAX_SIDES], sqrt_c[ST_MAX_SIDES];
    unsigned tag_base;
    unsigned long long timeout_ns;
};

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b)
{
    asm volatile("{ .reg .b64 t; mbarrier.arrive.shared::cta.b64 t, [%0]; }" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *b, uint32_t bytes)
{
    asm volatile("{ .reg .b64 t; mbarrier.arrive.expect_tx.shared::cta.b64 t, [%0], %1; }" ::"r"(smem_u32(b)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *b, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
// one row of q: global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_load_row(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void st_release_cta(unsigned *p, unsigned v)
{
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_cta(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_gpu64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu32(unsigned *p, unsigned v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_relaxed_gpu32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ------------------------------------------------------------------------------------------------ bounded waits
// A wait that does not come true within A.timeout_ns raises the device status word and the CTA's abort flag; from
// then on every wait of the CTA returns at once (and other CTAs see the status word in their slow path), so a
// protocol bug or a lost CTA ends the kernel with an error code instead of hanging the GPU.
enum { ST_W_QFULL = 1, ST_W_QEMPTY = 2, ST_W_WRITTEN = 3, ST_W_MAIL_UP = 4, ST_W_MAIL_DOWN = 5, ST_W_DONE = 6 };

struct Waiter {
    const StripArgs &A;
    unsigned *abort_flag;                    // shared memory
    unsigned long long t0 = 0;
    unsigned spins = 0;
    __device__ Waiter(const StripArgs &a, unsigned *f) : A(a), abort_flag(f) {}
    __device__ __forceinline__ void begin() { spins = 0; t0 = 0; }
    // call after a failed poll; true -> give up
    __device__ __noinline__ bool slow(int what)
    {
        if (*(volatile unsigned *)abort_flag) return true;
        if ((++spins & 63u) != 0) return false;
        const unsigned long long now = globaltimer_ns();
        if (t0 == 0) { t0 = now; return false; }
        if (ld_relaxed_gpu32(A.status) != 0 || now - t0 > A.timeout_ns) {
            atomicCAS(A.status, 0u, (unsigned)what | ((unsigned)blockIdx.x << 8));
            *(volatile unsigned *)abort_flag = 1u;
            return true;
        }
        return false;
    }
};

// ------------------------------------------------------------------------------------------------ window sums
// Sum over the S lanes of a window, delivered to every lane of it.  col = the lane's column sum; src = lane of the
// window's first column.  Order: pairs, then pairs of pairs, ... = the ascending xor tree of family_pass_kernel
// with zero padding to the next power of two, so both kernels round identically.
template <int S>
__device__ __forceinline__ float window_total(float col, int src)
{
    constexpr unsigned FULL = 0xffffffffu;
    if (S == 1) return col;
    const float a2 = col + __shfl_down_sync(FULL, col, 1);
    float t = a2;
    if (S == 3) t = a2 + __shfl_down_sync(FULL, col, 2);
    if (S >= 4) {
        const float a4 = a2 + __shfl_down_sync(FULL, a2, 2);
        t = a4;
        if (S == 5) t = a4 + __shfl_down_sync(FULL, col, 4);
        if (S == 6) t = a4 + __shfl_down_sync(FULL, a2, 4);
        if (S == 7) t = a4 + __shfl_down_sync(FULL, a2 + __shfl_down_sync(FULL, col, 2), 4);
        if (S == 8) t = a4 + __shfl_down_sync(FULL, a4, 4);
    }
    return __shfl_sync(FULL, t, src);
}

// ------------------------------------------------------------------------------------------------ one family step
// xt: the lane's column in the first active tile row; qs: same place in the staged q rows (HAS_Q) ; qg: same place
// in the family's q plane in HBM.  nb bands of S rows.  Row a2 of SURVEY.md 8(a); Eq. 14; Listing 3 PAPER.md:477-510.
// Lanes that are not `on` (beyond the last whole window of the chunk / the image) load from a clamped, valid column
// and take part in the shuffles, but store nothing; no active lane ever reads their values (windows are whole).
template <int S, bool HAS_Q>
__device__ __forceinline__ void family_step(float *xt, const float *qs, float *qg, int pitch, int Wq, int nb, bool on,
                                            int src, float cth, float sq, int NT)
{
    constexpr int NBMAX = ST_MAXROWS / S;
#pragma unroll
    for (int b = 0; b < NBMAX; ++b) {
        if (b < nb) {
            float v[S];
            float n2 = 0.0f;
#pragma unroll
            for (int r = 0; r < S; ++r) {
                const int row = b * S + r;
                const float xv = xt[row * pitch];
                v[r] = HAS_Q ? __fadd_rn(xv, qs[row * pitch]) : xv;
                n2 = fmaf(v[r], v[r], n2);
            }
            const float tot = window_total<S>(n2, src);
            const float alpha = ball_scale(tot, cth, sq);
            if (on) {
#pragma unroll
                for (int r = 0; r < S; ++r) {
                    float xn, qn;
                    ball_update(v[r], alpha, xn, qn);
                    xt[(b * S + r) * pitch] = xn;
                    __stcs(qg + (size_t)((b * S + r) * Wq), qn);
                }
            }
        }
    }
    bar_sync(1, NT);                 // every window of the next family overlaps windows of other warps
}

// ------------------------------------------------------------------------------------------------ compute side
__device__ __forceinline__ unsigned long long pack_word(unsigned tag, float v)
{
    return ((unsigned long long)tag << 32) | (unsigned long long)__float_as_uint(v);
}

struct ComputeState {
    int g = 0;            // family steps done
    int pos = 0;          // q ring: next free row
    unsigned n = 0;       // staged (non-empty) steps consumed so far
    unsigned mc = 0;      // transitions done
    unsigned done_up, done_down;    // cached progress of the strip above / below (flow control of the mailbox rings)
};

// Rows change owner between the families (s, oy, *) and (s2, oy2, *).  All compute threads of the CTA take part;
// on entry every tile write of the last step is visible (step barrier), on exit the tile holds the new row set.
// Sends come first and wait for nothing but ring space, so the hand-offs of one transition cannot form a cycle.
__device__ __forceinline__ void transition(const StripArgs &A, float *tile, int pitch, int j, int cta, int s, int oy,
                                           int s2, int oy2, ComputeState &cs, int tid, int NT, unsigned *written,
                                           Waiter &w)
{
    const int NS = A.NS, H = A.H, W = A.W, Wq = A.Wq;
    const int bt = st_boundary(j, NS, H, s, oy), bt2 = st_boundary(j, NS, H, s2, oy2);
    const int bb = st_boundary(j + 1, NS, H, s, oy), bb2 = st_boundary(j + 1, NS, H, s2, oy2);
    const unsigned mc = ++cs.mc;
    const unsigned tag = A.tag_base + mc;
    const int slot_base = ST_SLOT_OFF - j * ST_T;

    if (j >= 1 && bt2 > bt) {                                  // my top rows go to the strip above
        if (mc > (unsigned)ST_RU) {
            w.begin();
            while ((int)(tag - ST_RU - cs.done_up) > 0) {
                cs.done_up = ld_relaxed_gpu32(A.done + (size_t)(cta - 1) * 32);
                if ((int)(tag - ST_RU - cs.done_up) > 0 && w.slow(ST_W_DONE)) break;
            }
        }
        unsigned long long *dst = A.mail_up + ((size_t)(cta - 1) * ST_RU + mc % ST_RU) * A.max_up * Wq;
        for (int y = bt; y < bt2; ++y)
            for (int c = tid; c < W; c += NT)
                st_relaxed_gpu64(dst + (size_t)(y - bt) * Wq + c, pack_word(tag, tile[(y + slot_base) * pitch + c]));
    }
    if (j + 1 < NS && bb2 < bb) {                              // my bottom rows go to the strip below
        if (mc > (unsigned)ST_RD) {
            w.begin();
            while ((int)(tag - ST_RD - cs.done_down) > 0) {
                cs.done_down = ld_relaxed_gpu32(A.done + (size_t)(cta + 1) * 32);
                if ((int)(tag - ST_RD - cs.done_down) > 0 && w.slow(ST_W_DONE)) break;
            }
        }
        unsigned long long *dst = A.mail_down + ((size_t)(cta + 1) * ST_RD + mc % ST_RD) * A.max_down * Wq;
        for (int y = bb2; y < bb; ++y)
            for (int c = tid; c < W; c += NT)
                st_relaxed_gpu64(dst + (size_t)(y - bb2) * Wq + c, pack_word(tag, tile[(y + slot_base) * pitch + c]));
    }
    if (j + 1 < NS && bb2 > bb) {                              // rows arriving from below
        const unsigned long long *src = A.mail_up + ((size_t)cta * ST_RU + mc % ST_RU) * A.max_up * Wq;
        for (int y = bb; y < bb2; ++y)
            for (int c = tid; c < W; c += NT) {
                const unsigned long long *p = src + (size_t)(y - bb) * Wq + c;
                unsigned long long wd = ld_relaxed_gpu64(p);
                w.begin();
                while ((unsigned)(wd >> 32) != tag) {
                    if (w.slow(ST_W_MAIL_UP)) break;
                    wd = ld_relaxed_gpu64(p);
                }
                tile[(y + slot_base) * pitch + c] = __uint_as_float((unsigned)wd);
            }
    }
    if (j >= 1 && bt2 < bt) {                                  // rows arriving from above
        const unsigned long long *src = A.mail_down + ((size_t)cta * ST_RD + mc % ST_RD) * A.max_down * Wq;
        for (int y = bt2; y < bt; ++y)
            for (int c = tid; c < W; c += NT) {
                const unsigned long long *p = src + (size_t)(y - bt2) * Wq + c;
                unsigned long long wd = ld_relaxed_gpu64(p);
                w.begin();
                while ((unsigned)(wd >> 32) != tag) {
                    if (w.slow(ST_W_MAIL_DOWN)) break;
                    wd = ld_relaxed_gpu64(p);
                }
                tile[(y + slot_base) * pitch + c] = __uint_as_float((unsigned)wd);
            }
    }
    bar_sync(1, NT);
    if (tid == 0) {
        st_relaxed_gpu32(A.done + (size_t)cta * 32, tag);       // my mailbox slots of this transition are free again
        st_release_cta(written, (unsigned)cs.g);                // q of every step < g is on its way to HBM (loader: acquire)
    }
}

// One macro step: the S families (S, oy, 0..S-1) on the strip's bands; the strip interacts with nobody meanwhile.
template <int S>
__device__ __forceinline__ void macro_step(const StripArgs &A, int a, int oy, bool staged, float *tile, const float *ring,
                                           uint64_t *full, uint64_t *empty, int pitch, int Wq, int j, int frame,
                                           ComputeState &cs, int warp, int lane, int NT, Waiter &wt)
{
    constexpr int CW = (32 / S) * S;
    const int H = A.H, W = A.W, NS = A.NS;
    const int src = (lane / S) * S;
    const float cth = A.c[a], sq = A.sqrt_c[a];
    int lo, hi;
    st_active_rows(j, NS, H, S, oy, lo, hi);
    const int rows = hi - lo;
    const int nb = rows / S;
    float *xrow = tile + (lo - j * ST_T + ST_SLOT_OFF) * pitch;
    const float *qplane = A.q + ((size_t)(A.fam_base[a] + oy * S) * A.Btot + frame) * ((size_t)H * Wq) + (size_t)lo * Wq;
    const size_t fam_stride = (size_t)A.Btot * H * Wq;
#pragma unroll 1
    for (int ox = 0; ox < S; ++ox) {
        const int c = ox + warp * CW + lane;
        const bool on = (lane < CW) && (c < ox + ((W - ox) / S) * S);
        const int cl = c < W ? c : W - 1;                      // clamped: a valid column for the lanes that are off
        float *qg = const_cast<float *>(qplane) + (size_t)ox * fam_stride + cl;
        if (staged && rows > 0) {
            if (cs.pos + rows > A.NR) cs.pos = 0;
            const float *qs = ring + cs.pos * pitch + cl;
            cs.pos += rows;
            const unsigned stage = cs.n % ST_NSTG, parity = (cs.n / ST_NSTG) & 1u;
            ++cs.n;
            if (!mbar_try_wait(&full[stage], parity)) {
                wt.begin();
                while (!mbar_try_wait(&full[stage], parity))
                    if (wt.slow(ST_W_QFULL)) break;
            }
            family_step<S, true>(xrow + cl, qs, qg, pitch, Wq, nb, on, src, cth, sq, NT);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[stage]);          // the staged rows have been read
        } else {
            family_step<S, false>(xrow + cl, nullptr, qg, pitch, Wq, nb, on, src, cth, sq, NT);
        }
        ++cs.g;
    }
}

// ------------------------------------------------------------------------------------------------ q loader warp
template <int PITCH>
__device__ void loader_warp(const StripArgs &A, float *ring, uint64_t *full, uint64_t *empty, unsigned *written,
                            unsigned *abort_flag, unsigned short *qpos, unsigned short *qrows, int j, int frame, int lane)
{
    const int pitch = PITCH ? PITCH : A.Wq;
    const int Wq = PITCH ? PITCH : A.Wq;
    const int H = A.H, NS = A.NS;
    const size_t plane = (size_t)H * Wq;
    const uint32_t row_bytes = (uint32_t)Wq * 4u;
    Waiter wt(A, abort_flag);
    int pos = 0;
    unsigned n = 0, nt = 0;                 // issued / released stage counters
    unsigned have = 0;                      // last value read from `written`
    int g = A.F;
    for (int sweep = 1; sweep < A.n_sweeps; ++sweep)
        for (int a = 0; a < A.n_sides; ++a) {
            const int s = A.side[a];
            for (int oy = 0; oy < s; ++oy) {
                int lo, hi;
                st_active_rows(j, NS, H, s, oy, lo, hi);
                const int rows = hi - lo;
                for (int ox = 0; ox < s; ++ox, ++g) {
                    if (rows == 0) continue;
                    // (1) the rows were written one sweep ago, in step g - F: wait until the compute warps say so
                    const unsigned need = (unsigned)(g - A.F + 1);
                    if (have < need) {
                        wt.begin();
                        while ((have = ld_acquire_cta(written)) < need)
                            if (wt.slow(ST_W_WRITTEN)) break;
                    }
                    // (2) ring space: positions are a function of the step sequence alone (the compute warps
                    //     derive the same ones); wait until every older stage overlapping the new rows is released
                    const bool wrapped = pos + rows > A.NR;
                    const int npos = wrapped ? 0 : pos;
                    while (nt < n) {
                        const int fp = qpos[nt & 63u], fr = qrows[nt & 63u];
                        const bool need_pop = (n - nt >= (unsigned)ST_NSTG) || (fp < npos + rows && npos < fp + fr) ||
                                              (wrapped && fp >= pos);
                        if (!need_pop) break;
                        const unsigned stage = nt % ST_NSTG, parity = (nt / ST_NSTG) & 1u;
                        if (!mbar_try_wait(&empty[stage], parity)) {
                            wt.begin();
                            while (!mbar_try_wait(&empty[stage], parity))
                                if (wt.slow(ST_W_QEMPTY)) break;
                        }
                        ++nt;
                    }
                    __syncwarp();
                    if (lane == 0) { qpos[n & 63u] = (unsigned short)npos; qrows[n & 63u] = (unsigned short)rows; }
                    // (3) order the async-proxy reads behind the generic-proxy writes acquired in (1), then issue
                    fence_proxy_async();
                    uint64_t *bar = &full[n % ST_NSTG];
                    if (lane == 0) mbar_arrive_expect_tx(bar, (uint32_t)rows * row_bytes);
                    __syncwarp();
                    const float *srcp = A.q + ((size_t)(A.fam_base[a] + oy * s + ox) * A.Btot + frame) * plane +
                                        (size_t)lo * Wq;
                    for (int r = lane; r < rows; r += 32)
                        bulk_load_row(ring + (size_t)(npos + r) * pitch, srcp + (size_t)r * Wq, row_bytes, bar);
                    pos = npos + rows;
                    ++n;
                }
            }
        }
}

// ------------------------------------------------------------------------------------------------ kernel
template <int PITCH, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) strips_kernel(const __grid_constant__ StripArgs A)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int pitch = PITCH ? PITCH : A.Wq;
    float *tile = reinterpret_cast<float *>(smem_raw);
    float *ring = tile + ST_TR * pitch;
    uint64_t *full = reinterpret_cast<uint64_t *>(ring + (size_t)A.NR * pitch);
    uint64_t *empty = full + ST_NSTG;
    unsigned *written = reinterpret_cast<unsigned *>(empty + ST_NSTG);
    unsigned *abort_flag = written + 1;
    unsigned short *qpos = reinterpret_cast<unsigned short *>(written + 2);
    unsigned short *qrows = qpos + 64;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NWC = A.NWC, NT = NWC * 32;
    const int cta = blockIdx.x, fl = cta / A.NS, j = cta - fl * A.NS, frame = A.frame0 + fl;
    const int H = A.H, W = A.W, NS = A.NS;

    if (threadIdx.x == 0) {
        for (int i = 0; i < ST_NSTG; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NWC); }
        *written = 0u;
        *abort_flag = 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NWC) {
        loader_warp<PITCH>(A, ring, full, empty, written, abort_flag, qpos, qrows, j, frame, lane);
    } else {
        const int tid = threadIdx.x;
        // row a1: x <- y for the rows of the first family's geometry (q needs no zeroing: the first sweep reads none)
        const float *yim = A.y + (size_t)frame * H * W;
        {
            const int lo = st_boundary(j, NS, H, A.side[0], 0), hi = st_boundary(j + 1, NS, H, A.side[0], 0);
            for (int y = lo; y < hi; ++y)
                for (int c = tid; c < W; c += NT) tile[(y - j * ST_T + ST_SLOT_OFF) * pitch + c] = yim[(size_t)y * W + c];
        }
        bar_sync(1, NT);
        ComputeState cs;
        cs.done_up = cs.done_down = A.tag_base;
        Waiter wt(A, abort_flag);
        const int Wq = PITCH ? PITCH : A.Wq;
        for (int sweep = 0; sweep < A.n_sweeps; ++sweep)
            for (int a = 0; a < A.n_sides; ++a) {
                const int s = A.side[a];
                for (int oy = 0; oy < s; ++oy) {
#define SMRE_RUN(S_)                                                                                                   \
    case S_:                                                                                                           \
        macro_step<S_>(A, a, oy, sweep > 0, tile, ring, full, empty, pitch, Wq, j, frame, cs, warp, lane, NT, wt);     \
        break;
                    switch (s) {
                        SMRE_RUN(1) SMRE_RUN(2) SMRE_RUN(3) SMRE_RUN(4) SMRE_RUN(5) SMRE_RUN(6) SMRE_RUN(7) SMRE_RUN(8)
                    }
#undef SMRE_RUN
                    // next macro step: (s, oy + 1), or the first one of the next side; none after the very last one
                    int s2 = s, oy2 = oy + 1;
                    if (oy2 == s) {
                        if (a + 1 == A.n_sides && sweep + 1 == A.n_sweeps) break;
                        oy2 = 0;
                        s2 = A.side[(a + 1 == A.n_sides) ? 0 : a + 1];
                    }
                    transition(A, tile, pitch, j, cta, s, oy, s2, oy2, cs, tid, NT, written, wt);
                }
            }
        // row a9: the strip's rows under the last family's geometry
        {
            const int s = A.side[A.n_sides - 1];
            const int lo = st_boundary(j, NS, H, s, s - 1), hi = st_boundary(j + 1, NS, H, s, s - 1);
            float *xo = A.x_out + (size_t)frame * H * W;
            for (int y = lo; y < hi; ++y)
                for (int c = tid; c < W; c += NT) xo[(size_t)y * W + c] = tile[(y - j * ST_T + ST_SLOT_OFF) * pitch + c];
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned k = atomicAdd(A.finished, 1u);
        if (k + 1 == gridDim.x) {                               // last CTA: publish the health word to the host
            *(volatile unsigned *)A.status_host = ld_relaxed_gpu32(A.status);
            __threadfence_system();
            atomicExch(A.finished, 0u);                         // next launch of the same call (frame groups)
        }
    }
}

// ------------------------------------------------------------------------------------------------ host side
struct StripPlan {
    int H = 0, W = 0, B = 0, Wq = 0, NS = 0, NWC = 0, F = 0, NR = 0, max_up = 1, max_down = 1, frames_per_launch = 1;
    int n_sides = 0, side[ST_MAX_SIDES] = {}, fam_base[ST_MAX_SIDES] = {};
    float c[ST_MAX_SIDES] = {}, sqrt_c[ST_MAX_SIDES] = {};
    float *q = nullptr;
    unsigned long long *mail_up = nullptr, *mail_down = nullptr;
    unsigned *done = nullptr, *status = nullptr, *finished = nullptr;
    unsigned *status_host = nullptr;                             // pinned, mapped
    unsigned *status_host_dev = nullptr;
    size_t mail_up_bytes = 0, mail_down_bytes = 0, smem_bytes = 0;
    unsigned tag_base = 1;
    unsigned long long timeout_ns = 2000000000ull;
    int device = 0;
    const void *kernel = nullptr;
    int threads = 0;
};

static void set_why(char *why, size_t n, const char *fmt, ...)
{
    if (!why || !n) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(why, n, fmt, ap);
    va_end(ap);
}

bool strips_summary(int H, int W, int B, const int *sides, int n_sides, int sm_count, int smem_optin,
                    StripSummary *out, char *why, size_t why_len)
{
    if (n_sides > ST_MAX_SIDES) { set_why(why, why_len, "more than %d sides", ST_MAX_SIDES); return false; }
    int F = 0;
    for (int a = 0; a < n_sides; ++a) {
        if (sides[a] > ST_MAX_SIDE) { set_why(why, why_len, "side %d > %d", sides[a], ST_MAX_SIDE); return false; }
        F += sides[a] * sides[a];
    }
    const int NS = (H + ST_T - 1) / ST_T;
    if (NS > sm_count) {
        set_why(why, why_len, "%d strips of %d rows need more than the %d co-resident CTAs", NS, ST_T, sm_count);
        return false;
    }
    int NWC = 1;
    for (int a = 0; a < n_sides; ++a) {
        const int cw = st_chunk_width(sides[a]);
        NWC = std::max(NWC, (W + cw - 1) / cw);
    }
    if (NWC > ST_MAX_WARPS) {
        set_why(why, why_len, "width %d needs %d warps per strip (limit %d)", W, NWC, ST_MAX_WARPS);
        return false;
    }
    const int Wq = (W + 3) & ~3;
    // rows per step, rows moving per transition: brute force over one sweep (closed-form geometry, host only)
    int max_rows = 0, max_up = 1, max_down = 1;
    for (int a = 0; a < n_sides; ++a)
        for (int oy = 0; oy < sides[a]; ++oy) {
            int s2 = sides[a], oy2 = oy + 1;
            if (oy2 == s2) { oy2 = 0; s2 = sides[(a + 1) % n_sides]; }
            for (int j = 0; j < NS; ++j) {
                int lo, hi;
                st_active_rows(j, NS, H, sides[a], oy, lo, hi);
                max_rows = std::max(max_rows, hi - lo);
                const int hold = st_boundary(j + 1, NS, H, sides[a], oy) - st_boundary(j, NS, H, sides[a], oy);
                if (hold > ST_TR || st_boundary(j, NS, H, sides[a], oy) - j * ST_T + ST_SLOT_OFF < 0 ||
                    st_boundary(j + 1, NS, H, sides[a], oy) - j * ST_T + ST_SLOT_OFF > ST_TR) {
                    set_why(why, why_len, "strip %d does not fit its tile", j);
                    return false;
                }
                const int b_old = st_boundary(j, NS, H, sides[a], oy), b_new = st_boundary(j, NS, H, s2, oy2);
                const int d = b_new - b_old;
                if (d > 0) max_up = std::max(max_up, d);
                if (d < 0) max_down = std::max(max_down, -d);
                // a row that changes owner goes to a neighbouring strip (single hop)
                if ((d < 0 && b_new < st_boundary(j - 1, NS, H, sides[a], oy)) ||
                    (d > 0 && b_new > st_boundary(j + 1, NS, H, sides[a], oy))) {
                    set_why(why, why_len, "boundary %d moves past a whole strip", j);
                    return false;
                }
            }
        }
    if (max_rows > ST_MAXROWS) { set_why(why, why_len, "a strip has %d active rows (limit %d)", max_rows, ST_MAXROWS); return false; }
    const long long tile_bytes = (long long)ST_TR * Wq * 4;
    const long long fixed = ST_NSTG * 16 + 8 + 256 + 128;
    const long long ring_rows = (smem_optin - tile_bytes - fixed) / ((long long)Wq * 4);
    if (ring_rows < 3 * ST_MAXROWS) {
        set_why(why, why_len, "shared memory holds only %lld q rows of width %d", ring_rows, W);
        return false;
    }
    if (out) {
        out->strips = NS;
        out->warps = NWC;
        out->max_rows = max_rows;
        out->max_up = max_up;
        out->max_down = max_down;
        out->ring_rows = (int)std::min<long long>(ring_rows, 60000);
        out->frames_per_launch = std::max(1, std::min(B, sm_count / NS));
        const long long ctas = (long long)out->frames_per_launch * NS;
        out->workspace_bytes = ctas * ((long long)ST_RU * max_up + (long long)ST_RD * max_down) * Wq * 8 + ctas * 128;
    }
    (void)F;
    return true;
}

template <int PITCH, int MAXT>
static const void *kernel_ptr() { return (const void *)strips_kernel<PITCH, MAXT>; }

StripPlan *strips_plan_create(int H, int W, int B, int Wq, const int *sides, const float *c, int n_sides, float *q,
                              char *why, size_t why_len)
{
    int dev = 0, sms = 0, smem = 0, coop = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) { set_why(why, why_len, "device has no cooperative launch"); return nullptr; }
    StripSummary sm;
    if (!strips_summary(H, W, B, sides, n_sides, sms, smem, &sm, why, why_len)) return nullptr;

    StripPlan *p = new StripPlan;
    p->device = dev;
    p->H = H; p->W = W; p->B = B; p->Wq = Wq; p->q = q;
    p->NS = sm.strips; p->NWC = sm.warps; p->NR = sm.ring_rows;
    p->max_up = sm.max_up; p->max_down = sm.max_down; p->frames_per_launch = sm.frames_per_launch;
    p->n_sides = n_sides;
    int F = 0;
    for (int a = 0; a < n_sides; ++a) {
        p->side[a] = sides[a]; p->c[a] = c[a]; p->sqrt_c[a] = sqrtf(c[a]); p->fam_base[a] = F;
        F += sides[a] * sides[a];
    }
    p->F = F;
    p->threads = (p->NWC + 1) * 32;
    const bool big = p->threads > 672;
    if (Wq == 512) p->kernel = big ? kernel_ptr<512, 1024>() : kernel_ptr<512, 672>();
    else p->kernel = big ? kernel_ptr<0, 1024>() : kernel_ptr<0, 672>();
    p->smem_bytes = (size_t)ST_TR * Wq * 4 + (size_t)p->NR * Wq * 4 + ST_NSTG * 16 + 8 + 256;
    if (const char *e = getenv("SMRE_TIMEOUT_MS")) {
        const long long ms = atoll(e);
        if (ms > 0) p->timeout_ns = (unsigned long long)ms * 1000000ull;
    }
    const size_t ctas = (size_t)p->frames_per_launch * p->NS;
    p->mail_up_bytes = ctas * ST_RU * p->max_up * Wq * 8;
    p->mail_down_bytes = ctas * ST_RD * p->max_down * Wq * 8;
    cudaError_t e = cudaFuncSetAttribute(p->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&p->mail_up, p->mail_up_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&p->mail_down, p->mail_down_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&p->done, ctas * 128);
    if (e == cudaSuccess) e = cudaMalloc(&p->status, 256);
    if (e == cudaSuccess) e = cudaHostAlloc(&p->status_host, 64, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&p->status_host_dev, p->status_host, 0);
    if (e == cudaSuccess) e = cudaMemset(p->mail_up, 0, p->mail_up_bytes);
    if (e == cudaSuccess) e = cudaMemset(p->mail_down, 0, p->mail_down_bytes);
    if (e == cudaSuccess) e = cudaMemset(p->done, 0, ctas * 128);
    if (e == cudaSuccess) e = cudaMemset(p->status, 0, 256);
    int nb = 0;
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, p->kernel, p->threads, p->smem_bytes);
    if (e != cudaSuccess || nb < 1) {
        set_why(why, why_len, "strips workspace / occupancy: %s", e != cudaSuccess ? cudaGetErrorString(e) : "kernel does not fit an SM");
        cudaGetLastError();
        strips_plan_destroy(p);
        return nullptr;
    }
    p->finished = p->status + 32;
    *p->status_host = 0;
    return p;
}

void strips_plan_destroy(StripPlan *p)
{
    if (!p) return;
    if (p->mail_up) cudaFree(p->mail_up);
    if (p->mail_down) cudaFree(p->mail_down);
    if (p->done) cudaFree(p->done);
    if (p->status) cudaFree(p->status);
    if (p->status_host) cudaFreeHost(p->status_host);
    delete p;
}

void strips_plan_shape(const StripPlan *p, int *strips, int *warps)
{
    if (strips) *strips = p->NS;
    if (warps) *warps = p->NWC;
}

int strips_plan_status(const StripPlan *p) { return (int)*(volatile unsigned *)p->status_host; }

cudaError_t strips_run(StripPlan *p, const float *y, float *x_out, int n_sweeps, cudaStream_t st, long long *launches)
{
    int M = 0;
    for (int a = 0; a < p->n_sides; ++a) M += p->side[a];
    const unsigned long long total = (unsigned long long)n_sweeps * M + 2;
    if (total >= 0x40000000ull) return cudaErrorNotSupported;
    cudaError_t e = cudaMemsetAsync(p->status, 0, 256, st);
    if (e != cudaSuccess) return e;
    for (int f0 = 0; f0 < p->B; f0 += p->frames_per_launch) {
        const int nf = std::min(p->frames_per_launch, p->B - f0);
        if (p->tag_base + total < p->tag_base || p->tag_base + total > 0xfffffff0u) {     // 32-bit tags used up: start over
            e = cudaMemsetAsync(p->mail_up, 0, p->mail_up_bytes, st);
            if (e == cudaSuccess) e = cudaMemsetAsync(p->mail_down, 0, p->mail_down_bytes, st);
            if (e == cudaSuccess) e = cudaMemsetAsync(p->done, 0, (size_t)p->frames_per_launch * p->NS * 128, st);
            if (e != cudaSuccess) return e;
            p->tag_base = 1;
        }
        StripArgs A{};
        A.y = y; A.x_out = x_out; A.q = p->q;
        A.mail_up = p->mail_up; A.mail_down = p->mail_down; A.done = p->done;
        A.status = p->status; A.status_host = p->status_host_dev; A.finished = p->finished;
        A.H = p->H; A.W = p->W; A.Wq = p->Wq; A.Btot = p->B; A.frame0 = f0;
        A.NS = p->NS; A.NWC = p->NWC; A.n_sides = p->n_sides; A.F = p->F; A.n_sweeps = n_sweeps; A.NR = p->NR;
        A.max_up = p->max_up; A.max_down = p->max_down;
        for (int a = 0; a < p->n_sides; ++a) {
            A.side[a] = p->side[a]; A.fam_base[a] = p->fam_base[a]; A.c[a] = p->c[a]; A.sqrt_c[a] = p->sqrt_c[a];
        }
        A.tag_base = p->tag_base;
        A.timeout_ns = p->timeout_ns;
        p->tag_base += (unsigned)total;
        void *args[] = {&A};
        e = cudaLaunchCooperativeKernel(p->kernel, dim3((unsigned)(nf * p->NS)), dim3((unsigned)p->threads), args,
                                        p->smem_bytes, st);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
    return cudaSuccess;
}

}  // namespace smre
