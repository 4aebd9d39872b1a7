// "Strips" sweep scheduler of the standard variant: ONE persistent cooperative
// kernel runs all n_sweeps * F strictly ordered family steps (Alg. 2; order matters only for
// overlapping sets).  Geometry: smre_strips.cuh.  Per CTA = one strip of one frame:
//
//   * the x rows of the strip live in shared memory for the whole call (tile row = image row - j*T + T/2);
//   * compute warp k owns chunk k of every band: floor(32/s) windows, lane = image column; per family step it
//     reads x (+ q), reduces per window (column-serial fma chain, then a fixed shuffle tree over the s lanes of
//     the window -- the summation order of family_pass_kernel, so both schedulers agree bit for bit), scales
//     (Eq. 14), writes x back to the tile and q to HBM; one named barrier per family step;
//   * two more warps stream the q rows of the coming steps from HBM into a shared-memory ring with bulk async
//     copies (cp.async.bulk + mbarrier transaction counts), as deep as the ring allows.  The q of a pixel is always
//     written and read by the SAME CTA (the geometry does not depend on the sweep), so there is no cross-CTA
//     ordering of q at all; inside the CTA the copies are ordered behind the writes by the step barrier, a
//     release / acquire pair at CTA scope and a generic->async proxy fence;
//   * when the strip boundaries move (between macro steps) the rows that change owner travel through per-CTA
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
    unsigned long long *mail;       // [cta][ST_RING][tile rows][Wq] 8-byte words, written by the strips around
    unsigned *done;                 // [cta][32]: tag of the last transition this CTA has fully received
    unsigned *status;               // device word: 0 healthy, else code of the first wait that timed out
    unsigned *status_host;          // pinned host copy, written by the last CTA to finish
    unsigned *finished;             // CTAs that have finished (for status_host)
    int H, W, Wq, Btot, frame0;
    int T, NS, NWC, n_sides, F, n_sweeps, NR, max_rows;
    int side[ST_MAX_SIDES], fam_base[ST_MAX_SIDES];
    float c[ST_MAX_SIDES], sqrt_c[ST_MAX_SIDES];
    unsigned tag_base;
    // convergence control (Alg. 2: "while ||x_r - x_{r-1}||^2 > delta"); tol_mode 0: fixed n_sweeps
    int tol_mode;
    float delta;
    int NR_total;                   // ring rows the shared-memory layout was made for (NR of them are used as ring)
    double *partials;               // [2][cta]: this CTA's part of ||x_r - x_{r-1}||^2, by sweep parity
    unsigned *sweep_ctr;            // [frame of the launch][32]: CTAs that have delivered their part (monotonic)
    int *sweeps_done;               // [Btot] or null: sweeps run per frame
    int elim;                       // 1: stores that would not change memory are not issued
    unsigned long long timeout_ns;
#ifdef SMRE_ST_KO
    int ko;                         // timing experiments only (wrong results): parts of the kernel switched off
#endif
};
#ifdef SMRE_ST_KO
#define ST_KO(A, bit) (((A).ko & (bit)) != 0)
#else
#define ST_KO(A, bit) false
#endif

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
enum { ST_W_QFULL = 1, ST_W_ALLOW = 3, ST_W_MAIL = 4, ST_W_SWEEP = 5, ST_W_DONE = 6 };

// the rare part of a wait (every 64th failed poll): returns the new start time, or ~0 to give up
__device__ __noinline__ unsigned long long st_wait_check(const StripArgs &A, unsigned *abort_flag, unsigned long long t0, int what)
{
    const unsigned long long now = globaltimer_ns();
    if (t0 == 0) return now;
    if (ld_relaxed_gpu32(A.status) != 0 || now - t0 > A.timeout_ns) {
        atomicCAS(A.status, 0u, (unsigned)what | ((unsigned)blockIdx.x << 8));
        *(volatile unsigned *)abort_flag = 1u;
        return ~0ull;
    }
    return t0;
}
struct Waiter {
    const StripArgs &A;
    unsigned *abort_flag;                    // shared memory
    unsigned long long t0 = 0;
    unsigned spins = 0;
    __device__ Waiter(const StripArgs &a, unsigned *f) : A(a), abort_flag(f) {}
    __device__ __forceinline__ void begin() { spins = 0; t0 = 0; }
    // call after a failed poll; true -> give up
    __device__ __forceinline__ bool slow(int what)
    {
        if (*(volatile unsigned *)abort_flag) return true;
        if ((++spins & 63u) != 0) return false;
        t0 = st_wait_check(A, abort_flag, t0, what);
        return t0 == ~0ull;
    }
};

// ------------------------------------------------------------------------------------------------ macro-step table
// One entry per macro step (side index a, row offset oy) of a sweep, for THIS strip: built once at kernel start, so
// the steady state does no geometry arithmetic (the closed forms of smre_strips.cuh need integer divisions).
struct __align__(16) MacroEntry {
    short s, rows, lo, nb;              // side; active rows of the strip (whole bands); first active row; bands
    int fam0;                           // family index of (s, oy, 0)
    float c, sqrt_c;                    // threshold of the side (Eq. 5), its square root
    int xoff;                           // tile offset (floats) of the first active row
    long long qoff;                     // offset (floats) of (family fam0, this frame, row lo) in the q planes
    short hold_lo, hold_hi;             // rows the strip holds: [hold_lo, hold_hi)
    // hand-off to the NEXT macro step (cyclic): rows [send_lo[k], send_hi[k]) go to strip j + d,
    // d = -HOPS..-1, +1..+HOPS (k = 0..2*HOPS-1); rows [recv_lo[i], recv_hi[i]) arrive (above / below what is kept)
    short send_lo[2 * ST_HOPS], send_hi[2 * ST_HOPS];
    short recv_lo[2], recv_hi[2];
    int pad0;
    long long pad1;
    // the same hand-off in one 16-byte load, in TILE rows (image row - j T + T / 2, 0 .. T + 7): 10 bits per run,
    // first row in bits 0-3, number of rows in bits 4-9; splan: the six send runs (k = 0..5), rplan: the two arrival runs
    unsigned long long splan, rplan;
};
// The hand-off behind a macro step as a ready-made program (built once at kernel start): with every compute warp in
// the hand-off, the time it takes is set by the instructions the warps issue in front of and behind the one L2
// round trip, so nothing is decoded or multiplied there any more.
struct __align__(16) HandProg {
    int send_doff[3];           // run i: mailbox word offset of its first word from (slot, tile row 0, my column) of MY
                                // mailbox: d * dest_step + row * pitch
    unsigned send_meta[3];      // run i: tile row | rows << 8 | direction index k << 16
    unsigned counts;            // send runs | arriving rows << 8 | (more than 3 send runs: take the plan words) << 16
    unsigned recv_rows[4];      // the arriving tile rows, one byte each
    unsigned pad;
};
static_assert(sizeof(HandProg) == 48, "HandProg");
static_assert(sizeof(MacroEntry) == 96 && offsetof(MacroEntry, splan) % 16 == 0, "MacroEntry");

// ------------------------------------------------------------------------------------------------ window sums
// Sum over the S lanes of a window, delivered to every lane of it.  col = the lane's column sum; src = lane of the
// window's first column (windows start at lanes that are multiples of S).  Order: neighbouring columns first, then
// pairs of pairs, ... = the ascending xor tree of family_pass_kernel with zero padding to the next power of two,
// so both kernels round identically (fp addition is commutative: every lane of a power-of-two window gets the
// same bits from the butterfly).
template <int S>
__device__ __forceinline__ float window_total(float col, int src)
{
    constexpr unsigned FULL = 0xffffffffu;
    if (S == 1) return col;
    if (S == 2 || S == 4 || S == 8) {
        float t = col + __shfl_xor_sync(FULL, col, 1);
        if (S >= 4) t += __shfl_xor_sync(FULL, t, 2);
        if (S >= 8) t += __shfl_xor_sync(FULL, t, 4);
        return t;
    }
    const float a2 = col + __shfl_down_sync(FULL, col, 1);
    float t;
    if (S == 3) t = a2 + __shfl_down_sync(FULL, col, 2);
    else {
        const float a4 = a2 + __shfl_down_sync(FULL, a2, 2);
        if (S == 5) t = a4 + __shfl_down_sync(FULL, col, 4);
        else if (S == 6) t = a4 + __shfl_down_sync(FULL, a2, 4);
        else t = a4 + __shfl_down_sync(FULL, a2 + __shfl_down_sync(FULL, col, 2), 4);
    }
    return __shfl_sync(FULL, t, src);
}

// ------------------------------------------------------------------------------------------------ one family step
// G bands of S rows starting at tile row xt / staged row qs / plane row qg (all at the lane's column).  Band 0 is
// always there; bands >= nvalid load nothing and store nothing; lanes that are not `on` (their window is not fully
// inside the image, or beyond the chunk) load whatever lies at their address -- always inside shared memory -- and
// take part in the shuffles, but store nothing, and no active lane ever reads their values (windows are whole).
// Row a2 of SURVEY.md 8(a); Eq. 14; Listing 3 PAPER.md:477-510.
// Hand-off word {tag, value}: self-validating, so a row needs neither a fence nor a flag.
__device__ __forceinline__ unsigned long long pack_word(unsigned tag, float v)
{
    return ((unsigned long long)tag << 32) | (unsigned long long)__float_as_uint(v);
}

// ELIM: work that would not change memory is not done.  A lane's column of a window is LIVE if the window was
// scaled (alpha != 1) or any pixel of the column carried an increment; only live columns compute and store the
// update.  For the others x' = 1 * (x + 0) = x and q' = v - v = 0 are what memory already holds, bit for bit
// (the planes are zeroed at create, v - v is +0).  The q planes are still READ densely.  In the first sweep
// (!HAS_Q) the planes hold the previous call's increments, so every column is live and every q is written.
template <int S, int G, bool HAS_Q, int PITCH>
__device__ __forceinline__ void band_group(float *xt, const float *qs, float *qg, int pitch_rt, int nvalid, bool on,
                                           int src, float cth, float sq, int ko, bool elim)
{
    const int pitch = PITCH ? PITCH : pitch_rt;
    float v[G][S], n2[G], al[G];
    unsigned qbits[G];                                          // OR of the bit patterns of the column's increments
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const bool pb = i == 0 || i < nvalid;
        n2[i] = 0.0f;
        qbits[i] = 0u;
#pragma unroll
        for (int r = 0; r < S; ++r) {
            float xv = 0.0f, qv = 0.0f;
            if (pb) {
                xv = xt[(i * S + r) * pitch];
                if (HAS_Q) qv = qs[(i * S + r) * pitch];
            }
            if (HAS_Q) qbits[i] |= __float_as_uint(qv);
            v[i][r] = HAS_Q ? __fadd_rn(xv, qv) : xv;
            n2[i] = fmaf(v[i][r], v[i][r], n2[i]);
        }
    }
    // The decision "does this column change memory" does not wait for the scale factor: the window is scaled iff its
    // sum exceeds the threshold (the compare of ball_scale), which is known as soon as the shuffle tree is through;
    // the reciprocal square root and the products are only formed for the columns that go on.  (A window that is
    // scaled by a factor that rounds to exactly 1 is updated too: x' = v, q' = 0, what memory holds if q was 0.)
    bool go[G];
#pragma unroll
    for (int i = 0; i < G; ++i) {
        al[i] = window_total<S>(n2[i], src);                    // the sum for now
        const bool carried = !elim || !HAS_Q || (qbits[i] << 1) != 0u;
        go[i] = on && (i == 0 || i < nvalid) && (carried || al[i] > cth);
    }
#pragma unroll
    for (int i = 0; i < G; ++i) {
        if (go[i]) {
            al[i] = ball_scale(al[i], cth, sq);
#pragma unroll
            for (int r = 0; r < S; ++r) {
                float xn, qn;
                ball_update(v[i][r], al[i], xn, qn);
                xt[(i * S + r) * pitch] = xn;
                if (!(ko & 4)) __stcs(qg + (i * S + r) * pitch, qn);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ compute side

// q ring: where the rows of the next staged step go.  A pure function of the sequence of row counts, so the issuer
// and the compute warps derive the same positions independently.  A step's rows never wrap (immediate offsets).
__device__ __forceinline__ int ring_place(int &pos, int rows, int NR)
{
    if (pos + rows > NR) pos = 0;
    const int at = pos;
    pos += rows;
    return at;
}

struct ComputeState {
#ifdef SMRE_ST_KO
    long long t_send = 0, t_recv = 0, t_bar = 0, t_macro = 0, t_last = 0;
#endif
    int pos = 0;                        // q ring: next free row
    unsigned mc = 0;                    // transitions done
    float *tcol;                        // my column of the tile: tcol[t * pitch], t = tile row
    unsigned long long *box0;           // my column of slot 0 of my mailbox, addressed the same way
    long long slot_words, dest_step;    // next slot of my mailbox; same slot of the next strip's mailbox
    unsigned long long *box_next;       // my column of the slot of the NEXT transition (built after the previous one)
    bool mine;                          // my thread owns an image column
    unsigned *seen_sh;                  // shared memory [6]: cached progress words of strips j-3..j-1, j+1..j+3
                                        // (flow control of their mailbox rings)
};

// Mailboxes: CTA `cta` owns ST_RING slots of st_tile_rows(T) rows of Wq words; transition number mc uses slot
// mc % ST_RING; a row is filed under the RECEIVER's tile row.  The same slot of strip j + d lies d * st_dest_step()
// further on (next mailbox, tile rows shifted by T).
__device__ __forceinline__ long long st_dest_step(const StripArgs &A)
{
    return (long long)ST_RING * st_tile_rows(A.T) * A.Wq - (long long)A.T * A.Wq;
}

// Flow control of the mailbox rings: before strip j + d's slot of transition `tag` is written, that strip must have
// read the slot's previous message (transition tag - ST_RING).  `seen` is a cached copy of its progress word,
// refreshed at every transition without waiting, so this almost never has to wait.
__device__ __forceinline__ void st_ring_space(const StripArgs &A, int cta, int d, unsigned tag, unsigned mc, unsigned &seen,
                                              Waiter &w)
{
    if (mc <= (unsigned)ST_RING || (int)(tag - ST_RING - seen) <= 0 || ST_KO(A, 128)) return;
    w.begin();
    do {
        seen = ld_relaxed_gpu32(A.done + (size_t)(cta + d) * 32);
    } while ((int)(tag - ST_RING - seen) > 0 && !w.slow(ST_W_DONE));
}

// Rows change owner between macro step e (just finished) and the next one; e holds the plan.  All compute threads
// of the CTA take part; on entry every tile write of the last step is visible (step barrier), on exit the tile holds
// the new row set.  Most departing values have already left, straight from the registers of the macro step's last
// family (band_group); here only what that family did not touch is sent: rows outside the active rows (image top /
// bottom) and the columns outside its windows (left / right remainder).  Sends wait for nothing but ring space, so
// the hand-offs of one transition cannot form a cycle.  A thread owns column tid (W <= compute threads).
// A row travels to slot (receiver's tile row) of the receiver's mailbox, whoever sends it.
__device__ __forceinline__ void transition(const StripArgs &A, int pitch, int j, int cta, unsigned long long splan,
                                           const HandProg *prog, ComputeState &cs, int tid, int NT, Waiter &w)
{
    constexpr int MAXR = 8;                                    // rows requested at once
    static_assert(ST_HOPS == 3, "the sends below are written out for three hops");
    static_assert((ST_RING & (ST_RING - 1)) == 0, "ST_RING must be a power of two");
    const unsigned mc = ++cs.mc;
    const unsigned tag = A.tag_base + mc;
    if (ST_KO(A, 1)) { bar_sync(2, NT); return; }
#ifdef SMRE_ST_KO
    const long long c0 = clock64();
    cs.t_macro += c0 - cs.t_last;
#endif
    const bool mine = cs.mine;
    float *const trow = cs.tcol;                                // trow[t * pitch]: tile row t, my column
    unsigned long long *const box = cs.box_next;                // box[t * pitch]: slot mc % ST_RING of my mailbox
    const uint4 p0 = reinterpret_cast<const uint4 *>(prog)[0];   // send_doff[0..2], send_meta[0]
    const uint4 p1 = reinterpret_cast<const uint4 *>(prog)[1];   // send_meta[1..2], counts, recv_rows[0]
    const unsigned counts = p1.z;

    // departures first: they are what the strips around are waiting for
    auto send_run = [&](int k, int row, int n, unsigned long long *dst) {
        const int d = k < ST_HOPS ? k - ST_HOPS : k - ST_HOPS + 1;
        unsigned seen = *(volatile unsigned *)(cs.seen_sh + k);
        st_ring_space(A, cta, d, tag, mc, seen, w);
        if (!mine) return;
        const float *src = trow + row * pitch;
#pragma unroll 1
        for (int r = 0; r < n; ++r) st_relaxed_gpu64(dst + r * pitch, pack_word(tag, src[r * pitch]));
    };
    if (counts & 0xff0000u) {                                   // more than three runs (does not happen at T = 4, 8)
#pragma unroll 1
        for (int k = 0; k < 2 * ST_HOPS; ++k) {
            const unsigned f = (unsigned)(splan >> (10 * k)) & 1023u;
            if (f == 0u) continue;
            const int d = k < ST_HOPS ? k - ST_HOPS : k - ST_HOPS + 1;
            send_run(k, (int)(f & 15u), (int)(f >> 4), box + d * cs.dest_step + (int)(f & 15u) * pitch);
        }
    } else {
        const int nsend = (int)(counts & 255u);
        if (nsend > 0) send_run((int)(p0.w >> 16), (int)(p0.w & 255u), (int)(p0.w >> 8) & 255, box + (int)p0.x);
        if (nsend > 1) send_run((int)(p1.x >> 16), (int)(p1.x & 255u), (int)(p1.x >> 8) & 255, box + (int)p0.y);
        if (nsend > 2) send_run((int)(p1.y >> 16), (int)(p1.y & 255u), (int)(p1.y >> 8) & 255, box + (int)p0.z);
    }
#ifdef SMRE_ST_KO
    const long long c1 = clock64();
#endif
    // progress words of the strips around (flow control of the mailbox rings at the NEXT transitions): one thread per
    // neighbour asks now and files the answer in shared memory after the arrivals
    unsigned s_new = 0;
    const int nd = tid < ST_HOPS ? tid - ST_HOPS : tid - ST_HOPS + 1;       // tid 0..5 -> strip j-3..j-1, j+1..j+3
    const bool asks = tid < 2 * ST_HOPS && j + nd >= 0 && j + nd < A.NS;
    if (asks) s_new = ld_relaxed_gpu32(A.done + (size_t)(cta + nd) * 32);

    // arrivals: all words of a batch are requested at once; a word whose tag is right goes to the tile, the others
    // are requested again
    const int nrecv = (int)(counts >> 8) & 255;
    auto recv_batch = [&](auto rtag, unsigned lo4, unsigned hi4, int cnt) {
        constexpr int R = decltype(rtag)::value;                // rows requested at once
        int off[R];
#pragma unroll
        for (int r = 0; r < R; ++r) off[r] = (int)(((r < 4 ? lo4 : hi4) >> (8 * (r & 3))) & 255u) * pitch;
        unsigned missing = cnt >= R ? (1u << R) - 1u : (1u << cnt) - 1u;
        for (;;) {
            unsigned long long wd[R];
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (missing >> r & 1u) wd[r] = ld_relaxed_gpu64(box + off[r]);
#pragma unroll
            for (int r = 0; r < R; ++r)
                if ((missing >> r & 1u) && (unsigned)(wd[r] >> 32) == tag) {
                    trow[off[r]] = __uint_as_float((unsigned)wd[r]);
                    missing &= ~(1u << r);
                }
            if (ST_KO(A, 64)) missing = 0;
            if (!missing || w.slow(ST_W_MAIL)) break;
            if (w.spins > 2u) __nanosleep(256);                 // a long wait (an idle strip): stop hammering L2
        }
    };
    if (mine && nrecv > 0) {
        w.begin();
        if (nrecv <= 2) {                                       // the usual case: one row per moving boundary
            recv_batch(std::integral_constant<int, 2>{}, p1.w, 0u, nrecv);
        } else {
#pragma unroll 1
            for (int r0 = 0; r0 < nrecv; r0 += MAXR) {
                unsigned lo4 = p1.w, hi4;                        // rows r0 .. r0 + 3, r0 + 4 .. r0 + 7
                if (r0 == 0) hi4 = prog->recv_rows[1];
                else { lo4 = prog->recv_rows[2]; hi4 = prog->recv_rows[3]; }
                recv_batch(std::integral_constant<int, MAXR>{}, lo4, hi4, nrecv - r0);
            }
        }
    }
    if (asks) *(volatile unsigned *)(cs.seen_sh + tid) = s_new;
#ifdef SMRE_ST_KO
    const long long c2 = clock64();
#endif
    bar_sync(2, NT);
    if (tid == 0) st_relaxed_gpu32(A.done + (size_t)cta * 32, tag);   // my mailbox slot of this transition is free again
    // the next transition's slot, built now and kept (it was rebuilt from the kernel parameters and %ctaid in front
    // of the sends, on the critical path of the strips around)
    cs.box_next = cs.box0 + (size_t)((mc + 1) & (ST_RING - 1)) * cs.slot_words;
    asm volatile("" : "+l"(cs.box_next));
#ifdef SMRE_ST_KO
    const long long c3 = clock64();
    cs.t_send += c1 - c0; cs.t_recv += c2 - c1; cs.t_bar += c3 - c2; cs.t_last = c3;
#endif
}

// One macro step: the S families (S, oy, 0..S-1) on the strip's bands; the strip interacts with nobody meanwhile.
// One named barrier per family step (compute warps + the waiter warp): every window of the next family overlaps
// windows of this one that other warps own.
template <int S, int G, bool HAS_Q, int PITCH>
__device__ __forceinline__ void macro_steps(const StripArgs &A, const MacroEntry &e, float *tile, const float *ring,
                                            int j, int cta, ComputeState &cs, int warp, int lane, int NTL, bool handoff,
                                            Waiter &w)
{
    (void)j; (void)cta; (void)handoff; (void)w;
    constexpr int CW = (32 / S) * S;
    const int pitch = PITCH ? PITCH : A.Wq;
    int W = A.W, NR = A.NR;
    const int src = (lane / S) * S;
    const float cth = e.c, sq = e.sqrt_c;
    const int rows = e.rows, nb = e.nb;
#ifdef SMRE_ST_KO
    const int ko = A.ko;
#else
    constexpr int ko = 0;
#endif
    const int col0 = warp * CW + lane;
    int w_end = lane < CW ? warp * CW + src + S : (1 << 28);   // end of the lane's window at ox = 0
    float *xt = tile + e.xoff + col0;
    float *qg = A.q + e.qoff + col0;
    size_t q_step = (size_t)A.Btot * A.H * pitch + 1;          // next family's plane, next column
    asm volatile("" : "+l"(q_step));                            // kept in registers: rebuilt from the kernel parameters
    asm volatile("" : "+r"(NTL));                               // it sat on the path to the step barrier
    const float *qcol = ring + col0;
    int elim_i = A.elim;
    asm volatile("" : "+r"(W), "+r"(NR), "+r"(elim_i));
    const bool elim = elim_i != 0;
#pragma unroll 1
    for (int ox = 0; ox < S; ++ox) {
        const bool on = w_end <= W;                            // the window lies inside the image (reading A6)
        const float *qs = HAS_Q ? qcol + ring_place(cs.pos, rows, NR) * pitch : nullptr;
        if (!(ko & 8)) {
            band_group<S, G, HAS_Q, PITCH>(xt, qs, qg, pitch, nb, on, src, cth, sq, ko, elim);
            for (int b0 = G; b0 < nb; b0 += G)                 // strips taller than one group
                band_group<S, G, HAS_Q, PITCH>(xt + b0 * S * pitch, HAS_Q ? qs + b0 * S * pitch : nullptr,
                                               qg + b0 * S * pitch, pitch, nb - b0, on, src, cth, sq, ko, elim);
        }
        ++w_end;
        ++xt;
        ++qcol;
        qg += q_step;
        if (!(ko & 16)) bar_sync(1, NTL);
    }
}

template <int S, int PITCH>
__device__ __forceinline__ void macro_step(const StripArgs &A, const MacroEntry &e, bool staged, float *tile,
                                           const float *ring, int j, int cta, ComputeState &cs, int warp, int lane,
                                           int NTL, bool handoff, Waiter &w)
{
    constexpr int GM = S == 1 ? 4 : 2;                         // bands handled together when there are several
    if (e.rows == 0) {                                         // nothing of this strip is inside a window row
        for (int ox = 0; ox < S; ++ox)
            if (!ST_KO(A, 16)) bar_sync(1, NTL);
        return;
    }
    if (S == ST_MAX_SIDE || e.rows == S) {
        if (staged) macro_steps<S, 1, true, PITCH>(A, e, tile, ring, j, cta, cs, warp, lane, NTL, handoff, w);
        else macro_steps<S, 1, false, PITCH>(A, e, tile, ring, j, cta, cs, warp, lane, NTL, handoff, w);
    } else {
        if (staged) macro_steps<S, GM, true, PITCH>(A, e, tile, ring, j, cta, cs, warp, lane, NTL, handoff, w);
        else macro_steps<S, GM, false, PITCH>(A, e, tile, ring, j, cta, cs, warp, lane, NTL, handoff, w);
    }
}

// ------------------------------------------------------------------------------------------------ q streaming
// Two warps besides the compute warps:
//   * the WAITER takes part in the step barrier.  Before arriving at the barrier of step g it waits (mbarrier) until
//     the q rows of step g + 1 have landed, so the compute warps never wait for q themselves; after the barrier it
//     publishes progress = g + 1 with release semantics: by then every compute warp has read the staged rows of
//     step g and issued its q stores of step g (the barrier orders both at CTA scope).
//   * the ISSUER is decoupled: it walks the step sequence ahead of everybody and issues the bulk copies of whole
//     batches of steps (up to 32 rows = one copy per lane), as far ahead as the ring, the stage count and the
//     one-sweep dependency (the rows of step h were written in step h - F) allow.  It reads `progress` with acquire
//     semantics and orders its async-proxy reads behind the generic-proxy writes with a proxy fence.
__device__ void waiter_warp(const StripArgs &A, const MacroEntry *tab, int M, uint64_t *full, unsigned *progress,
                            unsigned *abort_flag, const unsigned *stopped, int lane, int NTL)
{
    Waiter wt(A, abort_flag);
    const bool tol_mode = A.tol_mode != 0;
    const bool off = ST_KO(A, 2);
    const int total = A.n_sweeps * A.F;
    unsigned cn = 0;                           // staged non-empty steps consumed
    int g = 0;
#ifdef SMRE_ST_KO
    long long t_wait = 0, t_bar = 0; int n_late = 0;
#endif
    for (int sweep = 0; sweep < A.n_sweeps; ++sweep) {
        if (tol_mode && sweep > 0) {
            // top of a sweep under convergence control: the compute warps decide (barrier A); if the run goes on, the
            // q rows of the sweep's first family are awaited here, since nothing was issued across the decision
            bar_sync(3, NTL);
            if (*(volatile const unsigned *)stopped) return;
            if (!off && tab[0].rows > 0) {
                const unsigned stage = cn % ST_NSTG, parity = (cn / ST_NSTG) & 1u;
                if (!mbar_try_wait(&full[stage], parity)) {
                    wt.begin();
                    while (!mbar_try_wait(&full[stage], parity))
                        if (wt.slow(ST_W_QFULL)) break;
                }
            }
            bar_sync(3, NTL);
        }
        for (int m = 0; m < M; ++m) {
            const int crows = tab[m].rows, cs_ = tab[m].s;
            const int nrows_macro = tab[(m + 1 == M) ? 0 : m + 1].rows;
            const bool cur_staged = sweep > 0 && crows > 0 && !off;
            for (int ox = 0; ox < cs_; ++ox, ++g) {
                const bool last_ox = ox + 1 == cs_;
                const int nrows = last_ox ? nrows_macro : crows;
                const bool sweep_end = last_ox && m + 1 == M;
                const bool nstaged = sweep_end ? !tol_mode : sweep > 0;       // tol mode: see the top of the sweep
                if (!off && g + 1 < total && nstaged && nrows > 0) {
                    const unsigned n1 = cn + (cur_staged ? 1u : 0u);
                    const unsigned stage = n1 % ST_NSTG, parity = (n1 / ST_NSTG) & 1u;
#ifdef SMRE_ST_KO
                    const long long w0 = clock64();
#endif
                    if (!mbar_try_wait(&full[stage], parity)) {
#ifdef SMRE_ST_KO
                        ++n_late;
#endif
                        wt.begin();
                        while (!mbar_try_wait(&full[stage], parity))
                            if (wt.slow(ST_W_QFULL)) break;
                    }
#ifdef SMRE_ST_KO
                    t_wait += clock64() - w0;
#endif
                }
#ifdef SMRE_ST_KO
                const long long b0 = clock64();
#endif
                if (!ST_KO(A, 16)) bar_sync(1, NTL);
                if (cur_staged) ++cn;
                if (lane == 0) st_release_cta(progress, (unsigned)(g + 1));
#ifdef SMRE_ST_KO
                t_bar += clock64() - b0;
#endif
            }
        }
    }
#ifdef SMRE_ST_KO
    if ((A.ko & 256) && lane == 0 && (blockIdx.x % 40) == 3)
        printf("waiter cta %d: steps %d  q-wait %lld cycles/step  late %d  barrier+release %lld cycles/step\n", blockIdx.x, g,
               t_wait / max(g, 1), n_late, t_bar / max(g, 1));
#endif
}

// Position in the sequence of STAGED (sweep >= 1), NON-EMPTY steps, with the ring_place state before the step.
struct StagedCursor {
    int m = 0, ox = 0;          // macro step, family inside it
    int g;                      // global step index
    int pos = 0;                // ring_place state before this step
    unsigned n = 0;             // staged non-empty steps before this one
};
// skip macro steps in which the strip has no rows (they are not staged)
__device__ __forceinline__ void staged_skip_empty(StagedCursor &k, const MacroEntry *tab, int M, int total)
{
    while (k.g < total && tab[k.m].rows == 0) {
        k.g += tab[k.m].s - k.ox;
        k.ox = 0;
        if (++k.m == M) k.m = 0;
    }
}

template <int PITCH>
__device__ void issuer_warp(const StripArgs &A, const MacroEntry *tab, int M, float *ring, uint64_t *full,
                            unsigned *progress, unsigned *abort_flag, const unsigned *allow, const unsigned *stopped,
                            int frame, int lane)
{
    constexpr int KMAX = 4;                                     // steps per batch (bookkeeping stays in registers)
    const int pitch = PITCH ? PITCH : A.Wq;
    const size_t plane = (size_t)A.H * pitch;
    const size_t fam_stride = (size_t)A.Btot * plane;
    const uint32_t row_bytes = (uint32_t)pitch * 4u;
    const int NR = A.NR, F = A.F;
    const int total = A.n_sweeps * F;
    if (ST_KO(A, 2) || A.n_sweeps < 2) return;
    Waiter wt(A, abort_flag);
    StagedCursor head, tail;                   // head: next step to load; tail: oldest step not yet known to be consumed
    head.g = tail.g = F;                       // the first staged step is step F = sweep 1, first family
    staged_skip_empty(head, tab, M, total);
    tail = head;
    unsigned have = 0;                         // last value read from `progress` (= family steps completed)
    while (head.g < total) {
        const MacroEntry he = tab[head.m];
        const int rows = he.rows;
        // batch: up to 32 rows (one bulk copy per lane), inside this macro step; at most F - 1 steps, because the
        // waiter may need the first step of the batch while only the steps before it are complete; small enough to
        // fit the ring next to the step being consumed
        int k = min(min(32 / rows, KMAX), he.s - head.ox);
        k = min(k, max(1, F - 1));
        k = min(k, total - head.g);
        k = min(k, max(1, (NR - 2 * A.max_rows) / rows));
        // ring rows of the batch; `gap` = rows at the end of the ring skipped by a wrap inside the batch
        int at[KMAX];
        int p = head.pos, gap_lo = NR;
#pragma unroll
        for (int i = 0; i < KMAX; ++i)
            if (i < k) {
                if (p + rows > NR) gap_lo = p;
                at[i] = ring_place(p, rows, NR);
            }
        // what must have happened before the copies may be issued, as a count of completed family steps:
        // (a) the batch's rows were written one sweep earlier;
        unsigned need = (unsigned)(head.g + k - F);
        // (b) every older step whose ring rows (or mbarrier stage) the batch takes over has been consumed
        while (tail.g < head.g) {
            const int trows = tab[tail.m].rows;
            int tp = tail.pos;
            const int tat = ring_place(tp, trows, NR);
            bool pop = head.n + (unsigned)k - tail.n > (unsigned)ST_NSTG || tat + trows > gap_lo;
#pragma unroll
            for (int i = 0; i < KMAX; ++i)
                if (i < k && tat < at[i] + rows && at[i] < tat + trows) pop = true;
            if (!pop) break;
            need = max(need, (unsigned)(tail.g + 1));
            tail.pos = tp;
            ++tail.n;
            ++tail.g;
            if (++tail.ox == tab[tail.m].s) { tail.ox = 0; if (++tail.m == M) tail.m = 0; }
            staged_skip_empty(tail, tab, M, total);
        }
        if (A.tol_mode) {
            // under convergence control nothing of a sweep is loaded before the sweep has been decided: a copy in
            // flight into the shared memory of a CTA that has stopped would outlive it
            const unsigned sweep_of_batch = (unsigned)(head.g / F);
            if (ld_acquire_cta(allow) <= sweep_of_batch) {
                wt.begin();
                while (ld_acquire_cta(allow) <= sweep_of_batch) {
                    if (*(volatile const unsigned *)stopped) return;
                    if (wt.slow(ST_W_ALLOW)) break;
                }
            }
        }
        if (have < need) {
            wt.begin();
            while ((have = ld_acquire_cta(progress)) < need) {
                __nanosleep(200);                               // far ahead of the compute warps: do not take their issue slots
                if (wt.slow(ST_W_QFULL)) break;
            }
        }
        fence_proxy_async();                                    // generic-proxy q stores -> async-proxy reads
        if (lane < k) mbar_arrive_expect_tx(&full[(head.n + lane) % ST_NSTG], (uint32_t)rows * row_bytes);
        __syncwarp();
        {
            const int i = lane / rows, r = lane - i * rows;     // lane -> (step of the batch, row of the step)
            int my_at = at[0];
#pragma unroll
            for (int t = 1; t < KMAX; ++t)
                if (t == i) my_at = at[t];
            if (i < k) {
                const float *src = A.q + ((size_t)(he.fam0 + head.ox + i) * A.Btot + frame) * plane +
                                   (size_t)(he.lo + r) * pitch;
                bulk_load_row(ring + (size_t)(my_at + r) * pitch, src, row_bytes, &full[(head.n + i) % ST_NSTG]);
            }
        }
        (void)fam_stride;
        head.pos = p;
        head.n += (unsigned)k;
        head.g += k;
        head.ox += k;
        if (head.ox == he.s) { head.ox = 0; if (++head.m == M) head.m = 0; }
        staged_skip_empty(head, tab, M, total);
    }
}

// ------------------------------------------------------------------------------------------------ kernel
template <int PITCH, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) strips_kernel(const __grid_constant__ StripArgs A)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int pitch = PITCH ? PITCH : A.Wq;
    const int T = A.T, TR = st_tile_rows(T);
    float *tile = reinterpret_cast<float *>(smem_raw);
    float *ring = tile + TR * pitch;
    float *xprev = ring + (size_t)A.NR * pitch;                 // tol mode: x_{r-1} of the rows held at the top of a sweep
    uint64_t *full = reinterpret_cast<uint64_t *>(ring + (size_t)A.NR_total * pitch);
    MacroEntry *tab = reinterpret_cast<MacroEntry *>(full + ST_NSTG);
    unsigned *abort_flag = reinterpret_cast<unsigned *>(tab + ST_MAX_SIDES * ST_MAX_SIDE);
    unsigned *progress = abort_flag + 1;
    unsigned *allow = abort_flag + 2;                           // tol mode: sweeps the run is allowed to execute so far
    unsigned *stopped = abort_flag + 3;                         // tol mode: the stop rule has fired
    double *wsum = reinterpret_cast<double *>(abort_flag + 4);  // [ST_MAX_WARPS + 1] per-warp parts of ||x_r - x_{r-1}||^2
    unsigned *seen_sh = reinterpret_cast<unsigned *>(wsum + ST_MAX_WARPS + 2);   // [2 * ST_HOPS], see transition()
    HandProg *prog = reinterpret_cast<HandProg *>(seen_sh + 8);  // [macro steps]: the hand-off behind each of them

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NWC = A.NWC, NT = NWC * 32, NTL = NT + (ST_KO(A, 32) ? 0 : 32);
    const int cta = blockIdx.x, fl = cta / A.NS, j = cta - fl * A.NS, frame = A.frame0 + fl;
    const int H = A.H, W = A.W, NS = A.NS;

    // macro-step table of this strip
    int M = 0;
    for (int a = 0; a < A.n_sides; ++a) M += A.side[a];
    if ((int)threadIdx.x < M) {
        int a = 0, m0 = 0;
        while ((int)threadIdx.x >= m0 + A.side[a]) { m0 += A.side[a]; ++a; }
        const int s = A.side[a], oy = (int)threadIdx.x - m0;
        int s2 = s, oy2 = oy + 1;                                // the next macro step (cyclic)
        if (oy2 == s) { oy2 = 0; s2 = A.side[a + 1 == A.n_sides ? 0 : a + 1]; }
        int lo, hi;
        st_active_rows(j, NS, H, T, s, oy, lo, hi);
        MacroEntry e;
        e.s = (short)s; e.rows = (short)(hi - lo); e.lo = (short)lo; e.nb = (short)((hi - lo) / s);
        e.fam0 = A.fam_base[a] + oy * s; e.c = A.c[a]; e.sqrt_c = A.sqrt_c[a];
        e.xoff = (lo - j * T + T / 2) * pitch;
        e.qoff = ((long long)e.fam0 * A.Btot + frame) * ((long long)H * pitch) + (long long)lo * pitch;
        const int olo = st_boundary(j, NS, H, T, s, oy), ohi = st_boundary(j + 1, NS, H, T, s, oy);
        const int nlo = st_boundary(j, NS, H, T, s2, oy2), nhi = st_boundary(j + 1, NS, H, T, s2, oy2);
        e.hold_lo = (short)olo; e.hold_hi = (short)ohi;
        for (int k = 0; k < 2 * ST_HOPS; ++k) {
            const int d = k < ST_HOPS ? k - ST_HOPS : k - ST_HOPS + 1, jd = j + d;
            int slo = 0, shi = 0;
            if (jd >= 0 && jd < NS) {                            // what I hold now and strip j + d holds next
                slo = max(olo, st_boundary(jd, NS, H, T, s2, oy2));
                shi = min(ohi, st_boundary(jd + 1, NS, H, T, s2, oy2));
                if (shi < slo) shi = slo;
            }
            e.send_lo[k] = (short)slo; e.send_hi[k] = (short)shi;
        }
        // what I hold next and do not hold now: above / below what I keep
        e.recv_lo[0] = (short)nlo; e.recv_hi[0] = (short)max(nlo, min(nhi, olo));
        e.recv_lo[1] = (short)min(nhi, max(nlo, ohi)); e.recv_hi[1] = (short)nhi;
        e.pad0 = 0; e.pad1 = 0;
        const int tb = T / 2 - j * T;                            // image row -> tile row
        e.splan = 0; e.rplan = 0;
        for (int k = 0; k < 2 * ST_HOPS; ++k)
            if (e.send_hi[k] > e.send_lo[k])
                e.splan |= (unsigned long long)((e.send_lo[k] + tb) | ((e.send_hi[k] - e.send_lo[k]) << 4)) << (10 * k);
        for (int i = 0; i < 2; ++i)
            if (e.recv_hi[i] > e.recv_lo[i])
                e.rplan |= (unsigned long long)((e.recv_lo[i] + tb) | ((e.recv_hi[i] - e.recv_lo[i]) << 4)) << (10 * i);
        tab[threadIdx.x] = e;
        HandProg hp;
        const int dest_step = (int)st_dest_step(A);
        int ns = 0, nr = 0;
        unsigned general = 0;
        for (int i = 0; i < 3; ++i) { hp.send_doff[i] = 0; hp.send_meta[i] = 0; }
        for (int i = 0; i < 4; ++i) hp.recv_rows[i] = 0;
        for (int k = 0; k < 2 * ST_HOPS; ++k) {
            const int n = e.send_hi[k] - e.send_lo[k];
            if (n <= 0) continue;
            if (ns == 3) { general = 1; continue; }
            const int d = k < ST_HOPS ? k - ST_HOPS : k - ST_HOPS + 1, row = e.send_lo[k] + tb;
            hp.send_doff[ns] = d * dest_step + row * pitch;
            hp.send_meta[ns] = (unsigned)row | (unsigned)n << 8 | (unsigned)k << 16;
            ++ns;
        }
        for (int i = 0; i < 2; ++i)
            for (int y = e.recv_lo[i]; y < e.recv_hi[i]; ++y, ++nr)
                if (nr < 16) hp.recv_rows[nr >> 2] |= (unsigned)(y + tb) << (8 * (nr & 3));
        hp.counts = (unsigned)ns | (unsigned)nr << 8 | general << 16;
        hp.pad = 0;
        prog[threadIdx.x] = hp;
    }
    if (threadIdx.x == 0) {
        for (int i = 0; i < ST_NSTG; ++i) mbar_init(&full[i], 1);
        *abort_flag = 0u;
        *progress = 0u;
        *allow = A.tol_mode ? 1u : (unsigned)A.n_sweeps;
        *stopped = 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NWC) {
        if (!ST_KO(A, 32)) waiter_warp(A, tab, M, full, progress, abort_flag, stopped, lane, NTL);
    } else if (warp == NWC + 1) {
        issuer_warp<PITCH>(A, tab, M, ring, full, progress, abort_flag, allow, stopped, frame, lane);
    } else {
        const int tid = threadIdx.x;
        const int slot_base = T / 2 - j * T;
        // row a1: x <- y for the rows the strip holds under the first family's geometry (q needs no zeroing: the
        // first sweep reads none)
        const float *yim = A.y + (size_t)frame * H * W;
        for (int y = tab[0].hold_lo; y < tab[0].hold_hi; ++y)
            for (int c = tid; c < W; c += NT) tile[(y + slot_base) * pitch + c] = yim[(size_t)y * W + c];
        if (tid < 2 * ST_HOPS) seen_sh[tid] = A.tag_base;
        bar_sync(2, NT);
        ComputeState cs;
#ifdef SMRE_ST_KO
        cs.t_last = clock64();
#endif
        cs.seen_sh = seen_sh;
        cs.tcol = tile + tid;
        cs.slot_words = (long long)st_tile_rows(T) * pitch;
        cs.box0 = A.mail + (long long)cta * ST_RING * cs.slot_words + tid;
        cs.dest_step = st_dest_step(A);
        cs.box_next = cs.box0 + cs.slot_words;                   // transition 1 uses slot 1
        cs.mine = tid < W;
        Waiter wt(A, abort_flag);
        bool stopped_early = false;
        const int h_lo = tab[0].hold_lo, h_hi = tab[0].hold_hi;      // rows held at the top of EVERY sweep
        for (int sweep = 0; sweep < A.n_sweeps; ++sweep) {
            if (A.tol_mode) {
                // ---- Alg. 2's stop rule: after sweep r, stop if ||x_r - x_{r-1}||^2 <= delta ----------
                if (sweep > 0) {
                    float acc = 0.0f;                            // my columns of the rows I hold (same rows as a sweep ago)
                    for (int y = h_lo; y < h_hi; ++y)
                        for (int c = tid; c < W; c += NT) {
                            const float d = tile[(y + slot_base) * pitch + c] - xprev[(y - h_lo) * pitch + c];
                            acc = fmaf(d, d, acc);
                        }
                    double part = (double)acc;                   // fixed order from here on: deterministic decision
#pragma unroll
                    for (int m2 = 1; m2 < 32; m2 <<= 1) part += __shfl_xor_sync(0xffffffffu, part, m2);
                    if (lane == 0) wsum[warp] = part;
                    bar_sync(2, NT);
                    if (tid == 0) {
                        double mine = 0.0;
                        for (int k = 0; k < NWC; ++k) mine += wsum[k];
                        A.partials[(size_t)(sweep & 1) * gridDim.x + cta] = mine;
                        __threadfence();
                        atomicAdd(A.sweep_ctr + (size_t)fl * 32, 1u);
                        // every strip of the frame has delivered its part of this sweep
                        const unsigned need = (unsigned)NS * (unsigned)sweep;
                        unsigned got;
                        wt.begin();
                        for (;;) {
                            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(got) : "l"(A.sweep_ctr + (size_t)fl * 32) : "memory");
                            if (got >= need || wt.slow(ST_W_SWEEP)) break;
                        }
                        double d2 = 0.0;
                        const double *pp = A.partials + (size_t)(sweep & 1) * gridDim.x + (size_t)fl * NS;
                        for (int k = 0; k < NS; ++k) d2 += __ldcg(pp + k);
                        const bool stop = !(d2 > (double)A.delta);
                        if (stop) {
                            *(volatile unsigned *)stopped = 1u;
                            if (j == 0 && A.sweeps_done) A.sweeps_done[frame] = sweep;
                        } else {
                            st_release_cta(allow, (unsigned)sweep + 1u);      // the issuer may load this sweep's rows
                        }
                    }
                    bar_sync(3, NTL);                            // A: decision published (compute warps + waiter)
                    if (*(volatile unsigned *)stopped) { stopped_early = true; break; }
                }
                for (int y = h_lo; y < h_hi; ++y)                // x_{r-1} for the next check
                    for (int c = tid; c < W; c += NT) xprev[(y - h_lo) * pitch + c] = tile[(y + slot_base) * pitch + c];
                if (sweep > 0) bar_sync(3, NTL);                 // B: the waiter has the first family's q rows
            }
            for (int m = 0; m < M; ++m) {
                const MacroEntry e = tab[m];
                const unsigned long long splan = e.splan;
                const bool staged = sweep > 0 && !ST_KO(A, 2);
                const bool handoff = !(m + 1 == M && sweep + 1 == A.n_sweeps);   // none after the very last one
#define SMRE_RUN(S_)                                                                                                   \
    case S_: macro_step<S_, PITCH>(A, e, staged, tile, ring, j, cta, cs, warp, lane, NTL, handoff, wt); break;
                switch (e.s) {
                    SMRE_RUN(1) SMRE_RUN(2) SMRE_RUN(3) SMRE_RUN(4) SMRE_RUN(5) SMRE_RUN(6) SMRE_RUN(7) SMRE_RUN(8)
                }
#undef SMRE_RUN
                if (!handoff) break;
                transition(A, pitch, j, cta, splan, prog + m, cs, tid, NT, wt);
            }
        }
        if (A.tol_mode && !stopped_early && j == 0 && tid == 0 && A.sweeps_done) A.sweeps_done[frame] = A.n_sweeps;
#ifdef SMRE_ST_KO
        if ((A.ko & 256) && (tid == 0 || tid == 200) && (j == NS / 2 || j == NS / 2 + 1 || j == 3))
            printf("strip %d tid %d: transitions %u  send %lld  recv %lld  bar %lld  macro %lld cycles (avg per transition)\n", j, tid,
                   cs.mc, cs.t_send / max(cs.mc, 1u), cs.t_recv / max(cs.mc, 1u), cs.t_bar / max(cs.mc, 1u), cs.t_macro / max(cs.mc, 1u));
#endif
        // row a9: the rows the strip holds under the last family's geometry
        // (after an early stop: under the first family's, which a strip holds at the top of every sweep)
        float *xo = A.x_out + (size_t)frame * H * W;
        const int o_lo = stopped_early ? h_lo : tab[M - 1].hold_lo, o_hi = stopped_early ? h_hi : tab[M - 1].hold_hi;
        for (int y = o_lo; y < o_hi; ++y)
            for (int c = tid; c < W; c += NT) xo[(size_t)y * W + c] = tile[(y + slot_base) * pitch + c];
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
    int H = 0, W = 0, B = 0, Wq = 0, T = 0, NS = 0, NWC = 0, F = 0, NR = 0, max_rows = 0, frames_per_launch = 1;
    int n_sides = 0, side[ST_MAX_SIDES] = {}, fam_base[ST_MAX_SIDES] = {};
    float c[ST_MAX_SIDES] = {}, sqrt_c[ST_MAX_SIDES] = {};
    float *q = nullptr;
    unsigned long long *mail = nullptr;
    unsigned *done = nullptr, *status = nullptr, *finished = nullptr, *sweep_ctr = nullptr;
    double *partials = nullptr;
    unsigned *status_host = nullptr;                             // pinned, mapped
    unsigned *status_host_dev = nullptr;
    size_t mail_bytes = 0, smem_bytes = 0;
    unsigned tag_base = 1;
    unsigned long long timeout_ns = 2000000000ull;
    int elim = 1;
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

static size_t strips_fixed_smem() { return ST_NSTG * 8 + ST_MAX_SIDES * ST_MAX_SIDE * sizeof(MacroEntry) + 16 + (ST_MAX_WARPS + 2) * 8 + 32 + ST_MAX_SIDES * ST_MAX_SIDE * sizeof(HandProg); }

// Brute-force check of one strip height against every geometry of a sweep (host only, closed forms).
static bool strips_check_T(int H, int NS, int T, const int *sides, int n_sides, int *max_rows, int *max_hop,
                           char *why, size_t why_len)
{
    const int TR = st_tile_rows(T);
    *max_rows = 0;
    *max_hop = 0;
    for (int a = 0; a < n_sides; ++a)
        for (int oy = 0; oy < sides[a]; ++oy) {
            int s2 = sides[a], oy2 = oy + 1;
            if (oy2 == s2) { oy2 = 0; s2 = sides[(a + 1) % n_sides]; }
            for (int j = 0; j < NS; ++j) {
                int lo, hi;
                st_active_rows(j, NS, H, T, sides[a], oy, lo, hi);
                *max_rows = std::max(*max_rows, hi - lo);
                const int bt = st_boundary(j, NS, H, T, sides[a], oy), bb = st_boundary(j + 1, NS, H, T, sides[a], oy);
                if (bb > bt && (bt - j * T + T / 2 < 0 || bb - j * T + T / 2 > TR)) {
                    set_why(why, why_len, "strip %d does not fit its tile", j);
                    return false;
                }
                for (int y = bt; y < bb; ++y) {                 // who holds row y next?
                    int j2 = j;
                    while (j2 > 0 && y < st_boundary(j2, NS, H, T, s2, oy2)) --j2;
                    while (j2 + 1 < NS && y >= st_boundary(j2 + 1, NS, H, T, s2, oy2)) ++j2;
                    *max_hop = std::max(*max_hop, std::abs(j2 - j));
                }
            }
        }
    if (*max_hop > ST_HOPS) { set_why(why, why_len, "rows move %d strips at once (limit %d)", *max_hop, ST_HOPS); return false; }
    return true;
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
    if (F < 2) { set_why(why, why_len, "a single family per sweep leaves nothing to prefetch"); return false; }
    if (H > 32000 || W > 32000) { set_why(why, why_len, "image too large"); return false; }
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
    // strip height: the smallest one whose strips are all co-resident (one CTA per SM): more, thinner strips mean
    // fewer rows per CTA and step -- a strip never holds more than one band of a side >= T
    int T = 0, NS = 0, max_rows = 0, max_hop = 0;
    const int forced = getenv("SMRE_STRIP_T") ? atoi(getenv("SMRE_STRIP_T")) : 0;
    for (int t : {4, 8}) {
        if (forced && t != forced) continue;
        const int ns = (H + t - 1) / t;
        if (ns > sm_count) continue;
        if (!strips_check_T(H, ns, t, sides, n_sides, &max_rows, &max_hop, why, why_len)) continue;
        T = t; NS = ns;
        break;
    }
    if (!T) {
        if (why && !why[0]) set_why(why, why_len, "%d rows need more strips than the %d co-resident CTAs", H, sm_count);
        return false;
    }
    const long long tile_bytes = (long long)st_tile_rows(T) * Wq * 4;
    const long long ring_rows = (smem_optin - tile_bytes - (long long)strips_fixed_smem() - 128) / ((long long)Wq * 4);
    if (ring_rows < 3 * max_rows + 8) {
        set_why(why, why_len, "shared memory holds only %lld q rows of width %d", ring_rows, W);
        return false;
    }
    if (out) {
        out->T = T;
        out->strips = NS;
        out->warps = NWC;
        out->max_rows = max_rows;
        out->max_hop = max_hop;
        out->ring_rows = (int)std::min<long long>(ring_rows, 30000);
        out->frames_per_launch = std::max(1, std::min(B, sm_count / NS));
        const long long ctas = (long long)out->frames_per_launch * NS;
        out->workspace_bytes = ctas * ST_RING * st_tile_rows(T) * Wq * 8 + ctas * 128;
    }
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
    if (why && why_len) why[0] = 0;
    if (!strips_summary(H, W, B, sides, n_sides, sms, smem, &sm, why, why_len)) return nullptr;

    StripPlan *p = new StripPlan;
    p->device = dev;
    p->H = H; p->W = W; p->B = B; p->Wq = Wq; p->q = q;
    p->T = sm.T; p->NS = sm.strips; p->NWC = sm.warps; p->NR = sm.ring_rows; p->max_rows = sm.max_rows;
    p->frames_per_launch = sm.frames_per_launch;
    p->n_sides = n_sides;
    int F = 0;
    for (int a = 0; a < n_sides; ++a) {
        p->side[a] = sides[a]; p->c[a] = c[a]; p->sqrt_c[a] = sqrtf(c[a]); p->fam_base[a] = F;
        F += sides[a] * sides[a];
    }
    p->F = F;
    p->threads = (p->NWC + 2) * 32;                               // compute warps + waiter + issuer
    // two builds: up to 18 warps with 96 registers, else 64 (measured on C1, 21 warps: 64 and 88 registers run alike)
    const bool big = p->threads > 672;
    if (Wq == 512) p->kernel = big ? kernel_ptr<512, 1024>() : kernel_ptr<512, 672>();
    else p->kernel = big ? kernel_ptr<0, 1024>() : kernel_ptr<0, 672>();
    p->smem_bytes = (size_t)st_tile_rows(p->T) * Wq * 4 + (size_t)p->NR * Wq * 4 + strips_fixed_smem();
    if (const char *e = getenv("SMRE_DENSE_STORES")) p->elim = atoi(e) ? 0 : 1;
    if (const char *e = getenv("SMRE_TIMEOUT_MS")) {
        const long long ms = atoll(e);
        if (ms > 0) p->timeout_ns = (unsigned long long)ms * 1000000ull;
    }
    const size_t ctas = (size_t)p->frames_per_launch * p->NS;
    p->mail_bytes = ctas * ST_RING * st_tile_rows(p->T) * Wq * 8;
    cudaError_t e = cudaFuncSetAttribute(p->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&p->mail, p->mail_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&p->done, ctas * 128);
    if (e == cudaSuccess) e = cudaMalloc(&p->status, 256);
    if (e == cudaSuccess) e = cudaMalloc(&p->partials, 2 * ctas * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&p->sweep_ctr, (size_t)p->frames_per_launch * 128);
    if (e == cudaSuccess) e = cudaHostAlloc(&p->status_host, 64, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&p->status_host_dev, p->status_host, 0);
    if (e == cudaSuccess) e = cudaMemset(p->mail, 0, p->mail_bytes);
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
    if (p->mail) cudaFree(p->mail);
    if (p->done) cudaFree(p->done);
    if (p->status) cudaFree(p->status);
    if (p->partials) cudaFree(p->partials);
    if (p->sweep_ctr) cudaFree(p->sweep_ctr);
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
    return strips_run_tol(p, y, x_out, n_sweeps, false, 0.0f, nullptr, st, launches);
}

cudaError_t strips_run_tol(StripPlan *p, const float *y, float *x_out, int n_sweeps, bool tol_mode, float delta,
                           int *sweeps_done, cudaStream_t st, long long *launches)
{
    const int xprev_rows = tol_mode ? st_tile_rows(p->T) : 0;           // x_{r-1} is taken out of the q ring
    if (p->NR - xprev_rows < 3 * p->max_rows + 8) return cudaErrorNotSupported;
    int M = 0;
    for (int a = 0; a < p->n_sides; ++a) M += p->side[a];
    const unsigned long long total = (unsigned long long)n_sweeps * M + 2;
    if (total >= 0x40000000ull || (unsigned long long)n_sweeps * p->F >= 0x7fffffffull) return cudaErrorNotSupported;
    cudaError_t e = cudaMemsetAsync(p->status, 0, 256, st);
    if (e != cudaSuccess) return e;
    for (int f0 = 0; f0 < p->B; f0 += p->frames_per_launch) {
        const int nf = std::min(p->frames_per_launch, p->B - f0);
        if (p->tag_base + total < p->tag_base || p->tag_base + total > 0xfffffff0u) {     // 32-bit tags used up: start over
            e = cudaMemsetAsync(p->mail, 0, p->mail_bytes, st);
            if (e == cudaSuccess) e = cudaMemsetAsync(p->done, 0, (size_t)p->frames_per_launch * p->NS * 128, st);
            if (e != cudaSuccess) return e;
            p->tag_base = 1;
        }
        StripArgs A{};
        A.y = y; A.x_out = x_out; A.q = p->q;
        A.mail = p->mail; A.done = p->done;
        A.status = p->status; A.status_host = p->status_host_dev; A.finished = p->finished;
        A.H = p->H; A.W = p->W; A.Wq = p->Wq; A.Btot = p->B; A.frame0 = f0;
        A.T = p->T; A.NS = p->NS; A.NWC = p->NWC; A.n_sides = p->n_sides; A.F = p->F; A.n_sweeps = n_sweeps;
        A.NR = p->NR - xprev_rows; A.NR_total = p->NR; A.max_rows = p->max_rows;
        A.tol_mode = tol_mode ? 1 : 0; A.delta = delta; A.partials = p->partials; A.sweep_ctr = p->sweep_ctr;
        A.sweeps_done = sweeps_done;
        if (tol_mode) {
            e = cudaMemsetAsync(p->sweep_ctr, 0, (size_t)p->frames_per_launch * 128, st);
            if (e != cudaSuccess) return e;
        }
        for (int a = 0; a < p->n_sides; ++a) {
            A.side[a] = p->side[a]; A.fam_base[a] = p->fam_base[a]; A.c[a] = p->c[a]; A.sqrt_c[a] = p->sqrt_c[a];
        }
        A.tag_base = p->tag_base;
        A.timeout_ns = p->timeout_ns;
        A.elim = p->elim;
#ifdef SMRE_ST_KO
        A.ko = getenv("SMRE_ST_KO") ? atoi(getenv("SMRE_ST_KO")) : 0;
#endif
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
