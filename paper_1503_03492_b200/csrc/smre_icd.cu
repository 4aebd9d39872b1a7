// Incomplete Dykstra (ICD), one shift: P_{Omega^i} of PAPER.md:373-381.
//
// The paper's kernel (Listing 3) gives one 32x32 tile to a 1024-thread block,
// one pixel per thread, q[6][1024] + two scratch arrays in shared memory and a shared-memory tree
// per level.  Here a tile of edge L = 2^K lives entirely in REGISTERS: every lane owns a 4x4 pixel
// block (P x P, P = min(L,4)) of x and of each level's increment q[k], so
//   * levels 1x1, 2x2, 4x4 are reduced inside the lane (no communication at all),
//   * levels 8, 16, 32 are a 4x4-block partial sum + an xor-shuffle tree over the 4 / 16 / 32 lanes
//     of the window (lanes are Morton-ordered inside the tile, so each window is an aligned lane
//     group); a 32x32 tile spans two warps and adds one shared-memory exchange,
//   * all n_cycles inner cycles of the shift run without touching memory; x is read once and
//     written once per shift; q never exists outside the register file (row a7).
// Tiles start at (2^i mod L) - L on both axes ("virtual" tiles overhang the border); windows that
// are not fully inside the image are skipped (reading A-ICD-13), pixels outside are never stored.
#include "smre_common.cuh"

namespace smre {

__device__ __forceinline__ int morton_even_bits(int t) {   // bits 0,2,4 of t -> 0,1,2
    return (t & 1) | ((t >> 1) & 2) | ((t >> 2) & 4);
}

// Pixel block per lane (LP = log2 of its edge): 4x4 is the throughput choice (fewest shuffles per pixel);
// 2x2 gives four times the lanes and a shorter dependent chain per level pass, which wins when the whole
// problem is too small to fill the machine (C2: 512^2, K = 3).  Tiles of 16x16 and 32x32 need 4x4 (a tile
// must fit in two warps).
// TOL: the stop rule of Listing 3: a tile stops after the first cycle whose sum over the
// tile's pixels and the cycle's levels of |x_old - x_new| is <= thresh = tol * L^2 (fp32; the lanes of a tile add
// their parts with an xor-shuffle tree), or after n_cycles cycles.  Tiles that have stopped keep x and q frozen
// while other tiles of the warp go on.  tile_cycles (may be null): cycles every tile ran.
template <int K, int LP, bool TOL>
__global__ void __launch_bounds__(128)
icd_shift_kernel(const float *src, float *dst, int H, int W, int org,
                 int nty, int ntx, long long n_tiles, int smin, IcdLevels lv, int n_cycles,
                 float thresh, int *tile_cycles)
{
    constexpr int L = 1 << K;
    constexpr int P = 1 << LP;                    // pixel block edge per lane: 1, 2, 2, 2, 4, 4
    constexpr int NB = L / P;                     // blocks per tile edge
    constexpr int LPT = NB * NB;                  // lanes per tile: 1, 1, 4, 16, 16, 64
    constexpr int KIN = K < LP ? K : LP;          // highest level reduced inside a lane
    constexpr int NP = P * P;

    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long tile = g / LPT;
    const int t = (int)(g % LPT);
    const bool tile_ok = tile < n_tiles;
    const long long per_frame = (long long)nty * ntx;
    const long long b = tile_ok ? tile / per_frame : 0;
    const int rem = (int)(tile_ok ? tile - b * per_frame : 0);
    const int tyi = rem / ntx, txi = rem - tyi * ntx;
    const int bx = morton_even_bits(t), by = morton_even_bits(t >> 1);
    const int ty0 = org + tyi * L, tx0 = org + txi * L;          // tile origin (may be < 0)
    const int gy0 = ty0 + by * P, gx0 = tx0 + bx * P;            // this lane's block origin
    const size_t frame = (size_t)b * H * W;

    // ---- load the block; outside pixels read as 0 and are never written ----------------------
    float x[NP];
    unsigned pix_in = 0;                                          // bit r*P+c: pixel inside image
#pragma unroll
    for (int r = 0; r < P; ++r)
#pragma unroll
        for (int c = 0; c < P; ++c) {
            const int gy = gy0 + r, gx = gx0 + c;
            const bool in = tile_ok && gy >= 0 && gy < H && gx >= 0 && gx < W;
            x[r * P + c] = in ? src[frame + (size_t)gy * W + gx] : 0.0f;
            pix_in |= (in ? 1u : 0u) << (r * P + c);
        }

    // ---- which windows are fully inside (per level) -------------------------------------------
    // in-lane levels: one bit per window of the block; higher levels: one flag per level
    unsigned win_ok[KIN + 1];
#pragma unroll
    for (int k = 0; k <= KIN; ++k) {
        const int S = 1 << k, NW = P >> k;
        unsigned m = 0;
#pragma unroll
        for (int wy = 0; wy < NW; ++wy)
#pragma unroll
            for (int wx = 0; wx < NW; ++wx) {
                bool ok = true;
#pragma unroll
                for (int r = 0; r < S; ++r)
#pragma unroll
                    for (int c = 0; c < S; ++c)
                        ok = ok && ((pix_in >> ((wy * S + r) * P + wx * S + c)) & 1u);
                m |= (ok ? 1u : 0u) << (wy * NW + wx);
            }
        win_ok[k] = m;
    }
    bool big_ok[K > KIN ? K - KIN : 1];
#pragma unroll
    for (int k = KIN + 1; k <= K; ++k) {
        const int S = 1 << k;
        const int wy0 = ty0 + (((by * P) >> k) << k), wx0 = tx0 + (((bx * P) >> k) << k);
        big_ok[k - KIN - 1] = tile_ok && wy0 >= 0 && wx0 >= 0 && wy0 + S <= H && wx0 + S <= W;
    }

    float q[K + 1][NP];
#pragma unroll
    for (int k = 0; k <= K; ++k)
#pragma unroll
        for (int p = 0; p < NP; ++p) q[k][p] = 0.0f;              // "Set q = 0"

    __shared__ float red[4];
    __shared__ float dred[4];
    bool active = true;                                           // TOL: the lane's tile still iterates
    int my_cycles = 0;

    for (int cyc = 0; cyc < n_cycles; ++cyc) {
        float delta = 0.0f;                                       // TOL: sum |x_old - x_new| of my pixels, this cycle
        if (TOL) {
            if (LPT > 32) { if (!__syncthreads_or(active)) break; }          // a tile spans two warps
            else if (!__any_sync(0xffffffffu, active)) break;
        }
        // coarse -> fine: for (s = K; s >= smin; s--)
#pragma unroll
        for (int k = K; k >= 0; --k) {
            if (k < smin) continue;                               // warp-uniform
            if (k > KIN) {
                // ---- window spans several lanes ----------------------------------------------
                float v[NP];
                float part = 0.0f;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    v[p] = x[p] + q[k][p];
                    part = fmaf(v[p], v[p], part);
                }
                const int lanes = 1 << (2 * (k - LP));            // 4, 16, 64
#pragma unroll
                for (int m = 1; m < 32; m <<= 1)
                    if (m < lanes) part += __shfl_xor_sync(0xffffffffu, part, m);
                if (lanes > 32) {                                 // K == 5 top level: two warps
                    const int w = threadIdx.x >> 5;
                    if ((threadIdx.x & 31) == 0) red[w] = part;
                    __syncthreads();
                    part = red[w & ~1] + red[w | 1];
                    __syncthreads();
                }
                const float alpha = big_ok[k > KIN ? k - KIN - 1 : 0]
                                        ? ball_scale(part, lv.c[k], lv.sqrt_c[k]) : 1.0f;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const float xn = alpha * v[p];
                    if (!TOL || active) {
                        if (TOL) delta += fabsf(x[p] - xn);
                        q[k][p] = v[p] - xn;
                        x[p] = xn;
                    }
                }
            } else {
                // ---- windows inside the lane's block ------------------------------------------
                const int S = 1 << k, NW = P >> k;
#pragma unroll
                for (int wy = 0; wy < NW; ++wy)
#pragma unroll
                    for (int wx = 0; wx < NW; ++wx) {
                        float v[16];
                        float n2 = 0.0f;
#pragma unroll
                        for (int r = 0; r < S; ++r)
#pragma unroll
                            for (int c = 0; c < S; ++c) {
                                const int p = (wy * S + r) * P + wx * S + c;
                                v[r * S + c] = x[p] + q[k][p];
                                n2 = fmaf(v[r * S + c], v[r * S + c], n2);
                            }
                        const bool ok = (win_ok[k <= KIN ? k : 0] >> (wy * NW + wx)) & 1u;
                        const float alpha = ok ? ball_scale(n2, lv.c[k], lv.sqrt_c[k]) : 1.0f;
#pragma unroll
                        for (int r = 0; r < S; ++r)
#pragma unroll
                            for (int c = 0; c < S; ++c) {
                                const int p = (wy * S + r) * P + wx * S + c;
                                const float xn = alpha * v[r * S + c];
                                if (!TOL || active) {
                                    if (TOL) delta += fabsf(x[p] - xn);
                                    q[k][p] = v[r * S + c] - xn;
                                    x[p] = xn;
                                }
                            }
                    }
            }
        }
        if (TOL) {                                                // the tile's delta: tree over its LPT lanes
#pragma unroll
            for (int m = 1; m < 32; m <<= 1)
                if (m < LPT) delta += __shfl_xor_sync(0xffffffffu, delta, m);
            if (LPT > 32) {
                const int w = threadIdx.x >> 5;
                if ((threadIdx.x & 31) == 0) dred[w] = delta;
                __syncthreads();
                delta = dred[w & ~1] + dred[w | 1];
            }
            if (active) {
                ++my_cycles;
                if (!(delta > thresh)) active = false;            // while (delta > tol*1024)
            }
        }
    }
    if (TOL && tile_cycles && tile_ok && t == 0) tile_cycles[tile] = my_cycles;

#pragma unroll
    for (int r = 0; r < P; ++r)
#pragma unroll
        for (int c = 0; c < P; ++c)
            if ((pix_in >> (r * P + c)) & 1u)
                dst[frame + (size_t)(gy0 + r) * W + (gx0 + c)] = x[r * P + c];
}

template <int K, int LP>
static cudaError_t launch_kp(const float *src, float *dst, int B, int H, int W, int shift_i,
                             const IcdLevels &lv, int n_cycles, cudaStream_t st, bool use_tol, float tol,
                             int *tile_cycles)
{
    constexpr int L = 1 << K;
    constexpr int P = 1 << LP;
    constexpr int LPT = (L / P) * (L / P);
    const int o = (1 << shift_i) % L;
    const int org = o ? o - L : 0;
    const int nty = (H - org + L - 1) / L, ntx = (W - org + L - 1) / L;
    const long long n_tiles = (long long)B * nty * ntx;
    const long long lanes = n_tiles * LPT;
    const int threads = 128;
    const long long blocks = (lanes + threads - 1) / threads;
    if (use_tol)
        icd_shift_kernel<K, LP, true><<<(unsigned)blocks, threads, 0, st>>>(src, dst, H, W, org, nty, ntx, n_tiles, shift_i, lv,
                                                                       n_cycles, tol * (float)(L * L), tile_cycles);
    else
        icd_shift_kernel<K, LP, false><<<(unsigned)blocks, threads, 0, st>>>(src, dst, H, W, org, nty, ntx, n_tiles, shift_i, lv,
                                                                        n_cycles, 0.0f, nullptr);
    return cudaGetLastError();
}

template <int K>
static cudaError_t launch_k(const float *src, float *dst, int B, int H, int W, int shift_i,
                            const IcdLevels &lv, int n_cycles, cudaStream_t st, bool use_tol, float tol,
                            int *tile_cycles)
{
    constexpr int LPmax = K < 2 ? K : 2;                   // 4x4 blocks where the tile allows it
    if constexpr (K == 2 || K == 3) {
        // lanes the 4x4 layout would give; below about half a machine of resident threads use 2x2 blocks
        const long long lanes4 = (long long)B * ((H + (1 << K) - 1) >> K) * ((W + (1 << K) - 1) >> K) * (1 << (2 * (K - 2)));
        if (lanes4 < 148ll * 1024) return launch_kp<K, 1>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
    }
    return launch_kp<K, LPmax>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
}

// tiles of shift i along an axis of extent N (tile edge 2^K): the layout of the per-tile cycle counts
int icd_tiles_along(int N, int K, int shift_i)
{
    const int L = 1 << K, o = (1 << shift_i) % L, org = o ? o - L : 0;
    return (N - org + L - 1) / L;
}

cudaError_t launch_icd_shift(const float *src, float *dst, int B, int H, int W, int K, int shift_i,
                             const IcdLevels &lv, int n_cycles, cudaStream_t st)
{
    return launch_icd_shift_tol(src, dst, B, H, W, K, shift_i, lv, n_cycles, st, false, 0.0f, nullptr);
}

cudaError_t launch_icd_shift_tol(const float *src, float *dst, int B, int H, int W, int K, int shift_i,
                                 const IcdLevels &lv, int n_cycles, cudaStream_t st, bool use_tol, float tol,
                                 int *tile_cycles)
{
    switch (K) {
        case 0: return launch_k<0>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        case 1: return launch_k<1>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        case 2: return launch_k<2>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        case 3: return launch_k<3>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        case 4: return launch_k<4>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        case 5: return launch_k<5>(src, dst, B, H, W, shift_i, lv, n_cycles, st, use_tol, tol, tile_cycles);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace smre
