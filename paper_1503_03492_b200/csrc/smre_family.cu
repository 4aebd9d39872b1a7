// Per-family projection pass as a stand-alone kernel: the building block
// of the SMRE_SCHED_GRAPH scheduler.  One launch = one family (s, oy, ox) over all frames.
//
// For every window S of the family (they are disjoint):
//     v = x_S + q_S;  n2 = sum v^2;  x_S = v * (n2 > c ? sqrt(c/n2) : 1);  q_S = v - x_S
// (Eq. 14; update rule Listing 3).
//
// Mapping: G = next power of two >= side lanes per window, lane j owns COLUMN j of its window and
// keeps the `side` values of that column in registers, so a warp touches 32/G neighbouring windows
// and every row access of the warp is one contiguous segment of (32/G)*side floats (coalesced).
// The sum of squares is a column-serial sum followed by a fixed xor-shuffle tree over the G lanes,
// neighbouring columns first: deterministic run to run, and the order the strip scheduler's sliding
// window sums use (smre_strips.cu, window_total), so both schedulers round identically.
#include "smre_common.cuh"

namespace smre {

template <int G>
__global__ void __launch_bounds__(256)
family_pass_kernel(float *__restrict__ x, float *__restrict__ q, int H, int W, int Wq, Family f,
                   int chunks_per_row)
{
    constexpr int WPW = 32 / G;                      // windows per warp
    const int lane = threadIdx.x & 31;
    const int warp = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    if (warp >= f.ny * chunks_per_row) return;       // warp-uniform
    const int wrow = warp / chunks_per_row;
    const int chunk = warp - wrow * chunks_per_row;
    const int wi = chunk * WPW + lane / G;           // window index along x
    const int j = lane % G;                          // column inside the window
    const bool on = (wi < f.nx) && (j < f.side);
    const size_t base = ((size_t)blockIdx.y * H + (size_t)(f.oy + wrow * f.side)) * W
                      + (size_t)(f.ox + wi * f.side + j);
    const size_t qbase = ((size_t)blockIdx.y * H + (size_t)(f.oy + wrow * f.side)) * Wq
                       + (size_t)(f.ox + wi * f.side + j);     // q planes have row pitch Wq

    float v[G];
    float part = 0.0f;
#pragma unroll
    for (int r = 0; r < G; ++r) {
        v[r] = 0.0f;
        if (r < f.side && on) {
            v[r] = __fadd_rn(x[base + (size_t)r * W], q[qbase + (size_t)r * Wq]);
        }
        part = fmaf(v[r], v[r], part);
    }
#pragma unroll
    for (int m = 1; m < G; m <<= 1) part += __shfl_xor_sync(0xffffffffu, part, m);     // pairs first: (c0+c1)+(c2+c3) ...

    const float alpha = ball_scale(part, f.c, f.sqrt_c);
#pragma unroll
    for (int r = 0; r < G; ++r) {
        if (r < f.side && on) {
            float xn, qn;
            ball_update(v[r], alpha, xn, qn);
            x[base + (size_t)r * W] = xn;
            q[qbase + (size_t)r * Wq] = qn;
        }
    }
}

template <int G>
static cudaError_t launch_g(float *x, float *q, int B, int H, int W, int Wq, const Family &f, cudaStream_t st)
{
    constexpr int WPW = 32 / G;
    const int chunks = (f.nx + WPW - 1) / WPW;
    const long long warps = (long long)f.ny * chunks;
    if (warps == 0) return cudaSuccess;
    const int warps_per_block = 8;
    dim3 grid((unsigned)((warps + warps_per_block - 1) / warps_per_block), (unsigned)B);
    family_pass_kernel<G><<<grid, warps_per_block * 32, 0, st>>>(x, q, H, W, Wq, f, chunks);
    return cudaGetLastError();
}

cudaError_t launch_family_pass(float *x, float *q_plane, int B, int H, int W, int Wq, const Family &f,
                               cudaStream_t st)
{
    const int s = f.side;
    if (s <= 1) return launch_g<1>(x, q_plane, B, H, W, Wq, f, st);
    if (s <= 2) return launch_g<2>(x, q_plane, B, H, W, Wq, f, st);
    if (s <= 4) return launch_g<4>(x, q_plane, B, H, W, Wq, f, st);
    if (s <= 8) return launch_g<8>(x, q_plane, B, H, W, Wq, f, st);
    if (s <= 16) return launch_g<16>(x, q_plane, B, H, W, Wq, f, st);
    return launch_g<32>(x, q_plane, B, H, W, Wq, f, st);
}

}  // namespace smre
