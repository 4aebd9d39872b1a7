// Shared declarations of the CUDA path (sm_100a).  Not used by, and shares nothing with, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace smre {

struct Family {
    int side, oy, ox;   // windows of edge `side` with origin == (oy, ox) mod side
    int ny, nx;         // floor((H-oy)/side), floor((W-ox)/side): windows fully inside (reading A6)
    float c;            // threshold c_S = 1/c_s(alpha)                                 (Eq. 5)
    float sqrt_c;       // sqrtf(c), rounded once on the host
};

// Eq. 14 in threshold form: scale factor alpha = sqrt(c/n2) of a window whose sum
// of squares is n2, 1 when the window is inside its ball.  Strict compare (reading A5).
// Default: sqrt(c) * rsqrt(n2) with the hardware reciprocal square root (MUFU.RSQ, <= 2 ulp):
// branch-free and ~4x shorter on the dependent chain that bounds a family step than IEEE
// division + square root.  -DSMRE_PRECISE_SCALE selects sqrt_rn(div_rn(c, n2)) for A/B checks.
// Every scheduler and both variants use this one function, so they agree bit for bit.
__device__ __forceinline__ float ball_scale(float n2, float c, float sqrt_c) {
#ifdef SMRE_PRECISE_SCALE
    (void)sqrt_c;
    return (n2 > c) ? __fsqrt_rn(__fdiv_rn(c, n2)) : 1.0f;
#else
    // rsqrt.approx.ftz: the bare MUFU.RSQ.  rsqrtf() wraps it in a denormal rescue that can never trigger
    // here (the branch is only taken for n2 > c > 0, far from the denormal range) but sits on the chain.
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(n2));
    return (n2 > c) ? sqrt_c * r : 1.0f;
#endif
}

// The update of one pixel of a projected window (Listing 3): x' = alpha*v, q' = v - x'.
// Written with explicit round-to-nearest operations so that no compiler contracts v - alpha*v into one fma
// in one kernel and not in another: every scheduler and both variants round identically.
__device__ __forceinline__ void ball_update(float v, float alpha, float &xn, float &qn)
{
    xn = __fmul_rn(alpha, v);
    qn = __fsub_rn(v, xn);
}

// smre_api.cu: text returned by smre_last_error() on the calling thread (for entry points in other files)
void set_last_error(const char *text);

// ---- launchers implemented in the .cu files --------------------------------------------------

// smre_family.cu: one family pass over all frames (schedule SMRE_SCHED_GRAPH).  x: [B][H][W];
// q_plane: [B][H][Wq], Wq = W rounded up to a multiple of 4 (16-byte aligned rows for cp.async).
cudaError_t launch_family_pass(float *x, float *q_plane, int B, int H, int W, int Wq, const Family &f,
                               cudaStream_t st);

// smre_icd.cu: one shift of the incomplete Dykstra (P_{Omega^i}).
struct IcdLevels {
    float c[6];         // c[k]: threshold of side 2^k, k = 0..K
    float sqrt_c[6];
};
// src may equal dst.  K <= 5.
cudaError_t launch_icd_shift(const float *src, float *dst, int B, int H, int W, int K, int shift_i,
                             const IcdLevels &lv, int n_cycles, cudaStream_t st);

// Same with the stop rule of Listing 3: every tile iterates until its sum |x_old - x_new| of one
// cycle is <= tol * L^2, at most n_cycles cycles.  tile_cycles: null or [B][tiles_y][tiles_x] ints (icd_tiles_along).
cudaError_t launch_icd_shift_tol(const float *src, float *dst, int B, int H, int W, int K, int shift_i,
                                 const IcdLevels &lv, int n_cycles, cudaStream_t st, bool use_tol, float tol,
                                 int *tile_cycles);
int icd_tiles_along(int N, int K, int shift_i);

}  // namespace smre
