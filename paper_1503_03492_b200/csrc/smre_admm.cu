// ADMM around the projection (Alg. 1, Eq. 9-13; readings A-ADMM-1..9 of
// DESIGN.md).  Everything of an iteration runs on the device; the host only enqueues and looks at the stop flag
// every `check_every` iterations (once the flag is up the remaining kernels of the batch return at once, so the
// state is that of the iteration that stopped).
//
// Per iteration, given x, A*x, eps, z, Y1, Y2 and w = rho1 (I - A*x - eps) + Y1:
//   1. rows / columns of A^T * w (= A * w: symmetric operator, A-ADMM-2); fused behind the column pass:
//      x <- x - (-A^T*w + rho2 (x - z) + Y2) / (2 gamma), partial sums of ||x_{r+1} - x_r||^2         (Eq. 11, A-ADMM-3)
//   2. rows / columns of A * x; fused behind the column pass: X = I - A*x + Y1 / rho1                   (argument of Eq. 12)
//   3. eps' = P_G(X): smre_project on the caller's handle (either variant, the hot path of this library)
//   4. z = (rho2 x + Y2) / (lambda + rho2), Y1 += alpha1 (I - A*x - eps'), Y2 += alpha2 (x - z), eps = eps',
//      the next w, partial sums of ||I - A*x - eps||^2                                                  (Alg. 1, A-ADMM-4, -7)
//   5. one block adds the partial sums in a fixed order, writes the two norms, counts the iteration and raises the
//      stop flag when both norms are <= delta                                                           (A-ADMM-6)
#include <cuda_runtime.h>
#include <cmath>
#include <cstdio>
#include <cstdint>
#include "../../include/smre.h"
#include "smre_common.cuh"

namespace smre {
namespace {

constexpr int ADMM_MAX_RADIUS = 32;
struct Taps { int radius; float g[2 * ADMM_MAX_RADIUS + 1]; };

struct AdmmState {
    const float *I;
    float *x, *Ax, *eps, *eps_next, *z, *Y1, *Y2, *w, *tmp, *X;
    double *part_dx, *part_res;        // [blocks]
    float *hist;                       // [2 * max_iter] or null
    int *iters;                        // iterations done
    int *stopped;                      // stop flag
    int H, W, blocks;
    float rho1, rho2, alpha1, alpha2, lambda, inv2gamma, delta;
};

// horizontal pass, zero outside the image
__global__ void admm_rows_kernel(const float *__restrict__ in, float *__restrict__ out, int H, int W, Taps t, const int *stopped)
{
    if (stopped && *stopped) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (c >= W) return;
    const float *row = in + (size_t)y * W;
    float a = 0.0f;
    for (int k = -t.radius; k <= t.radius; ++k) {
        const int cc = c + k;
        if (cc >= 0 && cc < W) a = fmaf(t.g[k + t.radius], row[cc], a);
    }
    out[(size_t)y * W + c] = a;
}

__device__ __forceinline__ float column_pass(const float *__restrict__ tmp, int H, int W, int y, int c, const Taps &t)
{
    float a = 0.0f;
    for (int k = -t.radius; k <= t.radius; ++k) {
        const int yy = y + k;
        if (yy >= 0 && yy < H) a = fmaf(t.g[k + t.radius], tmp[(size_t)yy * W + c], a);
    }
    return a;
}

__global__ void admm_cols_kernel(const float *__restrict__ tmp, float *__restrict__ out, int H, int W, Taps t)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (c < W) out[(size_t)y * W + c] = column_pass(tmp, H, W, y, c, t);
}

// normalised taps exp(-k^2 / 2 sigma^2), |k| <= ceil(3 sigma) (A-ADMM-2); computed in double, rounded once
bool make_taps(float sigma_psf, Taps &t)
{
    t.radius = (int)ceil(3.0 * (double)sigma_psf);
    if (t.radius > ADMM_MAX_RADIUS) return false;
    double g[2 * ADMM_MAX_RADIUS + 1], sum = 0.0;
    const double s = (double)sigma_psf;
    for (int k = -t.radius; k <= t.radius; ++k) { g[k + t.radius] = s > 0.0 ? exp(-(double)k * k / (2.0 * s * s)) : 1.0; sum += g[k + t.radius]; }
    for (int k = 0; k <= 2 * t.radius; ++k) t.g[k] = (float)(g[k] / sum);
    return true;
}

// block-wide sum of `v` in a fixed order, written to part[linear block index]
__device__ __forceinline__ void block_partial(double v, double *part)
{
    __shared__ double sh[32];
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < (int)(blockDim.x + 31) / 32; ++k) s += sh[k];
        part[blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
}

// column pass of A^T * w, then the x update
__global__ void admm_x_update_kernel(AdmmState S, Taps t)
{
    if (*S.stopped) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    double d2 = 0.0;
    if (c < S.W) {
        const size_t i = (size_t)y * S.W + c;
        const float Aw = column_pass(S.tmp, S.H, S.W, y, c, t);
        const float xo = S.x[i];
        const float g = -Aw + S.rho2 * (xo - S.z[i]) + S.Y2[i];
        const float xn = xo - g * S.inv2gamma;
        S.x[i] = xn;
        const float d = xn - xo;
        d2 = (double)d * (double)d;
    }
    block_partial(d2, S.part_dx);
}

// column pass of A * x, then the argument of the projection
__global__ void admm_residual_kernel(AdmmState S, Taps t)
{
    if (*S.stopped) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (c >= S.W) return;
    const size_t i = (size_t)y * S.W + c;
    const float Ax = column_pass(S.tmp, S.H, S.W, y, c, t);
    S.Ax[i] = Ax;
    S.X[i] = S.I[i] - Ax + S.Y1[i] / S.rho1;
}

// z, duals, eps <- eps', next w, residual norm
__global__ void admm_dual_kernel(AdmmState S)
{
    if (*S.stopped) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    double r2 = 0.0;
    if (c < S.W) {
        const size_t i = (size_t)y * S.W + c;
        const float x = S.x[i], e = S.eps_next[i];
        float Y2 = S.Y2[i];
        const float z = (S.rho2 * x + Y2) / (S.lambda + S.rho2);
        const float r1 = S.I[i] - S.Ax[i] - e;
        const float Y1 = S.Y1[i] + S.alpha1 * r1;
        Y2 += S.alpha2 * (x - z);
        S.z[i] = z;
        S.Y1[i] = Y1;
        S.Y2[i] = Y2;
        S.eps[i] = e;
        S.w[i] = S.rho1 * r1 + Y1;
        r2 = (double)r1 * (double)r1;
    }
    block_partial(r2, S.part_res);
}

__global__ void admm_decide_kernel(AdmmState S)
{
    if (*S.stopped) return;
    __shared__ double sh[2][256];
    double a = 0.0, b = 0.0;
    for (int k = threadIdx.x; k < S.blocks; k += 256) { a += S.part_dx[k]; b += S.part_res[k]; }
    sh[0][threadIdx.x] = a;
    sh[1][threadIdx.x] = b;
    __syncthreads();
    for (int m = 128; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) { sh[0][threadIdx.x] += sh[0][threadIdx.x + m]; sh[1][threadIdx.x] += sh[1][threadIdx.x + m]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double dx = sqrt(sh[0][0]), res = sqrt(sh[1][0]);
        const int r = *S.iters;
        if (S.hist) { S.hist[2 * r] = (float)dx; S.hist[2 * r + 1] = (float)res; }
        *S.iters = r + 1;
        if (!(dx > (double)S.delta || res > (double)S.delta)) *S.stopped = 1;
    }
}

__global__ void admm_init_kernel(AdmmState S)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (c >= S.W) return;
    const size_t i = (size_t)y * S.W + c;
    S.x[i] = S.Ax[i] = S.eps[i] = S.z[i] = S.Y1[i] = S.Y2[i] = 0.0f;      // A-ADMM-5
    S.w[i] = S.rho1 * S.I[i];
}

smre_status fail(smre_status s, const char *text) { set_last_error(text); return s; }

}  // namespace
}  // namespace smre

using namespace smre;

extern "C" smre_status smre_admm(smre_handle h, int H, int W, const float *I_dev, const smre_admm_params *p,
                                 float *x_out_dev, float *eps_out_dev, int *iters_out, float *hist_out_dev,
                                 void *cuda_stream)
{
    if (!h || !I_dev || !p || !x_out_dev || H <= 0 || W <= 0) return fail(SMRE_EINVAL, "smre_admm: null pointer or non-positive size");
    if (!(p->rho1 > 0.0f) || !(p->rho2 > 0.0f) || !(p->gamma > 0.0f) || p->lambda < 0.0f || p->sigma_psf < 0.0f ||
        p->max_iter <= 0 || p->n_sweeps <= 0 || !(p->delta >= 0.0f))
        return fail(SMRE_EINVAL, "smre_admm: rho1, rho2, gamma > 0, lambda, sigma_psf, delta >= 0, max_iter, n_sweeps >= 1");
    int hH = 0, hW = 0, hB = 0, hvariant = 0;
    if (smre_shape(h, &hH, &hW, &hB, &hvariant) != SMRE_OK) return SMRE_EINVAL;
    if (hH != H || hW != W || hB != 1) return fail(SMRE_EINVAL, "smre_admm: H, W must be the handle's and its batch must be 1");
    Taps t;
    if (!make_taps(p->sigma_psf, t)) return fail(SMRE_EUNSUPPORTED, "smre_admm: sigma_psf beyond the compiled limit (radius 32)");
    // The call is synchronous, so it runs on a stream of its own behind the work already queued on the caller's
    // stream: that stream can be captured (the caller's may be the legacy default stream, which cannot), and with the
    // incomplete variant one iteration is eleven small launches whose launch cost exceeds their run time.
    cudaStream_t user_st = (cudaStream_t)cuda_stream, st = nullptr;
    cudaEvent_t ev = nullptr;
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventRecord(ev, user_st) != cudaSuccess || cudaStreamWaitEvent(st, ev, 0) != cudaSuccess) {
        if (ev) cudaEventDestroy(ev);
        if (st) cudaStreamDestroy(st);
        return fail(SMRE_ECUDA, "smre_admm: could not create its stream");
    }
    const size_t N = (size_t)H * W;
    const dim3 block(128), grid((W + 127) / 128, H);
    const int blocks = (int)(grid.x * grid.y);
    const int check_every = p->check_every > 0 ? p->check_every : 8;

    // workspace of this call: 10 images, the partial sums, the two counters
    float *ws = nullptr;
    double *parts = nullptr;
    int *flags = nullptr, *flags_host = nullptr;
    cudaError_t e = cudaMalloc(&ws, 10 * N * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&parts, 2 * (size_t)blocks * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&flags, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMallocHost(&flags_host, 2 * sizeof(int));
    smre_status rc = SMRE_OK;
    if (e != cudaSuccess) { rc = fail(e == cudaErrorMemoryAllocation ? SMRE_ENOMEM : SMRE_ECUDA, cudaGetErrorString(e)); }
    if (rc == SMRE_OK) {
        AdmmState S;
        S.I = I_dev;
        S.x = ws; S.Ax = ws + N; S.eps = ws + 2 * N; S.eps_next = ws + 3 * N; S.z = ws + 4 * N; S.Y1 = ws + 5 * N;
        S.Y2 = ws + 6 * N; S.w = ws + 7 * N; S.tmp = ws + 8 * N; S.X = ws + 9 * N;
        S.part_dx = parts; S.part_res = parts + blocks;
        S.hist = hist_out_dev; S.iters = flags; S.stopped = flags + 1;
        S.H = H; S.W = W; S.blocks = blocks;
        S.rho1 = p->rho1; S.rho2 = p->rho2; S.alpha1 = p->alpha1; S.alpha2 = p->alpha2; S.lambda = p->lambda;
        S.inv2gamma = 1.0f / (2.0f * p->gamma); S.delta = p->delta;
        e = cudaMemsetAsync(flags, 0, 2 * sizeof(int), st);
        if (e == cudaSuccess) { admm_init_kernel<<<grid, block, 0, st>>>(S); e = cudaGetLastError(); }
        auto iteration = [&]() -> smre_status {
            admm_rows_kernel<<<grid, block, 0, st>>>(S.w, S.tmp, H, W, t, S.stopped);
            admm_x_update_kernel<<<grid, block, 0, st>>>(S, t);
            admm_rows_kernel<<<grid, block, 0, st>>>(S.x, S.tmp, H, W, t, S.stopped);
            admm_residual_kernel<<<grid, block, 0, st>>>(S, t);
            const smre_status r = smre_project(h, S.X, S.eps_next, p->n_sweeps, (void *)st);
            admm_dual_kernel<<<grid, block, 0, st>>>(S);
            admm_decide_kernel<<<1, 256, 0, st>>>(S);
            return r;
        };
        // incomplete variant: one iteration as a CUDA graph (plain launches only; the standard variant's projection is
        // one cooperative launch that dwarfs the rest, it stays as it is)
        cudaGraphExec_t exec = nullptr;
        if (e == cudaSuccess && hvariant == (int)SMRE_INCOMPLETE && cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const smre_status r = iteration();
            cudaGraph_t g = nullptr;
            const cudaError_t ce = cudaStreamEndCapture(st, &g);
            if (r != SMRE_OK || ce != cudaSuccess || !g || cudaGraphInstantiate(&exec, g, 0) != cudaSuccess) exec = nullptr;
            if (g) cudaGraphDestroy(g);
            cudaGetLastError();
        }
        int done = 0;
        while (e == cudaSuccess && rc == SMRE_OK && done < p->max_iter) {
            const int n = p->max_iter - done < check_every ? p->max_iter - done : check_every;
            for (int k = 0; k < n && rc == SMRE_OK; ++k) {
                if (exec) { if (cudaGraphLaunch(exec, st) != cudaSuccess) rc = fail(SMRE_ECUDA, "smre_admm: graph launch failed"); }
                else rc = iteration();
            }
            done += n;
            if (rc != SMRE_OK) break;
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaMemcpyAsync(flags_host, flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e == cudaSuccess && flags_host[1]) break;
        }
        if (e == cudaSuccess && rc == SMRE_OK) {
            e = cudaMemcpyAsync(flags_host, flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(x_out_dev, S.x, N * sizeof(float), cudaMemcpyDeviceToDevice, st);
            if (e == cudaSuccess && eps_out_dev) e = cudaMemcpyAsync(eps_out_dev, S.eps, N * sizeof(float), cudaMemcpyDeviceToDevice, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e == cudaSuccess && iters_out) *iters_out = flags_host[0];
        }
        if (e != cudaSuccess && rc == SMRE_OK) rc = fail(SMRE_ECUDA, cudaGetErrorString(e));
        if (exec) cudaGraphExecDestroy(exec);
    }
    cudaStreamSynchronize(st);
    if (ws) cudaFree(ws);
    if (parts) cudaFree(parts);
    if (flags) cudaFree(flags);
    if (flags_host) cudaFreeHost(flags_host);
    cudaEventDestroy(ev);
    cudaStreamDestroy(st);
    return rc;
}

// A * x alone (the PSF operator of the ADMM), for callers and tests: rows into tmp_dev, columns into out_dev
extern "C" smre_status smre_psf_apply(int H, int W, float sigma_psf, const float *in_dev, float *tmp_dev, float *out_dev,
                                      void *cuda_stream)
{
    if (!in_dev || !tmp_dev || !out_dev || H <= 0 || W <= 0 || !(sigma_psf >= 0.0f))
        return fail(SMRE_EINVAL, "smre_psf_apply: null pointer, non-positive size or negative sigma");
    Taps t;
    if (!make_taps(sigma_psf, t)) return fail(SMRE_EUNSUPPORTED, "smre_psf_apply: sigma_psf beyond the compiled limit (radius 32)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const dim3 block(128), grid((W + 127) / 128, H);
    admm_rows_kernel<<<grid, block, 0, st>>>(in_dev, tmp_dev, H, W, t, nullptr);
    admm_cols_kernel<<<grid, block, 0, st>>>(tmp_dev, out_dev, H, W, t);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SMRE_OK : fail(SMRE_ECUDA, cudaGetErrorString(e));
}
