// Threshold calibration (sec. 2.1, lines 89-113): the weights c_s(alpha) that balance
// the multi-scale test.  For a noise image eps
//     t_s = sum_{i in s} eps_i^2,  (t_s)^(1/4) ~ N(mu_s = (|s| - 0.5)^(1/4), sigma_s^2 = 1 / (8 sqrt|s|)),
//     Q_Omega = max_{s in Omega} ((t_s)^(1/4) - mu_s) / sigma_s
// over every square window of every side in sides[] at every shift (|s| = side^2), and
//     c_s(alpha) = 1 / (q_alpha sigma_s + mu_s)^4,   q_alpha = the alpha quantile of Q_Omega
// from n simulated noise images, which the caller supplies.  The library returns THRESHOLDS c_S = 1 / c_s(alpha).
//
//   q_stat_kernel    one CTA = one 32 x 32 block of window origins of one frame, all sides in one pass: the sums of
//                    side s grow out of those of side s - 1,
//                        t_s(y,x) = t_{s-1}(y,x) + C_{s-1}(y, x+s-1) + R_s(y+s-1, x),
//                    with running column sums C and row sums R kept in shared memory (only positive terms are ever
//                    added: no cancellation, unlike a summed-area table); frame maximum by an ordered-int atomicMax
//                    (a maximum does not depend on the order: bit-identical from run to run).
//   quantile_kernel  rank selection of the order statistic ceil(alpha n) among the n frame values, then the table.
#include "../../include/smre.h"
#include "smre_common.cuh"

#include <cmath>
#include <cstdint>
#include <cstdio>

namespace smre {

constexpr int CAL_TB = 32;                         // block of window origins per CTA (CAL_TB x CAL_TB)
constexpr int CAL_MAX_SIDE = SMRE_MAX_SIDE;        // 32
constexpr int CAL_TW = CAL_TB + CAL_MAX_SIDE - 1;  // 63: pixels a block of origins can reach
constexpr int CAL_TP = CAL_TW + 1;                 // pitch

struct CalSides {
    unsigned mask_lo;                              // bit (s - 1): side s is in sides[]
    float mu[CAL_MAX_SIDE + 1], inv_sigma[CAL_MAX_SIDE + 1], sigma[CAL_MAX_SIDE + 1];
};
struct CalList { int n; int side[CAL_MAX_SIDE]; };  // sides[] in the caller's order

// order-preserving map float -> unsigned, so that atomicMax on the image finds the float maximum
__device__ __forceinline__ unsigned ordered_bits(float f)
{
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __host__ __forceinline__ float ordered_float(unsigned o)
{
    const unsigned u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
#ifdef __CUDA_ARCH__
    return __uint_as_float(u);
#else
    float f; memcpy(&f, &u, 4); return f;
#endif
}

__global__ void __launch_bounds__(CAL_TB * CAL_TB)
q_stat_kernel(const float *eps, int H, int W, int smax, CalSides cs, unsigned *q_bits /* [frames], ordered bits */)
{
    __shared__ float v[CAL_TW * CAL_TP];           // squared pixels of the block's reach (0 outside the image)
    __shared__ float R[CAL_TW * CAL_TP];           // R_s(y,x) = sum_{k<s} v[y][x+k]
    __shared__ float C[CAL_TW * CAL_TP];           // C_s(y,x) = sum_{k<s} v[y+k][x]
    __shared__ float wmax[CAL_TB];
    const int tx = threadIdx.x & (CAL_TB - 1), ty = threadIdx.x / CAL_TB;
    const int x0 = blockIdx.x * CAL_TB, y0 = blockIdx.y * CAL_TB;
    const float *img = eps + (size_t)blockIdx.z * H * W;
    const int reach = CAL_TB + smax - 1;
    for (int i = threadIdx.x; i < reach * reach; i += CAL_TB * CAL_TB) {
        const int yy = i / reach, xx = i - yy * reach;
        const int gy = y0 + yy, gx = x0 + xx;
        const float e = (gy < H && gx < W) ? img[(size_t)gy * W + gx] : 0.0f;
        v[yy * CAL_TP + xx] = e * e;
        R[yy * CAL_TP + xx] = 0.0f;
        C[yy * CAL_TP + xx] = 0.0f;
    }
    __syncthreads();
    float t = 0.0f, best = -INFINITY;
    const int gy = y0 + ty, gx = x0 + tx;
    for (int s = 1; s <= smax; ++s) {
        // C_{s-1} is what the arrays hold now; t needs C_{s-1}(y, x+s-1) and the NEW R_s(y+s-1, x)
        const float c_prev = C[ty * CAL_TP + tx + s - 1];
        __syncthreads();
        for (int i = threadIdx.x; i < reach * reach; i += CAL_TB * CAL_TB) {
            const int yy = i / reach, xx = i - yy * reach;
            if (xx + s - 1 < reach) R[yy * CAL_TP + xx] += v[yy * CAL_TP + xx + s - 1];
            if (yy + s - 1 < reach) C[yy * CAL_TP + xx] += v[(yy + s - 1) * CAL_TP + xx];
        }
        __syncthreads();
        t += c_prev + R[(ty + s - 1) * CAL_TP + tx];
        if (((cs.mask_lo >> (s - 1)) & 1u) && gy + s <= H && gx + s <= W) {
            const float z = (sqrtf(sqrtf(t)) - cs.mu[s]) * cs.inv_sigma[s];
            best = fmaxf(best, z);
        }
    }
    for (int o = 16; o > 0; o >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, o));
    if (tx == 0) wmax[ty] = best;
    __syncthreads();
    if (threadIdx.x < CAL_TB) {
        float b = wmax[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) b = fmaxf(b, __shfl_xor_sync(0xffffffffu, b, o));
        if (threadIdx.x == 0 && b > -INFINITY) atomicMax(q_bits + blockIdx.z, ordered_bits(b));
    }
}

// q_bits -> floats in place, the order statistic of rank k (1-based) -> q_alpha, then the thresholds
__global__ void quantile_kernel(unsigned *q_bits, int n, int k, CalSides cs, CalList list, float *q_alpha_out,
                                float *c_out)
{
    float *q = reinterpret_cast<float *>(q_bits);
    for (int i = threadIdx.x; i < n; i += blockDim.x) q[i] = ordered_float(q_bits[i]);
    __syncthreads();
    __shared__ float qa;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const float mine = q[i];
        int less = 0, equal_before = 0;
        for (int j = 0; j < n; ++j) {
            const float o = q[j];
            less += o < mine;
            equal_before += (o == mine) && (j < i);
        }
        if (less + equal_before == k - 1) qa = mine;            // exactly one i has rank k
    }
    __syncthreads();
    if (threadIdx.x == 0 && q_alpha_out) *q_alpha_out = qa;
    if ((int)threadIdx.x < list.n) {
        const int s = list.side[threadIdx.x];
        const float base = fmaf(qa, cs.sigma[s], cs.mu[s]);
        c_out[threadIdx.x] = (base * base) * (base * base);
    }
}

}  // namespace smre

using namespace smre;

static smre_status cal_fail(smre_status st, const char *msg)
{
    set_last_error(msg);
    return st;
}

extern "C" smre_status smre_calibrate(int H, int W, int n_frames, const int *sides, int n_sides,
                                      const float *noise_dev, float alpha, float *q_stat_dev, float *q_alpha_dev,
                                      float *c_table_dev, void *cuda_stream)
{
    if (!sides || !noise_dev || !q_stat_dev || !c_table_dev)
        return cal_fail(SMRE_EINVAL, "smre_calibrate: NULL argument");
    if (H <= 0 || W <= 0 || n_frames <= 0 || n_sides <= 0 || n_sides > CAL_MAX_SIDE)
        return cal_fail(SMRE_EINVAL, "smre_calibrate: H, W, n_frames, n_sides must be positive (n_sides <= 32)");
    if (!(alpha > 0.0f) || !(alpha <= 1.0f)) return cal_fail(SMRE_EINVAL, "smre_calibrate: alpha must be in (0, 1]");
    if (n_frames > 65535) return cal_fail(SMRE_EUNSUPPORTED, "smre_calibrate: at most 65535 frames per call");
    CalSides cs{};
    CalList list{};
    list.n = n_sides;
    int smax = 0;
    for (int a = 0; a < n_sides; ++a) {
        const int s = sides[a];
        if (s < 1 || s > H || s > W) return cal_fail(SMRE_EINVAL, "smre_calibrate: side outside [1, min(H, W)]");
        if (s > CAL_MAX_SIDE) return cal_fail(SMRE_EUNSUPPORTED, "smre_calibrate: side exceeds SMRE_MAX_SIDE");
        if ((cs.mask_lo >> (s - 1)) & 1u) return cal_fail(SMRE_EINVAL, "smre_calibrate: duplicate side");
        cs.mask_lo |= 1u << (s - 1);
        const double n = (double)s * s;
        cs.mu[s] = (float)pow(n - 0.5, 0.25);                        // mu_s
        cs.inv_sigma[s] = (float)sqrt(8.0 * sqrt(n));                // 1 / sigma_s
        cs.sigma[s] = (float)sqrt(1.0 / (8.0 * sqrt(n)));
        list.side[a] = s;
        if (s > smax) smax = s;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemsetAsync(q_stat_dev, 0, (size_t)n_frames * sizeof(float), st);   // ordered bits 0 < any float
    if (e != cudaSuccess) return cal_fail(SMRE_ECUDA, cudaGetErrorString(e));
    dim3 grid((unsigned)((W + CAL_TB - 1) / CAL_TB), (unsigned)((H + CAL_TB - 1) / CAL_TB), (unsigned)n_frames);
    q_stat_kernel<<<grid, CAL_TB * CAL_TB, 0, st>>>(noise_dev, H, W, smax, cs, reinterpret_cast<unsigned *>(q_stat_dev));
    int k = (int)ceil((double)alpha * n_frames);
    k = k < 1 ? 1 : k > n_frames ? n_frames : k;
    quantile_kernel<<<1, 1024, 0, st>>>(reinterpret_cast<unsigned *>(q_stat_dev), n_frames, k, cs, list, q_alpha_dev,
                                        c_table_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cal_fail(SMRE_ECUDA, cudaGetErrorString(e));
    return SMRE_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// Second-order SOFI cumulant at zero time lag (Eq. 19):
//     C_2(r, 0) = <F^2(r, t)>_t - <F(r, t)>_t^2     per pixel over the n frames of a stack (e.g. the projected frames).
// HBM-bound: every frame is read once, coalesced (thread = 4 consecutive pixels, float4), the frame loop is unrolled
// for loads in flight.  The two moments are accumulated around the FIRST frame's value of the pixel (a shift leaves
// a cumulant of order >= 2 unchanged, and it removes the cancellation of <F^2> - <F>^2 on a bright background).
namespace smre {

__global__ void __launch_bounds__(256)
cumulant2_kernel(const float *__restrict__ stack, int n, long long N, float *__restrict__ c2)
{
    const long long i4 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i4 >= N) return;
    const float inv_n = 1.0f / (float)n;
    if (i4 + 4 <= N && (N & 3) == 0) {
        const float4 ref = *reinterpret_cast<const float4 *>(stack + i4);
        float4 s1 = make_float4(0.f, 0.f, 0.f, 0.f), s2 = s1;
#pragma unroll 4
        for (int t = 1; t < n; ++t) {
            const float4 v = __ldcs(reinterpret_cast<const float4 *>(stack + (long long)t * N + i4));
            const float dx = v.x - ref.x, dy = v.y - ref.y, dz = v.z - ref.z, dw = v.w - ref.w;
            s1.x += dx; s1.y += dy; s1.z += dz; s1.w += dw;
            s2.x = fmaf(dx, dx, s2.x); s2.y = fmaf(dy, dy, s2.y); s2.z = fmaf(dz, dz, s2.z); s2.w = fmaf(dw, dw, s2.w);
        }
        float4 o;
        o.x = fmaf(-(s1.x * inv_n), s1.x * inv_n, s2.x * inv_n);
        o.y = fmaf(-(s1.y * inv_n), s1.y * inv_n, s2.y * inv_n);
        o.z = fmaf(-(s1.z * inv_n), s1.z * inv_n, s2.z * inv_n);
        o.w = fmaf(-(s1.w * inv_n), s1.w * inv_n, s2.w * inv_n);
        *reinterpret_cast<float4 *>(c2 + i4) = o;
    } else {
        for (long long i = i4; i < min(i4 + 4, N); ++i) {
            const float ref = stack[i];
            float s1 = 0.f, s2 = 0.f;
            for (int t = 1; t < n; ++t) {
                const float d = stack[(long long)t * N + i] - ref;
                s1 += d;
                s2 = fmaf(d, d, s2);
            }
            c2[i] = fmaf(-(s1 * inv_n), s1 * inv_n, s2 * inv_n);
        }
    }
}

}  // namespace smre

extern "C" smre_status smre_cumulant2(int H, int W, int n_frames, const float *stack_dev, float *c2_out_dev,
                                      void *cuda_stream)
{
    if (!stack_dev || !c2_out_dev) return cal_fail(SMRE_EINVAL, "smre_cumulant2: NULL argument");
    if (H <= 0 || W <= 0 || n_frames <= 0) return cal_fail(SMRE_EINVAL, "smre_cumulant2: H, W, n_frames must be positive");
    if (((uintptr_t)stack_dev & 15) || ((uintptr_t)c2_out_dev & 15))
        return cal_fail(SMRE_EINVAL, "smre_cumulant2: pointers must be 16-byte aligned");
    const long long N = (long long)H * W;
    const long long threads = (N + 3) / 4;
    cumulant2_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(stack_dev, n_frames, N,
                                                                                           c2_out_dev);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cal_fail(SMRE_ECUDA, cudaGetErrorString(e));
    return SMRE_OK;
}
