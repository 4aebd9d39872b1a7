// smre_project_noalloc: the standard-variant projection for callers that must not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  No handle, no cudaMalloc / cudaFree / graph
// instantiation: the scratch of the per-family kernel (family_pass_kernel, smre_family.cu) -- one fp32 increment
// plane q_f per family (Alg. 2; storage PAPER.md:258) -- lives in ONE file-scope device array of
// SMRE_NOALLOC_MAX_BYTES that every GPU which loads the library holds until exit.  x_out itself is the work image.
//
// The array is shared by every call and keeps the last call's contents: each call zeroes the part it uses first
// (q_{0,s} = 0), and calls that overlap on the GPU (different streams, different threads) race -- serialise them.
#include "../../include/smre.h"
#include "smre_common.cuh"

#include <cmath>
#include <cstdio>
#include <mutex>

namespace smre {

// In HOST code this name is only a stand-in for the symbol, not a device address: its address is looked up per
// device with cudaGetSymbolAddress below and that pointer is what the kernels get.
static __device__ __align__(256) float g_noalloc_scratch[SMRE_NOALLOC_MAX_BYTES / sizeof(float)];

constexpr int kMaxDevices = 64;
static float *g_scratch_ptr[kMaxDevices] = {};      // device address of the array on each device, once looked up
static std::mutex g_scratch_mutex;

// Device address of the scratch array on the CURRENT device (looked up once per device, with that device current).
static cudaError_t scratch_on_current_device(float **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        float *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

}  // namespace smre

using namespace smre;

static smre_status na_fail(smre_status st, const char *fmt, long long a = 0, long long b = 0)
{
    char buf[400];
    snprintf(buf, sizeof buf, fmt, a, b);
    set_last_error(buf);
    return st;
}

extern "C" smre_status smre_project_noalloc(int H, int W, const int *sides, int n_sides, const float *c_table,
                                            const float *y_dev, float *x_out_dev, int n_sweeps, void *cuda_stream)
{
    if (!sides || !c_table || !y_dev || !x_out_dev) return na_fail(SMRE_EINVAL, "smre_project_noalloc: NULL argument");
    if (H <= 0 || W <= 0 || n_sides <= 0 || n_sweeps <= 0)
        return na_fail(SMRE_EINVAL, "smre_project_noalloc: H, W, n_sides, n_sweeps must be positive");
    long long F = 0;
    for (int a = 0; a < n_sides; ++a) {
        if (sides[a] < 1 || sides[a] > H || sides[a] > W)
            return na_fail(SMRE_EINVAL, "smre_project_noalloc: side %lld outside [1, min(H,W)]", sides[a]);
        if (sides[a] > SMRE_MAX_SIDE)
            return na_fail(SMRE_EUNSUPPORTED, "smre_project_noalloc: side %lld exceeds SMRE_MAX_SIDE = %lld", sides[a], SMRE_MAX_SIDE);
        if (!(c_table[a] >= 1.17549435e-38f) || !std::isfinite(c_table[a]))
            return na_fail(SMRE_EINVAL, "smre_project_noalloc: threshold of side %lld must be a normal positive float", sides[a]);
        for (int b = 0; b < a; ++b)
            if (sides[b] == sides[a]) return na_fail(SMRE_EINVAL, "smre_project_noalloc: duplicate side %lld", sides[a]);
        F += (long long)sides[a] * sides[a];
    }
    const int Wq = (W + 3) & ~3;                                  // row pitch of the planes, as in smre_create
    const long long plane = (long long)H * Wq;
    const long long need = F * plane * (long long)sizeof(float);
    if (need > (long long)SMRE_NOALLOC_MAX_BYTES)
        return na_fail(SMRE_EUNSUPPORTED, "smre_project_noalloc: the increment planes need %lld bytes, the static scratch "
                                          "holds SMRE_NOALLOC_MAX_BYTES = %lld; use smre_create / smre_project",
                       need, (long long)SMRE_NOALLOC_MAX_BYTES);
    float *q = nullptr;
    cudaError_t e = scratch_on_current_device(&q);
    if (e != cudaSuccess) return na_fail(SMRE_ECUDA, cudaGetErrorString(e));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // x <- y (row a1), q <- 0: the array keeps the last call's contents
    if (x_out_dev != y_dev) {
        e = cudaMemcpyAsync(x_out_dev, y_dev, (size_t)H * W * sizeof(float), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return na_fail(SMRE_ECUDA, cudaGetErrorString(e));
    }
    e = cudaMemsetAsync(q, 0, (size_t)need, st);
    if (e != cudaSuccess) return na_fail(SMRE_ECUDA, cudaGetErrorString(e));
    // the canonical family order of smre_create (A3), one kernel per family, n_sweeps sweeps
    for (int sweep = 0; sweep < n_sweeps; ++sweep) {
        long long f = 0;
        for (int a = 0; a < n_sides; ++a)
            for (int oy = 0; oy < sides[a]; ++oy)
                for (int ox = 0; ox < sides[a]; ++ox, ++f) {
                    const Family fam{sides[a], oy, ox, (H - oy) / sides[a], (W - ox) / sides[a], c_table[a],
                                     sqrtf(c_table[a])};
                    e = launch_family_pass(x_out_dev, q + f * plane, 1, H, W, Wq, fam, st);
                    if (e != cudaSuccess) return na_fail(SMRE_ECUDA, cudaGetErrorString(e));
                }
    }
    return SMRE_OK;
}
