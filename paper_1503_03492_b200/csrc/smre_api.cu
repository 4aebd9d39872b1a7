// C ABI of include/smre.h: handle, argument validation, family enumeration and the two sweep
// schedulers' host side.  Every step of the path runs in the kernels of smre_family.cu,
// smre_conveyor.cu and smre_icd.cu; there is no CPU path.
#include "../../include/smre.h"
#include "smre_common.cuh"
#include "smre_conveyor.cuh"
#include "smre_strips.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

using namespace smre;

static thread_local char g_err[512] = "";

static smre_status fail(smre_status st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}

static smre_status cuda_fail(cudaError_t e, const char *what)
{
    smre_status st = (e == cudaErrorMemoryAllocation) ? SMRE_ENOMEM : SMRE_ECUDA;
    return fail(st, "%s: %s", what, cudaGetErrorString(e));
}

#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);        \
    } while (0)

struct smre_handle_s {
    int H = 0, W = 0, B = 0;
    int Wq = 0;                        // row pitch of the q planes: W rounded up to a multiple of 4
    smre_variant variant = SMRE_STANDARD;
    std::vector<int> sides;
    std::vector<float> c;
    std::vector<Family> fams;          // standard: execution order; incomplete: level passes
    std::vector<int> pass_shift;       // incomplete: shift index of each level pass
    long long windows_per_sweep = 0;
    // standard
    float *q = nullptr;                // [F][B][H][Wq]
    float *xwork = nullptr;            // [B][H][W]
    size_t q_bytes = 0;
    smre_schedule schedule = SMRE_SCHED_AUTO;
    cudaGraphExec_t sweep_graph = nullptr;
    ConveyorPlan *plan = nullptr;      // null if the conveyor cannot tile this problem
    StripPlan *strips = nullptr;       // null if the strip kernel does not take this problem
    char strips_why[200] = "";         // ... and why
    // incomplete
    int K = 0;
    IcdLevels levels{};
    int *tile_cycles = nullptr;        // cycles every tile ran in the last smre_project_tol, shift-major
    std::vector<size_t> tile_off;      // offset of shift i in tile_cycles; [K + 1] = total
    // host staging for smre_project_host
    float *stage_in = nullptr, *stage_out = nullptr;
    // last launch
    int last_schedule = 0;
    long long last_launches = 0;
};

extern "C" const char *smre_last_error(void) { return g_err; }

namespace smre {
void set_last_error(const char *text) { snprintf(g_err, sizeof g_err, "%s", text ? text : ""); }
}

static smre_status build_sweep_graph(smre_handle h)
{
    cudaStream_t cs;
    CU(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    const size_t plane = (size_t)h->B * h->H * h->Wq;
    for (size_t f = 0; e == cudaSuccess && f < h->fams.size(); ++f)
        e = launch_family_pass(h->xwork, h->q + f * plane, h->B, h->H, h->W, h->Wq, h->fams[f], cs);
    cudaError_t e2 = cudaStreamEndCapture(cs, &g);
    if (e == cudaSuccess) e = e2;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&h->sweep_graph, g, 0);
    if (g) cudaGraphDestroy(g);
    cudaStreamDestroy(cs);
    if (e != cudaSuccess) return cuda_fail(e, "capturing the per-sweep family graph");
    return SMRE_OK;
}

extern "C" smre_status smre_create(smre_handle *out, int H, int W, int batch, const int *sides,
                                   int n_sides, const float *c_table, smre_variant variant)
{
    g_err[0] = 0;
    if (!out) return fail(SMRE_EINVAL, "out is NULL");
    *out = nullptr;
    if (!sides || !c_table) return fail(SMRE_EINVAL, "sides / c_table is NULL");
    if (H <= 0 || W <= 0 || batch <= 0 || n_sides <= 0)
        return fail(SMRE_EINVAL, "H, W, batch, n_sides must be positive");
    if (variant != SMRE_STANDARD && variant != SMRE_INCOMPLETE)
        return fail(SMRE_EINVAL, "unknown variant %d", (int)variant);
    int smax = 0;
    for (int a = 0; a < n_sides; ++a) {
        if (sides[a] < 1 || sides[a] > H || sides[a] > W)
            return fail(SMRE_EINVAL, "side %d outside [1, min(H,W)]", sides[a]);
        if (!(c_table[a] >= 1.17549435e-38f) || !std::isfinite(c_table[a]))     // FLT_MIN: rsqrt.approx.ftz
            return fail(SMRE_EINVAL, "threshold of side %d must be a normal positive float", sides[a]);
        for (int b = 0; b < a; ++b)
            if (sides[b] == sides[a]) return fail(SMRE_EINVAL, "duplicate side %d", sides[a]);
        if (sides[a] > smax) smax = sides[a];
    }
    if (smax > SMRE_MAX_SIDE)
        return fail(SMRE_EUNSUPPORTED, "side %d exceeds SMRE_MAX_SIDE = %d", smax, SMRE_MAX_SIDE);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(SMRE_ECUDA, "no CUDA device: this library has no CPU path");
    }

    smre_handle h = new (std::nothrow) smre_handle_s;
    if (!h) return fail(SMRE_ENOMEM, "host allocation failed");
    h->H = H; h->W = W; h->Wq = (W + 3) & ~3; h->B = batch; h->variant = variant;
    h->sides.assign(sides, sides + n_sides);
    h->c.assign(c_table, c_table + n_sides);

    if (variant == SMRE_STANDARD) {
        // canonical family order: sides[] as given, oy ascending, ox ascending (A3)
        for (int a = 0; a < n_sides; ++a)
            for (int oy = 0; oy < sides[a]; ++oy)
                for (int ox = 0; ox < sides[a]; ++ox) {
                    Family f{sides[a], oy, ox, (H - oy) / sides[a], (W - ox) / sides[a],
                             c_table[a], sqrtf(c_table[a])};
                    h->fams.push_back(f);
                    h->windows_per_sweep += (long long)f.ny * f.nx * batch;
                }
        const size_t plane = (size_t)batch * H * W * sizeof(float);
        h->q_bytes = (size_t)batch * H * h->Wq * sizeof(float) * h->fams.size();
        cudaError_t e = cudaMalloc(&h->q, h->q_bytes);
        if (e == cudaSuccess) e = cudaMalloc(&h->xwork, plane);
        if (e != cudaSuccess) { smre_status s = cuda_fail(e, "allocating increment planes"); smre_destroy(h); return s; }
        smre_status s = build_sweep_graph(h);
        if (s != SMRE_OK) { smre_destroy(h); return s; }
        // pixels outside every window of a family are never written: their increments stay 0 for the life of the handle
        e = cudaMemset(h->q, 0, h->q_bytes);
        if (e != cudaSuccess) { smre_status s2 = cuda_fail(e, "zeroing increment planes"); smre_destroy(h); return s2; }
        h->plan = conveyor_plan_create(H, W, batch, h->fams, h->q, h->xwork);     // may be null
        h->strips = strips_plan_create(H, W, batch, h->Wq, sides, c_table, n_sides, h->q, h->strips_why,
                                       sizeof h->strips_why);                                              // may be null
    } else {
        int K = 0;
        while ((2 << K) <= smax) ++K;
        h->K = K;
        for (int k = 0; k <= K; ++k) {
            int a = 0;
            while (a < n_sides && sides[a] != (1 << k)) ++a;
            if (a == n_sides) {
                delete h;
                return fail(SMRE_EINVAL, "SMRE_INCOMPLETE needs side %d (every 2^k up to %d) in sides[]",
                            1 << k, 1 << K);
            }
            h->levels.c[k] = c_table[a];
            h->levels.sqrt_c[k] = sqrtf(c_table[a]);
        }
        h->tile_off.assign(K + 2, 0);
        for (int i = 0; i <= K; ++i)
            h->tile_off[i + 1] = h->tile_off[i] + (size_t)batch * icd_tiles_along(H, K, i) * icd_tiles_along(W, K, i);
        if (cudaMalloc(&h->tile_cycles, h->tile_off[K + 1] * sizeof(int)) != cudaSuccess ||
            cudaMemset(h->tile_cycles, 0, h->tile_off[K + 1] * sizeof(int)) != cudaSuccess) {
            cudaGetLastError();
            smre_destroy(h);
            return fail(SMRE_ENOMEM, "allocating the per-tile cycle counters failed");
        }
        for (int i = 0; i <= K; ++i)
            for (int k = K; k >= i; --k) {
                const int side = 1 << k, o = (1 << i) % side;
                Family f{side, o, o, (H - o) / side, (W - o) / side, h->levels.c[k], h->levels.sqrt_c[k]};
                h->fams.push_back(f);
                h->pass_shift.push_back(i);
                h->windows_per_sweep += (long long)f.ny * f.nx * batch;
            }
    }
    *out = h;
    return SMRE_OK;
}

extern "C" smre_status smre_destroy(smre_handle h)
{
    if (!h) return SMRE_OK;
    if (h->plan) conveyor_plan_destroy(h->plan);
    if (h->strips) strips_plan_destroy(h->strips);
    if (h->sweep_graph) cudaGraphExecDestroy(h->sweep_graph);
    if (h->q) cudaFree(h->q);
    if (h->xwork) cudaFree(h->xwork);
    if (h->tile_cycles) cudaFree(h->tile_cycles);
    if (h->stage_in) cudaFree(h->stage_in);
    if (h->stage_out) cudaFree(h->stage_out);
    delete h;
    return SMRE_OK;
}

extern "C" smre_status smre_set_schedule(smre_handle h, smre_schedule schedule)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (schedule != SMRE_SCHED_AUTO && schedule != SMRE_SCHED_GRAPH && schedule != SMRE_SCHED_PERSISTENT &&
        schedule != SMRE_SCHED_STRIPS)
        return fail(SMRE_EUNSUPPORTED, "unknown schedule %d", (int)schedule);
    if (schedule == SMRE_SCHED_STRIPS && (h->variant != SMRE_STANDARD || !h->strips))
        return fail(SMRE_EUNSUPPORTED, "strip schedule unavailable for this handle: %s", h->strips_why);
    if (schedule == SMRE_SCHED_PERSISTENT && (h->variant != SMRE_STANDARD || !h->plan))
        return fail(SMRE_EUNSUPPORTED, "persistent schedule unavailable for this handle "
                                       "(incomplete variant, or tiles do not fit on chip)");
    h->schedule = schedule;
    return SMRE_OK;
}

extern "C" smre_status smre_project(smre_handle h, const float *y_dev, float *x_out_dev,
                                    int n_sweeps, void *cuda_stream)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (!y_dev || !x_out_dev) return fail(SMRE_EINVAL, "y_dev / x_out_dev is NULL");
    if (n_sweeps <= 0) return fail(SMRE_EINVAL, "n_sweeps must be positive");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = (size_t)h->B * h->H * h->W * sizeof(float);
    h->last_launches = 0;

    if (h->variant == SMRE_INCOMPLETE) {
        // Listing 2: one kernel per shift i = 0..K, ascending (A-ICD-2/3)
        h->last_schedule = SMRE_SCHED_GRAPH;
        for (int i = 0; i <= h->K; ++i) {
            const float *src = (i == 0) ? y_dev : x_out_dev;
            CU(launch_icd_shift(src, x_out_dev, h->B, h->H, h->W, h->K, i, h->levels, n_sweeps, st));
            ++h->last_launches;
        }
        return SMRE_OK;
    }

    // A wait of the previous strip-scheduled run on this handle that timed out (the kernel's last CTA writes the
    // health word to pinned host memory; reading it costs nothing and needs no synchronisation)
    if (h->strips && h->last_schedule == SMRE_SCHED_STRIPS && strips_plan_status(h->strips) != 0)
        return fail(SMRE_ECUDA, "the previous smre_project on this handle failed: a wait of the strip scheduler timed "
                                "out (code 0x%x), its result is invalid", strips_plan_status(h->strips));
    // SMRE_SCHED_AUTO: the strips where they take the problem (no host planning, nothing depends on n_sweeps), else
    // the conveyor where it can tile it, else one kernel per family
    if (h->strips && (h->schedule == SMRE_SCHED_STRIPS || h->schedule == SMRE_SCHED_AUTO)) {
        // in place is safe: a CTA writes a row only after the row's first owner has read it
        cudaError_t e = strips_run(h->strips, y_dev, x_out_dev, n_sweeps, st, &h->last_launches);
        if (e == cudaSuccess) { h->last_schedule = SMRE_SCHED_STRIPS; return SMRE_OK; }
        if (h->schedule == SMRE_SCHED_STRIPS) return cuda_fail(e, "strips_run");
        cudaGetLastError();                        // SMRE_SCHED_AUTO: any failure to launch falls through
        h->last_launches = 0;
    }
    if (h->plan && (h->schedule == SMRE_SCHED_PERSISTENT || h->schedule == SMRE_SCHED_AUTO)) {
        cudaError_t e = conveyor_run(h->plan, y_dev, x_out_dev, n_sweeps, st, &h->last_launches);
        if (e == cudaSuccess) { h->last_schedule = SMRE_SCHED_PERSISTENT; return SMRE_OK; }
        if (h->schedule == SMRE_SCHED_PERSISTENT) {
            if (e != cudaErrorNotSupported) return cuda_fail(e, "conveyor_run");
            return fail(SMRE_EUNSUPPORTED, "the conveyor cannot tile %d sweeps of this problem", n_sweeps);
        }
        cudaGetLastError();
        h->last_launches = 0;
    }
    // graph schedule: x <- y, q <- 0 (Alg. 2: q_{0,s} = 0), then n_sweeps replays of the sweep graph
    h->last_schedule = SMRE_SCHED_GRAPH;
    CU(cudaMemcpyAsync(h->xwork, y_dev, bytes, cudaMemcpyDeviceToDevice, st));
    CU(cudaMemsetAsync(h->q, 0, h->q_bytes, st));
    for (int s = 0; s < n_sweeps; ++s) CU(cudaGraphLaunch(h->sweep_graph, st));
    CU(cudaMemcpyAsync(x_out_dev, h->xwork, bytes, cudaMemcpyDeviceToDevice, st));
    h->last_launches = (long long)n_sweeps * (long long)h->fams.size();
    return SMRE_OK;
}

// max over ints (the largest cycle count of any tile), one block
__global__ void max_int_kernel(const int *v, size_t n, int *out)
{
    __shared__ int sm[32];
    int m = 0;
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) m = max(m, v[i]);
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < (int)(blockDim.x >> 5); ++k) m = max(m, sm[k]);
        *out = m;
    }
}

extern "C" smre_status smre_project_tol(smre_handle h, const float *y_dev, float *x_out_dev, int max_sweeps, float tol,
                                        int *sweeps_done_dev, void *cuda_stream)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (!y_dev || !x_out_dev) return fail(SMRE_EINVAL, "y_dev / x_out_dev is NULL");
    if (max_sweeps <= 0) return fail(SMRE_EINVAL, "max_sweeps must be positive");
    if (!(tol >= 0.0f) || !std::isfinite(tol)) return fail(SMRE_EINVAL, "tol must be finite and >= 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_launches = 0;
    if (h->variant == SMRE_INCOMPLETE) {
        // Listing 2 + the while loop of Listing 3: per shift, every tile until its own stop
        h->last_schedule = SMRE_SCHED_GRAPH;
        for (int i = 0; i <= h->K; ++i) {
            const float *src = (i == 0) ? y_dev : x_out_dev;
            CU(launch_icd_shift_tol(src, x_out_dev, h->B, h->H, h->W, h->K, i, h->levels, max_sweeps, st, true, tol,
                                    h->tile_cycles + h->tile_off[i]));
            ++h->last_launches;
        }
        if (sweeps_done_dev) {
            max_int_kernel<<<1, 256, 0, st>>>(h->tile_cycles, h->tile_off[h->K + 1], sweeps_done_dev);
            CU(cudaGetLastError());
            ++h->last_launches;
        }
        return SMRE_OK;
    }
    if (!h->strips)
        return fail(SMRE_EUNSUPPORTED, "convergence control of the standard variant runs on the strip scheduler, which "
                                       "does not take this problem: %s", h->strips_why);
    if (h->last_schedule == SMRE_SCHED_STRIPS && strips_plan_status(h->strips) != 0)
        return fail(SMRE_ECUDA, "the previous projection on this handle failed: a wait of the strip scheduler timed out "
                                "(code 0x%x), its result is invalid", strips_plan_status(h->strips));
    cudaError_t e = strips_run_tol(h->strips, y_dev, x_out_dev, max_sweeps, true, tol, sweeps_done_dev, st, &h->last_launches);
    if (e == cudaErrorNotSupported) return fail(SMRE_EUNSUPPORTED, "the strip scheduler has no room for x_{r-1} at this width");
    if (e != cudaSuccess) return cuda_fail(e, "strips_run_tol");
    h->last_schedule = SMRE_SCHED_STRIPS;
    return SMRE_OK;
}

extern "C" smre_status smre_export_tile_cycles(smre_handle h, int shift, int *cycles_out_dev, int *tiles_y, int *tiles_x,
                                               void *cuda_stream)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (h->variant != SMRE_INCOMPLETE) return fail(SMRE_EUNSUPPORTED, "only the incomplete variant iterates tile by tile");
    if (shift < 0 || shift > h->K) return fail(SMRE_EINVAL, "shift %d outside [0, %d]", shift, h->K);
    if (tiles_y) *tiles_y = icd_tiles_along(h->H, h->K, shift);
    if (tiles_x) *tiles_x = icd_tiles_along(h->W, h->K, shift);
    if (cycles_out_dev)
        CU(cudaMemcpyAsync(cycles_out_dev, h->tile_cycles + h->tile_off[shift],
                           (h->tile_off[shift + 1] - h->tile_off[shift]) * sizeof(int), cudaMemcpyDeviceToDevice,
                           (cudaStream_t)cuda_stream));
    return SMRE_OK;
}

extern "C" smre_status smre_project_host(smre_handle h, const float *y_host, float *x_out_host,
                                         int n_sweeps, void *cuda_stream)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (!y_host || !x_out_host) return fail(SMRE_EINVAL, "y_host / x_out_host is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = (size_t)h->B * h->H * h->W * sizeof(float);
    if (!h->stage_in) {
        CU(cudaMalloc(&h->stage_in, bytes));
        CU(cudaMalloc(&h->stage_out, bytes));
    }
    CU(cudaMemcpyAsync(h->stage_in, y_host, bytes, cudaMemcpyHostToDevice, st));
    smre_status s = smre_project(h, h->stage_in, h->stage_out, n_sweeps, cuda_stream);
    if (s != SMRE_OK) return s;
    CU(cudaMemcpyAsync(x_out_host, h->stage_out, bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    // the stream has drained: a hand-off of a persistent scheduler that timed out must not pass as a result
    if (h->last_schedule == SMRE_SCHED_STRIPS && h->strips && strips_plan_status(h->strips) != 0)
        return fail(SMRE_ECUDA, "strip scheduler: a wait timed out, code 0x%x (result invalid)", strips_plan_status(h->strips));
    if (h->last_schedule == SMRE_SCHED_PERSISTENT && h->plan && conveyor_plan_status(h->plan) != 0)
        return fail(SMRE_ECUDA, "conveyor scheduler: a neighbour hand-off timed out (result invalid)");
    return SMRE_OK;
}

extern "C" smre_status smre_shape(smre_handle h, int *H, int *W, int *batch, int *variant)
{
    if (!h) { set_last_error("smre_shape: null handle"); return SMRE_EINVAL; }
    if (H) *H = h->H;
    if (W) *W = h->W;
    if (batch) *batch = h->B;
    if (variant) *variant = (int)h->variant;
    return SMRE_OK;
}

extern "C" smre_status smre_info(smre_handle h, int *n_families, long long *windows_per_sweep,
                                 long long *increment_bytes)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (n_families) *n_families = (int)h->fams.size();
    if (windows_per_sweep) *windows_per_sweep = h->windows_per_sweep;
    if (increment_bytes) *increment_bytes = (long long)h->fams.size() * h->B * h->H * h->W * 4 * (h->q ? 1 : 0);
    return SMRE_OK;
}

extern "C" smre_status smre_family(smre_handle h, int idx, int *side, int *oy, int *ox, float *c)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (idx < 0 || idx >= (int)h->fams.size()) return fail(SMRE_EINVAL, "family index %d out of range", idx);
    const Family &f = h->fams[idx];
    if (side) *side = f.side;
    if (oy) *oy = f.oy;
    if (ox) *ox = f.ox;
    if (c) *c = f.c;
    return SMRE_OK;
}

extern "C" smre_status smre_export_increments(smre_handle h, float *q_out_dev, void *cuda_stream)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (!q_out_dev) return fail(SMRE_EINVAL, "q_out_dev is NULL");
    if (h->variant != SMRE_STANDARD)
        return fail(SMRE_EUNSUPPORTED, "the incomplete variant keeps no increments in device memory");
    CU(cudaMemcpy2DAsync(q_out_dev, (size_t)h->W * 4, h->q, (size_t)h->Wq * 4, (size_t)h->W * 4,
                         h->fams.size() * (size_t)h->B * h->H, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return SMRE_OK;
}

extern "C" smre_status smre_plan_check(int H, int W, const int *sides, int n_sides, int n_sweeps,
                                       int max_ctas, int *tiles_y, int *tiles_x, int *max_tile_h,
                                       int *max_tile_w, long long *table_bytes)
{
    g_err[0] = 0;
    if (!sides || H <= 0 || W <= 0 || n_sides <= 0 || n_sweeps <= 0 || max_ctas <= 0)
        return fail(SMRE_EINVAL, "smre_plan_check: bad argument");
    std::vector<Family> fams;
    for (int a = 0; a < n_sides; ++a) {
        if (sides[a] < 1 || sides[a] > H || sides[a] > W || sides[a] > SMRE_MAX_SIDE)
            return fail(SMRE_EINVAL, "side %d outside [1, min(H, W, SMRE_MAX_SIDE)]", sides[a]);
        for (int oy = 0; oy < sides[a]; ++oy)
            for (int ox = 0; ox < sides[a]; ++ox)
                fams.push_back(Family{sides[a], oy, ox, (H - oy) / sides[a], (W - ox) / sides[a], 1.0f, 1.0f});
    }
    ConveyorSummary cs;
    char why[200] = "";
    if (!conveyor_summary(H, W, fams, n_sweeps, max_ctas, &cs, why, sizeof why))
        return fail(SMRE_EUNSUPPORTED, "conveyor: %s", why);
    if (tiles_y) *tiles_y = cs.tiles_y;
    if (tiles_x) *tiles_x = cs.tiles_x;
    if (max_tile_h) *max_tile_h = cs.max_h;
    if (max_tile_w) *max_tile_w = cs.max_w;
    if (table_bytes) *table_bytes = cs.table_bytes;
    return SMRE_OK;
}

extern "C" smre_status smre_last_launch(smre_handle h, int *schedule_used, long long *kernel_launches,
                                        int *tiles_y, int *tiles_x)
{
    if (!h) return fail(SMRE_EINVAL, "handle is NULL");
    if (schedule_used) *schedule_used = h->last_schedule;
    if (kernel_launches) *kernel_launches = h->last_launches;
    int ty = 0, tx = 0;
    if (h->plan && h->last_schedule == SMRE_SCHED_PERSISTENT) {
        conveyor_plan_tiles(h->plan, &ty, &tx);
        if (conveyor_plan_status(h->plan) != 0)
            return fail(SMRE_ECUDA, "conveyor scheduler: a neighbour hand-off timed out (result invalid)");
    }
    if (h->strips && h->last_schedule == SMRE_SCHED_STRIPS) {
        strips_plan_shape(h->strips, &ty, &tx);
        cudaDeviceSynchronize();
        if (strips_plan_status(h->strips) != 0)
            return fail(SMRE_ECUDA, "strip scheduler: a wait timed out, code 0x%x (result invalid)", strips_plan_status(h->strips));
    }
    if (tiles_y) *tiles_y = ty;
    if (tiles_x) *tiles_x = tx;
    return SMRE_OK;
}
