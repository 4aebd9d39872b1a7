// Geometry and interface of the "strips" sweep scheduler (kernel and launch in smre_strips.cu).
// See DESIGN.md sec. 6.2.  Everything here is closed form: no tables, nothing depends on n_sweeps.
//
// A frame is cut into NS horizontal strips of nominal height T, one persistent CTA per strip; the strip keeps its
// rows of x in shared memory for the whole call.  At a family step (s, oy, ox) (windows of one family
// are disjoint) strip boundary j sits on the window-row grid of that family: it is the smallest grid line
//        b_j(s, oy) = oy + s*k  >=  j*T - T/2          (b_0 = 0, b_NS = H, clipped to H),
// so every window row ("band" of s image rows) lies inside exactly one strip and a boundary never leaves the
// s rows [j*T - T/2, j*T - T/2 + s).  While ox runs through 0..s-1 (a "macro step" = the s families (s, oy, *))
// the boundaries rest and strips do not interact at all; between macro steps each boundary moves by at most
// s - 1 rows, up or down, and the rows that change owner go to a strip at most ST_HOPS away.
// Along x the bands of a strip are cut into chunks of floor(32/s) windows, one warp each, lane = column.
#pragma once
#include "smre_common.cuh"

namespace smre {

constexpr int ST_MAX_SIDE = 8;                            // largest window side the strip kernel is compiled for
constexpr int ST_MAX_SIDES = 8;                           // entries of sides[]
constexpr int ST_HOPS = 3;                                // a row that changes owner moves at most this many strips
constexpr int ST_RING = 4;                                // mailbox ring depth (transitions)
constexpr int ST_MAX_WARPS = 30;                          // compute warps per CTA (+ the waiter and the issuer warp)
constexpr int ST_NSTG = 32;                               // q stages (mbarriers) in flight at most

// rows of x a strip keeps in shared memory: it only ever holds image rows in [j*T - T/2, j*T - T/2 + T + s - 1)
__host__ __device__ __forceinline__ int st_tile_rows(int T) { return T + ST_MAX_SIDE; }

// Row at which strip j begins while the families (s, oy, *) run.
__host__ __device__ __forceinline__ int st_boundary(int j, int NS, int H, int T, int s, int oy)
{
    if (j <= 0) return 0;
    if (j >= NS) return H;
    const int d = j * T - T / 2 - oy;
    const int b = oy + (d > 0 ? ((d + s - 1) / s) * s : 0);
    return b < H ? b : H;
}

// Active rows [lo, hi) of strip j in family (s, oy, *): whole window rows only (reading A6: windows fully inside).
__host__ __device__ __forceinline__ void st_active_rows(int j, int NS, int H, int T, int s, int oy, int &lo, int &hi)
{
    lo = st_boundary(j, NS, H, T, s, oy);
    if (lo < oy) lo = oy;
    hi = st_boundary(j + 1, NS, H, T, s, oy);
    const int ae = oy + ((H - oy) / s) * s;
    if (hi > ae) hi = ae;
    if (hi < lo) hi = lo;
}

__host__ __device__ __forceinline__ int st_chunk_width(int s) { return (32 / s) * s; }

struct StripPlan;      // host object: workspace + launch parameters

struct StripSummary {
    int T, strips, warps, max_rows, max_hop, ring_rows, frames_per_launch;
    long long workspace_bytes;
};

// Host-only feasibility check (no device needed when sm_count / smem_optin are given).
bool strips_summary(int H, int W, int B, const int *sides, int n_sides, int sm_count, int smem_optin,
                    StripSummary *out, char *why, size_t why_len);

// nullptr (reason in why) if the configuration is outside what the strip kernel supports.
StripPlan *strips_plan_create(int H, int W, int B, int Wq, const int *sides, const float *c, int n_sides, float *q,
                              char *why, size_t why_len);
void strips_plan_destroy(StripPlan *p);
void strips_plan_shape(const StripPlan *p, int *strips, int *warps);
// Health of the LAST finished run: 0 ok, > 0 a wait timed out (result invalid).  Reads a pinned host word the
// kernel's epilogue writes: no synchronisation; meaningful once the stream has drained.
int strips_plan_status(const StripPlan *p);
cudaError_t strips_run(StripPlan *p, const float *y, float *x_out, int n_sweeps, cudaStream_t st, long long *launches);
// Same under Alg. 2's stop rule: a frame stops after the first sweep r with ||x_r - x_{r-1}||^2 <= delta,
// at most n_sweeps sweeps; sweeps_done (device, [B] ints, may be null) receives r per frame.  The decision is taken
// on the device (one grid barrier per sweep among the strips of a frame); nothing returns to the host.
cudaError_t strips_run_tol(StripPlan *p, const float *y, float *x_out, int n_sweeps, bool tol_mode, float delta,
                           int *sweeps_done, cudaStream_t st, long long *launches);

}  // namespace smre
