// Interface of the conveyor sweep scheduler (host planner in smre_conveyor_plan.cu, kernel and launch in
// smre_conveyor.cu).  See DESIGN.md sec. 6.2 for the idea:
// tile boundaries MOVE so that at every family step they lie on that family's window grid; no
// window ever straddles a tile boundary, pixels change owner in one direction only (to the left /
// upper neighbour), and the neighbour latency is off the critical path.
#pragma once
#include "smre_common.cuh"
#include <vector>

namespace smre {

constexpr int CV_NCW = 16;              // compute warps per CTA
constexpr int CV_NST_T = (CV_NCW + 3) * 32;  // threads that take part in the step barrier: + one control, one sender, one receiver warp
constexpr int CV_NT = CV_NST_T + 32;        // + the planner warp, which runs ahead of the steps and never joins their barrier
constexpr int CV_PW = 64;               // edge of the torus-addressed x tile in shared memory
constexpr int CV_SD = 16;               // strip depth: a boundary moves < CV_SD pixels per step
constexpr int CV_D = 16;                // mailbox ring depth (steps)
constexpr int CV_PF = 7;                // q prefetch distance (steps)
constexpr int CV_NST = CV_PF + 1;       // q stages in shared memory
constexpr int CV_TR = 128;              // table ring entries in shared memory (steps)
constexpr int CV_DR = 64;               // step descriptor ring (steps)
constexpr int CV_BATCH = 16;            // the planner warp plans this many steps at once, one per lane
constexpr int CV_AHEAD = 16;            // ... starting this many steps ahead of the step that releases the batch
constexpr int CV_MBW = 2 * CV_SD * CV_PW;   // 8-byte words per mailbox slot
constexpr int CV_PROG_STRIDE = 64;       // progress counters 256 bytes apart: no line is shared by two CTAs
constexpr int CV_MAX_F = 1024;          // families kept in shared memory

// One axis of one tile slot at one step (16 bytes).  All positions are clipped to [0, N].
struct AxisEntry {
    short L, R;        // the tile owns pixels [L, R) along this axis at this step (empty if L == R)
    short A;           // pixels [A, R) were not held after the previous step: they ARRIVE
    short D;           // pixels [L, D) are not held at the next step: they DEPART after this step
    short w0, nw;      // windows of this step's family with origin in [L, R): first origin, count
    short e0, e1;      // y axis: blocks of cv_kr(side) window rows, rows of the window box (nw * side)
                       // x axis: first 4-aligned column c0 of the q box, 16-byte chunks per row of it
};

// Vertically stacked windows handled by one lane of the conveyor kernel, per window edge (the kernel's
// template instantiations and the planner's e0 must agree on this).
__host__ __device__ constexpr int cv_kr(int side) { return side == 1 ? 5 : side == 2 ? 3 : side <= 5 ? 2 : 1; }
static_assert(sizeof(AxisEntry) == 16, "AxisEntry must be 16 bytes");

// Tile-boundary trajectories of one axis for `total` steps.
struct AxisPlan {
    int N = 0;                         // image extent along the axis
    int T = 0;                         // nominal tile extent (0: one static tile)
    int slots = 0;                     // tile slots (CTAs) along the axis
    int max_extent = 0;                // largest R - L
    int max_move = 0;                  // largest boundary movement in one step (inside the image)
    long long drift = 0;               // total anchor movement
    int reach = 0;                     // largest slot distance from the reader of a q value to its writer one sweep earlier
    std::vector<AxisEntry> tab;        // [total][slots]
};

// (side, offset) of every step along one axis; total = n_sweeps * F steps, family order repeating.
// Returns false if no tiling with <= max_slots slots satisfies the kernel's invariants.
bool plan_axis(int N, const std::vector<Family> &fams, bool y_axis, int n_sweeps, int T,
               AxisPlan &out, char *why, size_t why_len);

// Checks the hand-off invariants of a pair of axis plans (partition, adjacency, strip depth,
// torus injectivity).  Pure host code; used by plan creation and by the CPU tests.
bool verify_axis(const AxisPlan &ap, char *why, size_t why_len);

struct ConveyorPlan;

// nullptr if the configuration is outside what the conveyor supports (then the graph schedule runs).
ConveyorPlan *conveyor_plan_create(int H, int W, int B, const std::vector<Family> &fams, float *q,
                                   float *xwork);
void conveyor_plan_destroy(ConveyorPlan *p);
void conveyor_plan_tiles(const ConveyorPlan *p, int *tiles_y, int *tiles_x);
int conveyor_plan_status(const ConveyorPlan *p);     // 0 healthy, 1 a poll timed out, -1 unreadable
cudaError_t conveyor_run(ConveyorPlan *p, const float *y, float *x_out, int n_sweeps,
                         cudaStream_t st, long long *launches);

// Host-only planning summary for tests / diagnostics (no device needed).
struct ConveyorSummary {
    int tiles_y, tiles_x, T_y, T_x, max_h, max_w, max_move_y, max_move_x, reach_y, reach_x;
    long long drift_y, drift_x, table_bytes;
};
bool conveyor_summary(int H, int W, const std::vector<Family> &fams, int n_sweeps, int max_ctas,
                      ConveyorSummary *out, char *why, size_t why_len);

}  // namespace smre
