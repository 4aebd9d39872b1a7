// Interface of the persistent sweep scheduler (smre_persistent.cu).
#pragma once
#include "smre_common.cuh"
#include <vector>

namespace smre {

struct PersistentPlan;   // tile decomposition + device workspace; opaque to the API layer

// Returns nullptr if the image cannot be tiled on chip (then only the graph schedule exists).
// q: [F][B][H][W] increment planes, xwork: [B][H][W]; both stay owned by the caller.
PersistentPlan *persistent_plan_create(int H, int W, int B, const std::vector<Family> &fams,
                                       float *q, float *xwork);
void persistent_plan_destroy(PersistentPlan *p);
void persistent_plan_tiles(const PersistentPlan *p, int *tiles_y, int *tiles_x);
// 0 = healthy, 1 = a mailbox poll timed out in some launch (protocol failure), -1 = cannot read.  Synchronises.
int persistent_plan_status(const PersistentPlan *p);

// Whole projection: x <- y, q <- 0, n_sweeps ordered sweeps, x_out <- x.  Asynchronous on st.
cudaError_t persistent_run(PersistentPlan *p, const float *y, float *x_out, int n_sweeps,
                           cudaStream_t st, long long *launches);

}  // namespace smre
