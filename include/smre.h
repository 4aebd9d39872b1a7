/*
 * smre.h -- C ABI of the B200-native Dykstra projection onto multi-scale window balls
 * (the hot path of arXiv 1503.03492, "Parallel Statistical Multi-resolution Estimation").
 *
 * What it computes.  Given a residual image y (the argument X of P_G in Eq. 12-13,
 * PAPER.md:159-164) the library runs Dykstra's algorithm (Alg. 2) with the
 * closed-form ball projection of Eq. 14 onto the sets
 *        tau_S = { x : sum_{i in S} x_i^2 <= c_S }          (Eq. 5)
 * for square windows S.  c_S here is a THRESHOLD: c_S = 1 / c_s(alpha) of the paper.
 *
 *   SMRE_STANDARD   -- the paper's "exact method" (Sec. 3.1; window set of
 *                      Fig. 5): every square window of every side in sides[], at
 *                      every shift, fully inside the image.  Windows sharing (side, oy, ox) are
 *                      disjoint (one "family") and are projected in parallel;
 *                      families run in the fixed order sides[] as given, then oy ascending, then
 *                      ox ascending.  One sweep = one pass over all sum(side^2) families.  One
 *                      fp32 increment plane q_f per family lives in device memory.
 *   SMRE_INCOMPLETE -- the paper's "incomplete Dykstra" (Sec. 3.2, Listing
 *                      2/3): K = floor(log2(max side)); for shift i = 0..K ascending, a Dykstra
 *                      run from q = 0 over the nested tilings of side 2^K, ..., 2^i (coarse to
 *                      fine) whose origin is (2^i mod side) on the diagonal; n_sweeps inner cycles
 *                      per shift.  Increments never leave the chip.
 *
 * All arithmetic is fp32.  Sums, products and differences are IEEE round-to-nearest; the
 * scale factor sqrt(c_S / sum) is evaluated as sqrtf(c_S) * rsqrt.approx.ftz(sum) (MUFU.RSQ, <= 2 ulp; build with
 * -DSMRE_PRECISE_SCALE for sqrt_rn(div_rn())), which is why thresholds must be normal floats (>= FLT_MIN).  The
 * comparison is strict (project iff sum > c_S, Eq. 14).  Images are dense row-major
 * [batch][H][W] fp32, idx = (b*H + row)*W + col, frames independent.
 *
 * Threading / streams.  Every call returns a status; nothing is thrown across the ABI.
 * smre_project only ENQUEUES work on the caller's CUDA stream: no host synchronisation, no host
 * round-trip between families.  One in-flight smre_project per handle.  Each call starts from
 * q = 0 (Alg. 2: q_{0,s} = 0); no state carries between calls.
 *
 * There is no CPU path: without a CUDA device smre_create fails with SMRE_ECUDA.
 */
#ifndef SMRE_H
#define SMRE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct smre_handle_s *smre_handle;

typedef enum {
    SMRE_OK = 0,
    SMRE_EINVAL = 1,        /* null pointer, non-positive size, side < 1 or > min(H,W), duplicate side,
                               non-positive threshold, missing power-of-two level for SMRE_INCOMPLETE */
    SMRE_EUNSUPPORTED = 2,  /* side beyond the compiled limit (SMRE_MAX_SIDE), unknown schedule */
    SMRE_ENOMEM = 3,        /* device allocation of the increment planes / workspace failed */
    SMRE_ECUDA = 4          /* any other CUDA runtime error (text in smre_last_error) */
} smre_status;

typedef enum { SMRE_STANDARD = 0, SMRE_INCOMPLETE = 1 } smre_variant;

/* How the ordered family sequence of SMRE_STANDARD is driven (the "sweep scheduler"). */
typedef enum {
    SMRE_SCHED_AUTO = 0,        /* persistent if the image tiles fit on chip, else graph */
    SMRE_SCHED_GRAPH = 1,       /* one kernel per family, one captured CUDA graph per sweep */
    SMRE_SCHED_PERSISTENT = 2,  /* "conveyor": one cooperative kernel per call; x tiles resident in
                                   shared memory, tile boundaries that follow each family's window
                                   grid, one-directional hand-off between CTAs, q streamed from HBM */
    SMRE_SCHED_STRIPS = 3       /* one cooperative kernel per call; one CTA per strip of 8 rows */
} smre_schedule;

#define SMRE_MAX_SIDE 32        /* largest window side (the paper's L_SMRE = 32) */

/*
 * Create a solver for [batch][H][W] images.
 *   out      (host, out)  receives the handle; owned by the caller until smre_destroy.
 *   sides    (host, in)   n_sides distinct window sides, 1 <= side <= min(H, W, SMRE_MAX_SIDE);
 *                         their order is the family order of SMRE_STANDARD.
 *   c_table  (host, in)   n_sides thresholds c_S > 0, c_table[a] belongs to sides[a].
 *   variant               SMRE_INCOMPLETE needs every 2^k, k <= floor(log2(max side)), in sides[];
 *                         other sides are ignored by it.
 * Allocates (device): SMRE_STANDARD  sum(side^2)*batch*H*Wq*4 bytes of increment planes (Wq = W rounded up
 * to a multiple of 4) plus a batch*H*W*4 work image and, if the conveyor can tile the problem, its mailboxes
 * (256 KiB per tile) and boundary tables; SMRE_INCOMPLETE nothing of image size.
 * The arrays sides / c_table are copied; the caller may free them on return.
 */
smre_status smre_create(smre_handle *out, int H, int W, int batch,
                        const int *sides, int n_sides, const float *c_table,
                        smre_variant variant);

/*
 * Project.  y_dev, x_out_dev: DEVICE pointers to batch*H*W contiguous fp32.  y_dev is only read;
 * x_out_dev == y_dev (in place) is allowed (the paper's kernels work in place on e,
 * PAPER.md:516).  n_sweeps >= 1: sweeps (standard) / inner cycles per shift (incomplete).
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Asynchronous, with one exception: the first
 * call of a handle with a given n_sweeps under the conveyor schedule plans the tile boundaries on the host
 * and uploads the tables (a few ms, cached per n_sweeps), which synchronises with the stream once.
 */
smre_status smre_project(smre_handle h, const float *y_dev, float *x_out_dev,
                         int n_sweeps, void *cuda_stream);

/*
 * Same projection with HOST buffers (pageable or pinned): copies y to the device, projects,
 * copies the result back, all on cuda_stream, and returns after the stream has drained.
 * The staging buffers belong to the handle.
 */
smre_status smre_project_host(smre_handle h, const float *y_host, float *x_out_host,
                              int n_sweeps, void *cuda_stream);

/*
 * Projection under the paper's own stopping rules instead of a fixed count (the paper "runs Dykstra until
 * convergence", tol 1e-3: PAPER.md:571, 752).  The decision is taken on the device; nothing returns to the host.
 *   SMRE_STANDARD   Alg. 2: stop after the first sweep r with ||x_r - x_{r-1}||_2^2 <= tol (tol is
 *                   Alg. 2's delta; x_0 = y), at most max_sweeps sweeps, each frame on its own.  The squared norm is
 *                   accumulated in fp32 per thread and in fp64 above (fixed order: the same input stops on the same
 *                   sweep every time).  Runs on the strip scheduler; SMRE_EUNSUPPORTED where that does not take the
 *                   problem.  sweeps_done_dev: DEVICE int[batch] or NULL, receives r per frame.
 *   SMRE_INCOMPLETE Listing 3: within each shift every L x L tile (L = 2^K) iterates until the
 *                   sum over its pixels and the cycle's levels of |x_old - x_new| is <= tol * L^2 (fp32), at most
 *                   max_sweeps cycles.  sweeps_done_dev: DEVICE int[1] or NULL, receives the largest cycle count of
 *                   any tile; smre_export_tile_cycles gives all of them.
 * tol >= 0.  Everything else as smre_project.
 */
smre_status smre_project_tol(smre_handle h, const float *y_dev, float *x_out_dev, int max_sweeps, float tol,
                             int *sweeps_done_dev, void *cuda_stream);

/* SMRE_INCOMPLETE: the cycles every tile ran in shift `shift` (0..K) of the last smre_project_tol, copied to
 * cycles_out_dev (DEVICE, [batch][tiles_y][tiles_x] ints, may be NULL to query the sizes only).  Tiles of a shift start
 * at (2^shift mod L) - L on both axes, those entirely above / left of the image left out. */
smre_status smre_export_tile_cycles(smre_handle h, int shift, int *cycles_out_dev, int *tiles_y, int *tiles_x,
                                    void *cuda_stream);

/* Frees every device and host resource of the handle.  NULL is accepted. */
smre_status smre_destroy(smre_handle h);

/* ---- diagnostics and test hooks (not on the hot path) -------------------------------------- */

/* Select the sweep scheduler of SMRE_STANDARD (default SMRE_SCHED_AUTO).  SMRE_EUNSUPPORTED if
 * the persistent schedule cannot hold this image on chip. */
smre_status smre_set_schedule(smre_handle h, smre_schedule schedule);

/* n_families: families per sweep (standard) / level passes per inner cycle summed over shifts
 * (incomplete).  windows_per_sweep: windows visited per sweep / per inner cycle, all frames.
 * increment_bytes: device bytes held for q.  Any pointer may be NULL. */
smre_status smre_info(smre_handle h, int *n_families, long long *windows_per_sweep,
                      long long *increment_bytes);

/* Family idx in execution order: side, row offset oy, column offset ox, threshold.  For
 * SMRE_INCOMPLETE idx runs over the level passes (shift-major), oy == ox. */
smre_status smre_family(smre_handle h, int idx, int *side, int *oy, int *ox, float *c);

/* SMRE_STANDARD only: copy the increment planes of the last smre_project to q_out_dev,
 * layout [F][batch][H][W] fp32 (device pointer).  Asynchronous on cuda_stream. */
smre_status smre_export_increments(smre_handle h, float *q_out_dev, void *cuda_stream);

/* Scheduler actually used by the last smre_project (smre_schedule value), number of kernels it
 * launched, and the persistent schedule's tile grid (0 x 0 if unused).  Pointers may be NULL.
 * After a persistent run this call SYNCHRONISES with the device to read the scheduler's health flag
 * and returns SMRE_ECUDA if a neighbour hand-off timed out (the result is then invalid). */
smre_status smre_last_launch(smre_handle h, int *schedule_used, long long *kernel_launches,
                             int *tiles_y, int *tiles_x);

/* Host-only planning check of the conveyor schedule (no device needed, nothing allocated): plans
 * the moving tile boundaries for n_sweeps sweeps of the standard variant over sides[] on an H x W
 * image with at most max_ctas tiles, verifies every hand-off invariant of the plan, and reports the
 * tile grid, the largest tile and the size of the boundary tables.  SMRE_EUNSUPPORTED (with the
 * reason in smre_last_error) if the conveyor cannot tile the problem.  Out pointers may be NULL. */
smre_status smre_plan_check(int H, int W, const int *sides, int n_sides, int n_sweeps, int max_ctas,
                            int *tiles_y, int *tiles_x, int *max_tile_h, int *max_tile_w,
                            long long *table_bytes);

/* ---- a projection that allocates nothing ------------------------------------------------------ */

/* Size of the file-scope device array that serves as the scratch of smre_project_noalloc: every GPU that loads
 * the library holds this much device memory until the process exits. */
#define SMRE_NOALLOC_MAX_BYTES (16 * 1024 * 1024)

/*
 * SMRE_STANDARD projection of ONE H x W image (Alg. 2; Eq. 14) for callers that
 * cannot allocate: no handle, and no cudaMalloc, cudaFree or any other allocating routine is called.  Same
 * arguments, family order and arithmetic as smre_create(..., SMRE_STANDARD) + smre_project under
 * SMRE_SCHED_GRAPH (bit-identical results); one kernel launch per family and sweep, enqueued on cuda_stream,
 * asynchronous.  y_dev / x_out_dev: DEVICE pointers to H*W fp32 (x_out_dev == y_dev allowed); sides / c_table:
 * HOST arrays.  The increment planes, sum(side^2) * H * Wq * 4 bytes (Wq = W rounded up to a multiple of 4), live
 * in a static device array of SMRE_NOALLOC_MAX_BYTES on the CURRENT device: a larger problem is refused with
 * SMRE_EUNSUPPORTED (64 x 64 with sides 1-4 needs 480 KiB; 256 x 256 with sides 1-4 7.5 MiB).
 * The array is shared by all calls and keeps the last call's contents; each call zeroes what it uses first.
 * Calls that overlap on the GPU (other streams, other threads) RACE on it: serialise them.
 */
smre_status smre_project_noalloc(int H, int W, const int *sides, int n_sides, const float *c_table,
                                 const float *y_dev, float *x_out_dev, int n_sweeps, void *cuda_stream);

/* ---- threshold calibration (sec. 2.1) ---------------------------------------------------- */

/*
 * The thresholds that balance the multi-scale test, from simulated noise.  noise_dev: DEVICE,
 * n_frames images [n_frames][H][W] of unit-variance noise drawn by the caller (the library draws no random numbers).
 * For every frame the extreme-value statistic
 *     Q = max over every window s of every side in sides[], at every shift, fully inside the image, of
 *         ((t_s)^(1/4) - mu_s) / sigma_s,   t_s = sum of squares over s,   mu_s = (|s| - 0.5)^(1/4),
 *         sigma_s^2 = 1 / (8 sqrt|s|),   |s| = side^2
 * is written to q_stat_dev (DEVICE, n_frames floats); q_alpha = the order statistic of rank ceil(alpha * n_frames)
 * (alpha as passed, a float, the product in double; clamped to [1, n_frames]) of
 * those values goes to q_alpha_dev (DEVICE, 1 float, may be NULL), and the THRESHOLD of every side,
 *     c_S = 1 / c_s(alpha) = (q_alpha sigma_s + mu_s)^4
 * to c_table_dev (DEVICE, n_sides floats, order of sides[]): the table smre_create takes.  sides: HOST, distinct,
 * 1 <= side <= min(H, W, SMRE_MAX_SIDE).  0 < alpha <= 1.  fp32; the window sums add positive terms only.
 * Asynchronous on cuda_stream; allocates nothing.
 */
smre_status smre_calibrate(int H, int W, int n_frames, const int *sides, int n_sides, const float *noise_dev,
                           float alpha, float *q_stat_dev, float *q_alpha_dev, float *c_table_dev, void *cuda_stream);

/*
 * Second-order SOFI cumulant at zero time lag (Eq. 19): C_2 = <F^2>_t - <F>_t^2 per pixel over the
 * n_frames frames of stack_dev (DEVICE, [n_frames][H][W] fp32, 16-byte aligned), e.g. the projected frames of a
 * batched smre_project; both means divide by n_frames.  c2_out_dev: DEVICE, H*W fp32, 16-byte aligned.
 * Asynchronous on cuda_stream; allocates nothing.
 */
smre_status smre_cumulant2(int H, int W, int n_frames, const float *stack_dev, float *c2_out_dev, void *cuda_stream);

/* Shape and variant the handle was created for (any pointer may be NULL). */
smre_status smre_shape(smre_handle h, int *H, int *W, int *batch, int *variant);

/* ---- The ADMM around the projection (Alg. 1, Eq. 9-13) -----------------
 * Solves Eq. 10,  min G(eps) + (lambda/2) ||z||^2  s.t.  I = A * x + eps,  z = x,  with G the multi-resolution
 * constraint of the handle (its sides and thresholds) and A a Gaussian PSF of standard deviation sigma_psf
 * (taps exp(-t^2 / 2 sigma^2), |t| <= ceil(3 sigma) <= 32, normalised, zero outside the image; 0 = identity).
 * One iteration, in Alg. 1's order (the readings A-ADMM-1..9 of DESIGN.md state what the paper leaves open):
 *     x   <- x - grad_x L / (2 gamma),  grad_x L = -A^T * (rho1 (I - A * x - eps) + Y1) + rho2 (x - z) + Y2   (Eq. 11)
 *     eps <- P_G(I - A * x + Y1 / rho1)          (Eq. 12: smre_project on `h`, n_sweeps sweeps / cycles from q = 0)
 *     z   <- (rho2 x + Y2) / (lambda + rho2)
 *     Y1  += alpha1 (I - A * x - eps),  Y2 += alpha2 (x - z)
 * from x = z = eps = Y = 0, until ||x_r - x_{r-1}||_2 <= delta and ||I - A * x_r - eps_r||_2 <= delta, at most
 * max_iter iterations.  All arithmetic is fp32 on the device (the two norms are summed in fp64 in a fixed order, so
 * a run is repeatable bit for bit); the host only enqueues and reads the stop flag every `check_every` iterations
 * (<= 0: 8); kernels enqueued behind the stop do nothing, so the result is that of the iteration that stopped.
 * App. B of the paper: rho1 = 6.192, rho2 = 1.8, alpha1 = 1.2, alpha2 = 0.12, lambda = 1, delta = 1e-3; gamma is
 * not given there: the x step is stable for 2 gamma >= rho1 + rho2.
 *   h             handle with batch 1 and the shape H x W (either variant; its schedule is used as set)
 *   I_dev         [H][W] device, read only;  x_out_dev [H][W] device: the estimate x;  eps_out_dev: the residual, or NULL
 *   iters_out     HOST int, or NULL: iterations done
 *   hist_out_dev  device [2 * max_iter] or NULL: the two norms after every iteration
 * Synchronous: it runs behind the work already queued on cuda_stream, on a stream of its own, and returns when it
 * has finished (with the incomplete variant one iteration is replayed as a CUDA graph).  Allocates and frees its
 * workspace (10 images) per call.
 * Errors: SMRE_EINVAL (pointers, shape mismatch, batch != 1, parameters out of range), SMRE_EUNSUPPORTED
 * (sigma_psf > 10.6), SMRE_ENOMEM, SMRE_ECUDA, and whatever smre_project returns. */
typedef struct {
    float sigma_psf;
    float rho1, rho2, alpha1, alpha2, lambda, gamma;
    float delta;
    int max_iter;
    int n_sweeps;
    int check_every;
} smre_admm_params;
smre_status smre_admm(smre_handle h, int H, int W, const float *I_dev, const smre_admm_params *p, float *x_out_dev,
                      float *eps_out_dev, int *iters_out, float *hist_out_dev, void *cuda_stream);

/* out = A * in with the PSF operator of smre_admm (rows into tmp_dev, columns into out_dev; all [H][W] device,
 * in_dev may not alias the others).  Asynchronous on cuda_stream. */
smre_status smre_psf_apply(int H, int W, float sigma_psf, const float *in_dev, float *tmp_dev, float *out_dev,
                           void *cuda_stream);

/* Text of the last error on the calling thread ("" if none).  Never NULL. */
const char *smre_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SMRE_H */
