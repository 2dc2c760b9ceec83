/* caspar_ba.h — C ABI of the B200 (sm_100a) bundle-adjustment hot path.
 *
 * One Levenberg-Marquardt iteration on a reprojection-error problem, after the generated
 * bundle-adjustment solver of "Caspar" (arxiv 2605.30583; /root/reference/PAPER.md):
 *   - residual of the Snavely reprojection factor, PAPER.md:182-204 (section VI-A):
 *       P = R(w) X + t,  p = -P_xy / P_z,  r = 1 + k1 |p|^2 + k2 |p|^4,  residual = f r p - pixel;
 *   - Levenberg-Marquardt with quality-based damping (Madsen et al.), PAPER.md:163 (section V);
 *   - preconditioned conjugate gradients with a block-Jacobi preconditioner, one block per node,
 *     applied matrix-free from per-observation Jacobians, PAPER.md:163,167-169;
 *   - one device memory block with views.
 * BASELINE.json `north_star` fixes the variant built here: the linear system is the
 * point-eliminated (Schur-complement) one, S = U' - W V'^-1 W^T, cameras are 9-vectors
 * (angle-axis w, translation t, f, k1, k2) updated additively.  DESIGN.md lists every reading.
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary.  Every call returns CASPAR_BA_OK (0) or a negative
 *     CASPAR_BA_E* code; caspar_ba_last_error() gives the text of the last failure on a handle.
 *   - "DEVICE" pointers are CUDA device pointers on the current device ("DEVICE or HOST" pointers are
 *     read with cudaMemcpyDefault, so either works).  "HOST" pointers are ordinary host memory.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the default stream).  All work is
 *     enqueued on it.  Calls that return host scalars synchronise that stream once before returning.
 *   - The library owns ONE device arena allocated in caspar_ba_create and freed in caspar_ba_destroy.
 *     Parameter arrays are BORROWED for the handle's lifetime and written only by an accepted
 *     caspar_ba_lm_step (or caspar_ba_solve / caspar_ba_set_parameters_host).
 *   - There is no CPU fallback: every step runs in the library's sm_100a kernels.
 *   - Not thread-safe per handle; distinct handles are independent.
 *
 * Layouts: cameras [num_cameras][9] row-major float32 = w0 w1 w2 t0 t1 t2 f k1 k2;
 * points [num_points][3] float32; observations [N][2] float32 pixels; indices int32.
 */
#ifndef CASPAR_BA_H
#define CASPAR_BA_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CASPAR_BA_OK 0
#define CASPAR_BA_EINVAL (-1)   /* null / negative sizes, index out of range, unsupported shape          */
#define CASPAR_BA_ECUDA (-2)    /* a CUDA runtime call failed (text in caspar_ba_last_error)             */
#define CASPAR_BA_ENOMEM (-3)   /* host or device allocation failed                                      */
#define CASPAR_BA_ENUMERIC (-4) /* non-finite cost, non-positive pivot in a 3x3 / 9x9 block, p.Sp <= 0   */
#define CASPAR_BA_ESTATE (-5)   /* call order, e.g. pcg_solve before linearize                           */

#define CASPAR_BA_MAX_TRACK 1024 /* longest supported track (observations of one point) */

typedef struct caspar_ba caspar_ba_t; /* opaque handle */

typedef struct {
  int32_t num_cameras, num_points;
  int64_t num_observations;
  float* cameras;              /* DEVICE [num_cameras][9]. Borrowed; updated in place by an accepted step. */
  float* points;               /* DEVICE [num_points][3].  Borrowed; updated in place by an accepted step. */
  const float* observations;   /* DEVICE or HOST [N][2] pixels.              Copied (reordered) at create. */
  const int32_t* camera_index; /* DEVICE or HOST [N], 0 <= v < num_cameras.  Copied at create.             */
  const int32_t* point_index;  /* DEVICE or HOST [N], 0 <= v < num_points.   Copied at create.             */
  int32_t robust_loss;         /* 0 = none (F = 1/2 sum |r|^2), 1 = Cauchy (F = 1/2 sum c^2 log(1+|r|^2/c^2)) */
  float robust_scale;          /* c in pixels (> 0 when robust_loss = 1)                                   */
  int32_t damping_mode;        /* 0 = lambda * max(diag(J^T J), 1e-6) (Marquardt scaling), 1 = lambda * I  */
  int32_t camera_model;        /* 0 = angle-axis 9-vector, additive update (north_star; C2);
                                  1 = the paper's Pose3 + calibration camera: the rotation is
                                      linearised in its tangent space, R(d) = R(w) Exp(d), and an accepted step
                                      retracts w <- Log(R(w) Exp(d_w)); t, f, k1, k2 stay additive (N3) */
  float depth_epsilon;         /* eps of d_safe = d + eps * sign_no_zero(d); 0 = no guard (C7)  */
} caspar_ba_problem;

typedef struct {
  int32_t iterations;  /* Schur matvecs performed                                 */
  int32_t converged;   /* 1 iff |r_k| <= rel_tol |b| was reached                  */
  double rel_residual; /* |r_k| / |b| of the recursive residual at exit           */
  double rz0, rz;      /* r.M^-1 r at start and at exit                           */
} caspar_ba_pcg_info;

typedef struct {
  double cost_before, cost_after; /* F at the current and at the trial parameters      */
  double model_decrease;          /* L(0) - L(delta) = -delta.g - 1/2 |J delta|^2      */
  double rho;                     /* gain ratio (cost_before - cost_after) / model_decrease */
  int32_t accepted;
  caspar_ba_pcg_info pcg;
} caspar_ba_step_info;

/* Environment (read once per caspar_ba_create; tuning / test switches, not needed in normal use):
 *   CASPAR_BA_TILE=128|192|256|512|1024  force the tile size T (default 256, doubled until it holds the
 *                                longest track);
 *   CASPAR_BA_PIPELINE=0         use the one-block-per-tile Schur pass instead of the persistent
 *                                TMA-pipelined matvec kernel (which serves tiles of <= 256 slots);
 *   CASPAR_BA_LIN_PIPELINE=0     use the one-block-per-tile linearize / cost kernels instead of the persistent
 *                                TMA-pipelined one (which serves tiles of <= 256 slots);
 *   CASPAR_BA_GRAPH=0            (read at the first solve) launch every PCG kernel on its own instead of
 *                                replaying chunks of 8 iterations as one CUDA graph. */

/* PAPER.md:167 (one device memory block, all arrays views into it), :137-149 (block-local sorted index built once
 * and reused: here the tile layout) -- step S0.
 * Build a solver for one problem on the CURRENT device: validates the indices (on the device when the index arrays
 * live there, else on the host in the pass that counts the tracks), reorders the observations (S0, on the host:
 * sorted by point into tiles of whole points, camera runs contiguous inside a tile), carves the arena.  Every later call on the handle runs on that device
 * whatever device is current in the calling thread.
 * Errors: EINVAL (bad sizes / indices / a track longer than CASPAR_BA_MAX_TRACK / CASPAR_BA_TILE not one of the
 * supported sizes), ENOMEM, ECUDA; the text is available from caspar_ba_last_error(NULL). */
int caspar_ba_create(const caspar_ba_problem* problem, void* cuda_stream, caspar_ba_t** out);

/* PAPER.md:182-204 (section VI-A, the reprojection factor: residual and its derivatives), :163 (block-Jacobi: one
 * block per node) -- steps S1-S4: read the caller's parameter arrays, evaluate residuals and Jacobians of every
 * observation, assemble the 9x9 camera and 3x3 point blocks and the gradient; cache them in the arena.
 * cost_out: HOST, nullable; F at the current parameters.  Errors: ENUMERIC (non-finite cost), ECUDA. */
int caspar_ba_linearize(caspar_ba_t* h, void* cuda_stream, double* cost_out);

/* PAPER.md:163 (normal equations, block-Jacobi preconditioned conjugate gradients), :167-169 (J and J^T applied
 * matrix-free from the per-observation Jacobians) -- steps S5-S8: solve (J^T J + lambda D) delta = -g through the Schur complement with block-Jacobi PCG,
 * x0 = 0, stop when |r_k| <= rel_tol |b| or after max_iter matvecs; back-substitute the point steps.
 * Leaves delta in the arena.  info: HOST, nullable.  Errors: ESTATE (no cached linearization),
 * ENUMERIC (block not positive definite, p.Sp <= 0; delta then holds the last good iterate). */
int caspar_ba_pcg_solve(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, void* cuda_stream,
                        caspar_ba_pcg_info* info);

/* PAPER.md:163 ("does not rely on Schur decomposition and instead solves the linear normal equations directly"),
 * :167-169 (PCG with normal residual: J and J^T applied separately, matrix-free) -- the paper's own linear solve
 * (N1): preconditioned CG on the FULL system (J^T J + lambda D) delta = -g over cameras and points, block
 * Jacobi with one block per node (U'_j, V'_k), x0 = 0, stop when |r_k| <= rel_tol |g| or after max_iter passes over
 * the Jacobians.  Same state machine, info and errors as caspar_ba_pcg_solve; leaves delta in the arena. */
int caspar_ba_pcgnr_solve(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, void* cuda_stream,
                          caspar_ba_pcg_info* info);
/* Linear solver of caspar_ba_lm_step / caspar_ba_solve: 0 = Schur PCG (north_star, default), 1 = caspar_ba_pcgnr_solve. */
int caspar_ba_set_linear_solver(caspar_ba_t* h, int32_t mode);

/* PAPER.md:163 (Levenberg-Marquardt, quality-based damping after Madsen et al.: the gain ratio decides) --
 * steps S1-S10: linearize if the cache is stale, pcg_solve, evaluate the trial point x + delta, gain ratio,
 * then commit (parameters updated in place, cache stale) or discard (cache stays valid).
 * accept_mode: 0 = accept iff rho > 0, the trial cost is finite AND lower than the current one (with a truncated fp32
 * solve both differences of the gain ratio can be negative: DESIGN.md 6.3), 1 = always, 2 = never (dry run).
 * info: HOST, required.
 * Linear-solve failures do not abort the iteration: a curvature breakdown
 * p.Sp <= 0 after at least one iteration truncates PCG at the last good iterate and the step is judged by its
 * gain ratio; a damped block that is not positive definite in fp32 (or a breakdown before the first iterate)
 * gives a REJECTED step whatever accept_mode says (accepted = 0, rho = -1, cost_after = cost_before, text in
 * caspar_ba_last_error), so that the caller's damping update raises lambda.  Errors: ENUMERIC (non-finite
 * cost at the CURRENT parameters), ECUDA, EINVAL. */
int caspar_ba_lm_step(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, int32_t accept_mode,
                      void* cuda_stream, caspar_ba_step_info* info);

/* PAPER.md:163 (the outer LM loop with the damping update of Madsen, Nielsen, Tingleff) --
 * `iterations` adaptive LM steps from lambda0 with Nielsen's damping update (accepted: lambda *=
 * max(1/3, 1 - (2 rho - 1)^3), nu = 2; rejected: lambda *= nu, nu *= 2).  infos[iterations] and
 * lambdas[iterations] (HOST, nullable) receive each step's record and the lambda it was solved with. */
int caspar_ba_solve(caspar_ba_t* h, int32_t iterations, float lambda0, float rel_tol, int32_t max_iter,
                    void* cuda_stream, caspar_ba_step_info* infos, float* lambdas);

/* PAPER.md:163 ("block Jacobi preconditioner ... one block per node") -- preconditioner of the Schur PCG:
 * 0 = blockdiag(U'_j), the damped camera blocks (default; C9); 1 = the diagonal 9x9 blocks of the Schur
 * complement itself, S_jj = U'_j - sum_{i in j} W_i V'^-1 W_i^T ("Schur-Jacobi", N4): one more
 * camera-ordered pass over the stored Jacobians per lambda; measured PCG iterations to tolerance: -2 % on the large grid
 * scene (its cap of 100 is hit because of the GLOBAL camera coupling), -10 % on mid, -30 % on the skewed scene.  Takes effect at the
 * next solve.  Errors: EINVAL. */
int caspar_ba_set_preconditioner(caspar_ba_t* h, int32_t mode);

/* PAPER.md:167-169 ("Separate kernels are used for the first iteration of the solver ... the initial score and the
 * Jacobian are calculated simultaneously, while subsequent runs use the score values from the previous iteration") --
 * the paper's fusion variant (N2).  mode 1: caspar_ba_lm_step evaluates the trial point x + delta with the
 * FULL linearization kernel (residuals, Jacobians, V_k, g_p and the cost in one pass) into a second set of arrays
 * (allocated here: 104 bytes per observation slot + 40 per point), and an accepted step swaps the two sets instead of
 * linearizing again: the next caspar_ba_lm_step starts at S4 with the cost it already knows.  A rejected step throws
 * the speculative Jacobians away.  Results are bit-identical to mode 0 (the same kernel at the same point).
 * mode 0 (default): S9 is the residual-only pass.  Errors: EINVAL, ENOMEM. */
int caspar_ba_set_fusion(caspar_ba_t* h, int32_t mode);

/* SURVEY.md 8(e) (the paper itself is single-GPU; its "shared add", taken across devices) --
 * POINT-SHARDED problem: the handle is ONE SHARD.  It was created with ALL cameras (replicated on every shard, the
 * same values) and a SUBSET of the points with all their observations (point ids local to the shard).  Every partial
 * sum over observations is then summed over the shards before it is used, through the caller's collective:
 *   fn(ctx, count, cuda_stream)  sum the first `count` DOUBLES of the exchange buffer over all shards, in place, result
 *                                on every shard (an all-reduce), enqueued on `cuda_stream`; return 0 on success.
 * exchange_buffer_dev: DEVICE, caller-owned, >= 54 * num_cameras + 8 doubles, borrowed until the next
 * caspar_ba_set_shard / destroy.  is_root: exactly one shard passes 1 (it contributes the replicated camera terms).
 * Exchanges per call: linearize 1 (U, g_c, cost); pcg_solve 1 for the right-hand side (+1 with the Schur-Jacobi
 * preconditioner) + ONE per iteration (q and p.q) + 1 (step scalars); lm_step 1 more (trial cost, |J delta|^2,
 * delta.g).  The PCG vector kernels run redundantly on every shard; their scalar sums are folded in a fixed order, so
 * alpha, beta, the direction scale and the stop decision -- hence x, r, p and the cameras -- are bit-identical on all
 * shards without any broadcast.  All shards must make the same calls in the same order.  The CUDA-graph PCG chunks,
 * caspar_ba_set_fusion and caspar_ba_pcgnr_solve are not used on a sharded handle.
 * fn = NULL returns the handle to a single-GPU problem.  Errors: EINVAL (buffer too small). */
typedef int (*caspar_ba_exchange_fn)(void* ctx, size_t count, void* cuda_stream);
int caspar_ba_set_shard(caspar_ba_t* h, caspar_ba_exchange_fn fn, void* ctx, double* exchange_buffer_dev,
                        size_t exchange_count, int32_t is_root);

/* PAPER.md:194-203 (residual only), :220 (fp32 summation is the paper's stated accuracy loss: the sum is fp64 here) --
 * step S9 without the update: F at the caller's current parameters.  cost_out: HOST, required. */
int caspar_ba_cost(caspar_ba_t* h, void* cuda_stream, double* cost_out);

/* PAPER.md:194-203 (residual only) -- step S9 for callers that cannot allocate (code under CUDA-graph capture, serving
 * loops, harnesses that forbid cudaMalloc): F = 1/2 sum rho(|r_i|^2) at the parameters in `problem`, with NO handle
 * and NO allocation.  The scratch the handle path keeps in its arena (the S1 camera table, the per-block partial
 * sums) is a fixed device array inside the library: 144 B x CASPAR_BA_STATIC_MAX_CAMERAS + 4.6 KiB = 2.25 MiB, held
 * by every GPU that loads the library until the process exits.
 *   problem: num_cameras <= CASPAR_BA_STATIC_MAX_CAMERAS; cameras, points, observations, camera_index, point_index
 *            are ALL DEVICE pointers on the CURRENT device (read only, caller's order; nothing is copied or kept);
 *            robust_loss / robust_scale / depth_epsilon as in caspar_ba_create; damping_mode and camera_model do not
 *            enter the cost and are ignored.
 *   cost_out_dev: DEVICE double, written by the last of the three kernels the call enqueues on `cuda_stream`.
 * Asynchronous: no synchronisation, no host result; calls cudaMalloc / cudaFree or any allocating routine never.
 * An index out of range cannot be reported without a round trip: it makes *cost_out_dev NaN (no fault).
 * ALL calls on one GPU share the scratch array: calls that overlap there (two streams, two host threads) race.  A
 * call writes every scratch word before it reads it, so nothing has to be cleared and the previous call's contents
 * never show.  The first call on a device resolves the array's address (and, with lazy module loading, loads the
 * kernels): make one call outside stream capture first.
 * Errors: EINVAL (null pointer, negative size, num_cameras > CASPAR_BA_STATIC_MAX_CAMERAS, robust_scale <= 0 with
 * robust_loss = 1, a pointer that is not device memory of the current device), ECUDA; the text is available from
 * caspar_ba_last_error(NULL). */
#define CASPAR_BA_STATIC_MAX_CAMERAS 16384
int caspar_ba_cost_static(const caspar_ba_problem* problem, double* cost_out_dev, void* cuda_stream);

/* frees the one arena (and the handle's events, graph, pinned scalars).  NULL is a no-op. */
void caspar_ba_destroy(caspar_ba_t* h);

/* Host-buffer convenience (end-to-end path): copy HOST parameter arrays ([Nc][9], [Np][3]; pinned memory
 * makes the copy asynchronous) into the borrowed device arrays and mark the cache stale / copy the
 * device arrays back to HOST buffers.  get synchronises the stream. */
int caspar_ba_set_parameters_host(caspar_ba_t* h, const float* cameras_host, const float* points_host,
                                  void* cuda_stream);
int caspar_ba_get_parameters_host(caspar_ba_t* h, float* cameras_host, float* points_host, void* cuda_stream);

/* ---- test-only exports: slow path, caller's observation / node order, array-of-structs float64 ---- */
enum {
  CASPAR_BA_RESIDUALS = 0, /* [N][2]          (robust-reweighted if enabled)   */
  CASPAR_BA_JC = 1,        /* [N][2][9]                                          */
  CASPAR_BA_JP = 2,        /* [N][2][3]                                          */
  CASPAR_BA_U = 3,         /* [Nc][9][9]                                         */
  CASPAR_BA_V = 4,         /* [Np][3][3]                                         */
  CASPAR_BA_G = 5,         /* [9 Nc + 3 Np]                                      */
  CASPAR_BA_SCHUR_RHS = 6, /* [9 Nc]        (after pcg_solve)                    */
  CASPAR_BA_DELTA = 7,     /* [9 Nc + 3 Np] (after pcg_solve)                    */
  CASPAR_BA_PRECONDITIONER = 8 /* [Nc][9][9] the blocks the preconditioner inverts (after pcg_solve / schur_matvec) */
};
/* device_dst: DEVICE double array with exactly `count` elements of the shape above. */
int caspar_ba_export(caspar_ba_t* h, int32_t what, double* device_dst, size_t count, void* cuda_stream);
/* q = S p at damping lambda from the cached linearization; p_dev, q_dev: DEVICE double [9 Nc]. */
int caspar_ba_schur_matvec(caspar_ba_t* h, float lambda, const double* p_dev, double* q_dev, void* cuda_stream);

/* ---- introspection ---- */
typedef struct {
  int32_t tile_slots;        /* T: observation slots (= threads) per tile                       */
  int32_t num_tiles;
  int64_t padded_slots;      /* num_tiles * T                                                   */
  int64_t camera_runs;       /* sum over tiles of distinct cameras in the tile                  */
  int64_t arena_bytes;
  int64_t kernels_launched;  /* kernels this handle has launched since create (or reset)         */
  /* CUDA-event time of the two dominant kernels, accumulated while profiling is on:              */
  double linearize_ms_total, matvec_ms_total;
  int64_t linearize_count, matvec_count;
  int32_t matvec_pipelined;  /* 1: the Schur matvec runs as the persistent TMA-pipelined kernel       */
  int32_t pipeline_stages;   /* shared-memory ring depth of that kernel (0 if not used)               */
  int32_t num_hot_cameras;   /* cameras whose q rows the pipelined matvec accumulates per CTA (> 0: HOT kernel) */
  int32_t device;            /* CUDA device the handle lives on                                       */
  double create_seconds;     /* host wall time of caspar_ba_create, of which ...                      */
  double reorder_seconds;    /* ... the S0 reordering (host, OpenMP)                                  */
  int32_t linearize_pipelined; /* 1: linearize and cost run as the persistent TMA-pipelined kernel      */
  int32_t reserved;
  int64_t speculative_hits;    /* caspar_ba_set_fusion(1): accepted steps whose trial linearization was reused ... */
  int64_t speculative_misses;  /* ... and rejected ones, whose trial linearization was thrown away                */
  int64_t arena2_bytes;        /* second set of linearization arrays (0 until caspar_ba_set_fusion(h, 1))         */
  int64_t shard_exchanges;     /* calls of the caspar_ba_set_shard collective so far                               */
} caspar_ba_stats;
/* Synchronises the stream the timed kernels ran on, then fills *out. */
int caspar_ba_get_stats(caspar_ba_t* h, caspar_ba_stats* out);
/* enable != 0: bracket every linearize and Schur-matvec kernel with CUDA events on its stream.
 * Also resets the accumulated times and the launch counter. */
int caspar_ba_set_profiling(caspar_ba_t* h, int32_t enable);
/* ---- step S0 on its own (host only, no CUDA call): the observation reordering that create performs ----
 * cam_index / point_index: HOST [n].  tile = 0 lets the library choose T, else 256 | 512 | 1024.
 * caspar_ba_layout_copy copies one of the planned arrays to HOST memory (`bytes` must match exactly):
 *   0 obs_of_slot int32[slots]   1 cam int32[slots]        2 rank uint16[slots]     3 tile_pt int32[tiles+1]
 *   4 run_begin int32[tiles+1]   5 run_cam int32[runs+tiles+1]  6 run_slot uint16[runs+tiles+1]
 *   7 pt_ptr int32[np_obs+1]     8 pt_perm int32[np]       9 cslot int32[n]         10 chunk_cam int32[chunks]
 *   11 chunk_begin int32[chunks+1] */
typedef struct caspar_ba_layout caspar_ba_layout_t;
typedef struct {
  int32_t tile_slots, num_tiles, observed_points, num_chunks;
  int64_t padded_slots, camera_runs;
} caspar_ba_layout_info;
int caspar_ba_layout_create(int32_t num_cameras, int32_t num_points, int64_t n, const int32_t* cam_index,
                            const int32_t* point_index, int32_t tile, caspar_ba_layout_t** out);
int caspar_ba_layout_get_info(const caspar_ba_layout_t* l, caspar_ba_layout_info* info);
int caspar_ba_layout_copy(const caspar_ba_layout_t* l, int32_t which, void* dst_host, size_t bytes);
void caspar_ba_layout_destroy(caspar_ba_layout_t* l);

/* Text of the last failure on the handle; valid until the next call on it; never NULL.
 * h = NULL: text of the last failed caspar_ba_create / caspar_ba_layout_create on the calling thread. */
const char* caspar_ba_last_error(const caspar_ba_t* h);

#ifdef __cplusplus
}
#endif
#endif
