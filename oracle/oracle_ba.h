/* oracle_ba.h — fp64 CPU ORACLE for one Levenberg-Marquardt iteration of bundle adjustment.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header, table or helper with
 * the CUDA path (paper_2605_30583_b200/csrc, include/caspar_ba.h) and neither includes the other.
 *
 * What it computes follows /root/reference/PAPER.md (arxiv 2605.30583, "Caspar"):
 *   - the Snavely reprojection residual, PAPER.md:182-204 (section VI-A);
 *   - Levenberg-Marquardt with quality-based damping after Madsen et al., PAPER.md:163 (section V);
 *   - block-Jacobi preconditioned conjugate gradients, one block per node, PAPER.md:163,167-169;
 * with the readings listed in DESIGN.md ("Readings of the paper"): the linear system is the
 * point-eliminated (Schur) one and cameras are 9-vectors updated additively, as
 * BASELINE.json `north_star` fixes.  The paper's own variants are here too, each behind a
 * switch that defaults to the north_star reading: the full-system solve without Schur elimination
 * (oracle_ba_pcgnr_solve), the tangent-space Pose3 rotation with retraction and the
 * d_safe depth guard (camera_model, depth_epsilon), and the block-Jacobi preconditioner
 * built from the diagonal blocks of the Schur complement itself (oracle_ba_set_preconditioner).
 *
 * All pointers are HOST pointers; all floating point is double.  Every call returns 0 on success,
 * a negative ORACLE_BA_E* code otherwise.
 */
#ifndef ORACLE_BA_H
#define ORACLE_BA_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORACLE_BA_OK 0
#define ORACLE_BA_EINVAL (-1)
#define ORACLE_BA_ENOMEM (-3)
#define ORACLE_BA_ENUMERIC (-4)
#define ORACLE_BA_ESTATE (-5)

typedef struct oracle_ba oracle_ba_t;

typedef struct {
  int32_t num_cameras, num_points;
  int64_t num_observations;
  double* cameras;               /* [num_cameras][9]: w0 w1 w2 t0 t1 t2 f k1 k2. Borrowed, updated in place. */
  double* points;                /* [num_points][3]. Borrowed, updated in place.                            */
  const double* observations;    /* [N][2] pixels. Borrowed.                                                 */
  const int32_t* camera_index;   /* [N]. Borrowed.                                                           */
  const int32_t* point_index;    /* [N]. Borrowed.                                                           */
  int32_t robust_loss;           /* 0 = none, 1 = Cauchy                                                     */
  double robust_scale;           /* c, pixels                                                                */
  int32_t damping_mode;          /* 0 = lambda * max(diag(J^T J), 1e-6), 1 = lambda * I                      */
  int32_t camera_model;          /* 0 = angle-axis, additive update; 1 = Pose3: rotation linearised in its tangent
                                    space, R(d) = R(w) Exp(d), retraction w <- Log(R(w) Exp(d_w)); t, f, k1, k2
                                    additive (N3)                             */
  double depth_epsilon;          /* eps of d_safe = d + eps sign_no_zero(d); 0 = none (C7)   */
} oracle_ba_problem;

typedef struct {
  int32_t iterations, converged;
  double rel_residual, rz0, rz;
} oracle_ba_pcg_info;

typedef struct {
  double cost_before, cost_after, model_decrease, rho;
  int32_t accepted;
  oracle_ba_pcg_info pcg;
} oracle_ba_step_info;

enum {
  ORACLE_BA_RESIDUALS = 0, /* [N][2]                    */
  ORACLE_BA_JC = 1,        /* [N][2][9]                 */
  ORACLE_BA_JP = 2,        /* [N][2][3]                 */
  ORACLE_BA_U = 3,         /* [Nc][9][9]                */
  ORACLE_BA_V = 4,         /* [Np][3][3]                */
  ORACLE_BA_G = 5,         /* [9 Nc + 3 Np]             */
  ORACLE_BA_SCHUR_RHS = 6, /* [9 Nc]                    */
  ORACLE_BA_DELTA = 7,     /* [9 Nc + 3 Np]             */
  ORACLE_BA_DAMPING = 8    /* [9 Nc + 3 Np], the diag D */
};

/* One observation: residual r (2), and if non-NULL d r / d camera (2x9 row-major) and d r / d point (2x3). */
void oracle_ba_observation(const double cam[9], const double pt[3], const double pixel[2],
                           double r[2], double jc[18], double jp[6]);
/* The same for either camera model and any depth guard: with camera_model = 1 the first three columns of jc are
 * d r / d d_w of the right perturbation R(w) Exp(d_w) at d_w = 0. */
void oracle_ba_observation_model(int32_t camera_model, double depth_epsilon, const double cam[9], const double pt[3],
                                 const double pixel[2], double r[2], double jc[18], double jp[6]);
/* Retraction of one camera: out = cam (+) delta.  camera_model 0: cam + delta; 1: w <- Log(Exp(w) Exp(delta_w)),
 * the other six entries additive. */
void oracle_ba_retract_camera(int32_t camera_model, const double cam[9], const double delta[9], double out[9]);
/* Rotation matrix R(w) (row-major 3x3) of the angle-axis vector w. */
void oracle_ba_rotation(const double w[3], double rot[9]);
/* Inverse of a symmetric positive-definite n x n matrix by Cholesky; nonzero if a pivot is not positive. */
int oracle_ba_spd_inverse(int n, const double* a, double* inv);

int oracle_ba_create(const oracle_ba_problem* problem, oracle_ba_t** out);
void oracle_ba_destroy(oracle_ba_t* h);
int oracle_ba_linearize(oracle_ba_t* h, double* cost_out);
int oracle_ba_cost(oracle_ba_t* h, double* cost_out);
int oracle_ba_pcg_solve(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, oracle_ba_pcg_info* info);
int oracle_ba_lm_step(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, int32_t accept_mode,
                      oracle_ba_step_info* info);
/* Adaptive LM run (Nielsen damping update): `iterations` steps from lambda0; infos[iterations],
 * lambdas[iterations] receive the step records and the lambda each step was solved with. */
int oracle_ba_solve(oracle_ba_t* h, int32_t iterations, double lambda0, double rel_tol, int32_t max_iter,
                    oracle_ba_step_info* infos, double* lambdas);
int oracle_ba_export(oracle_ba_t* h, int32_t what, double* dst, size_t count);
/* q = S p with S = U' - W V'^-1 W^T at damping lambda; p, q are [9 Nc]. */
int oracle_ba_schur_matvec(oracle_ba_t* h, double lambda, const double* p, double* q);
/* y = (J^T J + lambda D) x on the full (camera + point) system; x, y are [9 Nc + 3 Np]. */
int oracle_ba_full_matvec(oracle_ba_t* h, double lambda, const double* x, double* y);
/* The paper's own linear solve (PAPER.md:163 "does not rely on Schur decomposition", :167-169 PCG with normal
 * residual): preconditioned CG on the FULL damped normal equations (J^T J + lambda D) delta = -g, J and J^T applied
 * separately per observation, block-Jacobi preconditioner with one block per node: blockdiag(U'_j, V'_k).
 * x0 = 0; stop when |r_k| <= rel_tol |g|.  Leaves delta (cameras and points) like oracle_ba_pcg_solve. */
int oracle_ba_pcgnr_solve(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, oracle_ba_pcg_info* info);
/* Preconditioner of oracle_ba_pcg_solve: 0 = blockdiag(U'_j) (C9, the default); 1 = the diagonal 9x9
 * blocks of the Schur complement, S_jj = U'_j - sum_{i in j} W_i V'^-1_k(i) W_i^T ("Schur-Jacobi"). */
int oracle_ba_set_preconditioner(oracle_ba_t* h, int32_t mode);
/* Linear solver of oracle_ba_lm_step / oracle_ba_solve: 0 = Schur PCG (default), 1 = oracle_ba_pcgnr_solve. */
int oracle_ba_set_linear_solver(oracle_ba_t* h, int32_t mode);
/* The 9x9 blocks the current preconditioner inverts, [Nc][9][9] (after a solve or matvec at some lambda). */
int oracle_ba_export_preconditioner_blocks(oracle_ba_t* h, double* dst, size_t count);
int oracle_ba_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
