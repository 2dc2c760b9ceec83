/* oracle_ba.c — fp64 CPU ORACLE (TEST INFRASTRUCTURE ONLY; see oracle_ba.h).
 *
 * Plain loops over observations, cameras and points in the caller's order, array-of-structs,
 * double precision throughout.  No blocking, tiling, fusion or reordering beyond what each
 * definition states.  Every sum over "the observations of camera j" or "of point k" runs over
 * that node's observations in the caller's order; OpenMP (if enabled) only distributes whole
 * nodes or whole observations over threads, so results do not depend on the thread count
 * (the single exception, the scalar cost sum, is an fp64 reduction).
 *
 * Parity pins: tests/test_oracle_*.py (finite differences, scipy rotations, explicit sparse J,
 * dense Cholesky of the full damped system, noise-free convergence, limits; for the paper's variants:
 * finite differences through the retraction, scipy's rotation composition, the diagonal blocks of the dense
 * Schur complement, the dense solution of the full system).  No part of this file is "parity unpinned".
 */
#include "oracle_ba.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define D_MIN 1e-6 /* floor of the Marquardt scaling diag(J^T J); reading C5 */

struct oracle_ba {
  oracle_ba_problem pb;
  int64_t n_obs;
  int nc, np;
  /* observations grouped by node, caller's order inside each group */
  int64_t *cam_ptr, *cam_obs, *pt_ptr, *pt_obs;
  /* linearization at the current parameters (robust-reweighted if enabled) */
  double *r, *jc, *jp;    /* [N][2], [N][18], [N][6] */
  double *U, *V, *g, *D;  /* [Nc][81], [Np][9], [9Nc+3Np], [9Nc+3Np] */
  double cost;
  int linearized;
  /* damped blocks for the lambda in `prepared_lambda` */
  double *Ud, *Minv, *Vinv; /* [Nc][81], [Nc][81], [Np][9] */
  double* Pblk;             /* [Nc][81] the blocks the preconditioner inverts (U'_j or S_jj) */
  int preconditioner;       /* 0 = blockdiag(U'), 1 = diagonal blocks of S */
  int linear_solver;        /* what oracle_ba_lm_step calls: 0 = Schur PCG, 1 = full-system PCGNR */
  double prepared_lambda;
  int prepared;
  double *b, *delta; /* [9Nc], [9Nc+3Np] */
  int have_delta;
};

int oracle_ba_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* O1/O2: residual and Jacobians of one observation (O1, O2)       */
/* ------------------------------------------------------------------------------------------ */

/* a = sin(th)/th, b = (1-cos th)/th^2 and (1/th) d/dth of each; series below th^2 = 1e-4 (C3). */
static void angle_coefficients(double th2, double* a, double* b, double* a1, double* b1) {
  if (th2 < 1e-4) {
    double t2 = th2, t4 = th2 * th2, t6 = t4 * th2;
    *a = 1.0 - t2 / 6.0 + t4 / 120.0 - t6 / 5040.0;
    *b = 0.5 - t2 / 24.0 + t4 / 720.0 - t6 / 40320.0;
    *a1 = -1.0 / 3.0 + t2 / 30.0 - t4 / 840.0 + t6 / 45360.0;
    *b1 = -1.0 / 12.0 + t2 / 180.0 - t4 / 6720.0 + t6 / 453600.0;
  } else {
    double th = sqrt(th2), s = sin(th), c = cos(th);
    *a = s / th;
    *b = (1.0 - c) / th2;
    *a1 = (th * c - s) / (th2 * th);
    *b1 = (th * s - 2.0 * (1.0 - c)) / (th2 * th2);
  }
}

void oracle_ba_rotation(const double w[3], double rot[9]) {
  /* R = I + a [w]x + b [w]x^2, [w]x^2 = w w^T - th^2 I */
  double th2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
  double a, b, a1, b1;
  angle_coefficients(th2, &a, &b, &a1, &b1);
  double K[9] = {0.0, -w[2], w[1], w[2], 0.0, -w[0], -w[1], w[0], 0.0};
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double k2 = w[i] * w[j] - (i == j ? th2 : 0.0);
      rot[3 * i + j] = (i == j ? 1.0 : 0.0) + a * K[3 * i + j] + b * k2;
    }
}

void oracle_ba_observation(const double cam[9], const double X[3], const double m[2], double r[2], double jc[18],
                           double jp[6]) {
  oracle_ba_observation_model(0, 0.0, cam, X, m, r, jc, jp);
}

/* sign_no_zero(d) = +1 for d >= 0, -1 otherwise */
static double sign_no_zero(double d) { return d >= 0.0 ? 1.0 : -1.0; }

void oracle_ba_observation_model(int32_t camera_model, double depth_epsilon, const double cam[9], const double X[3],
                                 const double m[2], double r[2], double jc[18], double jp[6]) {
  const double* w = cam;
  const double* t = cam + 3;
  double f = cam[6], k1 = cam[7], k2 = cam[8];
  double R[9];
  oracle_ba_rotation(w, R);
  /* P = R X + t */
  double P[3];
  for (int i = 0; i < 3; ++i) P[i] = R[3 * i] * X[0] + R[3 * i + 1] * X[1] + R[3 * i + 2] * X[2] + t[i];
  /* p = -P_xy / d_safe, d_safe = d + eps sign_no_zero(d), d = P_z; eps = 0 is the north_star
   * reading C7 (no guard).  d d_safe / d d = 1, so the derivatives below only see d_safe in place of P_z. */
  double d_safe = P[2] + depth_epsilon * sign_no_zero(P[2]);
  double p[2] = {-P[0] / d_safe, -P[1] / d_safe};
  double n = p[0] * p[0] + p[1] * p[1];
  double rad = 1.0 + k1 * n + k2 * n * n;
  double uv[2] = {f * rad * p[0], f * rad * p[1]};
  r[0] = uv[0] - m[0];
  r[1] = uv[1] - m[1];
  if (!jc && !jp) return;

  /* d uv / d p = f (rad I + (2 k1 + 4 k2 n) p p^T) */
  double c = 2.0 * k1 + 4.0 * k2 * n;
  double duv_dp[4] = {f * (rad + c * p[0] * p[0]), f * c * p[0] * p[1], f * c * p[1] * p[0], f * (rad + c * p[1] * p[1])};
  /* d p / d P = (-1/d_safe) [[1, 0, p_x], [0, 1, p_y]] */
  double iz = -1.0 / d_safe;
  double dp_dP[6] = {iz, 0.0, iz * p[0], 0.0, iz, iz * p[1]};
  /* A = d uv / d P (2x3) */
  double A[6];
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 3; ++j) A[3 * i + j] = duv_dp[2 * i] * dp_dP[j] + duv_dp[2 * i + 1] * dp_dP[3 + j];

  if (jp) /* J_p = A R */
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 3; ++j) jp[3 * i + j] = A[3 * i] * R[j] + A[3 * i + 1] * R[3 + j] + A[3 * i + 2] * R[6 + j];

  if (jc) {
    /* d(RX)/dw = a1 q w^T - a [X]x + b1 (w s - th^2 X) w^T + b (s I + w X^T - 2 X w^T),  q = w x X, s = w.X */
    double th2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
    double a, b, a1, b1;
    angle_coefficients(th2, &a, &b, &a1, &b1);
    double q[3] = {w[1] * X[2] - w[2] * X[1], w[2] * X[0] - w[0] * X[2], w[0] * X[1] - w[1] * X[0]};
    double s = w[0] * X[0] + w[1] * X[1] + w[2] * X[2];
    double Xx[9] = {0.0, -X[2], X[1], X[2], 0.0, -X[0], -X[1], X[0], 0.0};
    double G[9];
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j)
        G[3 * i + j] = a1 * q[i] * w[j] - a * Xx[3 * i + j] + b1 * (w[i] * s - th2 * X[i]) * w[j] +
                       b * ((i == j ? s : 0.0) + w[i] * X[j] - 2.0 * X[i] * w[j]);
    if (camera_model == 1) {
      /* Pose3 (PAPER.md:163 "linearization ... in the tangent space"; :184 cam_T_world: sf.Pose3): the rotation is
       * perturbed on the right, R(d) = R Exp(d), so d(R Exp(d) X)/dd at d = 0 is R d(d x X)/dd = -R [X]x. */
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
          G[3 * i + j] = -(R[3 * i] * Xx[j] + R[3 * i + 1] * Xx[3 + j] + R[3 * i + 2] * Xx[6 + j]);
    }
    for (int i = 0; i < 2; ++i) {
      double* row = jc + 9 * i;
      for (int j = 0; j < 3; ++j) row[j] = A[3 * i] * G[j] + A[3 * i + 1] * G[3 + j] + A[3 * i + 2] * G[6 + j];
      for (int j = 0; j < 3; ++j) row[3 + j] = A[3 * i + j]; /* d/dt: dP/dt = I */
      row[6] = rad * p[i];                                   /* d/df  */
      row[7] = f * n * p[i];                                 /* d/dk1 */
      row[8] = f * n * n * p[i];                             /* d/dk2 */
    }
  }
}

/* ------------------------------------------------------------------------------------------ */
/* Retraction ("retraction are performed in the tangent space"; N3)      */
/* ------------------------------------------------------------------------------------------ */
/* unit quaternion (w, x, y, z) of the rotation vector v: (cos(th/2), sin(th/2) v/th) */
static void quat_of_rotvec(const double v[3], double q[4]) {
  double th2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  double th = sqrt(th2);
  double k = th2 < 1e-8 ? 0.5 - th2 / 48.0 : sin(0.5 * th) / th; /* sin(th/2)/th */
  q[0] = cos(0.5 * th);
  q[1] = k * v[0]; q[2] = k * v[1]; q[3] = k * v[2];
}

/* rotation vector of a unit quaternion, angle in [0, pi] */
static void rotvec_of_quat(const double qin[4], double v[3]) {
  double q[4] = {qin[0], qin[1], qin[2], qin[3]};
  if (q[0] < 0.0) for (int i = 0; i < 4; ++i) q[i] = -q[i]; /* same rotation, angle <= pi */
  double s = sqrt(q[1] * q[1] + q[2] * q[2] + q[3] * q[3]); /* sin(th/2) */
  double k = s < 1e-8 ? 2.0 / q[0] : 2.0 * atan2(s, q[0]) / s;
  v[0] = k * q[1]; v[1] = k * q[2]; v[2] = k * q[3];
}

void oracle_ba_retract_camera(int32_t camera_model, const double cam[9], const double delta[9], double out[9]) {
  for (int a = 0; a < 9; ++a) out[a] = cam[a] + delta[a];
  if (camera_model == 1) { /* w <- Log(Exp(w) Exp(delta_w)): quaternion product q(w) q(delta_w) */
    double a[4], b[4], c[4];
    quat_of_rotvec(cam, a);
    quat_of_rotvec(delta, b);
    c[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    c[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    c[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    c[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
    rotvec_of_quat(c, out);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* small dense helpers                                                                        */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_spd_inverse(int n, const double* a, double* inv) {
  /* Cholesky A = L L^T, then solve A x = e_c column by column. n <= 16. */
  double L[256];
  if (n > 16) return ORACLE_BA_EINVAL;
  memset(L, 0, sizeof L);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j <= i; ++j) {
      double s = a[n * i + j];
      for (int k = 0; k < j; ++k) s -= L[n * i + k] * L[n * j + k];
      if (i == j) {
        if (!(s > 0.0)) return ORACLE_BA_ENUMERIC;
        L[n * i + i] = sqrt(s);
      } else {
        L[n * i + j] = s / L[n * j + j];
      }
    }
  for (int c = 0; c < n; ++c) {
    double y[16], x[16];
    for (int i = 0; i < n; ++i) {
      double s = (i == c ? 1.0 : 0.0);
      for (int k = 0; k < i; ++k) s -= L[n * i + k] * y[k];
      y[i] = s / L[n * i + i];
    }
    for (int i = n - 1; i >= 0; --i) {
      double s = y[i];
      for (int k = i + 1; k < n; ++k) s -= L[n * k + i] * x[k];
      x[i] = s / L[n * i + i];
    }
    for (int i = 0; i < n; ++i) inv[n * i + c] = x[i];
  }
  return 0;
}

static void matvec_n(int n, const double* a, const double* x, double* y) {
  for (int i = 0; i < n; ++i) {
    double s = 0.0;
    for (int j = 0; j < n; ++j) s += a[n * i + j] * x[j];
    y[i] = s;
  }
}

/* group observation ids by node: ptr[n_nodes+1], list[N], caller's order inside each group */
static int group_by(const int32_t* idx, int64_t n, int n_nodes, int64_t** ptr_out, int64_t** list_out) {
  int64_t* ptr = (int64_t*)calloc((size_t)n_nodes + 1, sizeof(int64_t));
  int64_t* list = (int64_t*)malloc((size_t)(n > 0 ? n : 1) * sizeof(int64_t));
  int64_t* fill = (int64_t*)malloc(((size_t)n_nodes + 1) * sizeof(int64_t));
  if (!ptr || !list || !fill) { free(ptr); free(list); free(fill); return ORACLE_BA_ENOMEM; }
  for (int64_t i = 0; i < n; ++i) ptr[idx[i] + 1]++;
  for (int j = 0; j < n_nodes; ++j) ptr[j + 1] += ptr[j];
  memcpy(fill, ptr, ((size_t)n_nodes + 1) * sizeof(int64_t));
  for (int64_t i = 0; i < n; ++i) list[fill[idx[i]]++] = i;
  free(fill);
  *ptr_out = ptr;
  *list_out = list;
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* create / destroy                                                                           */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_create(const oracle_ba_problem* pb, oracle_ba_t** out) {
  if (!pb || !out || pb->num_cameras < 0 || pb->num_points < 0 || pb->num_observations < 0) return ORACLE_BA_EINVAL;
  if (pb->num_observations > 0 && (!pb->observations || !pb->camera_index || !pb->point_index)) return ORACLE_BA_EINVAL;
  if ((pb->num_cameras > 0 && !pb->cameras) || (pb->num_points > 0 && !pb->points)) return ORACLE_BA_EINVAL;
  if (pb->robust_loss != 0 && pb->robust_loss != 1) return ORACLE_BA_EINVAL;
  if (pb->robust_loss == 1 && !(pb->robust_scale > 0.0)) return ORACLE_BA_EINVAL;
  if (pb->camera_model != 0 && pb->camera_model != 1) return ORACLE_BA_EINVAL;
  if (!(pb->depth_epsilon >= 0.0)) return ORACLE_BA_EINVAL;
  for (int64_t i = 0; i < pb->num_observations; ++i)
    if (pb->camera_index[i] < 0 || pb->camera_index[i] >= pb->num_cameras || pb->point_index[i] < 0 ||
        pb->point_index[i] >= pb->num_points)
      return ORACLE_BA_EINVAL;
  oracle_ba_t* h = (oracle_ba_t*)calloc(1, sizeof *h);
  if (!h) return ORACLE_BA_ENOMEM;
  h->pb = *pb;
  h->n_obs = pb->num_observations;
  h->nc = pb->num_cameras;
  h->np = pb->num_points;
  size_t N = (size_t)(h->n_obs > 0 ? h->n_obs : 1), nc = (size_t)(h->nc > 0 ? h->nc : 1), np = (size_t)(h->np > 0 ? h->np : 1);
  size_t nv = 9 * nc + 3 * np;
  int rc = group_by(pb->camera_index, h->n_obs, h->nc, &h->cam_ptr, &h->cam_obs);
  if (!rc) rc = group_by(pb->point_index, h->n_obs, h->np, &h->pt_ptr, &h->pt_obs);
  h->r = (double*)malloc(N * 2 * sizeof(double));
  h->jc = (double*)malloc(N * 18 * sizeof(double));
  h->jp = (double*)malloc(N * 6 * sizeof(double));
  h->U = (double*)malloc(nc * 81 * sizeof(double));
  h->Ud = (double*)malloc(nc * 81 * sizeof(double));
  h->Minv = (double*)malloc(nc * 81 * sizeof(double));
  h->Pblk = (double*)malloc(nc * 81 * sizeof(double));
  h->V = (double*)malloc(np * 9 * sizeof(double));
  h->Vinv = (double*)malloc(np * 9 * sizeof(double));
  h->g = (double*)malloc(nv * sizeof(double));
  h->D = (double*)malloc(nv * sizeof(double));
  h->delta = (double*)calloc(nv, sizeof(double));
  h->b = (double*)malloc(9 * nc * sizeof(double));
  if (rc || !h->r || !h->jc || !h->jp || !h->U || !h->Ud || !h->Minv || !h->Pblk || !h->V || !h->Vinv || !h->g || !h->D ||
      !h->delta || !h->b) {
    oracle_ba_destroy(h);
    return ORACLE_BA_ENOMEM;
  }
  *out = h;
  return 0;
}

void oracle_ba_destroy(oracle_ba_t* h) {
  if (!h) return;
  free(h->cam_ptr); free(h->cam_obs); free(h->pt_ptr); free(h->pt_obs);
  free(h->r); free(h->jc); free(h->jp); free(h->U); free(h->Ud); free(h->Minv); free(h->Pblk); free(h->V); free(h->Vinv);
  free(h->g); free(h->D); free(h->delta); free(h->b);
  free(h);
}

/* ------------------------------------------------------------------------------------------ */
/* O3: cost F = 1/2 sum rho(|r|^2); rho(s) = s, or c^2 log(1 + s/c^2) for Cauchy               */
/* ------------------------------------------------------------------------------------------ */
static double cost_at(const oracle_ba_t* h, const double* cams, const double* pts) {
  double total = 0.0;
  double c2 = h->pb.robust_scale * h->pb.robust_scale;
  int robust = h->pb.robust_loss;
#pragma omp parallel for schedule(static) reduction(+ : total)
  for (int64_t i = 0; i < h->n_obs; ++i) {
    double r[2];
    oracle_ba_observation_model(h->pb.camera_model, h->pb.depth_epsilon, cams + 9 * (size_t)h->pb.camera_index[i],
                                pts + 3 * (size_t)h->pb.point_index[i], h->pb.observations + 2 * i, r, NULL, NULL);
    double s = r[0] * r[0] + r[1] * r[1];
    total += robust ? c2 * log1p(s / c2) : s;
  }
  return 0.5 * total;
}

int oracle_ba_cost(oracle_ba_t* h, double* cost_out) {
  if (!h || !cost_out) return ORACLE_BA_EINVAL;
  *cost_out = cost_at(h, h->pb.cameras, h->pb.points);
  return isfinite(*cost_out) ? 0 : ORACLE_BA_ENUMERIC;
}

/* ------------------------------------------------------------------------------------------ */
/* O2-O4: linearize and assemble g, U, V, D                                                    */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_linearize(oracle_ba_t* h, double* cost_out) {
  if (!h) return ORACLE_BA_EINVAL;
  int nc = h->nc, np = h->np;
  double c2 = h->pb.robust_scale * h->pb.robust_scale;
  int robust = h->pb.robust_loss;
  double total = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : total)
  for (int64_t i = 0; i < h->n_obs; ++i) {
    double* r = h->r + 2 * i;
    double* jc = h->jc + 18 * i;
    double* jp = h->jp + 6 * i;
    oracle_ba_observation_model(h->pb.camera_model, h->pb.depth_epsilon,
                                h->pb.cameras + 9 * (size_t)h->pb.camera_index[i],
                                h->pb.points + 3 * (size_t)h->pb.point_index[i], h->pb.observations + 2 * i, r, jc, jp);
    double s = r[0] * r[0] + r[1] * r[1];
    if (robust) {
      /* w = rho'(s) = 1 / (1 + s/c^2); r~ = sqrt(w) r, J~ = sqrt(w) J (first-order reweighting) */
      double sw = sqrt(1.0 / (1.0 + s / c2));
      total += c2 * log1p(s / c2);
      r[0] *= sw; r[1] *= sw;
      for (int k = 0; k < 18; ++k) jc[k] *= sw;
      for (int k = 0; k < 6; ++k) jp[k] *= sw;
    } else {
      total += s;
    }
  }
  h->cost = 0.5 * total;

  double* gc = h->g;
  double* gp = h->g + 9 * (size_t)nc;
  /* camera side: U_j = sum J_c^T J_c, g_c,j = sum J_c^T r over the observations of camera j */
#pragma omp parallel for schedule(dynamic, 16)
  for (int j = 0; j < nc; ++j) {
    double* U = h->U + 81 * (size_t)j;
    double* g = gc + 9 * (size_t)j;
    memset(U, 0, 81 * sizeof(double));
    memset(g, 0, 9 * sizeof(double));
    for (int64_t e = h->cam_ptr[j]; e < h->cam_ptr[j + 1]; ++e) {
      int64_t i = h->cam_obs[e];
      const double* J = h->jc + 18 * i;
      const double* r = h->r + 2 * i;
      for (int a = 0; a < 9; ++a) {
        for (int b = 0; b < 9; ++b) U[9 * a + b] += J[a] * J[b] + J[9 + a] * J[9 + b];
        g[a] += J[a] * r[0] + J[9 + a] * r[1];
      }
    }
    for (int a = 0; a < 9; ++a)
      h->D[9 * (size_t)j + a] = h->pb.damping_mode == 1 ? 1.0 : fmax(U[9 * a + a], D_MIN);
  }
  /* point side */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < np; ++k) {
    double* V = h->V + 9 * (size_t)k;
    double* g = gp + 3 * (size_t)k;
    memset(V, 0, 9 * sizeof(double));
    memset(g, 0, 3 * sizeof(double));
    for (int64_t e = h->pt_ptr[k]; e < h->pt_ptr[k + 1]; ++e) {
      int64_t i = h->pt_obs[e];
      const double* J = h->jp + 6 * i;
      const double* r = h->r + 2 * i;
      for (int a = 0; a < 3; ++a) {
        for (int b = 0; b < 3; ++b) V[3 * a + b] += J[a] * J[b] + J[3 + a] * J[3 + b];
        g[a] += J[a] * r[0] + J[3 + a] * r[1];
      }
    }
    for (int a = 0; a < 3; ++a)
      h->D[9 * (size_t)nc + 3 * (size_t)k + a] = h->pb.damping_mode == 1 ? 1.0 : fmax(V[3 * a + a], D_MIN);
  }
  h->linearized = 1;
  h->prepared = 0;
  h->have_delta = 0;
  if (cost_out) *cost_out = h->cost;
  return isfinite(h->cost) ? 0 : ORACLE_BA_ENUMERIC;
}

/* ------------------------------------------------------------------------------------------ */
/* O5: damped blocks U' = U + lambda D_c, V' = V + lambda D_p and their inverses               */
/* ------------------------------------------------------------------------------------------ */
static int prepare_damped(oracle_ba_t* h, double lambda) {
  if (h->prepared && h->prepared_lambda == lambda) return 0;
  int nc = h->nc, np = h->np, bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
  for (int k = 0; k < np; ++k) {
    double Vd[9];
    memcpy(Vd, h->V + 9 * (size_t)k, sizeof Vd);
    for (int a = 0; a < 3; ++a) Vd[3 * a + a] += lambda * h->D[9 * (size_t)nc + 3 * (size_t)k + a];
    if (oracle_ba_spd_inverse(3, Vd, h->Vinv + 9 * (size_t)k)) bad++;
  }
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : bad)
  for (int j = 0; j < nc; ++j) {
    double* Ud = h->Ud + 81 * (size_t)j;
    double* P = h->Pblk + 81 * (size_t)j;
    memcpy(Ud, h->U + 81 * (size_t)j, 81 * sizeof(double));
    for (int a = 0; a < 9; ++a) Ud[9 * a + a] += lambda * h->D[9 * (size_t)j + a];
    memcpy(P, Ud, 81 * sizeof(double));
    if (h->preconditioner == 1) {
      /* Schur-Jacobi: S_jj = U'_j - sum_{i in j} W_i V'^-1_k(i) W_i^T, W_i = J_c,i^T J_p,i (9x3) */
      for (int64_t e = h->cam_ptr[j]; e < h->cam_ptr[j + 1]; ++e) {
        int64_t i = h->cam_obs[e];
        const double* Jc = h->jc + 18 * i;
        const double* Jp = h->jp + 6 * i;
        const double* Vi = h->Vinv + 9 * (size_t)h->pb.point_index[i];
        double W[27], WV[27];
        for (int a = 0; a < 9; ++a)
          for (int c = 0; c < 3; ++c) W[3 * a + c] = Jc[a] * Jp[c] + Jc[9 + a] * Jp[3 + c];
        for (int a = 0; a < 9; ++a)
          for (int c = 0; c < 3; ++c)
            WV[3 * a + c] = W[3 * a] * Vi[c] + W[3 * a + 1] * Vi[3 + c] + W[3 * a + 2] * Vi[6 + c];
        for (int a = 0; a < 9; ++a)
          for (int c = 0; c < 9; ++c)
            P[9 * a + c] -= WV[3 * a] * W[3 * c] + WV[3 * a + 1] * W[3 * c + 1] + WV[3 * a + 2] * W[3 * c + 2];
      }
    }
    if (oracle_ba_spd_inverse(9, P, h->Minv + 81 * (size_t)j)) bad++;
  }
  if (bad) return ORACLE_BA_ENUMERIC;
  h->prepared = 1;
  h->prepared_lambda = lambda;
  return 0;
}

/* q = U' p - W V'^-1 W^T p, W_i = J_c,i^T J_p,i (never formed) */
static void schur_apply(const oracle_ba_t* h, const double* p, double* q, double* s_pts /* [Np][3] scratch */) {
  int nc = h->nc, np = h->np;
  /* s_k = V'^-1 sum_{i in k} J_p,i^T (J_c,i p_j(i)) */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < np; ++k) {
    double t[3] = {0.0, 0.0, 0.0};
    for (int64_t e = h->pt_ptr[k]; e < h->pt_ptr[k + 1]; ++e) {
      int64_t i = h->pt_obs[e];
      const double* Jc = h->jc + 18 * i;
      const double* Jp = h->jp + 6 * i;
      const double* pj = p + 9 * (size_t)h->pb.camera_index[i];
      double u0 = 0.0, u1 = 0.0;
      for (int a = 0; a < 9; ++a) { u0 += Jc[a] * pj[a]; u1 += Jc[9 + a] * pj[a]; }
      for (int a = 0; a < 3; ++a) t[a] += Jp[a] * u0 + Jp[3 + a] * u1;
    }
    matvec_n(3, h->Vinv + 9 * (size_t)k, t, s_pts + 3 * (size_t)k);
  }
  /* q_j = U'_j p_j - sum_{i in j} J_c,i^T (J_p,i s_k(i)) */
#pragma omp parallel for schedule(dynamic, 16)
  for (int j = 0; j < nc; ++j) {
    double* qj = q + 9 * (size_t)j;
    matvec_n(9, h->Ud + 81 * (size_t)j, p + 9 * (size_t)j, qj);
    for (int64_t e = h->cam_ptr[j]; e < h->cam_ptr[j + 1]; ++e) {
      int64_t i = h->cam_obs[e];
      const double* Jc = h->jc + 18 * i;
      const double* Jp = h->jp + 6 * i;
      const double* s = s_pts + 3 * (size_t)h->pb.point_index[i];
      double v0 = Jp[0] * s[0] + Jp[1] * s[1] + Jp[2] * s[2];
      double v1 = Jp[3] * s[0] + Jp[4] * s[1] + Jp[5] * s[2];
      for (int a = 0; a < 9; ++a) qj[a] -= Jc[a] * v0 + Jc[9 + a] * v1;
    }
  }
}

int oracle_ba_schur_matvec(oracle_ba_t* h, double lambda, const double* p, double* q) {
  if (!h || !p || !q) return ORACLE_BA_EINVAL;
  if (!h->linearized) return ORACLE_BA_ESTATE;
  int rc = prepare_damped(h, lambda);
  if (rc) return rc;
  double* s = (double*)malloc((size_t)(h->np > 0 ? h->np : 1) * 3 * sizeof(double));
  if (!s) return ORACLE_BA_ENOMEM;
  schur_apply(h, p, q, s);
  free(s);
  return 0;
}

int oracle_ba_full_matvec(oracle_ba_t* h, double lambda, const double* x, double* y) {
  if (!h || !x || !y) return ORACLE_BA_EINVAL;
  if (!h->linearized) return ORACLE_BA_ESTATE;
  int nc = h->nc, np = h->np;
  size_t nv = 9 * (size_t)nc + 3 * (size_t)np;
  /* y = J^T (J x) + lambda D x, one observation at a time (sequential: plain definition) */
  for (size_t a = 0; a < nv; ++a) y[a] = lambda * h->D[a] * x[a];
  for (int64_t i = 0; i < h->n_obs; ++i) {
    const double* Jc = h->jc + 18 * i;
    const double* Jp = h->jp + 6 * i;
    size_t oc = 9 * (size_t)h->pb.camera_index[i], op = 9 * (size_t)nc + 3 * (size_t)h->pb.point_index[i];
    double v[2];
    for (int row = 0; row < 2; ++row) {
      double s = 0.0;
      for (int a = 0; a < 9; ++a) s += Jc[9 * row + a] * x[oc + a];
      for (int a = 0; a < 3; ++a) s += Jp[3 * row + a] * x[op + a];
      v[row] = s;
    }
    for (int a = 0; a < 9; ++a) y[oc + a] += Jc[a] * v[0] + Jc[9 + a] * v[1];
    for (int a = 0; a < 3; ++a) y[op + a] += Jp[a] * v[0] + Jp[3 + a] * v[1];
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* O5/O6: Schur right-hand side, preconditioned CG, back-substitution                          */
/* ------------------------------------------------------------------------------------------ */
static double dot(const double* x, const double* y, size_t n) {
  double s = 0.0;
  for (size_t i = 0; i < n; ++i) s += x[i] * y[i];
  return s;
}

int oracle_ba_pcg_solve(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, oracle_ba_pcg_info* info) {
  if (!h || max_iter < 0) return ORACLE_BA_EINVAL;
  if (!h->linearized) return ORACLE_BA_ESTATE;
  int rc = prepare_damped(h, lambda);
  if (rc) return rc;
  int nc = h->nc, np = h->np;
  size_t n = 9 * (size_t)nc;
  const double* gc = h->g;
  const double* gp = h->g + n;
  double* x = h->delta; /* delta_c */
  double* work = (double*)malloc((4 * (n ? n : 1) + 3 * (size_t)(np > 0 ? np : 1)) * sizeof(double));
  if (!work) return ORACLE_BA_ENOMEM;
  double *res = work, *z = work + n, *p = work + 2 * n, *q = work + 3 * n, *s_pts = work + 4 * n;

  /* b_j = -g_c,j + sum_{i in j} J_c,i^T J_p,i V'^-1_k g_p,k */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < np; ++k) matvec_n(3, h->Vinv + 9 * (size_t)k, gp + 3 * (size_t)k, s_pts + 3 * (size_t)k);
#pragma omp parallel for schedule(dynamic, 16)
  for (int j = 0; j < nc; ++j) {
    double* bj = h->b + 9 * (size_t)j;
    for (int a = 0; a < 9; ++a) bj[a] = -gc[9 * (size_t)j + a];
    for (int64_t e = h->cam_ptr[j]; e < h->cam_ptr[j + 1]; ++e) {
      int64_t i = h->cam_obs[e];
      const double* Jc = h->jc + 18 * i;
      const double* Jp = h->jp + 6 * i;
      const double* s = s_pts + 3 * (size_t)h->pb.point_index[i];
      double v0 = Jp[0] * s[0] + Jp[1] * s[1] + Jp[2] * s[2];
      double v1 = Jp[3] * s[0] + Jp[4] * s[1] + Jp[5] * s[2];
      for (int a = 0; a < 9; ++a) bj[a] += Jc[a] * v0 + Jc[9 + a] * v1;
    }
  }

  /* textbook PCG (Saad, Alg. 9.1), x0 = 0, M = blockdiag(U'_j) */
  memset(x, 0, n * sizeof(double));
  memcpy(res, h->b, n * sizeof(double));
  for (int j = 0; j < nc; ++j) matvec_n(9, h->Minv + 81 * (size_t)j, res + 9 * (size_t)j, z + 9 * (size_t)j);
  memcpy(p, z, n * sizeof(double));
  double bnorm = sqrt(dot(h->b, h->b, n));
  double rz = dot(res, z, n), rz0 = rz;
  int iters = 0, converged = 0, status = 0;
  double rnorm = bnorm;
  if (bnorm == 0.0) converged = 1;
  while (!converged && iters < max_iter) {
    schur_apply(h, p, q, s_pts);
    ++iters;
    double pq = dot(p, q, n);
    if (!(pq > 0.0) || !isfinite(pq)) { status = ORACLE_BA_ENUMERIC; break; } /* C15 */
    double alpha = rz / pq;
    for (size_t a = 0; a < n; ++a) { x[a] += alpha * p[a]; res[a] -= alpha * q[a]; }
    rnorm = sqrt(dot(res, res, n));
    if (rnorm <= rel_tol * bnorm) { converged = 1; break; }
    for (int j = 0; j < nc; ++j) matvec_n(9, h->Minv + 81 * (size_t)j, res + 9 * (size_t)j, z + 9 * (size_t)j);
    double rz_new = dot(res, z, n);
    double beta = rz_new / rz;
    rz = rz_new;
    for (size_t a = 0; a < n; ++a) p[a] = z[a] + beta * p[a];
  }

  /* delta_p,k = -V'^-1_k (g_p,k + sum_{i in k} J_p,i^T J_c,i delta_c,j(i)) */
  double* dp = h->delta + n;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < np; ++k) {
    double t[3] = {gp[3 * (size_t)k], gp[3 * (size_t)k + 1], gp[3 * (size_t)k + 2]};
    for (int64_t e = h->pt_ptr[k]; e < h->pt_ptr[k + 1]; ++e) {
      int64_t i = h->pt_obs[e];
      const double* Jc = h->jc + 18 * i;
      const double* Jp = h->jp + 6 * i;
      const double* dc = x + 9 * (size_t)h->pb.camera_index[i];
      double u0 = 0.0, u1 = 0.0;
      for (int a = 0; a < 9; ++a) { u0 += Jc[a] * dc[a]; u1 += Jc[9 + a] * dc[a]; }
      for (int a = 0; a < 3; ++a) t[a] += Jp[a] * u0 + Jp[3 + a] * u1;
    }
    double s[3];
    matvec_n(3, h->Vinv + 9 * (size_t)k, t, s);
    for (int a = 0; a < 3; ++a) dp[3 * (size_t)k + a] = -s[a];
  }
  h->have_delta = 1;
  if (info) {
    info->iterations = iters;
    info->converged = converged;
    info->rel_residual = bnorm > 0.0 ? rnorm / bnorm : 0.0;
    info->rz0 = rz0;
    info->rz = rz;
  }
  free(work);
  return status;
}

/* ------------------------------------------------------------------------------------------ */
/* N1: the paper's own linear solve, PCG with normal residual on the FULL system, no Schur      */
/* (PAPER.md:163 "solves the linear normal equations directly", :167-169 PCGNR loop)            */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_pcgnr_solve(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, oracle_ba_pcg_info* info) {
  if (!h || max_iter < 0) return ORACLE_BA_EINVAL;
  if (!h->linearized) return ORACLE_BA_ESTATE;
  int save = h->preconditioner;
  h->preconditioner = 0; /* one block per node: U'_j for a camera, V'_k for a point */
  if (save != 0) h->prepared = 0;
  int rc = prepare_damped(h, lambda);
  h->preconditioner = save;
  if (save != 0) h->prepared = 0; /* Minv now holds U'^-1: the next Schur solve rebuilds its own */
  if (rc) return rc;
  int nc = h->nc, np = h->np;
  size_t ncv = 9 * (size_t)nc, n = ncv + 3 * (size_t)np;
  double* x = h->delta;
  double* work = (double*)malloc(4 * (n ? n : 1) * sizeof(double));
  if (!work) return ORACLE_BA_ENOMEM;
  double *res = work, *z = work + n, *p = work + 2 * n, *q = work + 3 * n;
#define APPLY_MINV(src, dst)                                                                                      \
  do {                                                                                                            \
    for (int j = 0; j < nc; ++j) matvec_n(9, h->Minv + 81 * (size_t)j, (src) + 9 * (size_t)j, (dst) + 9 * (size_t)j); \
    for (int k = 0; k < np; ++k)                                                                                  \
      matvec_n(3, h->Vinv + 9 * (size_t)k, (src) + ncv + 3 * (size_t)k, (dst) + ncv + 3 * (size_t)k);               \
  } while (0)
  /* textbook PCG (Saad, Alg. 9.1) on A = J^T J + lambda D, right-hand side -g, x0 = 0 */
  memset(x, 0, n * sizeof(double));
  for (size_t a = 0; a < n; ++a) res[a] = -h->g[a];
  APPLY_MINV(res, z);
  memcpy(p, z, n * sizeof(double));
  double bnorm = sqrt(dot(res, res, n));
  double rz = dot(res, z, n), rz0 = rz;
  int iters = 0, converged = 0, status = 0;
  double rnorm = bnorm;
  if (bnorm == 0.0) converged = 1;
  while (!converged && iters < max_iter) {
    /* normal-residual form: w = J p per observation, then q = J^T w + lambda D p (J and J^T applied separately) */
    rc = oracle_ba_full_matvec(h, lambda, p, q);
    if (rc) { status = rc; break; }
    ++iters;
    double pq = dot(p, q, n);
    if (!(pq > 0.0) || !isfinite(pq)) { status = ORACLE_BA_ENUMERIC; break; } /* C15 */
    double alpha = rz / pq;
    for (size_t a = 0; a < n; ++a) { x[a] += alpha * p[a]; res[a] -= alpha * q[a]; }
    rnorm = sqrt(dot(res, res, n));
    if (rnorm <= rel_tol * bnorm) { converged = 1; break; }
    APPLY_MINV(res, z);
    double rz_new = dot(res, z, n);
    double beta = rz_new / rz;
    rz = rz_new;
    for (size_t a = 0; a < n; ++a) p[a] = z[a] + beta * p[a];
  }
#undef APPLY_MINV
  h->have_delta = 1;
  memset(h->b, 0, ncv * sizeof(double)); /* no Schur right-hand side on this path */
  if (info) {
    info->iterations = iters;
    info->converged = converged;
    info->rel_residual = bnorm > 0.0 ? rnorm / bnorm : 0.0;
    info->rz0 = rz0;
    info->rz = rz;
  }
  free(work);
  return status;
}

int oracle_ba_set_preconditioner(oracle_ba_t* h, int32_t mode) {
  if (!h || (mode != 0 && mode != 1)) return ORACLE_BA_EINVAL;
  if (mode != h->preconditioner) h->prepared = 0;
  h->preconditioner = mode;
  return 0;
}

int oracle_ba_set_linear_solver(oracle_ba_t* h, int32_t mode) {
  if (!h || (mode != 0 && mode != 1)) return ORACLE_BA_EINVAL;
  h->linear_solver = mode;
  return 0;
}

int oracle_ba_export_preconditioner_blocks(oracle_ba_t* h, double* dst, size_t count) {
  if (!h || !dst) return ORACLE_BA_EINVAL;
  if (!h->prepared) return ORACLE_BA_ESTATE;
  if (count != 81 * (size_t)h->nc) return ORACLE_BA_EINVAL;
  memcpy(dst, h->Pblk, count * sizeof(double));
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* O7: one LM step and the adaptive schedule (Madsen, Nielsen, Tingleff 2004, Alg. 3.16)       */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_lm_step(oracle_ba_t* h, double lambda, double rel_tol, int32_t max_iter, int32_t accept_mode,
                      oracle_ba_step_info* info) {
  if (!h || !info || accept_mode < 0 || accept_mode > 2) return ORACLE_BA_EINVAL;
  int rc = 0;
  if (!h->linearized) {
    rc = oracle_ba_linearize(h, NULL);
    if (rc) return rc;
  }
  memset(info, 0, sizeof *info);
  info->cost_before = h->cost;
  rc = h->linear_solver == 1 ? oracle_ba_pcgnr_solve(h, lambda, rel_tol, max_iter, &info->pcg)
                             : oracle_ba_pcg_solve(h, lambda, rel_tol, max_iter, &info->pcg);
  if (rc) return rc;
  int nc = h->nc, np = h->np;
  size_t ncv = 9 * (size_t)nc, npv = 3 * (size_t)np;
  double* cams = (double*)malloc((ncv ? ncv : 1) * sizeof(double));
  double* pts = (double*)malloc((npv ? npv : 1) * sizeof(double));
  if (!cams || !pts) { free(cams); free(pts); return ORACLE_BA_ENOMEM; }
  /* trial point: additive update on all 9 Nc + 3 Np parameters (reading C2); with the Pose3 camera the rotation
   * is retracted on its manifold (N3) */
  for (int j = 0; j < nc; ++j)
    oracle_ba_retract_camera(h->pb.camera_model, h->pb.cameras + 9 * (size_t)j, h->delta + 9 * (size_t)j,
                             cams + 9 * (size_t)j);
  for (size_t a = 0; a < npv; ++a) pts[a] = h->pb.points[a] + h->delta[ncv + a];
  double f_new = cost_at(h, cams, pts);
  /* model decrease L(0) - L(delta) = -delta^T g - 1/2 |J delta|^2 (valid for an inexact delta; C11) */
  double dg = dot(h->delta, h->g, ncv + npv);
  double jd2 = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : jd2)
  for (int64_t i = 0; i < h->n_obs; ++i) {
    const double* Jc = h->jc + 18 * i;
    const double* Jp = h->jp + 6 * i;
    const double* dc = h->delta + 9 * (size_t)h->pb.camera_index[i];
    const double* dp = h->delta + ncv + 3 * (size_t)h->pb.point_index[i];
    for (int row = 0; row < 2; ++row) {
      double s = 0.0;
      for (int a = 0; a < 9; ++a) s += Jc[9 * row + a] * dc[a];
      for (int a = 0; a < 3; ++a) s += Jp[3 * row + a] * dp[a];
      jd2 += s * s;
    }
  }
  info->cost_after = f_new;
  info->model_decrease = -dg - 0.5 * jd2;
  info->rho = (info->cost_before - f_new) / info->model_decrease;
  int accept;
  if (accept_mode == 1) accept = 1;
  else if (accept_mode == 2) accept = 0;
  else accept = isfinite(f_new) && info->rho > 0.0;
  info->accepted = accept;
  if (accept) {
    memcpy(h->pb.cameras, cams, ncv * sizeof(double));
    memcpy(h->pb.points, pts, npv * sizeof(double));
    h->linearized = 0;
    h->prepared = 0;
  }
  free(cams);
  free(pts);
  return 0;
}

int oracle_ba_solve(oracle_ba_t* h, int32_t iterations, double lambda0, double rel_tol, int32_t max_iter,
                    oracle_ba_step_info* infos, double* lambdas) {
  if (!h || iterations < 0 || !infos || !lambdas) return ORACLE_BA_EINVAL;
  double lambda = lambda0, nu = 2.0;
  for (int it = 0; it < iterations; ++it) {
    lambdas[it] = lambda;
    int rc = oracle_ba_lm_step(h, lambda, rel_tol, max_iter, 0, &infos[it]);
    if (rc) return rc;
    if (infos[it].accepted) {
      double c = 2.0 * infos[it].rho - 1.0;
      lambda *= fmax(1.0 / 3.0, 1.0 - c * c * c);
      nu = 2.0;
    } else {
      lambda *= nu;
      nu *= 2.0;
    }
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* export                                                                                     */
/* ------------------------------------------------------------------------------------------ */
int oracle_ba_export(oracle_ba_t* h, int32_t what, double* dst, size_t count) {
  if (!h || !dst) return ORACLE_BA_EINVAL;
  size_t N = (size_t)h->n_obs, nc = (size_t)h->nc, np = (size_t)h->np;
  const double* src = NULL;
  size_t need = 0;
  switch (what) {
    case ORACLE_BA_RESIDUALS: src = h->r; need = 2 * N; break;
    case ORACLE_BA_JC: src = h->jc; need = 18 * N; break;
    case ORACLE_BA_JP: src = h->jp; need = 6 * N; break;
    case ORACLE_BA_U: src = h->U; need = 81 * nc; break;
    case ORACLE_BA_V: src = h->V; need = 9 * np; break;
    case ORACLE_BA_G: src = h->g; need = 9 * nc + 3 * np; break;
    case ORACLE_BA_DAMPING: src = h->D; need = 9 * nc + 3 * np; break;
    case ORACLE_BA_SCHUR_RHS: src = h->b; need = 9 * nc; break;
    case ORACLE_BA_DELTA: src = h->delta; need = 9 * nc + 3 * np; break;
    default: return ORACLE_BA_EINVAL;
  }
  if (what <= ORACLE_BA_DAMPING && what != ORACLE_BA_SCHUR_RHS && what != ORACLE_BA_DELTA && !h->linearized)
    return ORACLE_BA_ESTATE;
  if ((what == ORACLE_BA_SCHUR_RHS || what == ORACLE_BA_DELTA) && !h->have_delta) return ORACLE_BA_ESTATE;
  if (count != need) return ORACLE_BA_EINVAL;
  memcpy(dst, src, need * sizeof(double));
  return 0;
}
