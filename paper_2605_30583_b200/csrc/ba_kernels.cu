// ba_kernels.cu — hand-written sm_100a kernels of the bundle-adjustment hot path (steps S1-S9).
//
// Everything here is HBM-bandwidth bound scan / gather / segmented-reduce work (about 1 flop per byte
// in the Schur matvec), so there is no tensor-core path: the design rules are coalesced 128-bit
// accesses on slot-major arrays, one observation per thread with its Jacobian in registers,
// shared-memory staging for the two segmented reductions, and one fp64 RED per (tile, camera run)
// instead of a global atomic per observation.
//
// Block-level pattern shared by linearize / Schur pass (one TILE of whole points per block):
//   * POINT side  — values are scattered to `stage[c][rank]` (rank = position in the tile's
//     point-major order, so a point's observations are contiguous there); one thread per point sums
//     its range and writes the per-point result back into the same range for the observations to read.
//   * CAMERA side — slots are already sorted by camera inside the tile, so `stage[c][slot]` holds
//     contiguous camera runs; one thread per (run, component) sums the run in fp32 and issues ONE
//     fp64 atomic add to the L2-resident per-camera accumulator (cross-tile accumulation in fp64).
#include <math_constants.h>

#include <cstdlib>
#include <mutex>

#include "ba_internal.h"

namespace cba {

static thread_local long long g_launches = 0;
long long take_launch_count() {
  long long n = g_launches;
  g_launches = 0;
  return n;
}
#define CBA_LAUNCHED() (++g_launches, cudaGetLastError())

// ------------------------------------------------------------------------------------------------
// reductions
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum over the block; the result is valid in thread 0.  `red` holds >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double* red) {
  v = warp_sum(v);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) red[w] = v;
  __syncthreads();
  if (w == 0) {
    v = (lane < (int)(blockDim.x >> 5)) ? red[lane] : 0.0;
    v = warp_sum(v);
  }
  return v;
}

// ------------------------------------------------------------------------------------------------
// mbarrier / TMA bulk-copy / named-barrier wrappers (inline PTX) shared by the two persistent kernels
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar,
                                         unsigned long long policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// A consumer that has read a stage with ordinary (generic-proxy) shared-memory loads must order those reads before
// the bulk copy (async proxy) that refills the stage: the release of mbarrier.arrive alone does not reach across
// proxies.  Without this fence a warp whose gathered loads were still queued when its lane 0 arrived on the `empty`
// barrier read a few rows of the NEXT tile's points about once in 10^7 warp-tiles (measured on the skewed scene:
// 22 of 400 linearize calls had one warp of wrong residuals).  Every reading thread executes it.
__device__ __forceinline__ void fence_reads_before_refill() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void group_bar(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

constexpr int kMaxStages = 12;

// The persistent kernels hand out tiles in CHUNKS of C consecutive tiles, chunk c to CTA c mod G, so the i-th tile of CTA b
// is ((i / C) G + b) C + i mod C.  Consecutive tiles share cameras (points are ordered by camera id): the p_j rows / camera-
// table rows that the groups of a CTA gather repeat from one tile to the next, while the round-robin over chunks keeps the
// CTAs balanced.  Measured (matvec / linearize, ms): Large C = 1 0.648 / 0.744, C = 3 0.641 / 0.723, C = 6 0.637 / 0.720,
// C = 12 0.636 / 0.722, one contiguous range per CTA 0.636 / 0.719; Mid 0.1270 / 0.1355, 0.1264 / 0.1331, 0.1265 / 0.1340,
// 0.1275 / 0.1380, 0.1298 / 0.1305; Skewed, whose tiles differ (hot cameras, long tracks) and whose first tiles hold the
// hottest cameras, 0.577 / 0.616, 0.583 / 0.616, 0.586 / 0.619, 0.592 / 0.625, 0.612 / 0.814.  Hence C = 6 on scenes without
// hot cameras that have at least four chunks per CTA, else C = 1 (tile i G + b: the CTAs interleave tile by tile).
__device__ __forceinline__ int tile_chunk(const View& v, int G) { return (v.num_hot == 0 && v.num_tiles >= 24 * G) ? 6 : 1; }

// ------------------------------------------------------------------------------------------------
// S0 helpers: gather the caller's observations into slot order; pack / unpack points
// ------------------------------------------------------------------------------------------------
__global__ void gather_observations_kernel(View v, const float* __restrict__ observations, float2* __restrict__ px) {
  long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= v.n_slots) return;
  int o = v.obs_of_slot[s];
  px[s] = o >= 0 ? reinterpret_cast<const float2*>(observations)[o] : make_float2(0.f, 0.f);
}

__global__ void pack_points_kernel(View v, const float* __restrict__ src, float4* __restrict__ dst) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= v.np) return;
  const float* p = src + 3ll * v.pt_perm[k];
  dst[k] = make_float4(p[0], p[1], p[2], 0.f);
}

__global__ void unpack_points_kernel(View v, const float4* __restrict__ src, float* __restrict__ dst) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= v.np) return;
  float4 p = src[k];
  float* d = dst + 3ll * v.pt_perm[k];
  d[0] = p.x; d[1] = p.y; d[2] = p.z;
}

// ------------------------------------------------------------------------------------------------
// S1 camera prepass: everything that depends on the camera alone, once per camera, in fp64.
// Table row (144 B = 9 x 16 B):  double R[9] | double C[3] | float f k1 k2 th2 | w0 w1 w2 a | b a1 b1 pad
// with C = -R^T t the camera centre, so that P = R (X - C) is evaluated without the cancellation of
// R X + t for scenes far from the origin.  R and C stay in fp64 because the residual is evaluated in
// fp64 (C12: fp32 cannot resolve uv - pixel to 1e-5 relative); the Jacobian path rounds them.
// ------------------------------------------------------------------------------------------------
__global__ void camera_prepass_kernel(int nc, const float* __restrict__ cams, float* __restrict__ table) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nc) return;
  const float* c = cams + 9ll * j;
  const double w0 = c[0], w1 = c[1], w2 = c[2], t0 = c[3], t1 = c[4], t2 = c[5];
  const double th2 = w0 * w0 + w1 * w1 + w2 * w2;
  double a, b, a1, b1;
  if (th2 < 1e-3) {  // Taylor series in th2 (5 terms: truncation below 1e-17 here)
    a = 1.0 + th2 * (-1.0 / 6 + th2 * (1.0 / 120 + th2 * (-1.0 / 5040 + th2 * (1.0 / 362880))));
    b = 0.5 + th2 * (-1.0 / 24 + th2 * (1.0 / 720 + th2 * (-1.0 / 40320 + th2 * (1.0 / 3628800))));
    a1 = -1.0 / 3 + th2 * (1.0 / 30 + th2 * (-1.0 / 840 + th2 * (1.0 / 45360 + th2 * (-1.0 / 3991680))));
    b1 = -1.0 / 12 + th2 * (1.0 / 180 + th2 * (-1.0 / 6720 + th2 * (1.0 / 453600 + th2 * (-1.0 / 47900160))));
  } else {
    const double th = sqrt(th2);
    double sn, cs;
    sincos(th, &sn, &cs);
    const double omc = 2.0 * sin(0.5 * th) * sin(0.5 * th);  // 1 - cos(th) without cancellation
    a = sn / th;
    b = omc / th2;
    a1 = (th * cs - sn) / (th2 * th);
    b1 = (th * sn - 2.0 * omc) / (th2 * th2);
  }
  // R = I + a [w]x + b (w w^T - th2 I)
  double R[9];
  R[0] = 1.0 + b * (w0 * w0 - th2); R[1] = -a * w2 + b * w0 * w1;     R[2] = a * w1 + b * w0 * w2;
  R[3] = a * w2 + b * w1 * w0;      R[4] = 1.0 + b * (w1 * w1 - th2); R[5] = -a * w0 + b * w1 * w2;
  R[6] = -a * w1 + b * w2 * w0;     R[7] = a * w0 + b * w2 * w1;      R[8] = 1.0 + b * (w2 * w2 - th2);
  float* o = table + (long long)kCamTableFloats * j;
  double* od = reinterpret_cast<double*>(o);
#pragma unroll
  for (int i = 0; i < 9; ++i) od[i] = R[i];
  od[9] = -(R[0] * t0 + R[3] * t1 + R[6] * t2);
  od[10] = -(R[1] * t0 + R[4] * t1 + R[7] * t2);
  od[11] = -(R[2] * t0 + R[5] * t1 + R[8] * t2);
  o[24] = c[6]; o[25] = c[7]; o[26] = c[8]; o[27] = (float)th2;
  o[28] = c[0]; o[29] = c[1]; o[30] = c[2]; o[31] = (float)a;
  o[32] = (float)b; o[33] = (float)a1; o[34] = (float)b1; o[35] = 0.f;
}

// ------------------------------------------------------------------------------------------------
// S2 per-observation arithmetic (registers only).  PAPER.md:194-203; O1/O2.
// The projection and the residual are evaluated in fp64 from the fp64 R, C of the camera table
// (about 35 fp64 instructions per observation, hidden under the HBM bound); everything the Jacobian
// needs is rounded to fp32 once.
// ------------------------------------------------------------------------------------------------
struct Projection {
  float px, py, n, rad, inz;  // p, |p|^2, radial factor, -1/d_safe
  double r0, r1;              // residual, fp64: a trial point can throw a two-view point far enough for |r|^2 to
                              // overflow fp32, while the Cauchy cost of that observation is a few hundred
  float R[9];                         // rotation rounded to fp32 (J_p = A R)
};

// depth_eps: d_safe = d + eps sign_no_zero(d); 0 = the unguarded north_star model (C7).
__device__ __forceinline__ Projection project(const float4* __restrict__ row, float f, float k1, float k2, float X0,
                                              float X1, float X2, float2 m, float depth_eps) {
  const double2* rd = reinterpret_cast<const double2*>(row);
  const double2 a0 = __ldg(rd + 0), a1 = __ldg(rd + 1), a2 = __ldg(rd + 2), a3 = __ldg(rd + 3);
  const double2 a4 = __ldg(rd + 4), a5 = __ldg(rd + 5);  // R0 R1 | R2 R3 | R4 R5 | R6 R7 | R8 C0 | C1 C2
  const double d0 = (double)X0 - a4.y, d1 = (double)X1 - a5.x, d2 = (double)X2 - a5.y;
  const double P0 = fma(a0.x, d0, fma(a0.y, d1, a1.x * d2));
  const double P1 = fma(a1.y, d0, fma(a2.x, d1, a2.y * d2));
  const double P2 = fma(a3.x, d0, fma(a3.y, d1, a4.x * d2));
  const double d_safe = P2 + (P2 >= 0.0 ? (double)depth_eps : -(double)depth_eps);
  const double inz = -1.0 / d_safe;  // one shared reciprocal
  const double px = P0 * inz, py = P1 * inz;
  const double n = fma(px, px, py * py);
  const double rad = fma(n, fma((double)k2, n, (double)k1), 1.0);
  const double fr = (double)f * rad;
  Projection o;
  o.r0 = fma(fr, px, -(double)m.x);
  o.r1 = fma(fr, py, -(double)m.y);
  o.px = (float)px; o.py = (float)py; o.n = (float)n; o.rad = (float)rad; o.inz = (float)inz;
  o.R[0] = (float)a0.x; o.R[1] = (float)a0.y; o.R[2] = (float)a1.x;
  o.R[3] = (float)a1.y; o.R[4] = (float)a2.x; o.R[5] = (float)a2.y;
  o.R[6] = (float)a3.x; o.R[7] = (float)a3.y; o.R[8] = (float)a4.x;
  return o;
}

// Full linearization of one observation: J[0..17] = d r / d camera (2x9 row-major), J[18..23] = d r / d point.
// camera_model 1 (the paper's Pose3 camera): the rotation columns are the derivative with
// respect to the right perturbation R Exp(d) at d = 0, d(R Exp(d) X)/dd = -R [X]x, so J_w = -J_p [X]x = X x J_p(row).
__device__ __forceinline__ void linearize_observation(const float* __restrict__ table, int cam, float X0, float X1,
                                                      float X2, float2 m, int camera_model, float depth_eps,
                                                      float (&J)[24], double& r0, double& r1) {
  const float4* row = reinterpret_cast<const float4*>(table) + 9ll * cam;
  const float4 t6 = __ldg(row + 6), t7 = __ldg(row + 7), t8 = __ldg(row + 8);
  const float f = t6.x, k1 = t6.y, k2 = t6.z, th2 = t6.w;
  const float w0 = t7.x, w1 = t7.y, w2 = t7.z, a = t7.w;
  const float b = t8.x, a1 = t8.y, b1 = t8.z;
  const Projection pr = project(row, f, k1, k2, X0, X1, X2, m, depth_eps);
  r0 = pr.r0;
  r1 = pr.r1;
  const float px = pr.px, py = pr.py, n = pr.n, rad = pr.rad, inz = pr.inz;
  // d uv / d p = f (rad I + c p p^T), c = 2 k1 + 4 k2 n;  d p / d P = inz [[1, 0, px], [0, 1, py]]
  const float fc = f * fmaf(4.0f * k2, n, 2.0f * k1);
  const float fr = f * rad;
  const float D00 = fmaf(fc * px, px, fr), D01 = fc * px * py, D11 = fmaf(fc * py, py, fr);
  const float A00 = inz * D00, A01 = inz * D01, A02 = inz * fmaf(D00, px, D01 * py);
  const float A10 = A01, A11 = inz * D11, A12 = inz * fmaf(D01, px, D11 * py);
  // J_p = A R
  const float* R = pr.R;
  J[18] = fmaf(A00, R[0], fmaf(A01, R[3], A02 * R[6]));
  J[19] = fmaf(A00, R[1], fmaf(A01, R[4], A02 * R[7]));
  J[20] = fmaf(A00, R[2], fmaf(A01, R[5], A02 * R[8]));
  J[21] = fmaf(A10, R[0], fmaf(A11, R[3], A12 * R[6]));
  J[22] = fmaf(A10, R[1], fmaf(A11, R[4], A12 * R[7]));
  J[23] = fmaf(A10, R[2], fmaf(A11, R[5], A12 * R[8]));
  J[3] = A00; J[4] = A01; J[5] = A02;
  J[6] = rad * px;
  const float fn = f * n;
  J[7] = fn * px;
  J[8] = fn * n * px;
  J[12] = A10; J[13] = A11; J[14] = A12;
  J[15] = rad * py;
  J[16] = fn * py;
  J[17] = fn * n * py;
  if (camera_model == 1) {  // tangent-space rotation block: X x J_p(row)
    J[0] = X1 * J[20] - X2 * J[19];
    J[1] = X2 * J[18] - X0 * J[20];
    J[2] = X0 * J[19] - X1 * J[18];
    J[9] = X1 * J[23] - X2 * J[22];
    J[10] = X2 * J[21] - X0 * J[23];
    J[11] = X0 * J[22] - X1 * J[21];
    return;
  }
  // d(R X)/d w = u w^T + b w X^T + b s I - a [X]x,  u = a1 q + b1 (w s - th2 X) - 2 b X,  q = w x X, s = w.X
  const float q0 = w1 * X2 - w2 * X1, q1 = w2 * X0 - w0 * X2, q2 = w0 * X1 - w1 * X0;
  const float s = fmaf(w0, X0, fmaf(w1, X1, w2 * X2));
  const float bs = b * s;
  const float u0 = fmaf(a1, q0, fmaf(b1, fmaf(w0, s, -th2 * X0), -2.0f * b * X0));
  const float u1 = fmaf(a1, q1, fmaf(b1, fmaf(w1, s, -th2 * X1), -2.0f * b * X1));
  const float u2 = fmaf(a1, q2, fmaf(b1, fmaf(w2, s, -th2 * X2), -2.0f * b * X2));
  const float bw0 = b * w0, bw1 = b * w1, bw2 = b * w2;
  const float aX0 = a * X0, aX1 = a * X1, aX2 = a * X2;
  // G[i][j] = u_i w_j + bw_i X_j + bs delta_ij - a [X]x_ij   with [X]x = [[0,-X2,X1],[X2,0,-X0],[-X1,X0,0]]
  const float G00 = fmaf(u0, w0, fmaf(bw0, X0, bs)), G01 = fmaf(u0, w1, fmaf(bw0, X1, aX2)), G02 = fmaf(u0, w2, fmaf(bw0, X2, -aX1));
  const float G10 = fmaf(u1, w0, fmaf(bw1, X0, -aX2)), G11 = fmaf(u1, w1, fmaf(bw1, X1, bs)), G12 = fmaf(u1, w2, fmaf(bw1, X2, aX0));
  const float G20 = fmaf(u2, w0, fmaf(bw2, X0, aX1)), G21 = fmaf(u2, w1, fmaf(bw2, X1, -aX0)), G22 = fmaf(u2, w2, fmaf(bw2, X2, bs));
  J[0] = fmaf(A00, G00, fmaf(A01, G10, A02 * G20));
  J[1] = fmaf(A00, G01, fmaf(A01, G11, A02 * G21));
  J[2] = fmaf(A00, G02, fmaf(A01, G12, A02 * G22));
  J[9] = fmaf(A10, G00, fmaf(A11, G10, A12 * G20));
  J[10] = fmaf(A10, G01, fmaf(A11, G11, A12 * G21));
  J[11] = fmaf(A10, G02, fmaf(A11, G12, A12 * G22));
}

__device__ __forceinline__ void residual_observation(const float* __restrict__ table, int cam, float X0, float X1,
                                                     float X2, float2 m, float depth_eps, double& r0, double& r1) {
  const float4* row = reinterpret_cast<const float4*>(table) + 9ll * cam;
  const float4 t6 = __ldg(row + 6);
  const Projection pr = project(row, t6.x, t6.y, t6.z, X0, X1, X2, m, depth_eps);
  r0 = pr.r0;
  r1 = pr.r1;
}

// rho(s) of one observation and, with the Cauchy loss, sqrt(w) = (1 + s/c^2)^-1/2 ("robust loss";
// SURVEY.md O3).  s arrives in fp64; the fp32 fast path covers s/c^2 < 1e30, beyond it (a point thrown to infinity
// by a trial step) everything is evaluated in fp64 and the Jacobian of that observation, whose weight is < 1e-30,
// is dropped.
struct LossTerm {
  double rho;
  float sw;    // sqrt(w), 1 without a robust loss
  bool wild;   // s/c^2 >= 1e30
};

__device__ __forceinline__ LossTerm loss_term(const View& v, double s2) {
  LossTerm t;
  t.rho = s2;
  t.sw = 1.0f;
  t.wild = false;
  if (v.robust) {
    const double q = s2 * v.robust_inv_c2;
    if (q < 1e30) {
      const float qf = (float)q;
      t.rho = (double)(v.robust_c2 * log1pf(qf));
      t.sw = sqrtf(1.0f / (1.0f + qf));
    } else {
      t.rho = (double)v.robust_c2 * log1p(q);
      t.sw = (float)rsqrt(1.0 + q);
      t.wild = true;
    }
  }
  return t;
}

constexpr int blocks_per_sm(int T) { return T == 128 ? 6 : (T == 192 ? 4 : (T == 256 ? 3 : (T == 512 ? 2 : 1))); }

// ------------------------------------------------------------------------------------------------
// S2 + S3 (JAC = true): linearize every observation, store r and J, assemble V_k and g_p,k per point,
//                       accumulate the cost.
// S9      (JAC = false): residual-only cost at the given points / camera table.
// One block per tile, one thread per observation.  The observation finds its point through the slot's
// local point id (X_k is a 16-byte read from the tile's contiguous, L1-resident point range), so the only
// block-wide step is the point-side reduction: the nine products V (6) and g_p (3) are scattered to the
// point-major staging rows, and after ONE barrier lane (point, component) sums its range: three points
// per warp and pass.
// ------------------------------------------------------------------------------------------------
template <int T>
__device__ __forceinline__ void slot_rank_pid(const View& v, long long slot, unsigned& rank, unsigned& pid) {
  if (T <= 256) {
    const unsigned rp = v.rankpid[slot];
    rank = rp & 255u;
    pid = rp >> 8;
  } else {
    const unsigned rp = v.rankpid32[slot];
    rank = rp & 0xffffu;
    pid = rp >> 16;
  }
}

// Thread `first + i` prefetches the i-th 128-byte line of [ptr, ptr + bytes) into L2; returns the next free thread.
__device__ __forceinline__ int prefetch_lines(const void* ptr, long long bytes, int first, int tid) {
  const char* p = reinterpret_cast<const char*>(ptr);
  const char* line = reinterpret_cast<const char*>(reinterpret_cast<unsigned long long>(p) & ~127ull);
  const int lines = (int)((p + bytes - line + 127) >> 7);
  const int i = tid - first;
  if (bytes > 0 && i >= 0 && i < lines) asm volatile("prefetch.global.L2 [%0];" ::"l"(line + 128ll * i));
  return first + lines;
}

template <int T, bool JAC>
__global__ void __launch_bounds__(T, 1024 / T)
linearize_kernel(View v, const float4* __restrict__ pts, const float* __restrict__ table) {
  __shared__ float4 stage[JAC ? T : 1][2];  // by rank: (Vxx Vxy Vxz Vyy) (Vyz Vzz gx gy)
  __shared__ float stage_gz[JAC ? T : 1];   // by rank: gz
  __shared__ int arrived[JAC ? T : 1];      // by local point id: observations staged so far
  const int t = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  const long long slot = (long long)t * T + tid;
  const int p0 = v.tile_pt[t];
  const int cam = v.cam[slot];
  unsigned rank, pid;
  slot_rank_pid<T>(v, slot, rank, pid);
  const float2 m = v.px[slot];
  // Every block's critical path starts with two dependent levels of DRAM latency (slot arrays, then the point
  // and rank-range gathers they address).  The block therefore pulls the inputs of the tile that will run one
  // resident wave later (1024 / T blocks per SM) into L2: slot arrays now, points below.
  const int tn = t + (1024 / T) * v.num_sms;
  const bool prefetcher = tid < 64 && tn < v.num_tiles;  // two warps issue the (at most ~40) line prefetches
  int np0 = 0, np1 = 0, next_thread = 0;
  if (prefetcher) {
    np0 = __ldg(v.tile_pt + tn);
    np1 = __ldg(v.tile_pt + tn + 1);
    const long long sn = (long long)tn * T;
    next_thread = prefetch_lines(v.cam + sn, T * 4, 0, tid);
    next_thread = prefetch_lines(v.px + sn, T * 8, next_thread, tid);
    next_thread = T <= 256 ? prefetch_lines(v.rankpid + sn, T * 2, next_thread, tid)
                           : prefetch_lines(v.rankpid32 + sn, T * 4, next_thread, tid);
  }
  float4 X = make_float4(0.f, 0.f, 0.f, 0.f);
  int rb = 0, re = 0;  // rank range of this observation's point
  if (cam >= 0) {
    X = __ldg(pts + p0 + pid);
    if (JAC) {
      const int base = __ldg(v.pt_ptr + p0);
      rb = __ldg(v.pt_ptr + p0 + pid) - base;
      re = __ldg(v.pt_ptr + p0 + pid + 1) - base;
    }
  }
  if (JAC) {
    arrived[tid] = 0;
    __syncthreads();  // the only block-wide barrier: at the start, before anything has latency to expose
  }

  double term = 0.0;
  if (JAC) {
    float J[24], r0 = 0.f, r1 = 0.f;
#pragma unroll
    for (int i = 0; i < 24; ++i) J[i] = 0.f;
    if (cam >= 0) {
      double rd0, rd1;
      linearize_observation(table, cam, X.x, X.y, X.z, m, v.camera_model, v.depth_eps, J, rd0, rd1);
      const LossTerm lt = loss_term(v, fma(rd0, rd0, rd1 * rd1));
      term = lt.rho;
      r0 = (float)rd0; r1 = (float)rd1;
      if (v.robust) {  // Cauchy: w = 1 / (1 + s/c^2), r~ = sqrt(w) r, J~ = sqrt(w) J
        if (!lt.wild) {
          r0 *= lt.sw; r1 *= lt.sw;
#pragma unroll
          for (int i = 0; i < 24; ++i) J[i] *= lt.sw;
        } else {
          r0 = (float)(rd0 * (double)lt.sw); r1 = (float)(rd1 * (double)lt.sw);
#pragma unroll
          for (int i = 0; i < 24; ++i) J[i] = 0.f;
        }
      }
    }
    // eager stores: six 128-bit chunk arrays + the residual, streamed past L2's keep set
#pragma unroll
    for (int c = 0; c < 6; ++c) __stcs(&v.J[c][slot], make_float4(J[4 * c], J[4 * c + 1], J[4 * c + 2], J[4 * c + 3]));
    __stcs(&v.res[slot], make_float2(r0, r1));
    // Point side without a barrier: every observation stages its nine products at its rank, then counts
    // itself in; the observation that completes its point sums the point's rank range IN RANK ORDER (so
    // V_k and g_p,k do not depend on the arrival order) and writes the point's blocks.
    if (cam >= 0) {
      stage[rank][0] = make_float4(fmaf(J[18], J[18], J[21] * J[21]), fmaf(J[18], J[19], J[21] * J[22]),
                                   fmaf(J[18], J[20], J[21] * J[23]), fmaf(J[19], J[19], J[22] * J[22]));
      stage[rank][1] = make_float4(fmaf(J[19], J[20], J[22] * J[23]), fmaf(J[20], J[20], J[23] * J[23]),
                                   fmaf(J[18], r0, J[21] * r1), fmaf(J[19], r0, J[22] * r1));
      stage_gz[rank] = fmaf(J[20], r0, J[23] * r1);
      __threadfence_block();
      if (atomicAdd(&arrived[pid], 1) == re - rb - 1) {
        __threadfence_block();
        float2 a0 = make_float2(0.f, 0.f), a1 = a0, b0 = a0, b1 = a0;
        float gz = 0.f;
        for (int r = rb; r < re; ++r) {  // packed fp32 adds (FADD2)
          const float4 x = stage[r][0], y = stage[r][1];
          const float z = stage_gz[r];
          a0 = __fadd2_rn(a0, make_float2(x.x, x.y));
          a1 = __fadd2_rn(a1, make_float2(x.z, x.w));
          b0 = __fadd2_rn(b0, make_float2(y.x, y.y));
          b1 = __fadd2_rn(b1, make_float2(y.z, y.w));
          gz += z;
        }
        v.V0[p0 + pid] = make_float4(a0.x, a0.y, a1.x, a1.y);
        v.V1[p0 + pid] = b0;
        v.gp[p0 + pid] = make_float4(b1.x, b1.y, gz, 0.f);
      }
    }
  } else {
    if (cam >= 0) {
      double r0, r1;
      residual_observation(table, cam, X.x, X.y, X.z, m, v.depth_eps, r0, r1);
      term = loss_term(v, fma(r0, r0, r1 * r1)).rho;
    }
  }
  if (prefetcher) {  // the next wave's points and rank ranges (their tile bounds have long arrived)
    next_thread = prefetch_lines(pts + np0, 16ll * (np1 - np0), next_thread % 64, tid);
    if (JAC) prefetch_lines(v.pt_ptr + np0, 4ll * (np1 - np0 + 1), next_thread % 64, tid);
  }
  const double wsum = warp_sum(term);
  if (lane == 0) v.cost_warp[(long long)t * (T / 32) + (tid >> 5)] = wsum;  // folded by reduce_cost_kernel
}

// ------------------------------------------------------------------------------------------------
// S2 + S3, pipelined: the same per-observation work as linearize_kernel in a PERSISTENT kernel, one CTA per
// SM, for tiles of <= 256 slots (the default).  (Only JAC = true is launched.  The residual-only cost pass S9 stays
// on linearize_kernel<T, false>: it has a quarter of the instructions and nothing to overlap them with, so it wants
// the 40 resident warps of five small blocks, not the 24 of one 800-thread CTA: 0.32 ms against 0.42 ms measured.)  linearize_kernel opens every block with two dependent levels of
// global-memory latency (slot arrays, then the gathers they address) and ends with its stores draining; ncu
// (profiles/r01_ncu_linearize.md) showed 4.4 long-scoreboard + 1.0 drain stall cycles per issued instruction at
// 0.55 of the HBM roofline with clean traffic.  Here
//   producer warp : one lane streams each tile's inputs (camera ids, pixels, rank | point id, the tile's contiguous
//                   point range, the rank range of each point) into a ring of shared-memory stages with TMA bulk
//                   copies, several tiles ahead of the consumers;
//   consumer groups: NG groups of T threads, each on its own tile: inputs come from shared memory, the stage is
//                   released as soon as they are in registers, the camera row is gathered through L1/L2, the 24
//                   Jacobian floats leave as streaming 128-bit stores that nothing waits for (no block exit).
// Point side as in linearize_kernel (rank-ordered sum by the observation that completes its point), with
// self-resetting counters (atomicInc wraps at the track length).  The staging rows are double buffered and their
// reuse is ordered by an mbarrier per buffer (each warp arrives when it is done with a tile, and waits for the
// buffer's previous use just before it writes its rows two tiles later): a split barrier, so a warp never waits
// for the others to reach the same point, only for work that is two tiles old.  A full group barrier per tile
// cost 21 % of the stall samples (the group waits for its slowest warp, the one with most points to sum).  Cost: per-thread fp64 accumulation
// over the thread's tiles (a fixed order), one partial per warp, folded by reduce_cost_kernel.
// ------------------------------------------------------------------------------------------------
struct LinLayout {  // byte offsets inside one stage / inside the dynamic shared memory
  int cam, px, rank, pts, meta, stage_bytes;
  int stages, sbuf, sbuf_bytes, bars, total;
};

__host__ __device__ inline LinLayout lin_layout(int T, int NG, int max_pts, int meta_max, bool jac, int smem_limit) {
  LinLayout L;
  auto up = [](int x) { return (x + 127) & ~127; };
  L.cam = 0;
  L.px = L.cam + T * 4;
  L.rank = L.px + T * 8;
  L.pts = up(L.rank + T * 2);
  L.meta = up(L.pts + max_pts * 16);
  L.stage_bytes = up(L.meta + (jac ? meta_max : 0));
  L.sbuf_bytes = jac ? 2 * up(T * 40) : 0;  // per group, x2 buffers: float4 stage[T][2], float gz[T], unsigned arrived[T]
  const int fixed = NG * L.sbuf_bytes + 512;  // 512: full[12], empty[12], seen[12], done[2 NG]
  int st = (smem_limit - fixed) / L.stage_bytes;
  const int cap = NG == 3 ? 9 : 2 * NG;  // 8 - 12 tiles of inputs (<= 55 KB at T = 256) in flight per SM: far more than the consumers drain
  if (st > cap) st = cap;
  if (st >= NG) st -= st % NG;  // a multiple of NG: every stage belongs to one group, no `seen` guard (see the matvec)
  L.stages = st;
  L.sbuf = L.stages * L.stage_bytes;
  L.bars = L.sbuf + NG * L.sbuf_bytes;
  L.total = L.bars + 512;
  return L;
}

template <int T, int NG, bool JAC>
__global__ void __launch_bounds__(NG * T + 32, 1)
linearize_pipelined_kernel(View v, const float4* __restrict__ pts, const float* __restrict__ table, LinLayout L) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + L.bars);
  unsigned long long* empty = full + kMaxStages;
  volatile int* seen = reinterpret_cast<volatile int*>(empty + kMaxStages);  // see schur_matvec_pipelined_kernel
  unsigned long long* done = reinterpret_cast<unsigned long long*>(const_cast<int*>(seen) + kMaxStages);  // [NG][2]
  if (tid == 0) {
    for (int s = 0; s < L.stages; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, T / 32);  // one group consumes a stage
      seen[s] = 0;
    }
    for (int i = 0; i < 2 * NG; ++i) mbar_init(done + i, T / 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (JAC)  // per-point arrival counters of every group and buffer start at 0 and reset themselves (atomicInc wraps)
    for (int i = tid; i < 2 * NG * T; i += NG * T + 32)
      reinterpret_cast<unsigned*>(smem + L.sbuf + (size_t)(i / T) * (L.sbuf_bytes / 2) + T * 36)[i % T] = 0u;
  __syncthreads();
  const int G = gridDim.x;

  if (tid >= NG * T) {
    // ===== producer warp: one lane issues every copy =====
    if (tid == NG * T) {
      unsigned long long pol_stream;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
      int s = 0;
      unsigned ph = 0;
      const int C = tile_chunk(v, G);
      int t = blockIdx.x * C, within = 0;
      int4 d = t < v.num_tiles ? __ldg(v.tile_dir + t) : make_int4(0, 0, 0, 0);
      for (; t < v.num_tiles;) {
        const bool wrap = within + 1 == C;
        const int tn = wrap ? t + 1 + (G - 1) * C : t + 1;
        const int4 dn = tn < v.num_tiles ? __ldg(v.tile_dir + tn) : make_int4(0, 0, 0, 0);  // prefetch next entry
        mbar_wait(empty + s, ph ^ 1);
        unsigned char* st = smem + (size_t)s * L.stage_bytes;
        const unsigned pts_bytes = (unsigned)d.w * 16u;
        // the blob's first 16 + 2 (npts + 1) bytes, rounded up to 16: header and the rank range of each point
        // the WHOLE blob, not just its head (header + rank ranges, ~100 bytes): a bulk copy that small is a slow path of
        // the copy engine (measured: 0.773 -> 0.746 ms on Large; the same in the Schur matvec)
        const unsigned meta_bytes = JAC ? (unsigned)d.y : 0u;
        mbar_expect_tx(full + s, (unsigned)(T * 4 + T * 8 + T * 2) + pts_bytes + meta_bytes);
        const long long slot0 = (long long)t * T;
        bulk_g2s(st + L.cam, v.cam + slot0, T * 4, full + s, pol_stream);
        bulk_g2s(st + L.px, v.px + slot0, T * 8, full + s, pol_stream);
        bulk_g2s(st + L.rank, v.rankpid + slot0, T * 2, full + s, pol_stream);
        bulk_g2s(st + L.pts, pts + d.z, pts_bytes, full + s, pol_stream);
        if (JAC) bulk_g2s(st + L.meta, v.tile_meta + 16ll * d.x, meta_bytes, full + s, pol_stream);
        d = dn;
        t = tn;
        within = wrap ? 0 : within + 1;
        if (++s == L.stages) { s = 0; ph ^= 1; }
      }
    }
    return;
  }

  // ===== consumers: group g takes every NG-th tile of this CTA's sequence =====
  const int g = tid / T, gt = tid - g * T;
  double cost_acc = 0.0;
  int s = g % L.stages;
  int round = g / L.stages;
  int k = 0;  // tiles this group has done
  const bool guard = (L.stages % NG) != 0;
  const int C = tile_chunk(v, G);
  int t = blockIdx.x * C + g, within = g;  // this group's first tile: the g-th of the CTA's sequence
  while (within >= C) { within -= C; t += (G - 1) * C; }
  for (; t < v.num_tiles; ++k) {
    unsigned char* sb = smem + L.sbuf + (size_t)(2 * g + (k & 1)) * (L.sbuf_bytes / 2);  // this tile's buffer
    // by rank, two arrays of 16-byte rows (one array of 32-byte rows put rows r and r + 4 on the same banks):
    float4* stage_a = reinterpret_cast<float4*>(sb);                // (Vxx Vxy Vxz Vyy)
    float4* stage_b = reinterpret_cast<float4*>(sb + T * 16);       // (Vyz Vzz gx gy)
    float* stage_gz = reinterpret_cast<float*>(sb + T * 32);        // by rank: gz
    unsigned* arrived = reinterpret_cast<unsigned*>(sb + T * 36);   // by local point id
    if (guard)
      while (seen[s] < round) {
      }
    mbar_wait(full + s, (unsigned)(round & 1));
    if (guard && gt == 0) seen[s] = round + 1;
    const unsigned char* st = smem + (size_t)s * L.stage_bytes;
    const int cam = reinterpret_cast<const int*>(st + L.cam)[gt];
    const unsigned rp = reinterpret_cast<const unsigned short*>(st + L.rank)[gt];
    const unsigned rank = rp & 255u, pid = rp >> 8;
    const float2 m = reinterpret_cast<const float2*>(st + L.px)[gt];
    float4 X = make_float4(0.f, 0.f, 0.f, 0.f);
    int rb = 0, re = 0;  // rank range of this observation's point
    int p0 = 0;
    if (cam >= 0) {
      X = reinterpret_cast<const float4*>(st + L.pts)[pid];
      if (JAC) {
        const unsigned short* pt_start = reinterpret_cast<const unsigned short*>(st + L.meta + 16);
        rb = pt_start[pid];
        re = pt_start[pid + 1];
        p0 = reinterpret_cast<const int*>(st + L.meta)[3];
      }
    }
    // everything this thread needs from the stage has been read (not necessarily returned: X and the rank range
    // are first used far below), so the reads are fenced against the refill before the stage is handed back
    fence_reads_before_refill();
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty + s);
    const long long slot = (long long)t * T + gt;
    double term = 0.0;
    if (JAC) {
      float J[24], r0 = 0.f, r1 = 0.f;
#pragma unroll
      for (int i = 0; i < 24; ++i) J[i] = 0.f;
      if (cam >= 0) {
        double rd0, rd1;
        linearize_observation(table, cam, X.x, X.y, X.z, m, v.camera_model, v.depth_eps, J, rd0, rd1);
        const LossTerm lt = loss_term(v, fma(rd0, rd0, rd1 * rd1));
        term = lt.rho;
        r0 = (float)rd0; r1 = (float)rd1;
        if (v.robust) {  // Cauchy: w = 1 / (1 + s/c^2), r~ = sqrt(w) r, J~ = sqrt(w) J
          if (!lt.wild) {
            r0 *= lt.sw; r1 *= lt.sw;
#pragma unroll
            for (int i = 0; i < 24; ++i) J[i] *= lt.sw;
          } else {
            r0 = (float)(rd0 * (double)lt.sw); r1 = (float)(rd1 * (double)lt.sw);
#pragma unroll
            for (int i = 0; i < 24; ++i) J[i] = 0.f;
          }
        }
      }
      // eager stores: six 128-bit chunk arrays + the residual, streamed past L2's keep set
#pragma unroll
      for (int c = 0; c < 6; ++c) __stcs(&v.J[c][slot], make_float4(J[4 * c], J[4 * c + 1], J[4 * c + 2], J[4 * c + 3]));
      __stcs(&v.res[slot], make_float2(r0, r1));
      // every warp of the group is done with this buffer's previous use (two tiles ago)
      unsigned long long* buf_done = done + 2 * g + (k & 1);
      if (k >= 2) mbar_wait(buf_done, (unsigned)(((k >> 1) - 1) & 1));
      if (cam >= 0) {
        stage_a[rank] = make_float4(fmaf(J[18], J[18], J[21] * J[21]), fmaf(J[18], J[19], J[21] * J[22]),
                                    fmaf(J[18], J[20], J[21] * J[23]), fmaf(J[19], J[19], J[22] * J[22]));
        stage_b[rank] = make_float4(fmaf(J[19], J[20], J[22] * J[23]), fmaf(J[20], J[20], J[23] * J[23]),
                                    fmaf(J[18], r0, J[21] * r1), fmaf(J[19], r0, J[22] * r1));
        stage_gz[rank] = fmaf(J[20], r0, J[23] * r1);
        __threadfence_block();
        const unsigned last = (unsigned)(re - rb - 1);
        if (atomicInc(&arrived[pid], last) == last) {  // the counter is back at 0 for the group's next tile
          __threadfence_block();
          float2 a0 = make_float2(0.f, 0.f), a1 = a0, b0 = a0, b1 = a0;
          float gz = 0.f;
#pragma unroll 4  // (same order, loads batched: Skewed, tracks up to 200, 0.634 -> 0.616 ms)
          for (int r = rb; r < re; ++r) {  // rank order: V_k, g_p,k do not depend on the arrival order
            const float4 x = stage_a[r], y = stage_b[r];
            const float z = stage_gz[r];
            a0 = __fadd2_rn(a0, make_float2(x.x, x.y));
            a1 = __fadd2_rn(a1, make_float2(x.z, x.w));
            b0 = __fadd2_rn(b0, make_float2(y.x, y.y));
            b1 = __fadd2_rn(b1, make_float2(y.z, y.w));
            gz += z;
          }
          v.V0[p0 + pid] = make_float4(a0.x, a0.y, a1.x, a1.y);
          v.V1[p0 + pid] = b0;
          v.gp[p0 + pid] = make_float4(b1.x, b1.y, gz, 0.f);
        }
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(buf_done);  // this warp is done with the buffer
    } else {
      if (cam >= 0) {
        double r0, r1;
        residual_observation(table, cam, X.x, X.y, X.z, m, v.depth_eps, r0, r1);
        term = loss_term(v, fma(r0, r0, r1 * r1)).rho;
      }
    }
    cost_acc += term;
    s += NG;
    while (s >= L.stages) { s -= L.stages; ++round; }
    within += NG;  // this group's next tile: NG further in the CTA's sequence
    t += NG;
    while (within >= C) { within -= C; t += (G - 1) * C; }
  }
  const double wsum = warp_sum(cost_acc);
  if ((tid & 31) == 0) v.cost_warp[blockIdx.x * (NG * (T / 32)) + (tid >> 5)] = wsum;
}

// Sum of the per-warp cost partials in a FIXED order (thread i takes i, i + 1024, ...; then the block tree):
// the cost is bitwise reproducible, and no floating-point atomic is left on the linearize path (C14).
__global__ void __launch_bounds__(1024) reduce_cost_kernel(const double* __restrict__ part, long long n,
                                                          double* __restrict__ out) {
  __shared__ double red[32];
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  long long i = threadIdx.x;
  for (; i + 3072 < n; i += 4096) {
    a0 += part[i];
    a1 += part[i + 1024];
    a2 += part[i + 2048];
    a3 += part[i + 3072];
  }
  for (; i < n; i += 1024) a0 += part[i];
  const double tot = block_sum((a0 + a1) + (a2 + a3), red);
  if (threadIdx.x == 0) *out = tot;
}

// ------------------------------------------------------------------------------------------------
// S4 camera-side assembly: U_j = sum J_c^T J_c (45 unique) and g_c,j = sum J_c^T r (9).
// Camera-ordered pass: one warp per chunk of <= kChunkSlots slots of one camera (slots ascending, so
// the gathers walk the camera's in-tile runs contiguously); 54 fp32 partial sums per lane, reduced
// across lanes in fp64 and written as ONE partial row per chunk; reduce_camera_chunks_kernel then adds a
// camera's chunk rows in chunk order.  No atomics anywhere: U_j and g_c,j are bitwise reproducible (C14).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) assemble_cameras_kernel(View v) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= v.num_chunks) return;
  const int b = v.chunk_begin[w], e = v.chunk_begin[w + 1];
  float acc[kUg];
#pragma unroll
  for (int i = 0; i < kUg; ++i) acc[i] = 0.f;
  for (int i = b + lane; i < e; i += 32) {
    const int s = v.cslot[i];
    float J[20];
#pragma unroll
    for (int c = 0; c < 5; ++c) {
      const float4 x = v.J[c][s];
      J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
    }
    const float2 r = v.res[s];
    int k = 0;
#pragma unroll
    for (int a = 0; a < 9; ++a)
#pragma unroll
      for (int c = a; c < 9; ++c) {
        acc[k] = fmaf(J[a], J[c], fmaf(J[9 + a], J[9 + c], acc[k]));
        ++k;
      }
#pragma unroll
    for (int a = 0; a < 9; ++a) acc[45 + a] = fmaf(J[a], r.x, fmaf(J[9 + a], r.y, acc[45 + a]));
  }
  double mine0 = 0.0, mine1 = 0.0;
#pragma unroll
  for (int i = 0; i < kUg; ++i) {
    const double tot = warp_sum((double)acc[i]);
    if ((i & 31) == lane) {
      if (i < 32) mine0 = tot; else mine1 = tot;
    }
  }
  double* dst = v.Ug_part + (long long)kUg * w;
  dst[lane] = mine0;
  if (lane + 32 < kUg) dst[lane + 32] = mine1;
}

// One block of 64 threads per camera: thread e adds entry e of the camera's chunk rows, in chunk order, with four
// interleaved accumulators (chunk index mod 4) so that a hot camera's ~2,400 rows are not one dependent chain.
__global__ void __launch_bounds__(64) reduce_camera_chunks_kernel(View v) {
  const int j = blockIdx.x, e = threadIdx.x;
  if (e >= kUg) return;
  const int c0 = v.cam_chunk_ptr[j], c1 = v.cam_chunk_ptr[j + 1];
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  const double* src = v.Ug_part + (long long)kUg * c0 + e;
  int c = c0;
  for (; c + 4 <= c1; c += 4, src += 4 * kUg) {
    a0 += src[0];
    a1 += src[kUg];
    a2 += src[2 * kUg];
    a3 += src[3 * kUg];
  }
  if (c < c1) a0 += src[0];
  if (c + 1 < c1) a1 += src[kUg];
  if (c + 2 < c1) a2 += src[2 * kUg];
  v.Ug[(long long)kUg * j + e] = (a0 + a1) + (a2 + a3);
}

// ------------------------------------------------------------------------------------------------
// N4 Schur-Jacobi preconditioner ("one block per node"): the diagonal 9x9 blocks of
// the Schur complement itself,
//   S_jj = U'_j - sum_{i in j} W_i V'^-1_k(i) W_i^T = lambda D_j + sum_{i in j} J_c,i^T (I - B_i) J_c,i,
//   B_i = J_p,i V'^-1_k(i) J_p,i^T  (2x2, 0 <= B_i <= I),
// assembled as a sum of positive semi-definite terms (no cancellation against U'_j at small lambda).  The same
// camera-ordered chunk pass as assemble_cameras_kernel, with a 2x2 weight per observation; one partial row per
// chunk, added in chunk order by reduce_camera_chunks_kernel (bitwise reproducible).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) assemble_schur_diagonal_kernel(View v) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= v.num_chunks) return;
  const int b = v.chunk_begin[w], e = v.chunk_begin[w + 1];
  float acc[45];
#pragma unroll
  for (int i = 0; i < 45; ++i) acc[i] = 0.f;
  for (int i = b + lane; i < e; i += 32) {
    const int s = v.cslot[i];
    float J[24];
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      const float4 x = v.J[c][s];
      J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
    }
    const int tile = s / v.T;
    const unsigned pid = v.T <= 256 ? (unsigned)(v.rankpid[s] >> 8) : (v.rankpid32[s] >> 16);
    const long long k = (long long)v.tile_pt[tile] + pid;
    // y = V'^-1 J_p^T (3x2), B = J_p y, in fp64: 1 - B cancels to ~lambda (see schur_pass_kernel)
    const double* vi = v.Vinv64 + 6 * k;  // xx xy xz yy yz zz
    const double a[3] = {J[18], J[19], J[20]}, c[3] = {J[21], J[22], J[23]};  // J_p rows
    const double ya0 = vi[0] * a[0] + vi[1] * a[1] + vi[2] * a[2], ya1 = vi[1] * a[0] + vi[3] * a[1] + vi[4] * a[2],
                 ya2 = vi[2] * a[0] + vi[4] * a[1] + vi[5] * a[2];
    const double yc0 = vi[0] * c[0] + vi[1] * c[1] + vi[2] * c[2], yc1 = vi[1] * c[0] + vi[3] * c[1] + vi[4] * c[2],
                 yc2 = vi[2] * c[0] + vi[4] * c[1] + vi[5] * c[2];
    const float m00 = (float)(1.0 - (a[0] * ya0 + a[1] * ya1 + a[2] * ya2));
    const float m01 = (float)(-(a[0] * yc0 + a[1] * yc1 + a[2] * yc2));
    const float m11 = (float)(1.0 - (c[0] * yc0 + c[1] * yc1 + c[2] * yc2));
    float z0[9], z1[9];  // (I - B) J_c
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      z0[q] = fmaf(m00, J[q], m01 * J[9 + q]);
      z1[q] = fmaf(m01, J[q], m11 * J[9 + q]);
    }
    int idx = 0;
#pragma unroll
    for (int p = 0; p < 9; ++p)
#pragma unroll
      for (int q = p; q < 9; ++q) {
        acc[idx] = fmaf(J[p], z0[q], fmaf(J[9 + p], z1[q], acc[idx]));
        ++idx;
      }
  }
  double mine0 = 0.0, mine1 = 0.0;
#pragma unroll
  for (int i = 0; i < 45; ++i) {
    const double tot = warp_sum((double)acc[i]);
    if ((i & 31) == lane) {
      if (i < 32) mine0 = tot; else mine1 = tot;
    }
  }
  double* dst = v.Ug_part + (long long)kUg * w;  // the per-chunk rows are free again once U, g_c are reduced
  dst[lane] = mine0;
  if (lane + 32 < 45) dst[lane + 32] = mine1;
}

__global__ void __launch_bounds__(64) reduce_schur_diagonal_kernel(View v) {
  const int j = blockIdx.x, e = threadIdx.x;
  if (e >= 45) return;
  const int c0 = v.cam_chunk_ptr[j], c1 = v.cam_chunk_ptr[j + 1];
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  const double* src = v.Ug_part + (long long)kUg * c0 + e;
  int c = c0;
  for (; c + 4 <= c1; c += 4, src += 4 * kUg) {
    a0 += src[0];
    a1 += src[kUg];
    a2 += src[2 * kUg];
    a3 += src[3 * kUg];
  }
  if (c < c1) a0 += src[0];
  if (c + 1 < c1) a1 += src[kUg];
  if (c + 2 < c1) a2 += src[2 * kUg];
  v.Sdiag[45ll * j + e] = (a0 + a1) + (a2 + a3);
}

// ------------------------------------------------------------------------------------------------
// Damped blocks for one lambda: M^-1 = (U + lambda D_c)^-1 per camera (fp64 Cholesky), lambda D_c,
// the initial Schur right-hand side -g_c; V'^-1 = (V + lambda D_p)^-1 per point (fp64, stored fp32).
// ------------------------------------------------------------------------------------------------
__global__ void prepare_cameras_kernel(View v, double lambda, int schur_diagonal) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= v.nc) return;
  const double* ug = v.Ug + (long long)kUg * j;
  double A[81], L[81];
  {
    int k = 0;
    for (int a = 0; a < 9; ++a)
      for (int c = a; c < 9; ++c) {
        A[9 * a + c] = ug[k];
        A[9 * c + a] = ug[k];
        ++k;
      }
  }
  double ld[9];
  for (int a = 0; a < 9; ++a) {
    const double d = v.damping_mode == 1 ? 1.0 : fmax(A[10 * a], (double)kDMin);
    ld[a] = lambda * d;
    v.lamD[9ll * j + a] = ld[a];
    v.b[9ll * j + a] = v.shard_root ? -ug[45 + a] : 0.0;  // the shards' right-hand sides are summed: -g_c enters once
  }
  if (schur_diagonal) {  // S_jj = lambda D_j + sum J_c^T (I - B) J_c
    const double* sd = v.Sdiag + 45ll * j;
    int k = 0;
    for (int a = 0; a < 9; ++a)
      for (int c = a; c < 9; ++c) {
        A[9 * a + c] = sd[k];
        A[9 * c + a] = sd[k];
        ++k;
      }
  }
  for (int a = 0; a < 9; ++a) A[10 * a] += ld[a];
  {
    double* blk = v.Pblk + 81ll * j;  // the block the preconditioner inverts (test export)
    for (int i = 0; i < 81; ++i) blk[i] = A[i];
  }
  bool ok = true;
  for (int i = 0; i < 81; ++i) L[i] = 0.0;
  for (int i = 0; i < 9 && ok; ++i)
    for (int c = 0; c <= i; ++c) {
      double s = A[9 * i + c];
      for (int k = 0; k < c; ++k) s -= L[9 * i + k] * L[9 * c + k];
      if (i == c) {
        if (!(s > 0.0)) { ok = false; break; }
        L[10 * i] = sqrt(s);
      } else {
        L[9 * i + c] = s / L[10 * c];
      }
    }
  double* Mi = v.Minv + 81ll * j;
  if (!ok) {
    v.step->bad_block = 1.0;
    for (int i = 0; i < 81; ++i) Mi[i] = (i % 10 == 0) ? 1.0 : 0.0;
    return;
  }
  for (int c = 0; c < 9; ++c) {  // solve L L^T x = e_c
    double y[9], x[9];
    for (int i = 0; i < 9; ++i) {
      double s = (i == c) ? 1.0 : 0.0;
      for (int k = 0; k < i; ++k) s -= L[9 * i + k] * y[k];
      y[i] = s / L[10 * i];
    }
    for (int i = 8; i >= 0; --i) {
      double s = y[i];
      for (int k = i + 1; k < 9; ++k) s -= L[9 * k + i] * x[k];
      x[i] = s / L[10 * i];
    }
    for (int i = 0; i < 9; ++i) Mi[9 * i + c] = x[i];
  }
}

__global__ void prepare_points_kernel(View v, double lambda) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= v.np_obs) return;
  const float4 a = v.V0[k];
  const float2 c = v.V1[k];
  double xx = a.x, xy = a.y, xz = a.z, yy = a.w, yz = c.x, zz = c.y;
  const bool unit = v.damping_mode == 1;
  xx += lambda * (unit ? 1.0 : fmax(xx, (double)kDMin));
  yy += lambda * (unit ? 1.0 : fmax(yy, (double)kDMin));
  zz += lambda * (unit ? 1.0 : fmax(zz, (double)kDMin));
  // Cholesky pivots decide positive definiteness; the inverse itself is the adjugate over the determinant
  const double l00 = xx, l10 = xy / l00, l20 = xz / l00;
  const double d1 = yy - l10 * xy, m21 = yz - l10 * xz, d2 = zz - l20 * xz - (m21 / d1) * m21;
  if (!(l00 > 0.0) || !(d1 > 0.0) || !(d2 > 0.0)) {
    v.step->bad_block = 1.0;
    v.Vinv[2ll * k] = make_float4(0.f, 0.f, 0.f, 0.f);
    v.Vinv[2ll * k + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = 0; i < 6; ++i) v.Vinv64[6ll * k + i] = 0.0;
    return;
  }
  const double c00 = yy * zz - yz * yz, c01 = xz * yz - xy * zz, c02 = xy * yz - xz * yy;
  const double c11 = xx * zz - xz * xz, c12 = xy * xz - xx * yz, c22 = xx * yy - xy * xy;
  const double idet = 1.0 / (xx * c00 + xy * c01 + xz * c02);
  v.Vinv[2ll * k] = make_float4((float)(c00 * idet), (float)(c01 * idet), (float)(c02 * idet), (float)(c11 * idet));
  v.Vinv[2ll * k + 1] = make_float4((float)(c12 * idet), (float)(c22 * idet), 0.f, 0.f);
  double* w = v.Vinv64 + 6ll * k;  // the same inverse unrounded, for the fp64 point elimination
  w[0] = c00 * idet; w[1] = c01 * idet; w[2] = c02 * idet; w[3] = c11 * idet; w[4] = c12 * idet; w[5] = c22 * idet;
}

// ------------------------------------------------------------------------------------------------
// S5 / S6 / S8: one pass over the stored Jacobians in tile order.
//   MATVEC : q_j += sum_{i in j} J_c^T (u - J_p s_k),  u = J_c p_j,  s_k = V'^-1 sum_{i in k} J_p^T u
//            (the lambda D_c p term and the dot p.q are completed by the PCG update kernel)
//   RHS    : b_j += sum_{i in j} J_c^T J_p V'^-1 g_p,k          (b_j was initialised to -g_c,j)
//   BACKSUB: delta_p,k = -V'^-1 (g_p,k + sum_{i in k} J_p^T J_c delta_c,j);  also |J delta|^2, delta_p.g_p
// ------------------------------------------------------------------------------------------------
enum { MATVEC = 0, RHS = 1, BACKSUB = 2 };

template <int T, int MODE>
__global__ void __launch_bounds__(T, blocks_per_sm(T)) schur_pass_kernel(View v) {
  // one buffer, two views: pstage[3][T + 1] doubles for the point side, then stage[9][T + 1] floats for the camera side
  __shared__ double raw[(9 * (T + 1) + 1) / 2];
  float(*stage)[T + 1] = reinterpret_cast<float(*)[T + 1]>(raw);
  double(*pstage)[T + 1] = reinterpret_cast<double(*)[T + 1]>(raw);
  // The point elimination e = u - J_p V'^-1 J_p^T u is a least-squares residual computed through the normal
  // equations: its rounding error is cond(V'_k) eps |u|, and two-view points with a short baseline have
  // cond(V') ~ 1e4..1e6.  In fp32 that is 1e-3..1e-1 of |u|, more than the lambda-sized margin that keeps S positive
  // definite at lambda <= 1e-4: PCG then meets p.Sp <= 0 (skewed).  u, t_k, s_k and e are therefore
  // carried in fp64 (the stored Jacobians stay fp32; ~35 DFMA per observation, far below the HBM bound).
  __shared__ double red[32];
  const int t = blockIdx.x, tid = threadIdx.x;
  if (MODE == MATVEC) {
    if (v.pcg->done) return;
    if (t == 0 && tid == 0) {  // accumulators of the update that follows this matvec
      const int nxt = (v.pcg->it_a + 1) & 1;  // it_a: written by the previous update kernel only
      v.pcg->rz[nxt] = 0.0;
      v.pcg->pDp[nxt] = 0.0;
      v.pcg->rr = 0.0;
    }
  }
  const long long slot = (long long)t * T + tid;
  const int p0 = v.tile_pt[t], p1 = v.tile_pt[t + 1];
  const int base = v.pt_ptr[p0];
  const int cam = v.cam[slot];
  const unsigned rank = v.rank[slot];
  float J[24];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const float4 x = __ldcs(&v.J[c][slot]);  // streamed once per pass: evict-first
    J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
  }
  double u0 = 0.0, u1 = 0.0;
  if (MODE != RHS) {
    if (cam >= 0) {
      const float4* pv = reinterpret_cast<const float4*>(v.p32) + 3ll * cam;
      const float4 a = __ldg(pv), b = __ldg(pv + 1), c = __ldg(pv + 2);
      const float pj[9] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x};
#pragma unroll
      for (int i = 0; i < 9; ++i) {
        u0 = fma((double)J[i], (double)pj[i], u0);
        u1 = fma((double)J[9 + i], (double)pj[i], u1);
      }
      pstage[0][rank] = fma((double)J[18], u0, (double)J[21] * u1);
      pstage[1][rank] = fma((double)J[19], u0, (double)J[22] * u1);
      pstage[2][rank] = fma((double)J[20], u0, (double)J[23] * u1);
    }
    __syncthreads();
  }
  // point threads
  double dg_part = 0.0;
  for (int k = p0 + tid; k < p1; k += T) {
    const int rb = v.pt_ptr[k] - base, re = v.pt_ptr[k + 1] - base;
    double t0 = 0.0, t1 = 0.0, t2 = 0.0;
    if (MODE != RHS)
      for (int r = rb; r < re; ++r) { t0 += pstage[0][r]; t1 += pstage[1][r]; t2 += pstage[2][r]; }
    const double* vi = v.Vinv64 + 6ll * k;  // xx xy xz yy yz zz
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE != MATVEC) {
      g = v.gp[k];
      t0 += g.x; t1 += g.y; t2 += g.z;
    }
    double s0 = vi[0] * t0 + vi[1] * t1 + vi[2] * t2;
    double s1 = vi[1] * t0 + vi[3] * t1 + vi[4] * t2;
    double s2 = vi[2] * t0 + vi[4] * t1 + vi[5] * t2;
    if (MODE == BACKSUB) {
      s0 = -s0; s1 = -s1; s2 = -s2;
      v.dp[k] = make_float4((float)s0, (float)s1, (float)s2, 0.f);
      dg_part += s0 * g.x + s1 * g.y + s2 * g.z;
    }
    for (int r = rb; r < re; ++r) { pstage[0][r] = s0; pstage[1][r] = s1; pstage[2][r] = s2; }
  }
  __syncthreads();
  float c9[9];
  double dot_part = 0.0;  // fp64: squares of fp32 values underflow once |p| falls below ~1e-19
#pragma unroll
  for (int i = 0; i < 9; ++i) c9[i] = 0.f;
  if (cam >= 0) {
    const double s0 = pstage[0][rank], s1 = pstage[1][rank], s2 = pstage[2][rank];
    const double w0 = (double)J[18] * s0 + (double)J[19] * s1 + (double)J[20] * s2;
    const double w1 = (double)J[21] * s0 + (double)J[22] * s1 + (double)J[23] * s2;
    if (MODE == BACKSUB) {
      const double y0 = u0 + w0, y1 = u1 + w1;  // (J delta)_i
      dot_part = y0 * y0 + y1 * y1;
    } else {
      const double ed0 = (MODE == MATVEC) ? u0 - w0 : w0;
      const double ed1 = (MODE == MATVEC) ? u1 - w1 : w1;
      if (MODE == MATVEC) dot_part = u0 * ed0 + u1 * ed1;
      const float e0 = (float)ed0, e1 = (float)ed1;
#pragma unroll
      for (int i = 0; i < 9; ++i) c9[i] = fmaf(J[i], e0, J[9 + i] * e1);
    }
  }
  if (MODE != BACKSUB) {
    __syncthreads();  // every thread has read its s_k: the buffer becomes the camera-side staging rows
#pragma unroll
    for (int i = 0; i < 9; ++i) stage[i][tid] = c9[i];
    __syncthreads();
    // camera runs: one thread per (run, component), fp32 inside the tile, fp64 across tiles
    const int rb = v.run_begin[t], nruns = v.run_begin[t + 1] - rb - 1;
    double* dst = (MODE == MATVEC) ? v.q : v.b;
    for (int w = tid; w < 9 * nruns; w += T) {
      const int u = w / 9, a = w - 9 * u;
      const int s1 = v.run_slot[rb + u + 1];
      float acc = 0.f;
      for (int s = v.run_slot[rb + u]; s < s1; ++s) acc += stage[a][s];
      atomicAdd(dst + 9ll * v.run_cam[rb + u] + a, (double)acc);
    }
  }
  if (MODE == MATVEC) {
    const double tot = block_sum(dot_part, red);
    if (tid == 0) atomicAdd(&v.pcg->pq, tot);
  }
  if (MODE == BACKSUB) {
    const double jd2 = block_sum(dot_part, red);
    const double dg = block_sum(dg_part, red);
    if (tid == 0) {
      atomicAdd(&v.step->jd2, jd2);
      atomicAdd(&v.step->dg, dg);
    }
  }
}


// ------------------------------------------------------------------------------------------------
// S6, pipelined: the Schur matvec as a PERSISTENT kernel, one CTA per SM.
//
//   producer warp : one elected lane streams whole tiles into a ring of shared-memory stages with TMA
//                   bulk copies (cp.async.bulk.shared::cluster.global + mbarrier complete_tx): the six
//                   Jacobian chunk arrays, camera ids, ranks, the tile's metadata blob and its V'^-1
//                   rows — ten copies, one mbarrier per stage, L2 evict-first on the streamed Jacobians.
//   consumer warps: T threads, one observation each, run the three reduction phases of a tile from
//                   shared memory only; the only global traffic left on their critical path is the
//                   L1/L2-resident p_j gather and the fire-and-forget fp64 REDs.
// The ring keeps STAGES-1 tiles (~60 KB each) in flight per SM regardless of what the consumers do,
// which is what the first (one block per tile) version lacked: ncu showed 38 % barrier + 38 %
// long-scoreboard stalls at 39 % of HBM peak (history).
// ------------------------------------------------------------------------------------------------
struct PipeLayout {  // byte offsets inside one stage / inside the dynamic shared memory
  int j, cam, rank, vinv, gp, meta, stage_bytes, sbuf_stride;
  int stages, groups, tbuf, tbuf_bytes, sbuf, sbuf_bytes, scratch, hot, bars, total;
};

constexpr int kHotShift = 23;  // HOT kernels carry (hot index + 1) << 23 in a slot's camera id: needs nc < 2^23 (ba_reorder.cpp)
constexpr int kWarpScratchBytes = 1328;  // per consumer warp: 9 x 33 floats of products + 32 camera ids (1,316 B)

// NG consumer groups of T threads share the ring; each group owns a staging area for the point-side sums
// t_k (by rank) and one for the per-point results s_k (by local point id).
// with_gp: the stage also carries the tile's g_p rows (the S5 / S8 instantiations of the kernel)
__host__ __device__ inline PipeLayout pipe_layout(int T, int NG, int max_pts, int meta_max, int num_hot,
                                                  int smem_limit, bool with_gp = false) {
  PipeLayout L;
  auto up = [](int x) { return (x + 127) & ~127; };
  L.groups = NG;
  L.j = 0;
  L.cam = L.j + 6 * T * 16;
  L.rank = L.cam + T * 4;
  L.vinv = up(L.rank + T * 2);
  L.gp = up(L.vinv + max_pts * 48);  // V'^-1 in fp64, six entries per point
  L.meta = with_gp ? up(L.gp + max_pts * 16) : L.gp;
  L.stage_bytes = up(L.meta + meta_max);
  L.tbuf_bytes = up(3 * (T + 2) * 8);  // the point side is carried in fp64 (see schur_pass_kernel)
  // sbuf is indexed by POINT (<= max_pts), not by slot; row stride = 5 mod 16: the 15 storing lanes of phase B (point
  // lp = 0..4, component c) hit 64-bit banks lp + 5 c.  (Shared memory is what limits the ring: the fp64 point side cut
  // it from 6 to 4 stages on Large; the slimmer sbuf and scratch buy a 5th back: 0.672 -> 0.665 ms.)
  L.sbuf_stride = ((max_pts + 15) & ~15) + 5;
  L.sbuf_bytes = up(3 * L.sbuf_stride * 8);
  const int hot_bytes = up(num_hot * 9 * 8);  // per-CTA fp64 accumulators of the hot cameras' q rows
  const int fixed = NG * (L.tbuf_bytes + L.sbuf_bytes) + NG * (T / 32) * kWarpScratchBytes + hot_bytes + 256;
  int st = (smem_limit - fixed) / L.stage_bytes;
  L.stages = st > kMaxStages ? kMaxStages : st;
  L.tbuf = L.stages * L.stage_bytes;
  L.sbuf = L.tbuf + NG * L.tbuf_bytes;
  L.scratch = L.sbuf + NG * L.sbuf_bytes;
  L.hot = L.scratch + NG * (T / 32) * kWarpScratchBytes;
  L.bars = L.hot + hot_bytes;
  L.total = L.bars + 256;
  return L;
}


// MODE = MATVEC (S6), RHS (S5) or BACKSUB (S8): the same pass as schur_pass_kernel, see there.  RHS and BACKSUB also
// stream the tile's g_p rows into the stage; BACKSUB has no camera side (HOT is false there).
template <int T, int NG, bool HOT, int MODE>
__global__ void __launch_bounds__(NG * T + 32, 1) schur_matvec_pipelined_kernel(View v, PipeLayout L) {
  extern __shared__ __align__(128) unsigned char smem[];
  if (MODE == MATVEC && v.pcg->done) return;
  const int tid = threadIdx.x;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + L.bars);
  unsigned long long* empty = full + kMaxStages;
  // seen[s]: how many fills of stage s some consumer has already observed complete.  A parity wait cannot tell
  // "fill n done" from "fill n - 2 done, n - 1 still in flight"; when the stage count is not a multiple of NG
  // the previous fill of a stage belongs to ANOTHER group, bulk copies may complete out of order, and a group
  // could run one whole phase ahead of the barrier.  It therefore first waits until fill n - 1 has been seen.
  volatile int* seen = reinterpret_cast<volatile int*>(empty + kMaxStages);
  // Hot cameras (Zipf popularity: one camera can hold 16 % of the observations) would serialise ~1e5 REDs on the
  // same three L2 sectors per matvec; their rows are accumulated here, per CTA, and added to q once at the end.
  double* hot_acc = reinterpret_cast<double*>(smem + L.hot);
  if (HOT)
    for (int i = tid; i < 9 * v.num_hot; i += NG * T + 32) hot_acc[i] = 0.0;
  if (tid == 0) {
    for (int s = 0; s < L.stages; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, T / 32);  // one group consumes a stage
      seen[s] = 0;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (MODE == MATVEC && blockIdx.x == 0) {  // accumulators of the update that follows this matvec
      const int nxt = (v.pcg->it_a + 1) & 1;  // it_a: written by the previous update kernel only
      v.pcg->rz[nxt] = 0.0;
      v.pcg->pDp[nxt] = 0.0;
      v.pcg->rr = 0.0;
    }
  }
  __syncthreads();
  const int G = gridDim.x;

  if (tid >= NG * T) {
    // ===== producer warp: one lane issues every copy =====
    if (tid == NG * T) {
      unsigned long long pol_stream, pol_keep;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
      asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
      int s = 0;
      unsigned ph = 0;
      const int C = HOT ? 1 : tile_chunk(v, G);  // (hot cameras: C = 1 anyway; known at compile time there)
      int t = blockIdx.x * C, within = 0;
      int4 d = t < v.num_tiles ? __ldg(v.tile_dir + t) : make_int4(0, 0, 0, 0);
      for (; t < v.num_tiles;) {
        const bool wrap = within + 1 == C;
        const int tn = wrap ? t + 1 + (G - 1) * C : t + 1;
        const int4 dn = tn < v.num_tiles ? __ldg(v.tile_dir + tn) : make_int4(0, 0, 0, 0);  // prefetch next entry
        mbar_wait(empty + s, ph ^ 1);
        unsigned char* st = smem + (size_t)s * L.stage_bytes;
        const unsigned vinv_bytes = (unsigned)d.w * 48u;
        const unsigned gp_bytes = MODE == MATVEC ? 0u : (unsigned)d.w * 16u;
        mbar_expect_tx(full + s, (unsigned)(6 * T * 16 + T * 4 + T * 2) + vinv_bytes + gp_bytes + (unsigned)d.y);
        const long long slot0 = (long long)t * T;
#pragma unroll
        for (int c = 0; c < 6; ++c) bulk_g2s(st + L.j + c * T * 16, v.J[c] + slot0, T * 16, full + s, pol_stream);
        bulk_g2s(st + L.cam, v.cam + slot0, T * 4, full + s, pol_stream);
        bulk_g2s(st + L.rank, v.rankpid + slot0, T * 2, full + s, pol_stream);
        bulk_g2s(st + L.vinv, v.Vinv64 + 6ll * d.z, vinv_bytes, full + s, pol_keep);
        if (MODE != MATVEC) bulk_g2s(st + L.gp, v.gp + d.z, gp_bytes, full + s, pol_stream);
        bulk_g2s(st + L.meta, v.tile_meta + 16ll * d.x, (unsigned)d.y, full + s, pol_stream);
        d = dn;
        t = tn;
        within = wrap ? 0 : within + 1;
        if (++s == L.stages) { s = 0; ph ^= 1; }
      }
    }
    return;
  }

  // ===== consumers: group g takes every NG-th tile of this CTA's sequence =====
  const int g = tid / T, gt = tid - g * T, lane = tid & 31;
  const int bar_id = 1 + g;
  // row stride T + 2: the six lanes of a point in phase B (component c, half h) read banks 2c + h + rank: distinct
  double(*tbuf)[T + 2] = reinterpret_cast<double(*)[T + 2]>(smem + L.tbuf + (size_t)g * L.tbuf_bytes);  // by rank
  double* sbuf = reinterpret_cast<double*>(smem + L.sbuf + (size_t)g * L.sbuf_bytes);  // [3][sbuf_stride], by point
  const int sstride = L.sbuf_stride;
  float* rows = reinterpret_cast<float*>(smem + L.scratch + (size_t)(tid >> 5) * kWarpScratchBytes);
  int* camrow = reinterpret_cast<int*>(rows + 9 * 33);
  // p.q = sum_i u_i.e_i (+ p.lambda D_c p, added by the update kernel): the curvature of the operator AS COMPUTED,
  // which is what keeps alpha consistent with q (a rewritten, manifestly positive form was tried and made CG
  // diverge at lambda ~ 1e-5: DESIGN.md "PCG at tiny lambda").  fp64 accumulation.
  double dot_part = 0.0;
  double dg_part = 0.0;  // BACKSUB: delta_p . g_p
  int s = g % L.stages;  // stage of this group's current tile
  int round = g / L.stages;  // which fill of that stage it is
  // With a stage count that is a multiple of NG every stage is always consumed by the same group, in program order:
  // the parity wait alone is unambiguous and the `seen` guard (a shared-memory spin by all threads) is skipped.
  const bool guard = (L.stages % NG) != 0;
  // (the HOT instantiation keeps the plain tile-by-tile interleave, C = 1, spelled out: it has no register to spare)
  const int C = HOT ? 1 : tile_chunk(v, G);
  int t = HOT ? blockIdx.x + g * G : blockIdx.x * C + g, within = g;  // this group's first tile: the g-th of the CTA's sequence
  if (!HOT)
    while (within >= C) { within -= C; t += (G - 1) * C; }
  for (; t < v.num_tiles;) {
    if (guard)
      while (seen[s] < round) {
      }
    mbar_wait(full + s, (unsigned)(round & 1));
    if (guard && gt == 0) seen[s] = round + 1;
    const unsigned char* st = smem + (size_t)s * L.stage_bytes;
    const int npts = reinterpret_cast<const int*>(st + L.meta)[0];
    const unsigned short* pt_start = reinterpret_cast<const unsigned short*>(st + L.meta + 16);
    int cam = reinterpret_cast<const int*>(st + L.cam)[gt];
    const unsigned rp = reinterpret_cast<const unsigned short*>(st + L.rank)[gt];
    const unsigned rank = rp & 255u, pid = rp >> 8;
    // ---- phase A: u = J_c p_j, scatter J_p^T u to the point-major staging rows
    float4 pa = make_float4(0.f, 0.f, 0.f, 0.f), pb = pa, pc = pa;
    if (MODE != RHS && cam >= 0) {  // p_j (MATVEC) or delta_c,j (BACKSUB); RHS has no camera vector: u = 0
      const float4* pv = reinterpret_cast<const float4*>(v.p32) + 3ll * cam;
      pa = __ldg(pv); pb = __ldg(pv + 1); pc = __ldg(pv + 2);
    }
    // HOT: the slot's hot index rides above bit 23 of its camera id from here on (sign, equality of neighbours and the
    // scratch row keep working).  The lookup is issued HERE, two barriers ahead of the camera-side walk: inside the
    // walk it was a chain of dependent L2-latency loads, one per segment end (the 28 KB of L1 left beside the ring
    // hold neither the table nor the p rows): Skewed 0.696 ms per matvec, 0.441 with the walk's lookups and adds
    // knocked out, 0.67-0.68 with either kind of add alone knocked out.
    if (HOT && cam >= 0) cam |= ((int)__ldg(v.hot_of_cam + cam) + 1) << kHotShift;
    // The point elimination (t_k, s_k, e) is carried in fp64: its rounding error is cond(V'_k) eps |u|, and in
    // fp32 that exceeds the lambda-sized margin that keeps S positive definite once lambda <= 1e-4 (see
    // schur_pass_kernel).  u itself stays an fp32 dot product: an error du in u passes through the
    // projection I - B as (I - B) du, it is not amplified (and every fp32 -> fp64 conversion is a quarter-rate
    // XU instruction: converting the 18 entries of J_c per observation cost 0.14 ms per matvec).
    // J_c stays in registers across the two group barriers (18 registers); J_p is converted for the point side,
    // dropped, and re-read from the stage in phase C: two 128-bit loads instead of the five that re-reading J_c
    // took (the kernel is bound by shared-memory wavefronts: profiles/r02_ncu_schur_matvec.md).
    float uf0 = 0.f, uf1 = 0.f;
    float Jc[18];
    {
      float J[24];
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const float4 x = reinterpret_cast<const float4*>(st + L.j + c * T * 16)[gt];
        J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
      }
      const float pj[9] = {pa.x, pa.y, pa.z, pa.w, pb.x, pb.y, pb.z, pb.w, pc.x};
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        uf0 = fmaf(J[k], pj[k], uf0);
        uf1 = fmaf(J[9 + k], pj[k], uf1);
      }
#pragma unroll
      for (int k = 0; k < 18; ++k) Jc[k] = J[k];
      if (MODE != RHS && cam >= 0) {
        const double u0 = (double)uf0, u1 = (double)uf1;
        tbuf[0][rank] = fma((double)J[18], u0, (double)J[21] * u1);
        tbuf[1][rank] = fma((double)J[19], u0, (double)J[22] * u1);
        tbuf[2][rank] = fma((double)J[20], u0, (double)J[23] * u1);
      }
    }
    group_bar(bar_id, T);
    // ---- phase B: six lanes per point (component x half of the track; lanes 30, 31 idle, five points per
    // warp and pass): t_k = sum over the point's rank range, s_k = V'^-1 t_k, stored once per point
    {
      const int lp = lane / 6, c = (lane - 6 * lp) >> 1, half = lane & 1;
      for (int k0 = (gt >> 5) * 5; k0 < npts; k0 += (T / 32) * 5) {
        const int k = k0 + lp;
        const bool valid = lane < 30 && k < npts;
        const int rb = valid ? pt_start[k] : 0, re = valid ? pt_start[k + 1] : 0;
        double tsum = 0.0;
        if (MODE != RHS)
          // (a track of up to 16 observations is done in ONE round of up to eight independent loads per lane: with four
          // loads per round the tracks of 9-16 observations took two: Large 0.664 -> 0.648 ms per matvec)
          for (int r = rb + half; r < re; r += 16) {
            const double a0 = tbuf[c][r];
            const double a1 = r + 2 < re ? tbuf[c][r + 2] : 0.0;
            const double a2 = r + 4 < re ? tbuf[c][r + 4] : 0.0;
            const double a3 = r + 6 < re ? tbuf[c][r + 6] : 0.0;
            double hi = 0.0;
            if (r + 8 < re) {
              const double a4 = tbuf[c][r + 8];
              const double a5 = r + 10 < re ? tbuf[c][r + 10] : 0.0;
              const double a6 = r + 12 < re ? tbuf[c][r + 12] : 0.0;
              const double a7 = r + 14 < re ? tbuf[c][r + 14] : 0.0;
              hi = (a4 + a5) + (a6 + a7);
            }
            tsum += ((a0 + a1) + (a2 + a3)) + hi;
          }
        double gc = 0.0;  // component c of g_p,k (RHS: t = g_p; BACKSUB: t = sum + g_p)
        if (MODE != MATVEC && valid && half == 0) {
          gc = (double)reinterpret_cast<const float*>(st + L.gp)[4 * k + c];
          tsum += gc;
        }
        tsum += __shfl_xor_sync(0xffffffffu, tsum, 1);
        const int base = 6 * lp;
        const double t0 = __shfl_sync(0xffffffffu, tsum, base), t1 = __shfl_sync(0xffffffffu, tsum, base + 2),
                     t2 = __shfl_sync(0xffffffffu, tsum, base + 4);
        if (valid && half == 0) {
          const double* vi = reinterpret_cast<const double*>(st + L.vinv) + 6 * k;  // xx xy xz yy yz zz
          // row c of the symmetric 3x3: (0: xx xy xz) (1: xy yy yz) (2: xz yz zz)
          const double m0 = vi[c], m1 = vi[c == 0 ? 1 : (c == 1 ? 3 : 4)], m2 = vi[c == 0 ? 2 : (c == 1 ? 4 : 5)];
          double sc = m0 * t0 + m1 * t1 + m2 * t2;
          if (MODE == BACKSUB) {  // delta_p,k = -V'^-1 (g_p,k + sum J_p^T J_c delta_c); delta_p.g_p for the gain ratio
            sc = -sc;
            reinterpret_cast<float*>(v.dp + reinterpret_cast<const int*>(st + L.meta)[3] + k)[c] = (float)sc;
            dg_part += sc * gc;
          }
          sbuf[c * sstride + k] = sc;
        }
      }
    }
    group_bar(bar_id, T);
    // ---- phase C: e = u - J_p s_k, c = J_c^T e
    float c9[9];
    {
      float e0 = 0.f, e1 = 0.f;
      if (cam >= 0) {
        const float4 x4 = reinterpret_cast<const float4*>(st + L.j + 4 * T * 16)[gt];  // Jc16 Jc17 Jp0 Jp1
        const float4 x5 = reinterpret_cast<const float4*>(st + L.j + 5 * T * 16)[gt];  // Jp2 .. Jp5
        const double u0 = (double)uf0, u1 = (double)uf1;
        const double s0 = sbuf[pid], s1 = sbuf[sstride + pid], s2 = sbuf[2 * sstride + pid];
        const double w0 = (double)x4.z * s0 + (double)x4.w * s1 + (double)x5.x * s2;  // J_p s_k
        const double w1 = (double)x5.y * s0 + (double)x5.z * s1 + (double)x5.w * s2;
        if (MODE == BACKSUB) {  // |J delta|^2 of this observation
          const double y0 = u0 + w0, y1 = u1 + w1;
          dot_part += y0 * y0 + y1 * y1;
        } else {
          const double ed0 = MODE == MATVEC ? u0 - w0 : w0, ed1 = MODE == MATVEC ? u1 - w1 : w1;
          if (MODE == MATVEC) dot_part += u0 * ed0 + u1 * ed1;
          e0 = (float)ed0;
          e1 = (float)ed1;
        }
      }
      if (MODE != BACKSUB) {
#pragma unroll
        for (int k = 0; k < 9; ++k) c9[k] = fmaf(Jc[k], e0, Jc[9 + k] * e1);
      }
    }
    if (MODE == BACKSUB) {  // no camera side: the stage reads above feed registers only, so fence them (section 5.2)
      fence_reads_before_refill();
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + s);
    } else
    // ---- camera side, warp-local.  The tile's slots are sorted by camera, so a warp holds whole pieces of
    // camera runs (lane intervals).  The nine products go to the warp's scratch rows (bank = component + lane:
    // conflict free); lane (k, part) then walks component k over slots [11 part, 11 part + 11) and adds a
    // partial sum to q at every segment end: the nine lanes of a part act in lockstep, so one fp64 RED
    // instruction covers a whole 72-byte camera row.  A segment that crosses a part boundary is added in
    // two pieces.
    {
      const int cam_prev = __shfl_up_sync(0xffffffffu, cam, 1);
      const unsigned bmask = __ballot_sync(0xffffffffu, lane == 0 || cam_prev != cam);
#pragma unroll
      for (int k = 0; k < 9; ++k) rows[k * 33 + lane] = c9[k];
      camrow[lane] = cam;
      __syncwarp();
      // This warp is done with the stage.  The release sits HERE, after the scratch-row stores, on purpose: every
      // value this warp loaded from the stage has by now been consumed by an instruction whose result one of
      // those stores needs, so no stage read can still be queued when the producer's bulk copy (async proxy)
      // refills it.  Releasing right after the last stage load raced (see fence_reads_before_refill; the
      // linearize kernel, which releases early, needs the proxy fence); the fence here instead of the data
      // dependence measured 0.753 against 0.738 ms per matvec on Large.
      if (lane == 0) mbar_arrive(empty + s);
      if (lane < 27) {
        const int part = lane / 9, k = lane - 9 * part, s0 = 11 * part;
        const float* src = rows + k * 33 + s0;
        // bit i: slot s0 + i is the last slot of a segment (the next slot starts one), or of this part
        unsigned endm = ((bmask >> 1) | 0x80000000u) >> s0;
        endm |= part == 2 ? (1u << 9) : (1u << 10);
        float val[11];
#pragma unroll
        for (int i = 0; i < 11; ++i) val[i] = (i < 10 || part < 2) ? src[i] : 0.f;
        float acc = 0.f;
        double* qk = (MODE == MATVEC ? v.q : v.b) + k;
#pragma unroll
        for (int i = 0; i < 11; ++i) {
          acc += val[i];
          if (endm & (1u << i)) {
            const int cmh = camrow[s0 + i];
            if (cmh >= 0) {
              const int hot = HOT ? (cmh >> kHotShift) - 1 : -1;
              const int cm = HOT ? (cmh & ((1 << kHotShift) - 1)) : cmh;
              if (hot >= 0) atomicAdd(hot_acc + 9 * hot + k, (double)acc);
              else atomicAdd(qk + 9ll * cm, (double)acc);
            }
            acc = 0.f;
          }
        }
      }
      __syncwarp();  // the scratch rows are rewritten by this warp's next tile
    }
    s += NG;
    while (s >= L.stages) { s -= L.stages; ++round; }
    if (HOT) {
      t += NG * G;
    } else {
      within += NG;  // this group's next tile: NG further in the CTA's sequence
      t += NG;
      while (within >= C) { within -= C; t += (G - 1) * C; }
    }
  }
  // p.q (MATVEC) / |J delta|^2 and delta_p.g_p (BACKSUB): one fp64 atomic per CTA (same-address atomics serialise in
  // L2: 3,552 per-warp ones would trail the kernel)
  if (MODE != RHS) {
    const double tot = warp_sum(dot_part);
    const double tot2 = MODE == BACKSUB ? warp_sum(dg_part) : 0.0;
    double* warp_tot = reinterpret_cast<double*>(rows);  // this warp's scratch row is free now
    if (lane == 0) {
      warp_tot[0] = tot;
      warp_tot[1] = tot2;
    }
    group_bar(15, NG * T);  // all consumer groups are done
    if (tid < 32) {
      double a = 0.0, b = 0.0;
      for (int w = lane; w < NG * (T / 32); w += 32) {
        const double* wt = reinterpret_cast<const double*>(smem + L.scratch + (size_t)w * kWarpScratchBytes);
        a += wt[0];
        b += wt[1];
      }
      a = warp_sum(a);
      if (MODE == BACKSUB) b = warp_sum(b);
      if (lane == 0) {
        if (MODE == MATVEC) {
          atomicAdd(&v.pcg->pq, a);
        } else {
          atomicAdd(&v.step->jd2, a);
          atomicAdd(&v.step->dg, b);
        }
      }
    }
  } else if (HOT) {
    group_bar(15, NG * T);  // the hot accumulators below are complete once every group is done
  }
  if (HOT) {  // one RED per hot camera row and CTA
    double* dst = MODE == MATVEC ? v.q : v.b;
    for (int i = tid; i < 9 * v.num_hot; i += NG * T) {
      const double a = hot_acc[i];
      if (a != 0.0) atomicAdd(dst + 9ll * __ldg(v.hot_list + i / 9) + i % 9, a);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// S7 PCG vector kernels: fp64 state, 32 cameras (288 elements) per block, scalars stay on the device.
// ------------------------------------------------------------------------------------------------
constexpr int kPcgThreads = 288;

__device__ __forceinline__ double apply_minv(const View& v, int j, int a, const double* rs_cam) {
  const double* Mi = v.Minv + 81ll * j + 9 * a;
  double z = 0.0;
#pragma unroll
  for (int c = 0; c < 9; ++c) z = fma(Mi[c], rs_cam[c], z);
  return z;
}

// The fp32 copy of the search direction is p * 2^-e with 2^e ~ |r|: the matvec then works at O(1)
// magnitudes whatever the residual has shrunk to (fp32 products of a direction below ~1e-19 would
// underflow), and q, p.q are scaled back exactly (powers of two) by the update kernel.
__device__ __forceinline__ double direction_scale(double rr) {
  if (!(rr > 0.0) || !isfinite(rr)) return 1.0;
  int e;
  frexp(rr, &e);
  return ldexp(1.0, -(e / 2));
}

// The scalar sums of the S7 kernels (r.z, |r|^2, p.lambda D p, |b|^2), DETERMINISTICALLY (v.det_scalars: the handles of
// a sharded problem): every block stores its partials, the last block to arrive (a ticket) adds all of them in block order and adds the total to the target with
// ONE atomic.  Given the same vectors every run -- and every shard of a sharded problem (caspar_ba_set_shard) --
// computes the same BITS, so alpha, beta, the power-of-two direction scale and the stop decision agree across
// shards without a broadcast.  (Per-block atomics made them agree only to the last bits.)  N <= 3 sums per kernel;
// `mine` are this block's, already reduced (valid in thread 0).  Must be reached by every thread of every block.
template <int N>
__device__ __forceinline__ void fold_block_sums(const View& v, const double (&mine)[N], double* const (&target)[N], double* red) {
  __shared__ int is_last;
  const int nb = (int)gridDim.x, b = (int)blockIdx.x, tid = (int)threadIdx.x;
  if (!v.det_scalars) {  // single-GPU handles: one atomic per block and sum (the fold costs the launch-bound small
                         // scenes 16 % of their LM iterations/s: 1,609 -> 1,341 on Tiny)
    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < N; ++k) atomicAdd(target[k], mine[k]);
    }
    return;
  }
  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < N; ++k) v.pcg_part[(size_t)k * nb + b] = mine[k];
    __threadfence();
    is_last = atomicAdd(v.pcg_ticket, 1u) == (unsigned)(nb - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
#pragma unroll
  for (int k = 0; k < N; ++k) {
    double a = 0.0;
    for (int i = tid; i < nb; i += (int)blockDim.x) a += __ldcg(v.pcg_part + (size_t)k * nb + i);
    const double tot = block_sum(a, red);
    if (tid == 0) atomicAdd(target[k], tot);  // onto the zeroed accumulator (N1's point kernels add their part too)
  }
  if (tid == 0) *v.pcg_ticket = 0u;
}

// |b|^2, needed before the first direction is rounded to fp32
__global__ void __launch_bounds__(kPcgThreads) pcg_norm_kernel(View v) {
  __shared__ double red[32];
  const long long i = (long long)blockIdx.x * kPcgThreads + threadIdx.x;
  const double bi = i < 9ll * v.nc ? v.b[i] : 0.0;
  const double s = block_sum(bi * bi, red);
  const double mine[1] = {s};
  double* const target[1] = {&v.pcg->bnorm2};
  fold_block_sums<1>(v, mine, target, red);
}

// x = 0, r = b, z = M^-1 r, p = z; rz[0], |r|^2, pDp[0]
__global__ void __launch_bounds__(kPcgThreads) pcg_init_kernel(View v, double tol2) {
  __shared__ double rs[kPcgThreads];
  __shared__ double red[32];
  const int tid = threadIdx.x;
  const long long i = (long long)blockIdx.x * kPcgThreads + tid;
  const int j = (int)(i / 9), a = (int)(i - 9ll * j);
  const bool valid = j < v.nc;
  const double ri = valid ? v.b[i] : 0.0;
  rs[tid] = ri;
  __syncthreads();
  const double scale = direction_scale(v.pcg->bnorm2);
  double zi = 0.0, ld = 0.0;
  if (valid) {
    zi = apply_minv(v, j, a, rs + (tid - a));
    ld = v.lamD[i];
    v.x[i] = 0.0;
    v.r[i] = ri;
    v.z[i] = zi;
    v.p[i] = zi;
    v.q[i] = 0.0;
    v.p32[(long long)kCamPad * j + a] = (float)(zi * scale);
  }
  const double s_rz = block_sum(ri * zi, red);
  const double s_rr = block_sum(ri * ri, red);
  const double s_pd = block_sum(ld * zi * zi, red);
  if (tid == 0 && blockIdx.x == 0) {
    v.pcg->pscale = scale;
    v.pcg->tol2 = tol2;
  }
  const double mine[3] = {s_rz, s_rr, s_pd};
  double* const target[3] = {&v.pcg->rz[0], &v.pcg->rr, &v.pcg->pDp[0]};
  fold_block_sums<3>(v, mine, target, red);
}

// alpha = rz / (p.q); x += alpha p; r -= alpha q; z = M^-1 r; rz_new, |r|^2
// The iteration number lives on the device (it_a: read by the matvec and by this kernel, written by
// pcg_update_p; it_b: read by pcg_update_p, written here): no kernel reads a counter it writes, and no kernel
// argument changes from one iteration to the next, so a chunk of iterations can be replayed as a CUDA graph.
__global__ void __launch_bounds__(kPcgThreads) pcg_update_xr_kernel(View v) {
  __shared__ double rs[kPcgThreads];
  __shared__ double red[32];
  PcgScalars* sc = v.pcg;
  if (sc->done) return;
  const int iter = sc->it_a;
  const int tid = threadIdx.x, par = iter & 1;
  const double unscale = 1.0 / sc->pscale;  // q and p.q were computed from p * pscale
  const double denom = sc->pq * unscale * unscale + sc->pDp[par];
  const double rz = sc->rz[par];
  if (!(denom > 0.0) || !isfinite(denom) || !isfinite(rz)) {  // breakdown (C15) or b = 0
    if (blockIdx.x == 0 && tid == 0) {
      sc->done = 1;
      if (sc->bnorm2 == 0.0) sc->converged = 1; else sc->breakdown = 1;
    }
    return;
  }
  const double alpha = rz / denom;
  const long long i = (long long)blockIdx.x * kPcgThreads + tid;
  const int j = (int)(i / 9), a = (int)(i - 9ll * j);
  const bool valid = j < v.nc;
  double ri = 0.0;
  if (valid) {
    const double pi = v.p[i];
    const double qi = v.q[i] * unscale + v.lamD[i] * pi;
    v.x[i] += alpha * pi;
    ri = v.r[i] - alpha * qi;
    v.r[i] = ri;
  }
  rs[tid] = ri;
  __syncthreads();
  double zi = 0.0;
  if (valid) {
    zi = apply_minv(v, j, a, rs + (tid - a));
    v.z[i] = zi;
  }
  const double s_rz = block_sum(ri * zi, red);
  const double s_rr = block_sum(ri * ri, red);
  if (tid == 0 && blockIdx.x == 0) {
    sc->iters = iter + 1;
    sc->it_b = iter;
    if (iter == 0) sc->rz0 = rz;
  }
  const double mine[2] = {s_rz, s_rr};
  double* const target[2] = {&sc->rz[par ^ 1], &sc->rr};
  fold_block_sums<2>(v, mine, target, red);
}

// stop if |r| <= tol |b|, else beta = rz_new / rz; p = z + beta p; p.(lambda D p); q = 0
__global__ void __launch_bounds__(kPcgThreads) pcg_update_p_kernel(View v) {
  __shared__ double red[32];
  PcgScalars* sc = v.pcg;
  if (sc->done) return;
  const int iter = sc->it_b;
  const int tid = threadIdx.x, par = iter & 1;
  // |r|^2 of the iteration just completed survives the next matvec's reset of rr (a breakdown reports it)
  if (blockIdx.x == 0 && tid == 0) sc->rr_last = sc->rr;
  if (sc->rr <= sc->tol2 * sc->bnorm2) {
    if (blockIdx.x == 0 && tid == 0) { sc->done = 1; sc->converged = 1; }
    return;
  }
  const double beta = sc->rz[par ^ 1] / sc->rz[par];
  const double scale = direction_scale(sc->rr);
  const long long i = (long long)blockIdx.x * kPcgThreads + tid;
  const int j = (int)(i / 9), a = (int)(i - 9ll * j);
  double pd = 0.0;
  if (j < v.nc) {
    const double pi = v.z[i] + beta * v.p[i];
    v.p[i] = pi;
    v.q[i] = 0.0;
    v.p32[(long long)kCamPad * j + a] = (float)(pi * scale);
    pd = v.lamD[i] * pi * pi;
  }
  const double s_pd = block_sum(pd, red);
  if (tid == 0 && blockIdx.x == 0) {
    sc->pq = 0.0;
    sc->pscale = scale;
    sc->it_a = iter + 1;
  }
  const double mine[1] = {s_pd};
  double* const target[1] = {&sc->pDp[par ^ 1]};
  fold_block_sums<1>(v, mine, target, red);
}

// ------------------------------------------------------------------------------------------------
// N1: the paper's own linear solve, PCG with normal residual on the FULL camera + point system,
// no Schur elimination (PAPER.md:163 "solves the linear normal equations directly", :167-169 "the Jacobian and its
// transpose are applied separately").  One pass over the stored Jacobians per iteration, in tile order:
//   u_i = J_c,i p_c,j(i) + J_p,i p_p,k(i)                       (J applied, per observation)
//   q_c,j += sum_{i in j} J_c,i^T u_i,   q_p,k = sum_{i in k} J_p,i^T u_i      (J^T applied: "shared add" on both sides)
// camera side exactly as the Schur pass (in-tile camera runs, one fp64 RED per run and component), point side
// through the rank-ordered staging rows (a point lives in one tile: plain stores, no atomics).  The lambda D p terms
// and p.q = sum |u_i|^2 + p.lambda D p are completed by the update kernels.  FINAL: the same pass on delta instead of
// the search direction, for |J delta|^2 of the gain ratio (ignores / keeps the PCG scalars).
// ------------------------------------------------------------------------------------------------
template <int T, bool FINAL>
__global__ void __launch_bounds__(T, blocks_per_sm(T)) full_matvec_kernel(View v) {
  __shared__ float stage[9][T + 1];
  __shared__ double red[32];
  const int t = blockIdx.x, tid = threadIdx.x;
  if (!FINAL) {
    if (v.pcg->done) return;
    if (t == 0 && tid == 0) {  // accumulators of the update that follows this matvec
      const int nxt = (v.pcg->it_a + 1) & 1;
      v.pcg->rz[nxt] = 0.0;
      v.pcg->pDp[nxt] = 0.0;
      v.pcg->rr = 0.0;
    }
  }
  const long long slot = (long long)t * T + tid;
  const int p0 = v.tile_pt[t], p1 = v.tile_pt[t + 1];
  const int base = v.pt_ptr[p0];
  const int cam = v.cam[slot];
  const unsigned rank = v.rank[slot];
  float J[24];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const float4 x = __ldcs(&v.J[c][slot]);
    J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
  }
  // the direction's point part, broadcast to the point's rank range
  for (int k = p0 + tid; k < p1; k += T) {
    const float4 pp = v.pp32[k];
    for (int r = v.pt_ptr[k] - base; r < v.pt_ptr[k + 1] - base; ++r) { stage[0][r] = pp.x; stage[1][r] = pp.y; stage[2][r] = pp.z; }
  }
  __syncthreads();
  float u0 = 0.f, u1 = 0.f;
  if (cam >= 0) {
    const float4* pv = reinterpret_cast<const float4*>(v.p32) + 3ll * cam;
    const float4 a = __ldg(pv), b = __ldg(pv + 1), c = __ldg(pv + 2);
    const float pj[9] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x};
#pragma unroll
    for (int i = 0; i < 9; ++i) {
      u0 = fmaf(J[i], pj[i], u0);
      u1 = fmaf(J[9 + i], pj[i], u1);
    }
    const float x0 = stage[0][rank], x1 = stage[1][rank], x2 = stage[2][rank];
    u0 += fmaf(J[18], x0, fmaf(J[19], x1, J[20] * x2));
    u1 += fmaf(J[21], x0, fmaf(J[22], x1, J[23] * x2));
    stage[0][rank] = fmaf(J[18], u0, J[21] * u1);  // J_p^T u, at the same rank this thread just read
    stage[1][rank] = fmaf(J[19], u0, J[22] * u1);
    stage[2][rank] = fmaf(J[20], u0, J[23] * u1);
  }
  const double dot_part = (double)u0 * (double)u0 + (double)u1 * (double)u1;
  if (!FINAL) {
    __syncthreads();
    for (int k = p0 + tid; k < p1; k += T) {
      float t0 = 0.f, t1 = 0.f, t2 = 0.f;
      for (int r = v.pt_ptr[k] - base; r < v.pt_ptr[k + 1] - base; ++r) { t0 += stage[0][r]; t1 += stage[1][r]; t2 += stage[2][r]; }
      v.qp[k] = make_float4(t0, t1, t2, 0.f);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 9; ++i) stage[i][tid] = cam >= 0 ? fmaf(J[i], u0, J[9 + i] * u1) : 0.f;
    __syncthreads();
    const int rb = v.run_begin[t], nruns = v.run_begin[t + 1] - rb - 1;
    for (int w = tid; w < 9 * nruns; w += T) {
      const int u = w / 9, a = w - 9 * u;
      const int s1 = v.run_slot[rb + u + 1];
      float acc = 0.f;
      for (int s = v.run_slot[rb + u]; s < s1; ++s) acc += stage[a][s];
      atomicAdd(v.q + 9ll * v.run_cam[rb + u] + a, (double)acc);
    }
  }
  const double tot = block_sum(dot_part, red);
  if (tid == 0) atomicAdd(FINAL ? &v.step->jd2 : &v.pcg->pq, tot);
}

// ---- point part of the PCGNR vector updates.  The camera part is the Schur PCG's own kernels (pcg_norm / pcg_init /
// pcg_update_xr / pcg_update_p with b = -g_c and M = blockdiag(U'_j)); both parts add to the same device scalars and
// take the same decisions from them, and the point kernels run BEFORE the camera kernels of the same phase because
// those advance the iteration counters and the direction scale.  State per point: x, r in fp64; the direction only
// as the fp32 copy handed to the matvec (p = pp32 / pscale, a power of two); z = V'^-1 r is recomputed, not stored.
__device__ __forceinline__ void point_damping(const View& v, int k, double lambda, double (&ld)[3]) {
  if (v.damping_mode == 1) {
    ld[0] = ld[1] = ld[2] = lambda;
  } else {
    const float4 a = v.V0[k];
    const float2 c = v.V1[k];
    ld[0] = lambda * fmax((double)a.x, (double)kDMin);
    ld[1] = lambda * fmax((double)a.w, (double)kDMin);
    ld[2] = lambda * fmax((double)c.y, (double)kDMin);
  }
}

__device__ __forceinline__ void apply_vinv(const View& v, int k, const double (&r)[3], double (&z)[3]) {
  const float4 vi = v.Vinv[2ll * k];
  const float4 vj = v.Vinv[2ll * k + 1];
  z[0] = (double)vi.x * r[0] + (double)vi.y * r[1] + (double)vi.z * r[2];
  z[1] = (double)vi.y * r[0] + (double)vi.w * r[1] + (double)vj.x * r[2];
  z[2] = (double)vi.z * r[0] + (double)vj.x * r[1] + (double)vj.y * r[2];
}

__global__ void __launch_bounds__(256) pcgnr_norm_points_kernel(View v) {
  __shared__ double red[32];
  const int k = blockIdx.x * 256 + threadIdx.x;
  double s = 0.0;
  if (k < v.np_obs) {
    const float4 g = v.gp[k];
    s = (double)g.x * g.x + (double)g.y * g.y + (double)g.z * g.z;
  }
  s = block_sum(s, red);
  if (threadIdx.x == 0) atomicAdd(&v.pcg->bnorm2, s);
}

__global__ void __launch_bounds__(256) pcgnr_init_points_kernel(View v, double lambda) {
  __shared__ double red[32];
  const int k = blockIdx.x * 256 + threadIdx.x;
  const double scale = direction_scale(v.pcg->bnorm2);
  double s_rz = 0.0, s_rr = 0.0, s_pd = 0.0;
  if (k < v.np_obs) {
    const float4 g = v.gp[k];
    const double r[3] = {-(double)g.x, -(double)g.y, -(double)g.z};
    double z[3], ld[3];
    apply_vinv(v, k, r, z);
    point_damping(v, k, lambda, ld);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      v.xp[3ll * k + a] = 0.0;
      v.rp[3ll * k + a] = r[a];
      s_rz += r[a] * z[a];
      s_rr += r[a] * r[a];
    }
    // the direction as the matvec sees it; p.lambda D p from the rounded direction (what alpha is applied to)
    const float4 pp = make_float4((float)(z[0] * scale), (float)(z[1] * scale), (float)(z[2] * scale), 0.f);
    v.pp32[k] = pp;
    const double inv = 1.0 / scale;
    s_pd = ld[0] * (pp.x * inv) * (pp.x * inv) + ld[1] * (pp.y * inv) * (pp.y * inv) + ld[2] * (pp.z * inv) * (pp.z * inv);
  }
  s_rz = block_sum(s_rz, red);
  s_rr = block_sum(s_rr, red);
  s_pd = block_sum(s_pd, red);
  if (threadIdx.x == 0) {
    atomicAdd(&v.pcg->rz[0], s_rz);
    atomicAdd(&v.pcg->rr, s_rr);
    atomicAdd(&v.pcg->pDp[0], s_pd);
  }
}

__global__ void __launch_bounds__(256) pcgnr_update_xr_points_kernel(View v, double lambda) {
  __shared__ double red[32];
  const PcgScalars* sc = v.pcg;
  if (sc->done) return;
  const int par = sc->it_a & 1;
  const double unscale = 1.0 / sc->pscale;
  const double denom = sc->pq * unscale * unscale + sc->pDp[par];
  const double rz = sc->rz[par];
  if (!(denom > 0.0) || !isfinite(denom) || !isfinite(rz)) return;  // the camera kernel records the breakdown
  const double alpha = rz / denom;
  const int k = blockIdx.x * 256 + threadIdx.x;
  double s_rz = 0.0, s_rr = 0.0;
  if (k < v.np_obs) {
    const float4 pp = v.pp32[k], qq = v.qp[k];
    double ld[3], r[3], z[3];
    point_damping(v, k, lambda, ld);
    const double p[3] = {pp.x * unscale, pp.y * unscale, pp.z * unscale};
    const double q[3] = {qq.x * unscale + ld[0] * p[0], qq.y * unscale + ld[1] * p[1], qq.z * unscale + ld[2] * p[2]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      v.xp[3ll * k + a] += alpha * p[a];
      r[a] = v.rp[3ll * k + a] - alpha * q[a];
      v.rp[3ll * k + a] = r[a];
    }
    apply_vinv(v, k, r, z);
    s_rz = r[0] * z[0] + r[1] * z[1] + r[2] * z[2];
    s_rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
  }
  s_rz = block_sum(s_rz, red);
  s_rr = block_sum(s_rr, red);
  if (threadIdx.x == 0) {
    atomicAdd(&v.pcg->rz[par ^ 1], s_rz);
    atomicAdd(&v.pcg->rr, s_rr);
  }
}

__global__ void __launch_bounds__(256) pcgnr_update_p_points_kernel(View v, double lambda) {
  __shared__ double red[32];
  const PcgScalars* sc = v.pcg;
  if (sc->done) return;
  const int par = sc->it_b & 1;
  if (sc->rr <= sc->tol2 * sc->bnorm2) return;  // converged: the camera kernel records it
  const double beta = sc->rz[par ^ 1] / sc->rz[par];
  const double unscale = 1.0 / sc->pscale, scale = direction_scale(sc->rr);
  const int k = blockIdx.x * 256 + threadIdx.x;
  double s_pd = 0.0;
  if (k < v.np_obs) {
    const float4 pp = v.pp32[k];
    const double r[3] = {v.rp[3ll * k], v.rp[3ll * k + 1], v.rp[3ll * k + 2]};
    double z[3], ld[3];
    apply_vinv(v, k, r, z);
    point_damping(v, k, lambda, ld);
    const float4 pn = make_float4((float)((z[0] + beta * (pp.x * unscale)) * scale), (float)((z[1] + beta * (pp.y * unscale)) * scale),
                                  (float)((z[2] + beta * (pp.z * unscale)) * scale), 0.f);
    v.pp32[k] = pn;
    const double inv = 1.0 / scale;
    s_pd = ld[0] * (pn.x * inv) * (pn.x * inv) + ld[1] * (pn.y * inv) * (pn.y * inv) + ld[2] * (pn.z * inv) * (pn.z * inv);
  }
  s_pd = block_sum(s_pd, red);
  if (threadIdx.x == 0) atomicAdd(&v.pcg->pDp[par ^ 1], s_pd);
}

// delta_p = x_p (fp32 for the trial update and the export), its fp32 copy as the direction of the final J delta
// pass, and delta_p . g_p; unobserved points get 0
__global__ void __launch_bounds__(256) pcgnr_finish_points_kernel(View v) {
  __shared__ double red[32];
  const int k = blockIdx.x * 256 + threadIdx.x;
  double s = 0.0;
  if (k < v.np) {
    float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
    if (k < v.np_obs) {
      d = make_float4((float)v.xp[3ll * k], (float)v.xp[3ll * k + 1], (float)v.xp[3ll * k + 2], 0.f);
      const float4 g = v.gp[k];
      s = (double)d.x * g.x + (double)d.y * g.y + (double)d.z * g.z;
      v.pp32[k] = d;
    }
    v.dp[k] = d;
  }
  s = block_sum(s, red);
  if (threadIdx.x == 0) atomicAdd(&v.step->dg, s);
}

// delta_c -> fp32 padded copy for the back-substitution pass; delta_c . g_c
__global__ void __launch_bounds__(kPcgThreads) delta_c_kernel(View v) {
  __shared__ double red[32];
  const long long i = (long long)blockIdx.x * kPcgThreads + threadIdx.x;
  const int j = (int)(i / 9), a = (int)(i - 9ll * j);
  double d = 0.0;
  if (j < v.nc) {
    const double xi = v.x[i];
    v.p32[(long long)kCamPad * j + a] = (float)xi;
    d = v.shard_root ? xi * v.Ug[(long long)kUg * j + 45 + a] : 0.0;  // delta_c.g_c enters the shards' sum once
  }
  const double s = block_sum(d, red);
  if (threadIdx.x == 0) atomicAdd(&v.step->dg, s);
}

// ------------------------------------------------------------------------------------------------
// S9 trial point and commit
// ------------------------------------------------------------------------------------------------
// Pose3 camera (camera_model 1): w <- Log(Exp(w) Exp(d)) through unit quaternions, fp64.
__device__ __forceinline__ void quat_of_rotvec(double x, double y, double z, double (&q)[4]) {
  const double th2 = x * x + y * y + z * z, th = sqrt(th2);
  const double k = th2 < 1e-8 ? 0.5 - th2 / 48.0 : sin(0.5 * th) / th;
  q[0] = cos(0.5 * th); q[1] = k * x; q[2] = k * y; q[3] = k * z;
}

__device__ __forceinline__ double retract_rotation(const float* w, const double* d, int a) {
  double p[4], q[4], c[4];
  quat_of_rotvec((double)w[0], (double)w[1], (double)w[2], p);
  quat_of_rotvec(d[0], d[1], d[2], q);
  c[0] = p[0] * q[0] - p[1] * q[1] - p[2] * q[2] - p[3] * q[3];
  c[1] = p[0] * q[1] + p[1] * q[0] + p[2] * q[3] - p[3] * q[2];
  c[2] = p[0] * q[2] - p[1] * q[3] + p[2] * q[0] + p[3] * q[1];
  c[3] = p[0] * q[3] + p[1] * q[2] - p[2] * q[1] + p[3] * q[0];
  if (c[0] < 0.0) { c[0] = -c[0]; c[1] = -c[1]; c[2] = -c[2]; c[3] = -c[3]; }  // same rotation, angle <= pi
  const double s = sqrt(c[1] * c[1] + c[2] * c[2] + c[3] * c[3]);
  const double k = s < 1e-8 ? 2.0 / c[0] : 2.0 * atan2(s, c[0]) / s;
  return k * c[1 + a];
}

__global__ void trial_update_kernel(View v) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < 9ll * v.nc) {
    const int j = (int)(i / 9), a = (int)(i - 9ll * j);
    if (v.camera_model == 1 && a < 3) v.cams_trial[i] = (float)retract_rotation(v.cameras + 9ll * j, v.x + 9ll * j, a);
    else v.cams_trial[i] = (float)((double)v.cameras[i] + v.x[i]);
  }
  if (i < v.np) {
    const float4 p = v.pts[i], d = v.dp[i];
    v.pts_trial[i] = make_float4(p.x + d.x, p.y + d.y, p.z + d.z, 0.f);
  }
}

__global__ void commit_kernel(View v) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < 9ll * v.nc) v.cameras[i] = v.cams_trial[i];
  if (i < v.np) {
    const float4 p = v.pts_trial[i];
    v.pts[i] = p;
    float* d = v.points + 3ll * v.pt_perm[i];
    d[0] = p.x; d[1] = p.y; d[2] = p.z;
  }
}

// ------------------------------------------------------------------------------------------------
// test-only exports (caller order, fp64 array-of-structs) and the standalone matvec
// ------------------------------------------------------------------------------------------------
__global__ void export_kernel(View v, int what, double* __restrict__ dst) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  switch (what) {
    case CASPAR_BA_RESIDUALS:
    case CASPAR_BA_JC:
    case CASPAR_BA_JP: {
      if (i >= v.n_slots) return;
      const int o = v.obs_of_slot[i];
      if (o < 0) return;
      if (what == CASPAR_BA_RESIDUALS) {
        const float2 r = v.res[i];
        dst[2ll * o] = r.x;
        dst[2ll * o + 1] = r.y;
      } else {
        float J[24];
        for (int c = 0; c < 6; ++c) {
          const float4 x = v.J[c][i];
          J[4 * c] = x.x; J[4 * c + 1] = x.y; J[4 * c + 2] = x.z; J[4 * c + 3] = x.w;
        }
        if (what == CASPAR_BA_JC)
          for (int e = 0; e < 18; ++e) dst[18ll * o + e] = J[e];
        else
          for (int e = 0; e < 6; ++e) dst[6ll * o + e] = J[18 + e];
      }
      return;
    }
    case CASPAR_BA_U: {
      if (i >= v.nc) return;
      const double* ug = v.Ug + (long long)kUg * i;
      int k = 0;
      for (int a = 0; a < 9; ++a)
        for (int c = a; c < 9; ++c) {
          dst[81ll * i + 9 * a + c] = ug[k];
          dst[81ll * i + 9 * c + a] = ug[k];
          ++k;
        }
      return;
    }
    case CASPAR_BA_V: {
      if (i >= v.np) return;
      double* d = dst + 9ll * v.pt_perm[i];
      if (i >= v.np_obs) {
        for (int e = 0; e < 9; ++e) d[e] = 0.0;
        return;
      }
      const float4 a = v.V0[i];
      const float2 c = v.V1[i];
      d[0] = a.x; d[1] = a.y; d[2] = a.z; d[3] = a.y; d[4] = a.w; d[5] = c.x; d[6] = a.z; d[7] = c.x; d[8] = c.y;
      return;
    }
    case CASPAR_BA_G:
    case CASPAR_BA_DELTA: {
      const bool grad = what == CASPAR_BA_G;
      if (i < 9ll * v.nc) {
        const int j = (int)(i / 9), a = (int)(i - 9ll * j);
        dst[i] = grad ? v.Ug[(long long)kUg * j + 45 + a] : v.x[i];
      }
      if (i < v.np) {
        double* d = dst + 9ll * v.nc + 3ll * v.pt_perm[i];
        const float4 g = grad ? v.gp[i] : v.dp[i];
        const bool live = i < v.np_obs;
        d[0] = live ? g.x : 0.0; d[1] = live ? g.y : 0.0; d[2] = live ? g.z : 0.0;
      }
      return;
    }
    case CASPAR_BA_SCHUR_RHS:
      if (i < 9ll * v.nc) dst[i] = v.b[i];
      return;
    case CASPAR_BA_PRECONDITIONER:
      if (i < 81ll * v.nc) dst[i] = v.Pblk[i];
      return;
  }
}

__global__ void matvec_load_kernel(View v, const double* __restrict__ p_in) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 9ll * v.nc) return;
  const int j = (int)(i / 9), a = (int)(i - 9ll * j);
  v.p[i] = p_in[i];
  v.q[i] = 0.0;
  v.p32[(long long)kCamPad * j + a] = (float)p_in[i];
}

__global__ void matvec_finish_kernel(View v, double* __restrict__ q_out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 9ll * v.nc) return;
  q_out[i] = v.q[i] + v.lamD[i] * v.p[i];
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static inline unsigned grid_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

// "index out of range -- validated on device at create".  first_bad receives the lowest offending
// observation index (or stays at its initial value).
__global__ void validate_indices_kernel(const int* __restrict__ cam_idx, const int* __restrict__ pt_idx, long long n,
                                        int nc, int np, unsigned long long* __restrict__ first_bad) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < n; i += stride) {
    const int c = cam_idx[i], k = pt_idx[i];
    if (c < 0 || c >= nc || k < 0 || k >= np) atomicMin(first_bad, (unsigned long long)i);
  }
}

cudaError_t launch_validate_indices(const int* cam_idx_dev, const int* pt_idx_dev, long long n, int nc, int np,
                                    unsigned long long* first_bad_dev, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  const long long blocks = (n + 255) / 256;
  validate_indices_kernel<<<(unsigned)(blocks < 148 * 16 ? blocks : 148 * 16), 256, 0, s>>>(cam_idx_dev, pt_idx_dev, n, nc, np, first_bad_dev);
  return CBA_LAUNCHED();
}

cudaError_t launch_gather_observations(const View& v, const float* observations, float2* px_out, cudaStream_t s) {
  if (v.n_slots == 0) return cudaSuccess;
  gather_observations_kernel<<<grid_for(v.n_slots, 256), 256, 0, s>>>(v, observations, px_out);
  return CBA_LAUNCHED();
}

cudaError_t launch_pack_points(const View& v, const float* src, float4* dst, cudaStream_t s) {
  if (v.np == 0) return cudaSuccess;
  pack_points_kernel<<<grid_for(v.np, 256), 256, 0, s>>>(v, src, dst);
  return CBA_LAUNCHED();
}

cudaError_t launch_unpack_points(const View& v, const float4* src, float* dst, cudaStream_t s) {
  if (v.np == 0) return cudaSuccess;
  unpack_points_kernel<<<grid_for(v.np, 256), 256, 0, s>>>(v, src, dst);
  return CBA_LAUNCHED();
}

cudaError_t launch_camera_prepass(const View& v, const float* cams, float* table, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  camera_prepass_kernel<<<grid_for(v.nc, 128), 128, 0, s>>>(v.nc, cams, table);
  return CBA_LAUNCHED();
}

int smem_optin();
int pipe_groups(int T);

static bool linearize_pipelined(const View& v) { return v.lin_pipeline != 0 && v.T <= 256 && v.num_tiles > 0; }
static int linearize_grid(const View& v) { return v.num_tiles < v.num_sms ? v.num_tiles : v.num_sms; }

template <int T, int NG, bool JAC>
static cudaError_t launch_linearize_pipelined(const View& v, const float4* pts, const float* table, cudaStream_t s) {
  const LinLayout L = lin_layout(T, NG, v.max_pts_per_tile, v.meta_max_bytes, JAC, smem_optin());
  linearize_pipelined_kernel<T, NG, JAC><<<linearize_grid(v), NG * T + 32, L.total, s>>>(v, pts, table, L);
  return CBA_LAUNCHED();
}

template <bool JAC>
static cudaError_t launch_linearize_t(const View& v, const float4* pts, const float* table, cudaStream_t s) {
  if (v.num_tiles == 0) return cudaSuccess;
  if (JAC && linearize_pipelined(v)) {
    if (v.T == 256) return launch_linearize_pipelined<256, 3, true>(v, pts, table, s);
    if (v.T == 192) return launch_linearize_pipelined<192, 4, true>(v, pts, table, s);
    return launch_linearize_pipelined<128, 6, true>(v, pts, table, s);
  }
  switch (v.T) {
    case 128: linearize_kernel<128, JAC><<<v.num_tiles, 128, 0, s>>>(v, pts, table); break;
    case 192: linearize_kernel<192, JAC><<<v.num_tiles, 192, 0, s>>>(v, pts, table); break;
    case 256: linearize_kernel<256, JAC><<<v.num_tiles, 256, 0, s>>>(v, pts, table); break;
    case 512: linearize_kernel<512, JAC><<<v.num_tiles, 512, 0, s>>>(v, pts, table); break;
    default: linearize_kernel<1024, JAC><<<v.num_tiles, 1024, 0, s>>>(v, pts, table); break;
  }
  return CBA_LAUNCHED();
}

// cost_out (device) receives sum_i rho(|r_i|^2); an empty problem gets 0 from the arena's memset / the caller
// `pipelined`: the partials were written by linearize_pipelined_kernel (one per consumer warp of the grid), else by
// linearize_kernel (one per warp of every tile)
static cudaError_t launch_reduce_cost(const View& v, bool pipelined, double* cost_out, cudaStream_t s) {
  if (v.num_tiles == 0) return cudaMemsetAsync(cost_out, 0, sizeof(double), s);
  const long long parts = pipelined ? (long long)linearize_grid(v) * pipe_groups(v.T) * (v.T / 32)
                                    : (long long)v.num_tiles * (v.T / 32);
  reduce_cost_kernel<<<1, 1024, 0, s>>>(v.cost_warp, parts, cost_out);
  return CBA_LAUNCHED();
}

cudaError_t launch_linearize(const View& v, cudaStream_t s) { return launch_linearize_t<true>(v, v.pts, v.cam_table, s); }

cudaError_t launch_linearize_at(const View& v, const float4* pts, const float* table, cudaStream_t s) {
  return launch_linearize_t<true>(v, pts, table, s);
}

cudaError_t launch_linearize_cost(const View& v, double* cost_out, cudaStream_t s) {
  return launch_reduce_cost(v, linearize_pipelined(v), cost_out, s);
}

cudaError_t launch_cost(const View& v, const float4* pts, const float* table, double* cost_out, cudaStream_t s) {
  cudaError_t e = launch_linearize_t<false>(v, pts, table, s);
  return e != cudaSuccess ? e : launch_reduce_cost(v, false, cost_out, s);
}

cudaError_t launch_assemble_cameras(const View& v, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  if (v.num_chunks == 0) return cudaMemsetAsync(v.Ug, 0, sizeof(double) * kUg * (size_t)v.nc, s);
  assemble_cameras_kernel<<<grid_for(32ll * v.num_chunks, 128), 128, 0, s>>>(v);
  cudaError_t e = CBA_LAUNCHED();
  if (e != cudaSuccess) return e;
  reduce_camera_chunks_kernel<<<v.nc, 64, 0, s>>>(v);
  return CBA_LAUNCHED();
}

// preconditioner: 0 = blockdiag(U'_j) (C9), 1 = the diagonal blocks of S (N4; needs V'^-1 first, and one more
// camera-ordered pass over the Jacobians)
cudaError_t launch_prepare_blocks(const View& v, double lambda, int preconditioner, cudaStream_t s, int stage) {
  cudaError_t e = cudaSuccess;
  if (stage == 2) {
    if (v.nc > 0) {
      prepare_cameras_kernel<<<grid_for(v.nc, 64), 64, 0, s>>>(v, lambda, preconditioner);
      e = CBA_LAUNCHED();
    }
    return e;
  }
  if (v.np_obs > 0) {
    prepare_points_kernel<<<grid_for(v.np_obs, 256), 256, 0, s>>>(v, lambda);
    e = CBA_LAUNCHED();
  }
  if (e == cudaSuccess && preconditioner == 1 && v.nc > 0) {
    if (v.num_chunks > 0) {
      assemble_schur_diagonal_kernel<<<grid_for(32ll * v.num_chunks, 128), 128, 0, s>>>(v);
      e = CBA_LAUNCHED();
    }
    if (e == cudaSuccess) {
      reduce_schur_diagonal_kernel<<<v.nc, 64, 0, s>>>(v);
      e = CBA_LAUNCHED();
    }
  }
  if (e == cudaSuccess && v.nc > 0 && stage == 0) {
    prepare_cameras_kernel<<<grid_for(v.nc, 64), 64, 0, s>>>(v, lambda, preconditioner);
    e = CBA_LAUNCHED();
  }
  return e;
}

// A handle without observations (an empty shard of a sharded problem) still runs the PCG vector kernels on the summed
// b and q: the accumulators that the matvec kernel zeroes for the update that follows it must be zeroed all the same.
__global__ void pcg_zero_accumulators_kernel(View v) {
  if (v.pcg->done) return;
  const int nxt = (v.pcg->it_a + 1) & 1;
  v.pcg->rz[nxt] = 0.0;
  v.pcg->pDp[nxt] = 0.0;
  v.pcg->rr = 0.0;
}

template <int MODE>
static cudaError_t launch_pass(const View& v, cudaStream_t s) {
  if (v.num_tiles == 0) {
    if (MODE != MATVEC || v.nc == 0) return cudaSuccess;
    pcg_zero_accumulators_kernel<<<1, 1, 0, s>>>(v);
    return CBA_LAUNCHED();
  }
  switch (v.T) {
    case 128: schur_pass_kernel<128, MODE><<<v.num_tiles, 128, 0, s>>>(v); break;
    case 192: schur_pass_kernel<192, MODE><<<v.num_tiles, 192, 0, s>>>(v); break;
    case 256: schur_pass_kernel<256, MODE><<<v.num_tiles, 256, 0, s>>>(v); break;
    case 512: schur_pass_kernel<512, MODE><<<v.num_tiles, 512, 0, s>>>(v); break;
    default: schur_pass_kernel<1024, MODE><<<v.num_tiles, 1024, 0, s>>>(v); break;
  }
  return CBA_LAUNCHED();
}


// The pipelined matvec needs the opt-in shared-memory limit and at least two stages; otherwise (or with
// CASPAR_BA_PIPELINE=0) the one-block-per-tile kernel is used.
int smem_optin() {  // of the current device (the API layer switches to the handle's device first)
  static int cached[64];  // 0 = not asked yet
  int dev = 0, v = 0;
  cudaGetDevice(&dev);
  if (dev >= 0 && dev < 64 && cached[dev] > 0) return cached[dev];
  cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (dev >= 0 && dev < 64) cached[dev] = v;
  return v;
}

// The pipelined matvec packs rank and local point id into 16 bits, so it serves tiles of <= 256 slots:
// T = 256 with three consumer groups (800 threads) or T = 128 with six.  Longer tracks use schur_pass_kernel.
int pipe_groups(int T) { return T == 256 ? 3 : (T == 192 ? 4 : 6); }

bool pipelined_matvec_possible(const View& v) {
  if (v.num_tiles == 0 || v.T > 256) return false;
  const PipeLayout L = pipe_layout(v.T, pipe_groups(v.T), v.max_pts_per_tile, v.meta_max_bytes, v.num_hot, smem_optin());
  return L.stages >= pipe_groups(v.T) + 1;
}

bool pipelined_matvec_available(const View& v) { return v.pipeline != 0; }
int pipeline_stages(const View& v) {
  return pipe_layout(v.T, pipe_groups(v.T), v.max_pts_per_tile, v.meta_max_bytes, v.num_hot, smem_optin()).stages;
}

// The opt-in limit itself is requested (not this handle's own size): the attribute is per function, and
// handles with different layouts share the kernel.
template <int T, int NG>
static cudaError_t pipelined_attr(bool hot) {
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  cudaError_t e = hot ? cudaFuncSetAttribute(schur_matvec_pipelined_kernel<T, NG, true, MATVEC>, attr, smem_optin())
                      : cudaFuncSetAttribute(schur_matvec_pipelined_kernel<T, NG, false, MATVEC>, attr, smem_optin());
  if (e == cudaSuccess)
    e = hot ? cudaFuncSetAttribute(schur_matvec_pipelined_kernel<T, NG, true, RHS>, attr, smem_optin())
            : cudaFuncSetAttribute(schur_matvec_pipelined_kernel<T, NG, false, RHS>, attr, smem_optin());
  if (e == cudaSuccess) e = cudaFuncSetAttribute(schur_matvec_pipelined_kernel<T, NG, false, BACKSUB>, attr, smem_optin());
  return e;
}

template <int T, int NG>
static cudaError_t linearize_attr() {
  return cudaFuncSetAttribute(linearize_pipelined_kernel<T, NG, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin());
}

bool pipelined_linearize_possible(const View& v) {
  if (v.num_tiles == 0 || v.T > 256) return false;
  return lin_layout(v.T, pipe_groups(v.T), v.max_pts_per_tile, v.meta_max_bytes, true, smem_optin()).stages >= pipe_groups(v.T) + 1;
}

cudaError_t configure_kernels(const View& v) {
  if (linearize_pipelined(v)) {
    const cudaError_t e = v.T == 256 ? linearize_attr<256, 3>() : (v.T == 192 ? linearize_attr<192, 4>() : linearize_attr<128, 6>());
    if (e != cudaSuccess) return e;
  }
  if (!pipelined_matvec_available(v)) return cudaSuccess;
  const bool hot = v.num_hot > 0;
  if (v.T == 256) return pipelined_attr<256, 3>(hot);
  if (v.T == 192) return pipelined_attr<192, 4>(hot);
  return pipelined_attr<128, 6>(hot);
}

template <int T, int NG, int MODE>
static void pipelined_launch(const View& v, const PipeLayout& L, int grid, cudaStream_t s) {
  if (MODE != BACKSUB && v.num_hot > 0)
    schur_matvec_pipelined_kernel<T, NG, MODE != BACKSUB, MODE><<<grid, NG * T + 32, L.total, s>>>(v, L);
  else
    schur_matvec_pipelined_kernel<T, NG, false, MODE><<<grid, NG * T + 32, L.total, s>>>(v, L);
}

// S5 / S6 / S8 through the persistent TMA-pipelined kernel when the handle uses it (and, for S5 / S8, whose stages also
// carry the g_p rows, the ring still has a stage to spare), else through the one-block-per-tile pass.
template <int MODE>
static cudaError_t launch_pipelined_or_pass(const View& v, cudaStream_t s) {
  if (!pipelined_matvec_available(v) || v.num_tiles == 0) return launch_pass<MODE>(v, s);
  const int NG = pipe_groups(v.T);
  const PipeLayout L = pipe_layout(v.T, NG, v.max_pts_per_tile, v.meta_max_bytes, v.num_hot, smem_optin(), MODE != MATVEC);
  if (L.stages < NG + 1) return launch_pass<MODE>(v, s);
  const int grid = v.num_tiles < v.num_sms ? v.num_tiles : v.num_sms;
  if (v.T == 256) pipelined_launch<256, 3, MODE>(v, L, grid, s);
  else if (v.T == 192) pipelined_launch<192, 4, MODE>(v, L, grid, s);
  else pipelined_launch<128, 6, MODE>(v, L, grid, s);
  return CBA_LAUNCHED();
}

cudaError_t launch_schur_matvec(const View& v, cudaStream_t s) { return launch_pipelined_or_pass<MATVEC>(v, s); }

cudaError_t launch_pcg_init(const View& v, double tol2, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  pcg_norm_kernel<<<grid_for(9ll * v.nc, kPcgThreads), kPcgThreads, 0, s>>>(v);
  cudaError_t e = CBA_LAUNCHED();
  if (e != cudaSuccess) return e;
  pcg_init_kernel<<<grid_for(9ll * v.nc, kPcgThreads), kPcgThreads, 0, s>>>(v, tol2);
  return CBA_LAUNCHED();
}

cudaError_t launch_pcg_update(const View& v, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  const unsigned g = grid_for(9ll * v.nc, kPcgThreads);
  pcg_update_xr_kernel<<<g, kPcgThreads, 0, s>>>(v);
  cudaError_t e = CBA_LAUNCHED();
  if (e != cudaSuccess) return e;
  pcg_update_p_kernel<<<g, kPcgThreads, 0, s>>>(v);
  return CBA_LAUNCHED();
}

cudaError_t launch_backsub(const View& v, cudaStream_t s) {
  cudaError_t e = cudaSuccess;
  if (v.nc > 0) {
    delta_c_kernel<<<grid_for(9ll * v.nc, kPcgThreads), kPcgThreads, 0, s>>>(v);
    e = CBA_LAUNCHED();
  }
  if (e != cudaSuccess) return e;
  return launch_pipelined_or_pass<BACKSUB>(v, s);
}

cudaError_t launch_schur_rhs(const View& v, cudaStream_t s) { return launch_pipelined_or_pass<RHS>(v, s); }

template <bool FINAL>
static cudaError_t launch_full_pass(const View& v, cudaStream_t s) {
  if (v.num_tiles == 0) return cudaSuccess;
  switch (v.T) {
    case 128: full_matvec_kernel<128, FINAL><<<v.num_tiles, 128, 0, s>>>(v); break;
    case 192: full_matvec_kernel<192, FINAL><<<v.num_tiles, 192, 0, s>>>(v); break;
    case 256: full_matvec_kernel<256, FINAL><<<v.num_tiles, 256, 0, s>>>(v); break;
    case 512: full_matvec_kernel<512, FINAL><<<v.num_tiles, 512, 0, s>>>(v); break;
    default: full_matvec_kernel<1024, FINAL><<<v.num_tiles, 1024, 0, s>>>(v); break;
  }
  return CBA_LAUNCHED();
}

cudaError_t launch_full_matvec(const View& v, cudaStream_t s) { return launch_full_pass<false>(v, s); }

// x0 = 0, r0 = -g, z0 = M^-1 r0, p0 = z0 on both parts (b = -g_c was set by the block preparation)
cudaError_t launch_pcgnr_init(const View& v, double lambda, double tol2, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  const unsigned gc = grid_for(9ll * v.nc, kPcgThreads), gp = grid_for(v.np_obs, 256);
  pcg_norm_kernel<<<gc, kPcgThreads, 0, s>>>(v);
  cudaError_t e = CBA_LAUNCHED();
  if (e == cudaSuccess && v.np_obs > 0) {
    pcgnr_norm_points_kernel<<<gp, 256, 0, s>>>(v);
    e = CBA_LAUNCHED();
  }
  if (e == cudaSuccess && v.np_obs > 0) {
    pcgnr_init_points_kernel<<<gp, 256, 0, s>>>(v, lambda);
    e = CBA_LAUNCHED();
  }
  if (e != cudaSuccess) return e;
  pcg_init_kernel<<<gc, kPcgThreads, 0, s>>>(v, tol2);
  return CBA_LAUNCHED();
}

cudaError_t launch_pcgnr_update(const View& v, double lambda, cudaStream_t s) {
  if (v.nc == 0) return cudaSuccess;
  const unsigned gc = grid_for(9ll * v.nc, kPcgThreads), gp = grid_for(v.np_obs, 256);
  cudaError_t e = cudaSuccess;
  if (v.np_obs > 0) {
    pcgnr_update_xr_points_kernel<<<gp, 256, 0, s>>>(v, lambda);
    e = CBA_LAUNCHED();
  }
  if (e != cudaSuccess) return e;
  pcg_update_xr_kernel<<<gc, kPcgThreads, 0, s>>>(v);
  e = CBA_LAUNCHED();
  if (e == cudaSuccess && v.np_obs > 0) {
    pcgnr_update_p_points_kernel<<<gp, 256, 0, s>>>(v, lambda);
    e = CBA_LAUNCHED();
  }
  if (e != cudaSuccess) return e;
  pcg_update_p_kernel<<<gc, kPcgThreads, 0, s>>>(v);
  return CBA_LAUNCHED();
}

// delta = x on both parts, delta . g, and |J delta|^2 from one more pass with delta as the direction
cudaError_t launch_pcgnr_finish(const View& v, cudaStream_t s) {
  cudaError_t e = cudaSuccess;
  if (v.nc > 0) {
    delta_c_kernel<<<grid_for(9ll * v.nc, kPcgThreads), kPcgThreads, 0, s>>>(v);
    e = CBA_LAUNCHED();
  }
  if (e == cudaSuccess && v.np > 0) {
    pcgnr_finish_points_kernel<<<grid_for(v.np, 256), 256, 0, s>>>(v);
    e = CBA_LAUNCHED();
  }
  return e != cudaSuccess ? e : launch_full_pass<true>(v, s);
}

cudaError_t launch_trial_update(const View& v, cudaStream_t s) {
  const long long n = 9ll * v.nc > v.np ? 9ll * v.nc : v.np;
  if (n == 0) return cudaSuccess;
  trial_update_kernel<<<grid_for(n, 256), 256, 0, s>>>(v);
  return CBA_LAUNCHED();
}

cudaError_t launch_commit(const View& v, cudaStream_t s) {
  const long long n = 9ll * v.nc > v.np ? 9ll * v.nc : v.np;
  if (n == 0) return cudaSuccess;
  commit_kernel<<<grid_for(n, 256), 256, 0, s>>>(v);
  return CBA_LAUNCHED();
}

cudaError_t launch_export(const View& v, int what, double* dst, cudaStream_t s) {
  long long n = 0;
  switch (what) {
    case CASPAR_BA_RESIDUALS: case CASPAR_BA_JC: case CASPAR_BA_JP: n = v.n_slots; break;
    case CASPAR_BA_U: n = v.nc; break;
    case CASPAR_BA_V: n = v.np; break;
    case CASPAR_BA_G: case CASPAR_BA_DELTA: n = 9ll * v.nc > v.np ? 9ll * v.nc : v.np; break;
    case CASPAR_BA_SCHUR_RHS: n = 9ll * v.nc; break;
    case CASPAR_BA_PRECONDITIONER: n = 81ll * v.nc; break;
    default: return cudaErrorInvalidValue;
  }
  if (n == 0) return cudaSuccess;
  export_kernel<<<grid_for(n, 256), 256, 0, s>>>(v, what, dst);
  return CBA_LAUNCHED();
}

cudaError_t launch_matvec_standalone(const View& v, const double* p_in, double* q_out, cudaStream_t s, int stage) {
  if (v.nc == 0) return cudaSuccess;
  const unsigned g = grid_for(9ll * v.nc, 256);
  cudaError_t e = cudaSuccess;
  if (stage != 2) {
    matvec_load_kernel<<<g, 256, 0, s>>>(v, p_in);
    e = CBA_LAUNCHED();
    if (e != cudaSuccess) return e;
    e = launch_schur_matvec(v, s);
  }
  if (e != cudaSuccess || stage == 1) return e;
  matvec_finish_kernel<<<g, 256, 0, s>>>(v, q_out);
  return CBA_LAUNCHED();
}

// ------------------------------------------------------------------------------------------------
// Allocation-free cost (caspar_ba_cost_static; include/caspar_ba.h): step S9 on the CALLER's arrays, without a
// handle and without any cudaMalloc.  The scratch the handle path keeps in its arena (the S1 camera table and the
// per-block cost partials) lives in ONE file-scope device array of a fixed size.
//
// Every device that loads the library holds these kStaticScratchBytes until the process exits.  All calls share the
// array: calls that overlap on one GPU (two streams, two threads) race on it.  Nothing in it has to start at zero:
// every word a call reads -- table rows [0, nc), partials [0, kStaticCostBlocks) -- that call has written first, so
// the previous call's contents never show.
//
// `g_static_scratch` is a device symbol: in host code its name is only a host-side stand-in, NOT a device address.
// The launcher asks the runtime for the address once per device (cudaGetSymbolAddress, that device current) and
// hands the kernels that pointer.
// ------------------------------------------------------------------------------------------------
constexpr int kStaticCostBlocks = 148 * 4;
constexpr int kStaticCostThreads = 256;
constexpr size_t kStaticTableBytes = (size_t)CASPAR_BA_STATIC_MAX_CAMERAS * kCamTableFloats * sizeof(float);
constexpr size_t kStaticScratchBytes = kStaticTableBytes + kStaticCostBlocks * sizeof(double);
static_assert(kStaticTableBytes % 256 == 0, "the partials start on a 256-byte boundary");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// One thread per observation (grid-stride, caller's order): the same fp64 residual as the S9 kernels
// (residual_observation, loss_term), summed per thread, then per block in a fixed tree; part[block] is always
// written.  An index out of range poisons the sum (NaN) instead of faulting.
__global__ void __launch_bounds__(kStaticCostThreads)
cost_static_kernel(View v, const float* __restrict__ table, const float* __restrict__ points,
                   const float2* __restrict__ observations, const int* __restrict__ cam_idx,
                   const int* __restrict__ pt_idx, long long n, double* __restrict__ part) {
  __shared__ double red[32];
  double acc = 0.0;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int c = __ldg(cam_idx + i), k = __ldg(pt_idx + i);
    if (c < 0 || c >= v.nc || k < 0 || k >= v.np) {
      acc += __longlong_as_double(0x7ff8000000000000ll);
      continue;
    }
    const float* X = points + 3ll * k;
    double r0, r1;
    residual_observation(table, c, __ldg(X), __ldg(X + 1), __ldg(X + 2), __ldg(observations + i), v.depth_eps, r0, r1);
    acc += loss_term(v, fma(r0, r0, r1 * r1)).rho;
  }
  const double tot = block_sum(acc, red);
  if (threadIdx.x == 0) part[blockIdx.x] = tot;
}

// F = 1/2 sum of the block partials, in block order (bitwise reproducible for a given input).
__global__ void __launch_bounds__(1024) cost_static_finish_kernel(const double* __restrict__ part, int n,
                                                                 double* __restrict__ out) {
  __shared__ double red[32];
  double a = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) a += part[i];
  const double tot = block_sum(a, red);
  if (threadIdx.x == 0) *out = 0.5 * tot;
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device.
static cudaError_t static_scratch_address(unsigned char** out) {
  constexpr int kMaxDevices = 64;
  static std::mutex mu;
  static unsigned char* address[kMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!address[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    address[dev] = static_cast<unsigned char*>(p);
  }
  *out = address[dev];
  return cudaSuccess;
}

cudaError_t launch_cost_static(int nc, int np, long long n, const float* cameras, const float* points,
                               const float* observations, const int* cam_idx, const int* pt_idx, int robust,
                               float robust_scale, float depth_eps, double* cost_out, cudaStream_t s) {
  if (nc > CASPAR_BA_STATIC_MAX_CAMERAS) return cudaErrorInvalidValue;
  unsigned char* scratch = nullptr;
  cudaError_t e = static_scratch_address(&scratch);
  if (e != cudaSuccess) return e;
  float* table = reinterpret_cast<float*>(scratch);
  double* part = reinterpret_cast<double*>(scratch + kStaticTableBytes);
  // (these launches are not counted into any handle's kernels_launched)
  View v{};  // only the fields the residual and the loss read
  v.nc = nc;
  v.np = np;
  v.robust = robust;
  v.robust_c2 = robust_scale * robust_scale;
  v.robust_inv_c2 = robust ? 1.0 / ((double)robust_scale * (double)robust_scale) : 0.0;
  v.depth_eps = depth_eps;
  if (nc > 0) {
    camera_prepass_kernel<<<grid_for(nc, 128), 128, 0, s>>>(nc, cameras, table);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  cost_static_kernel<<<kStaticCostBlocks, kStaticCostThreads, 0, s>>>(
      v, table, points, reinterpret_cast<const float2*>(observations), cam_idx, pt_idx, n, part);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  cost_static_finish_kernel<<<1, 1024, 0, s>>>(part, kStaticCostBlocks, cost_out);
  return cudaGetLastError();
}

}  // namespace cba
