// ba_internal.h — internal layout of the B200 bundle-adjustment path (not part of the C ABI).
//
// Data layout in HBM:
//   * Observations are permuted once at create (S0): points are ordered by their lowest camera id
//     (camera locality per tile), packed greedily into TILES of whole points with T slots each
//     (T = threads per block = 256 | 512 | 1024), and inside a tile the slots are sorted by camera so
//     that equal-camera RUNS are contiguous.  Unused slots at the end of a tile are padding (cam = -1).
//   * Per-slot arrays (length num_tiles * T, slot-major, so a warp reads 32 consecutive elements):
//       px   float2   measured pixel
//       cam  int32    camera id (-1 = padding)
//       rank uint16   position of the slot's observation in the tile's POINT-major order
//       J    6 x float4 chunk arrays: the 24 floats (J_c 2x9 row-major, then J_p 2x3 row-major) of one
//                     observation, chunk c = floats [4c, 4c+4)  ("blocked struct of arrays")
//       res  float2   residual (robust-reweighted)
//   * Per-tile: first internal point, and a run table (camera id + first slot of each camera run).
//   * Per-point arrays are in INTERNAL point order (pt_perm maps internal -> caller id).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/caspar_ba.h"

namespace cba {

constexpr int kCamTableFloats = 36;  // per-camera table row (9 x 16 B: 12 doubles + 12 floats), see camera_prepass_kernel
constexpr int kCamPad = 12;          // fp32 camera-vector copies (p, delta_c) are padded 9 -> 12 floats
constexpr int kUg = 54;              // 45 upper-triangle entries of U_j + 9 of g_c,j, fp64 accumulators
constexpr int kChunkSlots = 1024;    // camera-ordered assembly: slots per work item
constexpr int kMaxHotCameras = 128;  // cameras whose q rows the pipelined matvec accumulates per CTA
constexpr float kDMin = 1e-6f;       // floor of diag(J^T J) in the damping matrix (C5)

// Scalars of the PCG recurrence, device resident (no host round trip inside the loop).
struct PcgScalars {
  double rz[2];   // r.z, parity = iteration & 1
  double pDp[2];  // p.(lambda D_c p), parity = iteration & 1
  double pq;      // sum_i u_i.e_i of the current matvec
  double rr;      // |r|^2 after the current update (zeroed by the next matvec)
  double rr_last; // |r|^2 after the last COMPLETED iteration: what a breakdown reports
  double bnorm2;  // |b|^2
  double rz0;
  double pscale;  // the fp32 direction handed to the matvec is p * pscale (a power of two)
  double tol2;    // squared relative tolerance of this solve
  int it_a;       // iteration number: read by the matvec and pcg_update_xr, written by pcg_update_p
  int it_b;       // the same, read by pcg_update_p, written by pcg_update_xr
  int done;       // set once converged / broken down: every later kernel returns immediately
  int converged;
  int breakdown;  // p.Sp <= 0 or non-finite
  int iters;
};

// Scalars of one LM step.
struct StepScalars {
  double cost;        // sum_i rho(|r_i|^2)   (F = cost / 2)
  double trial_cost;  // same at the trial point
  double jd2;         // |J delta|^2
  double dg;          // delta.g
  double bad_block;   // > 0: a 9x9 / 3x3 block was not positive definite (a double so that shards can sum it)
};

// Everything the kernels need, passed by value.
struct View {
  int nc, np, np_obs;  // cameras, points, points with at least one observation (internal ids [0, np_obs))
  int T, num_tiles;
  long long n_slots;
  int num_chunks;
  int robust;
  float robust_c2;
  double robust_inv_c2;  // 1 / c^2
  int damping_mode;
  int det_scalars;   // 1: the S7 kernels fold their scalar sums in a fixed order (sharded handles), 0: one atomic per block
  int shard_root;    // 1 unless this handle is a non-root shard of a point-sharded problem (caspar_ba_set_shard): only
                     // the root adds the replicated camera terms (-g_c in b, delta_c.g_c) that the shards then sum
  int camera_model;  // 0: angle-axis, additive; 1: Pose3 tangent-space rotation (right perturbation) + retraction
  float depth_eps;   // d_safe = d + eps sign_no_zero(d); 0 = no guard
  // caller's arrays (borrowed)
  float* cameras;
  float* points;
  // per slot
  const float2* px;
  const int* cam;
  const unsigned short* rank;
  const unsigned short* rankpid;  // rank | local point id << 8 (T <= 256): linearize, pipelined matvec
  const unsigned* rankpid32;      // rank | local point id << 16 (T > 256): linearize
  const int* obs_of_slot;  // caller observation id of a slot (-1 = padding)
  float4* J[6];
  float2* res;
  // per tile
  const int* tile_pt;     // [num_tiles + 1] first internal point of each tile
  const int* run_begin;   // [num_tiles + 1] index of the tile's first run in run_cam / run_slot
  const int* run_cam;     // camera id of each run; one terminator (-1) per tile
  const unsigned short* run_slot;  // first slot (within the tile) of each run; terminator = valid slots
  // per tile, for the pipelined (TMA bulk) kernels: one 16-byte aligned metadata blob per tile
  //   int4 header {npts, nruns, nvalid, first internal point}
  //   uint16 pt_start[npts + 1]   (rank range of each point, padded to 16 B)
  //   uint16 run_slot[nruns + 1]  (padded to 16 B)
  //   int32  run_cam[nruns]       (padded to 16 B)
  const int4* tile_dir;            // [num_tiles] {blob offset in 16-B units, blob bytes, first point, npts}
  const unsigned char* tile_meta;  // blobs
  int max_pts_per_tile, meta_max_bytes;
  int num_sms;
  int pipeline;                    // 1: Schur matvec runs as the persistent TMA-pipelined kernel
  int lin_pipeline;                // 1: linearize / cost run as the persistent TMA-pipelined kernel
  // per internal point
  const int* pt_ptr;      // [np_obs + 1] prefix sum of track lengths
  const int* pt_perm;     // [np] internal -> caller point id
  float4* pts;            // current points, internal order (w unused)
  float4* pts_trial;
  float4* V0;             // V_k: xx xy xz yy
  float2* V1;             // V_k: yz zz
  float4* gp;             // g_p,k (xyz, w unused)
  float4* Vinv;           // V'^-1, two float4 per point: (xx xy xz yy) (yz zz 0 0) — 32 B, bulk-copy aligned
  double* Vinv64;         // V'^-1 in fp64, six entries per point (xx xy xz yy yz zz): 48 B, bulk-copy aligned
  float4* dp;             // delta_p,k
  // full-system PCG (N1): point part of the state
  double* xp;             // [3 np] x_p
  double* rp;             // [3 np] r_p
  float4* pp32;           // [np] search direction * pscale
  float4* qp;             // [np] (J^T J p)_p of the current matvec, without the lambda D p term
  // per camera
  float* cams_trial;      // [nc][9]
  float* cam_table;       // [nc][kCamTableFloats]
  float* cam_table_trial;
  double* Ug;             // [nc][54]
  double* Minv;           // [nc][81]
  double* Pblk;           // [nc][81] the blocks Minv inverts: U'_j or S_jj (test export)
  double* Sdiag;          // [nc][45] sum_{i in j} J_c^T (I - B_i) J_c: the Schur-Jacobi blocks without lambda D_j
  double* lamD;           // [9 nc]
  double* b;              // [9 nc] Schur right-hand side
  double* x;              // [9 nc] delta_c
  double* r;              // [9 nc]
  double* z;              // [9 nc]
  double* p;              // [9 nc]
  double* q;              // [9 nc] matvec accumulator (without the lambda D_c p term)
  float* p32;             // [nc][12]
  // camera-ordered assembly work list
  const int* chunk_cam;   // [num_chunks]
  const int* chunk_begin; // [num_chunks + 1] into cslot
  const int* cslot;       // slots grouped by camera, ascending
  const int* cam_chunk_ptr;  // [nc + 1] first chunk of each camera (chunks are listed camera by camera)
  double* Ug_part;        // [num_chunks][54] per-chunk partial sums of (U_j, g_c,j)
  double* cost_warp;      // [num_tiles * T / 32] per-warp cost sums, folded in index order by reduce_cost_kernel
  // hot cameras (far more observations than average): index into the per-CTA accumulators, or -1
  const short* hot_of_cam;  // [nc]
  const int* hot_list;      // [num_hot] camera ids
  int num_hot;
  PcgScalars* pcg;
  StepScalars* step;
  double* pcg_part;         // [3][blocks of the S7 kernels] per-block partial sums, folded in block order by the last block
  unsigned* pcg_ticket;     // blocks of the running S7 kernel that have stored their partials (back at 0 when it ends)
};

// Host-side result of the S0 reordering (ba_reorder.cpp).
struct Reordered {
  int T = 0, num_tiles = 0, np_obs = 0;
  long long n_slots = 0;
  std::vector<int> obs_of_slot;           // [n_slots]
  std::vector<int> cam;                   // [n_slots]
  std::vector<unsigned short> rank;       // [n_slots]
  std::vector<unsigned short> rankpid;    // [n_slots] rank | local point id << 8 (tiles of <= 256 slots only)
  std::vector<unsigned> rankpid32;        // [n_slots] rank | local point id << 16 (tiles of > 256 slots only)
  std::vector<int> tile_pt;               // [num_tiles + 1]
  std::vector<int> run_begin;             // [num_tiles + 1]
  std::vector<int> run_cam;
  std::vector<unsigned short> run_slot;
  std::vector<int> pt_ptr;                // [np_obs + 1]
  std::vector<int> pt_perm;               // [np]
  std::vector<int> chunk_cam, chunk_begin, cslot, cam_chunk_ptr;
  std::vector<short> hot_of_cam;          // [nc]
  std::vector<int> hot_list;
  std::vector<int> tile_dir;              // [4 * num_tiles]
  std::vector<unsigned char> tile_meta;
  int max_pts_per_tile = 0, meta_max_bytes = 0;
  long long camera_runs = 0;
};

// Returns 0, or CASPAR_BA_EINVAL with `err` set.
int reorder_observations(int nc, int np, long long n, const int* cam_idx, const int* pt_idx, int forced_tile,
                         Reordered* out, std::string* err);

// ---- kernel launchers (ba_kernels.cu); all enqueue on `s` and return the launch status ----
cudaError_t launch_validate_indices(const int* cam_idx_dev, const int* pt_idx_dev, long long n, int nc, int np,
                                    unsigned long long* first_bad_dev, cudaStream_t s);
cudaError_t launch_gather_observations(const View& v, const float* observations, float2* px_out, cudaStream_t s);
cudaError_t launch_pack_points(const View& v, const float* points_caller, float4* dst, cudaStream_t s);
cudaError_t launch_unpack_points(const View& v, const float4* src, float* points_caller, cudaStream_t s);
cudaError_t launch_camera_prepass(const View& v, const float* cams, float* table, cudaStream_t s);
cudaError_t launch_linearize(const View& v, cudaStream_t s);
// the same at another point: reads pts / table, writes the linearization arrays of `v` (N2: the trial point)
cudaError_t launch_linearize_at(const View& v, const float4* pts, const float* table, cudaStream_t s);
cudaError_t launch_linearize_cost(const View& v, double* cost_out, cudaStream_t s);  // folds launch_linearize's partials
cudaError_t launch_cost(const View& v, const float4* pts, const float* table, double* cost_out, cudaStream_t s);
cudaError_t launch_assemble_cameras(const View& v, cudaStream_t s);
// `stage`: 0 = everything; 1 = point blocks (+ the Schur-diagonal sums for preconditioner 1) only; 2 = camera blocks only
// (a sharded handle sums Sdiag over the shards between 1 and 2)
cudaError_t launch_prepare_blocks(const View& v, double lambda, int preconditioner, cudaStream_t s, int stage = 0);
cudaError_t launch_schur_rhs(const View& v, cudaStream_t s);
cudaError_t launch_pcg_init(const View& v, double tol2, cudaStream_t s);
cudaError_t launch_schur_matvec(const View& v, cudaStream_t s);
cudaError_t configure_kernels(const View& v);  // once per handle: dynamic shared memory opt-in
bool pipelined_matvec_possible(const View& v);   // shape / shared-memory check, at create
bool pipelined_linearize_possible(const View& v);
bool pipelined_matvec_available(const View& v);  // = v.pipeline
int pipeline_stages(const View& v);
cudaError_t launch_pcg_update(const View& v, cudaStream_t s);  // two kernels
cudaError_t launch_backsub(const View& v, cudaStream_t s);
cudaError_t launch_full_matvec(const View& v, cudaStream_t s);
cudaError_t launch_pcgnr_init(const View& v, double lambda, double tol2, cudaStream_t s);
cudaError_t launch_pcgnr_update(const View& v, double lambda, cudaStream_t s);  // four kernels
cudaError_t launch_pcgnr_finish(const View& v, cudaStream_t s);
cudaError_t launch_trial_update(const View& v, cudaStream_t s);
cudaError_t launch_commit(const View& v, cudaStream_t s);
cudaError_t launch_export(const View& v, int what, double* dst, cudaStream_t s);
// `stage` (sharded handles): 0 = all, 1 = load + pass (leaves the shard's partial in v.q), 2 = finish (adds lambda D p)
cudaError_t launch_matvec_standalone(const View& v, const double* p_in, double* q_out, cudaStream_t s, int stage = 0);
// caspar_ba_cost_static: S1 + S9 on the caller's arrays with the scratch in a file-scope device array (no allocation)
cudaError_t launch_cost_static(int nc, int np, long long n, const float* cameras, const float* points,
                               const float* observations, const int* cam_idx, const int* pt_idx, int robust,
                               float robust_scale, float depth_eps, double* cost_out, cudaStream_t s);

}  // namespace cba
