// ba_api.cu — the C ABI of include/caspar_ba.h: arena, state machine, PCG loop, LM step.
// Host code only orchestrates launches and reads back a handful of scalars per call; every step of
// the path (S1-S9) runs in the kernels of ba_kernels.cu.  There is no CPU fallback.
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ba_internal.h"

namespace cba {
long long take_launch_count();
}

using namespace cba;

struct caspar_ba {
  caspar_ba_problem pb{};
  View v{};
  int device = 0;  // the CUDA device the handle was created on; every entry point switches to it
  double create_s = 0.0, reorder_s = 0.0;  // wall time of caspar_ba_create and of its host reordering (S0)
  void* arena = nullptr;
  size_t arena_bytes = 0;
  long long camera_runs = 0;
  bool linearized = false;
  bool have_delta = false;
  double prepared_lambda = -1.0;
  bool prepared = false;
  int prepared_preconditioner = 0;
  int linear_solver = 0;   // of lm_step / solve: 0 = Schur PCG, 1 = full-system PCGNR (caspar_ba_set_linear_solver)
  int preconditioner = 0;  // of the Schur PCG: 0 = blockdiag(U'_j), 1 = diagonal blocks of S (caspar_ba_set_preconditioner)
  double cost = 0.0;  // F at the cached linearization
  std::string err;
  long long launches = 0;
  // pinned host mirrors of the device scalars
  PcgScalars* h_pcg = nullptr;
  StepScalars* h_step = nullptr;
  int* h_flags = nullptr;  // done flags polled during a tolerance-driven PCG run
  // profiling
  bool profiling = false;
  std::vector<cudaEvent_t> ev_lin, ev_mv;  // start/stop pairs awaiting readout
  cudaStream_t prof_stream = nullptr;
  double lin_ms = 0.0, mv_ms = 0.0;
  long long lin_n = 0, mv_n = 0;
  std::vector<cudaEvent_t> ev_pool;
  cudaEvent_t poll_ev[2] = {nullptr, nullptr};
  // one chunk of PCG iterations (matvec + two update kernels, kPcgChunk times) as an instantiated CUDA graph:
  // no kernel argument changes between iterations (the iteration number is a device scalar), so the same graph
  // serves every chunk of every solve; captured once per handle on a private stream, launched on the caller's
  cudaStream_t capture_stream = nullptr;
  cudaGraphExec_t chunk_graph[2] = {nullptr, nullptr};  // one per set of linearization arrays (see `alt`)
  bool graph_tried[2] = {false, false};
  // N2: a second set of the arrays a linearization writes.  With fusion on, S9 evaluates the trial
  // point with the FULL linearize kernel into this set; an accepted step swaps the sets instead of linearizing again.
  struct LinSet {
    float4* J[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    float2* res = nullptr;
    float4* V0 = nullptr;
    float2* V1 = nullptr;
    float4* gp = nullptr;
  } alt;
  void* arena2 = nullptr;  // holds `alt`; allocated by caspar_ba_set_fusion(h, 1)
  size_t arena2_bytes = 0;
  int fusion = 0;
  int set_parity = 0;
  // point-sharded problem: this handle is one shard; `exchange` sums / broadcasts over the shards
  caspar_ba_exchange_fn exchange = nullptr;
  void* exchange_ctx = nullptr;
  double* xchg = nullptr;      // DEVICE exchange buffer (caller's), xchg_count doubles
  size_t xchg_count = 0;
  long long exchanges = 0;
  long long speculative_hits = 0, speculative_misses = 0;
};

constexpr int kPcgChunk = 8;

namespace {

// text of the last failure of caspar_ba_create / caspar_ba_layout_create on this thread (there is no handle to
// hold it): returned by caspar_ba_last_error(NULL)
thread_local std::string g_create_error;

int fail(caspar_ba* h, int code, const std::string& msg) {
  if (h) h->err = msg;
  return code;
}

int create_fail(int code, const std::string& msg) {
  g_create_error = msg;
  return code;
}

double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// Every entry point runs on the device the handle was created on, whatever device is current in the caller's
// thread, and restores the caller's device on return.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

int cuda_fail(caspar_ba* h, cudaError_t e, const char* where) {
  return fail(h, e == cudaErrorMemoryAllocation ? CASPAR_BA_ENOMEM : CASPAR_BA_ECUDA,
              std::string(where) + ": " + cudaGetErrorString(e));
}

#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);    \
  } while (0)

// bump allocator over the arena ("a single block of GPU memory ... all utilized arrays are views")
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <class T>
  T* take(size_t count) {
    off = (off + 255) & ~size_t(255);
    T* p = base ? (T*)(base + off) : nullptr;
    off += (count ? count : 1) * sizeof(T);
    return p;
  }
};

// One pass lays out the views; called with base = nullptr to size the arena, then with the real base.
size_t carve(caspar_ba* h, void* base, const Reordered& ro) {
  View& v = h->v;
  Carver c(base);
  const size_t S = (size_t)v.n_slots, NC = (size_t)v.nc, NP = (size_t)v.np;
  for (int i = 0; i < 6; ++i) v.J[i] = c.take<float4>(S);
  v.res = c.take<float2>(S);
  v.px = c.take<float2>(S);
  v.cam = c.take<int>(S);
  v.obs_of_slot = c.take<int>(S);
  v.rank = c.take<unsigned short>(S);
  v.rankpid = c.take<unsigned short>(ro.rankpid.size());
  v.rankpid32 = c.take<unsigned>(ro.rankpid32.size());
  v.tile_pt = c.take<int>(ro.tile_pt.size());
  v.run_begin = c.take<int>(ro.run_begin.size());
  v.run_cam = c.take<int>(ro.run_cam.size());
  v.run_slot = c.take<unsigned short>(ro.run_slot.size());
  v.tile_dir = c.take<int4>(ro.tile_dir.size() / 4);
  v.tile_meta = c.take<unsigned char>(ro.tile_meta.size());
  v.pt_ptr = c.take<int>(ro.pt_ptr.size());
  v.pt_perm = c.take<int>(NP);
  v.cslot = c.take<int>(ro.cslot.size());
  v.chunk_cam = c.take<int>(ro.chunk_cam.size());
  v.chunk_begin = c.take<int>(ro.chunk_begin.size());
  v.cam_chunk_ptr = c.take<int>(ro.cam_chunk_ptr.size());
  v.Ug_part = c.take<double>(kUg * ro.chunk_cam.size());
  v.cost_warp = c.take<double>((size_t)ro.num_tiles * (size_t)(ro.T / 32) + 32 * (size_t)v.num_sms);
  v.hot_of_cam = c.take<short>(ro.hot_of_cam.size());
  v.hot_list = c.take<int>(ro.hot_list.size());
  v.pts = c.take<float4>(NP);
  v.pts_trial = c.take<float4>(NP);
  v.V0 = c.take<float4>(NP);
  v.V1 = c.take<float2>(NP);
  v.gp = c.take<float4>(NP);
  v.Vinv = c.take<float4>(2 * NP);
  v.Vinv64 = c.take<double>(6 * NP);
  v.dp = c.take<float4>(NP);
  v.xp = c.take<double>(3 * NP);
  v.rp = c.take<double>(3 * NP);
  v.pp32 = c.take<float4>(NP);
  v.qp = c.take<float4>(NP);
  v.cams_trial = c.take<float>(9 * NC);
  v.cam_table = c.take<float>(kCamTableFloats * NC);
  v.cam_table_trial = c.take<float>(kCamTableFloats * NC);
  v.Ug = c.take<double>(kUg * NC);
  v.Minv = c.take<double>(81 * NC);
  v.Pblk = c.take<double>(81 * NC);
  v.Sdiag = c.take<double>(45 * NC);
  v.lamD = c.take<double>(9 * NC);
  v.b = c.take<double>(9 * NC);
  v.x = c.take<double>(9 * NC);
  v.r = c.take<double>(9 * NC);
  v.z = c.take<double>(9 * NC);
  v.p = c.take<double>(9 * NC);
  v.q = c.take<double>(9 * NC);
  v.p32 = c.take<float>(kCamPad * NC);
  v.pcg_part = c.take<double>(3 * (size_t)((9 * NC + 287) / 288 + 1));
  v.pcg_ticket = c.take<unsigned>(1);
  v.pcg = c.take<PcgScalars>(1);
  v.step = c.take<StepScalars>(1);
  return (c.off + 255) & ~size_t(255);
}

template <class T>
cudaError_t upload(const void* dst, const std::vector<T>& src, cudaStream_t s) {
  if (src.empty()) return cudaSuccess;
  return cudaMemcpyAsync(const_cast<void*>(dst), src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}

void account(caspar_ba* h) { h->launches += take_launch_count(); }

cudaEvent_t get_event(caspar_ba* h) {
  if (!h->ev_pool.empty()) {
    cudaEvent_t e = h->ev_pool.back();
    h->ev_pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

// Fold finished event pairs into the totals (the caller has synchronised the stream).
void drain_events(caspar_ba* h) {
  auto fold = [&](std::vector<cudaEvent_t>& evs, double& ms, long long& n) {
    for (size_t i = 0; i + 1 < evs.size(); i += 2) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, evs[i], evs[i + 1]) == cudaSuccess) {
        ms += t;
        n += 1;
      }
      h->ev_pool.push_back(evs[i]);
      h->ev_pool.push_back(evs[i + 1]);
    }
    evs.clear();
  };
  fold(h->ev_lin, h->lin_ms, h->lin_n);
  fold(h->ev_mv, h->mv_ms, h->mv_n);
}

struct Timed {  // brackets one kernel launch with events when profiling is on
  caspar_ba* h;
  std::vector<cudaEvent_t>* evs;
  cudaStream_t s;
  Timed(caspar_ba* h_, std::vector<cudaEvent_t>* e, cudaStream_t s_) : h(h_), evs(e), s(s_) {
    if (h->profiling) {
      cudaEvent_t a = get_event(h);
      cudaEventRecord(a, s);
      evs->push_back(a);
      h->prof_stream = s;
    }
  }
  ~Timed() {
    if (h->profiling) {
      cudaEvent_t b = get_event(h);
      cudaEventRecord(b, s);
      evs->push_back(b);
    }
  }
};

// ---- point-sharded mode: every partial sum over observations is summed over the shards before it is used ----
// The data goes through the caller's exchange buffer: vec[0..n) (+ up to 4 scalars behind it), one call of the caller's
// collective (an all-reduce sum of doubles), and back.
int shard_sum(caspar_ba* h, double* vec, size_t n, double* const* scalars, int ns, cudaStream_t s) {
  if (!h->exchange) return 0;
  if (n + (size_t)ns > h->xchg_count) return fail(h, CASPAR_BA_EINVAL, "exchange buffer too small");
  if (n) CK(cudaMemcpyAsync(h->xchg, vec, n * sizeof(double), cudaMemcpyDeviceToDevice, s));
  for (int i = 0; i < ns; ++i)
    CK(cudaMemcpyAsync(h->xchg + n + i, scalars[i], sizeof(double), cudaMemcpyDeviceToDevice, s));
  if (h->exchange(h->exchange_ctx, n + (size_t)ns, (void*)s) != 0)
    return fail(h, CASPAR_BA_ECUDA, "the shard exchange callback failed");
  if (n) CK(cudaMemcpyAsync(vec, h->xchg, n * sizeof(double), cudaMemcpyDeviceToDevice, s));
  for (int i = 0; i < ns; ++i)
    CK(cudaMemcpyAsync(scalars[i], h->xchg + n + i, sizeof(double), cudaMemcpyDeviceToDevice, s));
  ++h->exchanges;
  return 0;
}

int sync_step_scalars(caspar_ba* h, cudaStream_t s) {
  CK(cudaMemcpyAsync(h->h_step, h->v.step, sizeof(StepScalars), cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(h->h_pcg, h->v.pcg, sizeof(PcgScalars), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  if (h->profiling) drain_events(h);
  return 0;
}

int do_linearize(caspar_ba* h, cudaStream_t s) {
  View& v = h->v;
  CK(cudaMemsetAsync(v.step, 0, sizeof(StepScalars), s));
  CK(launch_pack_points(v, v.points, v.pts, s));
  CK(launch_camera_prepass(v, v.cameras, v.cam_table, s));
  {
    Timed t(h, &h->ev_lin, s);
    CK(launch_linearize(v, s));
  }
  CK(launch_linearize_cost(v, &v.step->cost, s));
  CK(launch_assemble_cameras(v, s));
  {  // shards: U_j, g_c,j and the cost are sums over every shard's observations
    double* sc[1] = {&v.step->cost};
    int rc = shard_sum(h, v.Ug, (size_t)kUg * (size_t)v.nc, sc, 1, s);
    if (rc) return rc;
  }
  account(h);
  h->linearized = true;
  h->prepared = false;
  h->have_delta = false;
  return 0;
}

int do_prepare(caspar_ba* h, double lambda, int preconditioner, cudaStream_t s) {
  if (h->prepared && h->prepared_lambda == lambda && h->prepared_preconditioner == preconditioner) return 0;
  if (h->exchange && preconditioner == 1) {  // the Schur-diagonal sums run over every shard's observations
    CK(launch_prepare_blocks(h->v, lambda, preconditioner, s, 1));
    int rc = shard_sum(h, h->v.Sdiag, 45 * (size_t)h->v.nc, nullptr, 0, s);
    if (rc) return rc;
    CK(launch_prepare_blocks(h->v, lambda, preconditioner, s, 2));
  } else {
    CK(launch_prepare_blocks(h->v, lambda, preconditioner, s));
  }
  account(h);
  h->prepared = true;
  h->prepared_lambda = lambda;
  h->prepared_preconditioner = preconditioner;
  return 0;
}

// Capture one chunk of iterations.  Failure is not an error: the loop then launches the kernels one by one.
static void build_chunk_graph(caspar_ba* h) {
  const int gp = h->set_parity;
  h->graph_tried[gp] = true;
  if (const char* env = std::getenv("CASPAR_BA_GRAPH"))
    if (env[0] == '0') return;
  if (!h->capture_stream && cudaStreamCreateWithFlags(&h->capture_stream, cudaStreamNonBlocking) != cudaSuccess) return;
  cudaGraph_t graph = nullptr;
  bool ok = cudaStreamBeginCapture(h->capture_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  for (int i = 0; ok && i < kPcgChunk; ++i)
    ok = launch_schur_matvec(h->v, h->capture_stream) == cudaSuccess &&
         launch_pcg_update(h->v, h->capture_stream) == cudaSuccess;
  const cudaError_t end = cudaStreamEndCapture(h->capture_stream, &graph);
  take_launch_count();  // captured launches are counted when the graph is launched
  if (ok && end == cudaSuccess && graph && cudaGraphInstantiate(&h->chunk_graph[gp], graph, 0) != cudaSuccess)
    h->chunk_graph[gp] = nullptr;
  if (graph) cudaGraphDestroy(graph);
  cudaGetLastError();
}

// Enqueue S5-S8.  No host synchronisation unless rel_tol > 0, where the device-side `done` flag is
// polled one chunk behind the launches so that the GPU never waits for the host.
int do_pcg(caspar_ba* h, double lambda, double rel_tol, int max_iter, cudaStream_t s) {
  View& v = h->v;
  h->prepared = false;  // the right-hand side b is rebuilt by prepare (it starts from -g_c)
  CK(cudaMemsetAsync(&v.step->jd2, 0, 3 * sizeof(double), s));  // jd2, dg, bad_block
  int rc = do_prepare(h, lambda, h->preconditioner, s);
  if (rc) return rc;
  CK(cudaMemsetAsync(v.pcg, 0, sizeof(PcgScalars), s));
  CK(launch_schur_rhs(v, s));
  rc = shard_sum(h, v.b, 9 * (size_t)v.nc, nullptr, 0, s);  // b = -g_c (root only) + sum over shards of W V'^-1 g_p
  if (rc) return rc;
  const double tol2 = rel_tol * rel_tol;
  // (the scalar sums of the S7 kernels are deterministic -- fold_block_sums -- so every shard computes the same alpha,
  // beta, direction scale and stop decision from the same summed b, q and p.q: no further exchange is needed)
  CK(launch_pcg_init(v, tol2, s));
  const int chunk = kPcgChunk;
  // whole chunks go out as one graph launch (not while per-launch profiling events are wanted)
  if (!h->graph_tried[h->set_parity] && v.nc > 0 && v.num_tiles > 0) {  // the kernel arguments hold the set's pointers
    account(h);
    build_chunk_graph(h);
  }
  cudaGraphExec_t chunk_graph = h->chunk_graph[h->set_parity];
  const bool use_graph = chunk_graph != nullptr && !h->profiling && !h->exchange;
  int polled = 0;  // chunks whose flag copy has been enqueued
  bool stop = false;
  for (int it = 0; it < max_iter && !stop; ++it) {
    if (use_graph && it % chunk == 0 && it + chunk <= max_iter) {
      CK(cudaGraphLaunch(chunk_graph, s));
      h->launches += 3ll * chunk;
      it += chunk - 1;
    } else {
      {
        Timed t(h, &h->ev_mv, s);
        CK(launch_schur_matvec(v, s));
      }
      if (h->exchange) {  // q and p.q are sums over the shards: the ONE exchange of a PCG iteration
        double* sc[1] = {&v.pcg->pq};
        rc = shard_sum(h, v.q, 9 * (size_t)v.nc, sc, 1, s);
        if (rc) return rc;
      }
      CK(launch_pcg_update(v, s));
    }
    // (shards: every shard computes the same flag and the copy sits at the same place of every shard's stream, so all
    // shards read the same value and stop after the same chunk: the collectives stay matched)
    if (rel_tol > 0.0 && (it + 1) % chunk == 0 && it + 1 < max_iter) {
      const int slot = polled & 1;
      if (polled >= 2) {  // wait for the copy enqueued two chunks ago (slot reuse) and look at it
        CK(cudaEventSynchronize(h->poll_ev[slot]));
        if (h->h_flags[slot]) stop = true;
      }
      if (!stop) {
        CK(cudaMemcpyAsync(&h->h_flags[slot], &v.pcg->done, sizeof(int), cudaMemcpyDeviceToHost, s));
        CK(cudaEventRecord(h->poll_ev[slot], s));
        ++polled;
      }
    }
  }
  CK(launch_backsub(v, s));
  account(h);
  h->have_delta = true;
  return 0;
}

// N1: enqueue the full-system PCG with normal residual (no Schur elimination).  Same device-side scalars, flags and
// polling as do_pcg; every iteration is one pass over the Jacobians plus four vector kernels.
int do_pcgnr(caspar_ba* h, double lambda, double rel_tol, int max_iter, cudaStream_t s) {
  View& v = h->v;
  h->prepared = false;  // b is rebuilt by prepare (it starts from -g_c)
  if (h->exchange) return fail(h, CASPAR_BA_ESTATE, "the full-system solve (N1) is not available on a sharded handle");
  CK(cudaMemsetAsync(&v.step->jd2, 0, 3 * sizeof(double), s));  // jd2, dg, bad_block
  int rc = do_prepare(h, lambda, 0, s);  // one block per node: U'_j and V'_k
  if (rc) return rc;
  CK(cudaMemsetAsync(v.pcg, 0, sizeof(PcgScalars), s));
  CK(launch_pcgnr_init(v, lambda, rel_tol * rel_tol, s));
  const int chunk = kPcgChunk;
  int polled = 0;
  bool stop = false;
  for (int it = 0; it < max_iter && !stop; ++it) {
    {
      Timed t(h, &h->ev_mv, s);
      CK(launch_full_matvec(v, s));
    }
    CK(launch_pcgnr_update(v, lambda, s));
    if (rel_tol > 0.0 && (it + 1) % chunk == 0 && it + 1 < max_iter) {
      const int slot = polled & 1;
      if (polled >= 2) {
        CK(cudaEventSynchronize(h->poll_ev[slot]));
        if (h->h_flags[slot]) stop = true;
      }
      if (!stop) {
        CK(cudaMemcpyAsync(&h->h_flags[slot], &v.pcg->done, sizeof(int), cudaMemcpyDeviceToHost, s));
        CK(cudaEventRecord(h->poll_ev[slot], s));
        ++polled;
      }
    }
  }
  CK(launch_pcgnr_finish(v, s));
  account(h);
  h->have_delta = true;
  h->prepared = false;  // v.b holds -g_c, not a Schur right-hand side
  return 0;
}

void fill_pcg_info(const caspar_ba* h, caspar_ba_pcg_info* info) {
  const PcgScalars& p = *h->h_pcg;
  info->iterations = p.iters;
  info->converged = p.converged;
  // after a breakdown rr belongs to an update that never ran: report the last completed iteration's residual
  const double rr = p.breakdown ? (p.iters > 0 ? p.rr_last : p.bnorm2) : p.rr;
  info->rel_residual = p.bnorm2 > 0.0 ? std::sqrt(rr / p.bnorm2) : 0.0;
  info->rz0 = p.iters > 0 ? p.rz0 : p.rz[0];
  info->rz = p.rz[p.iters & 1];
}

int check_numeric(caspar_ba* h) {
  if (h->h_step->bad_block) return fail(h, CASPAR_BA_ENUMERIC, "a damped 9x9 or 3x3 block is not positive definite");
  if (h->h_pcg->breakdown) return fail(h, CASPAR_BA_ENUMERIC, "PCG breakdown: p.Sp <= 0 or not finite");
  return 0;
}

}  // namespace

// =================================================================================================
extern "C" {

static int create_impl(const caspar_ba_problem* pb, void* cuda_stream, caspar_ba_t** out, caspar_ba*& h) {
  const double t_begin = now_s();
  if (pb->num_cameras < 0 || pb->num_points < 0 || pb->num_observations < 0)
    return create_fail(CASPAR_BA_EINVAL, "negative size");
  if (pb->num_observations > 0 && (!pb->observations || !pb->camera_index || !pb->point_index))
    return create_fail(CASPAR_BA_EINVAL, "null observation / index array");
  if ((pb->num_cameras > 0 && !pb->cameras) || (pb->num_points > 0 && !pb->points))
    return create_fail(CASPAR_BA_EINVAL, "null parameter array");
  if (pb->robust_loss != 0 && pb->robust_loss != 1) return create_fail(CASPAR_BA_EINVAL, "robust_loss must be 0 or 1");
  if (pb->robust_loss == 1 && !(pb->robust_scale > 0.f))
    return create_fail(CASPAR_BA_EINVAL, "robust_scale must be positive with the Cauchy loss");
  if (pb->damping_mode != 0 && pb->damping_mode != 1) return create_fail(CASPAR_BA_EINVAL, "damping_mode must be 0 or 1");
  if (pb->camera_model != 0 && pb->camera_model != 1) return create_fail(CASPAR_BA_EINVAL, "camera_model must be 0 or 1");
  if (!(pb->depth_epsilon >= 0.f)) return create_fail(CASPAR_BA_EINVAL, "depth_epsilon must be >= 0");
  if (pb->num_observations > 0 && (pb->num_cameras == 0 || pb->num_points == 0))
    return create_fail(CASPAR_BA_EINVAL, "observations without cameras or points");
  int forced = 0;
  if (const char* env = std::getenv("CASPAR_BA_TILE")) forced = std::atoi(env);
  h = new caspar_ba();
  h->pb = *pb;
  cudaGetDevice(&h->device);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const long long n = pb->num_observations;
  auto bail = [&](int code, const std::string& msg) {
    caspar_ba_destroy(h);
    h = nullptr;
    return create_fail(code, msg);
  };
  auto cuda_bail = [&](cudaError_t e, const char* where) {
    return bail(e == cudaErrorMemoryAllocation ? CASPAR_BA_ENOMEM : CASPAR_BA_ECUDA,
                std::string(where) + ": " + cudaGetErrorString(e));
  };
  // Index arrays that live on the DEVICE are validated there first: a bad index is reported without
  // moving 8 bytes per observation to the host.
  if (n > 0) {
    cudaPointerAttributes ac{}, ap{};
    const bool dev_c = cudaPointerGetAttributes(&ac, pb->camera_index) == cudaSuccess &&
                       (ac.type == cudaMemoryTypeDevice || ac.type == cudaMemoryTypeManaged);
    const bool dev_p = cudaPointerGetAttributes(&ap, pb->point_index) == cudaSuccess &&
                       (ap.type == cudaMemoryTypeDevice || ap.type == cudaMemoryTypeManaged);
    cudaGetLastError();
    if (dev_c && dev_p) {
      unsigned long long* flag = nullptr;
      unsigned long long bad = ~0ull;
      cudaError_t e = cudaMalloc(&flag, sizeof(unsigned long long));
      if (e == cudaSuccess) e = cudaMemcpyAsync(flag, &bad, sizeof bad, cudaMemcpyHostToDevice, s);
      if (e == cudaSuccess) e = launch_validate_indices(pb->camera_index, pb->point_index, n, pb->num_cameras, pb->num_points, flag, s);
      if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, flag, sizeof bad, cudaMemcpyDeviceToHost, s);
      if (e == cudaSuccess) e = cudaStreamSynchronize(s);
      if (flag) cudaFree(flag);
      take_launch_count();
      if (e != cudaSuccess) return cuda_bail(e, "validation of the index arrays");
      if (bad != ~0ull)
        return bail(CASPAR_BA_EINVAL, "camera_index / point_index out of range at observation " + std::to_string(bad) + " (validated on the device)");
    }
  }
  // S0 runs on the host, so the indices come to the host (the source may be device or host memory; host arrays are
  // validated there, in the same pass that counts the tracks).
  std::vector<int> cam_idx((size_t)n), pt_idx((size_t)n);
  if (n > 0) {
    cudaError_t e = cudaMemcpy(cam_idx.data(), pb->camera_index, sizeof(int) * (size_t)n, cudaMemcpyDefault);
    if (e == cudaSuccess) e = cudaMemcpy(pt_idx.data(), pb->point_index, sizeof(int) * (size_t)n, cudaMemcpyDefault);
    if (e != cudaSuccess) return cuda_bail(e, "copy of the index arrays");
  }
  Reordered ro;
  {
    std::string err;
    const double t0 = now_s();
    const int rc = reorder_observations(pb->num_cameras, pb->num_points, n, cam_idx.data(), pt_idx.data(), forced, &ro, &err);
    h->reorder_s = now_s() - t0;
    if (rc) return bail(rc, err);
  }
  View& v = h->v;
  v.nc = pb->num_cameras;
  v.np = pb->num_points;
  v.np_obs = ro.np_obs;
  v.T = ro.T;
  v.num_tiles = ro.num_tiles;
  v.n_slots = ro.n_slots;
  v.num_chunks = (int)ro.chunk_cam.size();
  v.num_hot = (int)ro.hot_list.size();
  v.robust = pb->robust_loss;
  v.robust_c2 = pb->robust_scale * pb->robust_scale;
  v.robust_inv_c2 = pb->robust_loss ? 1.0 / ((double)pb->robust_scale * (double)pb->robust_scale) : 0.0;
  v.damping_mode = pb->damping_mode;
  v.camera_model = pb->camera_model;
  v.shard_root = 1;
  v.depth_eps = pb->depth_epsilon;
  v.cameras = pb->cameras;
  v.points = pb->points;
  v.max_pts_per_tile = ro.max_pts_per_tile;
  v.meta_max_bytes = ro.meta_max_bytes;
  {
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device);
    v.num_sms = sms > 0 ? sms : 148;
  }
  {
    const char* env = std::getenv("CASPAR_BA_PIPELINE");  // "0" selects the one-block-per-tile Schur pass
    v.pipeline = (!(env && env[0] == '0') && pipelined_matvec_possible(v)) ? 1 : 0;
    env = std::getenv("CASPAR_BA_LIN_PIPELINE");  // "0" selects the one-block-per-tile linearize / cost kernels
    v.lin_pipeline = (!(env && env[0] == '0') && pipelined_linearize_possible(v)) ? 1 : 0;
  }
  h->camera_runs = ro.camera_runs;
  h->arena_bytes = carve(h, nullptr, ro);
  cudaError_t e = cudaMalloc(&h->arena, h->arena_bytes);
  if (e != cudaSuccess) return bail(CASPAR_BA_ENOMEM, "device arena of " + std::to_string(h->arena_bytes) + " bytes: " + cudaGetErrorString(e));
  carve(h, h->arena, ro);
  e = cudaMemsetAsync(h->arena, 0, h->arena_bytes, s);
  if (e == cudaSuccess) e = upload(v.cam, ro.cam, s);
  if (e == cudaSuccess) e = upload(v.obs_of_slot, ro.obs_of_slot, s);
  if (e == cudaSuccess) e = upload(v.rank, ro.rank, s);
  if (e == cudaSuccess) e = upload(v.rankpid, ro.rankpid, s);
  if (e == cudaSuccess) e = upload(v.rankpid32, ro.rankpid32, s);
  if (e == cudaSuccess) e = upload(v.tile_pt, ro.tile_pt, s);
  if (e == cudaSuccess) e = upload(v.run_begin, ro.run_begin, s);
  if (e == cudaSuccess) e = upload(v.run_cam, ro.run_cam, s);
  if (e == cudaSuccess) e = upload(v.run_slot, ro.run_slot, s);
  if (e == cudaSuccess) e = upload(v.tile_dir, ro.tile_dir, s);
  if (e == cudaSuccess) e = upload(v.tile_meta, ro.tile_meta, s);
  if (e == cudaSuccess) e = upload(v.pt_ptr, ro.pt_ptr, s);
  if (e == cudaSuccess) e = upload(v.pt_perm, ro.pt_perm, s);
  if (e == cudaSuccess) e = upload(v.cslot, ro.cslot, s);
  if (e == cudaSuccess) e = upload(v.chunk_cam, ro.chunk_cam, s);
  if (e == cudaSuccess) e = upload(v.chunk_begin, ro.chunk_begin, s);
  if (e == cudaSuccess) e = upload(v.cam_chunk_ptr, ro.cam_chunk_ptr, s);
  if (e == cudaSuccess) e = upload(v.hot_of_cam, ro.hot_of_cam, s);
  if (e == cudaSuccess) e = upload(v.hot_list, ro.hot_list, s);
  // pixels: the caller's array may live on either side; stage through the device if it is host memory
  float* obs_dev = nullptr;
  if (e == cudaSuccess && n > 0) {
    cudaPointerAttributes attr{};
    bool on_device = cudaPointerGetAttributes(&attr, pb->observations) == cudaSuccess &&
                     (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged);
    cudaGetLastError();
    const float* src = pb->observations;
    if (!on_device) {
      e = cudaMalloc(&obs_dev, sizeof(float) * 2 * (size_t)n);
      if (e == cudaSuccess) e = cudaMemcpyAsync(obs_dev, pb->observations, sizeof(float) * 2 * (size_t)n, cudaMemcpyDefault, s);
      src = obs_dev;
    }
    if (e == cudaSuccess) e = launch_gather_observations(v, src, const_cast<float2*>(v.px), s);
  }
  if (e == cudaSuccess) e = configure_kernels(v);
  if (e == cudaSuccess) e = cudaMallocHost(&h->h_pcg, sizeof(PcgScalars));
  if (e == cudaSuccess) e = cudaMallocHost(&h->h_step, sizeof(StepScalars));
  if (e == cudaSuccess) e = cudaMallocHost(&h->h_flags, 2 * sizeof(int));
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->poll_ev[0], cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->poll_ev[1], cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);  // the host vectors above die with this scope
  if (obs_dev) cudaFree(obs_dev);
  account(h);
  if (e != cudaSuccess) return cuda_bail(e, "caspar_ba_create");
  h->create_s = now_s() - t_begin;
  *out = h;
  return CASPAR_BA_OK;
}

int caspar_ba_create(const caspar_ba_problem* pb, void* cuda_stream, caspar_ba_t** out) {
  if (!pb || !out) return create_fail(CASPAR_BA_EINVAL, "null argument");
  *out = nullptr;
  caspar_ba* h = nullptr;
  try {  // no exception crosses the C ABI
    return create_impl(pb, cuda_stream, out, h);
  } catch (const std::bad_alloc&) {
    caspar_ba_destroy(h);
    return create_fail(CASPAR_BA_ENOMEM, "host allocation failed");
  } catch (...) {
    caspar_ba_destroy(h);
    return create_fail(CASPAR_BA_ENOMEM, "unexpected exception in caspar_ba_create");
  }
}

void caspar_ba_destroy(caspar_ba_t* h) {
  if (!h) return;
  DeviceGuard on_device(h->device);
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  for (cudaEvent_t e : h->ev_lin) cudaEventDestroy(e);
  for (cudaEvent_t e : h->ev_mv) cudaEventDestroy(e);
  for (cudaEvent_t e : h->poll_ev)
    if (e) cudaEventDestroy(e);
  for (cudaGraphExec_t g : h->chunk_graph)
    if (g) cudaGraphExecDestroy(g);
  if (h->arena2) cudaFree(h->arena2);
  if (h->capture_stream) cudaStreamDestroy(h->capture_stream);
  if (h->h_pcg) cudaFreeHost(h->h_pcg);
  if (h->h_step) cudaFreeHost(h->h_step);
  if (h->h_flags) cudaFreeHost(h->h_flags);
  if (h->arena) cudaFree(h->arena);
  delete h;
}

int caspar_ba_linearize(caspar_ba_t* h, void* cuda_stream, double* cost_out) {
  if (!h) return CASPAR_BA_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  int rc = do_linearize(h, s);
  if (rc) return rc;
  rc = sync_step_scalars(h, s);
  if (rc) return rc;
  h->cost = 0.5 * h->h_step->cost;
  if (cost_out) *cost_out = h->cost;
  if (!std::isfinite(h->cost)) {
    h->linearized = false;
    return fail(h, CASPAR_BA_ENUMERIC, "non-finite cost");
  }
  return CASPAR_BA_OK;
}

int caspar_ba_cost(caspar_ba_t* h, void* cuda_stream, double* cost_out) {
  if (!h || !cost_out) return CASPAR_BA_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  View& v = h->v;
  // evaluated in the trial buffers so that a cached linearization stays untouched
  CK(launch_pack_points(v, v.points, v.pts_trial, s));
  CK(launch_camera_prepass(v, v.cameras, v.cam_table_trial, s));
  CK(launch_cost(v, v.pts_trial, v.cam_table_trial, &v.step->trial_cost, s));
  account(h);
  int rc = shard_sum(h, &v.step->trial_cost, 1, nullptr, 0, s);
  if (rc) return rc;
  rc = sync_step_scalars(h, s);
  if (rc) return rc;
  *cost_out = 0.5 * h->h_step->trial_cost;
  return std::isfinite(*cost_out) ? CASPAR_BA_OK : fail(h, CASPAR_BA_ENUMERIC, "non-finite cost");
}

// S9 without a handle and without an allocation: the scratch is the fixed device array of ba_kernels.cu.  The success
// path touches no allocator (host or device); only a failure builds an error string.
int caspar_ba_cost_static(const caspar_ba_problem* pb, double* cost_out_dev, void* cuda_stream) {
  if (!pb || !cost_out_dev) return create_fail(CASPAR_BA_EINVAL, "null problem / cost_out_dev");
  if (pb->num_cameras < 0 || pb->num_points < 0 || pb->num_observations < 0)
    return create_fail(CASPAR_BA_EINVAL, "negative size");
  if (pb->num_cameras > CASPAR_BA_STATIC_MAX_CAMERAS)
    return create_fail(CASPAR_BA_EINVAL, "caspar_ba_cost_static: " + std::to_string(pb->num_cameras) +
                                             " cameras exceed CASPAR_BA_STATIC_MAX_CAMERAS = " +
                                             std::to_string(CASPAR_BA_STATIC_MAX_CAMERAS) +
                                             " (the fixed scratch array holds one 144-byte table row per camera)");
  if (pb->num_observations > 0 && (!pb->observations || !pb->camera_index || !pb->point_index))
    return create_fail(CASPAR_BA_EINVAL, "null observation / index array");
  if ((pb->num_cameras > 0 && !pb->cameras) || (pb->num_points > 0 && !pb->points))
    return create_fail(CASPAR_BA_EINVAL, "null parameter array");
  if (pb->robust_loss != 0 && pb->robust_loss != 1) return create_fail(CASPAR_BA_EINVAL, "robust_loss must be 0 or 1");
  if (pb->robust_loss == 1 && !(pb->robust_scale > 0.f))
    return create_fail(CASPAR_BA_EINVAL, "robust_scale must be positive with the Cauchy loss");
  if (!(pb->depth_epsilon >= 0.f)) return create_fail(CASPAR_BA_EINVAL, "depth_epsilon must be >= 0");
  int device = -1;
  cudaError_t e = cudaGetDevice(&device);
  if (e != cudaSuccess) return create_fail(CASPAR_BA_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  // the kernels dereference every pointer on the current device: a host pointer would fault there
  const void* ptrs[] = {pb->cameras, pb->points, pb->observations, pb->camera_index, pb->point_index, cost_out_dev};
  const char* names[] = {"cameras", "points", "observations", "camera_index", "point_index", "cost_out_dev"};
  for (int i = 0; i < 6; ++i) {
    if (!ptrs[i]) continue;
    cudaPointerAttributes a;
    const bool ok = cudaPointerGetAttributes(&a, ptrs[i]) == cudaSuccess &&
                    (a.type == cudaMemoryTypeManaged || (a.type == cudaMemoryTypeDevice && a.device == device));
    if (!ok) {
      cudaGetLastError();
      return create_fail(CASPAR_BA_EINVAL, std::string("caspar_ba_cost_static: ") + names[i] +
                                               " is not device memory of the current device");
    }
  }
  e = launch_cost_static(pb->num_cameras, pb->num_points, pb->num_observations, pb->cameras, pb->points,
                         pb->observations, pb->camera_index, pb->point_index, pb->robust_loss, pb->robust_scale,
                         pb->depth_epsilon, cost_out_dev, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess)
    return create_fail(CASPAR_BA_ECUDA, std::string("caspar_ba_cost_static: ") + cudaGetErrorString(e));
  return CASPAR_BA_OK;
}

int caspar_ba_pcg_solve(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, void* cuda_stream,
                        caspar_ba_pcg_info* info) {
  if (!h || max_iter < 0 || !(lambda >= 0.f) || !(rel_tol >= 0.f)) return CASPAR_BA_EINVAL;
  if (!h->linearized) return fail(h, CASPAR_BA_ESTATE, "pcg_solve before linearize");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  int rc = do_pcg(h, (double)lambda, (double)rel_tol, max_iter, s);
  if (rc) return rc;
  rc = shard_sum(h, &h->v.step->jd2, 3, nullptr, 0, s);  // shards: jd2, dg, bad_block
  if (rc) return rc;
  rc = sync_step_scalars(h, s);
  if (rc) return rc;
  if (info) fill_pcg_info(h, info);
  return check_numeric(h);
}

int caspar_ba_pcgnr_solve(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, void* cuda_stream,
                          caspar_ba_pcg_info* info) {
  if (!h || max_iter < 0 || !(lambda >= 0.f) || !(rel_tol >= 0.f)) return CASPAR_BA_EINVAL;
  if (!h->linearized) return fail(h, CASPAR_BA_ESTATE, "pcgnr_solve before linearize");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  int rc = do_pcgnr(h, (double)lambda, (double)rel_tol, max_iter, s);
  if (rc) return rc;
  rc = sync_step_scalars(h, s);
  if (rc) return rc;
  if (info) fill_pcg_info(h, info);
  return check_numeric(h);
}

int caspar_ba_set_linear_solver(caspar_ba_t* h, int32_t mode) {
  if (!h || (mode != 0 && mode != 1)) return CASPAR_BA_EINVAL;
  h->linear_solver = mode;
  return CASPAR_BA_OK;
}

int caspar_ba_lm_step(caspar_ba_t* h, float lambda, float rel_tol, int32_t max_iter, int32_t accept_mode,
                      void* cuda_stream, caspar_ba_step_info* info) {
  if (!h || !info || max_iter < 0 || accept_mode < 0 || accept_mode > 2 || !(lambda >= 0.f) || !(rel_tol >= 0.f))
    return CASPAR_BA_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  View& v = h->v;
  std::memset(info, 0, sizeof *info);
  int rc;
  const bool fresh = !h->linearized;
  if (fresh) {
    rc = do_linearize(h, s);
    if (rc) return rc;
  }
  rc = h->linear_solver == 1 ? do_pcgnr(h, (double)lambda, (double)rel_tol, max_iter, s)
                             : do_pcg(h, (double)lambda, (double)rel_tol, max_iter, s);
  if (rc) return rc;
  // trial point and its cost (S9)
  CK(launch_trial_update(v, s));
  CK(launch_camera_prepass(v, v.cams_trial, v.cam_table_trial, s));
  // N2: with fusion on, the trial point gets the FULL linearization (r, J, V, g_p and the cost in one pass) in the
  // other set of arrays; if the step is accepted that IS the next iteration's linearization ("the
  // initial score and the Jacobian are calculated simultaneously, while subsequent runs use the score values from the
  // previous iteration").  (A forced rejection, accept_mode 2, speculates too: the tests use it for rejected steps.)
  const bool speculate = h->fusion != 0 && h->arena2 != nullptr && !h->exchange;  // (not on a sharded handle)
  if (speculate) {
    View w = v;
    for (int i = 0; i < 6; ++i) w.J[i] = h->alt.J[i];
    w.res = h->alt.res; w.V0 = h->alt.V0; w.V1 = h->alt.V1; w.gp = h->alt.gp;
    {
      Timed t(h, &h->ev_lin, s);
      CK(launch_linearize_at(w, v.pts_trial, v.cam_table_trial, s));
    }
    CK(launch_linearize_cost(w, &v.step->trial_cost, s));
  } else {
    CK(launch_cost(v, v.pts_trial, v.cam_table_trial, &v.step->trial_cost, s));
  }
  // shards: the trial cost, |J delta|^2, delta.g and the bad-block count are sums over the shards (contiguous scalars)
  rc = shard_sum(h, &v.step->trial_cost, 4, nullptr, 0, s);
  if (rc) return rc;
  account(h);
  rc = sync_step_scalars(h, s);  // the one host synchronisation of the step
  if (rc) return rc;
  if (fresh) h->cost = 0.5 * h->h_step->cost;
  if (!std::isfinite(h->cost)) {
    h->linearized = false;
    return fail(h, CASPAR_BA_ENUMERIC, "non-finite cost");
  }
  fill_pcg_info(h, &info->pcg);
  // A curvature breakdown after at least one good iteration truncates the solve at the last good iterate
  // (Steihaug-style truncated CG): with fp32 Jacobians the computed Schur operator can lose positive
  // definiteness at lambda ~ 1e-6.  The step is then judged by its gain ratio like any other.
  if (h->h_pcg->breakdown && h->h_pcg->iters >= 1 && !h->h_step->bad_block) h->h_pcg->breakdown = 0;
  // A failed linear solve (a damped block that is not positive definite in fp32, or a breakdown before the
  // first iterate) is a REJECTED step, not an error: parameters and the cached linearization stay, the caller's
  // damping update raises lambda (what every LM driver does with a failed solve).  accept_mode cannot override
  // it: there is no step to accept.
  if (h->h_step->bad_block || h->h_pcg->breakdown) {
    h->err = h->h_step->bad_block ? "linear solve failed: a damped 9x9 or 3x3 block is not positive definite"
                                  : "linear solve failed: PCG breakdown before the first iterate";
    info->cost_before = info->cost_after = h->cost;
    info->model_decrease = 0.0;
    info->rho = -1.0;
    info->accepted = 0;
    info->pcg.converged = 0;
    h->have_delta = false;
    return CASPAR_BA_OK;
  }
  // S10 gain ratio (host scalars)
  info->cost_before = h->cost;
  info->cost_after = 0.5 * h->h_step->trial_cost;
  info->model_decrease = -h->h_step->dg - 0.5 * h->h_step->jd2;
  info->rho = (info->cost_before - info->cost_after) / info->model_decrease;
  bool accept;
  if (accept_mode == 1) accept = true;
  else if (accept_mode == 2) accept = false;
  else  // rho > 0 with an actual decrease: a truncated fp32 solve can make BOTH differences negative
    accept = std::isfinite(info->cost_after) && info->rho > 0.0 && info->cost_after < info->cost_before;
  info->accepted = accept ? 1 : 0;
  if (accept) {
    CK(launch_commit(v, s));
    h->linearized = false;
    h->prepared = false;
    if (speculate && std::isfinite(info->cost_after)) {
      // the trial linearization becomes the current one: swap the two sets, assemble the camera side (S4) from it
      for (int i = 0; i < 6; ++i) std::swap(v.J[i], h->alt.J[i]);
      std::swap(v.res, h->alt.res); std::swap(v.V0, h->alt.V0); std::swap(v.V1, h->alt.V1); std::swap(v.gp, h->alt.gp);
      h->set_parity ^= 1;
      CK(launch_assemble_cameras(v, s));
      h->linearized = true;
      h->have_delta = false;
      h->cost = info->cost_after;
      ++h->speculative_hits;
    }
    account(h);
  } else if (speculate) {
    ++h->speculative_misses;
  }
  return CASPAR_BA_OK;
}

int caspar_ba_set_shard(caspar_ba_t* h, caspar_ba_exchange_fn fn, void* ctx, double* exchange_buffer_dev,
                        size_t exchange_count, int32_t is_root) {
  if (!h) return CASPAR_BA_EINVAL;
  if (!fn) {  // back to a single-GPU problem
    h->exchange = nullptr;
    h->exchange_ctx = nullptr;
    h->xchg = nullptr;
    h->xchg_count = 0;
    h->v.shard_root = 1;
    h->v.det_scalars = 0;
  } else {
    const size_t need = (size_t)kUg * (size_t)h->v.nc + 8;
    if (!exchange_buffer_dev || exchange_count < need)
      return fail(h, CASPAR_BA_EINVAL, "exchange buffer: need at least 54 * num_cameras + 8 doubles (" + std::to_string(need) + ")");
    h->exchange = fn;
    h->exchange_ctx = ctx;
    h->xchg = exchange_buffer_dev;
    h->xchg_count = exchange_count;
    h->v.shard_root = is_root ? 1 : 0;
    h->v.det_scalars = 1;
  }
  h->linearized = false;
  h->prepared = false;
  h->have_delta = false;
  return CASPAR_BA_OK;
}

int caspar_ba_set_fusion(caspar_ba_t* h, int32_t mode) {
  if (!h || (mode != 0 && mode != 1)) return CASPAR_BA_EINVAL;
  DeviceGuard on_device(h->device);
  if (mode == 1 && !h->arena2) {
    const size_t S = (size_t)h->v.n_slots, NP = (size_t)h->v.np;
    Carver sizer(nullptr);
    auto lay = [&](Carver& c) {
      for (int i = 0; i < 6; ++i) h->alt.J[i] = c.take<float4>(S);
      h->alt.res = c.take<float2>(S);
      h->alt.V0 = c.take<float4>(NP);
      h->alt.V1 = c.take<float2>(NP);
      h->alt.gp = c.take<float4>(NP);
    };
    lay(sizer);
    h->arena2_bytes = (sizer.off + 255) & ~size_t(255);
    cudaError_t e = cudaMalloc(&h->arena2, h->arena2_bytes);
    if (e != cudaSuccess) {
      h->arena2 = nullptr;
      h->alt = caspar_ba::LinSet();
      return fail(h, CASPAR_BA_ENOMEM, "second set of linearization arrays (" + std::to_string(h->arena2_bytes) + " bytes): " + cudaGetErrorString(e));
    }
    e = cudaMemset(h->arena2, 0, h->arena2_bytes);  // padding slots and unobserved points stay zero, as in the arena
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemset(arena2)");
    Carver real(h->arena2);
    lay(real);
  }
  h->fusion = mode;
  return CASPAR_BA_OK;
}

int caspar_ba_solve(caspar_ba_t* h, int32_t iterations, float lambda0, float rel_tol, int32_t max_iter,
                    void* cuda_stream, caspar_ba_step_info* infos, float* lambdas) {
  if (!h || iterations < 0) return CASPAR_BA_EINVAL;
  double lambda = lambda0, nu = 2.0;
  for (int it = 0; it < iterations; ++it) {
    caspar_ba_step_info info;
    if (lambdas) lambdas[it] = (float)lambda;
    int rc = caspar_ba_lm_step(h, (float)lambda, rel_tol, max_iter, 0, cuda_stream, &info);
    if (rc) return rc;
    if (infos) infos[it] = info;
    if (info.accepted) {  // Nielsen's update (Madsen, Nielsen, Tingleff 2004, eq. 3.16 / PAPER.md:163)
      const double c = 2.0 * info.rho - 1.0;
      lambda *= std::fmax(1.0 / 3.0, 1.0 - c * c * c);
      nu = 2.0;
    } else {
      lambda *= nu;
      nu *= 2.0;
    }
  }
  return CASPAR_BA_OK;
}

int caspar_ba_set_parameters_host(caspar_ba_t* h, const float* cameras_host, const float* points_host,
                                  void* cuda_stream) {
  if (!h || (h->v.nc > 0 && !cameras_host) || (h->v.np > 0 && !points_host)) return CASPAR_BA_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  if (h->v.nc > 0)
    CK(cudaMemcpyAsync(h->v.cameras, cameras_host, sizeof(float) * 9 * (size_t)h->v.nc, cudaMemcpyHostToDevice, s));
  if (h->v.np > 0)
    CK(cudaMemcpyAsync(h->v.points, points_host, sizeof(float) * 3 * (size_t)h->v.np, cudaMemcpyHostToDevice, s));
  h->linearized = false;
  h->prepared = false;
  h->have_delta = false;
  return CASPAR_BA_OK;
}

int caspar_ba_get_parameters_host(caspar_ba_t* h, float* cameras_host, float* points_host, void* cuda_stream) {
  if (!h || (h->v.nc > 0 && !cameras_host) || (h->v.np > 0 && !points_host)) return CASPAR_BA_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  if (h->v.nc > 0)
    CK(cudaMemcpyAsync(cameras_host, h->v.cameras, sizeof(float) * 9 * (size_t)h->v.nc, cudaMemcpyDeviceToHost, s));
  if (h->v.np > 0)
    CK(cudaMemcpyAsync(points_host, h->v.points, sizeof(float) * 3 * (size_t)h->v.np, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return CASPAR_BA_OK;
}

int caspar_ba_export(caspar_ba_t* h, int32_t what, double* device_dst, size_t count, void* cuda_stream) {
  if (!h || !device_dst) return CASPAR_BA_EINVAL;
  const size_t N = (size_t)h->pb.num_observations, nc = (size_t)h->v.nc, np = (size_t)h->v.np;
  size_t need = 0;
  switch (what) {
    case CASPAR_BA_RESIDUALS: need = 2 * N; break;
    case CASPAR_BA_JC: need = 18 * N; break;
    case CASPAR_BA_JP: need = 6 * N; break;
    case CASPAR_BA_U: need = 81 * nc; break;
    case CASPAR_BA_V: need = 9 * np; break;
    case CASPAR_BA_G: case CASPAR_BA_DELTA: need = 9 * nc + 3 * np; break;
    case CASPAR_BA_SCHUR_RHS: need = 9 * nc; break;
    case CASPAR_BA_PRECONDITIONER: need = 81 * nc; break;
    default: return fail(h, CASPAR_BA_EINVAL, "unknown export id");
  }
  if (count != need) return fail(h, CASPAR_BA_EINVAL, "export: wrong element count");
  const bool solve_product = what == CASPAR_BA_SCHUR_RHS || what == CASPAR_BA_DELTA;
  if (what == CASPAR_BA_PRECONDITIONER ? !h->prepared : (solve_product ? !h->have_delta : !h->linearized))
    return fail(h, CASPAR_BA_ESTATE, "export: nothing cached");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  CK(launch_export(h->v, what, device_dst, s));
  account(h);
  CK(cudaStreamSynchronize(s));
  return CASPAR_BA_OK;
}

int caspar_ba_schur_matvec(caspar_ba_t* h, float lambda, const double* p_dev, double* q_dev, void* cuda_stream) {
  if (!h || !p_dev || !q_dev || !(lambda >= 0.f)) return CASPAR_BA_EINVAL;
  if (!h->linearized) return fail(h, CASPAR_BA_ESTATE, "schur_matvec before linearize");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  DeviceGuard on_device(h->device);
  int rc = do_prepare(h, (double)lambda, h->preconditioner, s);
  if (rc) return rc;
  CK(cudaMemsetAsync(h->v.pcg, 0, sizeof(PcgScalars), s));
  {
    Timed t(h, &h->ev_mv, s);  // brackets load + pass + finish; the pass dominates
    if (h->exchange) {
      CK(launch_matvec_standalone(h->v, p_dev, q_dev, s, 1));
      rc = shard_sum(h, h->v.q, 9 * (size_t)h->v.nc, nullptr, 0, s);
      if (rc) return rc;
      CK(launch_matvec_standalone(h->v, p_dev, q_dev, s, 2));
    } else {
      CK(launch_matvec_standalone(h->v, p_dev, q_dev, s));
    }
  }
  account(h);
  h->have_delta = false;  // x / p buffers were reused
  rc = sync_step_scalars(h, s);
  if (rc) return rc;
  return check_numeric(h);
}

int caspar_ba_set_preconditioner(caspar_ba_t* h, int32_t mode) {
  if (!h || (mode != 0 && mode != 1)) return CASPAR_BA_EINVAL;
  h->preconditioner = mode;  // do_prepare rebuilds the blocks when the mode they were built for differs
  return CASPAR_BA_OK;
}

int caspar_ba_get_stats(caspar_ba_t* h, caspar_ba_stats* out) {
  if (!h || !out) return CASPAR_BA_EINVAL;
  DeviceGuard on_device(h->device);
  if (h->profiling && (!h->ev_lin.empty() || !h->ev_mv.empty())) {
    CK(cudaStreamSynchronize(h->prof_stream));
    drain_events(h);
  }
  out->tile_slots = h->v.T;
  out->num_tiles = h->v.num_tiles;
  out->padded_slots = h->v.n_slots;
  out->camera_runs = h->camera_runs;
  out->arena_bytes = (int64_t)h->arena_bytes;
  out->kernels_launched = h->launches;
  out->linearize_ms_total = h->lin_ms;
  out->matvec_ms_total = h->mv_ms;
  out->linearize_count = h->lin_n;
  out->matvec_count = h->mv_n;
  out->matvec_pipelined = h->v.pipeline;
  out->pipeline_stages = h->v.pipeline ? pipeline_stages(h->v) : 0;
  out->num_hot_cameras = h->v.num_hot;
  out->linearize_pipelined = h->v.lin_pipeline;
  out->device = h->device;
  out->create_seconds = h->create_s;
  out->reorder_seconds = h->reorder_s;
  out->speculative_hits = h->speculative_hits;
  out->speculative_misses = h->speculative_misses;
  out->arena2_bytes = (int64_t)h->arena2_bytes;
  out->shard_exchanges = h->exchanges;
  return CASPAR_BA_OK;
}

int caspar_ba_set_profiling(caspar_ba_t* h, int32_t enable) {
  if (!h) return CASPAR_BA_EINVAL;
  DeviceGuard on_device(h->device);
  if (h->prof_stream || !h->ev_lin.empty() || !h->ev_mv.empty()) {
    cudaStreamSynchronize(h->prof_stream);
    drain_events(h);
  }
  h->profiling = enable != 0;
  h->lin_ms = h->mv_ms = 0.0;
  h->lin_n = h->mv_n = 0;
  h->launches = 0;
  return CASPAR_BA_OK;
}

const char* caspar_ba_last_error(const caspar_ba_t* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

// ---- S0 on its own (host only) ------------------------------------------------------------------
struct caspar_ba_layout {
  Reordered ro;
};

int caspar_ba_layout_create(int32_t nc, int32_t np, int64_t n, const int32_t* cam_index, const int32_t* point_index,
                            int32_t tile, caspar_ba_layout_t** out) {
  if (!out || nc < 0 || np < 0 || n < 0 || (n > 0 && (!cam_index || !point_index)))
    return create_fail(CASPAR_BA_EINVAL, "null argument or negative size");
  *out = nullptr;
  caspar_ba_layout* l = nullptr;
  std::string err;
  int rc;
  try {
    l = new caspar_ba_layout();
    rc = reorder_observations(nc, np, n, cam_index, point_index, tile, &l->ro, &err);
  } catch (const std::bad_alloc&) {
    rc = CASPAR_BA_ENOMEM;
    err = "host allocation failed";
  } catch (...) {
    rc = CASPAR_BA_ENOMEM;
    err = "unexpected exception in caspar_ba_layout_create";
  }
  if (rc) {
    delete l;
    return create_fail(rc, err);
  }
  *out = l;
  return CASPAR_BA_OK;
}

int caspar_ba_layout_get_info(const caspar_ba_layout_t* l, caspar_ba_layout_info* info) {
  if (!l || !info) return CASPAR_BA_EINVAL;
  info->tile_slots = l->ro.T;
  info->num_tiles = l->ro.num_tiles;
  info->observed_points = l->ro.np_obs;
  info->num_chunks = (int32_t)l->ro.chunk_cam.size();
  info->padded_slots = l->ro.n_slots;
  info->camera_runs = l->ro.camera_runs;
  return CASPAR_BA_OK;
}

int caspar_ba_layout_copy(const caspar_ba_layout_t* l, int32_t which, void* dst, size_t bytes) {
  if (!l || !dst) return CASPAR_BA_EINVAL;
  const Reordered& r = l->ro;
  const void* src = nullptr;
  size_t have = 0;
  const size_t slots = (size_t)r.n_slots;
  auto pick = [&](const void* p, size_t n) { src = p; have = n; };
  switch (which) {
    case 0: pick(r.obs_of_slot.data(), slots * sizeof(int)); break;
    case 1: pick(r.cam.data(), slots * sizeof(int)); break;
    case 2: pick(r.rank.data(), slots * sizeof(unsigned short)); break;
    case 3: pick(r.tile_pt.data(), r.tile_pt.size() * sizeof(int)); break;
    case 4: pick(r.run_begin.data(), r.run_begin.size() * sizeof(int)); break;
    case 5: pick(r.run_cam.data(), r.run_cam.size() * sizeof(int)); break;
    case 6: pick(r.run_slot.data(), r.run_slot.size() * sizeof(unsigned short)); break;
    case 7: pick(r.pt_ptr.data(), r.pt_ptr.size() * sizeof(int)); break;
    case 8: pick(r.pt_perm.data(), r.pt_perm.size() * sizeof(int)); break;
    case 9: pick(r.cslot.data(), (size_t)(r.pt_ptr.empty() ? 0 : r.pt_ptr.back()) * sizeof(int)); break;
    case 10: pick(r.chunk_cam.data(), r.chunk_cam.size() * sizeof(int)); break;
    case 11: pick(r.chunk_begin.data(), r.chunk_begin.size() * sizeof(int)); break;
    default: return CASPAR_BA_EINVAL;
  }
  if (bytes != have) return CASPAR_BA_EINVAL;
  if (have) std::memcpy(dst, src, have);
  return CASPAR_BA_OK;
}

void caspar_ba_layout_destroy(caspar_ba_layout_t* l) { delete l; }

}  // extern "C"
