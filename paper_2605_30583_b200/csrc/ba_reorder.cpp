// ba_reorder.cpp — step S0: one-off reordering of the observations at create (host side).
//
// "observations reordered (sorted by point, with camera-side segments)" — BASELINE.json north_star.
// The tile metadata built here plays the role of the paper's SharedIndex arrays:
// a block-local sorted list of unique camera indices plus a per-thread target, built once and reused
// by every kernel.  Nothing below is copied from the paper; it describes no algorithm for this.
//
//   1. points are ordered by (lowest camera id that observes them, caller id): points that share
//      cameras end up in the same tile, which keeps the number of camera runs per tile small;
//      unobserved points go last and belong to no tile;
//   2. points are packed greedily into tiles of at most T observations (whole points only);
//   3. inside a tile, slots are sorted by (camera id, internal point id): equal-camera runs are
//      contiguous; `rank` gives each slot's position in the tile's point-major order;
//   4. a camera-ordered list of slots (chunks of <= kChunkSlots) drives the camera-block assembly.
#include <algorithm>
#include <cstdlib>
#include <numeric>

#include "ba_internal.h"

namespace cba {

int reorder_observations(int nc, int np, long long n, const int* cam_idx, const int* pt_idx, int forced_tile,
                         Reordered* out, std::string* err) {
  if (n >= (1LL << 31) - 4096) {
    *err = "more than 2^31 observations are not supported";
    return CASPAR_BA_EINVAL;
  }
  // --- validate, count tracks, lowest camera per point -----------------------------------------
  std::vector<int> track(np, 0), key(np, nc), key_hi(np, -1);
  for (long long i = 0; i < n; ++i) {
    int c = cam_idx[i], k = pt_idx[i];
    if (c < 0 || c >= nc || k < 0 || k >= np) {
      *err = "camera_index / point_index out of range at observation " + std::to_string(i);
      return CASPAR_BA_EINVAL;
    }
    track[k]++;
    if (c < key[k]) key[k] = c;
    if (c > key_hi[k]) key_hi[k] = c;
  }
  int max_track = 0;
  for (int k = 0; k < np; ++k) max_track = std::max(max_track, track[k]);
  if (max_track > CASPAR_BA_MAX_TRACK) {
    *err = "a point has " + std::to_string(max_track) + " observations; the limit is " +
           std::to_string(CASPAR_BA_MAX_TRACK);
    return CASPAR_BA_EINVAL;
  }
  int T = forced_tile;
  if (T != 0 && T != 128 && T != 192 && T != 256 && T != 512 && T != 1024) {
    *err = "tile size must be 0 (automatic), 128, 192, 256, 512 or 1024; got " + std::to_string(forced_tile);
    return CASPAR_BA_EINVAL;
  }
  if (T == 0) T = 256;  // three consumer groups of the pipelined matvec per SM
  while (T < max_track) T = T == 192 ? 256 : T * 2;  // a tile holds whole points: grow to the longest track

  // --- 1. internal point order: counting sort by key (stable -> ties by caller id) --------------
  std::vector<int> bucket(nc + 2, 0);
  for (int k = 0; k < np; ++k) bucket[key[k] + 1]++;
  for (int c = 0; c <= nc; ++c) bucket[c + 1] += bucket[c];
  std::vector<int>& perm = out->pt_perm;
  perm.assign(np, 0);
  std::vector<int> internal_of(np);
  {
    std::vector<int> fill(bucket.begin(), bucket.end() - 1);
    for (int k = 0; k < np; ++k) {
      int pos = fill[key[k]]++;
      perm[pos] = k;
      internal_of[k] = pos;
    }
  }
  int np_obs = bucket[nc];  // points with key < nc, i.e. observed at least once
  // Inside a lowest-camera bucket the points go by their HIGHEST camera id (ties by caller id): points that agree on
  // both ends of their camera set mostly agree on the rest, so a tile of ~40 consecutive points sees fewer distinct
  // cameras -- 0.180 -> 0.125 camera runs per observation on Large, 0.65 -> 0.56 on Skewed, 0.095 -> 0.071 on Mid --
  // i.e. fewer segment ends in the camera-side walk, fewer REDs and camera-row gathers: Schur matvec 0.719 -> 0.679 ms on
  // Large.  A greedy fill with a 64 / 256-point lookahead on top gained only 0.125 -> 0.121 / 0.118.
#pragma omp parallel for schedule(dynamic, 16)
  for (int c = 0; c < nc; ++c)
    std::stable_sort(perm.begin() + bucket[c], perm.begin() + bucket[c + 1],
                     [&](int a, int b) { return key_hi[a] < key_hi[b]; });
  for (int pos = 0; pos < np_obs; ++pos) internal_of[perm[pos]] = pos;
  out->np_obs = np_obs;
  out->pt_ptr.assign(np_obs + 1, 0);
  for (int a = 0; a < np_obs; ++a) out->pt_ptr[a + 1] = out->pt_ptr[a] + track[perm[a]];

  // observations grouped by internal point (caller's order inside a point)
  std::vector<int> obs_by_pt(n > 0 ? n : 1);
  {
    std::vector<int> fill(out->pt_ptr.begin(), out->pt_ptr.end() - 1);
    for (long long i = 0; i < n; ++i) obs_by_pt[fill[internal_of[pt_idx[i]]]++] = (int)i;
  }

  // --- 2. greedy tiles of whole points ---------------------------------------------------------
  std::vector<int>& tile_pt = out->tile_pt;
  tile_pt.clear();
  tile_pt.push_back(0);
  {
    int used = 0;
    for (int a = 0; a < np_obs; ++a) {
      int len = track[perm[a]];
      if (used + len > T) {
        tile_pt.push_back(a);
        used = 0;
      }
      used += len;
    }
    if (np_obs > 0) tile_pt.push_back(np_obs);
  }
  int num_tiles = (int)tile_pt.size() - 1;
  out->T = T;
  out->num_tiles = num_tiles;
  out->n_slots = (long long)num_tiles * T;
  out->obs_of_slot.assign(out->n_slots > 0 ? out->n_slots : 1, -1);
  out->cam.assign(out->n_slots > 0 ? out->n_slots : 1, -1);
  out->rank.assign(out->n_slots > 0 ? out->n_slots : 1, 0);
  // rank | local point id << 8, for the pipelined matvec (tiles of <= 256 slots: both fit a byte)
  out->rankpid.assign(T <= 256 && out->n_slots > 0 ? out->n_slots : 1, 0);
  out->rankpid32.assign(T > 256 && out->n_slots > 0 ? out->n_slots : 1, 0);
  out->run_begin.assign(num_tiles + 1, 0);

  // --- 3. in-tile sort by (camera, point-major position) and run tables -------------------------
  std::vector<int> runs_per_tile(num_tiles, 0);
#pragma omp parallel
  {
    std::vector<unsigned long long> keys;
    std::vector<unsigned short> pid_of_r;
    std::vector<unsigned char> taken;
#pragma omp for schedule(dynamic, 64)
    for (int t = 0; t < num_tiles; ++t) {
      int base = out->pt_ptr[tile_pt[t]];
      int cnt = out->pt_ptr[tile_pt[t + 1]] - base;
      keys.resize(cnt);
      for (int r = 0; r < cnt; ++r)  // r = position in point-major order
        keys[r] = ((unsigned long long)cam_idx[obs_by_pt[base + r]] << 16) | (unsigned)r;
      std::sort(keys.begin(), keys.end());
      pid_of_r.resize(cnt);
      for (int a = tile_pt[t]; a < tile_pt[t + 1]; ++a)
        for (int r = out->pt_ptr[a] - base; r < out->pt_ptr[a + 1] - base; ++r) pid_of_r[r] = (unsigned short)(a - tile_pt[t]);
      long long s0 = (long long)t * T;
      int runs = 0, prev = -1;
      // Bank-aware ranks.  A slot's rank must lie in its point's range [pt_ptr[k], pt_ptr[k + 1]) - base, but WHICH
      // position of the range it takes is free.  The kernels scatter per-observation products to shared-memory rows
      // indexed by rank (Schur matvec: 8-byte rows, 16 lanes per wavefront; linearize: 16-byte rows, 8 lanes per
      // wavefront), and with ranks in point-major input order those stores ran at 2.9x their ideal wavefronts
      // (profiles/r02_ncu_schur_matvec.md).  Greedy: walking the slots in order, a slot takes the free position of
      // its point whose bank (rank mod 16, rank mod 8) is unused so far in its half-warp / quarter-warp.
      taken.assign(cnt, 0);
      unsigned half_used = 0, quarter_used = 0;
      for (int s = 0; s < cnt; ++s) {
        const int r0 = (int)(keys[s] & 0xFFFFu), c = (int)(keys[s] >> 16);
        const int a = tile_pt[t] + pid_of_r[r0];
        const int lo = out->pt_ptr[a] - base, hi = out->pt_ptr[a + 1] - base;
        if ((s & 15) == 0) half_used = 0;
        if ((s & 7) == 0) quarter_used = 0;
        int best = -1, best_cost = 4;
        for (int r = lo; r < hi && best_cost > 0; ++r) {
          if (taken[r]) continue;
          const int cost = 2 * (int)((half_used >> (r & 15)) & 1u) + (int)((quarter_used >> (r & 7)) & 1u);
          if (cost < best_cost) { best_cost = cost; best = r; }
        }
        const int r = best;
        taken[r] = 1;
        half_used |= 1u << (r & 15);
        quarter_used |= 1u << (r & 7);
        out->obs_of_slot[s0 + s] = obs_by_pt[base + r0];
        out->cam[s0 + s] = c;
        out->rank[s0 + s] = (unsigned short)r;
        if (T <= 256) out->rankpid[s0 + s] = (unsigned short)(r | (pid_of_r[r] << 8));
        else out->rankpid32[s0 + s] = (unsigned)r | ((unsigned)pid_of_r[r] << 16);
        if (c != prev) { runs++; prev = c; }
      }
      runs_per_tile[t] = runs;
    }
  }
  long long total_runs = 0;
  for (int t = 0; t < num_tiles; ++t) {
    out->run_begin[t] = (int)(total_runs + t);  // + t: one terminator entry per earlier tile
    total_runs += runs_per_tile[t];
  }
  out->run_begin[num_tiles] = (int)(total_runs + num_tiles);
  out->camera_runs = total_runs;
  out->run_cam.assign(total_runs + num_tiles + 1, -1);
  out->run_slot.assign(total_runs + num_tiles + 1, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int t = 0; t < num_tiles; ++t) {
    long long s0 = (long long)t * T;
    int cnt = out->pt_ptr[tile_pt[t + 1]] - out->pt_ptr[tile_pt[t]];
    int w = out->run_begin[t], prev = -1;
    for (int s = 0; s < cnt; ++s) {
      int c = out->cam[s0 + s];
      if (c != prev) {
        out->run_cam[w] = c;
        out->run_slot[w] = (unsigned short)s;
        ++w;
        prev = c;
      }
    }
    out->run_cam[w] = -1;  // terminator: first slot past the tile's valid ones
    out->run_slot[w] = (unsigned short)cnt;
  }

  // --- 3b. per-tile metadata blobs for the TMA-bulk pipelined kernels --------------------------------
  {
    auto pad16 = [](size_t bytes) { return (bytes + 15) & ~size_t(15); };
    std::vector<size_t> off(num_tiles + 1, 0);
    for (int t = 0; t < num_tiles; ++t) {
      const int npts = tile_pt[t + 1] - tile_pt[t], nruns = runs_per_tile[t];
      const size_t bytes = 16 + pad16(2 * (size_t)(npts + 1)) + pad16(2 * (size_t)(nruns + 1)) + pad16(4 * (size_t)nruns);
      off[t + 1] = off[t] + bytes;
      out->max_pts_per_tile = std::max(out->max_pts_per_tile, npts);
      out->meta_max_bytes = std::max(out->meta_max_bytes, (int)bytes);
    }
    out->tile_meta.assign(off[num_tiles] ? off[num_tiles] : 16, 0);
    out->tile_dir.assign(4 * (size_t)(num_tiles ? num_tiles : 1), 0);
#pragma omp parallel for schedule(static)
    for (int t = 0; t < num_tiles; ++t) {
      const int npts = tile_pt[t + 1] - tile_pt[t], nruns = runs_per_tile[t];
      const int base = out->pt_ptr[tile_pt[t]];
      unsigned char* blob = out->tile_meta.data() + off[t];
      int* hdr = reinterpret_cast<int*>(blob);
      hdr[0] = npts; hdr[1] = nruns; hdr[2] = out->pt_ptr[tile_pt[t + 1]] - base; hdr[3] = tile_pt[t];
      unsigned short* pt_start = reinterpret_cast<unsigned short*>(blob + 16);
      for (int a = 0; a <= npts; ++a) pt_start[a] = (unsigned short)(out->pt_ptr[tile_pt[t] + a] - base);
      unsigned short* rs = reinterpret_cast<unsigned short*>(blob + 16 + pad16(2 * (size_t)(npts + 1)));
      int* rc = reinterpret_cast<int*>(blob + 16 + pad16(2 * (size_t)(npts + 1)) + pad16(2 * (size_t)(nruns + 1)));
      const int rb = out->run_begin[t];
      for (int u = 0; u <= nruns; ++u) rs[u] = out->run_slot[rb + u];
      for (int u = 0; u < nruns; ++u) rc[u] = out->run_cam[rb + u];
      out->tile_dir[4 * (size_t)t + 0] = (int)(off[t] / 16);
      out->tile_dir[4 * (size_t)t + 1] = (int)(off[t + 1] - off[t]);
      out->tile_dir[4 * (size_t)t + 2] = tile_pt[t];
      out->tile_dir[4 * (size_t)t + 3] = npts;
    }
  }

  // --- 4. camera-ordered slot list in chunks ---------------------------------------------------
  std::vector<long long> cptr(nc + 1, 0);
  for (long long i = 0; i < n; ++i) cptr[cam_idx[i] + 1]++;
  for (int c = 0; c < nc; ++c) cptr[c + 1] += cptr[c];
  out->cslot.assign(n > 0 ? n : 1, 0);
  {
    std::vector<long long> fill(cptr.begin(), cptr.end() - 1);
    for (long long s = 0; s < out->n_slots; ++s) {  // ascending slots -> each camera's list is ascending
      int c = out->cam[s];
      if (c >= 0) out->cslot[fill[c]++] = (int)s;
    }
  }
  out->chunk_cam.clear();
  out->chunk_begin.clear();
  out->cam_chunk_ptr.assign(nc + 1, 0);
  for (int c = 0; c < nc; ++c) {
    out->cam_chunk_ptr[c] = (int)out->chunk_cam.size();
    for (long long b = cptr[c]; b < cptr[c + 1]; b += kChunkSlots) {
      out->chunk_cam.push_back(c);
      out->chunk_begin.push_back((int)b);
    }
  }
  out->cam_chunk_ptr[nc] = (int)out->chunk_cam.size();
  out->chunk_begin.push_back((int)n);

  // --- 5. hot cameras: far more observations than the average camera (Zipf popularity).  Their rows of q are
  // accumulated per CTA in shared memory by the pipelined matvec; every other camera goes straight to L2.
  out->hot_of_cam.assign(nc > 0 ? nc : 1, -1);
  out->hot_list.clear();
  if (nc > 0 && nc < (1 << 23) && n > 0) {  // (the HOT kernels carry the hot index above bit 23 of a camera id)
    const long long limit = std::max<long long>(8192, 4 * (n / nc));
    std::vector<std::pair<long long, int>> big;
    for (int c = 0; c < nc; ++c)
      if (cptr[c + 1] - cptr[c] > limit) big.push_back({cptr[c + 1] - cptr[c], c});
    std::sort(big.begin(), big.end(), [](const auto& a, const auto& b) { return a.first > b.first || (a.first == b.first && a.second < b.second); });
    if ((int)big.size() > kMaxHotCameras) big.resize(kMaxHotCameras);
    for (size_t i = 0; i < big.size(); ++i) {
      out->hot_of_cam[big[i].second] = (short)i;
      out->hot_list.push_back(big[i].second);
    }
  }
  return 0;
}

}  // namespace cba
