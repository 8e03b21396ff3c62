// S5 - track selector (BASELINE.json north_star (5)): deduplicates tracklets by shared
// clusters.  Every cluster goes to the tracklet with the largest key = (n_hits << 32 | ~tracklet id)
// among those holding it (u64 atomicMax); a tracklet survives if it still owns min_track_hits
// clusters.  Tracklet ids, track ids and the CSR offsets are ranks from scans (deterministic).
//   k_owner      owner[cluster] = max key                 (one warp per tracklet, coalesced hit rows)
//   k_owned      owned count, first/last owned row, ownership bit mask per tracklet
//                -> scans -> track ids, CSR starts
//   k_finalize   capacity checks, n_tracks
//   k_write      trk_cl_idx (input indices, ascending row), cluster_track  (warp per track; reads the masks, not owner[])
//   k_params     tracks SoA (thread per track id: coalesced stores)
//   k_kept / scan / k_tracklet_ids   tracklet ids for the debug view (off the critical path: the key carries the
//                seed id, which orders kept tracklets exactly as their tracklet id would)
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;

// Ownership key: larger n_hits wins, then the smaller id.  64-bit in general; when every seed id fits 24 bits and
// n_hits fits 8 (max_seeds <= 2^24, n_rows <= 255) a 32-bit key gives the same order and owner[] is half as large -
// S5 is bound by random DRAM sectors of that array.
template <class K> __device__ __forceinline__ K make_key(int n_hits, int id);
template <> __device__ __forceinline__ unsigned long long make_key<unsigned long long>(int n_hits, int id) {
  return ((unsigned long long)(unsigned)n_hits << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)id);
}
template <> __device__ __forceinline__ unsigned make_key<unsigned>(int n_hits, int id) {
  return ((unsigned)n_hits << 24) | (0xFFFFFFu - (unsigned)id);
}

template <class K>
__global__ void __launch_bounds__(kThreads) k_init_out(Ctx c, OutPtrs o) {
  // owner = 0, cluster_track = -1 (vectorised where aligned; n is host-known)
  const long long n = c.n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    reinterpret_cast<K*>(c.owner)[i] = 0;
    o.cluster_track[i] = -1;
  }
}

// kept flag per seed + tracklet ids: only the debug view / the n_tracklets counter need them (the ownership key uses the
// seed id, which orders kept tracklets exactly like their tracklet id does)
__global__ void __launch_bounds__(kThreads) k_kept(Ctx c) {
  if (c.cnt->status) return;
  const int ns = c.cnt->n_seeds;
  for (int sd = blockIdx.x * blockDim.x + threadIdx.x; sd < ns; sd += gridDim.x * blockDim.x)
    c.kept_scan[sd] = c.t_n_hits[sd] >= c.min_tracklet_hits;
}

__global__ void __launch_bounds__(kThreads) k_tracklet_ids(Ctx c) {
  if (c.cnt->status) {
    if (blockIdx.x == 0 && threadIdx.x == 0) c.cnt->n_tracklets = 0;
    return;
  }
  const int ns = c.cnt->n_seeds;
  for (int sd = blockIdx.x * blockDim.x + threadIdx.x; sd < ns; sd += gridDim.x * blockDim.x) {
    const int inc = c.kept_scan[sd], prev = sd ? c.kept_scan[sd - 1] : 0;
    c.tracklet_of_seed[sd] = inc != prev ? inc - 1 : -1;
  }
}

// The hit tables are read once per pass and never again: streaming loads keep them from evicting the owner[] / perm[]
// lines of the sector being worked on out of L2.
template <class K>
__global__ void __launch_bounds__(kThreads) k_owner(Ctx c) {
  if (c.cnt->status) return;
  const int ns = c.cnt->n_seeds, R = c.R;
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  for (int sd = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; sd < ns; sd += warps) {
    const int nh = c.t_n_hits[sd];
    if (nh < c.min_tracklet_hits) continue;
    const K key = make_key<K>(nh, sd);
    K* owner = reinterpret_cast<K*>(c.owner);
    const int* hit = c.t_hit + (size_t)sd * R;
    const int last = c.t_last_row[sd];
    for (int r = c.t_first_row[sd] + lane; r <= last; r += 32) {   // the table is defined on [first_row, last_row] only
      const int cl = __ldcs(hit + r);
      if (cl >= 0) atomicMax(owner + cl, key);
    }
  }
}

// owned count, first / last owned row and the ownership bit mask (bit k of word w: row first_row + 32 w + k is owned)
template <class K>
__global__ void __launch_bounds__(kThreads) k_owned(Ctx c) {
  if (c.cnt->status) return;
  const int ns = c.cnt->n_seeds, R = c.R;
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  for (int sd = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; sd < ns; sd += warps) {
    const int nh = c.t_n_hits[sd];
    const bool kept = nh >= c.min_tracklet_hits;
    int owned = 0, first = 0x7FFFFFFF, last = -1;
    unsigned mine = 0;                                   // lane w keeps mask word w
    if (kept) {
      const K key = make_key<K>(nh, sd);
      const K* owner = reinterpret_cast<const K*>(c.owner);
      const int* hit = c.t_hit + (size_t)sd * R;
      const int hi = c.t_last_row[sd];
      int w = 0;
      for (int rb = c.t_first_row[sd]; rb <= hi; rb += 32, ++w) {
        const int r = rb + lane;
        bool own = false;
        if (r <= hi) {
          const int cl = __ldcs(hit + r);
          own = cl >= 0 && owner[cl] == key;
        }
        const unsigned m = __ballot_sync(0xffffffffu, own);
        if (lane == w) mine = m;
        if (m) {
          owned += __popc(m);
          first = min(first, rb + __ffs(m) - 1);
          last = rb + 31 - __clz(m);
        }
      }
    }
    if (lane < c.mask_words) c.own_mask[(size_t)sd * c.mask_words + lane] = mine;
    if (lane == 0) {
      const bool surv = kept && owned >= c.min_track_hits;
      c.k_owned[sd] = owned; c.k_first[sd] = first; c.k_last[sd] = last;
      c.surv_scan[sd] = surv;
      c.owned_scan[sd] = surv ? owned : 0;
    }
  }
}

__global__ void k_finalize(Ctx c, OutPtrs o) {
  Counters& k = *c.cnt;
  if (!k.status && (k.n_tracks > o.max_tracks || k.n_track_clusters > o.max_track_clusters))
    k.status |= TPC_STATUS_TRACKS_OVERFLOW;
  if (k.status) { k.n_tracks = 0; k.n_track_clusters = 0; k.n_tracklets = 0; }
  *o.n_tracks = k.n_tracks;
  *o.status = k.status;
  if (k.status) o.trk_cl_start[0] = 0;
}

__global__ void __launch_bounds__(kThreads) k_write(Ctx c, OutPtrs o) {
  if (c.cnt->status) return;
  const int ns = c.cnt->n_seeds, R = c.R;
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  if (blockIdx.x == 0 && threadIdx.x == 0) o.trk_cl_start[0] = 0;
  for (int sd = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; sd < ns; sd += warps) {
    const int inc = c.surv_scan[sd], prev = sd ? c.surv_scan[sd - 1] : 0;
    if (inc == prev) continue;
    const int id = inc - 1;
    const int end = c.owned_scan[sd];
    int off = end - c.k_owned[sd];
    const int* hit = c.t_hit + (size_t)sd * R;
    const int hi = c.t_last_row[sd];
    const unsigned* mask = c.own_mask + (size_t)sd * c.mask_words;
    for (int rb = c.t_first_row[sd]; rb <= hi; rb += 32, ++mask) {
      const unsigned m = *mask;                          // rows of this chunk the track owns (k_owned)
      if ((m >> lane) & 1u) {
        const int cl = __ldcs(hit + rb + lane);
        const int in_idx = c.perm[cl];
        o.trk_cl_idx[off + __popc(m & ((1u << lane) - 1))] = in_idx;
        o.cluster_track[in_idx] = id;
      }
      off += __popc(m);
    }
    if (lane == 0) {
      c.track_seed[id] = sd;                         // seed of track id, for k_params and the refit
      o.trk_cl_start[id + 1] = end;
    }
  }
}

// pseudo-z of the track at the beam line, assuming a primary from the origin
__device__ __forceinline__ float beam_z(float kb, float x, float y, float z, float t, float q) {
  const float cv = kb * q;
  const float d = sqrtf(x * x + y * y);
  float a = fabsf((0.5f * cv) * d);
  if (!(a < 1.0f)) a = 1.0f;
  const float c1 = sqrtf(1.0f - a * a);
  const float a1 = a / sqrtf(2.0f * (1.0f + c1));
  const float c2 = sqrtf(1.0f - a1 * a1);
  const float a2 = a1 / sqrtf(2.0f * (1.0f + c2));
  const float w = a2 * a2;
  const float ser = 1.0f + w * ((float)(1.0 / 6.0) + w * ((float)(3.0 / 40.0) + w * ((float)(5.0 / 112.0) + w * (float)(35.0 / 1152.0))));
  const float ratio = a > 0.0f ? (4.0f * (a2 * ser)) / a : 1.0f;
  const float path = d * ratio;
  return z - t * path;
}

// Track parameters: one thread per TRACK id, so every output component is written with coalesced full-sector stores
// (one warp per track wrote 29 scattered 4-byte stores per track: 50 M partial sectors on cfg5).
__global__ void __launch_bounds__(kThreads) k_params(Ctx c, OutPtrs o) {
  if (c.cnt->status) return;
  const int nt = c.cnt->n_tracks, R = c.R;
  const size_t mt = (size_t)o.max_tracks;
  for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < nt; id += gridDim.x * blockDim.x) {
    const int sd = c.track_seed[id];
    const float* p = c.t_par + (size_t)sd * 5;
    const float* q = c.t_cov + (size_t)sd * 15;
#pragma unroll
    for (int i = 0; i < 5; ++i) o.par[i * mt + id] = p[i];
#pragma unroll
    for (int i = 0; i < 15; ++i) o.cov[i * mt + id] = q[i];
    const int low = c.t_first_row[sd];
    o.sector[id] = (int)c.srow[c.seed_head[sd]] >> 8;
    o.first_row[id] = c.k_first[sd];
    o.last_row[id] = c.k_last[sd];
    o.n_clusters[id] = c.k_owned[sd];
    o.x_ref[id] = c.rowtab[low].x;
    o.z_ref[id] = c.t_zref[sd];
    o.chi2[id] = c.t_chi2[sd];
    o.ndf[id] = 2 * c.t_n_hits[sd] - 5;
    o.z_beam[id] = beam_z(c.kb, c.rowtab[low].x, p[0], c.t_zref[sd] + p[1], p[3], p[4]);
  }
  (void)R;
}

inline unsigned grid_for(long long n, int per_block, int n_sms, int waves) {
  long long g = (n + per_block - 1) / per_block;
  const long long cap = (long long)n_sms * waves;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (unsigned)g;
}

}  // namespace

int launches_s5() { return 8 + 9; }
int launch_s5(const Ctx& c, const OutPtrs& o, cudaStream_t st) {
  const unsigned gn = grid_for(c.n, kThreads, c.n_sms, 8);
  const unsigned gs = grid_for(c.max_seeds, kThreads, c.n_sms, 8);          // thread per seed
  const unsigned gw = grid_for((long long)c.max_seeds * 32, kThreads, c.n_sms, 8);   // warp per seed
  if (c.max_seeds <= (1 << 24) && c.R <= 255) {
    k_init_out<unsigned><<<gn, kThreads, 0, st>>>(c, o);
    k_owner<unsigned><<<gw, kThreads, 0, st>>>(c);
    k_owned<unsigned><<<gw, kThreads, 0, st>>>(c);
  } else {
    k_init_out<unsigned long long><<<gn, kThreads, 0, st>>>(c, o);
    k_owner<unsigned long long><<<gw, kThreads, 0, st>>>(c);
    k_owned<unsigned long long><<<gw, kThreads, 0, st>>>(c);
  }
  if (launch_scan_inclusive(c.surv_scan, &c.cnt->n_seeds, 0, c.max_seeds, c.tile_sums, &c.cnt->n_tracks, c.n_sms, st)) return -1;
  if (launch_scan_inclusive(c.owned_scan, &c.cnt->n_seeds, 0, c.max_seeds, c.tile_sums, &c.cnt->n_track_clusters, c.n_sms, st)) return -1;
  k_finalize<<<1, 1, 0, st>>>(c, o);
  k_write<<<gw, kThreads, 0, st>>>(c, o);
  k_params<<<grid_for(o.max_tracks, kThreads, c.n_sms, 8), kThreads, 0, st>>>(c, o);
  // tracklet ids (debug view, n_tracklets counter): nothing downstream waits for them
  k_kept<<<gs, kThreads, 0, st>>>(c);
  if (launch_scan_inclusive(c.kept_scan, &c.cnt->n_seeds, 0, c.max_seeds, c.tile_sums, &c.cnt->n_tracklets, c.n_sms, st)) return -1;
  k_tracklet_ids<<<gs, kThreads, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
