// S8 - cluster protection for hit removal, "strategy B": a cluster is kept iff it
// is attached to a track or lies, in its own (sector, row), inside the closed rectangle +-road_y x +-road_z around a
// cluster some track owns.  A separate call (tpc_tracker_protect), not part of the timed hot path; it reads the sorted
// clusters and the grid the last tpc_track_timeframe left in the workspace and the caller's cluster_track array.
//   k_mark   thread per sorted position: an owned cluster marks the members of the rectangle around itself
//   k_out    keep[input index] = mark[sorted position]
#include <mutex>

#include "../../include/tpc_tracker.h"
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 256;

// Mark bytes of tpc_tracker_protect_static (include/tpc_tracker.h): one byte per sorted position, in an array that is part
// of the library image instead of the caller's workspace, for callers that cannot obtain device memory at run time.
// One copy per device that loads this module, shared by every handle and stream of the process.  In HOST code this
// name is only a handle for cudaGetSymbolAddress - it is not a device address and must never be handed to a kernel.
static __device__ __align__(256) unsigned char g_static_mark[TPC_PROTECT_STATIC_MAX_CLUSTERS];

__global__ void __launch_bounds__(kThreads) k_mark(Ctx c, const int* __restrict__ cluster_track, float road_y, float road_z,
                                                   unsigned char* __restrict__ mark) {
  if (c.cnt->status) return;
  const long long n = c.n;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (long long)gridDim.x * blockDim.x) {
    if (__ldg(cluster_track + c.perm[o]) < 0) continue;
    const int sr = c.srow[o];                            // (sector << 8) | row
    const int s = sr >> 8, r = sr & 255;
    const float2 me = c.yz[o];
    RowGrid g;
    g.b0 = __ldg(c.bin_base + s * c.R + r);
    g.ny = __ldg(&c.rowtab[r].ny);
    g.nz = __ldg(c.nz + s);
    g.ymax = __ldg(&c.rowtab[r].ymax);
    g.zmin = __ldg(c.zmin + s);
    for_each_in_rect(g, c.inv_cy, c.inv_cz, c.bins, c.yz, me.x - road_y, me.x + road_y, me.y - road_z, me.y + road_z,
                     [&](int j, float, float) { mark[j] = 1; });
  }
}

__global__ void __launch_bounds__(kThreads) k_out(Ctx c, const unsigned char* __restrict__ mark, unsigned char* __restrict__ keep) {
  if (c.cnt->status) return;
  const long long n = c.n;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (long long)gridDim.x * blockDim.x)
    keep[c.perm[o]] = mark[o];
}

// ---- hit removal, "strategy A": class of every track, then of every input cluster
__global__ void __launch_bounds__(kThreads) k_track_class(Ctx c, RemovePtrs o) {
  const int nt = c.cnt->status ? 0 : min(c.cnt->n_tracks, c.max_tracks);
  const size_t mt = (size_t)c.max_tracks, ft = (size_t)o.fit_stride, gt = (size_t)o.mrg_stride;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nt; k += gridDim.x * blockDim.x) {
    // a track outside every merged track (-1: link cycle), a merge that did not run (status bit) or an id
    // that cannot be one is classified from its own segment only - and never used as an index
    int m = o.merged_of_track[k];
    if (c.mcnt->status || m >= c.mcnt->n_merged) m = -1;
    int cls = 1;
    if (m >= 0 && o.apex_leg[m] == 1) cls = 2;
    else if (m >= 0 && fabsf(o.mrg_par[4 * gt + m]) * o.min_pt > 1.0f) cls = 3;
    else if (fabsf(o.fit_par[2 * ft + k]) > o.max_incl && fabsf(c.up_par[2 * mt + k]) > o.max_incl) cls = 4;
    c.m_bin_of[k] = cls;                                  // per-track scratch of the merger, free by now
  }
}

__global__ void __launch_bounds__(kThreads) k_cluster_class(Ctx c, RemovePtrs o, int* __restrict__ good_track) {
  const long long n = c.n;
  const bool dead = c.cnt->status != 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int k = dead ? -1 : o.cluster_track[i];
    const int cls = k >= 0 ? c.m_bin_of[k] : 0;
    o.cls[i] = (unsigned char)cls;
    good_track[i] = cls == 1 ? k : -1;
  }
}

__global__ void __launch_bounds__(kThreads) k_removable(Ctx c, RemovePtrs o, const unsigned char* __restrict__ keep) {
  const long long n = c.n;
  const bool dead = c.cnt->status != 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    o.remove[i] = (!dead && o.cls[i] >= 2 && !keep[i]) ? 1 : 0;
}

}  // namespace

int launch_protect(const Ctx& c, const int* cluster_track, float road_y, float road_z, unsigned char* keep, cudaStream_t st);

int launch_removable(const Ctx& c, const RemovePtrs& o, cudaStream_t st) {
  if (c.n == 0) return 0;
  // scratch: the S1 record buffer (16 bytes per cluster) is dead after S1: the good-track map and the keep flags live there
  int* good_track = reinterpret_cast<int*>(c.rec);
  unsigned char* keep = reinterpret_cast<unsigned char*>(good_track + c.n);
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 256;
  if (g > cap) g = cap;
  long long gk = ((long long)c.max_tracks + kThreads - 1) / kThreads;
  if (gk > cap) gk = cap;
  k_track_class<<<(unsigned)gk, kThreads, 0, st>>>(c, o);
  k_cluster_class<<<(unsigned)g, kThreads, 0, st>>>(c, o, good_track);
  if (cudaMemsetAsync(keep, 0, (size_t)c.n, st) != cudaSuccess) return -1;   // a dead run marks nothing
  if (launch_protect(c, good_track, o.road_y, o.road_z, keep, st)) return -1;
  k_removable<<<(unsigned)g, kThreads, 0, st>>>(c, o, keep);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launch_protect(const Ctx& c, const int* cluster_track, float road_y, float road_z, unsigned char* keep, cudaStream_t st) {
  unsigned char* mark = reinterpret_cast<unsigned char*>(c.flag_scan);      // scratch, free after S3
  if (c.n == 0) return 0;
  if (cudaMemsetAsync(mark, 0, (size_t)c.n, st) != cudaSuccess) return -1;
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 256;
  if (g > cap) g = cap;
  k_mark<<<(unsigned)g, kThreads, 0, st>>>(c, cluster_track, road_y, road_z, mark);
  k_out<<<(unsigned)g, kThreads, 0, st>>>(c, mark, keep);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// ---- tpc_tracker_protect_static: the same two kernels, the marks in g_static_mark.  No allocation of any kind here.
namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_mark_addr[kMaxDevices];   // device address of g_static_mark per device ordinal; null = not looked up yet
}  // namespace

int launch_protect_static(const Ctx& c, const int* cluster_track, float road_y, float road_z, unsigned char* keep, cudaStream_t st) {
  if (c.n == 0) return 0;
  if ((long long)c.n > (long long)TPC_PROTECT_STATIC_MAX_CLUSTERS) return -1;   // (the C entry point has refused this already)
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
  unsigned char* mark = nullptr;
  {
    // first call on this device: ask the runtime where the array lives HERE (the current device's copy)
    std::lock_guard<std::mutex> lock(g_static_mutex);
    mark = g_static_mark_addr[dev];
    if (!mark) {
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_static_mark) != cudaSuccess || !p) { cudaGetLastError(); return -1; }
      mark = g_static_mark_addr[dev] = static_cast<unsigned char*>(p);
    }
  }
  // the array still holds the previous call's marks: clear the part this frame uses, on the caller's stream
  if (cudaMemsetAsync(mark, 0, (size_t)c.n, st) != cudaSuccess) return -1;
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 256;
  if (g > cap) g = cap;
  k_mark<<<(unsigned)g, kThreads, 0, st>>>(c, cluster_track, road_y, road_z, mark);
  k_out<<<(unsigned)g, kThreads, 0, st>>>(c, mark, keep);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
