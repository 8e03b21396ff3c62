// S8 - cluster protection for hit removal, "strategy B": a cluster is kept iff it
// is attached to a track or lies, in its own (sector, row), inside the closed rectangle +-road_y x +-road_z around a
// cluster some track owns.  A separate call (tpc_tracker_protect), not part of the timed hot path; it reads the sorted
// clusters and the grid the last tpc_track_timeframe left in the workspace and the caller's cluster_track array.
//   k_mark   thread per sorted position: an owned cluster marks the members of the rectangle around itself
//   k_out    keep[input index] = mark[sorted position]
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 256;

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

}  // namespace

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

}  // namespace tpc
