// S2 - neighbours finder (BASELINE.json north_star (2)): for every cluster of row
// r the best (up, down) link pair in rows r+-1 (widening to r+-2) by minimal straight-line deviation
// inside a search window.  One thread per sorted position; consecutive positions are neighbours in
// (z, y) of the same row, so a warp's rectangle queries hit the same few cache lines of the rows
// above and below.  The per-row tables sit in shared memory.  Division-free, no candidate cap:
// up to kCap candidates per side are kept in shared-memory lists, beyond that the thread
// re-walks the rectangles (same visiting order, same result).
// Measured and rejected on cfg5 (this version: 6.1 ms): one flat per-lane loop over (query, bin row, candidate) from
// global memory 14.5 ms and from shared-memory tiles 17.8 ms; a warp-cooperative flattened (slot, candidate) item list
// 14.1 ms; the five phases (up k=1, up k=2, down k=1, down k=2, scoring) on compacted CTA work lists with the cluster
// state in shared memory 10.4 ms (twelve CTA barriers per tile cost more than the idle lanes they remove); the k = 2 up
// retries (40 % of the clusters, 2 ms of the kernel) deferred to a second, compacted launch 6.5 ms.
// Round 2 (profiles/r02_s2_regions.md: 49 % of the instructions are the rectangle query at 10 - 18 lanes, 20 % the pair
// scoring at 9.6 lanes; DRAM traffic = 1.0 x the algorithmic bytes).  Three more designs measured and rejected on cfg5
// (this version: 5.74 ms), all bit-exact:
//  * the rectangle query split in two halves (bin cover + the four bin_start loads / the candidate walk) so that the
//    loads of the up and the down query of a cluster are in flight together before either walk starts: 6.12 ms - the
//    down query is then computed for the 15 % of the clusters whose up window turns out empty, and eight more live
//    values per thread cost more than the overlapped latency (the kernel is issue-bound, 75 % of the slots busy);
//  * the candidate lists keep (position, y, z) so that the scoring does not gather the candidates a second time
//    (kCap 4 to keep 5 CTAs per SM): 7.77 ms - the second gather hits L1 anyway, while the lists' shared-memory
//    traffic triples and windows with 5 - 8 candidates fall back to the re-walk;
//  * warp tiles: the warp finds, per target row, the one contiguous run of positions that holds all 32 windows (two
//    bin_start loads), streams it through a 32-entry shared-memory tile with coalesced loads, and every lane tests every
//    candidate of the tile against its own rectangle (broadcast reads, uniform control flow, no divergence): 13.7 ms.
//    The run holds ~36 candidates for windows that accept ~1.5 each, and a test costs ~12 instructions: the uniform scan
//    does ten times the comparisons the bin lookup does, which costs more than all the idle lanes it removes.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 256;
constexpr int kCap = 8;


__device__ __forceinline__ RowGrid make_grid(const Ctx& c, const RowTab* tab, int s, int t) {
  RowGrid g;
  g.b0 = __ldg(c.bin_base + s * c.R + t);
  g.ny = tab[t].ny;
  g.nz = __ldg(c.nz + s);
  g.ymax = tab[t].ymax;
  g.zmin = __ldg(c.zmin + s);
  return g;
}

__global__ void __launch_bounds__(kThreads, 5) k_neighbours(Ctx c) {
  extern __shared__ RowTab tab[];
  // candidate lists: sorted positions only, [entry][thread] in shared memory (dynamic indexing of a register array
  // would put them in local memory: 13 % of the instructions of round 1b)
  int* listU = reinterpret_cast<int*>(tab + c.R) + threadIdx.x;
  int* listD = listU + kCap * kThreads;
  for (int i = threadIdx.x; i < c.R * (int)(sizeof(RowTab) / 4); i += blockDim.x)
    reinterpret_cast<int*>(tab)[i] = __ldg(reinterpret_cast<const int*>(c.rowtab) + i);
  __syncthreads();
  if (c.cnt->status) return;
  const float2* __restrict__ yz = c.yz;
  const int* __restrict__ bin_start = c.bins;
  const long long n = c.n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int sr = c.srow[i];                            // (sector << 8) | row
    const int s = sr >> 8, r = sr & 255;
    const float2 me = yz[i];
    const float y = me.x, z = me.y;
    int lu = -1, ld = -1;

    int nU = 0, nD = 0;
    int ku = 0, kd = 0;
    float uylo = 0, uyhi = 0, uzlo = 0, uzhi = 0, dylo = 0, dyhi = 0, dzlo = 0, dzhi = 0;
    RowGrid gu = {}, gd = {};
    for (int k = 1; k <= 2 && nU == 0; ++k) {
      if (r + k >= c.R) break;
      const float yc = y * tab[r].up_ratio[k - 1], wy = tab[r].up_wy[k - 1], wz = tab[r].up_wz[k - 1];
      uylo = yc - wy; uyhi = yc + wy; uzlo = z - wz; uzhi = z + wz;
      gu = make_grid(c, tab, s, r + k);
      for_each_in_rect(gu, c.inv_cy, c.inv_cz, bin_start, yz, uylo, uyhi, uzlo, uzhi, [&](int j, float yj, float zj) {
        if (nU < kCap) listU[nU * kThreads] = j;
        ++nU;
      });
      ku = k;
    }
    if (nU > 0) {
      for (int k = 1; k <= 2 && nD == 0; ++k) {
        if (r - k < 0) break;
        const float yc = y * tab[r].dn_ratio[k - 1], wy = tab[r].dn_wy[k - 1], wz = tab[r].dn_wz[k - 1];
        dylo = yc - wy; dyhi = yc + wy; dzlo = z - wz; dzhi = z + wz;
        gd = make_grid(c, tab, s, r - k);
        for_each_in_rect(gd, c.inv_cy, c.inv_cz, bin_start, yz, dylo, dyhi, dzlo, dzhi, [&](int j, float yj, float zj) {
          if (nD < kCap) listD[nD * kThreads] = j;
          ++nD;
        });
        kd = k;
      }
    }
    if (nU > 0 && nD > 0) {
      const float dxu = tab[r].up_dx[ku - 1], dxd = tab[r].dn_dx[kd - 1];
      const float cut = c.link_T * ((dxu * dxd) * (dxu * dxd));
      float best = INFINITY;
      int bu = -1, bd = -1;
      auto score = [&](int u, float yu, float zu, int d, float yd, float zd) {
        const float Dy = dxd * (yu - y) - dxu * (y - yd);
        const float Dz = dxd * (zu - z) - dxu * (z - zd);
        const float Dv = Dy * Dy + Dz * Dz;
        if (Dv < best) { best = Dv; bu = u; bd = d; }
      };
      if (nU <= kCap && nD <= kCap) {
        for (int a = 0; a < nU; ++a) {
          const int u = listU[a * kThreads];
          const float2 pu = __ldg(yz + u);
          for (int b = 0; b < nD; ++b) {
            const int d = listD[b * kThreads];
            const float2 pd = __ldg(yz + d);
            score(u, pu.x, pu.y, d, pd.x, pd.y);
          }
        }
      } else {   // rare: crowded window, walk the rectangles again
        for_each_in_rect(gu, c.inv_cy, c.inv_cz, bin_start, yz, uylo, uyhi, uzlo, uzhi, [&](int u, float yu, float zu) {
          for_each_in_rect(gd, c.inv_cy, c.inv_cz, bin_start, yz, dylo, dyhi, dzlo, dzhi,
                           [&](int d, float yd, float zd) { score(u, yu, zu, d, yd, zd); });
        });
      }
      if (best <= cut) { lu = bu; ld = bd; }
    }
    c.link_up_raw[i] = lu;
    c.link_dn_raw[i] = ld;
  }
}

}  // namespace

int launches_s2() { return 1; }
int launch_s2(const Ctx& c, cudaStream_t st) {
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 160;   // measured on cfg5: 5 -> 6.9 ms, 32 -> 6.2, 64 -> 5.9, 160 -> 5.76, 320 -> 5.84, 1280 -> 6.3, no cap -> 6.7
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  k_neighbours<<<(unsigned)g, kThreads, c.R * sizeof(RowTab) + 2 * kCap * kThreads * sizeof(int), st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
