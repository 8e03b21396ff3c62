// S1 - per-sector, per-row cluster sort and 2-D (y,z) grid binning (BASELINE.json north_star (1);
// DESIGN.md section 3.1).  Counting sort over the global bin id:
//   k_zrange   per-sector exact min/max of z (block-local smem reduction on order-preserving keys)
//   k_tables   nz_s, bin_base[(s,r)], N_b                                   (one block)
//   k_zero     bins[0 .. N_b+2) = 0
//   k_count    gbin[i]; histogram into bins[gbin+2]
//   scan       inclusive: bins[g+1] = first position of bin g
//   k_scatter  pos = bins[gbin+1]++  -> tmp_idx[pos] = i   (arrival order inside a bin is arbitrary;
//              afterwards bins[0..N_b] is exactly the CSR bin_start)
//   k_place    stable fix-up: rank of i among the indices of its bin, final position = start + rank;
//              writes perm, ys, zs, srow                   (bins hold ~1-3 clusters)
//   k_rowstart row_start[sr] = bin_start[bin_base[sr]]
// The result equals std::stable_sort by (sector,row,bin) whatever order the atomics resolved in.
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(256) k_reset(Ctx c) {
  const int i = threadIdx.x;
  if (i < c.S) { c.zmin_key[i] = 0x7FFFFFFF; c.zmax_key[i] = (int)0x80000000; }
  if (i == 0) {
    Counters z = {};
    *c.cnt = z;
  }
}

// ---------------------------------------------------------------------------------- z range
__global__ void __launch_bounds__(kThreads) k_zrange(Ctx c) {
  __shared__ int smin[kMaxRows], smax[kMaxRows];
  for (int i = threadIdx.x; i < c.S; i += blockDim.x) { smin[i] = 0x7FFFFFFF; smax[i] = (int)0x80000000; }
  __syncthreads();
  bool bad = false;
  const long long n = c.n;
  // 4 clusters per thread per step: one 32-bit load of the sector bytes, one float4 of z
  const long long n4 = n >> 2;
  const uint32_t* sec4 = reinterpret_cast<const uint32_t*>(c.in_sector);
  const float4* z4 = reinterpret_cast<const float4*>(c.in_z);
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (long long)gridDim.x * blockDim.x) {
    const uint32_t sw = __ldg(sec4 + q);
    const float4 zv = __ldg(z4 + q);
    const float zz[4] = {zv.x, zv.y, zv.z, zv.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int s = (sw >> (8 * k)) & 0xFF;
      if (s >= c.S) { bad = true; continue; }
      const int key = float_key(zz[k]);
      if (key < smin[s]) atomicMin(&smin[s], key);
      if (key > smax[s]) atomicMax(&smax[s], key);
    }
  }
  if (blockIdx.x == 0 && threadIdx.x < (int)(n & 3)) {   // ragged tail
    const long long i = (n4 << 2) + threadIdx.x;
    const int s = c.in_sector[i];
    if (s >= c.S) bad = true;
    else {
      const int key = float_key(c.in_z[i]);
      atomicMin(&smin[s], key);
      atomicMax(&smax[s], key);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < c.S; i += blockDim.x) {
    if (smin[i] != 0x7FFFFFFF) atomicMin(&c.zmin_key[i], smin[i]);
    if (smax[i] != (int)0x80000000) atomicMax(&c.zmax_key[i], smax[i]);
  }
  if (bad) atomicOr(&c.cnt->status, (int)TPC_STATUS_BAD_CLUSTER);
}

// ---------------------------------------------------------------------------------- tables
__global__ void __launch_bounds__(1024) k_tables(Ctx c) {
  __shared__ long long sbase[kMaxRows + 1];
  __shared__ int snz[kMaxRows];
  if (threadIdx.x == 0) {
    long long acc = 0;
    for (int s = 0; s < c.S; ++s) {
      const int kmin = c.zmin_key[s], kmax = c.zmax_key[s];
      int nz = 0;
      float zmin = 0.f, zmax = 0.f;
      if (kmin <= kmax) {
        zmin = key_float(kmin); zmax = key_float(kmax);
        nz = (int)floorf((zmax - zmin) * c.inv_cz) + 1;
      }
      c.zmin[s] = zmin; c.zmax[s] = zmax; c.nz[s] = nz; snz[s] = nz;
      sbase[s] = acc;
      acc += (long long)nz * c.ny_total;
    }
    sbase[c.S] = acc;
    int st = 0;
    if (acc > 2147483647LL - 2 || acc > (long long)c.max_bins) { st = TPC_STATUS_BINS_OVERFLOW; acc = 0; }
    if (st) atomicOr(&c.cnt->status, st);
    c.cnt->n_bins = (int)acc;
  }
  __syncthreads();
  const bool ok = (sbase[c.S] <= 2147483647LL - 2) && (sbase[c.S] <= (long long)c.max_bins);
  for (int sr = threadIdx.x; sr <= c.SR; sr += blockDim.x) {
    int v = 0;
    if (ok) {
      if (sr == c.SR) v = (int)sbase[c.S];
      else {
        const int s = sr / c.R, r = sr - s * c.R;
        v = (int)(sbase[s] + (long long)snz[s] * c.rowtab[r].ny_prefix);
      }
    }
    c.bin_base[sr] = v;
  }
}

__global__ void __launch_bounds__(kThreads) k_zero_bins(Ctx c) {
  if (c.cnt->status) return;
  const long long m = (long long)c.cnt->n_bins + 2;
  const long long m4 = m >> 2;
  int4* b4 = reinterpret_cast<int4*>(c.bins);
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < m4; q += (long long)gridDim.x * blockDim.x)
    b4[q] = make_int4(0, 0, 0, 0);
  if (blockIdx.x == 0 && threadIdx.x < (int)(m & 3)) c.bins[(m4 << 2) + threadIdx.x] = 0;
}

// ---------------------------------------------------------------------------------- count
__device__ __forceinline__ int global_bin(const Ctx& c, int s, int r, float y, float z) {
  const RowTab& t = c.rowtab[r];
  const int ny = __ldg(&t.ny);
  const int iy = floor_clamp((y + __ldg(&t.ymax)) * c.inv_cy, ny - 1);
  const int iz = floor_clamp((z - __ldg(c.zmin + s)) * c.inv_cz, __ldg(c.nz + s) - 1);
  return __ldg(c.bin_base + s * c.R + r) + iz * ny + iy;
}

__global__ void __launch_bounds__(kThreads) k_count(Ctx c) {
  if (c.cnt->status) return;
  bool bad = false;
  const long long n = c.n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int s = __ldg(c.in_sector + i), r = __ldg(c.in_row + i);
    if (s >= c.S || r >= c.R) { bad = true; c.gbin[i] = -1; continue; }
    const int g = global_bin(c, s, r, __ldg(c.in_y + i), __ldg(c.in_z + i));
    c.gbin[i] = g;
    atomicAdd(c.bins + g + 2, 1);
  }
  if (bad) atomicOr(&c.cnt->status, (int)TPC_STATUS_BAD_CLUSTER);
}

__global__ void __launch_bounds__(kThreads) k_scatter(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int g = __ldg(c.gbin + i);
    const int pos = atomicAdd(c.bins + g + 1, 1);
    c.tmp_idx[pos] = (int)i;
  }
}

// stable fix-up + gather of the sorted payload
__global__ void __launch_bounds__(kThreads) k_place(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (long long)gridDim.x * blockDim.x) {
    const int i = __ldg(c.tmp_idx + p);
    const int g = __ldg(c.gbin + i);
    const int bs = c.bins[g], be = c.bins[g + 1];
    int rank = 0;
    for (int j = bs; j < be; ++j) rank += (__ldg(c.tmp_idx + j) < i);
    const int fp = bs + rank;
    c.perm[fp] = i;
    c.yz[fp] = make_float2(__ldg(c.in_y + i), __ldg(c.in_z + i));
    c.srow[fp] = (uint16_t)((int)__ldg(c.in_sector + i) * c.R + (int)__ldg(c.in_row + i));
  }
}

__global__ void __launch_bounds__(kThreads) k_rowstart(Ctx c) {
  const bool dead = c.cnt->status != 0;
  for (int sr = blockIdx.x * blockDim.x + threadIdx.x; sr <= c.SR; sr += gridDim.x * blockDim.x)
    c.row_start[sr] = dead ? 0 : c.bins[c.bin_base[sr]];
}

inline unsigned grid_for(long long n, int per_block, int n_sms, int waves) {
  long long g = (n + per_block - 1) / per_block;
  const long long cap = (long long)n_sms * waves;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (unsigned)g;
}

}  // namespace

int launches_reset() { return 1; }
int launch_reset(const Ctx& c, cudaStream_t st) {
  k_reset<<<1, 256, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launches_s1() { return 7 + 3; }
int launch_s1(const Ctx& c, cudaStream_t st) {
  const unsigned g = grid_for(c.n, kThreads, c.n_sms, 8);
  k_zrange<<<grid_for(c.n / 4 + 1, kThreads, c.n_sms, 4), kThreads, 0, st>>>(c);
  k_tables<<<1, 1024, 0, st>>>(c);
  k_zero_bins<<<grid_for((long long)c.max_bins / 4 + 1, kThreads, c.n_sms, 8), kThreads, 0, st>>>(c);
  k_count<<<g, kThreads, 0, st>>>(c);
  if (launch_scan_inclusive(c.bins, &c.cnt->n_bins, 2, (long long)c.max_bins + 2, c.tile_sums, nullptr, c.n_sms, st)) return -1;
  k_scatter<<<g, kThreads, 0, st>>>(c);
  k_place<<<g, kThreads, 0, st>>>(c);
  k_rowstart<<<grid_for(c.SR + 1, kThreads, c.n_sms, 1), kThreads, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
