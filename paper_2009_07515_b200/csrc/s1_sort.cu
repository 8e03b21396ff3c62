// S1 - per-sector, per-row cluster sort and 2-D (y,z) grid binning (BASELINE.json north_star (1);
// DESIGN.md section 3.1).  Two-level counting sort whose random accesses stay inside L2:
//   k_zrange_count  one streaming pass over (sector,row,z): exact per-sector min/max of z and the
//                   number of clusters per (sector,row)               (smem reductions, then atomics)
//   k_tables        nz_s, bin_base[(s,r)], N_b, row_start = exclusive scan of the (s,r) counts   (one block)
//   k_partition     streaming pass over the input: every cluster goes to the bucket of its
//                   (sector,row) as one 16-byte record (y, z, input index, -) - arrival order; the
//                   5472 bucket heads live in L2, which merges the 16-byte stores into full lines
//   k_binsort       one CTA per (sector,row) bucket (~17 k clusters, a few 10 k bins: L2 resident):
//                   zero its bins, histogram (the atomic returns the arrival rank inside the bin),
//                   CTA-wide exclusive scan -> CSR bin_start (the bucket's base is row_start, so no
//                   device-wide scan), scatter perm / (y,z) / srow, then a stable fix-up that orders
//                   the clusters of every multiply-occupied bin by input index
// The result equals std::stable_sort by (sector,row,bin) whatever order the atomics resolved in.
// (Round 1a-c used one device-wide counting sort over the ~N global bins: every one of its ~8 accesses
// per cluster was a random 32-byte DRAM sector; 15.1 ms on cfg5, see profiles/.)
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;
constexpr int kHistMaxSR = 12288;   // (sector,row) histogram kept in shared memory up to this many buckets (48 KB)

__global__ void __launch_bounds__(256) k_reset(Ctx c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < c.S) { c.zmin_key[i] = 0x7FFFFFFF; c.zmax_key[i] = (int)0x80000000; }
  for (int j = i; j < c.SR; j += gridDim.x * blockDim.x) c.sr_count[j] = 0;
  if (i == 0) {
    Counters z = {};
    *c.cnt = z;
  }
}

// ---------------------------------------------------------------------------------- z range + (s,r) counts
__global__ void __launch_bounds__(kThreads) k_zrange_count(Ctx c, int use_smem_hist) {
  extern __shared__ int s_hist[];                 // [SR] when use_smem_hist
  __shared__ int smin[kMaxRows], smax[kMaxRows];
  for (int i = threadIdx.x; i < c.S; i += blockDim.x) { smin[i] = 0x7FFFFFFF; smax[i] = (int)0x80000000; }
  if (use_smem_hist)
    for (int i = threadIdx.x; i < c.SR; i += blockDim.x) s_hist[i] = 0;
  __syncthreads();
  bool bad = false;
  const long long n = c.n;
  auto one = [&](int s, int r, float z) {
    if (s >= c.S || r >= c.R) { bad = true; return; }
    const int key = float_key(z);
    if (key < smin[s]) atomicMin(&smin[s], key);
    if (key > smax[s]) atomicMax(&smax[s], key);
    if (use_smem_hist) atomicAdd(&s_hist[s * c.R + r], 1);
    else atomicAdd(c.sr_count + s * c.R + r, 1);
  };
  // 4 clusters per thread per step: one 32-bit load of the sector bytes, one of the row bytes, one float4 of z
  const long long n4 = n >> 2;
  const uint32_t* sec4 = reinterpret_cast<const uint32_t*>(c.in_sector);
  const uint32_t* row4 = reinterpret_cast<const uint32_t*>(c.in_row);
  const float4* z4 = reinterpret_cast<const float4*>(c.in_z);
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (long long)gridDim.x * blockDim.x) {
    const uint32_t sw = __ldg(sec4 + q), rw = __ldg(row4 + q);
    const float4 zv = __ldg(z4 + q);
    one(sw & 0xFF, rw & 0xFF, zv.x);
    one((sw >> 8) & 0xFF, (rw >> 8) & 0xFF, zv.y);
    one((sw >> 16) & 0xFF, (rw >> 16) & 0xFF, zv.z);
    one(sw >> 24, rw >> 24, zv.w);
  }
  if (blockIdx.x == 0 && threadIdx.x < (int)(n & 3)) {   // ragged tail
    const long long i = (n4 << 2) + threadIdx.x;
    one(c.in_sector[i], c.in_row[i], c.in_z[i]);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < c.S; i += blockDim.x) {
    if (smin[i] != 0x7FFFFFFF) atomicMin(&c.zmin_key[i], smin[i]);
    if (smax[i] != (int)0x80000000) atomicMax(&c.zmax_key[i], smax[i]);
  }
  if (use_smem_hist)
    for (int i = threadIdx.x; i < c.SR; i += blockDim.x) {
      const int v = s_hist[i];
      if (v) atomicAdd(c.sr_count + i, v);
    }
  if (bad) atomicOr(&c.cnt->status, (int)TPC_STATUS_BAD_CLUSTER);
}

// ---------------------------------------------------------------------------------- tables
// exclusive prefix of `v` over the block (any blockDim <= 1024); *total = block sum.  smem: 33 ints.
__device__ __forceinline__ int block_exclusive(int v, int* smem, int* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  int inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int o = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += o;
  }
  if (lane == 31) smem[w] = inc;
  __syncthreads();
  if (w == 0) {
    const int s = lane < nw ? smem[lane] : 0;
    int si = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int o = __shfl_up_sync(0xffffffffu, si, d);
      if (lane >= d) si += o;
    }
    smem[lane] = si - s;                       // exclusive warp offsets
    if (lane == 31) smem[32] = si;
  }
  __syncthreads();
  const int r = smem[w] + inc - v;
  *total = smem[32];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(1024) k_tables(Ctx c) {
  __shared__ long long sbase[kMaxRows + 1];
  __shared__ int snz[kMaxRows];
  __shared__ int sscan[33];
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
  // row_start = exclusive scan of the (sector,row) counts; the partition cursors start there
  const bool dead = *reinterpret_cast<volatile int*>(&c.cnt->status) != 0;   // set before the barrier above (thread 0) or by k_zrange_count
  int carry = 0;
  for (int b = 0; b < c.SR; b += blockDim.x) {
    const int i = b + threadIdx.x;
    const int v = (i < c.SR && !dead) ? c.sr_count[i] : 0;
    int total;
    const int ex = block_exclusive(v, sscan, &total);
    if (i < c.SR) { c.row_start[i] = carry + ex; c.sr_cursor[i] = carry + ex; }
    carry += total;
  }
  if (threadIdx.x == 0) {
    c.row_start[c.SR] = carry;
    if (ok) c.bins[(int)sbase[c.S]] = carry;   // bin_start[N_b] = N
  }
}

// ---------------------------------------------------------------------------------- partition by (sector,row)
__global__ void __launch_bounds__(kThreads) k_partition(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  auto one = [&](int s, int r, float y, float z, long long i) {
    const int pos = atomicAdd(c.sr_cursor + s * c.R + r, 1);
    c.rec[pos] = make_float4(y, z, __int_as_float((int)i), 0.0f);
  };
  const long long n4 = n >> 2;
  const uint32_t* sec4 = reinterpret_cast<const uint32_t*>(c.in_sector);
  const uint32_t* row4 = reinterpret_cast<const uint32_t*>(c.in_row);
  const float4* y4 = reinterpret_cast<const float4*>(c.in_y);
  const float4* z4 = reinterpret_cast<const float4*>(c.in_z);
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (long long)gridDim.x * blockDim.x) {
    const uint32_t sw = __ldg(sec4 + q), rw = __ldg(row4 + q);
    const float4 yv = __ldg(y4 + q), zv = __ldg(z4 + q);
    const long long i = q << 2;
    one(sw & 0xFF, rw & 0xFF, yv.x, zv.x, i);
    one((sw >> 8) & 0xFF, (rw >> 8) & 0xFF, yv.y, zv.y, i + 1);
    one((sw >> 16) & 0xFF, (rw >> 16) & 0xFF, yv.z, zv.z, i + 2);
    one(sw >> 24, rw >> 24, yv.w, zv.w, i + 3);
  }
  if (blockIdx.x == 0 && threadIdx.x < (int)(n & 3)) {
    const long long i = (n4 << 2) + threadIdx.x;
    one(c.in_sector[i], c.in_row[i], c.in_y[i], c.in_z[i], i);
  }
}

// ---------------------------------------------------------------------------------- bin sort inside a (sector,row) bucket
// One CTA per bucket, buckets handed out by a ticket.  Everything the CTA touches at random (its bins,
// its slice of rec / perm / yz) was written moments ago and sits in L2; DRAM sees each array once.
// Reads of data that atomics or other threads of the CTA wrote go through L2 (__ldcg), never a stale L1 line.
template <int kT, int kMinCtas>
__global__ void __launch_bounds__(kT, kMinCtas) k_binsort(Ctx c) {
  __shared__ int s_scan[33];
  __shared__ int s_sr;
  if (c.cnt->status) return;
  const int tid = threadIdx.x;
  for (;;) {
    if (tid == 0) s_sr = atomicAdd(&c.cnt->s1_ticket, 1);
    __syncthreads();
    const int sr = s_sr;
    __syncthreads();
    if (sr >= c.SR) break;
    const int b0 = __ldg(c.bin_base + sr), nb = __ldg(c.bin_base + sr + 1) - b0;
    if (nb == 0) continue;                        // empty sector
    const int p0 = __ldg(c.row_start + sr), p1 = __ldg(c.row_start + sr + 1);
    const int s = sr / c.R, r = sr - s * c.R;
    const int ny = __ldg(&c.rowtab[r].ny), nzm1 = __ldg(c.nz + s) - 1;
    const float ymax = __ldg(&c.rowtab[r].ymax), zmin = __ldg(c.zmin + s);
    int* __restrict__ bins = c.bins + b0;
    auto local_bin = [&](float y, float z) {     // DESIGN.md section 3.1 step 3
      const int iy = floor_clamp((y + ymax) * c.inv_cy, ny - 1);
      const int iz = floor_clamp((z - zmin) * c.inv_cz, nzm1);
      return iz * ny + iy;
    };

    for (int j = tid; j < nb; j += kT) bins[j] = 0;
    __syncthreads();

    // histogram; the atomic's return value is the cluster's arrival rank inside its bin
#pragma unroll 4
    for (int i = p0 + tid; i < p1; i += kT) {
      const float4 v = __ldcg(c.rec + i);
      const int a = atomicAdd(bins + local_bin(v.x, v.y), 1);
      reinterpret_cast<int*>(c.rec + i)[3] = a;
    }
    __syncthreads();

    // exclusive scan of the bucket's bins, starting at row_start: bins[] becomes the CSR bin_start
    int carry = p0;
    for (int base = 0; base < nb; base += kT * 4) {
      const int j = base + tid * 4;
      int x[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) x[k] = (j + k < nb) ? __ldcg(bins + j + k) : 0;
      int total;
      int o = carry + block_exclusive((x[0] + x[1]) + (x[2] + x[3]), s_scan, &total);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (j + k < nb) bins[j + k] = o;
        o += x[k];
      }
      carry += total;
    }
    __syncthreads();

    // scatter (arrival order inside a bin)
#pragma unroll 4
    for (int i = p0 + tid; i < p1; i += kT) {
      const float4 v = __ldcg(c.rec + i);
      const int pos = __ldcg(bins + local_bin(v.x, v.y)) + __float_as_int(v.w);
      c.perm[pos] = __float_as_int(v.z);
      c.yz[pos] = make_float2(v.x, v.y);
      c.srow[pos] = (uint16_t)sr;
    }
    __syncthreads();

    // stable fix-up: order the clusters of a multiply-occupied bin by input index (bins hold ~1-3 clusters)
    for (int j = tid; j < nb; j += kT) {
      const int bs = __ldcg(bins + j), be = (j + 1 < nb) ? __ldcg(bins + j + 1) : p1;
      if (be - bs < 2) continue;
      for (int a = bs + 1; a < be; ++a) {          // insertion sort on (perm, yz)
        const int pa = __ldcg(c.perm + a);
        const float2 va = __ldcg(c.yz + a);
        int b = a - 1;
        while (b >= bs) {
          const int pb = __ldcg(c.perm + b);
          if (pb < pa) break;
          c.perm[b + 1] = pb;
          c.yz[b + 1] = __ldcg(c.yz + b);
          --b;
        }
        if (b + 1 != a) { c.perm[b + 1] = pa; c.yz[b + 1] = va; }
      }
    }
  }
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
  k_reset<<<(c.SR + 255) / 256 < 64 ? (c.SR + 255) / 256 : 64, 256, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launches_s1() { return 4; }
int launch_s1(const Ctx& c, cudaStream_t st) {
  const int smem_hist = c.SR <= kHistMaxSR;
  k_zrange_count<<<grid_for(c.n / 4 + 1, kThreads, c.n_sms, 8), kThreads, smem_hist ? c.SR * sizeof(int) : 0, st>>>(c, smem_hist);
  k_tables<<<1, 1024, 0, st>>>(c);
  k_partition<<<grid_for(c.n / 4 + 1, kThreads, c.n_sms, 8), kThreads, 0, st>>>(c);
  // big buckets: 1024 threads per bucket, two buckets per SM in flight; small ones: 256 threads, eight per SM
  if ((long long)c.n >= 2048LL * c.SR) k_binsort<1024, 2><<<grid_for(c.SR, 1, c.n_sms, 2), 1024, 0, st>>>(c);
  else k_binsort<256, 8><<<grid_for(c.SR, 1, c.n_sms, 8), 256, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
