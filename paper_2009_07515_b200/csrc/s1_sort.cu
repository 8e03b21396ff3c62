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
//                   device-wide scan), scatter perm / (y,z) / srow; the clusters of a multiply-occupied
//                   bin take their stable rank (members with a smaller input index) in a final pass
// The result equals std::stable_sort by (sector,row,bin) whatever order the atomics resolved in.
// (Round 1a-c used one device-wide counting sort over the ~N global bins: every one of its ~8 accesses
// per cluster was a random 32-byte DRAM sector; 15.1 ms on cfg5, see profiles/.)
// Round 2, measured and rejected: the partition without global atomics (per-chunk (sector,row) histograms from the count
// pass, offsets by a scan over the chunks, shared-memory cursors per CTA): S1 4.45 -> 6.98 ms.  Each of the 1184 CTAs then
// owns its own 5472 write positions, ~14 records = 224 bytes per run: 6.5 M open write streams instead of 5472, and L2 no
// longer merges the 16-byte stores into full lines.  The shared global cursors are what keeps the writes dense.
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;
constexpr int kHistMaxSR = 11776;   // (sector,row) histogram kept in shared memory up to this many buckets: 46 KB dynamic + the 2 KB
                                    // of static smin/smax stay inside the 48 KB a kernel gets without opting in

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
  auto one = [&](int s, int r, float zin) {
    const float z = input_z(c, s, zin);                  // cm as given, or converted from the native time (section 3.0a)
    // a non-finite z has no bin (and an infinite one would make the z range, hence the bin count, meaningless)
    if (s >= c.S || r >= c.R || !(fabsf(z) < INFINITY)) { bad = true; return; }
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
    bool too_many = false;
    for (int s = 0; s < c.S; ++s) {
      const int kmin = c.zmin_key[s], kmax = c.zmax_key[s];
      int nz = 0;
      float zmin = 0.f, zmax = 0.f;
      if (kmin <= kmax) {
        zmin = key_float(kmin); zmax = key_float(kmax);
        // the row count stays a float until it is known to fit: a huge |z| (1e30) would saturate the conversion and the
        // "+ 1" would wrap; such a grid is a BINS_OVERFLOW like any other grid that is too large
        const float rows = floorf((zmax - zmin) * c.inv_cz);
        if (!(rows < 2147483646.0f)) { too_many = true; nz = 0; }
        else nz = (int)rows + 1;
      }
      c.zmin[s] = zmin; c.zmax[s] = zmax; c.nz[s] = nz; snz[s] = nz;
      sbase[s] = acc;
      acc += (long long)nz * c.ny_total;
    }
    sbase[c.S] = acc;
    int st = 0;
    if (too_many) sbase[c.S] = acc = 2147483647LL;             // every thread sees "not ok" below
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
  bool bad = false;
  auto one = [&](int s, int r, float yin, float zin, long long i) {
    const float z = input_z(c, s, zin);
    const float y = input_y(c, r, yin);                 // cm as given, or converted from the pad coordinate (section 3.0b)
    if (!(fabsf(y) < INFINITY)) bad = true;             // precondition: finite coordinates (z was checked by k_zrange_count)
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
  if (bad) atomicOr(&c.cnt->status, (int)TPC_STATUS_BAD_CLUSTER);
}

// ---------------------------------------------------------------------------------- bin sort inside a (sector,row) bucket
// One CTA per bucket, buckets handed out by a ticket.
//
// Slab path (the normal one).  A bucket of cfg5 holds ~17 k clusters and ~10^5 bins: with two buckets per SM in
// flight the bins + records of all of them (~1 MB each) do not fit L2, and every random access to them was a DRAM
// sector (19 GB of DRAM traffic for 4 GB of useful bytes, profiles/).  So the CTA first splits its bucket into z-slabs
// of whole bin rows (a counting sort over <= 64 slab ids, shared-memory counters, records copied rec -> rec2), then
// bin-sorts one slab at a time ENTIRELY in shared memory: the slab's records arrive with one 1-D TMA bulk copy
// (cp.async.bulk + mbarrier) while the bins are cleared, then slab histogram (shared atomics), exclusive scan, CSR
// written out once with coalesced stores, stable rank inside multiply-occupied bins from a shared-memory table of
// input indices.  Global memory sees: rec read twice, rec2 written and read once, outputs and bin_start written once
// (7.7 GB of DRAM traffic on cfg5; 10.5 GB when the three sub-steps each re-read rec2, 19 GB before the slab split).
// Global path (fallback when a slab's bins or clusters do not fit the shared-memory tables): the same steps on
// the whole bucket with the bins in global memory.
// Reads of data that atomics or other threads of the CTA wrote go through L2 (__ldcg), never a stale L1 line.
constexpr int kMaxSlabs = 128;
constexpr int kSlabTarget = 768;  // clusters per slab aimed at (cap / target = 2.7: no bucket of cfg5 falls back; 1024 -> 10 % did)
constexpr int kSlabBinCap = 8192;     // bins of one slab held in shared memory (48 KB)
constexpr int kSlabCluCap = 2048;     // clusters of one slab whose input indices fit the shared-memory table (16 KB)

struct BucketGeom {
  int sr, b0, nb, p0, p1, ny, nzm1;
  uint16_t srow;                      // (sector << 8) | row, what the sorted srow[] array holds
  float ymax, zmin;
};

__device__ __forceinline__ int local_bin_of(const Ctx& c, const BucketGeom& g, float y, float z) {   // DESIGN.md 3.1 step 3
  const int iy = floor_clamp((y + g.ymax) * c.inv_cy, g.ny - 1);
  const int iz = floor_clamp((z - g.zmin) * c.inv_cz, g.nzm1);
  return iz * g.ny + iy;
}

template <int kT>
__device__ void bucket_global(const Ctx& c, const BucketGeom& g, int* s_scan) {
  const int tid = threadIdx.x;
  const int nb = g.nb, p0 = g.p0, p1 = g.p1;
  int* __restrict__ bins = c.bins + g.b0;
  for (int j = tid; j < nb; j += kT) bins[j] = 0;
  __syncthreads();
  // histogram; the atomic's return value is the cluster's arrival rank inside its bin
#pragma unroll 4
  for (int i = p0 + tid; i < p1; i += kT) {
    const float4 v = __ldcg(c.rec + i);
    const int a = atomicAdd(bins + local_bin_of(c, g, v.x, v.y), 1);
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
  // scatter: alone in its bin -> final place; else park the input index at bin_start + arrival rank
  int* __restrict__ tmp = c.flag_scan;          // free until S3
#pragma unroll 4
  for (int i = p0 + tid; i < p1; i += kT) {
    const float4 v = __ldcg(c.rec + i);
    const int b = local_bin_of(c, g, v.x, v.y);
    const int bs = __ldcg(bins + b), be = (b + 1 < nb) ? __ldcg(bins + b + 1) : p1;
    if (be - bs == 1) {
      c.perm[bs] = __float_as_int(v.z);
      c.yz[bs] = make_float2(v.x, v.y);
      c.srow[bs] = g.srow;
    } else {
      tmp[bs + __float_as_int(v.w)] = __float_as_int(v.z);
    }
  }
  __syncthreads();
  // multiply-occupied bins: stable rank = number of members with a smaller input index
#pragma unroll 2
  for (int i = p0 + tid; i < p1; i += kT) {
    const float4 v = __ldcg(c.rec + i);
    const int b = local_bin_of(c, g, v.x, v.y);
    const int bs = __ldcg(bins + b), be = (b + 1 < nb) ? __ldcg(bins + b + 1) : p1;
    if (be - bs == 1) continue;
    const int idx = __float_as_int(v.z);
    int rank = 0;
    for (int q = bs; q < be; ++q) rank += (__ldcg(tmp + q) < idx);
    const int pos = bs + rank;
    c.perm[pos] = idx;
    c.yz[pos] = make_float2(v.x, v.y);
    c.srow[pos] = g.srow;
  }
}

struct SlabShared {
  float4 recs[kSlabCluCap];           // the records of the slab in flight: one 1-D TMA bulk copy from rec2 (32 KB)
  unsigned long long mbar;            // mbarrier the bulk copy completes on
  int bins[kSlabBinCap];              // slab histogram, then exclusive offsets inside the slab
  int idx[kSlabCluCap];               // input indices of the clusters of multiply-occupied bins, at offset + arrival rank
  int cnt[kMaxSlabs + 1];             // clusters per slab, then exclusive offsets (cnt[n_slab] = bucket size)
  int cur[kMaxSlabs];                 // write cursors of the slab split
  int scan[33];
  int sr;
  int fits;
};

// ---- 1-D TMA bulk copy global -> shared, completion on an mbarrier (cp.async.bulk; SASS UBLKCP)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* mbar) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* mbar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(mbar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* mbar, unsigned parity) {
  unsigned done;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(done)
                 : "r"(smem_u32(mbar)), "r"(parity)
                 : "memory");
  } while (!done);
}

template <int kT>
__device__ void bucket_slabs(const Ctx& c, const BucketGeom& g, SlabShared& sh, int n_slab, int slab_rows, unsigned& parity) {
  const int tid = threadIdx.x;
  const int p0 = g.p0, p1 = g.p1, ny = g.ny, nz = g.nzm1 + 1;
  float4* __restrict__ rec2 = c.rec2;
  // ---- split the bucket into z-slabs: count, offsets, copy rec -> rec2 (arrival order inside a slab is arbitrary)
  auto slab_of = [&](float z) { return floor_clamp((z - g.zmin) * c.inv_cz, g.nzm1) / slab_rows; };
  for (int i = p0 + tid; i < p1; i += kT) atomicAdd(&sh.cnt[slab_of(__ldcg(c.rec + i).y)], 1);
  __syncthreads();
  if (tid == 0) {
    int acc = 0, fits = 1;
    for (int k = 0; k < n_slab; ++k) {
      const int v = sh.cnt[k];
      if (v > kSlabCluCap) fits = 0;
      sh.cnt[k] = acc; sh.cur[k] = acc;
      acc += v;
    }
    sh.cnt[n_slab] = acc;
    sh.fits = fits;
  }
  __syncthreads();
  if (!sh.fits) {
    if (tid == 0) atomicAdd(&c.cnt->s1_global, 1);
    bucket_global<kT>(c, g, sh.scan);
    return;
  }     // a slab with too many clusters: whole bucket the slow way
#pragma unroll 4
  for (int i = p0 + tid; i < p1; i += kT) {
    const float4 v = __ldcg(c.rec + i);
    rec2[p0 + atomicAdd(&sh.cur[slab_of(v.y)], 1)] = v;
  }
  asm volatile("fence.proxy.async;" ::: "memory");      // these generic-proxy stores are read back by the TMA engine
  __syncthreads();

  // ---- one slab at a time, in shared memory
  for (int k = 0; k < n_slab; ++k) {
    const int q0 = p0 + sh.cnt[k], m = sh.cnt[k + 1] - sh.cnt[k];
    const int rows = min(slab_rows, nz - k * slab_rows);
    const int nbs = rows * ny, bbase = k * slab_rows * ny;
    // the slab's records come in with one bulk copy while the bins are being cleared
    if (tid == 0 && m > 0) tma_load_1d(sh.recs, rec2 + q0, (unsigned)m * 16u, &sh.mbar);
    for (int j = tid; j < nbs; j += kT) sh.bins[j] = 0;
    __syncthreads();
    if (m > 0) { mbar_wait(&sh.mbar, parity); parity ^= 1u; }
    // histogram: arrival rank inside the bin is the atomic's return value, kept in the (shared) record
    for (int i = tid; i < m; i += kT) {
      const float4 v = sh.recs[i];
      const int a = atomicAdd(&sh.bins[local_bin_of(c, g, v.x, v.y) - bbase], 1);
      reinterpret_cast<int*>(sh.recs + i)[3] = a;
    }
    __syncthreads();
    // exclusive scan in place; the CSR goes out with coalesced stores
    int carry = 0;
    for (int base = 0; base < nbs; base += kT * 4) {
      const int j = base + tid * 4;
      int x[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) x[e] = (j + e < nbs) ? sh.bins[j + e] : 0;
      int total;
      int o = carry + block_exclusive((x[0] + x[1]) + (x[2] + x[3]), sh.scan, &total);
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if (j + e < nbs) { sh.bins[j + e] = o; c.bins[g.b0 + bbase + j + e] = q0 + o; }
        o += x[e];
      }
      carry += total;
    }
    __syncthreads();
    // alone in its bin -> final place; else park the input index in the shared table
    for (int i = tid; i < m; i += kT) {
      const float4 v = sh.recs[i];
      const int bl = local_bin_of(c, g, v.x, v.y) - bbase;
      const int bs = sh.bins[bl], be = (bl + 1 < nbs) ? sh.bins[bl + 1] : m;
      if (be - bs == 1) {
        c.perm[q0 + bs] = __float_as_int(v.z);
        c.yz[q0 + bs] = make_float2(v.x, v.y);
        c.srow[q0 + bs] = g.srow;
      } else {
        sh.idx[bs + __float_as_int(v.w)] = __float_as_int(v.z);
      }
    }
    __syncthreads();
    // multiply-occupied bins: stable rank = number of members with a smaller input index
    for (int i = tid; i < m; i += kT) {
      const float4 v = sh.recs[i];
      const int bl = local_bin_of(c, g, v.x, v.y) - bbase;
      const int bs = sh.bins[bl], be = (bl + 1 < nbs) ? sh.bins[bl + 1] : m;
      if (be - bs == 1) continue;
      const int idx = __float_as_int(v.z);
      int rank = 0;
      for (int q = bs; q < be; ++q) rank += (sh.idx[q] < idx);
      const int pos = q0 + bs + rank;
      c.perm[pos] = idx;
      c.yz[pos] = make_float2(v.x, v.y);
      c.srow[pos] = g.srow;
    }
    __syncthreads();                               // sh.bins / sh.idx are reused by the next slab
  }
}

template <int kT, int kMinCtas>
__global__ void __launch_bounds__(kT, kMinCtas) k_binsort(Ctx c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SlabShared& sh = *reinterpret_cast<SlabShared*>(smem_raw);
  if (c.cnt->status) return;
  const int tid = threadIdx.x;
  if (tid == 0) mbar_init(&sh.mbar);
  unsigned parity = 0;                            // phase of sh.mbar the next bulk copy completes (same in every thread)
  for (;;) {
    __syncthreads();                               // everybody is done with the previous bucket's shared state
    if (tid == 0) sh.sr = atomicAdd(&c.cnt->s1_ticket, 1);
    for (int k = tid; k <= kMaxSlabs; k += kT) sh.cnt[k] = 0;
    __syncthreads();
    BucketGeom g;
    g.sr = sh.sr;
    if (g.sr >= c.SR) break;
    g.b0 = __ldg(c.bin_base + g.sr); g.nb = __ldg(c.bin_base + g.sr + 1) - g.b0;
    if (g.nb == 0) continue;                       // empty sector
    g.p0 = __ldg(c.row_start + g.sr); g.p1 = __ldg(c.row_start + g.sr + 1);
    const int s = g.sr / c.R, r = g.sr - s * c.R;
    g.srow = (uint16_t)((s << 8) | r);
    g.ny = __ldg(&c.rowtab[r].ny); g.nzm1 = __ldg(c.nz + s) - 1;
    g.ymax = __ldg(&c.rowtab[r].ymax); g.zmin = __ldg(c.zmin + s);
    const int m = g.p1 - g.p0, nz = g.nzm1 + 1;
    if (m == 0) {                                  // a row without clusters: its bins all start at row_start
      for (int j = tid; j < g.nb; j += kT) c.bins[g.b0 + j] = g.p0;
      continue;
    }
    int n_slab = (m + kSlabTarget - 1) / kSlabTarget;
    const long long by_bins = ((long long)nz * g.ny + kSlabBinCap - 1) / kSlabBinCap;   // a slab's bins must fit too
    if (by_bins > n_slab) n_slab = (int)(by_bins < kMaxSlabs ? by_bins : kMaxSlabs);
    if (n_slab > kMaxSlabs) n_slab = kMaxSlabs;
    if (n_slab > nz) n_slab = nz;
    const int slab_rows = (nz + n_slab - 1) / n_slab;
    n_slab = (nz + slab_rows - 1) / slab_rows;
    if ((long long)slab_rows * g.ny <= kSlabBinCap) bucket_slabs<kT>(c, g, sh, n_slab, slab_rows, parity);
    else {
      if (tid == 0) atomicAdd(&c.cnt->s1_global, 1);
      bucket_global<kT>(c, g, sh.scan);
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

// per device, once per tracker (tpc_tracker_create): the bin sort needs more than 48 KB of dynamic shared memory
int init_s1() {
  if (cudaFuncSetAttribute(k_binsort<512, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SlabShared)) != cudaSuccess ||
      cudaFuncSetAttribute(k_binsort<256, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SlabShared)) != cudaSuccess)
    return -1;
  return 0;
}

int launches_s1() { return 4; }
int launch_s1(const Ctx& c, cudaStream_t st) {
  const int smem_hist = c.SR <= kHistMaxSR;
  k_zrange_count<<<grid_for(c.n / 4 + 1, kThreads, c.n_sms, 8), kThreads, smem_hist ? c.SR * sizeof(int) : 0, st>>>(c, smem_hist);
  k_tables<<<1, 1024, 0, st>>>(c);
  k_partition<<<grid_for(c.n / 4 + 1, kThreads, c.n_sms, 128), kThreads, 0, st>>>(c);
  // big buckets: 512 threads per bucket, three buckets per SM in flight (73 KB of shared memory each); small ones: 256
  // threads, three per SM
  if ((long long)c.n >= 2048LL * c.SR) k_binsort<512, 3><<<grid_for(c.SR, 1, c.n_sms, 3), 512, sizeof(SlabShared), st>>>(c);
  else k_binsort<256, 3><<<grid_for(c.SR, 1, c.n_sms, 3), 256, sizeof(SlabShared), st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
