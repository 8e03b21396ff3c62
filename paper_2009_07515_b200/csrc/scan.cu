// Device-wide in-place inclusive scan (int32) whose length lives on the device.
// Reduce-then-scan in three launches: per-tile sums, one-block scan of the tile sums, per-tile
// rescan with the tile offset.  Used by S1 (bin histogram -> CSR), S3 (seed ids), S5 (tracklet /
// track ids, CSR of attached clusters): every id in the pipeline is a rank from a scan, never the
// return value of an atomic, so ids are deterministic.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 256;
constexpr int kItems = kScanTile / kThreads;   // 8
static_assert(kItems == 8, "two int4 per thread");

__device__ __forceinline__ int warp_inclusive(int v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// exclusive prefix of `v` over the block; *total = block sum.  smem: 32 ints.
__device__ __forceinline__ int block_exclusive(int v, int* smem, int* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int inc = warp_inclusive(v, lane);
  if (lane == 31) smem[w] = inc;
  __syncthreads();
  if (w == 0) {
    const int s = lane < nw ? smem[lane] : 0;
    const int si = warp_inclusive(s, lane);
    smem[lane] = si - s;                       // exclusive warp offsets
    if (lane == nw - 1) smem[32] = si;
  }
  __syncthreads();
  const int r = smem[w] + inc - v;
  *total = smem[32];
  __syncthreads();
  return r;
}

__device__ __forceinline__ void load_tile(const int* __restrict__ data, long long base, long long n, int (&x)[kItems]) {
  const long long o = base + (long long)threadIdx.x * kItems;
  if (base + kScanTile <= n) {
    const int4 a = *reinterpret_cast<const int4*>(data + o);
    const int4 b = *reinterpret_cast<const int4*>(data + o + 4);
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
  } else {
#pragma unroll
    for (int i = 0; i < kItems; ++i) x[i] = (o + i < n) ? data[o + i] : 0;
  }
}

__global__ void __launch_bounds__(kThreads) k_scan_reduce(const int* __restrict__ data, const int* __restrict__ n_ptr,
                                                          int n_add, int* __restrict__ tile_sums) {
  __shared__ int sm[33];
  const long long n = (long long)*n_ptr + n_add;
  const long long tiles = (n + kScanTile - 1) / kScanTile;
  for (long long t = blockIdx.x; t < tiles; t += gridDim.x) {
    int x[kItems];
    load_tile(data, t * kScanTile, n, x);
    int s = 0;
#pragma unroll
    for (int i = 0; i < kItems; ++i) s += x[i];
    int total;
    block_exclusive(s, sm, &total);
    if (threadIdx.x == 0) tile_sums[t] = total;
  }
}

// one block: exclusive scan of tile_sums[0..tiles) in place, carry across chunks of blockDim
__global__ void __launch_bounds__(1024) k_scan_sums(int* __restrict__ tile_sums, const int* __restrict__ n_ptr, int n_add,
                                                    int* __restrict__ total_out) {
  __shared__ int sm[33];
  const long long n = (long long)*n_ptr + n_add;
  const int tiles = (int)((n + kScanTile - 1) / kScanTile);
  int carry = 0;
  for (int b = 0; b < tiles; b += blockDim.x) {
    const int i = b + threadIdx.x;
    const int v = i < tiles ? tile_sums[i] : 0;
    int total;
    const int ex = block_exclusive(v, sm, &total);
    if (i < tiles) tile_sums[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(kThreads) k_scan_apply(int* __restrict__ data, const int* __restrict__ n_ptr, int n_add,
                                                         const int* __restrict__ tile_sums) {
  __shared__ int sm[33];
  const long long n = (long long)*n_ptr + n_add;
  const long long tiles = (n + kScanTile - 1) / kScanTile;
  for (long long t = blockIdx.x; t < tiles; t += gridDim.x) {
    const long long base = t * kScanTile;
    int x[kItems];
    load_tile(data, base, n, x);
#pragma unroll
    for (int i = 1; i < kItems; ++i) x[i] += x[i - 1];
    int total;
    const int off = block_exclusive(x[kItems - 1], sm, &total) + tile_sums[t];
    const long long o = base + (long long)threadIdx.x * kItems;
    if (base + kScanTile <= n) {
      *reinterpret_cast<int4*>(data + o) = make_int4(x[0] + off, x[1] + off, x[2] + off, x[3] + off);
      *reinterpret_cast<int4*>(data + o + 4) = make_int4(x[4] + off, x[5] + off, x[6] + off, x[7] + off);
    } else {
#pragma unroll
      for (int i = 0; i < kItems; ++i)
        if (o + i < n) data[o + i] = x[i] + off;
    }
  }
}

}  // namespace

int launch_scan_inclusive(int* data, const int* n_ptr, int n_add, long long max_n, int* tile_sums, int* total_out,
                          int n_sms, cudaStream_t st) {
  const long long max_tiles = (max_n + kScanTile - 1) / kScanTile;
  long long g = (long long)n_sms * 8;
  if (g > max_tiles) g = max_tiles;
  if (g < 1) g = 1;
  k_scan_reduce<<<(unsigned)g, kThreads, 0, st>>>(data, n_ptr, n_add, tile_sums);
  k_scan_sums<<<1, 1024, 0, st>>>(tile_sums, n_ptr, n_add, total_out);
  k_scan_apply<<<(unsigned)g, kThreads, 0, st>>>(data, n_ptr, n_add, tile_sums);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
