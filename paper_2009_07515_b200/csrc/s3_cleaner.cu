// S3 - cellular-automaton link cleaner (BASELINE.json north_star (3)): keeps a link
// only if it is reciprocal, finds chain heads, assigns chain lengths and numbers the seeds.
//   k_clean   out of place from the raw arrays: link_up/link_dn
//   k_heads   flag[i] = chain length if i is a head with length >= min_chain_len, else 0;
//             head_bit[i] = (flag[i] != 0)
//   scan      inclusive scan of head_bit -> seed id = rank (ascending head position: deterministic)
//   k_seeds   seed_head[id] = i, seed_len[id] = length
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads) k_clean(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  int linked = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int u = c.link_up_raw[i], d = c.link_dn_raw[i];
    const int lu = (u >= 0 && __ldg(c.link_dn_raw + u) == (int)i) ? u : -1;
    const int ld = (d >= 0 && __ldg(c.link_up_raw + d) == (int)i) ? d : -1;
    c.link_up[i] = lu;
    c.link_dn[i] = ld;
    linked += (lu >= 0);
  }
  // chain edges, for the bytes model only
  for (int o = 16; o; o >>= 1) linked += __shfl_xor_sync(0xffffffffu, linked, o);
  if ((threadIdx.x & 31) == 0 && linked) atomicAdd(&c.cnt->n_linked, linked);
}

__global__ void __launch_bounds__(kThreads) k_heads(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  bool cycle = false;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    int len = 0;
    if (c.link_up[i] >= 0 && c.link_dn[i] < 0) {
      for (int p = (int)i; p >= 0; p = __ldg(c.link_up + p)) {
        if (++len > c.R) { cycle = true; break; }   // links always go up in row: cannot happen
      }
      if (len < c.min_chain_len) len = 0;
    }
    c.flag[i] = len;
    c.flag_scan[i] = len != 0;
  }
  if (cycle) atomicOr(&c.cnt->status, (int)TPC_STATUS_CHAIN_CYCLE);
}

__global__ void k_seed_count(Ctx c) {
  if (c.cnt->status) { c.cnt->n_seeds = 0; return; }
  if (c.cnt->n_seeds > c.max_seeds) {
    atomicOr(&c.cnt->status, (int)TPC_STATUS_SEEDS_OVERFLOW);
    c.cnt->n_seeds = 0;
  }
}

__global__ void __launch_bounds__(kThreads) k_seeds(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int len = c.flag[i];
    if (len) {
      const int id = c.flag_scan[i] - 1;
      c.seed_head[id] = (int)i;
      c.seed_len[id] = len;
    }
  }
}

}  // namespace

int launches_s3() { return 4 + 3; }
int launch_s3(const Ctx& c, cudaStream_t st) {
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 16;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  k_clean<<<(unsigned)g, kThreads, 0, st>>>(c);
  k_heads<<<(unsigned)g, kThreads, 0, st>>>(c);
  // host-known length: *n_ptr = 0 (cnt->zero), n_add = n
  if (launch_scan_inclusive(c.flag_scan, &c.cnt->zero, c.n, c.n, c.tile_sums, &c.cnt->n_seeds, c.n_sms, st)) return -1;
  k_seed_count<<<1, 1, 0, st>>>(c);
  k_seeds<<<(unsigned)g, kThreads, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
