// S3 - cellular-automaton link cleaner (BASELINE.json north_star (3)): keeps a link
// only if it is reciprocal, finds chain heads, assigns chain lengths and numbers the seeds.
//   k_clean   out of place from the raw arrays: link_up/link_dn; seed bit = head of a chain with >= min_chain_len nodes
//   scan      inclusive scan of the seed bits -> seed id = rank (ascending head position: deterministic)
//   k_seeds   seed_head[id] = i          (seed_len[id] = full chain length is counted by S4 while it follows the chain)
#include "tpc_internal.cuh"
#include "../../include/tpc_tracker.h"

namespace tpc {
namespace {

constexpr int kThreads = 256;

// Out of place from the raw arrays.  A head (cleaned up-link, no cleaned down-link) is a seed iff its chain has at
// least min_chain_len nodes: that needs min_chain_len - 2 further steps only, taken on the RAW arrays (a cleaned link
// p -> q exists iff raw_up[p] == q and raw_dn[q] == p).  The full chain length (seed_len) is counted by S4, which walks
// the whole chain anyway (round 1b walked every chain here as well: 2.8 ms of dependent loads at 6.7 lanes).
__global__ void __launch_bounds__(kThreads) k_clean(Ctx c) {
  if (c.cnt->status) return;
  const long long n = c.n;
  const int* __restrict__ ru = c.link_up_raw;
  const int* __restrict__ rd = c.link_dn_raw;
  int linked = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int u = ru[i], d = rd[i];
    const int lu = (u >= 0 && __ldg(rd + u) == (int)i) ? u : -1;
    const int ld = (d >= 0 && __ldg(ru + d) == (int)i) ? d : -1;
    c.link_up[i] = lu;
    c.link_dn[i] = ld;
    linked += (lu >= 0);
    int seed = 0;
    if (lu >= 0 && ld < 0) {
      int len = 2, p = lu;
      while (len < c.min_chain_len) {
        const int q = __ldg(ru + p);
        if (q < 0 || __ldg(rd + q) != p) break;
        p = q; ++len;
      }
      seed = len >= c.min_chain_len;
    }
    c.flag_scan[i] = seed;
  }
  // chain edges, for the bytes model only
  for (int o = 16; o; o >>= 1) linked += __shfl_xor_sync(0xffffffffu, linked, o);
  if ((threadIdx.x & 31) == 0 && linked) atomicAdd(&c.cnt->n_linked, linked);
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
    const int inc = c.flag_scan[i], prev = i ? c.flag_scan[i - 1] : 0;
    if (inc != prev) {                                   // seed_len[id] is written by S4
      const int id = inc - 1;
      c.seed_head[id] = (int)i;
      // everything S4 needs to start the tracklet, gathered here (3 dependent loads per seed that S4's refill would
      // otherwise take with one active lane): head, next, their (y,z), (sector << 8 | row) of the head, row of next
      const int nx = c.link_up[i];
      const float2 ph = c.yz[i], pn = c.yz[nx];
      const int srh = c.srow[i], r1 = c.srow[nx] & 255;
      c.seed_rec[2 * (size_t)id] = make_float4(ph.x, ph.y, pn.x, pn.y);
      c.seed_rec[2 * (size_t)id + 1] = make_float4(__int_as_float((int)i), __int_as_float(nx), __int_as_float(srh), __int_as_float(r1));
    }
  }
}

}  // namespace

int launches_s3() { return 3 + 3; }
int launch_s3(const Ctx& c, cudaStream_t st) {
  long long g = ((long long)c.n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 8;     // one resident wave (measured: 8 -> 1.09 ms, 16 -> 1.30, 64 -> 1.28)
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  k_clean<<<(unsigned)g, kThreads, 0, st>>>(c);
  // host-known length: *n_ptr = 0 (cnt->zero), n_add = n
  if (launch_scan_inclusive(c.flag_scan, &c.cnt->zero, c.n, c.n, c.tile_sums, &c.cnt->n_seeds, c.n_sms, st)) return -1;
  k_seed_count<<<1, 1, 0, st>>>(c);
  k_seeds<<<(unsigned)g, kThreads, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
