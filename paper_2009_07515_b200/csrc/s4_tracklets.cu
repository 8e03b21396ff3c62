// S4 - tracklet constructor (BASELINE.json north_star (4)): per seed, follow the chain
// upward with Kalman updates (phase A), extrapolate further up picking up gated nearest clusters
// (phase B), turn round with a reset covariance and refit downward with pick-up (phase C).
// 5-parameter filter (y, z - z_ref, sin(phi), tan(lambda), q/pT) in the sector-local frame, exact
// circle propagation in a uniform Bz, full 5x5 symmetric covariance (15 unique entries) in
// registers, textbook update.
//
// Persistent kernel, one thread per tracklet, ONE uniform step loop for all three phases: every
// iteration each lane resolves its next row (chain cluster, row above, row below), then all lanes run
// the same propagate -> candidate (known cluster or grid search) -> update code together, whatever
// phase they are in.  A lane that finishes writes its tracklet and takes the next seed from a global
// ticket (idle lanes of a warp are served by one atomic: ballot + popc), so lanes never wait for the
// longest chain of a batch.  (Round 1a ran the three phases as three loops per 32-seed batch and
// measured 3.7 active lanes per instruction; see profiles/.)
//
// Hit table t_hit[seed][row]: no clearing pass.  A lane writes every row it visits between the lowest
// updated row and the turning row (a position, or -1 for a skipped / empty row), so the entries in
// [first_row, last_row] are all defined and nothing outside that range is ever read (S5 and the debug
// view honour the range).
//
// Measured and rejected on cfg5 (this version: 12.8 ms): the searches of a warp laid end to end and tested 32
// candidates at a time (warp scan, owner lookup, 64-bit shared-memory atomicMin of (d2, position)): 12.9 ms, bit-exact
// but no faster; the known-cluster loads hoisted above the transport: no change; S5's ownership votes cast by the
// finishing lane: S4 +4.2 ms for S5 -2.8 ms; 8 CTAs per SM (64 registers, spills): 14.7 ms; an L2 prefetch of the next
// row's bin_start entry at the linearly extrapolated position, issued one step ahead: 15.9 ms (20 more instructions
// in a divergent region cost more than the latency they hide).
//
// Round 2, measured on cfg5 with ncu source-level counters (profiles/r02_s4_regions.md): the transport and the update
// run at 29.9 and 28.4 of 32 lanes; the grid search runs at 9.4 lanes (3.6 inside its candidate loop), is 36 % of the
// warp instructions and 55 % of the stall samples (two dependent gathers, bin_start then (y,z)).  Tried and rejected,
// all bit-exact:
//  * searches batched inside the warp (lanes that need a search wait until 8 .. 28 lanes do, then search together):
//    14.1 ms at 8, 15.0 at 16, 27 at 28 lanes - searches come in runs per lane (phase B, below the head), so waiting
//    lanes idle for many steps and the memory-level parallelism drops;
//  * the bin_start line of the next search prefetched (prefetch.global.L1 / .L2, or a real load kept in a register)
//    at the straight-line prediction before the transport: 13.0 - 13.4 ms against 12.9 for the same code without it;
//    ncu: L1 hits rose by the number of prefetches, the stall at the first use of bin_start did not move - a warp waits
//    for the slowest of its ~9 searching lanes (second bin row, rare misprediction), not for the average one;
//  * streaming stores / loads (st.global.cs, ld.global.cs) for the hit table: 12.26 ms against 12.06;
//  * covariance in shared memory, two buffers (live / last update, no copy), transport staged row by row: 64 registers,
//    8 CTAs per SM, occupancy 37 -> 49 %: 11.8 ms (7 CTAs 11.7, 9 CTAs 12.8, 10 CTAs 19.8), but DRAM reads 10.5 -> 16.7 GB
//    and L2 hit rate 53 -> 47 %: the lanes in flight (608-byte hit table each, plus the rows they walk) already exceed
//    L2, so more warps buy latency hiding with cache misses - occupancy is not the lever, the working set is;
//  * L2 warm-up: every refill asks (prefetch.global.L2::evict_last) for its slice of bin_start, (y,z) and link_up 0.5 - 4
//    sectors ahead of the ticket: 13.2 ms, DRAM reads 10.5 -> 15.8 GB, L2 hit rate 53 -> 45 % - the kernel refills all of
//    L2 every 0.14 ms (875 GB/s of misses into 126 MB) while a tracklet lives 0.4 ms, so nothing asked for ahead of time
//    survives until it is used.
//
// Arithmetic is written operation by operation in the order of DESIGN.md section 3.4 (compiled with
// -fmad=false; fused multiply-adds only where the text writes fma(), as __fmaf_rn): the transport J C J^T skips only
// the terms that are structurally 0*x or 1*x.
#include "kf.cuh"
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 128;
constexpr int kW = 2;                         // candidates of a search loaded together (measured: 1 -> 13.2 ms, 2 -> 12.0, 3 -> 12.8, 4 -> 12.6; 3 and 4 spill)
constexpr int kCtasPerSm = 6;              // 80 registers per thread (measured: 4 -> 17.7 ms, 5 -> 15.5, 6 -> 13.9, 7 -> 13.9, 8 spills -> 14.7)

// nearest gated cluster of row r of sector s, or -1
__device__ __forceinline__ int kf_search(const Ctx& c, int b0, int ny, float ymax, int nz, float zmin, const KF& k,
                                         float zref, float* ym, float* zm) {
  const float cut = c.pick_chi2_cut;
  const float sy2 = k.c[CI(0, 0)] + c.err_y2, sz2 = k.c[CI(1, 1)] + c.err_z2;
  const float hy = sqrtf(cut * sy2), hz = sqrtf(cut * sz2);
  const float zabs = zref + k.p[1];
  const float ylo = k.p[0] - hy, yhi = k.p[0] + hy, zlo = zabs - hz, zhi = zabs + hz;
  const float wy = 1.0f / sy2, wz = 1.0f / sz2;
  float best = INFINITY;
  int arg = -1;
  const int iy0 = floor_clamp((ylo + ymax) * c.inv_cy, ny - 1);
  const int iy1 = floor_clamp((yhi + ymax) * c.inv_cy, ny - 1);
  const int iz0 = floor_clamp((zlo - zmin) * c.inv_cz, nz - 1);
  const int iz1 = floor_clamp((zhi - zmin) * c.inv_cz, nz - 1);
  const int* __restrict__ bins = c.bins;
  const float2* __restrict__ yz = c.yz;
  // The window almost always covers one or two bin rows: their four bin_start entries are loaded together and the
  // two candidate runs are walked as ONE loop (a nested row / candidate loop pays the load latency once per level
  // and once per row).  Visiting order (row ascending, position ascending) is that of DESIGN.md section 3.1.
  for (int iz = iz0; iz <= iz1; iz += 2) {
    const int b = b0 + iz * ny;
    const bool two = iz + 1 <= iz1;
    const int jb0 = __ldg(bins + b + iy0), je0 = __ldg(bins + b + iy1 + 1);
    const int jb1 = two ? __ldg(bins + b + ny + iy0) : 0, je1 = two ? __ldg(bins + b + ny + iy1 + 1) : 0;
    const int n0 = je0 - jb0, total = n0 + (je1 - jb1);
    const int shift = jb1 - n0;                   // t >= n0: j = jb1 + (t - n0)
    for (int t = 0; t < total; t += kW) {         // kW candidates in flight
      int j[kW];
      float2 v[kW];
#pragma unroll
      for (int e = 0; e < kW; ++e) {
        const int te = t + e;
        j[e] = te < n0 ? jb0 + te : shift + te;
        if (te < total) v[e] = __ldg(yz + j[e]);
      }
#pragma unroll
      for (int e = 0; e < kW; ++e) {
        if (t + e < total && v[e].x >= ylo && v[e].x <= yhi && v[e].y >= zlo && v[e].y <= zhi) {
          const float dy = v[e].x - k.p[0];
          const float dz = (v[e].y - zref) - k.p[1];
          const float d2 = (dy * dy) * wy + (dz * dz) * wz;
          if (d2 <= cut && d2 < best) { best = d2; arg = j[e]; *ym = v[e].x; *zm = v[e].y; }
        }
      }
    }
  }
  return arg;
}

enum : int { kIdle = 0, kPhaseA = 1, kPhaseB = 2, kPhaseC = 3 };

template <int kCtas>
__global__ void __launch_bounds__(kThreads, kCtas) k_tracklets(Ctx c) {
  extern __shared__ float smem[];
  const int R = c.R;
  float* tx = smem;                               // row_x[r]
  float* tymax = smem + R;                        // ymax_r
  int* tny = reinterpret_cast<int*>(smem + 2 * R);   // ny_r
  for (int i = threadIdx.x; i < R; i += blockDim.x) {
    tx[i] = c.rowtab[i].x; tymax[i] = c.rowtab[i].ymax; tny[i] = c.rowtab[i].ny;
  }
  __syncthreads();
  if (c.cnt->status) return;
  const int n_seeds = c.cnt->n_seeds;
  const int lane = threadIdx.x & 31;
  const float2* __restrict__ yz = c.yz;
  const int* __restrict__ link_up = c.link_up;
  const float ey2 = c.err_y2, ez2 = c.err_z2, kb = c.kb, msp = c.max_sinphi, ymargin = c.y_margin;
  const int max_gap = c.max_gap;

  unsigned long long steps = 0, hits_kept = 0;
  bool exhausted = false;                         // warp-uniform: the ticket ran out

  // per-lane tracklet state
  int phase = kIdle;
  int sd = 0, sR = 0, r0 = 0, cur = 0, gap = 0, nh = 0, last_row = 0, low = 0, nextcl = -1, nz = 0;
  float zref = 0.f, zmin = 0.f;
  int* hit = nullptr;
  KF k;
  // sv: state at the last update (A/B: parameters only; C: the output).  It lives in shared memory ([entry][thread],
  // conflict-free): 21 registers fewer per thread buy a fifth and sixth resident CTA per SM.
  float* sv = smem + 3 * R + threadIdx.x;         // entry e at sv[e * kThreads]: 0-4 parameters, 5-19 covariance, 20 chi2
#pragma unroll
  for (int i = 0; i < 5; ++i) k.p[i] = 0.f;
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = 0.f;
  k.chi2 = 0.f;

  for (;;) {
    // ---- refill idle lanes from the ticket
    const unsigned idle = __ballot_sync(0xffffffffu, phase == kIdle);
    if (idle && !exhausted) {
      const int leader = __ffs(idle) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(&c.cnt->s4_ticket, __popc(idle));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (base + __popc(idle) >= n_seeds) exhausted = true;
      if (phase == kIdle) {
        const int mine = base + __popc(idle & ((1u << lane) - 1u));
        if (mine < n_seeds) {
          sd = mine;
          hit = c.t_hit + (size_t)sd * R;
          const float4 sa = __ldg(c.seed_rec + 2 * (size_t)sd), sb = __ldg(c.seed_rec + 2 * (size_t)sd + 1);   // written by S3's k_seeds
          const int h = __float_as_int(sb.x), nx = __float_as_int(sb.y), srh = __float_as_int(sb.z), r1 = __float_as_int(sb.w);
          const int s = srh >> 8;                 // srh = (sector << 8) | row
          sR = s * R; r0 = srh & 255;
          nz = __ldg(c.nz + s); zmin = __ldg(c.zmin + s);
          const float2 ph = make_float2(sa.x, sa.y), pn = make_float2(sa.z, sa.w);
          zref = ph.y;
          const float dx = tx[r1] - tx[r0];
          const float dy = pn.x - ph.x;
          const float dz = pn.y - zref;
          const float dl = sqrtf(dx * dx + dy * dy);
          k.p[0] = ph.x; k.p[1] = 0.0f; k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = 0.0f;
          kf_reset_cov(k, c);
#pragma unroll
          for (int i = 0; i < 5; ++i) sv[i * kThreads] = k.p[i];
          hit[r0] = h;
          cur = r0; last_row = r0; low = r0; nh = 1; gap = 0; nextcl = nx;
          phase = kPhaseA;
        }
      }
    }
    if (!__any_sync(0xffffffffu, phase != kIdle)) break;

    // ---- resolve this lane's next row r and its known cluster cl (or -1: search)
    bool act = false, go_c = false, done = false;
    int r = 0, cl = -1;
    if (phase == kPhaseA) {
      if (nextcl >= 0) {
        cl = nextcl;
        r = cur + 1 + (cl >= __ldg(c.row_start + sR + cur + 2));   // links go up one row or two
        act = true;
      } else {
        c.seed_len[sd] = nh;                      // end of the chain: every node was absorbed (S3 leaves the count to us)
        phase = kPhaseB; gap = 0;
      }
    }
    if (phase == kPhaseB) {
      if (cur + 1 < R) { r = cur + 1; act = true; }
      else go_c = true;
    } else if (phase == kPhaseC) {
      if (cur >= 1) { r = cur - 1; cl = (r >= r0) ? hit[r] : -1; act = true; }
      else done = true;
    }

    // ---- one Kalman step, the same code for every phase.  The explicit barrier makes the lanes of the three
    // phases reconverge here: without it the compiler keeps the phase branches apart and runs the step once per
    // phase group (round 1b: 28.0 M executions of the step for 8.7 M loop iterations, 9.5 lanes each).
    __syncwarp();
    if (act) {
      ++steps;
      bool stop = false;
      if (!kf_propagate(k, kb, tx[r] - tx[cur], msp)) stop = true;
      else {
        const int prev = cur;
        cur = r;
        if (phase != kPhaseA && !(fabsf(k.p[0]) <= tymax[r] + ymargin)) stop = true;
        else {
          float ym, zm;
          const bool known = cl >= 0;
          if (known) { const float2 v = __ldg(yz + cl); ym = v.x; zm = v.y; }
          else cl = kf_search(c, __ldg(c.bin_base + sR + r), tny[r], tymax[r], nz, zmin, k, zref, &ym, &zm);
          if (cl >= 0) {
            kf_update(k, ym, zm - zref, ey2, ez2);
            gap = 0;
            if (!known) { hit[r] = cl; ++nh; }
#pragma unroll
            for (int i = 0; i < 5; ++i) sv[i * kThreads] = k.p[i];
            if (phase == kPhaseC) {
#pragma unroll
              for (int i = 0; i < 15; ++i) sv[(5 + i) * kThreads] = k.c[i];
              sv[20 * kThreads] = k.chi2;
              low = r;
            } else {
              last_row = r;
              if (phase == kPhaseA) {
                hit[r] = cl; ++nh;
                if (r == prev + 2) hit[prev + 1] = -1;
                nextcl = __ldg(link_up + cl);
              }
            }
          } else {
            if (phase == kPhaseB || r < r0) hit[r] = -1;
            if (++gap > max_gap) stop = true;
          }
        }
      }
      if (stop) {
        if (phase == kPhaseC) done = true;
        else {
          go_c = true;                            // a failed step of A skips B
          if (phase == kPhaseA) {                 // rare: count the chain nodes the filter did not reach
            int len = nh;
            for (int p = nextcl; p >= 0; p = __ldg(link_up + p)) ++len;
            c.seed_len[sd] = len;
          }
        }
      }
    }

    // ---- turn round: back to the last updated state, covariance and chi2 reset
    if (go_c) {
#pragma unroll
      for (int i = 0; i < 5; ++i) k.p[i] = sv[i * kThreads];
      kf_reset_cov(k, c);
#pragma unroll
      for (int i = 0; i < 15; ++i) sv[(5 + i) * kThreads] = k.c[i];
      sv[20 * kThreads] = 0.0f;
      cur = last_row; low = last_row; gap = 0;
      phase = kPhaseC;
    }

    // ---- finished: write the tracklet, become idle
    if (done) {
      for (int rr = r0; rr < low; ++rr) nh -= (hit[rr] >= 0);   // only if phase C stopped above the head
      c.t_first_row[sd] = low; c.t_last_row[sd] = last_row; c.t_n_hits[sd] = nh;
      float* op = c.t_par + (size_t)sd * 5;
      float* oc = c.t_cov + (size_t)sd * 15;
#pragma unroll
      for (int i = 0; i < 5; ++i) op[i] = sv[i * kThreads];
#pragma unroll
      for (int i = 0; i < 15; ++i) oc[i] = sv[(5 + i) * kThreads];
      c.t_chi2[sd] = sv[20 * kThreads]; c.t_zref[sd] = zref;
      if (nh >= c.min_tracklet_hits) hits_kept += nh;
      phase = kIdle;
    }
  }

  for (int o = 16; o; o >>= 1) {
    steps += __shfl_xor_sync(0xffffffffu, steps, o);
    hits_kept += __shfl_xor_sync(0xffffffffu, hits_kept, o);
  }
  if (lane == 0) {
    if (steps) atomicAdd(&c.cnt->kf_steps, steps);
    if (hits_kept) atomicAdd(&c.cnt->n_hits, hits_kept);
  }
}

}  // namespace

int launches_s4() { return 1; }
int launch_s4(const Ctx& c, cudaStream_t st) {
  // persistent: every SM filled with resident CTAs; lanes pull seeds until the ticket runs out
  k_tracklets<kCtasPerSm><<<c.n_sms * kCtasPerSm, kThreads, (3 * c.R + 21 * kThreads) * sizeof(float), st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
