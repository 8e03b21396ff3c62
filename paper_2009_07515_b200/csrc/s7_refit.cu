// S7 - refit of every track over the clusters it owns after the selector (the first slice of
// "Track Fit").  A separate call (tpc_tracker_refit), not part of the timed hot path: it reads what
// the last tpc_track_timeframe left in the workspace (hit tables, ownership masks, sorted clusters, the seed of every
// track) and writes one fitted state per track.
// One thread per track.  The owned clusters are walked from the top row down through the ownership bit mask; the seed
// direction comes from the top two, q/pT from the track, then propagate + update (no gate) cluster by cluster.
// Round 2, measured and rejected: the S4 pattern (persistent kernel, every lane pulls its next track from a ticket, one
// propagate + update step per loop iteration) - 10 -> ~25 of 32 lanes active, but 2.79 ms against 2.83: the kernel waits for
// the random 32-byte sectors of (y,z) behind the hit table (2.6 GB for 82 M clusters), not for idle lanes.
#include "kf.cuh"
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 128;

// walks the owned rows of a tracklet in DESCENDING order: next() returns the row or -1
struct OwnedRows {
  const unsigned* mask;
  int first, w;
  unsigned m;
  __device__ __forceinline__ OwnedRows(const unsigned* mask_, int first_, int words) : mask(mask_), first(first_), w(words - 1) {
    m = mask[w];
  }
  __device__ __forceinline__ int next() {
    while (m == 0) {
      if (--w < 0) return -1;
      m = mask[w];
    }
    const int bit = 31 - __clz(m);
    m &= ~(1u << bit);
    return first + 32 * w + bit;
  }
};

// a residual as a signed 16-bit count of steps - one fp32 product, round to nearest with ties
// to even (rintf), saturation at +-32767 with the comparisons written out (a NaN counts as below the range)
__device__ __forceinline__ short quantise_residual(float res, float inv_step) {
  const float v = res * inv_step;
  const float r = rintf(v);
  if (!(r > -32767.0f)) return (short)-32767;
  if (r >= 32767.0f) return (short)32767;
  return (short)(int)r;
}

__global__ void __launch_bounds__(kThreads) k_refit(Ctx c, FitPtrs o) {
  extern __shared__ float tx[];                         // row_x[r]
  for (int i = threadIdx.x; i < c.R; i += blockDim.x) tx[i] = c.rowtab[i].x;
  __syncthreads();
  if (c.cnt->status) return;
  const int nt = min(c.cnt->n_tracks, o.max_tracks), R = c.R;
  const size_t mt = (size_t)o.max_tracks;
  const float2* __restrict__ yz = c.yz;
  for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < nt; id += gridDim.x * blockDim.x) {
    const int sd = c.track_seed[id];
    const int* hit = c.t_hit + (size_t)sd * R;
    const int first = c.t_first_row[sd], last = c.t_last_row[sd];
    const int words = (last - first) / 32 + 1;          // mask words that can hold a bit
    OwnedRows rows(c.own_mask + (size_t)sd * c.mask_words, first, words);
    const int r_top = rows.next();
    OwnedRows rows2 = rows;                              // positioned after the top cluster
    const int r_nxt = rows.next();
    // residual slots: the owned clusters of track id sit at trk_cl_start[id] .. in ASCENDING row, the walk is descending
    const bool want_res = o.res_y != nullptr, want_q = o.qres_y != nullptr;
    int slot = want_res ? o.trk_cl_start[id + 1] - 1 : 0;
    const int slot0 = want_res ? o.trk_cl_start[id] : 0;
    KF k;
    int cur = r_top, nfit = 0;
    float zref = 0.f;
#pragma unroll
    for (int i = 0; i < 5; ++i) k.p[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 15; ++i) k.c[i] = 0.f;
    k.chi2 = 0.f;
    if (r_top >= 0 && r_nxt >= 0) {
      const float2 pt = __ldg(yz + hit[r_top]), pn = __ldg(yz + hit[r_nxt]);
      zref = pt.y;
      const float dx = tx[r_top] - tx[r_nxt];
      const float dy = pt.x - pn.x, dz = pt.y - pn.y;
      const float dl = sqrtf(dx * dx + dy * dy);
      k.p[0] = pt.x; k.p[1] = 0.0f; k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = c.t_par[(size_t)sd * 5 + 4];
      kf_reset_cov(k, c);
      nfit = 1;
      if (want_res) {
        o.res_y[slot] = 0.0f; o.res_z[slot] = 0.0f;
        if (want_q) { o.qres_y[slot] = 0; o.qres_z[slot] = 0; }
        --slot;
      }
      for (int r = rows2.next(); r >= 0; r = rows2.next()) {
        if (!kf_propagate(k, c.kb, tx[r] - tx[cur], c.max_sinphi)) break;
        const float2 v = __ldg(yz + hit[r]);
        if (want_res) {
          const float ry = v.x - k.p[0], rz = (v.y - zref) - k.p[1];
          o.res_y[slot] = ry; o.res_z[slot] = rz;
          if (want_q) { o.qres_y[slot] = quantise_residual(ry, o.inv_step_y); o.qres_z[slot] = quantise_residual(rz, o.inv_step_z); }
          --slot;
        }
        kf_update(k, v.x, v.y - zref, c.err_y2, c.err_z2);
        cur = r; ++nfit;
      }
    }
    if (want_res)
      for (; slot >= slot0; --slot) {                                                   // clusters that did not enter the fit
        o.res_y[slot] = 0.0f; o.res_z[slot] = 0.0f;
        if (want_q) { o.qres_y[slot] = 0; o.qres_z[slot] = 0; }
      }
#pragma unroll
    for (int i = 0; i < 5; ++i) o.par[i * mt + id] = k.p[i];
#pragma unroll
    for (int i = 0; i < 15; ++i) o.cov[i * mt + id] = k.c[i];
    o.chi2[id] = k.chi2;
    o.x_ref[id] = nfit ? tx[cur] : 0.f;
    o.z_ref[id] = zref;
    o.n_fit[id] = nfit;
    o.ndf[id] = nfit ? 2 * nfit - 5 : 0;
    c.fit_row[id] = nfit ? cur : 0;                     // for the merger (S9)
  }
}

}  // namespace

int launches_refit() { return 1; }
int launch_refit(const Ctx& c, const FitPtrs& o, cudaStream_t st) {
  long long g = ((long long)o.max_tracks + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * 256;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  k_refit<<<(unsigned)g, kThreads, c.R * sizeof(float), st>>>(c, o);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
