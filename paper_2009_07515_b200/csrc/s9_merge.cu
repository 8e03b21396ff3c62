// S9 - track merger (the second slice of "Track Fit"): the segments a
// physical track was found in - one per sector it crosses, one per stretch between holes longer than max_gap - are
// joined by comparing the state at the outer end of one with the state at the inner end of the other, and every
// joined track is refitted over all its clusters.  A separate call (tpc_tracker_merge) after tpc_track_timeframe and
// tpc_tracker_refit; it reads what those left in the workspace and the refit's output.
//
//   k_merge_tables   one thread: a z grid per sector for the inner ends (bin width = dz_win, doubled until the bins fit)
//   k_refit_up       thread per track: upward refit (3.9.1) -> state at the outer end; z of both ends, sector; counts the
//                    inner end into its (sector, z) bin
//   scan + k_merge_fill   counting sort of 16-byte inner-end records by (sector, z bin): "extensive use of sort" - here
//                    a hand-written counting sort (no Thrust / CUB), the window of 3.9.3 is then a contiguous run of bins
//   k_merge_match    warp per outer end: candidates of 3.9.3 from the bins around z_out, score 3.9.4 (rotation +
//                    helix step + chi2), best partner of the outer end by a warp reduction (ties -> lowest id), best partner of
//                    every inner end by a 64-bit atomicMin of (chi2 bits, id) - both independent of the visiting order
//   k_merge_link     mutual best -> links (3.9.5);  flags + scan -> merged ids (3.9.6)
//   k_chain_len / scan / k_chain_fill   chains followed from their heads: merged_of_track, CSR merged -> segments
//   k_refit_merged   thread per merged track: downward refit through all segments, the frame turned at sector changes (3.9.7)
//
// Arithmetic: fp32, -fmad=false, the operations of DESIGN.md section 3.9 in the order written (the helix step and the
// update are those of S4, kf.cuh); bit-identical to the oracle.
#include "kf.cuh"
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 128;

// the state turned into the frame rotated by the angle with sine sa and cosine ca
__device__ __forceinline__ bool kf_rotate(KF& k, float kb, float x, float sa, float ca, float max_sinphi, float* x_new) {
  const float y = k.p[0], s = k.p[2], t = k.p[3], q = k.p[4];
  if (!(fabsf(s) < max_sinphi)) return false;
  const float c = sqrtf(1.0f - s * s);
  const float s1 = s * ca - c * sa;
  const float c1 = c * ca + s * sa;
  if (!(fabsf(s1) < max_sinphi) || !(c1 > 0.0f)) return false;
  const float xn = x * ca + y * sa;
  const float yn = y * ca - x * sa;
  const float j00 = c / c1;
  const float j10 = ((0.0f - sa) * t) / c1;
  const float j20 = (0.0f - kb * q) * sa;
  const float j22 = c1 / c;
  // M = J C: rows 3 and 4 of J are unit rows; M0 = j00 C0, M1 = j10 C0 + C1, M2 = j20 C0 + j22 C2
  float m0[5], m1[5], m2[5];
#pragma unroll
  for (int l = 0; l < 5; ++l) {
    m0[l] = j00 * k.c[CI(0, l)];
    m1[l] = j10 * k.c[CI(0, l)] + k.c[CI(1, l)];
    m2[l] = j20 * k.c[CI(0, l)] + j22 * k.c[CI(2, l)];
  }
  // C'[i][0] = M[i][0] j00;  C'[i][1] = M[i][0] j10 + M[i][1];  C'[i][2] = M[i][0] j20 + M[i][2] j22;  C'[i][3,4] = M[i][3,4]
  float n[15];
  n[CI(0, 0)] = m0[0] * j00;
  n[CI(1, 0)] = m1[0] * j00;
  n[CI(2, 0)] = m2[0] * j00;
  n[CI(3, 0)] = k.c[CI(3, 0)] * j00;
  n[CI(4, 0)] = k.c[CI(4, 0)] * j00;
  n[CI(1, 1)] = m1[0] * j10 + m1[1];
  n[CI(2, 1)] = m2[0] * j10 + m2[1];
  n[CI(3, 1)] = k.c[CI(3, 0)] * j10 + k.c[CI(3, 1)];
  n[CI(4, 1)] = k.c[CI(4, 0)] * j10 + k.c[CI(4, 1)];
  n[CI(2, 2)] = m2[0] * j20 + m2[2] * j22;
  n[CI(3, 2)] = k.c[CI(3, 0)] * j20 + k.c[CI(3, 2)] * j22;
  n[CI(4, 2)] = k.c[CI(4, 0)] * j20 + k.c[CI(4, 2)] * j22;
  n[CI(3, 3)] = k.c[CI(3, 3)];
  n[CI(4, 3)] = k.c[CI(4, 3)];
  n[CI(4, 4)] = k.c[CI(4, 4)];
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = n[i];
  k.p[0] = yn; k.p[2] = s1;
  *x_new = xn;
  return true;
}

// owned rows of a tracklet in ASCENDING order
struct OwnedRowsUp {
  const unsigned* mask;
  int first, w, words;
  unsigned m;
  __device__ __forceinline__ OwnedRowsUp(const unsigned* mask_, int first_, int words_) : mask(mask_), first(first_), w(0), words(words_) {
    m = mask[0];
  }
  __device__ __forceinline__ int next() {
    while (m == 0) {
      if (++w >= words) return -1;
      m = mask[w];
    }
    const int bit = __ffs(m) - 1;
    m &= m - 1;
    return first + 32 * w + bit;
  }
};
// ... and in DESCENDING order
struct OwnedRowsDown {
  const unsigned* mask;
  int first, w;
  unsigned m;
  __device__ __forceinline__ OwnedRowsDown(const unsigned* mask_, int first_, int words) : mask(mask_), first(first_), w(words - 1) {
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

__device__ __forceinline__ int n_tracks_of(const Ctx& c, const MergePtrs& o) { return min(c.cnt->n_tracks, o.max_tracks); }

// ---------------------------------------------------------------------------------- z grid of the inner ends
__global__ void k_merge_tables(Ctx c, float w0, int new_merge) {
  if (threadIdx.x || blockIdx.x) return;
  MergeCounters& mc = *c.mcnt;
  if (new_merge) mc.n_merged = 0;
  mc.status = 0;
  // bins a quarter of the window wide: a query reads 9-10 bins, 1.25 x the window instead of 3 x with bins of dz_win
  float w = w0;
  for (int it = 0; it < 64; ++it, w = w * 2.0f) {
    const float inv_w = 1.0f / w;
    long long acc = 0;
    for (int s = 0; s < c.S; ++s) {
      c.m_bin_base[s] = (int)acc;
      int nzb = 0;
      if (c.nz[s] > 0) {
        const float rows = floorf((c.zmax[s] - c.zmin[s]) * inv_w);
        nzb = rows < 1.0e9f ? (int)rows + 1 : 2000000000;
      }
      c.m_nzb[s] = nzb;
      acc += nzb;
      if (acc > c.max_merge_bins) break;
    }
    if (acc <= c.max_merge_bins) {
      c.m_bin_base[c.S] = (int)acc;
      mc.n_bins = (int)acc; mc.inv_w = inv_w;
      return;
    }
  }
  mc.n_bins = 0; mc.inv_w = 0.0f; mc.status = 1;      // cannot happen for finite z ranges: 2^64 * dz_win covers everything
}

__global__ void __launch_bounds__(kThreads) k_merge_clear(Ctx c, MergePtrs o) {
  const int nb = c.mcnt->n_bins;
  const int nt = n_tracks_of(c, o);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= nb; i += gridDim.x * blockDim.x) c.m_bin_start[i] = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += gridDim.x * blockDim.x) {
    c.m_best_b[i] = -1; c.m_chi_b[i] = -1.0f; c.m_dir_b[i] = 0;
    c.m_best_a[i] = ~0ull;
    c.m_next[i] = -1; c.m_prev[i] = -1; c.m_dir[i] = 0;
    // -1 = in no merged track: what a track keeps when no chain head reaches it (a cycle of links) and
    // what every track has when the run was aborted by a status bit - never the previous content of the caller's buffer
    o.merged_of_track[i] = -1;
  }
}

__device__ __forceinline__ int merge_bin(const Ctx& c, int s, float z, float inv_w) {
  return c.m_bin_base[s] + floor_clamp((z - c.zmin[s]) * inv_w, c.m_nzb[s] - 1);
}

// ---------------------------------------------------------------------------------- 3.9.1 upward refit + end bookkeeping
__global__ void __launch_bounds__(kThreads) k_refit_up(Ctx c, FitPtrs f, MergePtrs o) {
  extern __shared__ float tx[];
  for (int i = threadIdx.x; i < c.R; i += blockDim.x) tx[i] = c.rowtab[i].x;
  __syncthreads();
  if (c.cnt->status || c.mcnt->status) return;
  const int nt = n_tracks_of(c, o), R = c.R;
  const size_t mt = (size_t)c.max_tracks, ft = (size_t)f.max_tracks;
  const float inv_w = c.mcnt->inv_w;
  const float2* __restrict__ yz = c.yz;
  for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < nt; id += gridDim.x * blockDim.x) {
    const int sd = c.track_seed[id];
    const int* hit = c.t_hit + (size_t)sd * R;
    const int first = c.t_first_row[sd], last = c.t_last_row[sd];
    const int words = (last - first) / 32 + 1;
    OwnedRowsUp rows(c.own_mask + (size_t)sd * c.mask_words, first, words);
    const int r_bot = rows.next();
    const int r_nxt = rows.next();
    KF k;
#pragma unroll
    for (int i = 0; i < 5; ++i) k.p[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 15; ++i) k.c[i] = 0.f;
    k.chi2 = 0.f;
    int cur = max(r_bot, 0), nfit = 0, sector = 0;
    float zref = 0.f;
    if (r_bot >= 0) sector = c.srow[hit[r_bot]] >> 8;
    if (r_bot >= 0 && r_nxt >= 0) {
      const float2 pb = __ldg(yz + hit[r_bot]), pn = __ldg(yz + hit[r_nxt]);
      zref = pb.y;
      const float dx = tx[r_nxt] - tx[r_bot];
      const float dy = pn.x - pb.x, dz = pn.y - pb.y;
      const float dl = sqrtf(dx * dx + dy * dy);
      k.p[0] = pb.x; k.p[1] = 0.0f; k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = f.par[4 * ft + id];
      kf_reset_cov(k, c);
      nfit = 1;
      for (int r = r_nxt; r >= 0; r = rows.next()) {
        if (!kf_propagate(k, c.kb, tx[r] - tx[cur], c.max_sinphi)) break;
        const float2 v = __ldg(yz + hit[r]);
        kf_update(k, v.x, v.y - zref, c.err_y2, c.err_z2);
        cur = r; ++nfit;
      }
    }
#pragma unroll
    for (int i = 0; i < 5; ++i) c.up_par[i * mt + id] = k.p[i];
#pragma unroll
    for (int i = 0; i < 15; ++i) c.up_cov[i * mt + id] = k.c[i];
    c.up_chi2[id] = k.chi2;
    c.up_x[id] = nfit ? tx[cur] : 0.f;
    c.up_zref[id] = zref;
    c.up_row[id] = nfit ? cur : 0;
    c.up_n[id] = nfit;
    c.m_sector[id] = sector;
    const float z_in = f.z_ref[id] + f.par[1 * ft + id];
    c.m_zin[id] = z_in;
    c.m_zout[id] = zref + k.p[1];
    // the inner end goes into its (sector, z) bin (every track: those that take no part are skipped when read) - unless
    // its sector has no grid (a track without an owned row is filed under sector 0, which may be empty): no bin then
    const int b = c.m_nzb[sector] > 0 ? merge_bin(c, sector, z_in, inv_w) : -1;
    c.m_bin_of[id] = b;
    // the record the candidate scan reads: z_in, the row of the inner state (-1: takes no part), the id, x of the inner state
    c.m_rec[id] = make_float4(z_in, __int_as_float(nfit >= 2 && f.n_fit[id] >= 2 ? c.fit_row[id] : -1), __int_as_float(id), f.x_ref[id]);
    if (b >= 0) atomicAdd(c.m_bin_start + b + 1, 1);  // counts at b + 1: the inclusive scan leaves the CSR starts in place
  }
}

__global__ void __launch_bounds__(kThreads) k_merge_fill(Ctx c, MergePtrs o) {
  if (c.cnt->status || c.mcnt->status) return;
  const int nt = n_tracks_of(c, o);
  for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < nt; id += gridDim.x * blockDim.x) {
    const int b = c.m_bin_of[id];
    if (b < 0) continue;
    const int pos = c.m_bin_start[b] + atomicAdd(c.m_bin_fill + b, 1);
    c.m_srec[pos] = c.m_rec[id];
  }
}

__global__ void __launch_bounds__(kThreads) k_merge_zero_fill(Ctx c) {
  const int nb = c.mcnt->n_bins;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nb; i += gridDim.x * blockDim.x) c.m_bin_fill[i] = 0;
}

// ---------------------------------------------------------------------------------- 3.9.3 - 3.9.5 candidates, score, choice
// One WARP per outer end: the lanes read the window's run of 16-byte records together (coalesced; a thread per outer end
// walked ~130 records one dependent load after the other: 35 ms on cfg5), apply the cheap cuts, and the few lanes whose
// record survives score their pair.  Lane-local best (chi2, then id), then a warp reduction with the same order.
__global__ void __launch_bounds__(kThreads) k_merge_match(Ctx c, FitPtrs f, MergePtrs o) {
  extern __shared__ float sm[];
  float* tymax = sm;
  for (int i = threadIdx.x; i < c.R; i += blockDim.x) tymax[i] = c.rowtab[i].ymax;
  __syncthreads();
  if (c.cnt->status || c.mcnt->status) return;
  const int nt = n_tracks_of(c, o), n_az = c.S >> 1;
  const size_t mt = (size_t)c.max_tracks, ft = (size_t)f.max_tracks;
  const float inv_w = c.mcnt->inv_w;
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  for (int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; a < nt; a += warps) {
    if (c.up_n[a] < 2 || f.n_fit[a] < 2) continue;       // warp-uniform
    const int s_a = c.m_sector[a], r_a = c.up_row[a];
    const float y_a = c.up_par[0 * mt + a];
    const float x_a = c.up_x[a], zref_a = c.up_zref[a], z_out = c.m_zout[a];
    const float zlo = z_out - o.dz_win, zhi = z_out + o.dz_win;
    float best = 0.f;
    int bb = -1, bdir = 0;
    for (int pass = 0; pass < 2; ++pass) {
      int dir = 0, s_b = s_a;
      if (pass == 1) {
        if (n_az < 1) continue;                           // a one-sector geometry has no neighbour
        if (!(fabsf(y_a) >= tymax[r_a] - o.edge)) continue;
        dir = y_a >= 0.0f ? 1 : -1;
        s_b = (s_a / n_az) * n_az + ((s_a % n_az) + dir + n_az) % n_az;
        if (s_b == s_a) continue;
      }
      if (c.m_nzb[s_b] == 0) continue;
      // 3.9.4, first half (once per pass, every lane the same): the outer state, turned into the neighbour's frame
      KF k0;
#pragma unroll
      for (int i = 0; i < 5; ++i) k0.p[i] = c.up_par[i * mt + a];
#pragma unroll
      for (int i = 0; i < 15; ++i) k0.c[i] = c.up_cov[i * mt + a];
      k0.chi2 = 0.f;
      float x0 = x_a;
      if (dir != 0 && !kf_rotate(k0, c.kb, x0, dir > 0 ? o.sin_a : 0.0f - o.sin_a, o.cos_a, c.max_sinphi, &x0)) continue;
      const float zslope = k0.p[3] / sqrtf(1.0f - k0.p[2] * k0.p[2]);   // the road of 3.9.3: dz/dx of a straight continuation
      const int b0 = merge_bin(c, s_b, zlo, inv_w), b1 = merge_bin(c, s_b, zhi, inv_w);
      const int j0 = c.m_bin_start[b0], j1 = c.m_bin_start[b1 + 1];
      for (int j = j0 + lane; j < j1; j += 32) {
        const float4 rec = __ldg(c.m_srec + j);         // (z_in, row of the inner state or -1, id, x of the inner state)
        const int b = __float_as_int(rec.z), r_b = __float_as_int(rec.y);
        const float z_b = rec.x;
        if (b == a || r_b < 0) continue;
        if (!(z_b >= zlo && z_b <= zhi)) continue;
        if (dir == 0 ? (r_b < r_a + 1 || r_b > r_a + o.max_rows) : (r_b < r_a - o.back_rows || r_b > r_a + o.max_rows)) continue;
        const float dxb = rec.w - x0;
        if (!(fabsf(z_b - (z_out + dxb * zslope)) <= o.road_z0 + o.road_z1 * fabsf(dxb))) continue;
        KF k = k0;
        if (!kf_propagate(k, c.kb, dxb, c.max_sinphi)) continue;
        float d[5];
        d[0] = f.par[0 * ft + b] - k.p[0];
        d[1] = z_b - (zref_a + k.p[1]);
        d[2] = f.par[2 * ft + b] - k.p[2];
        d[3] = f.par[3 * ft + b] - k.p[3];
        d[4] = f.par[4 * ft + b] - k.p[4];
        float chi = 0.0f;
#pragma unroll
        for (int i = 0; i < 5; ++i) chi = chi + (d[i] * d[i]) / (k.c[CI(i, i)] + f.cov[(size_t)CI(i, i) * ft + b]);
        if (!(chi <= o.chi2_cut)) continue;
        if (bb < 0 || chi < best || (chi == best && b < bb)) { best = chi; bb = b; bdir = dir; }
        // high word: order-preserving unsigned key of chi (fp32 variances can come out slightly negative, and then so
        // does chi); low word = id -> ties go to the lowest a
        const unsigned cb = __float_as_uint(chi + 0.0f);   // -0 -> +0: the oracle's `chi == best` makes no difference between them
        const unsigned ck = (cb & 0x80000000u) ? ~cb : (cb | 0x80000000u);
        atomicMin(c.m_best_a + b, ((unsigned long long)ck << 32) | (unsigned)a);
      }
    }
    __syncwarp();
#pragma unroll
    for (int off = 16; off; off >>= 1) {
      const float ochi = __shfl_xor_sync(0xffffffffu, best, off);
      const int ob = __shfl_xor_sync(0xffffffffu, bb, off), od = __shfl_xor_sync(0xffffffffu, bdir, off);
      if (ob >= 0 && (bb < 0 || ochi < best || (ochi == best && ob < bb))) { best = ochi; bb = ob; bdir = od; }
    }
    if (lane == 0) { c.m_best_b[a] = bb; c.m_dir_b[a] = bdir; c.m_chi_b[a] = bb >= 0 ? best : -1.0f; }
  }
}

__global__ void __launch_bounds__(kThreads) k_merge_link(Ctx c, MergePtrs o) {
  if (c.cnt->status || c.mcnt->status) return;
  const int nt = n_tracks_of(c, o);
  for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < nt; a += gridDim.x * blockDim.x) {
    const int b = c.m_best_b[a];
    if (b >= 0 && (int)(c.m_best_a[b] & 0xFFFFFFFFull) == a) { c.m_next[a] = b; c.m_prev[b] = a; c.m_dir[a] = c.m_dir_b[a]; }
  }
}

__global__ void __launch_bounds__(kThreads) k_merge_heads(Ctx c, MergePtrs o) {
  const int nt = (c.cnt->status || c.mcnt->status) ? 0 : n_tracks_of(c, o);
  if (blockIdx.x == 0 && threadIdx.x == 0) c.mcnt->n_scan = nt;
  for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < nt; a += gridDim.x * blockDim.x) c.m_head_scan[a] = c.m_prev[a] < 0;
}

// merged id of a head = its rank; the chain is followed once for the length and the members' ids ...
__global__ void __launch_bounds__(kThreads) k_chain_len(Ctx c, MergePtrs o) {
  const int nt = c.mcnt->n_scan;
  if (blockIdx.x == 0 && threadIdx.x == 0) { *o.n_merged = nt ? c.m_head_scan[nt - 1] : 0; c.mcnt->n_merged = nt ? c.m_head_scan[nt - 1] : 0; }
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < nt; h += gridDim.x * blockDim.x) {
    if (c.m_prev[h] >= 0) continue;
    const int m = c.m_head_scan[h] - 1;
    int len = 0;
    for (int k = h; k >= 0 && len < nt; k = c.m_next[k], ++len) o.merged_of_track[k] = m;
    c.m_seg_scan[m] = len;
    c.m_head_of[m] = h;
  }
}

// ... and once more to write the CSR (seg_scan is now the inclusive scan of the lengths)
__global__ void __launch_bounds__(kThreads) k_chain_fill(Ctx c, MergePtrs o) {
  const int nm = c.mcnt->n_merged, nt = c.mcnt->n_scan;
  if (blockIdx.x == 0 && threadIdx.x == 0) o.seg_start[0] = 0;
  for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < nm; m += gridDim.x * blockDim.x) {
    const int end = c.m_seg_scan[m];
    o.seg_start[m + 1] = end;
    int pos = m ? c.m_seg_scan[m - 1] : 0;
    int len = 0;
    for (int k = c.m_head_of[m]; k >= 0 && len < nt; k = c.m_next[k], ++len) o.seg_idx[pos++] = k;
  }
}

// ---------------------------------------------------------------------------------- 3.9.7 merged refit
__global__ void __launch_bounds__(kThreads) k_refit_merged(Ctx c, MergePtrs o) {
  extern __shared__ float tx[];
  for (int i = threadIdx.x; i < c.R; i += blockDim.x) tx[i] = c.rowtab[i].x;
  __syncthreads();
  const int nm = c.mcnt->n_merged, R = c.R;
  const size_t mo = (size_t)o.max_tracks;
  const float2* __restrict__ yz = c.yz;
  for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < nm; m += gridDim.x * blockDim.x) {
    const int s0 = o.seg_start[m], s1 = o.seg_start[m + 1];
    KF k;
#pragma unroll
    for (int i = 0; i < 5; ++i) k.p[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 15; ++i) k.c[i] = 0.f;
    k.chi2 = 0.f;
    float x = 0.f, zref = 0.f;
    int nfit = 0, ncl = 0, sector = 0;
    bool ok = true, started = false;
    for (int q = s1 - 1; q >= s0; --q) {
      const int seg = o.seg_idx[q];
      const int sd = c.track_seed[seg];
      ncl += c.k_owned[sd];
      if (!ok) continue;                                // only the cluster count goes on
      const int* hit = c.t_hit + (size_t)sd * R;
      const int first = c.t_first_row[sd], last = c.t_last_row[sd];
      OwnedRowsDown rows(c.own_mask + (size_t)sd * c.mask_words, first, (last - first) / 32 + 1);
      int r = rows.next();
      if (q == s1 - 1) {
        OwnedRowsDown peek = rows;
        const int r_nxt = peek.next();
        if (r < 0 || r_nxt < 0) { ok = false; continue; }
        sector = c.m_sector[seg];
        const float2 pt = __ldg(yz + hit[r]), pn = __ldg(yz + hit[r_nxt]);
        zref = pt.y;
        const float dx = tx[r] - tx[r_nxt];
        const float dy = pt.x - pn.x, dz = pt.y - pn.y;
        const float dl = sqrtf(dx * dx + dy * dy);
        k.p[0] = pt.x; k.p[1] = 0.0f; k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = c.t_par[(size_t)sd * 5 + 4];
        kf_reset_cov(k, c);
        x = tx[r]; nfit = 1; started = true;
        r = rows.next();
      } else {
        const int dir = c.m_dir[seg];
        if (dir != 0) {
          const float sd_ = dir > 0 ? o.sin_a : 0.0f - o.sin_a;
          const float2 pc = __ldg(yz + hit[r]);
          const float xt = tx[r] * o.cos_a + pc.x * sd_;
          if (!kf_propagate(k, c.kb, xt - x, c.max_sinphi)) { ok = false; continue; }
          x = xt;
          if (!kf_rotate(k, c.kb, x, 0.0f - sd_, o.cos_a, c.max_sinphi, &x)) { ok = false; continue; }
        }
        sector = c.m_sector[seg];
      }
      for (; r >= 0; r = rows.next()) {
        if (!kf_propagate(k, c.kb, tx[r] - x, c.max_sinphi)) { ok = false; break; }
        x = tx[r];
        const float2 v = __ldg(yz + hit[r]);
        kf_update(k, v.x, v.y - zref, c.err_y2, c.err_z2);
        ++nfit;
      }
    }
#pragma unroll
    for (int i = 0; i < 5; ++i) o.par[i * mo + m] = k.p[i];
#pragma unroll
    for (int i = 0; i < 15; ++i) o.cov[i * mo + m] = k.c[i];
    o.chi2[m] = k.chi2;
    o.x_ref[m] = started ? x : 0.f;
    o.z_ref[m] = zref;
    o.n_fit[m] = nfit;
    o.ndf[m] = nfit ? 2 * nfit - 5 : 0;
    o.sector[m] = sector;
    o.n_clusters[m] = ncl;
  }
}


// ---------------------------------------------------------------------------------- 3.9.8 apex links (looper following)
// k_apex_prep   thread per merged track: its tail's circle (centre, radius, curvature), end point, dip, z_out; the steep
//               ones are counted into (sector, z_out) bins
// k_apex_fill   counting sort of 16-byte records (z_out, id, tan(lambda), curvature): what the cheap cuts need
// k_apex_match  warp per tail: the sectors the track curls through, the window's run of records read together, exact
//               pre-cuts (z window, curvature signs, the dip term alone above the cut), score, lane-local best, warp reduction
// k_apex_link   mutual best -> partners; secondary-leg label
__global__ void __launch_bounds__(kThreads) k_apex_prep(Ctx c, MergePtrs m, ApexPtrs o) {
  const int nm = c.mcnt->n_merged;
  const float inv_w = c.mcnt->inv_w;
  const size_t mt = (size_t)c.max_tracks;
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < nm; A += gridDim.x * blockDim.x) {
    const int t = m.seg_idx[m.seg_start[A + 1] - 1];
    const float x = c.up_x[t], y = c.up_par[0 * mt + t], s = c.up_par[2 * mt + t], tl = c.up_par[3 * mt + t];
    const float cv = c.kb * c.up_par[4 * mt + t];
    const float zo = c.up_zref[t] + c.up_par[1 * mt + t];
    const int sector = c.m_sector[t];
    const bool steep = c.up_n[t] >= 2 && fabsf(s) >= o.min_s && fabsf(s) < 1.0f && cv != 0.0f;
    float xc = 0.f, yc = 0.f, R = 0.f;
    if (steep) {
      xc = x - s / cv;
      yc = y + sqrtf(1.0f - s * s) / cv;
      R = 1.0f / fabsf(cv);
    }
    c.a_c4[A] = make_float4(xc, yc, R, cv);
    c.a_p4[A] = make_float4(x, y, tl, zo);
    c.a_sector[A] = steep ? (sector | (s >= 0.0f ? 0x100 : 0)) : -1;     // bit 8: curls to +y
    c.a_best[A] = -1; c.a_score[A] = -1.0f;
    o.apex_partner[A] = -1; o.apex_leg[A] = 0;
    int b = -1;
    if (steep && c.m_nzb[sector] > 0) {
      b = merge_bin(c, sector, zo, inv_w);
      atomicAdd(c.m_bin_start + b + 1, 1);
    }
    c.m_bin_of[A] = b;
  }
}

__global__ void __launch_bounds__(kThreads) k_apex_clear(Ctx c) {
  const int nb = c.mcnt->n_bins;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= nb; i += gridDim.x * blockDim.x) {
    c.m_bin_start[i] = 0;
    if (i < nb) c.m_bin_fill[i] = 0;
  }
}

__global__ void __launch_bounds__(kThreads) k_apex_fill(Ctx c) {
  const int nm = c.mcnt->n_merged;
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < nm; A += gridDim.x * blockDim.x) {
    const int b = c.m_bin_of[A];
    if (b < 0) continue;
    const int pos = c.m_bin_start[b] + atomicAdd(c.m_bin_fill + b, 1);
    const float4 p = c.a_p4[A];
    c.m_srec[pos] = make_float4(p.w, __int_as_float(A), p.z, c.a_c4[A].w);
  }
}

__global__ void __launch_bounds__(kThreads) k_apex_match(Ctx c, MergePtrs m, ApexPtrs o) {
  const int nm = c.mcnt->n_merged, n_az = c.S >> 1;
  const float inv_w = c.mcnt->inv_w;
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  const float tz2 = o.tol_z * o.tol_z, tt2 = o.tol_t * o.tol_t;
  for (int A = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; A < nm; A += warps) {
    const int sa = c.a_sector[A];
    if (sa < 0) continue;                                 // warp-uniform
    const int s_a = sa & 0xFF, dirA = (sa & 0x100) ? 1 : -1;
    const float4 cA = c.a_c4[A], pA = c.a_p4[A];          // (xc, yc, R, c), (x, y, t, z_out)
    const float zlo = pA.w - o.dz_win, zhi = pA.w + o.dz_win;
    float best = 0.f;
    int bb = -1;
    float sk = 0.0f, ck = 1.0f;
    for (int k = 0; k <= o.max_k; ++k) {
      if (k > 0) {
        const float s2 = sk * m.cos_a + ck * m.sin_a, c2 = ck * m.cos_a - sk * m.sin_a;
        sk = s2; ck = c2;
      }
      if (k > 0 && n_az < 1) break;
      const int s_b = n_az < 1 ? s_a : (s_a / n_az) * n_az + ((((s_a % n_az) + dirA * k) % n_az) + n_az) % n_az;
      if (k > 0 && s_b == s_a) break;
      if (c.m_nzb[s_b] == 0) continue;
      const float sd = dirA > 0 ? sk : 0.0f - sk;
      // |z_out(B) - z_out(A)| <= dz_win: the bins of [zlo, zhi] hold every such B (monotone clamped floor); the
      // predicate itself is applied below with the written expression
      // (one more bin on either side: zlo / zhi are rounded sums, the predicate below is a rounded difference)
      const int base = c.m_bin_base[s_b];
      const int b0 = max(base, merge_bin(c, s_b, zlo, inv_w) - 1), b1 = min(base + c.m_nzb[s_b] - 1, merge_bin(c, s_b, zhi, inv_w) + 1);
      const int j0 = c.m_bin_start[b0], j1 = c.m_bin_start[b1 + 1];
      for (int j = j0 + lane; j < j1; j += 32) {
        const float4 rec = __ldg(c.m_srec + j);           // (z_out, id, tan(lambda), curvature)
        const int B = __float_as_int(rec.y);
        if (B == A) continue;
        if (!(fabsf(rec.x - pA.w) <= o.dz_win)) continue;
        if (!(cA.w * rec.w < 0.0f)) continue;
        const float dt = pA.z + rec.z;
        const float term_t = (dt * dt) / tt2;
        if (!(term_t <= o.cut)) continue;                 // exact pre-cut: the other two terms are >= 0 and rounding is monotone
        const float4 cB = c.a_c4[B], pB = c.a_p4[B];
        const float xcB = cB.x * ck - cB.y * sd, ycB = cB.x * sd + cB.y * ck;
        const float xB = pB.x * ck - pB.y * sd, yB = pB.x * sd + pB.y * ck;
        const float Rm = 0.5f * (cA.z + cB.z);
        const float dcx = cA.x - xcB, dcy = cA.y - ycB;
        const float dc2 = dcx * dcx + dcy * dcy;
        const float ex = xB - pA.x, ey = yB - pA.y;
        const float d = sqrtf(ex * ex + ey * ey);
        const float h = (0.5f * d) / Rm;
        if (!(h < 0.98f)) continue;
        const float h1 = h / sqrtf(2.0f * (1.0f + sqrtf(1.0f - h * h)));
        const float w = h1 * h1;
        const float ser = 1.0f + w * ((float)(1.0 / 6.0) + w * ((float)(3.0 / 40.0) + w * ((float)(5.0 / 112.0) + w * (float)(35.0 / 1152.0))));
        const float arc = (4.0f * Rm) * (h1 * ser);
        const float dz = rec.x - (pA.w + pA.z * arc);
        const float tc = o.tol_c * Rm;
        const float score = dc2 / (tc * tc) + (dz * dz) / tz2 + term_t;
        if (!(score <= o.cut)) continue;
        if (bb < 0 || score < best || (score == best && B < bb)) { best = score; bb = B; }
      }
    }
    __syncwarp();
#pragma unroll
    for (int off = 16; off; off >>= 1) {
      const float os = __shfl_xor_sync(0xffffffffu, best, off);
      const int ob = __shfl_xor_sync(0xffffffffu, bb, off);
      if (ob >= 0 && (bb < 0 || os < best || (os == best && ob < bb))) { best = os; bb = ob; }
    }
    if (lane == 0) { c.a_best[A] = bb; c.a_score[A] = bb >= 0 ? best : -1.0f; }
  }
}

__global__ void __launch_bounds__(kThreads) k_apex_link(Ctx c, ApexPtrs o) {
  const int nm = c.mcnt->n_merged, n_az = c.S >> 1;
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < nm; A += gridDim.x * blockDim.x) {
    const int B = c.a_best[A];
    if (B < 0 || c.a_best[B] != A) continue;
    o.apex_partner[A] = B;
    const float zA = c.a_p4[A].w, zB = c.a_p4[B].w;
    const bool a_side = (c.a_sector[A] & 0xFF) < n_az;
    const bool later = a_side ? zA > zB : zA < zB;
    o.apex_leg[A] = (later || (zA == zB && A > B)) ? 1 : 0;
  }
}

unsigned grid_for(long long n, const Ctx& c, int per_sm) {
  long long g = (n + kThreads - 1) / kThreads;
  const long long cap = (long long)c.n_sms * per_sm;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (unsigned)g;
}

}  // namespace

int launches_merge() { return 12 + 6; }
int launch_merge(const Ctx& c, const FitPtrs& f, const MergePtrs& o, cudaStream_t st) {
  const unsigned gt = grid_for(c.max_tracks, c, 64), gb = grid_for(c.max_merge_bins, c, 16);
  const size_t sh = c.R * sizeof(float);
  k_merge_tables<<<1, 32, 0, st>>>(c, o.dz_win * 0.25f, 1);
  k_merge_clear<<<gt > gb ? gt : gb, kThreads, 0, st>>>(c, o);
  k_refit_up<<<gt, kThreads, sh, st>>>(c, f, o);
  // CSR starts of the (sector, z) bins: inclusive scan of the counts written at b + 1 (entry 0 stays 0)
  if (launch_scan_inclusive(c.m_bin_start, &c.mcnt->n_bins, 1, (long long)c.max_merge_bins + 1, c.tile_sums, nullptr, c.n_sms, st)) return -1;
  k_merge_zero_fill<<<gb, kThreads, 0, st>>>(c);
  k_merge_fill<<<gt, kThreads, 0, st>>>(c, o);
  k_merge_match<<<grid_for((long long)c.max_tracks * 32, c, 64), kThreads, sh, st>>>(c, f, o);
  k_merge_link<<<gt, kThreads, 0, st>>>(c, o);
  k_merge_heads<<<gt, kThreads, 0, st>>>(c, o);
  if (launch_scan_inclusive(c.m_head_scan, &c.mcnt->n_scan, 0, c.max_tracks, c.tile_sums, nullptr, c.n_sms, st)) return -1;
  k_chain_len<<<gt, kThreads, 0, st>>>(c, o);
  if (launch_scan_inclusive(c.m_seg_scan, &c.mcnt->n_merged, 0, c.max_tracks, c.tile_sums, nullptr, c.n_sms, st)) return -1;
  k_chain_fill<<<gt, kThreads, 0, st>>>(c, o);
  k_refit_merged<<<gt, kThreads, sh, st>>>(c, o);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launches_apex() { return 6 + 3; }
int launch_apex(const Ctx& c, const MergePtrs& m, const ApexPtrs& o, cudaStream_t st) {
  const unsigned gt = grid_for(c.max_tracks, c, 64), gb = grid_for(c.max_merge_bins, c, 16);
  k_merge_tables<<<1, 32, 0, st>>>(c, o.dz_win * 0.25f, 0);   // n_merged of the merge call stays
  k_apex_clear<<<gb, kThreads, 0, st>>>(c);
  k_apex_prep<<<gt, kThreads, 0, st>>>(c, m, o);
  if (launch_scan_inclusive(c.m_bin_start, &c.mcnt->n_bins, 1, (long long)c.max_merge_bins + 1, c.tile_sums, nullptr, c.n_sms, st)) return -1;
  k_apex_fill<<<gt, kThreads, 0, st>>>(c);
  k_apex_match<<<grid_for((long long)c.max_tracks * 32, c, 64), kThreads, 0, st>>>(c, m, o);
  k_apex_link<<<gt, kThreads, 0, st>>>(c, o);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
