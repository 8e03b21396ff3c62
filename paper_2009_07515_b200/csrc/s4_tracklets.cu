// S4 - tracklet constructor (BASELINE.json north_star (4)): per seed, follow the chain
// upward with Kalman updates (phase A), extrapolate further up picking up gated nearest clusters
// (phase B), turn round with a reset covariance and refit downward with pick-up (phase C).
// 5-parameter filter (y, z - z_ref, sin(phi), tan(lambda), q/pT) in the sector-local frame, exact
// circle propagation in a uniform Bz, full 5x5 symmetric covariance (15 unique entries) in
// registers, textbook update.
//
// Persistent kernel: one thread per tracklet, warps fetch 32 consecutive seeds from a global
// ticket counter (one atomic per warp), so SMs stay busy whatever the chain-length mix.  The hit
// table [seed][row] of a warp's 32 seeds is one contiguous 32*R*4-byte block and is cleared
// cooperatively with coalesced stores.
//
// Arithmetic is written operation by operation in the order of DESIGN.md section 3.4 (compiled with
// -fmad=false): the transport J C J^T skips only the terms that are structurally 0*x or 1*x.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int kThreads = 128;

// symmetric 5x5, lower triangle row-major: index(i,j) = i*(i+1)/2 + j for i >= j
#define CI(i, j) ((i) >= (j) ? ((i) * ((i) + 1) / 2 + (j)) : ((j) * ((j) + 1) / 2 + (i)))

struct KF {
  float p[5];
  float c[15];
  float chi2;
};

__device__ __forceinline__ void kf_reset_cov(KF& k, const Ctx& c) {
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = 0.0f;
  k.c[CI(0, 0)] = c.err_y2; k.c[CI(1, 1)] = c.err_z2;
  k.c[CI(2, 2)] = c.init_c_ss; k.c[CI(3, 3)] = c.init_c_tt; k.c[CI(4, 4)] = c.init_c_qq;
  k.chi2 = 0.0f;
}

// DESIGN.md section 3.4.1
__device__ __forceinline__ bool kf_propagate(KF& k, float kb, float dx, float max_sinphi) {
  const float y = k.p[0], z = k.p[1], s = k.p[2], t = k.p[3], q = k.p[4];
  const float cv = kb * q;
  const float s1 = s + cv * dx;
  if (!(fabsf(s) < max_sinphi) || !(fabsf(s1) < max_sinphi)) return false;
  const float c0 = sqrtf(1.0f - s * s);
  const float c1 = sqrtf(1.0f - s1 * s1);
  const float cc = c0 + c1;
  const float ss = s + s1;
  const float Tn = ss / cc;
  const float y1 = y + dx * Tn;
  const float dl = dx * sqrtf(1.0f + Tn * Tn);
  const float u = (0.5f * cv) * dl;
  const float w = u * u;
  const float ser = 1.0f + w * ((float)(1.0 / 6.0) + w * ((float)(3.0 / 40.0) + w * ((float)(5.0 / 112.0) + w * (float)(35.0 / 1152.0))));
  const float arc = dl * ser;
  const float z1 = z + t * arc;

  const float c0c1 = c0 * c1;
  const float kdx = kb * dx;
  const float j02 = dx * (c0 + s * Tn) / c0c1;
  const float j04 = (kdx * dx) * (c1 * cc + s1 * ss) / (c1 * (cc * cc));
  const float j24 = kdx;
  const float j13 = arc;
  const float j12 = (t * dx) * Tn / c0c1;
  const float sm = s + (0.5f * cv) * dx;
  const float cm = sqrtf(1.0f - sm * sm);
  const float j14 = ((t * kdx) * dx) * (float)(1.0 / 6.0) * (2.0f * sm / (cm * cm * cm) + s1 / (c1 * c1 * c1));

  // M = J C (rows 3 and 4 of J are unit rows), then C1 = M J^T, lower triangle
  float m0[5], m1[5], m2[5];
#pragma unroll
  for (int l = 0; l < 5; ++l) {
    m0[l] = (k.c[CI(0, l)] + j02 * k.c[CI(2, l)]) + j04 * k.c[CI(4, l)];
    m1[l] = ((k.c[CI(1, l)] + j12 * k.c[CI(2, l)]) + j13 * k.c[CI(3, l)]) + j14 * k.c[CI(4, l)];
    m2[l] = k.c[CI(2, l)] + j24 * k.c[CI(4, l)];
  }
  float n[15];
  n[CI(0, 0)] = (m0[0] + m0[2] * j02) + m0[4] * j04;
  n[CI(1, 0)] = (m1[0] + m1[2] * j02) + m1[4] * j04;
  n[CI(2, 0)] = (m2[0] + m2[2] * j02) + m2[4] * j04;
  n[CI(3, 0)] = (k.c[CI(3, 0)] + k.c[CI(3, 2)] * j02) + k.c[CI(3, 4)] * j04;
  n[CI(4, 0)] = (k.c[CI(4, 0)] + k.c[CI(4, 2)] * j02) + k.c[CI(4, 4)] * j04;
  n[CI(1, 1)] = ((m1[1] + m1[2] * j12) + m1[3] * j13) + m1[4] * j14;
  n[CI(2, 1)] = ((m2[1] + m2[2] * j12) + m2[3] * j13) + m2[4] * j14;
  n[CI(3, 1)] = ((k.c[CI(3, 1)] + k.c[CI(3, 2)] * j12) + k.c[CI(3, 3)] * j13) + k.c[CI(3, 4)] * j14;
  n[CI(4, 1)] = ((k.c[CI(4, 1)] + k.c[CI(4, 2)] * j12) + k.c[CI(4, 3)] * j13) + k.c[CI(4, 4)] * j14;
  n[CI(2, 2)] = m2[2] + m2[4] * j24;
  n[CI(3, 2)] = k.c[CI(3, 2)] + k.c[CI(3, 4)] * j24;
  n[CI(4, 2)] = k.c[CI(4, 2)] + k.c[CI(4, 4)] * j24;
  n[CI(3, 3)] = k.c[CI(3, 3)];
  n[CI(4, 3)] = k.c[CI(4, 3)];
  n[CI(4, 4)] = k.c[CI(4, 4)];
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = n[i];
  k.p[0] = y1; k.p[1] = z1; k.p[2] = s1;
  return true;
}

// DESIGN.md section 3.4.2
__device__ __forceinline__ void kf_update(KF& k, float ym, float zm, float err_y2, float err_z2) {
  const float r0 = ym - k.p[0];
  const float r1 = zm - k.p[1];
  const float S00 = k.c[CI(0, 0)] + err_y2;
  const float S10 = k.c[CI(1, 0)];
  const float S11 = k.c[CI(1, 1)] + err_z2;
  const float det = S00 * S11 - S10 * S10;
  const float idet = 1.0f / det;
  const float I00 = S11 * idet, I10 = (0.0f - S10) * idet, I11 = S00 * idet;
  k.chi2 = k.chi2 + ((r0 * r0) * I00 + (2.0f * (r0 * r1)) * I10 + (r1 * r1) * I11);
  float K0[5], K1[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    K0[i] = k.c[CI(i, 0)] * I00 + k.c[CI(i, 1)] * I10;
    K1[i] = k.c[CI(i, 0)] * I10 + k.c[CI(i, 1)] * I11;
  }
  float n[15];
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 0; j <= i; ++j) n[CI(i, j)] = k.c[CI(i, j)] - (K0[i] * k.c[CI(0, j)] + K1[i] * k.c[CI(1, j)]);
#pragma unroll
  for (int i = 0; i < 5; ++i) k.p[i] = k.p[i] + (K0[i] * r0 + K1[i] * r1);
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = n[i];
}

struct Grid {
  const int* __restrict__ bin_start;
  const float* __restrict__ ys;
  const float* __restrict__ zs;
  const int* __restrict__ bin_base_s;   // bin_base + s*R
  int nz;
  float zmin;
};

// nearest gated cluster of row r, or -1
__device__ __forceinline__ int kf_search(const Ctx& c, const RowTab* tab, const Grid& G, int r, const KF& k, float zref,
                                         float* ym, float* zm) {
  const float cut = c.pick_chi2_cut;
  const float sy2 = k.c[CI(0, 0)] + c.err_y2, sz2 = k.c[CI(1, 1)] + c.err_z2;
  const float hy = sqrtf(cut * sy2), hz = sqrtf(cut * sz2);
  const float zabs = zref + k.p[1];
  const float ylo = k.p[0] - hy, yhi = k.p[0] + hy, zlo = zabs - hz, zhi = zabs + hz;
  const float wy = 1.0f / sy2, wz = 1.0f / sz2;
  float best = INFINITY;
  int arg = -1;
  RowGrid g;
  g.b0 = __ldg(G.bin_base_s + r); g.ny = tab[r].ny; g.nz = G.nz; g.ymax = tab[r].ymax; g.zmin = G.zmin;
  for_each_in_rect(g, c.inv_cy, c.inv_cz, G.bin_start, G.ys, G.zs, ylo, yhi, zlo, zhi, [&](int j, float yj, float zj) {
    const float dy = yj - k.p[0];
    const float dz = (zj - zref) - k.p[1];
    const float d2 = (dy * dy) * wy + (dz * dz) * wz;
    if (d2 <= cut && d2 < best) { best = d2; arg = j; *ym = yj; *zm = zj; }
  });
  return arg;
}

__global__ void __launch_bounds__(kThreads) k_tracklets(Ctx c) {
  extern __shared__ RowTab tab[];
  for (int i = threadIdx.x; i < c.R * (int)(sizeof(RowTab) / 4); i += blockDim.x)
    reinterpret_cast<int*>(tab)[i] = __ldg(reinterpret_cast<const int*>(c.rowtab) + i);
  __syncthreads();
  if (c.cnt->status) return;
  const int n_seeds = c.cnt->n_seeds;
  const int R = c.R;
  const int lane = threadIdx.x & 31;
  const float* __restrict__ ys = c.ys;
  const float* __restrict__ zs = c.zs;
  const int* __restrict__ link_up = c.link_up;
  unsigned long long steps = 0, hits_kept = 0;
  int kept_cnt = 0;

  for (;;) {
    int base = 0;
    if (lane == 0) base = atomicAdd(&c.cnt->s4_ticket, 32);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base >= n_seeds) break;
    const int cnt = min(32, n_seeds - base);
    {   // clear the warp's hit tables (contiguous cnt*R ints)
      int* h0 = c.t_hit + (size_t)base * R;
      for (int i = lane; i < cnt * R; i += 32) h0[i] = -1;
    }
    __syncwarp();
    const int sd = base + lane;
    if (sd < n_seeds) {
      int* __restrict__ hit = c.t_hit + (size_t)sd * R;
      const int h = __ldg(c.seed_head + sd), nx = __ldg(link_up + h);
      const int srh = c.srow[h];
      const int s = srh / R, r0 = srh - s * R;
      const int r1 = (int)c.srow[nx] - s * R;
      Grid G;
      G.bin_start = c.bins; G.ys = ys; G.zs = zs; G.bin_base_s = c.bin_base + s * R;
      G.nz = __ldg(c.nz + s); G.zmin = __ldg(c.zmin + s);
      const float zref = __ldg(zs + h);
      const float ey2 = c.err_y2, ez2 = c.err_z2, kb = c.kb, msp = c.max_sinphi;

      KF k;
      {
        const float dx = tab[r1].x - tab[r0].x;
        const float dy = __ldg(ys + nx) - __ldg(ys + h);
        const float dz = __ldg(zs + nx) - zref;
        const float dl = sqrtf(dx * dx + dy * dy);
        k.p[0] = __ldg(ys + h); k.p[1] = 0.0f; k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = 0.0f;
        kf_reset_cov(k, c);
      }
      hit[r0] = h;
      int cur = r0;
      float lp[5];
#pragma unroll
      for (int i = 0; i < 5; ++i) lp[i] = k.p[i];
      int last_row = r0;

      // Phase A
      bool up_ok = true;
      for (int cl = nx; cl >= 0; cl = __ldg(link_up + cl)) {
        const int rc = (int)c.srow[cl] - s * R;
        ++steps;
        if (!kf_propagate(k, kb, tab[rc].x - tab[cur].x, msp)) { up_ok = false; break; }
        cur = rc;
        kf_update(k, __ldg(ys + cl), __ldg(zs + cl) - zref, ey2, ez2);
        hit[rc] = cl;
#pragma unroll
        for (int i = 0; i < 5; ++i) lp[i] = k.p[i];
        last_row = rc;
      }
      // Phase B
      if (up_ok) {
        int gap = 0;
        for (int r = cur + 1; r < R; ++r) {
          ++steps;
          if (!kf_propagate(k, kb, tab[r].x - tab[cur].x, msp)) break;
          cur = r;
          if (!(fabsf(k.p[0]) <= tab[r].ymax + c.y_margin)) break;
          float ym, zm;
          const int cl = kf_search(c, tab, G, r, k, zref, &ym, &zm);
          if (cl >= 0) {
            kf_update(k, ym, zm - zref, ey2, ez2);
            hit[r] = cl; gap = 0;
#pragma unroll
            for (int i = 0; i < 5; ++i) lp[i] = k.p[i];
            last_row = r;
          } else if (++gap > c.max_gap) break;
        }
      }
      // Phase C
#pragma unroll
      for (int i = 0; i < 5; ++i) k.p[i] = lp[i];
      cur = last_row;
      kf_reset_cov(k, c);
      KF out = k;
      int low = last_row;
      {
        int gap = 0;
        for (int r = cur - 1; r >= 0; --r) {
          ++steps;
          if (!kf_propagate(k, kb, tab[r].x - tab[cur].x, msp)) break;
          cur = r;
          if (!(fabsf(k.p[0]) <= tab[r].ymax + c.y_margin)) break;
          int cl = hit[r];
          float ym, zm;
          if (cl >= 0) { ym = __ldg(ys + cl); zm = __ldg(zs + cl); }
          else cl = kf_search(c, tab, G, r, k, zref, &ym, &zm);
          if (cl >= 0) {
            kf_update(k, ym, zm - zref, ey2, ez2);
            hit[r] = cl; gap = 0;
            out = k; low = r;
          } else if (++gap > c.max_gap) break;
        }
      }
      int nh = 0;
      for (int r = 0; r < R; ++r) {
        if (r < low) hit[r] = -1;
        else nh += hit[r] >= 0;
      }
      c.t_first_row[sd] = low; c.t_last_row[sd] = last_row; c.t_n_hits[sd] = nh;
#pragma unroll
      for (int i = 0; i < 5; ++i) c.t_par[(size_t)sd * 5 + i] = out.p[i];
#pragma unroll
      for (int i = 0; i < 15; ++i) c.t_cov[(size_t)sd * 15 + i] = out.c[i];
      c.t_chi2[sd] = out.chi2; c.t_zref[sd] = zref;
      if (nh >= c.min_tracklet_hits) { hits_kept += nh; ++kept_cnt; }
    }
    __syncwarp();
  }
  for (int o = 16; o; o >>= 1) {
    steps += __shfl_xor_sync(0xffffffffu, steps, o);
    hits_kept += __shfl_xor_sync(0xffffffffu, hits_kept, o);
  }
  if (lane == 0) {
    if (steps) atomicAdd(&c.cnt->kf_steps, steps);
    if (hits_kept) atomicAdd(&c.cnt->n_hits, hits_kept);
  }
  (void)kept_cnt;
}

}  // namespace

int launches_s4() { return 1; }
int launch_s4(const Ctx& c, cudaStream_t st) {
  // persistent: enough CTAs to fill every SM; each warp pulls work until the ticket runs out
  const int per_sm = 4;
  k_tracklets<<<c.n_sms * per_sm, kThreads, c.R * sizeof(RowTab), st>>>(c);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace tpc
