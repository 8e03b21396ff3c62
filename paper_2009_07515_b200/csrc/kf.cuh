// The 5-parameter Kalman filter pieces shared by S4 (tracklet constructor) and S7 (refit): state
// (y, z - z_ref, sin(phi), tan(lambda), q/pT) at a pad-row plane, full symmetric 5x5 covariance as 15 registers.
// DESIGN.md sections 3.4.1 (helix step + transport) and 3.4.2 (update), operation by operation; fused multiply-adds
// exactly where the text writes fma().  Nothing here is shared with oracle/.
#pragma once
#include "tpc_internal.cuh"

namespace tpc {

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
  const float s1 = __fmaf_rn(cv, dx, s);
  if (!(fabsf(s) < max_sinphi) || !(fabsf(s1) < max_sinphi)) return false;
  const float c0 = sqrtf(__fmaf_rn(-s, s, 1.0f));
  const float c1 = sqrtf(__fmaf_rn(-s1, s1, 1.0f));
  const float cc = c0 + c1;
  const float ss = s + s1;
  const float Tn = ss / cc;
  const float y1 = __fmaf_rn(dx, Tn, y);
  const float dl = dx * sqrtf(__fmaf_rn(Tn, Tn, 1.0f));
  const float u = (0.5f * cv) * dl;
  const float w = u * u;
  const float ser = __fmaf_rn(w, __fmaf_rn(w, __fmaf_rn(w, __fmaf_rn(w, (float)(35.0 / 1152.0), (float)(5.0 / 112.0)), (float)(3.0 / 40.0)), (float)(1.0 / 6.0)), 1.0f);
  const float arc = dl * ser;
  const float z1 = __fmaf_rn(t, arc, z);

  const float c0c1 = c0 * c1;
  const float kdx = kb * dx;
  const float j02 = dx * __fmaf_rn(s, Tn, c0) / c0c1;
  const float j04 = (kdx * dx) * __fmaf_rn(s1, ss, c1 * cc) / (c1 * (cc * cc));
  const float j24 = kdx;
  const float j13 = arc;
  const float j12 = (t * dx) * Tn / c0c1;
  const float sm = __fmaf_rn(0.5f * cv, dx, s);
  const float cm = sqrtf(__fmaf_rn(-sm, sm, 1.0f));
  const float j14 = ((t * kdx) * dx) * (float)(1.0 / 6.0) * (2.0f * sm / (cm * cm * cm) + s1 / (c1 * c1 * c1));

  // M = J C (rows 3 and 4 of J are unit rows), then C1 = M J^T, lower triangle
  float m0[5], m1[5], m2[5];
#pragma unroll
  for (int l = 0; l < 5; ++l) {
    m0[l] = __fmaf_rn(j04, k.c[CI(4, l)], __fmaf_rn(j02, k.c[CI(2, l)], k.c[CI(0, l)]));
    m1[l] = __fmaf_rn(j14, k.c[CI(4, l)], __fmaf_rn(j13, k.c[CI(3, l)], __fmaf_rn(j12, k.c[CI(2, l)], k.c[CI(1, l)])));
    m2[l] = __fmaf_rn(j24, k.c[CI(4, l)], k.c[CI(2, l)]);
  }
  float n[15];
  n[CI(0, 0)] = __fmaf_rn(m0[4], j04, __fmaf_rn(m0[2], j02, m0[0]));
  n[CI(1, 0)] = __fmaf_rn(m1[4], j04, __fmaf_rn(m1[2], j02, m1[0]));
  n[CI(2, 0)] = __fmaf_rn(m2[4], j04, __fmaf_rn(m2[2], j02, m2[0]));
  n[CI(3, 0)] = __fmaf_rn(k.c[CI(3, 4)], j04, __fmaf_rn(k.c[CI(3, 2)], j02, k.c[CI(3, 0)]));
  n[CI(4, 0)] = __fmaf_rn(k.c[CI(4, 4)], j04, __fmaf_rn(k.c[CI(4, 2)], j02, k.c[CI(4, 0)]));
  n[CI(1, 1)] = __fmaf_rn(m1[4], j14, __fmaf_rn(m1[3], j13, __fmaf_rn(m1[2], j12, m1[1])));
  n[CI(2, 1)] = __fmaf_rn(m2[4], j14, __fmaf_rn(m2[3], j13, __fmaf_rn(m2[2], j12, m2[1])));
  n[CI(3, 1)] = __fmaf_rn(k.c[CI(3, 4)], j14, __fmaf_rn(k.c[CI(3, 3)], j13, __fmaf_rn(k.c[CI(3, 2)], j12, k.c[CI(3, 1)])));
  n[CI(4, 1)] = __fmaf_rn(k.c[CI(4, 4)], j14, __fmaf_rn(k.c[CI(4, 3)], j13, __fmaf_rn(k.c[CI(4, 2)], j12, k.c[CI(4, 1)])));
  n[CI(2, 2)] = __fmaf_rn(m2[4], j24, m2[2]);
  n[CI(3, 2)] = __fmaf_rn(k.c[CI(3, 4)], j24, k.c[CI(3, 2)]);
  n[CI(4, 2)] = __fmaf_rn(k.c[CI(4, 4)], j24, k.c[CI(4, 2)]);
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
  const float det = __fmaf_rn(S00, S11, -(S10 * S10));
  const float idet = 1.0f / det;
  const float I00 = S11 * idet, I10 = (0.0f - S10) * idet, I11 = S00 * idet;
  k.chi2 = k.chi2 + __fmaf_rn(r1 * r1, I11, __fmaf_rn(2.0f * (r0 * r1), I10, (r0 * r0) * I00));
  float K0[5], K1[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    K0[i] = __fmaf_rn(k.c[CI(i, 1)], I10, k.c[CI(i, 0)] * I00);
    K1[i] = __fmaf_rn(k.c[CI(i, 1)], I11, k.c[CI(i, 0)] * I10);
  }
  float n[15];
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 0; j <= i; ++j) n[CI(i, j)] = __fmaf_rn(-K1[i], k.c[CI(1, j)], __fmaf_rn(-K0[i], k.c[CI(0, j)], k.c[CI(i, j)]));
#pragma unroll
  for (int i = 0; i < 5; ++i) k.p[i] = __fmaf_rn(K1[i], r1, __fmaf_rn(K0[i], r0, k.p[i]));
#pragma unroll
  for (int i = 0; i < 15; ++i) k.c[i] = n[i];
}

}  // namespace tpc
