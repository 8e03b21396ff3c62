// =============================================================================================
// TEST INFRASTRUCTURE - NOT PART OF THE PRODUCT.
//
// Plain, slow, single-threaded CPU oracle for the TPC sector track finder ("Track Finding",
// PAPER.md:137 Table 1; section 6).  The paper names the step but defers the algorithm
// to references that are not available; the five steps come from BASELINE.json `north_star`
// (sort+bin, neighbours finder, link cleaner, Kalman tracklet constructor, selector) and every
// formula below is the reading fixed in DESIGN.md section 3 ("The method, step by step").  This file
// follows that text in its order and notation; DESIGN.md is the authority when the two differ.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this.  It shares no code, header, table or constant generator with
// paper_2009_07515_b200/csrc (the CUDA product) and neither includes the other.
//
// Arithmetic contract: fp32, round-to-nearest-even, one rounding per written
// operation, evaluation order exactly as written, no FMA contraction by the compiler (build with
// -ffp-contract=off, no -ffast-math), only + - * / sqrt floor fabs and - in the Kalman transport and update of
// stage 4 only - the fused multiply-add std::fma exactly where DESIGN.md sections 3.4.1 / 3.4.2 write fma().  Stage 4 is templated on the
// scalar: the float instance is the parity reference, the double instance exists for the
// analytic pins (tests/test_oracle_*.py) and to measure the fp32 error.
//
// Pins (tests/, -m "not gpu"): S1 vs numpy lexsort + independent bin recomputation; S2 vs
// brute-force all-pairs search; S3 invariants + brute-force chain walk; helix step vs closed-form
// circle, Jacobian vs finite differences; KF vs closed-form weighted line fit at Bz=0 and vs
// generator truth (q/pT 1e-4 rel.) on noise-free helices, pulls on smeared input; S5 vs
// brute-force ownership; the S4 phase logic (chain, pick-up across holes, gap rule, downward pass) vs
// generator truth on isolated noise-free helices with rows removed (tests/test_oracle_phases.py);
// the field constant vs the textbook radius of curvature (tests/golden/helix_radius.txt); the two CHOICES among
// several candidates - the S4 search (gate, strict minimum, tie -> lowest position, window, weights) and the S2 pair
// choice and link cut - on hand-built dyadic constructions whose answers are known by hand, plus a whole-row scan
// (tests/test_oracle_choice_pins.py; each case lists the mutations it kills); the native time input, the track merger
// (rotation, upward and merged refit, candidates / score / mutual choice / chains) and the apex links of loopers in
// tests/test_oracle_time_input.py, test_oracle_merge.py, test_oracle_apex.py (DESIGN.md section 9 lists the pins and the
// twenty mutations they kill).  Nothing is left "parity unpinned".
// =============================================================================================
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <map>
#include <numeric>
#include <string>
#include <vector>

namespace {

constexpr int kMaxRows = 256;

struct Params {             // mirrors the ctypes Structure in oracle/oracle.py (not the product header)
  int32_t n_sectors, n_rows;
  float row_x[kMaxRows];
  float tan_half_sector, bz_tesla, err_y2, err_z2, cell_y, cell_z;
  float link_ay, link_az, link_b, link_T;
  int32_t min_chain_len, max_gap, min_tracklet_hits, min_track_hits;
  float pick_chi2_cut, max_sinphi, y_margin, init_c_ss, init_c_tt, init_c_qq;
  int32_t z_is_time; float cm_per_time_unit, drift_length;   // native time input, DESIGN.md section 3.0a
  int32_t y_is_pad;                                          // native pad input, DESIGN.md section 3.0b
  int32_t n_pads[kMaxRows];                                  //   pads of row r
  float pad_pitch[kMaxRows];                                 //   pad width of row r, cm
};

// DESIGN.md section 3.7a ("tailored custom fixed ... point data formats using only exactly as many bits as
// needed", "stored as residuals to the extrapolated track position"): a residual as a signed 16-bit count
// of steps.  fp32: one product with the reciprocal step, round to nearest with ties to even, saturation at +-32767
// (-32768 is never produced; a NaN - no residual is one - counts as below the range).
inline int32_t quantise_residual(float res, float inv_step) {
  const float v = res * inv_step;
  const float r = std::nearbyint(v);                    // default rounding mode: to nearest, ties to even
  if (!(r > -32767.0f)) return -32767;
  if (r >= 32767.0f) return 32767;
  return (int32_t)r;
}

// floor(v) clamped to [0, hi]; defined for every v (NaN and negatives -> 0), DESIGN.md section 3.1 (3)
inline int floor_clamp(float v, int hi) {
  const float f = std::floor(v);
  if (!(f >= 0.0f)) return 0;
  if (f >= (float)hi) return hi;
  return (int)f;
}

// ------------------------------------------------------------------------------------------
// Kalman filter pieces.  State p = (y, z_rel, s=sin(phi), t=tan(lambda), q=q/pT) at a
// pad-row plane x; C is the full symmetric 5x5 (lower triangle computed, upper mirrored).
// ------------------------------------------------------------------------------------------
template <class T>
struct KF {
  T p[5];
  T C[5][5];
  T chi2;
};

// Beam-line z of a track ("Track seeds are extrapolated to the beam line and the most
// likely z coordinate is computed under the assumption that the track is a primary and the vertex is at the origin").
// A primary's circle passes through the origin of the xy plane: the chord d from the origin to (x, y) subtends the
// turning angle theta with sin(theta/2) = |c| d / 2, the path length is d * asin(a)/a with a = |c| d / 2, and
// z_beam = z - tan(lambda) * path.  asin(a)/a without libm: two half-angle reductions sin(t/2) = sin t / sqrt(2 (1 +
// cos t)), then the 5-term series of section 3.4.1.
template <class T>
T beam_z(T kb, T x, T y, T z, T t, T q) {
  const T c = kb * q;
  const T d = std::sqrt(x * x + y * y);
  T a = std::fabs((T(0.5) * c) * d);
  if (!(a < T(1))) a = T(1);
  const T c1 = std::sqrt(T(1) - a * a);
  const T a1 = a / std::sqrt(T(2) * (T(1) + c1));
  const T c2 = std::sqrt(T(1) - a1 * a1);
  const T a2 = a1 / std::sqrt(T(2) * (T(1) + c2));
  const T w = a2 * a2;
  const T ser = T(1) + w * (T(1.0 / 6.0) + w * (T(3.0 / 40.0) + w * (T(5.0 / 112.0) + w * T(35.0 / 1152.0))));
  const T ratio = a > T(0) ? (T(4) * (a2 * ser)) / a : T(1);
  const T path = d * ratio;
  return z - t * path;
}

// Helix step x -> x+dx in a uniform Bz (exact circle in xy), DESIGN.md section 3.4.1.
// Returns false and leaves (p, C) untouched if |s| or |s1| >= max_sinphi.
template <class T>
bool kf_propagate(KF<T>& k, T kb, T dx, T max_sinphi, T* jac_out /*25, row-major, may be null*/) {
  const T y = k.p[0], z = k.p[1], s = k.p[2], t = k.p[3], q = k.p[4];
  const T c = kb * q;                                   // curvature
  const T s1 = std::fma(c, dx, s);
  if (!(std::fabs(s) < max_sinphi) || !(std::fabs(s1) < max_sinphi)) return false;
  const T c0 = std::sqrt(std::fma(-s, s, T(1)));
  const T c1 = std::sqrt(std::fma(-s1, s1, T(1)));
  const T cc = c0 + c1;
  const T ss = s + s1;
  const T Tn = ss / cc;                                 // tan of the chord direction
  const T y1 = std::fma(dx, Tn, y);
  const T dl = dx * std::sqrt(std::fma(Tn, Tn, T(1)));  // signed chord length
  const T u = (T(0.5) * c) * dl;
  const T w = u * u;
  // asin(u)/u = 1 + w/6 + 3w^2/40 + 5w^3/112 + 35w^4/1152 + ...   (no libm transcendental)
  const T ser = std::fma(w, std::fma(w, std::fma(w, std::fma(w, T(35.0 / 1152.0), T(5.0 / 112.0)), T(3.0 / 40.0)), T(1.0 / 6.0)), T(1));
  const T arc = dl * ser;                               // signed xy arc length
  const T z1 = std::fma(t, arc, z);

  // Jacobian d(p1)/d(p0); identity except the six entries below.
  const T c0c1 = c0 * c1;
  const T kdx = kb * dx;
  const T j_ys = dx * std::fma(s, Tn, c0) / c0c1;
  const T j_yq = (kdx * dx) * std::fma(s1, ss, c1 * cc) / (c1 * (cc * cc));
  const T j_sq = kdx;
  const T j_zt = arc;
  const T j_zs = (t * dx) * Tn / c0c1;
  const T sm = std::fma(T(0.5) * c, dx, s);             // sin(phi) at the step midpoint (Simpson)
  const T cm = std::sqrt(std::fma(-sm, sm, T(1)));
  const T j_zq = ((t * kdx) * dx) * T(1.0 / 6.0) * (T(2) * sm / (cm * cm * cm) + s1 / (c1 * c1 * c1));

  T J[5][5];
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) J[i][j] = (i == j) ? T(1) : T(0);
  J[0][2] = j_ys; J[0][4] = j_yq; J[1][2] = j_zs; J[1][3] = j_zt; J[1][4] = j_zq; J[2][4] = j_sq;

  // C1 = J C J^T: M = J C (k ascending), C1[i][j] = sum_l M[i][l] J[j][l] (l ascending) for i >= j, mirrored; every
  // term enters its sum by one fused multiply-add.
  T M[5][5];
  for (int i = 0; i < 5; ++i)
    for (int l = 0; l < 5; ++l) {
      T acc = T(0);
      for (int kk = 0; kk < 5; ++kk) acc = std::fma(J[i][kk], k.C[kk][l], acc);
      M[i][l] = acc;
    }
  T C1[5][5];
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) {
      T acc = T(0);
      for (int l = 0; l < 5; ++l) acc = std::fma(M[i][l], J[j][l], acc);
      C1[i][j] = acc;
      C1[j][i] = acc;
    }
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) k.C[i][j] = C1[i][j];
  k.p[0] = y1; k.p[1] = z1; k.p[2] = s1;                // t, q unchanged
  if (jac_out)
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < 5; ++j) jac_out[i * 5 + j] = J[i][j];
  return true;
}

// Textbook Kalman update with the measurement m = (y_m, z_m - z_ref), V = diag(err_y2, err_z2), H = [I2 0]
// (DESIGN.md section 3.4.2).  No gate here.
template <class T>
void kf_update(KF<T>& k, T ym, T zm, T err_y2, T err_z2) {
  const T r0 = ym - k.p[0];
  const T r1 = zm - k.p[1];
  const T S00 = k.C[0][0] + err_y2;
  const T S10 = k.C[1][0];
  const T S11 = k.C[1][1] + err_z2;
  const T det = std::fma(S00, S11, -(S10 * S10));
  const T idet = T(1) / det;
  const T I00 = S11 * idet, I10 = (T(0) - S10) * idet, I11 = S00 * idet;   // S^-1 (symmetric)
  k.chi2 = k.chi2 + std::fma(r1 * r1, I11, std::fma(T(2) * (r0 * r1), I10, (r0 * r0) * I00));
  T K0[5], K1[5];                                       // gain K = C H^T S^-1   (5x2)
  for (int i = 0; i < 5; ++i) {
    K0[i] = std::fma(k.C[i][1], I10, k.C[i][0] * I00);
    K1[i] = std::fma(k.C[i][1], I11, k.C[i][0] * I10);
  }
  T C1[5][5];
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) {                      // C -= K (H C), lower triangle then mirror
      const T v = std::fma(-K1[i], k.C[1][j], std::fma(-K0[i], k.C[0][j], k.C[i][j]));
      C1[i][j] = v;
      C1[j][i] = v;
    }
  for (int i = 0; i < 5; ++i) k.p[i] = std::fma(K1[i], r1, std::fma(K0[i], r0, k.p[i]));
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) k.C[i][j] = C1[i][j];
}

template <class T>
void kf_reset_cov(KF<T>& k, const Params& P) {
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) k.C[i][j] = T(0);
  k.C[0][0] = T(P.err_y2); k.C[1][1] = T(P.err_z2);
  k.C[2][2] = T(P.init_c_ss); k.C[3][3] = T(P.init_c_tt); k.C[4][4] = T(P.init_c_qq);
  k.chi2 = T(0);
}


// Rotation of the state into the sector frame turned by alpha about the beam axis (sa = sin(alpha), ca = cos(alpha)),
// DESIGN.md section 3.9.2.  The point and the direction turn rigidly; the state is then given at the plane
// x' = x*ca + y*sa of the new frame (returned in *x_new), so the covariance moves with the Jacobian of "turn, then
// slide along the track back onto that plane".  Plain operations, one rounding each (no fma).  Returns false and leaves
// the state untouched if the track is too steep in either frame.
template <class T>
bool kf_rotate(KF<T>& k, T kb, T x, T sa, T ca, T max_sinphi, T* x_new) {
  const T y = k.p[0], s = k.p[2], t = k.p[3], q = k.p[4];
  if (!(std::fabs(s) < max_sinphi)) return false;
  const T c = std::sqrt(T(1) - s * s);
  const T s1 = s * ca - c * sa;
  const T c1 = c * ca + s * sa;
  if (!(std::fabs(s1) < max_sinphi) || !(c1 > T(0))) return false;
  const T xn = x * ca + y * sa;
  const T yn = y * ca - x * sa;
  T J[5][5];
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) J[i][j] = (i == j) ? T(1) : T(0);
  J[0][0] = c / c1;                           // d y'/d y: the slide along the track back to the plane x' = const
  J[1][0] = ((T(0) - sa) * t) / c1;           // d z'/d y
  J[2][0] = (T(0) - kb * q) * sa;             // d s'/d y: the curvature acts over the slide
  J[2][2] = c1 / c;                           // d sin(phi - alpha)/d sin(phi)
  T M[5][5], C1[5][5];
  for (int i = 0; i < 5; ++i)
    for (int l = 0; l < 5; ++l) {
      T acc = T(0);
      for (int kk = 0; kk < 5; ++kk) acc = acc + J[i][kk] * k.C[kk][l];
      M[i][l] = acc;
    }
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) {
      T acc = T(0);
      for (int l = 0; l < 5; ++l) acc = acc + M[i][l] * J[j][l];
      C1[i][j] = acc; C1[j][i] = acc;
    }
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) k.C[i][j] = C1[i][j];
  k.p[0] = yn; k.p[2] = s1;
  *x_new = xn;
  return true;
}

// ------------------------------------------------------------------------------------------
struct Oracle {
  Params P;
  int n_sr = 0;                        // n_sectors * n_rows
  float kb = 0.f;                      // curvature constant
  float inv_cy = 0.f, inv_cz = 0.f;
  std::vector<float> ymax;             // [n_rows]
  std::vector<int32_t> ny;             // [n_rows]
  // link tables, index [row][k-1], k = row step 1 or 2
  std::vector<float> up_dx, up_ratio, up_wy, up_wz, dn_dx, dn_ratio, dn_wy, dn_wz;

  // input (borrowed for the duration of run())
  int64_t n = 0;
  const uint8_t* in_sector = nullptr; const uint8_t* in_row = nullptr;
  const float* in_y = nullptr; const float* in_z = nullptr;
  std::vector<float> z_from_time;      // pseudo-z computed from the native time, when z_is_time
  std::vector<float> y_from_pad;       // sector-local y computed from the native pad coordinate (section 3.0b), when y_is_pad

  // S1
  std::vector<float> zmin, zmax; std::vector<int32_t> nz;         // per sector
  std::vector<int32_t> bin_base;                                  // [n_sr+1]
  std::vector<int32_t> gbin;                                      // [n] global bin of input cluster
  std::vector<int32_t> perm;                                      // [n] sorted position -> input index
  std::vector<float> ys, zs;                                      // [n] sorted
  std::vector<int32_t> s_sector, s_row;                           // [n] sorted (oracle convenience)
  std::vector<int32_t> bin_start;                                 // [n_bins+1]
  std::vector<int32_t> row_start;                                 // [n_sr+1]
  // S2
  std::vector<int32_t> link_up_raw, link_dn_raw;
  // S3
  std::vector<int32_t> link_up, link_dn, seed_head, seed_len;
  // S4 (per seed; values held as double, exact for the float instance)
  std::vector<int32_t> t_hit;                                     // [n_seeds * n_rows] sorted position or -1
  std::vector<int32_t> t_first_row, t_last_row, t_n_hits, t_kept, t_ndf, t_sector;
  std::vector<double> t_par, t_cov, t_x_ref, t_z_ref, t_chi2;     // par [n_seeds*5], cov [n_seeds*15]
  std::vector<int64_t> t_kf_steps;                                // [1] total propagate calls (for bytes model)
  // S5
  std::vector<int32_t> tracklet_of_seed;                          // [n_seeds] rank among kept or -1
  std::vector<uint64_t> owner;                                    // [n] by sorted position
  std::vector<int32_t> k_owned;                                   // [n_seeds]
  std::vector<int32_t> trk_seed, trk_sector, trk_first_row, trk_last_row, trk_n_clusters, trk_ndf;
  std::vector<double> trk_par, trk_cov, trk_x_ref, trk_z_ref, trk_chi2, trk_z_beam;
  std::vector<int32_t> trk_cl_pos;                                 // sorted positions parallel to trk_cl_idx
  // S7 refit over the owned clusters
  std::vector<double> fit_par, fit_cov, fit_x_ref, fit_z_ref, fit_chi2;
  std::vector<int32_t> fit_ndf, fit_n;
  std::vector<double> fit_res_y, fit_res_z;                        // parallel to trk_cl_idx: residual to the extrapolated track
  std::vector<int32_t> fit_qres_y, fit_qres_z;                     // the same as counts of steps
  // S8 cluster protection, "strategy B"
  std::vector<int32_t> keep;                                       // [n] by INPUT index: 1 protected, 0 removable
  // S9 track merger
  std::vector<int32_t> fit_row;                                    // [n_tracks] row of the state of the downward refit
  std::vector<double> up_par, up_cov, up_x_ref, up_z_ref, up_chi2; // upward refit: state at the highest fitted row
  std::vector<int32_t> up_row, up_n;
  std::vector<int32_t> mrg_best_b, mrg_best_a, mrg_next, mrg_prev, mrg_dir;   // [n_tracks]
  std::vector<double> mrg_chi2_b;                                  // [n_tracks] score of best_b (or -1)
  std::vector<int32_t> mrg_of_track, mrg_seg_start, mrg_seg_idx;   // merged id of every track; CSR merged -> tracks, inner to outer
  std::vector<double> mrg_par, mrg_cov, mrg_x_ref, mrg_z_ref, mrg_chi2;
  std::vector<int32_t> mrg_n_fit, mrg_ndf, mrg_sector, mrg_n_clusters;
  // S9 apex links of loopers
  std::vector<int32_t> apx_best, apx_partner, apx_leg;             // [n_merged]
  std::vector<double> apx_score;                                   // [n_merged] score of apx_best or -1
  // hit removal, strategy A
  std::vector<int32_t> rem_class, rem_good_track, rem_remove;      // [n] by INPUT index
  int s4_prec = 32;
  std::vector<int32_t> trk_cl_start, trk_cl_idx, cluster_track;
  std::vector<double> stage_seconds;                              // [5]

  explicit Oracle(const Params& p) : P(p) { derive(); }

  // ---- host-side derived tables, each one stated fp32 expression
  void derive() {
    n_sr = P.n_sectors * P.n_rows;
    kb = -0.00299792458f * P.bz_tesla;
    inv_cy = 1.0f / P.cell_y;
    inv_cz = 1.0f / P.cell_z;
    ymax.resize(P.n_rows); ny.resize(P.n_rows);
    for (int r = 0; r < P.n_rows; ++r) {
      ymax[r] = P.row_x[r] * P.tan_half_sector;
      ny[r] = (int)std::floor((2.0f * ymax[r]) * inv_cy) + 1;
    }
    auto tab = [&](std::vector<float>& v) { v.assign(P.n_rows * 2, 0.f); };
    tab(up_dx); tab(up_ratio); tab(up_wy); tab(up_wz); tab(dn_dx); tab(dn_ratio); tab(dn_wy); tab(dn_wz);
    for (int r = 0; r < P.n_rows; ++r)
      for (int k = 1; k <= 2; ++k) {
        if (r + k < P.n_rows) {
          const float dx = P.row_x[r + k] - P.row_x[r];
          up_dx[r * 2 + k - 1] = dx;
          up_ratio[r * 2 + k - 1] = P.row_x[r + k] / P.row_x[r];
          up_wy[r * 2 + k - 1] = P.link_ay * dx + P.link_b;
          up_wz[r * 2 + k - 1] = P.link_az * dx + P.link_b;
        }
        if (r - k >= 0) {
          const float dx = P.row_x[r] - P.row_x[r - k];
          dn_dx[r * 2 + k - 1] = dx;
          dn_ratio[r * 2 + k - 1] = P.row_x[r - k] / P.row_x[r];
          dn_wy[r * 2 + k - 1] = P.link_ay * dx + P.link_b;
          dn_wz[r * 2 + k - 1] = P.link_az * dx + P.link_b;
        }
      }
  }

  // grid coordinates (DESIGN.md section 3.1 (3)); v already fp32
  int bin_iy(float y, int r) const { return floor_clamp((y + ymax[r]) * inv_cy, ny[r] - 1); }
  int bin_iz(float z, int s) const { return floor_clamp((z - zmin[s]) * inv_cz, nz[s] - 1); }

  // ------------------------------------------------------------------------------ S1
  int stage1() {
    zmin.assign(P.n_sectors, INFINITY); zmax.assign(P.n_sectors, -INFINITY); nz.assign(P.n_sectors, 0);
    for (int64_t i = 0; i < n; ++i) {
      if (in_sector[i] >= P.n_sectors || in_row[i] >= P.n_rows) return -1;
      if (!std::isfinite(in_y[i]) || !std::isfinite(in_z[i])) return -1;      // precondition: finite coordinates
      const int s = in_sector[i];
      zmin[s] = std::min(zmin[s], in_z[i]);
      zmax[s] = std::max(zmax[s], in_z[i]);
    }
    for (int s = 0; s < P.n_sectors; ++s) {
      if (!(zmin[s] <= zmax[s])) continue;
      const float rows = std::floor((zmax[s] - zmin[s]) * inv_cz);
      if (!(rows < 2147483646.0f)) return -2;                                   // more bin rows than an int32 holds: N_b > INT32_MAX
      nz[s] = (int)rows + 1;
    }
    bin_base.assign(n_sr + 1, 0);
    int64_t acc = 0;
    for (int s = 0; s < P.n_sectors; ++s)
      for (int r = 0; r < P.n_rows; ++r) {
        bin_base[s * P.n_rows + r] = (int32_t)acc;
        acc += (int64_t)ny[r] * nz[s];
        if (acc > INT32_MAX) return -2;
      }
    bin_base[n_sr] = (int32_t)acc;
    const int64_t n_bins = acc;
    gbin.resize(n);
    for (int64_t i = 0; i < n; ++i) {
      const int s = in_sector[i], r = in_row[i];
      gbin[i] = bin_base[s * P.n_rows + r] + bin_iz(in_z[i], s) * ny[r] + bin_iy(in_y[i], r);
    }
    // order = ascending (sector,row,bin) = ascending global bin, ties by input index: std::stable_sort
    perm.resize(n);
    std::iota(perm.begin(), perm.end(), 0);
    std::stable_sort(perm.begin(), perm.end(), [&](int32_t a, int32_t b) { return gbin[a] < gbin[b]; });
    ys.resize(n); zs.resize(n); s_sector.resize(n); s_row.resize(n);
    bin_start.assign(n_bins + 1, 0);
    for (int64_t pos = 0; pos < n; ++pos) {
      const int32_t i = perm[pos];
      ys[pos] = in_y[i]; zs[pos] = in_z[i]; s_sector[pos] = in_sector[i]; s_row[pos] = in_row[i];
      bin_start[gbin[i] + 1]++;
    }
    for (int64_t b = 0; b < n_bins; ++b) bin_start[b + 1] += bin_start[b];   // CSR: bin b = [bin_start[b], bin_start[b+1])
    row_start.resize(n_sr + 1);
    for (int sr = 0; sr <= n_sr; ++sr) row_start[sr] = bin_start[bin_base[sr]];
    return 0;
  }

  // positions of row t of sector s whose (y,z) lies in the closed rectangle, visited in ascending position
  template <class F>
  void for_each_in_rect(int s, int t, float ylo, float yhi, float zlo, float zhi, F&& f) const {
    if (nz[s] == 0) return;
    const int b0 = bin_base[s * P.n_rows + t];
    const int iy0 = bin_iy(ylo, t), iy1 = bin_iy(yhi, t), iz0 = bin_iz(zlo, s), iz1 = bin_iz(zhi, s);
    for (int iz = iz0; iz <= iz1; ++iz) {
      const int jb = bin_start[b0 + iz * ny[t] + iy0], je = bin_start[b0 + iz * ny[t] + iy1 + 1];
      for (int j = jb; j < je; ++j)
        if (ys[j] >= ylo && ys[j] <= yhi && zs[j] >= zlo && zs[j] <= zhi) f(j);
    }
  }

  // ------------------------------------------------------------------------------ S2
  void stage2() {
    link_up_raw.assign(n, -1); link_dn_raw.assign(n, -1);
    std::vector<int32_t> U, D;
    for (int64_t i = 0; i < n; ++i) {
      const int s = s_sector[i], r = s_row[i];
      const float y = ys[i], z = zs[i];
      int ku = 0, kd = 0;
      U.clear(); D.clear();
      for (int k = 1; k <= 2 && U.empty(); ++k) {
        if (r + k >= P.n_rows) break;
        const float yc = y * up_ratio[r * 2 + k - 1], wy = up_wy[r * 2 + k - 1], wz = up_wz[r * 2 + k - 1];
        for_each_in_rect(s, r + k, yc - wy, yc + wy, z - wz, z + wz, [&](int j) { U.push_back(j); });
        ku = k;
      }
      for (int k = 1; k <= 2 && D.empty(); ++k) {
        if (r - k < 0) break;
        const float yc = y * dn_ratio[r * 2 + k - 1], wy = dn_wy[r * 2 + k - 1], wz = dn_wz[r * 2 + k - 1];
        for_each_in_rect(s, r - k, yc - wy, yc + wy, z - wz, z + wz, [&](int j) { D.push_back(j); });
        kd = k;
      }
      if (U.empty() || D.empty()) continue;
      const float dxu = up_dx[r * 2 + ku - 1], dxd = dn_dx[r * 2 + kd - 1];
      const float cut = P.link_T * ((dxu * dxd) * (dxu * dxd));
      float best = INFINITY; int bu = -1, bd = -1;
      for (int u : U)                       // ascending u, then ascending d; strict '<' keeps the first minimum
        for (int d : D) {
          const float Dy = dxd * (ys[u] - y) - dxu * (y - ys[d]);
          const float Dz = dxd * (zs[u] - z) - dxu * (z - zs[d]);
          const float Dv = Dy * Dy + Dz * Dz;
          if (Dv < best) { best = Dv; bu = u; bd = d; }
        }
      if (best <= cut) { link_up_raw[i] = bu; link_dn_raw[i] = bd; }
    }
  }

  // ------------------------------------------------------------------------------ S3
  void stage3() {
    link_up.assign(n, -1); link_dn.assign(n, -1);
    for (int64_t i = 0; i < n; ++i) {
      const int u = link_up_raw[i], d = link_dn_raw[i];
      if (u >= 0 && link_dn_raw[u] == i) link_up[i] = u;
      if (d >= 0 && link_up_raw[d] == i) link_dn[i] = d;
    }
    seed_head.clear(); seed_len.clear();
    for (int64_t i = 0; i < n; ++i) {
      if (!(link_up[i] >= 0 && link_dn[i] < 0)) continue;
      int len = 0;
      for (int c = (int)i; c >= 0; c = link_up[c]) ++len;
      if (len >= P.min_chain_len) { seed_head.push_back((int32_t)i); seed_len.push_back(len); }
    }
  }

  // ------------------------------------------------------------------------------ S4
  // nearest gated cluster of row r; returns sorted position or -1
  template <class T>
  int search(int s, int r, const KF<T>& k, T zref) const {
    const T cut = T(P.pick_chi2_cut);
    const T sy2 = k.C[0][0] + T(P.err_y2), sz2 = k.C[1][1] + T(P.err_z2);
    const T hy = std::sqrt(cut * sy2), hz = std::sqrt(cut * sz2);
    const T zabs = zref + k.p[1];
    const T ylo = k.p[0] - hy, yhi = k.p[0] + hy, zlo = zabs - hz, zhi = zabs + hz;
    const T wy = T(1) / sy2, wz = T(1) / sz2;
    T best = T(INFINITY); int arg = -1;
    for_each_in_rect(s, r, (float)ylo, (float)yhi, (float)zlo, (float)zhi, [&](int j) {
      if (T(ys[j]) < ylo || T(ys[j]) > yhi || T(zs[j]) < zlo || T(zs[j]) > zhi) return;
      const T dy = T(ys[j]) - k.p[0];
      const T dz = (T(zs[j]) - zref) - k.p[1];
      const T d2 = (dy * dy) * wy + (dz * dz) * wz;
      if (d2 <= cut && d2 < best) { best = d2; arg = j; }
    });
    return arg;
  }

  template <class T>
  void tracklet(int sd) {
    const int R = P.n_rows;
    int32_t* hit = &t_hit[(size_t)sd * R];
    std::fill(hit, hit + R, -1);
    const int h = seed_head[sd], nx = link_up[h];
    const int s = s_sector[h], r0 = s_row[h], r1 = s_row[nx];
    const T kbT = T(kb), msp = T(P.max_sinphi), ey2 = T(P.err_y2), ez2 = T(P.err_z2);
    const T zref = T(zs[h]);
    int64_t steps = 0;

    // seed: straight line through the first two chain clusters
    KF<T> k;
    {
      const T dx = T(P.row_x[r1]) - T(P.row_x[r0]);
      const T dy = T(ys[nx]) - T(ys[h]);
      const T dz = T(zs[nx]) - T(zs[h]);
      const T dl = std::sqrt(dx * dx + dy * dy);
      k.p[0] = T(ys[h]); k.p[1] = T(0); k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = T(0);
      kf_reset_cov(k, P);
    }
    hit[r0] = h;
    int cur = r0;                               // row the state lives on
    KF<T> last = k; int last_row = r0;          // "last updated" state (phase A/B)

    // Phase A: follow the chain upward, update without gate
    bool up_ok = true;
    for (int c = nx; c >= 0; c = link_up[c]) {
      const int rc = s_row[c];
      ++steps;
      if (!kf_propagate(k, kbT, T(P.row_x[rc]) - T(P.row_x[cur]), msp, (T*)nullptr)) { up_ok = false; break; }
      cur = rc;
      kf_update(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
      hit[rc] = c;
      last = k; last_row = rc;
    }
    // Phase B: extrapolate upward, pick up gated nearest clusters
    if (up_ok) {
      int gap = 0;
      for (int r = cur + 1; r < R; ++r) {
        ++steps;
        if (!kf_propagate(k, kbT, T(P.row_x[r]) - T(P.row_x[cur]), msp, (T*)nullptr)) break;
        cur = r;
        if (!(std::fabs(k.p[0]) <= T(ymax[r]) + T(P.y_margin))) break;   // left the sector (NaN-safe)
        const int c = search<T>(s, r, k, zref);
        if (c >= 0) {
          kf_update(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
          hit[r] = c; gap = 0;
          last = k; last_row = r;
        } else if (++gap > P.max_gap) break;
      }
    }
    // Phase C: turn round at the last updated cluster, reset C and chi2, refit downward with pick-up
    k = last; cur = last_row;
    kf_reset_cov(k, P);
    KF<T> out = k; int low = last_row;
    {
      int gap = 0;
      for (int r = cur - 1; r >= 0; --r) {
        ++steps;
        if (!kf_propagate(k, kbT, T(P.row_x[r]) - T(P.row_x[cur]), msp, (T*)nullptr)) break;
        cur = r;
        if (!(std::fabs(k.p[0]) <= T(ymax[r]) + T(P.y_margin))) break;   // left the sector (NaN-safe)
        const int c = hit[r] >= 0 ? hit[r] : search<T>(s, r, k, zref);
        if (c >= 0) {
          kf_update(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
          hit[r] = c; gap = 0;
          out = k; low = r;
        } else if (++gap > P.max_gap) break;
      }
    }
    for (int r = 0; r < low; ++r) hit[r] = -1;
    int nh = 0;
    for (int r = 0; r < R; ++r) nh += hit[r] >= 0;
    t_first_row[sd] = low; t_last_row[sd] = last_row; t_n_hits[sd] = nh; t_sector[sd] = s;
    t_ndf[sd] = 2 * nh - 5;
    t_kept[sd] = nh >= P.min_tracklet_hits;
    for (int i = 0; i < 5; ++i) t_par[(size_t)sd * 5 + i] = (double)out.p[i];
    for (int i = 0, m = 0; i < 5; ++i)
      for (int j = 0; j <= i; ++j, ++m) t_cov[(size_t)sd * 15 + m] = (double)out.C[i][j];
    t_x_ref[sd] = (double)P.row_x[low]; t_z_ref[sd] = (double)zref; t_chi2[sd] = (double)out.chi2;
    t_kf_steps[0] += steps;
  }

  template <class T>
  void stage4() {
    const size_t K = seed_head.size();
    t_hit.assign(K * P.n_rows, -1);
    t_first_row.assign(K, 0); t_last_row.assign(K, 0); t_n_hits.assign(K, 0); t_kept.assign(K, 0);
    t_ndf.assign(K, 0); t_sector.assign(K, 0);
    t_par.assign(K * 5, 0.0); t_cov.assign(K * 15, 0.0);
    t_x_ref.assign(K, 0.0); t_z_ref.assign(K, 0.0); t_chi2.assign(K, 0.0);
    t_kf_steps.assign(1, 0);
    for (size_t sd = 0; sd < K; ++sd) tracklet<T>((int)sd);
  }

  // ------------------------------------------------------------------------------ S5
  void stage5() {
    const size_t K = seed_head.size();
    const int R = P.n_rows;
    tracklet_of_seed.assign(K, -1);
    int32_t nk = 0;
    for (size_t sd = 0; sd < K; ++sd)
      if (t_kept[sd]) tracklet_of_seed[sd] = nk++;
    auto key = [&](size_t sd) {
      return ((uint64_t)(uint32_t)t_n_hits[sd] << 32) | (uint64_t)(0xFFFFFFFFu - (uint32_t)tracklet_of_seed[sd]);
    };
    owner.assign(n, 0);
    for (size_t sd = 0; sd < K; ++sd) {
      if (!t_kept[sd]) continue;
      const uint64_t kk = key(sd);
      for (int r = 0; r < R; ++r) {
        const int c = t_hit[sd * R + r];
        if (c >= 0) owner[c] = std::max(owner[c], kk);
      }
    }
    k_owned.assign(K, 0);
    for (size_t sd = 0; sd < K; ++sd) {
      if (!t_kept[sd]) continue;
      const uint64_t kk = key(sd);
      for (int r = 0; r < R; ++r) {
        const int c = t_hit[sd * R + r];
        if (c >= 0 && owner[c] == kk) k_owned[sd]++;
      }
    }
    trk_seed.clear(); trk_sector.clear(); trk_first_row.clear(); trk_last_row.clear(); trk_n_clusters.clear();
    trk_ndf.clear(); trk_par.clear(); trk_cov.clear(); trk_x_ref.clear(); trk_z_ref.clear(); trk_chi2.clear(); trk_z_beam.clear();
    trk_cl_start.assign(1, 0); trk_cl_idx.clear(); trk_cl_pos.clear();
    cluster_track.assign(n, -1);
    for (size_t sd = 0; sd < K; ++sd) {
      if (!t_kept[sd] || k_owned[sd] < P.min_track_hits) continue;
      const int32_t id = (int32_t)trk_seed.size();
      const uint64_t kk = key(sd);
      int first = -1, lastr = -1;
      for (int r = 0; r < R; ++r) {
        const int c = t_hit[sd * R + r];
        if (c >= 0 && owner[c] == kk) {
          if (first < 0) first = r;
          lastr = r;
          trk_cl_idx.push_back(perm[c]);
          trk_cl_pos.push_back(c);
          cluster_track[perm[c]] = id;
        }
      }
      trk_cl_start.push_back((int32_t)trk_cl_idx.size());
      trk_seed.push_back((int32_t)sd); trk_sector.push_back(t_sector[sd]);
      trk_first_row.push_back(first); trk_last_row.push_back(lastr); trk_n_clusters.push_back(k_owned[sd]);
      trk_ndf.push_back(t_ndf[sd]);
      for (int i = 0; i < 5; ++i) trk_par.push_back(t_par[sd * 5 + i]);
      for (int i = 0; i < 15; ++i) trk_cov.push_back(t_cov[sd * 15 + i]);
      trk_x_ref.push_back(t_x_ref[sd]); trk_z_ref.push_back(t_z_ref[sd]); trk_chi2.push_back(t_chi2[sd]);
      // section 3.6: absolute pseudo-z of the state = z_ref + z_rel (one rounding), then the beam-line extrapolation
      const double* pp = &t_par[sd * 5];
      if (s4_prec == 64)
        trk_z_beam.push_back(beam_z<double>((double)kb, t_x_ref[sd], pp[0], t_z_ref[sd] + pp[1], pp[3], pp[4]));
      else
        trk_z_beam.push_back((double)beam_z<float>(kb, (float)t_x_ref[sd], (float)pp[0], (float)t_z_ref[sd] + (float)pp[1],
                                                   (float)pp[3], (float)pp[4]));
    }
  }

  // ---------------------------------------------------------------------------------------- S7
  // Refit of every track over the clusters it OWNS after the selector, top row downwards (
  // PAPER.md:99, 138 "Track Fit": the step after track finding; here without merging and without corrections).
  // Seed at the top owned cluster from the direction to the next lower one (the S4 seed rule, oriented towards +x),
  // q/pT of the track as the starting value, initial covariance, chi2 = 0; then propagate + update (no gate) through
  // the owned clusters in descending row.  A failed propagation stops the fit at the last updated cluster.
  template <class T>
  void stage6() {
    const size_t nt = trk_seed.size();
    fit_par.assign(nt * 5, 0.0); fit_cov.assign(nt * 15, 0.0); fit_x_ref.assign(nt, 0.0); fit_z_ref.assign(nt, 0.0);
    fit_chi2.assign(nt, 0.0); fit_ndf.assign(nt, 0); fit_n.assign(nt, 0); fit_row.assign(nt, 0);
    fit_res_y.assign(trk_cl_idx.size(), 0.0); fit_res_z.assign(trk_cl_idx.size(), 0.0);
    const T kbT = T(kb), msp = T(P.max_sinphi), ey2 = T(P.err_y2), ez2 = T(P.err_z2);
    for (size_t id = 0; id < nt; ++id) {
      const int32_t* cl = &trk_cl_pos[trk_cl_start[id]];
      const int m = trk_cl_start[id + 1] - trk_cl_start[id];
      if (m < 2) continue;                                  // cannot happen with min_track_hits >= 2
      const int top = cl[m - 1], nxt = cl[m - 2];
      const T zref = T(zs[top]);
      const T dx = T(P.row_x[s_row[top]]) - T(P.row_x[s_row[nxt]]);
      const T dy = T(ys[top]) - T(ys[nxt]), dz = T(zs[top]) - T(zs[nxt]);
      const T dl = std::sqrt(dx * dx + dy * dy);
      KF<T> k;
      k.p[0] = T(ys[top]); k.p[1] = T(0); k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = T(trk_par[id * 5 + 4]);
      kf_reset_cov(k, P);
      int cur = s_row[top], nfit = 1;
      for (int i = m - 2; i >= 0; --i) {
        const int c = cl[i], r = s_row[c];
        if (!kf_propagate<T>(k, kbT, T(P.row_x[r]) - T(P.row_x[cur]), msp, (T*)nullptr)) break;
        // residual of the cluster to the extrapolated track position: the
        // innovation of the update that follows
        fit_res_y[trk_cl_start[id] + i] = (double)(T(ys[c]) - k.p[0]);
        fit_res_z[trk_cl_start[id] + i] = (double)((T(zs[c]) - zref) - k.p[1]);
        kf_update<T>(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
        cur = r; ++nfit;
      }
      store_kf(k, &fit_par[id * 5], &fit_cov[id * 15], &fit_chi2[id]);
      fit_x_ref[id] = (double)P.row_x[cur]; fit_z_ref[id] = (double)zref; fit_row[id] = cur;
      fit_n[id] = nfit; fit_ndf[id] = 2 * nfit - 5;
    }
  }


  // the residuals of the last stage6 as 16-bit counts of `step_y` / `step_z` (cm).  The residual is
  // the fp32 one (in the double instance: the double residual cast to fp32 first); inv_step = 1 / step, one fp32 division.
  void quantise_residuals(float step_y, float step_z) {
    const float iy = 1.0f / step_y, iz = 1.0f / step_z;
    fit_qres_y.resize(fit_res_y.size()); fit_qres_z.resize(fit_res_z.size());
    for (size_t i = 0; i < fit_res_y.size(); ++i) {
      fit_qres_y[i] = quantise_residual((float)fit_res_y[i], iy);
      fit_qres_z[i] = quantise_residual((float)fit_res_z[i], iz);
    }
  }

  // ---------------------------------------------------------------------------------------- S9
  // Track merger ("Track Fit" of PAPER.md:99, 131, 138: the segments a track was found in - one per
  // sector it crosses, and one per stretch between holes longer than max_gap - are joined and refitted).  Runs after
  // stage6 (the downward refit gives every segment's state at its INNER end).
  //   9.1 upward refit: the state at the OUTER end;  9.2-9.4 candidates and score;  9.5 mutual best;  9.6 chains;
  //   9.7 downward refit of every merged track through all its segments, turning the frame at sector changes.
  struct MergeCuts { int32_t max_rows, back_rows; float edge, dz_win, chi2_cut, road_z0, road_z1; };

  template <class T>
  void stage9(const MergeCuts& mc) {
    const int nt = (int)trk_seed.size(), n_az = P.n_sectors / 2;
    const T kbT = T(kb), msp = T(P.max_sinphi), ey2 = T(P.err_y2), ez2 = T(P.err_z2);
    // sin and cos of the sector angle (twice the half-sector angle) from tan_half_sector alone: no libm (section 3.0)
    const T th = T(P.tan_half_sector);
    const T den = T(1) + th * th;
    const T sin_a = (T(2) * th) / den, cos_a = (T(1) - th * th) / den;

    // ---- 9.1 upward refit: seed at the lowest owned cluster from the direction to the next one, q/pT of the downward
    // refit as the starting value, then propagate + update (no gate) through the owned clusters in ascending row
    up_par.assign((size_t)nt * 5, 0.0); up_cov.assign((size_t)nt * 15, 0.0); up_x_ref.assign(nt, 0.0); up_z_ref.assign(nt, 0.0);
    up_chi2.assign(nt, 0.0); up_row.assign(nt, 0); up_n.assign(nt, 0);
    for (int id = 0; id < nt; ++id) {
      const int32_t* cl = &trk_cl_pos[trk_cl_start[id]];
      const int m = trk_cl_start[id + 1] - trk_cl_start[id];
      if (m < 2) continue;
      const int bot = cl[0], nxt = cl[1];
      const T zref = T(zs[bot]);
      const T dx = T(P.row_x[s_row[nxt]]) - T(P.row_x[s_row[bot]]);
      const T dy = T(ys[nxt]) - T(ys[bot]), dz = T(zs[nxt]) - T(zs[bot]);
      const T dl = std::sqrt(dx * dx + dy * dy);
      KF<T> k;
      k.p[0] = T(ys[bot]); k.p[1] = T(0); k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = T(fit_par[(size_t)id * 5 + 4]);
      kf_reset_cov(k, P);
      int cur = s_row[bot], nfit = 1;
      for (int i = 1; i < m; ++i) {
        const int c = cl[i], r = s_row[c];
        if (!kf_propagate<T>(k, kbT, T(P.row_x[r]) - T(P.row_x[cur]), msp, (T*)nullptr)) break;
        kf_update<T>(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
        cur = r; ++nfit;
      }
      store_kf(k, &up_par[(size_t)id * 5], &up_cov[(size_t)id * 15], &up_chi2[id]);
      up_x_ref[id] = (double)P.row_x[cur]; up_z_ref[id] = (double)zref; up_row[id] = cur; up_n[id] = nfit;
    }

    // ---- 9.2 absolute z of the two ends (one rounding each)
    std::vector<T> z_in(nt), z_out(nt);
    for (int id = 0; id < nt; ++id) {
      z_in[id] = T(fit_z_ref[id]) + T(fit_par[(size_t)id * 5 + 1]);
      z_out[id] = T(up_z_ref[id]) + T(up_par[(size_t)id * 5 + 1]);
    }
    // tracks of a sector ordered by z_in (a library sort as a step: it only speeds the window scan up, the candidate set
    // is defined by the predicate of 9.3)
    std::vector<std::vector<int32_t>> by_sector(P.n_sectors);
    for (int id = 0; id < nt; ++id) by_sector[trk_sector[id]].push_back(id);
    for (auto& v : by_sector) std::sort(v.begin(), v.end(), [&](int32_t a, int32_t b) { return z_in[a] < z_in[b] || (z_in[a] == z_in[b] && a < b); });

    // ---- 9.3 / 9.4 / 9.5: score of every candidate pair; best partner of every outer end and of every inner end
    mrg_best_b.assign(nt, -1); mrg_best_a.assign(nt, -1); mrg_chi2_b.assign(nt, -1.0); mrg_dir.assign(nt, 0);
    std::vector<T> best_a_chi2(nt, T(0));
    std::vector<int32_t> best_b_dir(nt, 0), best_a_dir(nt, 0);
    const T dzw = T(mc.dz_win), cut = T(mc.chi2_cut);
    for (int a = 0; a < nt; ++a) {
      if (up_n[a] < 2 || fit_n[a] < 2) continue;
      const int sa_ = trk_sector[a], ra = up_row[a];
      const T ya = T(up_par[(size_t)a * 5 + 0]);
      T best = T(0); int bb = -1, bdir = 0;
      for (int pass = 0; pass < 2; ++pass) {
        int dir = 0, sb = sa_;
        if (pass == 1) {
          // the neighbour the outer end is heading for: only if that end lies within `edge` of the sector boundary
          if (n_az < 1) continue;                         // a one-sector geometry has no neighbour
          if (!(std::fabs(ya) >= T(ymax[ra]) - T(mc.edge))) continue;
          dir = ya >= T(0) ? 1 : -1;
          sb = (sa_ / n_az) * n_az + ((sa_ % n_az) + dir + n_az) % n_az;
          if (sb == sa_) continue;                        // a one-sector geometry has no neighbour
        }
        // 9.4 (first half) the outer state of a, turned into the neighbour's frame if that is where this pass looks
        KF<T> k0; load_kf(k0, &up_par[(size_t)a * 5], &up_cov[(size_t)a * 15], 0.0);
        T x0 = T(up_x_ref[a]);
        if (dir != 0 && !kf_rotate<T>(k0, kbT, x0, dir > 0 ? sin_a : T(0) - sin_a, cos_a, msp, &x0)) continue;
        // the road: where a straight continuation of that state has its z at a given x
        const T zslope = k0.p[3] / std::sqrt(T(1) - k0.p[2] * k0.p[2]);
        const auto& lst = by_sector[sb];
        const T zlo = z_out[a] - dzw, zhi = z_out[a] + dzw;
        auto it = std::lower_bound(lst.begin(), lst.end(), zlo, [&](int32_t b, T v) { return z_in[b] < v; });
        for (; it != lst.end() && z_in[*it] <= zhi; ++it) {
          const int b = *it;
          if (b == a || up_n[b] < 2 || fit_n[b] < 2) continue;
          const int rb = fit_row[b];
          if (dir == 0 ? (rb < ra + 1 || rb > ra + mc.max_rows) : (rb < ra - mc.back_rows || rb > ra + mc.max_rows)) continue;
          const T dxb = T(fit_x_ref[b]) - x0;
          if (!(std::fabs(z_in[b] - (z_out[a] + dxb * zslope)) <= T(mc.road_z0) + T(mc.road_z1) * std::fabs(dxb))) continue;
          // 9.4 (second half) moved to b's inner plane
          KF<T> k = k0;
          if (!kf_propagate<T>(k, kbT, dxb, msp, (T*)nullptr)) continue;
          const double* pb = &fit_par[(size_t)b * 5]; const double* cb = &fit_cov[(size_t)b * 15];
          T d[5];
          d[0] = T(pb[0]) - k.p[0];
          d[1] = z_in[b] - (T(up_z_ref[a]) + k.p[1]);
          d[2] = T(pb[2]) - k.p[2]; d[3] = T(pb[3]) - k.p[3]; d[4] = T(pb[4]) - k.p[4];
          T chi = T(0);
          for (int i = 0; i < 5; ++i) chi = chi + (d[i] * d[i]) / (k.C[i][i] + T(cb[i * (i + 1) / 2 + i]));
          if (!(chi <= cut)) continue;
          // 9.5 the best partner of a's outer end (ties -> lowest b) and of b's inner end (ties -> lowest a)
          if (bb < 0 || chi < best || (chi == best && b < bb)) { best = chi; bb = b; bdir = dir; }
          if (mrg_best_a[b] < 0 || chi < best_a_chi2[b] || (chi == best_a_chi2[b] && a < mrg_best_a[b])) {
            best_a_chi2[b] = chi; mrg_best_a[b] = a; best_a_dir[b] = dir;
          }
        }
      }
      mrg_best_b[a] = bb; best_b_dir[a] = bdir; mrg_chi2_b[a] = bb >= 0 ? (double)best : -1.0;
    }
    // ---- 9.6 mutual links and chains
    mrg_next.assign(nt, -1); mrg_prev.assign(nt, -1);
    for (int a = 0; a < nt; ++a) {
      const int b = mrg_best_b[a];
      if (b >= 0 && mrg_best_a[b] == a) { mrg_next[a] = b; mrg_prev[b] = a; mrg_dir[a] = best_b_dir[a]; }
    }
    mrg_of_track.assign(nt, -1); mrg_seg_start.assign(1, 0); mrg_seg_idx.clear();
    for (int h = 0; h < nt; ++h) {
      if (mrg_prev[h] >= 0) continue;                     // heads in ascending track id
      const int32_t id = (int32_t)mrg_seg_start.size() - 1;
      int len = 0;
      for (int k2 = h; k2 >= 0 && len < nt; k2 = mrg_next[k2], ++len) { mrg_of_track[k2] = id; mrg_seg_idx.push_back(k2); }
      mrg_seg_start.push_back((int32_t)mrg_seg_idx.size());
    }
    // ---- 9.7 downward refit of every merged track: from the top cluster of the outermost segment through all owned
    // clusters of all segments in turn, the frame turned back at every sector change
    const int nm = (int)mrg_seg_start.size() - 1;
    mrg_par.assign((size_t)nm * 5, 0.0); mrg_cov.assign((size_t)nm * 15, 0.0); mrg_x_ref.assign(nm, 0.0); mrg_z_ref.assign(nm, 0.0);
    mrg_chi2.assign(nm, 0.0); mrg_n_fit.assign(nm, 0); mrg_ndf.assign(nm, 0); mrg_sector.assign(nm, 0); mrg_n_clusters.assign(nm, 0);
    for (int mId = 0; mId < nm; ++mId) {
      const int s0 = mrg_seg_start[mId], s1 = mrg_seg_start[mId + 1];
      int ncl = 0;
      for (int q = s0; q < s1; ++q) ncl += trk_cl_start[mrg_seg_idx[q] + 1] - trk_cl_start[mrg_seg_idx[q]];
      mrg_n_clusters[mId] = ncl;
      const int last = mrg_seg_idx[s1 - 1];
      const int32_t* cl = &trk_cl_pos[trk_cl_start[last]];
      const int m = trk_cl_start[last + 1] - trk_cl_start[last];
      if (m < 2) continue;
      const int top = cl[m - 1], nxt = cl[m - 2];
      const T zref = T(zs[top]);
      const T dx = T(P.row_x[s_row[top]]) - T(P.row_x[s_row[nxt]]);
      const T dy = T(ys[top]) - T(ys[nxt]), dz = T(zs[top]) - T(zs[nxt]);
      const T dl = std::sqrt(dx * dx + dy * dy);
      KF<T> k;
      k.p[0] = T(ys[top]); k.p[1] = T(0); k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = T(trk_par[(size_t)last * 5 + 4]);   // as section 3.7
      kf_reset_cov(k, P);
      T x = T(P.row_x[s_row[top]]);
      int nfit = 1, sector = trk_sector[last];
      bool ok = true;
      for (int q = s1 - 1; q >= s0 && ok; --q) {
        const int seg = mrg_seg_idx[q];
        const int32_t* c2 = &trk_cl_pos[trk_cl_start[seg]];
        const int m2 = trk_cl_start[seg + 1] - trk_cl_start[seg];
        if (q < s1 - 1) {                                 // coming down from segment q+1 into segment q
          const int dir = mrg_dir[seg];                   // the link seg -> next went `dir` sectors up; go back
          if (dir != 0) {
            // first, still in the upper segment's frame, to the plane through the top cluster of segment q (its x in
            // that frame: the point turned by +dir), where the track is no steeper than the finder saw it; then turn
            const int ct = c2[m2 - 1];
            const T sd = dir > 0 ? sin_a : T(0) - sin_a;
            const T xt = T(P.row_x[s_row[ct]]) * cos_a + T(ys[ct]) * sd;
            if (!kf_propagate<T>(k, kbT, xt - x, msp, (T*)nullptr)) break;
            x = xt;
            if (!kf_rotate<T>(k, kbT, x, T(0) - sd, cos_a, msp, &x)) break;
          }
          sector = trk_sector[seg];
        }
        for (int i = (q == s1 - 1 ? m2 - 2 : m2 - 1); i >= 0; --i) {
          const int c = c2[i], r = s_row[c];
          if (!kf_propagate<T>(k, kbT, T(P.row_x[r]) - x, msp, (T*)nullptr)) { ok = false; break; }
          x = T(P.row_x[r]);
          kf_update<T>(k, T(ys[c]), T(zs[c]) - zref, ey2, ez2);
          ++nfit;
        }
      }
      store_kf(k, &mrg_par[(size_t)mId * 5], &mrg_cov[(size_t)mId * 15], &mrg_chi2[mId]);
      mrg_x_ref[mId] = (double)x; mrg_z_ref[mId] = (double)zref; mrg_n_fit[mId] = nfit; mrg_ndf[mId] = 2 * nfit - 5;
      mrg_sector[mId] = sector;
    }
  }


  // ---------------------------------------------------------------------------------------- S9, part 2
  // Apex links: looper following ("secondary legs of looping tracks", PAPER.md:107
  // "the following of looping tracks").  A track that curls up inside the TPC is found as two merged tracks, the outgoing
  // leg and the returning leg (which the finder walks outwards, against the particle's motion); they are never
  // joined by 3.9.3 because the stretch around the apex, where |sin(phi)| >= max_sinphi, cannot be parametrised in x.
  // Both legs end steeply at the apex side and lie on ONE circle: their OUTER ends are compared through the circle
  // centres, the z advance along the arc between the two end points and the dip angles.
  struct ApexCuts { int32_t max_k; float min_s, dz_win, tol_c, tol_z, tol_t, cut; };

  template <class T>
  void stage10(const ApexCuts& ac) {
    const int nm = (int)mrg_seg_start.size() - 1, n_az = P.n_sectors / 2;
    const T kbT = T(kb);
    const T th = T(P.tan_half_sector);
    const T den = T(1) + th * th;
    const T sin_a = (T(2) * th) / den, cos_a = (T(1) - th * th) / den;
    apx_best.assign(nm, -1); apx_partner.assign(nm, -1); apx_leg.assign(nm, 0); apx_score.assign(nm, -1.0);
    std::vector<int32_t> tail(nm);
    std::vector<T> zo(nm);
    for (int m = 0; m < nm; ++m) {
      tail[m] = mrg_seg_idx[mrg_seg_start[m + 1] - 1];
      zo[m] = T(up_z_ref[tail[m]]) + T(up_par[(size_t)tail[m] * 5 + 1]);
    }
    // a tail takes part iff its outer state is steep (it ends because the track curls over) and has a curvature
    auto steep = [&](int m) {
      const int t = tail[m];
      const T s = T(up_par[(size_t)t * 5 + 2]);
      return up_n[t] >= 2 && std::fabs(s) >= T(ac.min_s) && std::fabs(s) < T(1) && kbT * T(up_par[(size_t)t * 5 + 4]) != T(0);
    };
    // circle centre of a tail in its own sector frame: xc = x - sin(phi)/c, yc = y + cos(phi)/c
    auto centre = [&](int t, T* xc, T* yc, T* R, T* c) {
      const T s = T(up_par[(size_t)t * 5 + 2]);
      *c = kbT * T(up_par[(size_t)t * 5 + 4]);
      *xc = T(up_x_ref[t]) - s / *c;
      *yc = T(up_par[(size_t)t * 5 + 0]) + std::sqrt(T(1) - s * s) / *c;
      *R = T(1) / std::fabs(*c);
    };
    for (int A = 0; A < nm; ++A) {
      if (!steep(A)) continue;
      const int a = tail[A], s_a = trk_sector[a];
      const T xA = T(up_x_ref[a]), yA = T(up_par[(size_t)a * 5 + 0]), tA = T(up_par[(size_t)a * 5 + 3]);
      const int dirA = T(up_par[(size_t)a * 5 + 2]) >= T(0) ? 1 : -1;   // the side the track curls to
      T xcA, ycA, RA, cA;
      centre(a, &xcA, &ycA, &RA, &cA);
      T best = T(0); int bb = -1;
      T sk = T(0), ck = T(1);                               // sine and cosine of k sector angles
      for (int k = 0; k <= ac.max_k; ++k) {
        if (k > 0) {
          const T s2 = sk * cos_a + ck * sin_a, c2 = ck * cos_a - sk * sin_a;
          sk = s2; ck = c2;
        }
        if (k > 0 && n_az < 1) break;                       // a one-sector geometry: the tail's own sector only
        const int s_b = n_az < 1 ? s_a : (s_a / n_az) * n_az + ((((s_a % n_az) + dirA * k) % n_az) + n_az) % n_az;
        if (k > 0 && s_b == s_a) break;                     // once round
        const T sd = dirA > 0 ? sk : T(0) - sk;             // sector s_b is the frame of s_a turned by dirA * k sector angles
        for (int B = 0; B < nm; ++B) {                       // plain scan; the predicates below define the set
          if (B == A || !steep(B)) continue;
          const int b = tail[B];
          if (trk_sector[b] != s_b) continue;
          if (!(std::fabs(zo[B] - zo[A]) <= T(ac.dz_win))) continue;
          T xcB, ycB, RB, cB;
          centre(b, &xcB, &ycB, &RB, &cB);
          if (!(cA * cB < T(0))) continue;                  // the returning leg is walked against the motion
          // b's centre and end point in a's frame
          const T xcB_a = xcB * ck - ycB * sd, ycB_a = xcB * sd + ycB * ck;
          const T xB = T(up_x_ref[b]), yB = T(up_par[(size_t)b * 5 + 0]);
          const T xB_a = xB * ck - yB * sd, yB_a = xB * sd + yB * ck;
          const T Rm = T(0.5) * (RA + RB);
          const T dcx = xcA - xcB_a, dcy = ycA - ycB_a;
          const T dc2 = dcx * dcx + dcy * dcy;
          const T ex = xB_a - xA, ey = yB_a - yA;
          const T d = std::sqrt(ex * ex + ey * ey);
          const T h = (T(0.5) * d) / Rm;                    // sine of half the turning angle between the two end points
          if (!(h < T(0.98))) continue;
          // arc = 2 Rm asin(h) = 4 Rm asin(h1), h1 = sine of a quarter of the turning angle; 5-term series of section 3.4.1
          const T h1 = h / std::sqrt(T(2) * (T(1) + std::sqrt(T(1) - h * h)));
          const T w = h1 * h1;
          const T ser = T(1) + w * (T(1.0 / 6.0) + w * (T(3.0 / 40.0) + w * (T(5.0 / 112.0) + w * T(35.0 / 1152.0))));
          const T arc = (T(4) * Rm) * (h1 * ser);
          const T dz = zo[B] - (zo[A] + tA * arc);
          const T dt = tA + T(up_par[(size_t)b * 5 + 3]);
          const T tc = T(ac.tol_c) * Rm;
          const T score = dc2 / (tc * tc) + (dz * dz) / (T(ac.tol_z) * T(ac.tol_z)) + (dt * dt) / (T(ac.tol_t) * T(ac.tol_t));
          if (!(score <= T(ac.cut))) continue;
          if (bb < 0 || score < best || (score == best && B < bb)) { best = score; bb = B; }
        }
      }
      apx_best[A] = bb; apx_score[A] = bb >= 0 ? (double)best : -1.0;
    }
    for (int A = 0; A < nm; ++A) {
      const int B = apx_best[A];
      if (B >= 0 && apx_best[B] == A) apx_partner[A] = B;
    }
    // Which leg is the returning ("secondary") one: a primary moves away from the central electrode, so |z| grows along
    // its motion - on the A side the leg whose apex-side end has the larger z comes later, on the C side the one with the
    // smaller z (the time shift of continuous readout moves both ends alike).  Ties -> the higher id.
    for (int A = 0; A < nm; ++A) {
      const int B = apx_partner[A];
      if (B < 0) continue;
      const bool a_side = trk_sector[tail[A]] < n_az;
      const bool later = a_side ? zo[A] > zo[B] : zo[A] < zo[B];
      apx_leg[A] = (later || (zo[A] == zo[B] && A > B)) ? 1 : 0;
    }
  }


  // ---------------------------------------------------------------------------------------- S8a
  // Hit removal, "strategy A": "positive identification of all hits that can
  // safely be removed" - hits of "tracks of very low momentum", "secondary legs of looping tracks", "track segments with
  // high inclination angle" - while "the online tracking identifies the good tracks used for physics and protects all hits
  // in their vicinity from removal".  Class of an input cluster: 0 not attached; else, for its track k and merged track m:
  // 2 if m is the secondary leg of a looper (3.9.8); else 3 if |q/pT| of the merged fit times min_pt exceeds 1 (low
  // momentum); else 4 if both ends of the segment k are steeper than max_incl; else 1 (good).  Good tracks protect the
  // clusters inside their road exactly as in section 3.8; a cluster is removable iff its class is >= 2 and it is not
  // protected.
  void stage11(float min_pt, float max_incl, float road_y, float road_z) {
    const int nt = (int)trk_seed.size();
    std::vector<int32_t> cls_of_track(nt, 1);
    for (int k = 0; k < nt; ++k) {
      const int m = mrg_of_track[k];
      if (m >= 0 && apx_leg[m] == 1) cls_of_track[k] = 2;
      else if (m >= 0 && std::fabs((float)mrg_par[(size_t)m * 5 + 4]) * min_pt > 1.0f) cls_of_track[k] = 3;
      else if (std::fabs((float)fit_par[(size_t)k * 5 + 2]) > max_incl && std::fabs((float)up_par[(size_t)k * 5 + 2]) > max_incl) cls_of_track[k] = 4;
    }
    rem_class.assign(n, 0); rem_good_track.assign(n, -1); rem_remove.assign(n, 0);
    for (int64_t i = 0; i < n; ++i) {
      const int k = cluster_track[i];
      if (k < 0) continue;
      rem_class[i] = cls_of_track[k];
      if (cls_of_track[k] == 1) rem_good_track[i] = k;
    }
    // protection by the good tracks only (the road of section 3.8 around every cluster a good track owns)
    std::vector<int32_t> kept(n, 0);
    for (int id = 0; id < nt; ++id) {
      if (cls_of_track[id] != 1) continue;
      for (int32_t q = trk_cl_start[id]; q < trk_cl_start[id + 1]; ++q) {
        const int o = trk_cl_pos[q];
        const float y = ys[o], z = zs[o];
        for_each_in_rect(s_sector[o], s_row[o], y - road_y, y + road_y, z - road_z, z + road_z,
                         [&](int j) { kept[perm[j]] = 1; });
      }
    }
    for (int64_t i = 0; i < n; ++i) rem_remove[i] = rem_class[i] >= 2 && !kept[i];
  }

  // ---------------------------------------------------------------------------------------- S8
  // Cluster protection for hit removal, "strategy B": "runs only the online tracking and removes all hits not in the
  // vicinity of good tracks".  A cluster is protected iff it is attached to a track or
  // lies, in its own (sector, row), inside the closed rectangle +-road_y x +-road_z around a cluster some track owns.
  void stage7_protect(float road_y, float road_z) {
    keep.assign(n, 0);
    for (size_t id = 0; id < trk_seed.size(); ++id)
      for (int32_t q = trk_cl_start[id]; q < trk_cl_start[id + 1]; ++q) {
        const int o = trk_cl_pos[q];
        const float y = ys[o], z = zs[o];
        for_each_in_rect(s_sector[o], s_row[o], y - road_y, y + road_y, z - road_z, z + road_z,
                         [&](int j) { keep[perm[j]] = 1; });
      }
  }

  int run(int64_t n_, const uint8_t* sec, const uint8_t* row, const float* y, const float* z, int prec, int last_stage) {
    n = n_; in_sector = sec; in_row = row; in_y = y; in_z = z;
    if (P.z_is_time) {
      // the input holds the cluster time t in time units; its pseudo-z (vertex
      // time 0) is the drift distance left at time t, positive on the A side (sectors < n_sectors / 2), negative on the C
      // side.  fp32, the product and the difference rounded separately.
      z_from_time.resize(n);
      for (int64_t i = 0; i < n; ++i) {
        const float zc = P.drift_length - z[i] * P.cm_per_time_unit;
        z_from_time[i] = (int)sec[i] < P.n_sectors / 2 ? zc : 0.0f - zc;
      }
      in_z = z_from_time.data();
    }
    if (P.y_is_pad) {
      // DESIGN.md section 3.0b (hits arrive in "native pad, row, and time coordinates"): the input holds
      // the pad coordinate p of the cluster (centre of pad 0 = 0, centre of the last pad = n_pads_r - 1, fractional for a
      // centroid).  The pads of a row lie symmetric about the sector axis, so y = (p - (n_pads_r - 1) / 2) * pitch_r.
      // fp32: the half pad count is exact, the difference and the product are rounded separately.  A row out of
      // range is rejected by stage 1 below; its y is left as given.
      y_from_pad.resize(n);
      for (int64_t i = 0; i < n; ++i) {
        const int r = row[i];
        if (r >= P.n_rows) { y_from_pad[i] = y[i]; continue; }
        const float centre = 0.5f * (float)(P.n_pads[r] - 1);
        const float d = y[i] - centre;
        y_from_pad[i] = d * P.pad_pitch[r];
      }
      in_y = y_from_pad.data();
    }
    stage_seconds.assign(5, 0.0);
    auto now = [] { return std::chrono::steady_clock::now(); };
    auto secs = [](auto a, auto b) { return std::chrono::duration<double>(b - a).count(); };
    auto t0 = now();
    int rc = stage1();
    auto t1 = now(); stage_seconds[0] = secs(t0, t1);
    if (rc != 0 || last_stage < 2) return rc;
    stage2();
    auto t2 = now(); stage_seconds[1] = secs(t1, t2);
    if (last_stage < 3) return 0;
    stage3();
    auto t3 = now(); stage_seconds[2] = secs(t2, t3);
    if (last_stage < 4) return 0;
    s4_prec = prec;
    if (prec == 64) stage4<double>(); else stage4<float>();
    auto t4 = now(); stage_seconds[3] = secs(t3, t4);
    if (last_stage < 5) return 0;
    stage5();
    auto t5 = now(); stage_seconds[4] = secs(t4, t5);
    if (last_stage < 6) return 0;
    if (prec == 64) stage6<double>(); else stage6<float>();
    return 0;
  }
};

template <class V>
int give(const V& v, const void** ptr, int64_t* n, int* kind, int k) {
  *ptr = v.data(); *n = (int64_t)v.size(); *kind = k;
  return 0;
}

template <class T>
void load_kf(KF<T>& k, const double* par, const double* cov15, double chi2) {
  for (int i = 0; i < 5; ++i) k.p[i] = (T)par[i];
  for (int i = 0, m = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j, ++m) { k.C[i][j] = (T)cov15[m]; k.C[j][i] = (T)cov15[m]; }
  k.chi2 = (T)chi2;
}
template <class T>
void store_kf(const KF<T>& k, double* par, double* cov15, double* chi2) {
  for (int i = 0; i < 5; ++i) par[i] = (double)k.p[i];
  for (int i = 0, m = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j, ++m) cov15[m] = (double)k.C[i][j];
  if (chi2) *chi2 = (double)k.chi2;
}

template <class T>
int kf_propagate_entry(const Params& P, double* par, double* cov15, double x0, double x1, double* jac25) {
  KF<T> k; load_kf(k, par, cov15, 0.0);
  T J[25];
  const T kbT = T(-0.00299792458f * P.bz_tesla);
  const bool ok = kf_propagate<T>(k, kbT, T(x1) - T(x0), T(P.max_sinphi), J);
  if (!ok) return 0;
  store_kf(k, par, cov15, nullptr);
  if (jac25) for (int i = 0; i < 25; ++i) jac25[i] = (double)J[i];
  return 1;
}

// KF over an explicit point list with the S4 seed rule + phase-A updates (no search), ending on the last point.
template <class T>
int kf_fit_entry(const Params& P, int npt, const double* x, const double* y, const double* z, double* par, double* cov15,
                 double* chi2) {
  if (npt < 2) return 0;
  KF<T> k;
  const T zref = T(z[0]);
  const T dx = T(x[1]) - T(x[0]), dy = T(y[1]) - T(y[0]), dz = T(z[1]) - T(z[0]);
  const T dl = std::sqrt(dx * dx + dy * dy);
  k.p[0] = T(y[0]); k.p[1] = T(0); k.p[2] = dy / dl; k.p[3] = dz / dl; k.p[4] = T(0);
  kf_reset_cov(k, P);
  const T kbT = T(-0.00299792458f * P.bz_tesla);
  for (int i = 1; i < npt; ++i) {
    if (!kf_propagate<T>(k, kbT, T(x[i]) - T(x[i - 1]), T(P.max_sinphi), (T*)nullptr)) return 0;
    kf_update<T>(k, T(y[i]), T(z[i]) - zref, T(P.err_y2), T(P.err_z2));
  }
  store_kf(k, par, cov15, chi2);
  return 1;
}

}  // namespace

// =============================================================================================
extern "C" {

void* orc_create(const void* params) { return new Oracle(*reinterpret_cast<const Params*>(params)); }
void orc_destroy(void* h) { delete reinterpret_cast<Oracle*>(h); }
int orc_params_size() { return (int)sizeof(Params); }

// prec: 32 (parity reference) or 64; last_stage: 1..5, 6 = also the refit of section 3.7
int orc_run(void* h, int64_t n, const uint8_t* sector, const uint8_t* row, const float* y, const float* z, int prec,
            int last_stage) {
  return reinterpret_cast<Oracle*>(h)->run(n, sector, row, y, z, prec, last_stage);
}

// kind: 0 int32, 1 float32, 2 float64, 3 uint64, 4 int64
int orc_get(void* h, const char* name, const void** ptr, int64_t* n, int* kind) {
  Oracle& o = *reinterpret_cast<Oracle*>(h);
  const std::string s(name);
#define I32(f) if (s == #f) return give(o.f, ptr, n, kind, 0)
#define F32(f) if (s == #f) return give(o.f, ptr, n, kind, 1)
#define F64(f) if (s == #f) return give(o.f, ptr, n, kind, 2)
#define U64(f) if (s == #f) return give(o.f, ptr, n, kind, 3)
#define I64(f) if (s == #f) return give(o.f, ptr, n, kind, 4)
  F32(ymax); I32(ny); F32(zmin); F32(zmax); I32(nz); I32(bin_base); I32(gbin); I32(perm); F32(ys); F32(zs);
  I32(s_sector); I32(s_row); I32(bin_start); I32(row_start);
  I32(link_up_raw); I32(link_dn_raw); I32(link_up); I32(link_dn); I32(seed_head); I32(seed_len);
  I32(t_hit); I32(t_first_row); I32(t_last_row); I32(t_n_hits); I32(t_kept); I32(t_ndf); I32(t_sector);
  F64(t_par); F64(t_cov); F64(t_x_ref); F64(t_z_ref); F64(t_chi2); I64(t_kf_steps);
  I32(tracklet_of_seed); U64(owner); I32(k_owned);
  I32(trk_seed); I32(trk_sector); I32(trk_first_row); I32(trk_last_row); I32(trk_n_clusters); I32(trk_ndf);
  F64(trk_par); F64(trk_cov); F64(trk_x_ref); F64(trk_z_ref); F64(trk_chi2); F64(trk_z_beam);
  I32(trk_cl_start); I32(trk_cl_idx); I32(trk_cl_pos); I32(cluster_track); F64(stage_seconds);
  I32(fit_qres_y); I32(fit_qres_z);
  I32(keep); F64(fit_res_y); F64(fit_res_z); F64(fit_par); F64(fit_cov); F64(fit_x_ref); F64(fit_z_ref); F64(fit_chi2); I32(fit_ndf); I32(fit_n);
  I32(fit_row); F64(up_par); F64(up_cov); F64(up_x_ref); F64(up_z_ref); F64(up_chi2); I32(up_row); I32(up_n);
  I32(mrg_best_b); I32(mrg_best_a); I32(mrg_next); I32(mrg_prev); I32(mrg_dir); F64(mrg_chi2_b);
  I32(mrg_of_track); I32(mrg_seg_start); I32(mrg_seg_idx);
  I32(rem_class); I32(rem_good_track); I32(rem_remove);
  I32(apx_best); I32(apx_partner); I32(apx_leg); F64(apx_score);
  F64(mrg_par); F64(mrg_cov); F64(mrg_x_ref); F64(mrg_z_ref); F64(mrg_chi2); I32(mrg_n_fit); I32(mrg_ndf); I32(mrg_sector); I32(mrg_n_clusters);
  F32(up_dx); F32(up_ratio); F32(up_wy); F32(up_wz); F32(dn_dx); F32(dn_ratio); F32(dn_wy); F32(dn_wz);
#undef I32
#undef F32
#undef F64
#undef U64
#undef I64
  return -1;
}

int orc_kf_propagate(const void* params, int prec, double* par, double* cov15, double x0, double x1, double* jac25) {
  const Params& P = *reinterpret_cast<const Params*>(params);
  return prec == 64 ? kf_propagate_entry<double>(P, par, cov15, x0, x1, jac25)
                    : kf_propagate_entry<float>(P, par, cov15, x0, x1, jac25);
}

void orc_kf_update(const void* params, int prec, double* par, double* cov15, double ym, double zm_rel, double* chi2) {
  const Params& P = *reinterpret_cast<const Params*>(params);
  if (prec == 64) {
    KF<double> k; load_kf(k, par, cov15, *chi2);
    kf_update<double>(k, ym, zm_rel, (double)P.err_y2, (double)P.err_z2);
    store_kf(k, par, cov15, chi2);
  } else {
    KF<float> k; load_kf(k, par, cov15, *chi2);
    kf_update<float>(k, (float)ym, (float)zm_rel, P.err_y2, P.err_z2);
    store_kf(k, par, cov15, chi2);
  }
}

int orc_kf_fit(const void* params, int prec, int npt, const double* x, const double* y, const double* z, double* par,
               double* cov15, double* chi2) {
  const Params& P = *reinterpret_cast<const Params*>(params);
  return prec == 64 ? kf_fit_entry<double>(P, npt, x, y, z, par, cov15, chi2)
                    : kf_fit_entry<float>(P, npt, x, y, z, par, cov15, chi2);
}

// S8 on the tracks of the last orc_run (last_stage >= 5)
void orc_quantise_residuals(void* h, float step_y, float step_z) { reinterpret_cast<Oracle*>(h)->quantise_residuals(step_y, step_z); }
// test entry: the scalar rule on caller-given values
void orc_quantise_values(const float* res, int64_t n, float step, int32_t* out) {
  const float inv = 1.0f / step;
  for (int64_t i = 0; i < n; ++i) out[i] = quantise_residual(res[i], inv);
}

void orc_protect(void* h, float road_y, float road_z) { reinterpret_cast<Oracle*>(h)->stage7_protect(road_y, road_z); }

// S9 on the tracks and the refit of the last orc_run (last_stage >= 6)
void orc_merge(void* h, int max_rows, int back_rows, float edge, float dz_win, float chi2_cut, float road_z0, float road_z1) {
  Oracle* o = reinterpret_cast<Oracle*>(h);
  const Oracle::MergeCuts mc{max_rows, back_rows, edge, dz_win, chi2_cut, road_z0, road_z1};
  if (o->s4_prec == 64) o->stage9<double>(mc); else o->stage9<float>(mc);
}

// apex links on the merged tracks of the last orc_merge
void orc_apex(void* h, int max_k, float min_s, float dz_win, float tol_c, float tol_z, float tol_t, float cut) {
  Oracle* o = reinterpret_cast<Oracle*>(h);
  const Oracle::ApexCuts ac{max_k, min_s, dz_win, tol_c, tol_z, tol_t, cut};
  if (o->s4_prec == 64) o->stage10<double>(ac); else o->stage10<float>(ac);
}

// strategy-A classification on the results of the last orc_merge + orc_apex
void orc_removable(void* h, float min_pt, float max_incl, float road_y, float road_z) {
  reinterpret_cast<Oracle*>(h)->stage11(min_pt, max_incl, road_y, road_z);
}

// one rotation of DESIGN.md section 3.9.2 (for the pins): par / cov15 in place, returns the new x or NaN on failure
double orc_kf_rotate(const void* params, int prec, double* par, double* cov15, double x, double sa, double ca) {
  const Params& P = *reinterpret_cast<const Params*>(params);
  const float kbf = -0.00299792458f * P.bz_tesla;
  if (prec == 64) {
    KF<double> k; load_kf(k, par, cov15, 0.0); double xn = 0;
    if (!kf_rotate<double>(k, (double)kbf, x, sa, ca, (double)P.max_sinphi, &xn)) return NAN;
    store_kf(k, par, cov15, nullptr); return xn;
  }
  KF<float> k; load_kf(k, par, cov15, 0.0); float xn = 0;
  if (!kf_rotate<float>(k, kbf, (float)x, (float)sa, (float)ca, P.max_sinphi, &xn)) return NAN;
  store_kf(k, par, cov15, nullptr); return (double)xn;
}

// S4 search of one state in row `row` of sector `sector`, on the grid of the last orc_run
// (last_stage >= 1): sorted position of the nearest gated cluster or -1.  For the pins (tests/test_oracle_search.py).
int orc_search(void* h, int prec, const double* par, const double* cov15, double zref, int sector, int row) {
  Oracle& o = *reinterpret_cast<Oracle*>(h);
  if (prec == 64) {
    KF<double> k; load_kf(k, par, cov15, 0.0);
    return o.search<double>(sector, row, k, zref);
  }
  KF<float> k; load_kf(k, par, cov15, 0.0);
  return o.search<float>(sector, row, k, (float)zref);
}

// beam-line z of one state, for the pins (prec 32 or 64)
double orc_beam_z(const void* params, int prec, double x, double y, double z, double tanl, double qpt) {
  const Params& P = *static_cast<const Params*>(params);
  const float kb = -0.00299792458f * P.bz_tesla;
  if (prec == 64) return beam_z<double>((double)kb, x, y, z, tanl, qpt);
  return (double)beam_z<float>(kb, (float)x, (float)y, (float)z, (float)tanl, (float)qpt);
}

}  // extern "C"
