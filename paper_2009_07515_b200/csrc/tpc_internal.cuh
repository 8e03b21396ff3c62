// Internal declarations shared by the CUDA translation units of libtpc_tracker.so (sm_100a only).
// Nothing here is visible across the C ABI (include/tpc_tracker.h) and nothing is shared with oracle/.
//
// Arithmetic contract: fp32, one rounding per written operation, no FMA
// contraction - every .cu file is compiled with `nvcc -fmad=false` and without --use_fast_math, so
// + - * / sqrtf floorf are IEEE-correctly rounded and the decisions (bins, windows, link choice,
// gates) come out bit-identical to any other IEEE implementation of DESIGN.md section 3.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

constexpr int kMaxRows = 256;      // row ids are uint8
constexpr int kScanTile = 2048;    // items per scan tile (256 threads x 8)

// Per-row derived tables, one stated fp32 expression each; built on the host at create.
struct RowTab {
  float x;            // row_x[r]
  float ymax;         // row_x[r] * tan_half_sector
  int ny;             // (int)floor((2*ymax)*inv_cy) + 1
  int ny_prefix;      // sum of ny over rows < r
  float up_dx[2], up_ratio[2], up_wy[2], up_wz[2];   // index k-1, k = row step 1 or 2
  float dn_dx[2], dn_ratio[2], dn_wy[2], dn_wz[2];
};
static_assert(sizeof(RowTab) == 80, "RowTab layout");

// Device counter block (lives in the workspace).  All written by kernels.
struct Counters {
  int n_bins;             // N_b
  int n_seeds;
  int n_tracklets;
  int n_tracks;
  int n_track_clusters;
  int n_linked;
  int status;             // tpc_status_bits
  int zero;               // always 0 (a device-resident "n = 0" for scans of host-known length)
  unsigned long long kf_steps;
  unsigned long long n_hits;
  int s4_ticket;          // dynamic work counter of the S4 persistent kernel
  int s1_ticket;          // dynamic (sector,row) bucket counter of the S1 bin-sort kernel
  int s1_global;          // buckets bin-sorted on the global-memory path
  int pad[1];
};

// Device counter block of the merger (S9).
struct MergeCounters {
  int n_bins;             // (sector, z) bins of the inner ends
  float inv_w;            // 1 / bin width
  int n_merged;
  int n_scan;             // n_tracks of the call (device-resident scan length)
  int status;             // != 0: the z grid could not be built
  int pad[3];
};

// Everything a kernel needs, passed by value (a few hundred bytes).
struct Ctx {
  // geometry / cuts
  int S, R, SR;
  int ny_total;                       // sum over rows of ny
  float inv_cy, inv_cz, kb;
  float err_y2, err_z2, link_T;
  int min_chain_len, max_gap, min_tracklet_hits, min_track_hits;
  float pick_chi2_cut, max_sinphi, y_margin, init_c_ss, init_c_tt, init_c_qq;
  int z_is_time; float cm_per_time_unit, drift_length;   // native time input
  int y_is_pad; const float2* padtab; // native pad input: [R] (0.5 (n_pads_r - 1), pad_pitch_r)
  const RowTab* rowtab;               // [R]
  // capacities
  int max_clusters; int max_bins; int max_seeds; int max_tracks; int max_track_clusters;
  // input of the current call
  int n;
  const uint8_t* in_sector; const uint8_t* in_row; const float* in_y; const float* in_z;
  // S1
  int* zmin_key; int* zmax_key;       // [S] order-preserving integer keys of the floats during the reduction
  float* zmin; float* zmax; int* nz;  // [S]
  int* bin_base;                      // [SR+1]
  int* row_start;                     // [SR+1]
  int* sr_count;                      // [SR] clusters per (sector,row)
  int* sr_cursor;                     // [SR] write cursor of the (sector,row) bucket during the partition
  float4* rec;                        // [n] clusters grouped by (sector,row), arrival order: (y, z, input index, rank in bin)
  float4* rec2;                       // [n] the same records grouped by (sector,row,z-slab); shares memory with the four link arrays
  int* bins;                          // [max_bins+2]; after S1 bins[0..N_b] is the CSR bin_start
  int* perm; float2* yz; uint16_t* srow;              // [n] sorted: input index, (y,z) pair, (sector << 8) | row
  int* tile_sums;                     // scan scratch
  // S2 / S3
  int* link_up_raw; int* link_dn_raw; int* link_up; int* link_dn;
  int* flag_scan;                     // [n] S3: seed bit per sorted position, then its inclusive scan
  int* seed_head; int* seed_len;      // [max_seeds]
  float4* seed_rec;                   // [max_seeds][2] (y,z) of head and next; head, next, (sector << 8 | row) of head, row of next
  // S4
  int* t_hit;                         // [max_seeds][R]
  int* t_first_row; int* t_last_row; int* t_n_hits;   // [max_seeds]
  float* t_par; float* t_cov; float* t_chi2; float* t_zref;   // [max_seeds][5], [max_seeds][15], ...
  // S5
  int* kept_scan;                     // [max_seeds] inclusive scan of kept flags
  int* tracklet_of_seed;              // [max_seeds]
  unsigned long long* owner;          // [n]
  int* k_owned; int* k_first; int* k_last;   // [max_seeds]
  int* surv_scan; int* owned_scan;    // [max_seeds] inclusive scans
  int* track_seed;                    // [max_seeds] seed of track id (S5 k_write; read by k_params and the refit)
  unsigned* own_mask; int mask_words; // [max_seeds][mask_words] bit k of word w: row first_row + 32 w + k is owned
  // S7 / S9 (per track, [max_tracks]; SoA [component][max_tracks] for par / cov)
  int* fit_row;                       // row of the state the downward refit (S7) ended on
  float* up_par; float* up_cov; float* up_chi2; float* up_x; float* up_zref; int* up_row; int* up_n;   // upward refit (3.9.1)
  int* m_sector; float* m_zin; float* m_zout;
  int max_merge_bins;
  int* m_bin_base; int* m_nzb;        // [S+1], [S]
  int* m_bin_start; int* m_bin_fill;  // [max_merge_bins+2], [max_merge_bins]
  int* m_bin_of; float4* m_rec; float4* m_srec;   // [max_tracks]: bin, inner-end record (z_in, row or -1, id, x_in), records sorted by bin
  int* m_best_b; float* m_chi_b; int* m_dir_b; unsigned long long* m_best_a;
  int* m_next; int* m_prev; int* m_dir;
  int* m_head_scan; int* m_seg_scan; int* m_head_of;
  float4* a_c4; float4* a_p4; int* a_sector; int* a_best; float* a_score;   // apex links (3.9.8), per merged track
  MergeCounters* mcnt;
  Counters* cnt;
  int n_sms;
};

// ---- host launchers, one per stage (each only enqueues kernels on `st`)
int init_s1();                                      // kernel attributes, per device (called at create)
int launch_s1(const Ctx& c, cudaStream_t st);
int launch_s2(const Ctx& c, cudaStream_t st);
int launch_s3(const Ctx& c, cudaStream_t st);
int launch_s4(const Ctx& c, cudaStream_t st);
struct OutPtrs {
  int* n_tracks; int* status; int* sector; int* first_row; int* last_row; int* n_clusters; float* par; float* cov;
  float* x_ref; float* z_ref; float* chi2; int* ndf; int* trk_cl_start; int* trk_cl_idx; int* cluster_track;
  float* z_beam;
  int max_tracks; int max_track_clusters;
};
int launch_s5(const Ctx& c, const OutPtrs& o, cudaStream_t st);
int launch_reset(const Ctx& c, cudaStream_t st);
struct FitPtrs {
  float* par; float* cov; float* x_ref; float* z_ref; float* chi2; int* ndf; int* n_fit;
  const int* trk_cl_start; float* res_y; float* res_z;   // optional (null: no residuals)
  short* qres_y; short* qres_z; float inv_step_y, inv_step_z;   // optional residual codes
  int max_tracks;
};
int launch_refit(const Ctx& c, const FitPtrs& o, cudaStream_t st);   // S7, separate call
struct MergePtrs {                    // S9: cuts + the caller's outputs
  int max_rows, back_rows; float edge, dz_win, chi2_cut, road_z0, road_z1;
  float sin_a, cos_a;                 // sine / cosine of the sector angle, host-computed in fp32
  int* n_merged; int* merged_of_track; int* seg_start; int* seg_idx;
  float* par; float* cov; float* x_ref; float* z_ref; float* chi2; int* ndf; int* n_fit; int* sector; int* n_clusters;
  int max_tracks;
};
int launch_merge(const Ctx& c, const FitPtrs& f, const MergePtrs& o, cudaStream_t st);   // S9, separate call
int launches_merge();
struct ApexPtrs {                     // apex links: cuts + the caller's outputs
  int max_k; float min_s, dz_win, tol_c, tol_z, tol_t, cut;
  int* apex_partner; int* apex_leg;
  int max_tracks;
};
int launch_apex(const Ctx& c, const MergePtrs& m, const ApexPtrs& o, cudaStream_t st);
int launches_apex();
int launch_protect(const Ctx& c, const int* cluster_track, float road_y, float road_z, unsigned char* keep, cudaStream_t st);   // S8
// the same with the mark bytes in the library's own static array (n <= TPC_PROTECT_STATIC_MAX_CLUSTERS); allocates nothing
int launch_protect_static(const Ctx& c, const int* cluster_track, float road_y, float road_z, unsigned char* keep, cudaStream_t st);
struct RemovePtrs {                   // hit removal, strategy A
  float min_pt, max_incl, road_y, road_z;
  const int* cluster_track; const int* merged_of_track; const int* apex_leg;
  const float* mrg_par; int mrg_stride; const float* fit_par; int fit_stride;
  unsigned char* cls; unsigned char* remove;
};
int launch_removable(const Ctx& c, const RemovePtrs& o, cudaStream_t st);

// In-place inclusive scan of data[0 .. *n_ptr + n_add) (int32), length known only on the device.
// max_n bounds the grid; tile_sums needs ceil(max_n / kScanTile) + 1 ints.  total_out (nullable)
// receives the grand total.  3 launches.
int launch_scan_inclusive(int* data, const int* n_ptr, int n_add, long long max_n, int* tile_sums, int* total_out,
                          int n_sms, cudaStream_t st);

// number of kernel launches per call of each launcher (kept next to the launch code)
int launches_reset(); int launches_s1(); int launches_s2(); int launches_s3(); int launches_s4(); int launches_s5();

// ---------------------------------------------------------------------------- device helpers
#ifdef __CUDACC__
// floor(v) clamped to [0, hi]; NaN and negatives -> 0
__device__ __forceinline__ int floor_clamp(float v, int hi) {
  // cvt.rmi.s32.f32 is floor() with saturation and NaN -> 0, so this is exactly
  //   f = floorf(v); !(f >= 0) ? 0 : f >= (float)hi ? hi : (int)f      (hi >= 0)
  // in three instructions
  return min(max(__float2int_rd(v), 0), hi);
}

// the pseudo-z of an input cluster of sector s whose z entry is v (cm, or time units when
// z_is_time).  -fmad=false: the product and the difference are rounded separately, like the oracle's.
__device__ __forceinline__ float input_z(const Ctx& c, int s, float v) {
  if (!c.z_is_time) return v;
  const float zc = c.drift_length - v * c.cm_per_time_unit;
  return s < (c.S >> 1) ? zc : 0.0f - zc;
}

// the sector-local y of an input cluster of row r (< R) whose y entry is v (cm, or the pad
// coordinate when y_is_pad).  -fmad=false: the difference and the product are rounded separately, like the oracle's.
__device__ __forceinline__ float input_y(const Ctx& c, int r, float v) {
  if (!c.y_is_pad) return v;
  const float2 t = __ldg(c.padtab + r);
  const float d = v - t.x;
  return d * t.y;
}

// order-preserving float <-> int key (signed compare)
__device__ __forceinline__ int float_key(float f) {
  const int i = __float_as_int(f);
  return i >= 0 ? i : i ^ 0x7FFFFFFF;
}
__device__ __forceinline__ float key_float(int k) { return __int_as_float(k >= 0 ? k : k ^ 0x7FFFFFFF); }

// The (y,z) grid of one (sector,row): what a rectangle query needs.
struct RowGrid {
  int b0;        // bin_base[s*R + t]
  int ny;        // bins along y
  int nz;        // bins along z (sector-wide)
  float ymax, zmin;
};

// Visits the sorted positions of one row whose (y,z) lies in the closed rectangle, in ascending
// position (iz ascending, then position) - the "rectangle query" of DESIGN.md section 3.1.
template <class F>
__device__ __forceinline__ void for_each_in_rect(const RowGrid& g, float inv_cy, float inv_cz,
                                                 const int* __restrict__ bin_start, const float2* __restrict__ yz,
                                                 float ylo, float yhi, float zlo, float zhi, F&& f) {
  const int iy0 = floor_clamp((ylo + g.ymax) * inv_cy, g.ny - 1);
  const int iy1 = floor_clamp((yhi + g.ymax) * inv_cy, g.ny - 1);
  const int iz0 = floor_clamp((zlo - g.zmin) * inv_cz, g.nz - 1);
  const int iz1 = floor_clamp((zhi - g.zmin) * inv_cz, g.nz - 1);
  // two bin rows per step: their four bin_start entries are loaded together and both candidate runs are walked as one
  // loop, two candidates in flight (same visiting order: row ascending, position ascending)
  for (int iz = iz0; iz <= iz1; iz += 2) {
    const int b = g.b0 + iz * g.ny;
    const bool two = iz + 1 <= iz1;
    const int jb0 = __ldg(bin_start + b + iy0), je0 = __ldg(bin_start + b + iy1 + 1);
    const int jb1 = two ? __ldg(bin_start + b + g.ny + iy0) : 0, je1 = two ? __ldg(bin_start + b + g.ny + iy1 + 1) : 0;
    const int n0 = je0 - jb0, total = n0 + (je1 - jb1);
    const int shift = jb1 - n0;                   // t >= n0: j = jb1 + (t - n0)
    for (int t = 0; t < total; t += 2) {
      const int ja = t < n0 ? jb0 + t : shift + t;
      const int jc = t + 1 < n0 ? jb0 + t + 1 : shift + t + 1;
      const float2 va = __ldg(yz + ja);
      float2 vc = va;
      if (t + 1 < total) vc = __ldg(yz + jc);
      if (va.x >= ylo && va.x <= yhi && va.y >= zlo && va.y <= zhi) f(ja, va.x, va.y);
      if (t + 1 < total && vc.x >= ylo && vc.x <= yhi && vc.y >= zlo && vc.y <= zhi) f(jc, vc.x, vc.y);
    }
  }
}
#endif

}  // namespace tpc
