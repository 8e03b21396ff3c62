// C-ABI boundary of libtpc_tracker.so (include/tpc_tracker.h): argument checks, host-side derived
// tables, workspace carving, stage orchestration on the caller's stream.  No device allocation.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <new>
#include <vector>

#include "../../include/tpc_tracker.h"
#include "tpc_internal.cuh"

using namespace tpc;

constexpr int kMaxSlots = 3;          // host_io = number of staging slots (0 none, 1 synchronous host path, 2-3 pipelined)

struct tpc_tracker {
  tpc_params_t params;            // row_x pointer is NOT kept (copied into rowtab)
  Ctx ctx;                        // pointers into the workspace; input fields set per call
  int64_t max_clusters, max_bins, max_seeds, max_tracks, max_track_clusters;
  int host_io;
  // staging for the host variants (device): slot 0 serves tpc_track_timeframe_host, slots 0 and 1 the pipelined pair
  struct Slot {
    uint8_t* sector; uint8_t* row; float* y; float* z;
    OutPtrs out;
    int64_t n;
    cudaEvent_t h2d_done, in_free, done, out_free;   // pipelined path only
    bool busy;
  } slot[kMaxSlots];
  cudaStream_t s_in, s_compute, s_out;                // pipelined path only (host_io >= 2)
  int* h_counts;                                      // pinned host: [slot][4] = n_tracks, status, n_track_clusters, -
  cudaStream_t last_stream;
  // optional CUDA graph of the S1..S5 launch sequence (tpc_tracker_enable_graph): one cached executable, replayed while the
  // call's arguments (n and every pointer) stay the same, re-captured when they change
  bool use_graph;
  cudaGraphExec_t graph_exec;
  tpc_clusters_t graph_in;
  OutPtrs graph_out;
  bool timing;
  cudaEvent_t ev[6];
  int64_t last_n;
  int64_t last_max_tracks;        // out->max_tracks of the last track call: n_tracks <= it (S5 raises TRACKS_OVERFLOW otherwise)
  // call order of the optional calls: frame_seq counts the track calls; the others remember the frame they ran on
  // (0 = never).  refit -> merge -> apex -> removable each need their predecessors to have run on the CURRENT frame,
  // because they read what those left in the workspace (fit_row, up_*, MergeCounters).
  uint64_t frame_seq, refit_seq, merge_seq, apex_seq;
};

namespace {

constexpr size_t kAlign = 256;
inline size_t up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

// Walks the workspace layout; with base == nullptr only sizes it.
struct Carver {
  char* base; size_t off;
  template <class T> T* take(size_t count) {
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += up(count * sizeof(T));
    return p;
  }
};

bool params_ok(const tpc_params_t* p) {
  if (!p || !p->row_x) return false;
  if (p->n_sectors < 1 || p->n_sectors > 256 || p->n_rows < 3 || p->n_rows > kMaxRows) return false;
  if ((int64_t)p->n_sectors * p->n_rows > 65535) return false;
  if (!(p->cell_y > 0.f) || !(p->cell_z > 0.f) || !(p->tan_half_sector > 0.f)) return false;
  if (p->min_chain_len < 2 || p->max_gap < 0) return false;
  if (p->z_is_time && (!(p->cm_per_time_unit > 0.f) || !(p->cm_per_time_unit < INFINITY) || !(std::fabs(p->drift_length) < INFINITY)))
    return false;
  if (p->y_is_pad) {
    if (!p->n_pads || !p->pad_pitch) return false;
    for (int r = 0; r < p->n_rows; ++r)
      if (p->n_pads[r] < 1 || !(p->pad_pitch[r] > 0.f) || !(p->pad_pitch[r] < INFINITY)) return false;
  }
  for (int r = 0; r < p->n_rows; ++r) {
    if (!(p->row_x[r] > 0.f)) return false;
    if (r && !(p->row_x[r] > p->row_x[r - 1])) return false;
  }
  return true;
}

void layout(tpc_tracker* t, char* base, size_t* total) {
  Carver cv{base, 0};
  Ctx& c = t->ctx;
  const size_t N = (size_t)t->max_clusters, NB = (size_t)t->max_bins, K = (size_t)t->max_seeds;
  const int S = t->params.n_sectors, R = t->params.n_rows, SR = S * R;
  c.cnt = cv.take<Counters>(1);
  c.rowtab = cv.take<RowTab>(R);
  c.padtab = cv.take<float2>(R);
  c.zmin_key = cv.take<int>(S); c.zmax_key = cv.take<int>(S);
  c.zmin = cv.take<float>(S); c.zmax = cv.take<float>(S); c.nz = cv.take<int>(S);
  c.bin_base = cv.take<int>(SR + 1); c.row_start = cv.take<int>(SR + 1);
  c.sr_count = cv.take<int>(SR); c.sr_cursor = cv.take<int>(SR);
  c.rec = cv.take<float4>(N);
  c.bins = cv.take<int>(NB + 2 + 8);
  c.perm = cv.take<int>(N); c.yz = cv.take<float2>(N); c.srow = cv.take<uint16_t>(N);
  const size_t T = (size_t)t->max_tracks;
  c.max_merge_bins = 1 << 18;                       // (sector, z) bins of the merger's inner ends (S9)
  size_t max_scan = N > NB + 2 ? N : NB + 2;
  if (K > max_scan) max_scan = K;
  if (T > max_scan) max_scan = T;
  if ((size_t)c.max_merge_bins + 2 > max_scan) max_scan = (size_t)c.max_merge_bins + 2;
  c.tile_sums = cv.take<int>(max_scan / kScanTile + 2);
  // S1's second record buffer and the four link arrays of S2/S3 are never live together: one 16 N byte slice serves both
  c.rec2 = cv.take<float4>(N);
  c.link_up_raw = base ? reinterpret_cast<int*>(c.rec2) : nullptr;
  c.link_dn_raw = base ? c.link_up_raw + N : nullptr;
  c.link_up = base ? c.link_dn_raw + N : nullptr;
  c.link_dn = base ? c.link_up + N : nullptr;
  c.flag_scan = cv.take<int>(N);
  c.seed_head = cv.take<int>(K); c.seed_len = cv.take<int>(K);
  c.seed_rec = cv.take<float4>(2 * K);
  c.t_hit = cv.take<int>(K * R);
  c.t_first_row = cv.take<int>(K); c.t_last_row = cv.take<int>(K); c.t_n_hits = cv.take<int>(K);
  c.t_par = cv.take<float>(K * 5); c.t_cov = cv.take<float>(K * 15); c.t_chi2 = cv.take<float>(K); c.t_zref = cv.take<float>(K);
  c.kept_scan = cv.take<int>(K); c.tracklet_of_seed = cv.take<int>(K);
  c.owner = cv.take<unsigned long long>(N);
  c.k_owned = cv.take<int>(K); c.k_first = cv.take<int>(K); c.k_last = cv.take<int>(K);
  c.surv_scan = cv.take<int>(K); c.owned_scan = cv.take<int>(K);
  c.track_seed = cv.take<int>(K);
  c.mask_words = (R + 31) / 32;
  c.own_mask = cv.take<unsigned>(K * (size_t)c.mask_words);
  // S7 / S9: per track
  c.fit_row = cv.take<int>(T);
  c.up_par = cv.take<float>(5 * T); c.up_cov = cv.take<float>(15 * T); c.up_chi2 = cv.take<float>(T);
  c.up_x = cv.take<float>(T); c.up_zref = cv.take<float>(T); c.up_row = cv.take<int>(T); c.up_n = cv.take<int>(T);
  c.m_sector = cv.take<int>(T); c.m_zin = cv.take<float>(T); c.m_zout = cv.take<float>(T);
  c.m_bin_base = cv.take<int>(S + 1); c.m_nzb = cv.take<int>(S);
  c.m_bin_start = cv.take<int>((size_t)c.max_merge_bins + 2); c.m_bin_fill = cv.take<int>((size_t)c.max_merge_bins);
  c.m_bin_of = cv.take<int>(T); c.m_rec = cv.take<float4>(T); c.m_srec = cv.take<float4>(T);
  c.m_best_b = cv.take<int>(T); c.m_chi_b = cv.take<float>(T); c.m_dir_b = cv.take<int>(T);
  c.m_best_a = cv.take<unsigned long long>(T);
  c.m_next = cv.take<int>(T); c.m_prev = cv.take<int>(T); c.m_dir = cv.take<int>(T);
  c.m_head_scan = cv.take<int>(T); c.m_seg_scan = cv.take<int>(T); c.m_head_of = cv.take<int>(T);
  c.a_c4 = cv.take<float4>(T); c.a_p4 = cv.take<float4>(T); c.a_sector = cv.take<int>(T); c.a_best = cv.take<int>(T);
  c.a_score = cv.take<float>(T);
  c.mcnt = cv.take<MergeCounters>(1);
  for (int k = 0; k < t->host_io; ++k) {
    const size_t TC = (size_t)t->max_track_clusters;
    tpc_tracker::Slot& sl = t->slot[k];
    sl.sector = cv.take<uint8_t>(N); sl.row = cv.take<uint8_t>(N);
    sl.y = cv.take<float>(N); sl.z = cv.take<float>(N);
    OutPtrs& o = sl.out;
    o.n_tracks = cv.take<int>(1); o.status = cv.take<int>(1);
    o.sector = cv.take<int>(T); o.first_row = cv.take<int>(T); o.last_row = cv.take<int>(T); o.n_clusters = cv.take<int>(T);
    o.par = cv.take<float>(T * 5); o.cov = cv.take<float>(T * 15);
    o.x_ref = cv.take<float>(T); o.z_ref = cv.take<float>(T); o.chi2 = cv.take<float>(T); o.ndf = cv.take<int>(T);
    o.trk_cl_start = cv.take<int>(T + 1); o.trk_cl_idx = cv.take<int>(TC); o.cluster_track = cv.take<int>(N);
    o.z_beam = cv.take<float>(T);
    o.max_tracks = (int)T; o.max_track_clusters = (int)TC;
  }
  *total = cv.off;
}

bool caps_ok(int64_t max_clusters, int64_t max_bins, int64_t max_seeds, int64_t max_tracks, int64_t max_track_clusters) {
  const int64_t lim = 2147483647LL - 16;
  return max_clusters >= 1 && max_clusters <= lim && max_bins >= 1 && max_bins <= lim && max_seeds >= 1 &&
         max_seeds <= lim && max_tracks >= 1 && max_tracks <= lim && max_track_clusters >= 1 && max_track_clusters <= lim;
}

void fill_ctx_constants(tpc_tracker* t, std::vector<RowTab>& tab) {
  const tpc_params_t& p = t->params;
  Ctx& c = t->ctx;
  const int R = p.n_rows;
  c.S = p.n_sectors; c.R = R; c.SR = p.n_sectors * R;
  // each a single fp32 expression, DESIGN.md section 3.0
  c.kb = -0.00299792458f * p.bz_tesla;
  c.inv_cy = 1.0f / p.cell_y;
  c.inv_cz = 1.0f / p.cell_z;
  c.err_y2 = p.err_y2; c.err_z2 = p.err_z2; c.link_T = p.link_T;
  c.min_chain_len = p.min_chain_len; c.max_gap = p.max_gap;
  c.min_tracklet_hits = p.min_tracklet_hits; c.min_track_hits = p.min_track_hits;
  c.pick_chi2_cut = p.pick_chi2_cut; c.max_sinphi = p.max_sinphi; c.y_margin = p.y_margin;
  c.init_c_ss = p.init_c_ss; c.init_c_tt = p.init_c_tt; c.init_c_qq = p.init_c_qq;
  c.z_is_time = p.z_is_time != 0; c.cm_per_time_unit = p.cm_per_time_unit; c.drift_length = p.drift_length;
  tab.assign(R, RowTab{});
  int acc = 0;
  for (int r = 0; r < R; ++r) {
    RowTab& e = tab[r];
    e.x = p.row_x[r];
    e.ymax = p.row_x[r] * p.tan_half_sector;
    e.ny = (int)std::floor((2.0f * e.ymax) * c.inv_cy) + 1;
    e.ny_prefix = acc;
    acc += e.ny;
    for (int k = 1; k <= 2; ++k) {
      if (r + k < R) {
        const float dx = p.row_x[r + k] - p.row_x[r];
        e.up_dx[k - 1] = dx;
        e.up_ratio[k - 1] = p.row_x[r + k] / p.row_x[r];
        e.up_wy[k - 1] = p.link_ay * dx + p.link_b;
        e.up_wz[k - 1] = p.link_az * dx + p.link_b;
      }
      if (r - k >= 0) {
        const float dx = p.row_x[r] - p.row_x[r - k];
        e.dn_dx[k - 1] = dx;
        e.dn_ratio[k - 1] = p.row_x[r - k] / p.row_x[r];
        e.dn_wy[k - 1] = p.link_ay * dx + p.link_b;
        e.dn_wz[k - 1] = p.link_az * dx + p.link_b;
      }
    }
  }
  c.ny_total = acc;
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int run_device(tpc_tracker* t, const tpc_clusters_t* in, const OutPtrs& o, cudaStream_t st, cudaEvent_t after_s1 = nullptr) {
  Ctx& c = t->ctx;
  c.n = (int)in->n;
  c.in_sector = in->sector; c.in_row = in->row; c.in_y = in->y; c.in_z = in->z;
  t->last_stream = st;
  t->last_n = in->n;
  t->last_max_tracks = o.max_tracks;
  ++t->frame_seq;
  const bool tm = t->timing;
  if (tm) cudaEventRecord(t->ev[0], st);
  if (launch_reset(c, st)) return TPC_ERR_CUDA;
  if (launch_s1(c, st)) return TPC_ERR_CUDA;
  if (after_s1) cudaEventRecord(after_s1, st);     // the input arrays are not read again
  if (tm) cudaEventRecord(t->ev[1], st);
  if (launch_s2(c, st)) return TPC_ERR_CUDA;
  if (tm) cudaEventRecord(t->ev[2], st);
  if (launch_s3(c, st)) return TPC_ERR_CUDA;
  if (tm) cudaEventRecord(t->ev[3], st);
  if (launch_s4(c, st)) return TPC_ERR_CUDA;
  if (tm) cudaEventRecord(t->ev[4], st);
  if (launch_s5(c, o, st)) return TPC_ERR_CUDA;
  if (tm) cudaEventRecord(t->ev[5], st);
  return cudaGetLastError() == cudaSuccess ? TPC_OK : TPC_ERR_CUDA;
}

// host outputs may leave cluster_track NULL: it is then not copied back (it is recomputable from the CSR)
bool out_ok(const tpc_tracks_t* o, bool host = false) {
  return o && o->n_tracks && o->status && o->sector && o->first_row && o->last_row && o->n_clusters && o->par && o->cov &&
         o->x_ref && o->z_ref && o->chi2 && o->ndf && o->trk_cl_start && o->trk_cl_idx && (host || o->cluster_track) && o->z_beam &&
         o->max_tracks >= 1 && o->max_track_clusters >= 1;
}

OutPtrs to_out(const tpc_tracks_t* o) {
  OutPtrs r;
  r.n_tracks = o->n_tracks; r.status = o->status; r.sector = o->sector; r.first_row = o->first_row;
  r.last_row = o->last_row; r.n_clusters = o->n_clusters; r.par = o->par; r.cov = o->cov; r.x_ref = o->x_ref;
  r.z_ref = o->z_ref; r.chi2 = o->chi2; r.ndf = o->ndf; r.trk_cl_start = o->trk_cl_start; r.trk_cl_idx = o->trk_cl_idx;
  r.cluster_track = o->cluster_track; r.z_beam = o->z_beam; r.max_tracks = (int)o->max_tracks; r.max_track_clusters = (int)o->max_track_clusters;
  return r;
}

// D2H of exactly the tracks found (T tracks, n_tc attached clusters) from the staging outputs `o` to the caller's HOST
// buffers, enqueued on `st`.
bool copy_tracks_d2h(const OutPtrs& o, const tpc_tracks_t* out, size_t n, size_t T, size_t n_tc, cudaStream_t st) {
  const size_t mt = (size_t)out->max_tracks;
  auto d2h = [&](void* dst, const void* src, size_t bytes) {
    return bytes == 0 || cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  };
  bool ok = true;
  if (T) {
    ok = d2h(out->sector, o.sector, T * 4) && d2h(out->first_row, o.first_row, T * 4) &&
         d2h(out->last_row, o.last_row, T * 4) && d2h(out->n_clusters, o.n_clusters, T * 4) &&
         d2h(out->x_ref, o.x_ref, T * 4) && d2h(out->z_ref, o.z_ref, T * 4) && d2h(out->chi2, o.chi2, T * 4) &&
         d2h(out->ndf, o.ndf, T * 4) && d2h(out->z_beam, o.z_beam, T * 4) &&
         d2h(out->trk_cl_start, o.trk_cl_start, (T + 1) * 4);
    for (int i = 0; i < 5 && ok; ++i) ok = d2h(out->par + i * mt, o.par + i * mt, T * 4);
    for (int i = 0; i < 15 && ok; ++i) ok = d2h(out->cov + i * mt, o.cov + i * mt, T * 4);
    ok = ok && d2h(out->trk_cl_idx, o.trk_cl_idx, n_tc * 4);
  } else {
    out->trk_cl_start[0] = 0;
  }
  return ok && (!out->cluster_track || d2h(out->cluster_track, o.cluster_track, n * 4));
}

}  // namespace

extern "C" {

size_t tpc_tracker_workspace_bytes(const tpc_params_t* params, int64_t max_clusters, int64_t max_bins, int64_t max_seeds,
                                   int64_t max_tracks, int64_t max_track_clusters, int32_t host_io) {
  if (!params_ok(params) || !caps_ok(max_clusters, max_bins, max_seeds, max_tracks, max_track_clusters)) return 0;
  if (host_io < 0 || host_io > kMaxSlots) return 0;
  tpc_tracker tmp{};
  tmp.params = *params;
  tmp.max_clusters = max_clusters; tmp.max_bins = max_bins; tmp.max_seeds = max_seeds;
  tmp.max_tracks = max_tracks; tmp.max_track_clusters = max_track_clusters; tmp.host_io = host_io;
  size_t total = 0;
  layout(&tmp, nullptr, &total);
  return total;
}

int tpc_tracker_create(const tpc_params_t* params, int64_t max_clusters, int64_t max_bins, int64_t max_seeds,
                       int64_t max_tracks, int64_t max_track_clusters, int32_t host_io, void* d_workspace,
                       size_t workspace_bytes, tpc_tracker_t** out) {
  if (!out) return TPC_ERR_INVALID_ARG;
  *out = nullptr;
  if (!params_ok(params) || !caps_ok(max_clusters, max_bins, max_seeds, max_tracks, max_track_clusters)) return TPC_ERR_INVALID_ARG;
  if (host_io < 0 || host_io > kMaxSlots) return TPC_ERR_INVALID_ARG;
  if (!d_workspace || !aligned(d_workspace, kAlign)) return TPC_ERR_INVALID_ARG;
  tpc_tracker* t = new (std::nothrow) tpc_tracker{};
  if (!t) return TPC_ERR_INVALID_ARG;
  t->params = *params;
  t->max_clusters = max_clusters; t->max_bins = max_bins; t->max_seeds = max_seeds;
  t->max_tracks = max_tracks; t->max_track_clusters = max_track_clusters; t->host_io = host_io;
  size_t total = 0;
  layout(t, static_cast<char*>(d_workspace), &total);
  if (total > workspace_bytes) { delete t; return TPC_ERR_CAPACITY; }   // nothing but the host struct exists yet
  std::vector<RowTab> tab;
  fill_ctx_constants(t, tab);
  // native pad input: per row the half pad count (exact in fp32) and the pitch
  std::vector<float2> padtab((size_t)params->n_rows, make_float2(0.f, 1.f));
  t->ctx.y_is_pad = params->y_is_pad != 0;
  if (params->y_is_pad)
    for (int r = 0; r < params->n_rows; ++r) padtab[r] = make_float2(0.5f * (float)(params->n_pads[r] - 1), params->pad_pitch[r]);
  t->params.row_x = nullptr; t->params.n_pads = nullptr; t->params.pad_pitch = nullptr;   // the caller's tables are not kept
  Ctx& c = t->ctx;
  c.max_clusters = (int)max_clusters; c.max_bins = (int)max_bins; c.max_seeds = (int)max_seeds;
  c.max_tracks = (int)max_tracks; c.max_track_clusters = (int)max_track_clusters;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    delete t; return TPC_ERR_CUDA;
  }
  c.n_sms = sms;
  if (init_s1()) { delete t; return TPC_ERR_CUDA; }
  if (cudaMemcpy(const_cast<RowTab*>(c.rowtab), tab.data(), tab.size() * sizeof(RowTab), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(const_cast<float2*>(c.padtab), padtab.data(), padtab.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemset(c.cnt, 0, sizeof(Counters)) != cudaSuccess || cudaMemset(c.mcnt, 0, sizeof(MergeCounters)) != cudaSuccess) {
    delete t; return TPC_ERR_CUDA;
  }
  // from here on a failure goes through tpc_tracker_destroy, which releases whatever was created so far
  for (auto& e : t->ev)
    if (cudaEventCreate(&e) != cudaSuccess) { tpc_tracker_destroy(t); return TPC_ERR_CUDA; }
  if (host_io >= 2) {
    bool ok = cudaStreamCreateWithFlags(&t->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&t->s_compute, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&t->s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaHostAlloc(reinterpret_cast<void**>(&t->h_counts), 4 * kMaxSlots * sizeof(int), cudaHostAllocDefault) == cudaSuccess;
    for (auto& sl : t->slot)
      for (cudaEvent_t* e : {&sl.h2d_done, &sl.in_free, &sl.done, &sl.out_free})
        ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { tpc_tracker_destroy(t); return TPC_ERR_CUDA; }
  }
  *out = t;
  return TPC_OK;
}

int tpc_track_timeframe(tpc_tracker_t* t, const tpc_clusters_t* in, const tpc_tracks_t* out, void* cuda_stream) {
  if (!t || !in || !out_ok(out)) return TPC_ERR_INVALID_ARG;
  if (in->n < 0 || (in->n > 0 && (!in->sector || !in->row || !in->y || !in->z))) return TPC_ERR_INVALID_ARG;
  if (in->n > t->max_clusters || out->max_tracks > t->max_tracks || out->max_track_clusters > t->max_track_clusters)
    return TPC_ERR_CAPACITY;
  if (!aligned(in->sector, 4) || !aligned(in->row, 4) || !aligned(in->z, 16) || !aligned(in->y, 16)) return TPC_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const OutPtrs o = to_out(out);
  if (!t->use_graph || t->timing || st == nullptr) return run_device(t, in, o, st);   // (the legacy default stream cannot capture)
  // a stream the caller is already capturing (the framework around the tracker records its own graph): a second
  // BeginCapture would fail and could invalidate that capture - enqueue the plain launches into the caller's graph instead
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); return TPC_ERR_CUDA; }
  if (cap != cudaStreamCaptureStatusNone) return run_device(t, in, o, st);
  const bool same = t->graph_exec && t->graph_in.n == in->n && t->graph_in.sector == in->sector && t->graph_in.row == in->row &&
                    t->graph_in.y == in->y && t->graph_in.z == in->z && std::memcmp(&t->graph_out, &o, sizeof(OutPtrs)) == 0;
  if (!same) {
    if (t->graph_exec) { cudaGraphExecDestroy(t->graph_exec); t->graph_exec = nullptr; }
    cudaGraph_t g = nullptr;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return TPC_ERR_CUDA;
    const int rc = run_device(t, in, o, st);
    const cudaError_t ce = cudaStreamEndCapture(st, &g);
    if (rc != TPC_OK || ce != cudaSuccess || !g) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return rc != TPC_OK ? rc : TPC_ERR_CUDA; }
    const cudaError_t ie = cudaGraphInstantiate(&t->graph_exec, g, 0);
    cudaGraphDestroy(g);
    if (ie != cudaSuccess) { t->graph_exec = nullptr; return TPC_ERR_CUDA; }
    t->graph_in = *in; t->graph_out = o;
  }
  t->last_stream = st; t->last_n = in->n; t->last_max_tracks = o.max_tracks;
  ++t->frame_seq;
  t->ctx.n = (int)in->n;
  t->ctx.in_sector = in->sector; t->ctx.in_row = in->row; t->ctx.in_y = in->y; t->ctx.in_z = in->z;
  return cudaGraphLaunch(t->graph_exec, st) == cudaSuccess ? TPC_OK : TPC_ERR_CUDA;
}

int tpc_tracker_enable_graph(tpc_tracker_t* t, int32_t enable) {
  if (!t) return TPC_ERR_INVALID_ARG;
  t->use_graph = enable != 0;
  if (!t->use_graph && t->graph_exec) { cudaGraphExecDestroy(t->graph_exec); t->graph_exec = nullptr; }
  return TPC_OK;
}

int tpc_track_timeframe_host(tpc_tracker_t* t, const tpc_clusters_t* in, const tpc_tracks_t* out, void* cuda_stream) {
  if (!t || !in || !out_ok(out, true) || !t->host_io) return TPC_ERR_INVALID_ARG;
  if (in->n < 0 || (in->n > 0 && (!in->sector || !in->row || !in->y || !in->z))) return TPC_ERR_INVALID_ARG;
  if (in->n > t->max_clusters || out->max_tracks > t->max_tracks || out->max_track_clusters > t->max_track_clusters)
    return TPC_ERR_CAPACITY;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t n = (size_t)in->n;
  tpc_clusters_t d = *in;
  tpc_tracker::Slot& sl = t->slot[0];
  d.sector = sl.sector; d.row = sl.row; d.y = sl.y; d.z = sl.z; d.x = nullptr;
  if (n) {
    if (cudaMemcpyAsync(sl.sector, in->sector, n, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(sl.row, in->row, n, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(sl.y, in->y, n * 4, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(sl.z, in->z, n * 4, cudaMemcpyHostToDevice, st) != cudaSuccess)
      return TPC_ERR_CUDA;
  }
  OutPtrs o = sl.out;
  o.max_tracks = (int)out->max_tracks; o.max_track_clusters = (int)out->max_track_clusters;
  const int rc = run_device(t, &d, o, st);
  if (rc != TPC_OK) return rc;
  // counts first, then exactly the tracks found
  int head[2] = {0, 0};
  if (cudaMemcpyAsync(&head[0], o.n_tracks, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(&head[1], o.status, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return TPC_ERR_CUDA;
  *out->n_tracks = head[0]; *out->status = head[1];
  int n_tc = 0;
  if (head[0] && (cudaMemcpyAsync(&n_tc, &t->ctx.cnt->n_track_clusters, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                  cudaStreamSynchronize(st) != cudaSuccess))
    return TPC_ERR_CUDA;
  if (!copy_tracks_d2h(o, out, n, (size_t)head[0], (size_t)n_tc, st) || cudaStreamSynchronize(st) != cudaSuccess) return TPC_ERR_CUDA;
  return TPC_OK;
}

// ---- pipelined host path (host_io = 2 or 3 staging slots): H2D of frame i+1 and D2H of frame i-1 overlap the
// kernels of frame i (with 3 slots the next upload does not have to wait for the previous download to be collected).
// Three library-owned streams; two staging slots; events order the reuse of a slot's input staging (free once S1 of
// the frame that used it has run), of its output staging (free once its D2H has finished) and of the single workspace
// (frames compute one after the other on s_compute).
int tpc_track_timeframe_host_begin(tpc_tracker_t* t, const tpc_clusters_t* in, int32_t slot) {
  if (!t || !in || t->host_io < 2 || slot < 0 || slot >= t->host_io) return TPC_ERR_INVALID_ARG;
  if (in->n < 0 || (in->n > 0 && (!in->sector || !in->row || !in->y || !in->z))) return TPC_ERR_INVALID_ARG;
  if (in->n > t->max_clusters) return TPC_ERR_CAPACITY;
  tpc_tracker::Slot& sl = t->slot[slot];
  if (sl.busy) return TPC_ERR_INVALID_ARG;          // begin / end must alternate per slot
  const size_t n = (size_t)in->n;
  sl.n = in->n;
  // A failure after something was enqueued must not leave copies or kernels in flight on a slot the caller believes
  // free (a retry would overwrite staging that is still being read): drain the library's streams before returning.
  auto fail = [&](int code) {
    cudaStreamSynchronize(t->s_in); cudaStreamSynchronize(t->s_compute);
    return code;
  };
  if (cudaStreamWaitEvent(t->s_in, sl.in_free, 0) != cudaSuccess) return TPC_ERR_CUDA;
  if (n) {
    if (cudaMemcpyAsync(sl.sector, in->sector, n, cudaMemcpyHostToDevice, t->s_in) != cudaSuccess ||
        cudaMemcpyAsync(sl.row, in->row, n, cudaMemcpyHostToDevice, t->s_in) != cudaSuccess ||
        cudaMemcpyAsync(sl.y, in->y, n * 4, cudaMemcpyHostToDevice, t->s_in) != cudaSuccess ||
        cudaMemcpyAsync(sl.z, in->z, n * 4, cudaMemcpyHostToDevice, t->s_in) != cudaSuccess)
      return fail(TPC_ERR_CUDA);
  }
  if (cudaEventRecord(sl.h2d_done, t->s_in) != cudaSuccess ||
      cudaStreamWaitEvent(t->s_compute, sl.h2d_done, 0) != cudaSuccess ||
      cudaStreamWaitEvent(t->s_compute, sl.out_free, 0) != cudaSuccess)
    return fail(TPC_ERR_CUDA);
  tpc_clusters_t d = *in;
  d.sector = sl.sector; d.row = sl.row; d.y = sl.y; d.z = sl.z; d.x = nullptr;
  const int rc = run_device(t, &d, sl.out, t->s_compute, sl.in_free);
  if (rc != TPC_OK) return fail(rc);
  int* hc = t->h_counts + 4 * slot;
  if (cudaMemcpyAsync(hc + 0, sl.out.n_tracks, 4, cudaMemcpyDeviceToHost, t->s_compute) != cudaSuccess ||
      cudaMemcpyAsync(hc + 1, sl.out.status, 4, cudaMemcpyDeviceToHost, t->s_compute) != cudaSuccess ||
      cudaMemcpyAsync(hc + 2, &t->ctx.cnt->n_track_clusters, 4, cudaMemcpyDeviceToHost, t->s_compute) != cudaSuccess ||
      cudaEventRecord(sl.done, t->s_compute) != cudaSuccess)
    return fail(TPC_ERR_CUDA);
  sl.busy = true;
  return TPC_OK;
}

int tpc_track_timeframe_host_end(tpc_tracker_t* t, const tpc_tracks_t* out, int32_t slot) {
  if (!t || !out_ok(out, true) || t->host_io < 2 || slot < 0 || slot >= t->host_io) return TPC_ERR_INVALID_ARG;
  tpc_tracker::Slot& sl = t->slot[slot];
  if (!sl.busy) return TPC_ERR_INVALID_ARG;
  if (out->max_tracks != t->max_tracks || out->max_track_clusters != t->max_track_clusters) return TPC_ERR_INVALID_ARG;
  if (cudaEventSynchronize(sl.done) != cudaSuccess) return TPC_ERR_CUDA;
  const int* hc = t->h_counts + 4 * slot;
  *out->n_tracks = hc[0]; *out->status = hc[1];
  const bool ok = copy_tracks_d2h(sl.out, out, (size_t)sl.n, (size_t)hc[0], (size_t)hc[2], t->s_out);
  if (!ok || cudaEventRecord(sl.out_free, t->s_out) != cudaSuccess || cudaStreamSynchronize(t->s_out) != cudaSuccess)
    return TPC_ERR_CUDA;
  sl.busy = false;
  return TPC_OK;
}

int tpc_tracker_refit(tpc_tracker_t* t, const tpc_fit_t* out, void* cuda_stream) {
  if (!t || !out || !out->par || !out->cov || !out->x_ref || !out->z_ref || !out->chi2 || !out->ndf || !out->n_fit)
    return TPC_ERR_INVALID_ARG;
  // room for every track the last frame can have found (its out->max_tracks): nothing is ever cut off silently
  if (out->max_tracks < 1 || out->max_tracks > t->max_tracks || out->max_tracks < t->last_max_tracks) return TPC_ERR_CAPACITY;
  FitPtrs o;
  o.par = out->par; o.cov = out->cov; o.x_ref = out->x_ref; o.z_ref = out->z_ref; o.chi2 = out->chi2; o.ndf = out->ndf;
  o.n_fit = out->n_fit; o.max_tracks = (int)out->max_tracks;
  const int nres = (out->trk_cl_start != nullptr) + (out->res_y != nullptr) + (out->res_z != nullptr);
  if (nres != 0 && nres != 3) return TPC_ERR_INVALID_ARG;
  o.trk_cl_start = out->trk_cl_start; o.res_y = out->res_y; o.res_z = out->res_z;
  // residual codes: both or none, only next to the residuals, steps finite and > 0
  const int nq = (out->qres_y != nullptr) + (out->qres_z != nullptr);
  if (nq == 1 || (nq == 2 && nres != 3)) return TPC_ERR_INVALID_ARG;
  o.qres_y = nullptr; o.qres_z = nullptr; o.inv_step_y = 0.f; o.inv_step_z = 0.f;
  if (nq == 2) {
    if (!(out->res_step_y > 0.f) || !(out->res_step_y < INFINITY) || !(out->res_step_z > 0.f) || !(out->res_step_z < INFINITY))
      return TPC_ERR_INVALID_ARG;
    o.qres_y = out->qres_y; o.qres_z = out->qres_z;
    o.inv_step_y = 1.0f / out->res_step_y; o.inv_step_z = 1.0f / out->res_step_z;   // one fp32 division each
  }
  if (!t->frame_seq) return TPC_ERR_INVALID_ARG;      // no frame tracked yet
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  if (launch_refit(t->ctx, o, st)) return TPC_ERR_CUDA;
  t->refit_seq = t->frame_seq;
  return TPC_OK;
}

int tpc_tracker_merge(tpc_tracker_t* t, const tpc_fit_t* fit, const tpc_merge_cuts_t* cuts, const tpc_merged_t* out,
                      void* cuda_stream) {
  if (!t || !fit || !cuts || !out) return TPC_ERR_INVALID_ARG;
  if (!fit->par || !fit->cov || !fit->x_ref || !fit->z_ref || !fit->n_fit) return TPC_ERR_INVALID_ARG;
  if (!out->n_merged || !out->merged_of_track || !out->seg_start || !out->seg_idx || !out->par || !out->cov || !out->x_ref ||
      !out->z_ref || !out->chi2 || !out->ndf || !out->n_fit || !out->sector || !out->n_clusters)
    return TPC_ERR_INVALID_ARG;
  if (cuts->max_rows < 0 || cuts->back_rows < 0 || !(cuts->edge >= 0.f) || !(cuts->dz_win > 0.f) || !(cuts->dz_win < INFINITY) ||
      !(cuts->chi2_cut >= 0.f) || !(cuts->road_z0 >= 0.f) || !(cuts->road_z1 >= 0.f))
    return TPC_ERR_INVALID_ARG;
  if (fit->max_tracks < 1 || fit->max_tracks > t->max_tracks || out->max_tracks < 1 || out->max_tracks > t->max_tracks)
    return TPC_ERR_CAPACITY;
  // the kernels index `fit` and `out` by track id up to n_tracks: both must hold every track of the last frame
  if (fit->max_tracks < t->last_max_tracks || out->max_tracks < t->last_max_tracks) return TPC_ERR_CAPACITY;
  FitPtrs f{};
  f.par = fit->par; f.cov = fit->cov; f.x_ref = fit->x_ref; f.z_ref = fit->z_ref; f.chi2 = fit->chi2; f.ndf = fit->ndf;
  f.n_fit = fit->n_fit; f.max_tracks = (int)fit->max_tracks;
  MergePtrs o{};
  o.max_rows = cuts->max_rows; o.back_rows = cuts->back_rows; o.edge = cuts->edge; o.dz_win = cuts->dz_win; o.chi2_cut = cuts->chi2_cut;
  o.road_z0 = cuts->road_z0; o.road_z1 = cuts->road_z1;
  // sine and cosine of the sector angle from tan_half_sector alone, fp32, one rounding per operation
  const float th = t->params.tan_half_sector;
  const float den = 1.0f + th * th;
  o.sin_a = (2.0f * th) / den; o.cos_a = (1.0f - th * th) / den;
  o.n_merged = out->n_merged; o.merged_of_track = out->merged_of_track; o.seg_start = out->seg_start; o.seg_idx = out->seg_idx;
  o.par = out->par; o.cov = out->cov; o.x_ref = out->x_ref; o.z_ref = out->z_ref; o.chi2 = out->chi2; o.ndf = out->ndf;
  o.n_fit = out->n_fit; o.sector = out->sector; o.n_clusters = out->n_clusters; o.max_tracks = (int)out->max_tracks;
  if (!t->frame_seq || t->refit_seq != t->frame_seq) return TPC_ERR_INVALID_ARG;   // needs the refit of THIS frame
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  if (launch_merge(t->ctx, f, o, st)) return TPC_ERR_CUDA;
  t->merge_seq = t->frame_seq;
  return TPC_OK;
}

int tpc_tracker_apex(tpc_tracker_t* t, const tpc_merged_t* merged, const tpc_apex_cuts_t* cuts, const tpc_apex_t* out,
                     void* cuda_stream) {
  if (!t || !merged || !cuts || !out || !merged->seg_start || !merged->seg_idx || !out->apex_partner || !out->apex_leg)
    return TPC_ERR_INVALID_ARG;
  if (cuts->max_k < 0 || !(cuts->min_s >= 0.f) || !(cuts->dz_win > 0.f) || !(cuts->dz_win < INFINITY) || !(cuts->tol_c > 0.f) ||
      !(cuts->tol_z > 0.f) || !(cuts->tol_t > 0.f) || !(cuts->cut >= 0.f))
    return TPC_ERR_INVALID_ARG;
  if (out->max_tracks < 1 || out->max_tracks > t->max_tracks || merged->max_tracks < 1 || merged->max_tracks > t->max_tracks)
    return TPC_ERR_CAPACITY;
  // entries [0, n_merged) are read / written and n_merged <= n_tracks <= the last frame's max_tracks
  if (out->max_tracks < t->last_max_tracks || merged->max_tracks < t->last_max_tracks) return TPC_ERR_CAPACITY;
  MergePtrs m{};
  const float th = t->params.tan_half_sector;
  const float den = 1.0f + th * th;
  m.sin_a = (2.0f * th) / den; m.cos_a = (1.0f - th * th) / den;
  m.seg_start = merged->seg_start; m.seg_idx = merged->seg_idx; m.max_tracks = (int)merged->max_tracks;
  ApexPtrs o{};
  o.max_k = cuts->max_k; o.min_s = cuts->min_s; o.dz_win = cuts->dz_win; o.tol_c = cuts->tol_c; o.tol_z = cuts->tol_z;
  o.tol_t = cuts->tol_t; o.cut = cuts->cut;
  o.apex_partner = out->apex_partner; o.apex_leg = out->apex_leg; o.max_tracks = (int)out->max_tracks;
  if (!t->frame_seq || t->merge_seq != t->frame_seq) return TPC_ERR_INVALID_ARG;   // needs the merge of THIS frame
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  if (launch_apex(t->ctx, m, o, st)) return TPC_ERR_CUDA;
  t->apex_seq = t->frame_seq;
  return TPC_OK;
}

int tpc_tracker_removable(tpc_tracker_t* t, const int32_t* cluster_track, const tpc_fit_t* fit, const tpc_merged_t* merged,
                          const tpc_apex_t* apex, const tpc_removal_cuts_t* cuts, uint8_t* cls, uint8_t* remove, void* cuda_stream) {
  if (!t || !cluster_track || !fit || !merged || !apex || !cuts || !cls || !remove) return TPC_ERR_INVALID_ARG;
  if (!fit->par || !merged->merged_of_track || !merged->par || !apex->apex_leg) return TPC_ERR_INVALID_ARG;
  if (!(cuts->min_pt >= 0.f) || !(cuts->max_incl >= 0.f) || !(cuts->road_y >= 0.f) || !(cuts->road_z >= 0.f)) return TPC_ERR_INVALID_ARG;
  if (fit->max_tracks > t->max_tracks || merged->max_tracks > t->max_tracks || fit->max_tracks < 1 || merged->max_tracks < 1 ||
      apex->max_tracks < 1 || apex->max_tracks > t->max_tracks)
    return TPC_ERR_CAPACITY;
  if (fit->max_tracks < t->last_max_tracks || merged->max_tracks < t->last_max_tracks || apex->max_tracks < t->last_max_tracks)
    return TPC_ERR_CAPACITY;
  RemovePtrs o{};
  o.min_pt = cuts->min_pt; o.max_incl = cuts->max_incl; o.road_y = cuts->road_y; o.road_z = cuts->road_z;
  o.cluster_track = cluster_track; o.merged_of_track = merged->merged_of_track; o.apex_leg = apex->apex_leg;
  o.mrg_par = merged->par; o.mrg_stride = (int)merged->max_tracks; o.fit_par = fit->par; o.fit_stride = (int)fit->max_tracks;
  o.cls = cls; o.remove = remove;
  if (!t->frame_seq || t->merge_seq != t->frame_seq || t->apex_seq != t->frame_seq) return TPC_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  return launch_removable(t->ctx, o, st) ? TPC_ERR_CUDA : TPC_OK;
}

int tpc_tracker_protect(tpc_tracker_t* t, const int32_t* cluster_track, float road_y, float road_z, uint8_t* keep,
                        void* cuda_stream) {
  if (!t || !keep || !cluster_track || !(road_y >= 0.f) || !(road_z >= 0.f)) return TPC_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  return launch_protect(t->ctx, cluster_track, road_y, road_z, keep, st) ? TPC_ERR_CUDA : TPC_OK;
}

// Strategy-B protection with the mark bytes in the static array of s8_protect.cu (see the header): no cudaMalloc / cudaFree,
// no workspace scratch.  The size check comes first so that an oversized frame enqueues nothing.
int tpc_tracker_protect_static(tpc_tracker_t* t, const int32_t* cluster_track, float road_y, float road_z, uint8_t* keep,
                               void* cuda_stream) {
  if (!t || !keep || !cluster_track || !(road_y >= 0.f) || !(road_z >= 0.f)) return TPC_ERR_INVALID_ARG;
  if (t->last_n > (int64_t)TPC_PROTECT_STATIC_MAX_CLUSTERS) return TPC_ERR_STATIC_SCRATCH;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  t->last_stream = st;
  return launch_protect_static(t->ctx, cluster_track, road_y, road_z, keep, st) ? TPC_ERR_CUDA : TPC_OK;
}

int tpc_tracker_counters(tpc_tracker_t* t, tpc_counters_t* out) {
  if (!t || !out) return TPC_ERR_INVALID_ARG;
  Counters k;
  if (cudaStreamSynchronize(t->last_stream) != cudaSuccess ||
      cudaMemcpy(&k, t->ctx.cnt, sizeof(k), cudaMemcpyDeviceToHost) != cudaSuccess)
    return TPC_ERR_CUDA;
  out->n_clusters = t->last_n; out->n_bins = k.n_bins; out->n_seeds = k.n_seeds; out->n_tracklets = k.n_tracklets;
  out->n_tracks = k.n_tracks; out->n_track_clusters = k.n_track_clusters; out->n_linked = k.n_linked;
  out->kf_steps = (int64_t)k.kf_steps; out->n_hits = (int64_t)k.n_hits; out->status = k.status; out->s1_global_buckets = k.s1_global;
  return TPC_OK;
}

int tpc_tracker_enable_stage_timing(tpc_tracker_t* t, int32_t enable) {
  if (!t) return TPC_ERR_INVALID_ARG;
  t->timing = enable != 0;
  return TPC_OK;
}

int tpc_tracker_stage_ms(tpc_tracker_t* t, float* out_ms5) {
  if (!t || !out_ms5 || !t->timing) return TPC_ERR_INVALID_ARG;
  if (cudaEventSynchronize(t->ev[5]) != cudaSuccess) return TPC_ERR_CUDA;
  for (int i = 0; i < 5; ++i)
    if (cudaEventElapsedTime(&out_ms5[i], t->ev[i], t->ev[i + 1]) != cudaSuccess) return TPC_ERR_CUDA;
  return TPC_OK;
}

int tpc_tracker_stage_view(tpc_tracker_t* t, int32_t which, tpc_stage_view_t* out) {
  if (!t || !out || which < 0 || which >= TPC_VIEW_COUNT_) return TPC_ERR_INVALID_ARG;
  Counters k;
  if (cudaStreamSynchronize(t->last_stream) != cudaSuccess ||
      cudaMemcpy(&k, t->ctx.cnt, sizeof(k), cudaMemcpyDeviceToHost) != cudaSuccess)
    return TPC_ERR_CUDA;
  const Ctx& c = t->ctx;
  const int64_t n = t->last_n, ns = k.n_seeds, SR1 = c.SR + 1;
  auto set = [&](const void* p, int64_t cnt, int eb, int fl) { out->ptr = p; out->n = cnt; out->elem_bytes = eb; out->is_float = fl; };
  switch (which) {
    case TPC_VIEW_PERM: set(c.perm, n, 4, 0); break;
    case TPC_VIEW_YZ: set(c.yz, 2 * n, 4, 1); break;
    case TPC_VIEW_SROW: set(c.srow, n, 2, 0); break;
    case TPC_VIEW_BIN_START: set(c.bins, (int64_t)k.n_bins + 1, 4, 0); break;
    case TPC_VIEW_ROW_START: set(c.row_start, SR1, 4, 0); break;
    case TPC_VIEW_BIN_BASE: set(c.bin_base, SR1, 4, 0); break;
    case TPC_VIEW_ZMIN: set(c.zmin, c.S, 4, 1); break;
    case TPC_VIEW_ZMAX: set(c.zmax, c.S, 4, 1); break;
    case TPC_VIEW_NZ: set(c.nz, c.S, 4, 0); break;
    case TPC_VIEW_LINK_UP_RAW: set(c.link_up_raw, n, 4, 0); break;
    case TPC_VIEW_LINK_DN_RAW: set(c.link_dn_raw, n, 4, 0); break;
    case TPC_VIEW_LINK_UP: set(c.link_up, n, 4, 0); break;
    case TPC_VIEW_LINK_DN: set(c.link_dn, n, 4, 0); break;
    case TPC_VIEW_SEED_HEAD: set(c.seed_head, ns, 4, 0); break;
    case TPC_VIEW_SEED_LEN: set(c.seed_len, ns, 4, 0); break;
    case TPC_VIEW_T_HIT: set(c.t_hit, ns * c.R, 4, 0); break;
    case TPC_VIEW_T_FIRST_ROW: set(c.t_first_row, ns, 4, 0); break;
    case TPC_VIEW_T_LAST_ROW: set(c.t_last_row, ns, 4, 0); break;
    case TPC_VIEW_T_N_HITS: set(c.t_n_hits, ns, 4, 0); break;
    case TPC_VIEW_T_PAR: set(c.t_par, ns * 5, 4, 1); break;
    case TPC_VIEW_T_COV: set(c.t_cov, ns * 15, 4, 1); break;
    case TPC_VIEW_T_CHI2: set(c.t_chi2, ns, 4, 1); break;
    case TPC_VIEW_T_ZREF: set(c.t_zref, ns, 4, 1); break;
    case TPC_VIEW_TRACKLET_OF_SEED: set(c.tracklet_of_seed, ns, 4, 0); break;
    case TPC_VIEW_OWNED: set(c.k_owned, ns, 4, 0); break;
    case TPC_VIEW_FIT_ROW: set(c.fit_row, k.n_tracks, 4, 0); break;
    case TPC_VIEW_UP_PAR: set(c.up_par, 5 * (int64_t)c.max_tracks, 4, 1); break;
    case TPC_VIEW_UP_COV: set(c.up_cov, 15 * (int64_t)c.max_tracks, 4, 1); break;
    case TPC_VIEW_UP_X: set(c.up_x, k.n_tracks, 4, 1); break;
    case TPC_VIEW_UP_ZREF: set(c.up_zref, k.n_tracks, 4, 1); break;
    case TPC_VIEW_UP_ROW: set(c.up_row, k.n_tracks, 4, 0); break;
    case TPC_VIEW_UP_N: set(c.up_n, k.n_tracks, 4, 0); break;
    case TPC_VIEW_MRG_BEST_B: set(c.m_best_b, k.n_tracks, 4, 0); break;
    case TPC_VIEW_MRG_BEST_A: set(c.m_best_a, k.n_tracks, 8, 0); break;
    case TPC_VIEW_MRG_CHI_B: set(c.m_chi_b, k.n_tracks, 4, 1); break;
    case TPC_VIEW_MRG_NEXT: set(c.m_next, k.n_tracks, 4, 0); break;
    case TPC_VIEW_MRG_PREV: set(c.m_prev, k.n_tracks, 4, 0); break;
    case TPC_VIEW_MRG_DIR: set(c.m_dir, k.n_tracks, 4, 0); break;
    case TPC_VIEW_APEX_BEST: set(c.a_best, c.max_tracks, 4, 0); break;
    case TPC_VIEW_APEX_SCORE: set(c.a_score, c.max_tracks, 4, 1); break;
    default: return TPC_ERR_INVALID_ARG;
  }
  return TPC_OK;
}

int tpc_tracker_launches_per_call(const tpc_tracker_t* t) {
  if (!t) return TPC_ERR_INVALID_ARG;
  return launches_reset() + launches_s1() + launches_s2() + launches_s3() + launches_s4() + launches_s5();
}

int tpc_tracker_destroy(tpc_tracker_t* t) {
  if (!t) return TPC_ERR_INVALID_ARG;
  for (auto& e : t->ev)
    if (e) cudaEventDestroy(e);
  if (t->s_compute) cudaStreamSynchronize(t->s_compute);
  if (t->s_out) cudaStreamSynchronize(t->s_out);
  for (auto& sl : t->slot)
    for (cudaEvent_t e : {sl.h2d_done, sl.in_free, sl.done, sl.out_free})
      if (e) cudaEventDestroy(e);
  for (cudaStream_t st : {t->s_in, t->s_compute, t->s_out})
    if (st) cudaStreamDestroy(st);
  if (t->h_counts) cudaFreeHost(t->h_counts);
  if (t->graph_exec) cudaGraphExecDestroy(t->graph_exec);
  delete t;
  return TPC_OK;
}

const char* tpc_error_string(int code) {
  switch (code) {
    case TPC_OK: return "ok";
    case TPC_ERR_INVALID_ARG: return "invalid argument";
    case TPC_ERR_CAPACITY: return "capacity exceeded";
    case TPC_ERR_CUDA: return "CUDA error";
    case TPC_ERR_STATIC_SCRATCH: return "frame has more clusters than the library's built-in scratch array holds (TPC_PROTECT_STATIC_MAX_CLUSTERS)";
    default: return "unknown error";
  }
}

}  // extern "C"
