/* A plain C program on the C ABI of libtpc_tracker.so (include/tpc_tracker.h): no Python, no torch.  It reads one time
 * frame from a binary dump, allocates the device buffers with the CUDA runtime, runs tpc_track_timeframe and prints
 * "n_tracks status n_attached".  tests/test_c_abi_program.py writes the dump, builds this file with gcc, runs it on the
 * GPU box and compares the numbers with the oracle's.
 *
 * dump layout (little endian): int64 n; int32 n_sectors, n_rows; float row_x[n_rows]; float f[16] = tan_half_sector,
 * bz_tesla, err_y2, err_z2, cell_y, cell_z, link_ay, link_az, link_b, link_T, pick_chi2_cut, max_sinphi, y_margin,
 * init_c_ss, init_c_tt, init_c_qq; int32 i[4] = min_chain_len, max_gap, min_tracklet_hits, min_track_hits;
 * int64 max_bins; uint8 sector[n]; uint8 row[n]; float y[n]; float z[n]. */
#include <cuda_runtime_api.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "tpc_tracker.h"

#define CK(x) do { if ((x) != 0) { fprintf(stderr, "failed: %s (line %d)\n", #x, __LINE__); return 1; } } while (0)

static void* dev(size_t bytes, const void* host) {
  void* p = NULL;
  if (cudaMalloc(&p, bytes ? bytes : 1) != cudaSuccess) return NULL;
  if (host && bytes && cudaMemcpy(p, host, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return NULL;
  return p;
}

int main(int argc, char** argv) {
  if (argc < 2) return 2;
  FILE* f = fopen(argv[1], "rb");
  if (!f) return 2;
  int64_t n, max_bins; int32_t geo[2], iv[4]; float rx[256], fv[16];
  CK(fread(&n, 8, 1, f) != 1); CK(fread(geo, 4, 2, f) != 2); CK(fread(rx, 4, geo[1], f) != (size_t)geo[1]);
  CK(fread(fv, 4, 16, f) != 16); CK(fread(iv, 4, 4, f) != 4); CK(fread(&max_bins, 8, 1, f) != 1);
  uint8_t* sec = malloc(n); uint8_t* row = malloc(n); float* y = malloc(4 * n); float* z = malloc(4 * n);
  CK(fread(sec, 1, n, f) != (size_t)n); CK(fread(row, 1, n, f) != (size_t)n);
  CK(fread(y, 4, n, f) != (size_t)n); CK(fread(z, 4, n, f) != (size_t)n);
  fclose(f);

  tpc_params_t p; memset(&p, 0, sizeof p);
  p.n_sectors = geo[0]; p.n_rows = geo[1]; p.row_x = rx;
  p.tan_half_sector = fv[0]; p.bz_tesla = fv[1]; p.err_y2 = fv[2]; p.err_z2 = fv[3]; p.cell_y = fv[4]; p.cell_z = fv[5];
  p.link_ay = fv[6]; p.link_az = fv[7]; p.link_b = fv[8]; p.link_T = fv[9]; p.pick_chi2_cut = fv[10]; p.max_sinphi = fv[11];
  p.y_margin = fv[12]; p.init_c_ss = fv[13]; p.init_c_tt = fv[14]; p.init_c_qq = fv[15];
  p.min_chain_len = iv[0]; p.max_gap = iv[1]; p.min_tracklet_hits = iv[2]; p.min_track_hits = iv[3];

  const int64_t max_seeds = n / 2 + 1024, max_tracks = n / 8 + 1024, max_tc = n + 1;
  const size_t ws = tpc_tracker_workspace_bytes(&p, n, max_bins, max_seeds, max_tracks, max_tc, 0);
  CK(ws == 0);
  void* d_ws = dev(ws, NULL); CK(d_ws == NULL);
  tpc_tracker_t* t = NULL;
  CK(tpc_tracker_create(&p, n, max_bins, max_seeds, max_tracks, max_tc, 0, d_ws, ws, &t));

  tpc_clusters_t in; memset(&in, 0, sizeof in);
  in.n = n; in.sector = dev(n, sec); in.row = dev(n, row); in.y = dev(4 * n, y); in.z = dev(4 * n, z);
  tpc_tracks_t out; memset(&out, 0, sizeof out);
  out.max_tracks = max_tracks; out.max_track_clusters = max_tc;
  out.n_tracks = dev(4, NULL); out.status = dev(4, NULL);
  out.sector = dev(4 * max_tracks, NULL); out.first_row = dev(4 * max_tracks, NULL); out.last_row = dev(4 * max_tracks, NULL);
  out.n_clusters = dev(4 * max_tracks, NULL); out.par = dev(20 * max_tracks, NULL); out.cov = dev(60 * max_tracks, NULL);
  out.x_ref = dev(4 * max_tracks, NULL); out.z_ref = dev(4 * max_tracks, NULL); out.chi2 = dev(4 * max_tracks, NULL);
  out.ndf = dev(4 * max_tracks, NULL); out.z_beam = dev(4 * max_tracks, NULL);
  out.trk_cl_start = dev(4 * (max_tracks + 1), NULL); out.trk_cl_idx = dev(4 * max_tc, NULL); out.cluster_track = dev(4 * n, NULL);

  CK(tpc_track_timeframe(t, &in, &out, NULL));
  CK(cudaDeviceSynchronize() != cudaSuccess);
  int32_t nt = -1, st = -1;
  CK(cudaMemcpy(&nt, out.n_tracks, 4, cudaMemcpyDeviceToHost) != cudaSuccess);
  CK(cudaMemcpy(&st, out.status, 4, cudaMemcpyDeviceToHost) != cudaSuccess);
  int32_t* ct = malloc(4 * n);
  CK(cudaMemcpy(ct, out.cluster_track, 4 * n, cudaMemcpyDeviceToHost) != cudaSuccess);
  int64_t attached = 0;
  for (int64_t i = 0; i < n; ++i) attached += ct[i] >= 0;
  tpc_counters_t k; CK(tpc_tracker_counters(t, &k));
  printf("%d %d %lld %lld\n", nt, st, (long long)attached, (long long)k.n_seeds);
  CK(tpc_tracker_destroy(t));
  return 0;
}
