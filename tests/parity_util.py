"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded time frame
and compare stage by stage (test infrastructure; imports both sides, which share no code)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import Oracle
from tpc_synth import default_params

INT_STAGES = ["perm", "bin_start", "row_start", "bin_base", "nz", "link_up_raw", "link_dn_raw", "link_up", "link_dn",
              "seed_head", "seed_len"]


def run_gpu(tf, params=None, host=False, caps=None, timing=False):
    import paper_2009_07515_b200 as tpc
    P = params or default_params(tf)
    c = tpc.suggest_capacities(tf.n, P)
    c["max_bins"] = tpc.max_bins_bound(tf.sector, tf.z, P)
    if caps:
        c.update(caps)
    trk = tpc.Tracker(P, c["max_clusters"], c["max_bins"], c["max_seeds"], c["max_tracks"], c["max_track_clusters"],
                      host_io=host)
    if timing:
        trk.enable_stage_timing(True)
    th = lambda a: torch.from_numpy(np.ascontiguousarray(a))  # noqa: E731
    if host:
        ins = [th(a).pin_memory() for a in (tf.sector, tf.row, tf.y, tf.z)]
        out = trk.new_tracks(tf.n, host=True)
        trk.track_timeframe_host(*ins, out)
    else:
        ins = [th(a).cuda() for a in (tf.sector, tf.row, tf.y, tf.z)]
        out = trk.new_tracks(tf.n)
        trk.track_timeframe(*ins, out)
        torch.cuda.synchronize()
    return P, trk, out


def run_oracle(tf, P, last_stage=6):
    return Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=last_stage)


def compare_integer_stages(trk, o, upto=3):
    """bit-exact comparison of S1..S3; returns a dict name -> #mismatches."""
    bad = {}
    names = ["perm", "bin_start", "row_start", "bin_base", "nz"]
    if upto >= 2:
        names += ["link_up_raw", "link_dn_raw"]
    if upto >= 3:
        names += ["link_up", "link_dn", "seed_head", "seed_len"]
    for name in names:
        a = trk.stage_view(name); b = o.get(name)
        if a.shape != b.shape:
            bad[name] = f"shape {a.shape} vs {b.shape}"
        elif not np.array_equal(a, b):
            bad[name] = int((a != b).sum())
    yz = trk.stage_view("yz").reshape(-1, 2)
    for name, a in (("ys", yz[:, 0]), ("zs", yz[:, 1]), ("zmin", None), ("zmax", None)):
        a = trk.stage_view(name) if a is None else a
        b = o.get(name)
        if name in ("zmin", "zmax"):
            keep = o.get("nz") > 0
            a, b = a[keep], b[keep]
        if a.shape != b.shape or not np.array_equal(a, b):
            bad[name] = "differs"
    R = trk.params["n_rows"]
    srow = trk.stage_view("srow").astype(np.int64)
    if not np.array_equal(srow, o.get("s_sector").astype(np.int64) * 256 + o.get("s_row")):   # (sector << 8) | row
        bad["srow"] = "differs"
    return bad


def rel_err(a, b, floor):
    """max |a-b| / max(|b|, floor)"""
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    if a.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), floor)))


def compare_tracklets(trk, o):
    """S4 per seed: hit tables bit-exact?  parameters / covariance relative error."""
    R = trk.params["n_rows"]
    res = {}
    hit_g = trk.stage_view("t_hit").reshape(-1, R).copy(); hit_o = o.get("t_hit").reshape(-1, R)
    # the CUDA table is defined on [t_first_row, t_last_row] only (tpc_tracker.h); the oracle's holds -1 outside
    rows = np.arange(R)[None, :]
    outside = (rows < trk.stage_view("t_first_row")[:, None]) | (rows > trk.stage_view("t_last_row")[:, None])
    hit_g[outside] = -1
    res["n_seeds"] = (hit_g.shape[0], hit_o.shape[0])
    if hit_g.shape != hit_o.shape:
        res["hit_mismatch_seeds"] = -1
        return res
    res["hit_mismatch_seeds"] = int((hit_g != hit_o).any(axis=1).sum())
    for nm in ("t_first_row", "t_last_row", "t_n_hits"):
        res[nm + "_mismatch"] = int((trk.stage_view(nm) != o.get(nm)).sum())
    same = ~(hit_g != hit_o).any(axis=1)
    par_g = trk.stage_view("t_par").reshape(-1, 5)[same]; par_o = o.get("t_par").reshape(-1, 5)[same]
    cov_g = trk.stage_view("t_cov").reshape(-1, 15)[same]; cov_o = o.get("t_cov").reshape(-1, 15)[same]
    res["par_bitexact"] = bool(np.array_equal(par_g.astype(np.float32), par_o.astype(np.float32)))
    res["cov_bitexact"] = bool(np.array_equal(cov_g.astype(np.float32), cov_o.astype(np.float32)))
    res["chi2_bitexact"] = bool(np.array_equal(trk.stage_view("t_chi2")[same], o.get("t_chi2").astype(np.float32)[same]))
    # relative error with a per-parameter floor (parameters cross zero): y, z_rel in cm, sin, tan, q/pT
    floors = np.array([1.0, 1.0, 0.1, 0.1, 0.1])
    res["par_rel"] = float(np.max(np.abs(par_g - par_o) / np.maximum(np.abs(par_o), floors))) if par_g.size else 0.0
    diag = [0, 2, 5, 9, 14]
    sig = np.sqrt(np.maximum(cov_o[:, diag], 0))
    idx = [(i, j) for i in range(5) for j in range(i + 1)]
    scale = np.stack([sig[:, i] * sig[:, j] for i, j in idx], axis=1)
    res["cov_rel"] = float(np.max(np.abs(cov_g - cov_o) / np.maximum(scale, 1e-30))) if cov_g.size else 0.0
    return res


def compare_tracks(out_np: dict, o, n_in: int):
    """S5: exact equality of the assignment + matching statistics (>= 90 % shared clusters)."""
    res = {}
    ct_g = out_np["cluster_track"]; ct_o = o.get("cluster_track")
    res["n_tracks"] = (out_np["n_tracks"], int(o.get("trk_seed").shape[0]))
    res["cluster_track_equal"] = bool(np.array_equal(ct_g, ct_o))
    res["csr_equal"] = bool(np.array_equal(out_np["trk_cl_start"], o.get("trk_cl_start")) and
                            np.array_equal(out_np["trk_cl_idx"], o.get("trk_cl_idx")))
    # matching: for every oracle track the GPU track sharing most of its clusters
    To = int(o.get("trk_seed").shape[0])
    matched = 0
    if To:
        st = o.get("trk_cl_start"); idx = o.get("trk_cl_idx")
        for t in range(To):
            cl = idx[st[t]:st[t + 1]]
            g = ct_g[cl]
            g = g[g >= 0]
            if g.size and np.bincount(g).max() >= 0.9 * cl.size:
                matched += 1
    res["matched_frac"] = matched / To if To else 1.0
    return res
