"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded time frame
and compare stage by stage (test infrastructure; imports both sides, which share no code)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import Oracle
from tpc_synth import default_params

INT_STAGES = ["perm", "bin_start", "row_start", "bin_base", "nz", "link_up_raw", "link_dn_raw", "link_up", "link_dn",
              "seed_head", "seed_len"]


def run_gpu(tf, params=None, host=False, caps=None, timing=False, guard_bytes=0):
    import paper_2009_07515_b200 as tpc
    P = params or default_params(tf)
    c = tpc.suggest_capacities(tf.n, P)
    c["max_bins"] = tpc.max_bins_bound(tf.sector, tf.z, P)
    if caps:
        c.update(caps)
    trk = tpc.Tracker(P, c["max_clusters"], c["max_bins"], c["max_seeds"], c["max_tracks"], c["max_track_clusters"],
                      host_io=host, guard_bytes=guard_bytes)
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


# ------------------------------------------------------------------------------------------------------------------
# Whole-frame parity, sector by sector.  Sectors are independent (section 3.1: one z range per sector;
# S2..S5 never leave a sector), so the oracle run on the clusters of ONE sector must reproduce, array by array and bit for
# bit, the slice of the CUDA result that belongs to that sector.  The sectors are checked in a fork()ed process pool:
# the children inherit the host copies of the CUDA arrays (module global _FRAME), run the plain oracle and compare; they
# never touch CUDA.
_FRAME = None


def collect_gpu_frame(tf, P, trk, out, road=(1.0, 1.0)):
    """Host copies of every stage array, the outputs, the refit (with residuals) and the keep flags of one CUDA run."""
    g = out.numpy()
    fit = trk.refit(g["n_tracks"], tracks=out)
    keep = trk.protect(out, *road)
    torch.cuda.synchronize()
    views = {nm: trk.stage_view(nm) for nm in (
        "perm", "yz", "srow", "bin_start", "row_start", "bin_base", "zmin", "zmax", "nz", "link_up_raw", "link_dn_raw",
        "link_up", "link_dn", "seed_head", "seed_len", "t_hit", "t_first_row", "t_last_row", "t_n_hits", "t_par", "t_cov",
        "t_chi2", "t_zref", "tracklet_of_seed", "k_owned")}
    return dict(tf=tf, P=P, out=g, fit=fit, keep=keep.cpu().numpy()[: tf.n].astype(np.int32), road=road, **views)


def _eq(bad, name, a, b):
    a = np.asarray(a); b = np.asarray(b)
    if a.shape != b.shape:
        bad.append(f"{name}: shape {a.shape} vs {b.shape}")
    elif not np.array_equal(a, b):
        bad.append(f"{name}: {int((a != b).sum())} of {a.size} differ")


def check_sector(s: int):
    """Oracle on sector `s` of _FRAME['tf'] against the CUDA arrays restricted to that sector: list of mismatches."""
    from tpc_synth import select_sectors
    F = _FRAME
    tf, P, g, fit = F["tf"], F["P"], F["out"], F["fit"]
    R = P["n_rows"]
    sub, idx = select_sectors(tf, [s])
    o = Oracle(P).run(sub.sector, sub.row, sub.y, sub.z, precision=32, last_stage=6)
    bad = []
    f32 = np.float32
    a, b = int(F["row_start"][s * R]), int(F["row_start"][(s + 1) * R])
    if b - a != sub.n:
        return s, [f"row_start: sector holds {b - a} positions, {sub.n} clusters"], {}
    off = lambda v: np.where(v >= 0, v.astype(np.int64) + a, -1)   # noqa: E731  oracle positions -> frame positions
    # ---- S1
    _eq(bad, "perm", F["perm"][a:b], idx[o.get("perm")])
    yz = F["yz"].reshape(-1, 2)[a:b]
    _eq(bad, "ys", yz[:, 0], o.get("ys")); _eq(bad, "zs", yz[:, 1], o.get("zs"))
    _eq(bad, "srow", F["srow"][a:b].astype(np.int64), o.get("s_sector").astype(np.int64) * 256 + o.get("s_row"))
    bb0, bb1 = int(F["bin_base"][s * R]), int(F["bin_base"][(s + 1) * R])
    _eq(bad, "bin_base", F["bin_base"][s * R:(s + 1) * R + 1].astype(np.int64) - bb0, o.get("bin_base")[s * R:(s + 1) * R + 1])
    _eq(bad, "bin_start", F["bin_start"][bb0:bb1 + 1].astype(np.int64) - a, o.get("bin_start"))
    _eq(bad, "row_start", F["row_start"][s * R:(s + 1) * R + 1].astype(np.int64) - a, o.get("row_start")[s * R:(s + 1) * R + 1])
    _eq(bad, "nz", F["nz"][s], o.get("nz")[s]); _eq(bad, "zmin", F["zmin"][s], o.get("zmin")[s]); _eq(bad, "zmax", F["zmax"][s], o.get("zmax")[s])
    # ---- S2 / S3
    for nm in ("link_up_raw", "link_dn_raw", "link_up", "link_dn"):
        _eq(bad, nm, F[nm][a:b], off(o.get(nm)))
    k0, k1 = int(np.searchsorted(F["seed_head"], a)), int(np.searchsorted(F["seed_head"], b))
    _eq(bad, "seed_head", F["seed_head"][k0:k1], off(o.get("seed_head")))
    _eq(bad, "seed_len", F["seed_len"][k0:k1], o.get("seed_len"))
    K = k1 - k0
    # ---- S4 (the CUDA hit table is defined on [t_first_row, t_last_row] only; the oracle's holds -1 outside)
    if K == o.get("seed_head").shape[0]:
        hit = F["t_hit"].reshape(-1, R)[k0:k1].copy()
        rows = np.arange(R)[None, :]
        hit[(rows < F["t_first_row"][k0:k1, None]) | (rows > F["t_last_row"][k0:k1, None])] = -1
        _eq(bad, "t_hit", hit, off(o.get("t_hit").reshape(-1, R)))
        for nm in ("t_first_row", "t_last_row", "t_n_hits"):
            _eq(bad, nm, F[nm][k0:k1], o.get(nm))
        _eq(bad, "t_par", F["t_par"].reshape(-1, 5)[k0:k1], o.get("t_par").astype(f32).reshape(-1, 5))
        _eq(bad, "t_cov", F["t_cov"].reshape(-1, 15)[k0:k1], o.get("t_cov").astype(f32).reshape(-1, 15))
        _eq(bad, "t_chi2", F["t_chi2"][k0:k1], o.get("t_chi2").astype(f32))
        _eq(bad, "t_zref", F["t_zref"][k0:k1], o.get("t_z_ref").astype(f32))
        tos_g = F["tracklet_of_seed"][k0:k1].astype(np.int64); tos_o = o.get("tracklet_of_seed")
        first_kept = tos_g[tos_g >= 0].min() if (tos_g >= 0).any() else 0
        _eq(bad, "tracklet_of_seed", np.where(tos_g >= 0, tos_g - first_kept, -1), tos_o)
        _eq(bad, "k_owned", F["k_owned"][k0:k1], o.get("k_owned"))
    # ---- S5: tracks of a sector have consecutive ids (seed order is sector-major)
    mine = np.nonzero(g["sector"] == s)[0]
    t0, t1 = (int(mine[0]), int(mine[-1]) + 1) if mine.size else (0, 0)
    To = int(o.get("trk_seed").shape[0])
    if t1 - t0 != To or (mine.size and not np.array_equal(mine, np.arange(t0, t1))):
        bad.append(f"tracks: {t1 - t0} vs oracle {To}")
    else:
        ct = g["cluster_track"][idx].astype(np.int64)
        _eq(bad, "cluster_track", np.where(ct >= 0, ct - t0, -1), o.get("cluster_track"))
        st = g["trk_cl_start"][t0:t1 + 1].astype(np.int64)
        c0, c1 = (int(st[0]), int(st[-1])) if To else (0, 0)
        _eq(bad, "trk_cl_start", st - c0 if To else np.zeros(1, np.int64), o.get("trk_cl_start"))
        _eq(bad, "trk_cl_idx", g["trk_cl_idx"][c0:c1], idx[o.get("trk_cl_idx")] if To else np.empty(0, np.int64))
        for nm in ("first_row", "last_row", "n_clusters", "ndf"):
            _eq(bad, nm, g[nm][t0:t1], o.get("trk_" + nm))
        _eq(bad, "par", g["par"][t0:t1], o.get("trk_par").astype(f32).reshape(-1, 5))
        _eq(bad, "cov", g["cov"][t0:t1], o.get("trk_cov").astype(f32).reshape(-1, 15))
        for nm in ("x_ref", "z_ref", "chi2", "z_beam"):
            _eq(bad, nm, g[nm][t0:t1], o.get("trk_" + nm).astype(f32))
        # ---- refit + residuals
        _eq(bad, "fit_par", fit["par"][t0:t1], o.get("fit_par").astype(f32).reshape(-1, 5))
        _eq(bad, "fit_cov", fit["cov"][t0:t1], o.get("fit_cov").astype(f32).reshape(-1, 15))
        for nm in ("x_ref", "z_ref", "chi2"):
            _eq(bad, "fit_" + nm, fit[nm][t0:t1], o.get("fit_" + nm).astype(f32))
        _eq(bad, "fit_n", fit["n_fit"][t0:t1], o.get("fit_n")); _eq(bad, "fit_ndf", fit["ndf"][t0:t1], o.get("fit_ndf"))
        _eq(bad, "res_y", fit["res_y"][c0:c1], o.get("fit_res_y").astype(f32))
        _eq(bad, "res_z", fit["res_z"][c0:c1], o.get("fit_res_z").astype(f32))
    # ---- protection flags
    _eq(bad, "keep", F["keep"][idx], o.protect(*F["road"]))
    stats = dict(n=sub.n, seeds=K, tracks=To, attached=int((o.get("cluster_track") >= 0).sum()))
    return s, bad, stats


def check_sectors_parallel(frame: dict, sectors, procs=None):
    """Runs check_sector over `sectors` in a fork()ed pool (children: numpy + the CPU oracle only).  Returns
    ({sector: [mismatch, ...]}, {sector: stats}, processes used)."""
    import multiprocessing as mp
    import os
    global _FRAME
    _FRAME = frame
    sectors = list(sectors)
    procs = max(1, min(len(sectors), procs or (os.cpu_count() or 1)))
    try:
        if procs == 1:
            res = [check_sector(s) for s in sectors]
        else:
            with mp.get_context("fork").Pool(procs) as pool:
                res = pool.map(check_sector, sectors, chunksize=1)
    finally:
        _FRAME = None
    return {s: b for s, b, _ in res}, {s: st for s, _, st in res}, procs
