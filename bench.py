#!/usr/bin/env python
"""bench.py - TPC clusters/s tracked per B200 on a synthetic time frame (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl ours|reference]

A step = one pass of the whole hot path (S1..S5, tpc_track_timeframe) over one time frame.
`value`  : clusters/s, device-timed (CUDA events), inputs resident in HBM.
`e2e`    : the same through tpc_track_timeframe_host (pinned HOST buffers in and out).
`roofline`: the dominant kernel against the measured HBM peak (MEASURED_PEAKS.json), algorithmic
            bytes per DESIGN.md section 6, duration from CUDA events recorded inside the library.
`cpu_baseline`: the oracle, as it stands, single-threaded, on a bounded sample (whole sectors).
N > 1: replicas only - every rank tracks its own time frame, no collective on the
data path; value = clusters of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "TPC clusters/sec tracked per B200 (time frame, device-timed)"
UNIT = "clusters/s"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", help="cfg1..cfg5 (BASELINE.json configs[0..4]); cfg5 = the metric's")
    ap.add_argument("--collisions", type=int, default=0, help="override n_collisions (debug; 0 = the config's own)")
    ap.add_argument("--cell-y", type=float, default=0.0, help="override the grid cell along y, cm (debug; 0 = tpc_synth.choose_cell)")
    ap.add_argument("--cell-z", type=float, default=0.0, help="override the grid cell along z, cm (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parity-sectors", type=int, default=2,
                    help="sectors of the timed frame checked against the oracle before timing (0: skip)")
    ap.add_argument("--repeats", type=int, default=10, help="separately-evented steps for median / best (>= 10)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-optional", action="store_true", help="skip the optional calls (refit / merge / apex / removable / protect)")
    return ap.parse_args()


def _capture_is_current(src_file: str, sha1: str) -> bool:
    """A committed ncu capture describes the kernel only as long as the kernel's source file is the one it was taken from:
    the CSV rows carry the sha1 of that file at capture time."""
    import hashlib
    try:
        with open(os.path.join(ROOT, "paper_2009_07515_b200", "csrc", src_file), "rb") as f:
            return hashlib.sha1(f.read()).hexdigest() == sha1.strip()
    except Exception:
        return False


def ncu_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on cfg5, copied from the committed
    `ncu --set full` capture (profiles/traffic.csv names the capture and the sha1 of the kernel's source file it was taken
    from); None if there is none or if the source has changed since (a stale capture is not reported)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            head = f.readline().strip().split(",")
            for ln in f:
                d = dict(zip(head, ln.strip().split(",")))
                if d["kernel"] == kernel:
                    return float(d["dram_bytes_per_launch"]) if _capture_is_current(d["source_file"], d["source_sha1"]) else None
    except Exception:
        pass
    return None


def ncu_counters(kernel: str):
    """Issue-slot utilisation, active lanes, occupancy, L2 hit rate of `kernel` on cfg5 and what actually bounds it,
    copied from the committed `ncu --set full` capture (profiles/kernel_counters.csv names it); None if there is none."""
    try:
        with open(os.path.join(ROOT, "profiles", "kernel_counters.csv")) as f:
            head = f.readline().strip().split(",")
            for ln in f:
                p = ln.strip().split(",")
                if p[0] == kernel:
                    d = dict(zip(head, p))
                    if not _capture_is_current(d["source_file"], d["source_sha1"]):
                        return None
                    return {"issue_slots_busy": float(d["issue_slots_busy_pct"]) / 100, "active_lanes_of_32": float(d["active_lanes_per_instruction"]),
                            "achieved_occupancy": float(d["achieved_occupancy_pct"]) / 100, "l2_hit_rate": float(d["l2_hit_rate_pct"]) / 100,
                            "bound_by": d["bound_by"], "source": d["source"]}
    except Exception:
        pass
    return None


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# The two legs that execute oracle/ (test infrastructure, never on the product path): the pre-timing parity check of
# the timed configuration ("each config is also run once through the parity checker before it is
# timed") and the CPU baseline.  Both run the oracle on whole sectors (sectors are independent) in
# fork()ed children that inherit the host arrays through _SHARED and never touch CUDA.
_SHARED = None


def _sector_slices(tf):
    """Input indices of every sector, in input order: one stable argsort instead of 36 masks."""
    order = np.argsort(tf.sector, kind="stable")
    counts = np.bincount(tf.sector, minlength=tf.geometry.n_sectors)
    ends = np.cumsum(counts)
    return order, ends - counts, ends


def _oracle_sector(s: int):
    """Child: the oracle, as it stands, on sector s; returns (clusters, seconds)."""
    from oracle import Oracle
    F = _SHARED
    tf, idx = F["tf"], F["order"][F["lo"][s]:F["hi"][s]]
    sec, row, y, z = tf.sector[idx], tf.row[idx], tf.y[idx], tf.z[idx]
    t0 = time.perf_counter()
    Oracle(F["P"]).run(sec, row, y, z)
    return int(idx.size), time.perf_counter() - t0


def _parity_sector(s: int):
    """Child: oracle on sector s against the CUDA result restricted to that sector; list of mismatching arrays."""
    from oracle import Oracle
    F = _SHARED
    tf, P, g = F["tf"], F["P"], F["out"]
    R = int(P["n_rows"])
    idx = F["order"][F["lo"][s]:F["hi"][s]]
    o = Oracle(P).run(tf.sector[idx], tf.row[idx], tf.y[idx], tf.z[idx])
    a, b = int(F["row_start"][s * R]), int(F["row_start"][(s + 1) * R])
    bad = []

    def eq(name, x, y_):
        x = np.asarray(x); y_ = np.asarray(y_)
        if x.shape != y_.shape or not np.array_equal(x, y_):
            bad.append(name)

    off = lambda v: np.where(v >= 0, v.astype(np.int64) + a, -1)   # noqa: E731  oracle positions -> frame positions
    eq("perm", F["perm"][a:b], idx[o.get("perm")])
    for nm in ("link_up_raw", "link_dn_raw", "link_up", "link_dn"):
        eq(nm, F[nm][a:b], off(o.get(nm)))
    mine = np.nonzero(g["sector"] == s)[0]
    t0, t1 = (int(mine[0]), int(mine[-1]) + 1) if mine.size else (0, 0)
    To = int(o.get("trk_seed").shape[0])
    if t1 - t0 != To:
        bad.append(f"n_tracks {t1 - t0} vs {To}")
    else:
        ct = g["cluster_track"][idx].astype(np.int64)
        eq("cluster_track", np.where(ct >= 0, ct - t0, -1), o.get("cluster_track"))
        st = g["trk_cl_start"][t0:t1 + 1].astype(np.int64)
        c0, c1 = (int(st[0]), int(st[-1])) if To else (0, 0)
        eq("trk_cl_idx", g["trk_cl_idx"][c0:c1], idx[o.get("trk_cl_idx")] if To else np.empty(0, np.int64))
        eq("par", g["par"][t0:t1], o.get("trk_par").astype(np.float32).reshape(-1, 5))
        eq("cov", g["cov"][t0:t1], o.get("trk_cov").astype(np.float32).reshape(-1, 15))
        eq("chi2", g["chi2"][t0:t1], o.get("trk_chi2").astype(np.float32))
    return s, bad, int(idx.size), To


def _fork_map(fn, items, procs):
    import multiprocessing as mp
    if procs <= 1 or len(items) <= 1:
        return [fn(i) for i in items]
    with mp.get_context("fork").Pool(procs) as pool:
        return pool.map(fn, items, chunksize=1)


def parity_precheck(tf, P, trk, out, n_sectors: int) -> dict:
    """The timed configuration through the parity checker before it is timed: `n_sectors` whole sectors of the frame,
    S1 order, raw and cleaned links, assignment, CSR and track parameters, all compared exactly."""
    global _SHARED
    S = tf.geometry.n_sectors
    counts = np.bincount(tf.sector, minlength=S)
    filled = [s for s in range(S) if counts[s] > 0]
    # spread over both sides of the TPC
    pick = sorted({filled[int((i + 0.5) * len(filled) / n_sectors)] for i in range(n_sectors)}) if filled else []
    order, lo, hi = _sector_slices(tf)
    shared = dict(tf=tf, P=P, out=out.numpy(), order=order, lo=lo, hi=hi)
    for nm in ("perm", "row_start", "link_up_raw", "link_dn_raw", "link_up", "link_dn"):
        shared[nm] = trk.stage_view(nm)
    _SHARED = shared
    t0 = time.perf_counter()
    try:
        res = _fork_map(_parity_sector, pick, min(len(pick), os.cpu_count() or 1))
    finally:
        _SHARED = None
    bad = {int(s): b for s, b, _, _ in res if b}
    return {"checked": "oracle vs CUDA, exact: perm, raw + cleaned links, cluster_track, trk_cl_idx, par, cov, chi2",
            "sectors": [int(s) for s in pick], "clusters": int(sum(n for _, _, n, _ in res)),
            "tracks": int(sum(t for _, _, _, t in res)), "ok": not bad, "mismatches": bad,
            "seconds": round(time.perf_counter() - t0, 1)}


def cpu_baseline(tf, P, one_thread_clusters=8_000_000) -> dict:
    """The oracle as it stands on this box's host cores: (i) one thread on a bounded sample of whole
    sectors, (ii) sector-parallel over P = os.cpu_count() processes on all sectors of the frame (36 independent units;
    cf. PAPER.md:129).  The headline `value` / `cores` is (ii)."""
    from oracle import Oracle
    global _SHARED
    S = tf.geometry.n_sectors
    order, lo, hi = _sector_slices(tf)
    counts = hi - lo
    take, tot = [], 0
    for s in range(S):
        if take and tot + counts[s] > one_thread_clusters:
            break
        take.append(s); tot += int(counts[s])
    idx = np.sort(order[lo[take[0]]:hi[take[-1]]])
    sub = [a[idx] for a in (tf.sector, tf.row, tf.y, tf.z)]
    t0 = time.perf_counter()
    o = Oracle(P).run(*sub)
    dt1 = time.perf_counter() - t0
    one = {"value": idx.size / dt1, "unit": UNIT, "cores": 1,
           "sample": f"sectors {take[0]}..{take[-1]} of {tf.name} ({idx.size} of {tf.n} clusters), all five stages, fp32, {dt1:.1f} s",
           "stage_seconds": [float(v) for v in o.get("stage_seconds")]}
    filled = [s for s in range(S) if counts[s] > 0]
    procs = max(1, min(os.cpu_count() or 1, len(filled)))
    # bounded: all sectors if that is <= ~30 s of wall at the measured one-thread rate, else the first sectors that fit
    budget_clusters = one["value"] * procs * 30.0
    sectors, tot = [], 0
    for s in filled:
        if sectors and tot + counts[s] > budget_clusters:
            break
        sectors.append(s); tot += int(counts[s])
    procs = min(procs, len(sectors))
    _SHARED = dict(tf=tf, P=P, order=order, lo=lo, hi=hi)
    t0 = time.perf_counter()
    try:
        res = _fork_map(_oracle_sector, sectors, procs)
    finally:
        _SHARED = None
    dtp = time.perf_counter() - t0
    n_par = sum(n for n, _ in res)
    return {"value": n_par / dtp, "unit": UNIT, "cores": procs, "kind": "oracle",
            "sample": f"sectors {sectors[0]}..{sectors[-1]} of {tf.name} ({n_par} of {tf.n} clusters), one oracle process per sector over "
                      f"{procs} processes (os.cpu_count() = {os.cpu_count()}), all five stages, fp32, {dtp:.1f} s wall, "
                      f"{sum(t for _, t in res):.1f} core-seconds",
            "one_thread": one}


def optional_parity(tfl, P) -> dict:
    """refit -> merge through the parity checker before the optional calls are timed: four whole sectors of the looper
    frame (the 17|0 wrap on the A side and its mirror on the C side: full z span and density of the frame) as a frame of
    their own, CUDA against one oracle run, every output compared exactly.  apex / removable are NOT re-checked here: the
    oracle's apex step is an all-pairs scan (minutes at this density); tests/test_gpu_merge.py compares them at this
    density on two sectors."""
    import torch
    import paper_2009_07515_b200 as tpc
    from oracle import Oracle
    from tpc_synth import select_sectors
    S = tfl.geometry.n_sectors
    pick = sorted({0, S // 2 - 1, S // 2, S - 1})
    sub, _ = select_sectors(tfl, pick)
    t0 = time.perf_counter()
    c = tpc.suggest_capacities(sub.n, P)
    trk = tpc.Tracker(P, c["max_clusters"], tpc.max_bins_bound(sub.sector, sub.z, P), c["max_seeds"], c["max_tracks"], c["max_track_clusters"])
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (sub.sector, sub.row, sub.y, sub.z)]
    out = trk.new_tracks(sub.n)
    trk.track_timeframe(*ins, out)
    T = out.numpy()["n_tracks"]
    m = trk.merge(T)
    ct = out.numpy()["cluster_track"]
    trk.destroy(); del trk, out, ins
    torch.cuda.empty_cache()
    o = Oracle(P).run(sub.sector, sub.row, sub.y, sub.z, precision=32, last_stage=6).merge()
    bad = []

    def eq(name, x, y_):
        x = np.asarray(x); y_ = np.asarray(y_)
        if x.shape != y_.shape or not np.array_equal(x, y_):
            bad.append(name)
    eq("cluster_track", ct, o.get("cluster_track"))
    eq("merged_of_track", m["merged_of_track"], o.get("mrg_of_track"))
    eq("seg_start", m["seg_start"], o.get("mrg_seg_start")); eq("seg_idx", m["seg_idx"], o.get("mrg_seg_idx"))
    eq("mrg_par", m["par"], o.get("mrg_par").astype(np.float32).reshape(-1, 5))
    eq("mrg_cov", m["cov"], o.get("mrg_cov").astype(np.float32).reshape(-1, 15))
    eq("mrg_n_fit", m["n_fit"], o.get("mrg_n_fit"))
    return {"checked": "oracle vs CUDA, exact: cluster_track, merged_of_track, seg_start, seg_idx, merged par / cov / n_fit "
                       "(apex / removable: tests/test_gpu_merge.py, same density)", "sectors": pick, "clusters": int(sub.n), "tracks": int(T),
            "merged": int(m["n_merged"]), "ok": not bad, "mismatches": bad,
            "seconds": round(time.perf_counter() - t0, 1)}


def optional_calls(args, tf, P, dev, stream, rank) -> dict:
    """Device times of the optional calls on the looper twin of the timed frame (same recipe + `loopers`)."""
    import torch
    import paper_2009_07515_b200 as tpc
    from tpc_synth import generate_config
    over = {"loopers": True}
    if args.collisions:
        over["n_collisions"] = args.collisions
    if rank:
        over["seed"] = replica_seed(args.workload, rank)
    tfl = generate_config(args.workload, device="cuda", **over)
    parity = optional_parity(tfl, P) if (args.parity_sectors > 0 and rank == 0) else None
    if parity and not parity["ok"]:
        raise RuntimeError(f"parity check of the optional calls failed before timing: {parity['mismatches']}")
    c = tpc.suggest_capacities(tfl.n, P)
    trk = tpc.Tracker(P, c["max_clusters"], tpc.max_bins_bound(tfl.sector, tfl.z, P), c["max_seeds"], c["max_tracks"],
                      c["max_track_clusters"], device=dev)
    d_in = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (tfl.sector, tfl.row, tfl.y, tfl.z)]
    out = trk.new_tracks(tfl.n)
    trk.track_timeframe(*d_in, out)
    k = trk.counters()
    if k["status"] != 0:
        raise RuntimeError(f"tracker status {k['status']} on the looper frame")
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn):                                         # one warm-up, one timed call, device time
        fn()
        ev0.record(stream)
        fn()
        ev1.record(stream)
        torch.cuda.synchronize(dev)
        return ev0.elapsed_time(ev1)
    fit_buf = trk.new_fit(); mg_buf = trk.new_merged(); ax_buf = trk.new_apex()
    refit_ms = timed(lambda: trk.refit_into(fit_buf))
    merge_ms = timed(lambda: trk.merge_into(fit_buf, mg_buf))
    n_merged = int(mg_buf["n_merged"].item())
    apex_ms = timed(lambda: trk.apex_into(mg_buf, ax_buf))
    n_apex = int((ax_buf["apex_partner"][:n_merged] >= 0).sum().item()) // 2
    cls = torch.zeros(tfl.n, dtype=torch.uint8, device=dev); rem = torch.zeros(tfl.n, dtype=torch.uint8, device=dev)
    removable_ms = timed(lambda: trk.removable_into(out, fit_buf, mg_buf, ax_buf, cls, rem))
    removed_frac = float(rem.float().mean().item())
    sec_leg_frac = float((cls == 2).float().mean().item())
    keep = torch.empty(tfl.n, dtype=torch.uint8, device=dev)
    protect_ms = timed(lambda: trk.protect(out, 1.0, 1.0, keep=keep))
    kept_frac = float(keep.float().mean().item())
    # truth: tracks the generator gave both legs (>= 20 clusters each)
    tid = tfl.track_id
    nmax = int(tid.max()) + 1
    c0 = np.bincount(tid[(tid >= 0) & (tfl.leg == 0)], minlength=nmax); c1 = np.bincount(tid[(tid >= 0) & (tfl.leg == 1)], minlength=nmax)
    truth_pairs = int(((c0 >= 20) & (c1 >= 20)).sum())
    res = {"frame": {"workload": tfl.name, "n_clusters": int(tfl.n), "returning_leg_clusters": int((tfl.leg == 1).sum()),
                     "n_tracks": int(k["n_tracks"])},
           "parity_before_timing": parity,
           "refit": {"what": "tpc_tracker_refit: all tracks refitted over their owned clusters", "ms": refit_ms},
           "merge": {"what": "tpc_tracker_merge: segments joined across sector borders and long holes, upward + merged downward refit",
                     "ms": merge_ms, "n_merged": n_merged},
           "apex": {"what": "tpc_tracker_apex: looper legs paired through their circles, returning leg labelled", "ms": apex_ms,
                    "pairs": n_apex, "truth_pairs_with_20_clusters_per_leg": truth_pairs},
           "removable": {"what": "tpc_tracker_removable alone (strategy A: class per cluster, protection by good tracks), buffers "
                                 "pre-allocated, device ms", "ms": removable_ms, "removed_fraction": removed_frac,
                         "secondary_leg_fraction": sec_leg_frac},
           "protect": {"what": "tpc_tracker_protect: strategy-B keep flag per cluster, 1 cm road", "ms": protect_ms,
                       "kept_fraction": kept_frac}}
    trk.destroy()
    return res


def make_timeframe(args, rank: int):
    from tpc_synth import generate_config
    import torch
    over = {}
    if args.collisions:
        over["n_collisions"] = args.collisions
    if rank:
        over["seed"] = replica_seed(args.workload, rank)                # replicas track different time frames
    dev = "cuda" if torch.cuda.is_available() and args.impl == "ours" else "cpu"
    return generate_config(args.workload, device=dev, **over)


def algorithmic_bytes(k: dict) -> dict:
    """what the method itself must move, ideal caching."""
    N, Nb, S, H, K, T = k["n_clusters"], k["n_bins"], k["kf_steps"], k["n_hits"], k["n_seeds"], k["n_tracks"]
    L = k["n_linked"]
    Ho = k["n_track_clusters"]
    b = {
        "S1": 53 * N + 8 * Nb,
        "S2": 20 * N + 4 * Nb,
        "S3": 24 * N + 4 * L + 8 * K,
        "S4": 20 * S + 8 * H + 120 * K,
        "S5": 12 * N + 32 * H + 4 * Ho + 100 * T,
    }
    b["total"] = sum(b.values())
    # the same total (i) with SURVEY.md section 8(d)'s own S2 formula (16 N + 4 N_b: no srow read) and (ii) at the 1.1 bins per
    # cluster section 8(d) assumed - the harness's cell rule (tpc_synth.choose_cell, scale 0.5) gives ~3 bins per cluster
    # because that is faster for S2 / S4, and those extra bin_start entries are bytes the method does not need
    b["total_survey_S2"] = b["total"] - 4 * N
    nb11 = int(1.1 * N)
    b["total_at_1p1_bins_per_cluster"] = b["total_survey_S2"] - (8 + 4) * (Nb - nb11)
    return b


def aggregate_over_ranks(ms_device: float, ms_e2e: float, n_clusters: int, world: int, device=None):
    """Replicas only: the job's time is the MAX over ranks, its work the SUM of the ranks'
    clusters.  The only torch.distributed traffic of the bench (besides the barriers); works on nccl and gloo."""
    if world <= 1:
        return ms_device, ms_e2e, n_clusters
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_device, ms_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    nn = torch.tensor([n_clusters], dtype=torch.int64, device=device)
    dist.all_reduce(nn, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), int(nn[0])


def replica_seed(workload: str, rank: int) -> int:
    """Rank r tracks its own time frame: the workload's seed + 1000 r."""
    from tpc_synth import CONFIGS
    return CONFIGS[workload]["seed"] + 1000 * rank


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload."""
    from oracle import Oracle
    from tpc_synth import default_params, select_sectors
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    tf = make_timeframe(args, 0)
    P = default_params(tf)           # cell chosen on the full workload, as for the CUDA arm
    # calibrate on one sector, then take as many whole sectors as fit ~100 s / (K+W) per step
    sub, _ = select_sectors(tf, [0])
    t0 = time.perf_counter()
    Oracle(P).run(sub.sector, sub.row, sub.y, sub.z)
    rate = sub.n / max(1e-9, time.perf_counter() - t0)
    budget = 100.0 / max(1, args.steps + args.warmup)
    order = list(range(tf.geometry.n_sectors))
    counts = np.bincount(tf.sector, minlength=tf.geometry.n_sectors)
    take, tot = [], 0
    for s in order:
        if take and (tot + counts[s]) / rate > budget:
            break
        take.append(s); tot += int(counts[s])
    sub, _ = select_sectors(tf, take)
    o = Oracle(P)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        o.run(sub.sector, sub.row, sub.y, sub.z)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    dt = float(np.mean(times))
    val = sub.n / dt
    sample = f"sectors {take[0]}..{take[-1]} of {tf.name} ({sub.n} of {tf.n} clusters), all five stages, fp32"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": tf.name, "n_clusters": tf.n, "sample_clusters": sub.n},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2009_07515_b200 as tpc
    from tpc_synth import default_params, select_sectors

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    t_gen = time.perf_counter()
    tf = make_timeframe(args, rank)
    t_gen = time.perf_counter() - t_gen
    P = default_params(tf)
    if args.cell_y > 0:
        P["cell_y"] = np.float32(args.cell_y)
    if args.cell_z > 0:
        P["cell_z"] = np.float32(args.cell_z)
    caps = tpc.suggest_capacities(tf.n, P)
    caps["max_bins"] = tpc.max_bins_bound(tf.sector, tf.z, P)

    # sizing run with loose capacities, then a tracker with capacities fitted to this workload
    # (x1.25): the workspace the timed runs use is what a deployment would allocate.
    th = lambda a: torch.from_numpy(np.ascontiguousarray(a))  # noqa: E731
    d_in = [th(a).to(dev) for a in (tf.sector, tf.row, tf.y, tf.z)]
    trk = tpc.Tracker(P, caps["max_clusters"], caps["max_bins"], caps["max_seeds"], caps["max_tracks"],
                      caps["max_track_clusters"], device=dev)
    out = trk.new_tracks(tf.n)
    trk.track_timeframe(*d_in, out)
    k0 = trk.counters()
    if k0["status"] != 0:
        raise RuntimeError(f"tracker status {k0['status']}")
    trk.destroy(); del trk, out
    torch.cuda.empty_cache()
    fit = lambda v, lo=1024: int(max(lo, v * 1.25 + 1))  # noqa: E731
    caps.update(max_bins=fit(k0["n_bins"]), max_seeds=fit(k0["n_seeds"]), max_tracks=fit(k0["n_tracks"]),
                max_track_clusters=fit(k0["n_track_clusters"]))
    trk = tpc.Tracker(P, caps["max_clusters"], caps["max_bins"], caps["max_seeds"], caps["max_tracks"],
                      caps["max_track_clusters"], host_io=0 if args.no_e2e else 3, device=dev)
    out = trk.new_tracks(tf.n)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- the timed configuration through the parity checker before it is timed (rank 0, a few whole sectors)
    parity = None
    if args.parity_sectors > 0 and rank == 0:
        trk.track_timeframe(*d_in, out)
        torch.cuda.synchronize(dev)
        parity = parity_precheck(tf, P, trk, out, args.parity_sectors)
        if not parity["ok"]:
            raise RuntimeError(f"parity check failed before timing: {parity['mismatches']}")

    # ---- device-timed: K steps back to back, inputs resident
    for _ in range(args.warmup):
        trk.track_timeframe(*d_in, out)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        trk.track_timeframe(*d_in, out)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    k = trk.counters()

    # ---- the same step, separately evented (>= 10 repeats): median and best next to the mean
    reps = max(10, args.repeats)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
    evs[0].record(stream)
    for i in range(reps):
        trk.track_timeframe(*d_in, out)
        evs[i + 1].record(stream)
    torch.cuda.synchronize(dev)
    per_step = np.array([evs[i].elapsed_time(evs[i + 1]) for i in range(reps)])

    # ---- the same step replayed from the cached CUDA graph (tpc_tracker_enable_graph; needs a non-default stream)
    gs = torch.cuda.Stream(device=dev)
    trk.enable_graph(True)
    with torch.cuda.stream(gs):
        for _ in range(2):
            trk.track_timeframe(*d_in, out, stream=gs)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(gs)
        for _ in range(args.steps):
            trk.track_timeframe(*d_in, out, stream=gs)
        g1.record(gs)
        gs.synchronize()
    graph_ms = g0.elapsed_time(g1) / args.steps
    trk.enable_graph(False)

    # ---- per-stage device times (events recorded inside the library, separate untimed-by-value runs)
    trk.enable_stage_timing(True)
    stage = np.zeros(5)
    for _ in range(args.steps):
        trk.track_timeframe(*d_in, out)
        stage += np.array(trk.stage_ms())
    stage /= args.steps
    trk.enable_stage_timing(False)

    # ---- the optional calls (refit, merge, apex, removable, protect: separate calls, not part of the step).  They are timed
    # on the frame they were built for: the same workload WITH the returning legs of the loopers (generator key `loopers`),
    # on a tracker of its own, after a parity check of exactly these calls against the oracle.
    opt = optional_calls(args, tf, P, dev, stream, rank) if not args.no_optional else None

    # ---- end to end through the host entry points (pinned host buffers in and out).  Time frames arrive one after the
    # other, so the pipelined begin/end pair is the call a user makes: every step still does the H2D
    # copy of its own inputs and the D2H copy of its own tracks, but the copies of one frame overlap the kernels of
    # its neighbours.  Wall clock around K steps, nothing in flight before or after.
    e2e = None
    if not args.no_e2e:
        h_in = [th(a).pin_memory() for a in (tf.sector, tf.row, tf.y, tf.z)]
        NS = 3                                         # staging slots = frames in flight
        h_out = [trk.new_tracks(tf.n, host=True) for _ in range(NS)]
        for i in range(min(2, args.warmup)):
            trk.track_timeframe_host_begin(*h_in, i % NS)
            trk.track_timeframe_host_end(h_out[i % NS], i % NS)
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            trk.track_timeframe_host_begin(*h_in, i % NS)
            if i >= NS - 1:
                j = i - (NS - 1)
                trk.track_timeframe_host_end(h_out[j % NS], j % NS)
        for j in range(max(0, args.steps - (NS - 1)), args.steps):
            trk.track_timeframe_host_end(h_out[j % NS], j % NS)
        torch.cuda.synchronize(dev)
        ms_e2e = (time.perf_counter() - t0) * 1e3
        barrier()
        # the same pipeline without the per-cluster assignment in the download (cluster_track = NULL: the CSR carries it)
        h_csr = [trk.new_tracks(tf.n, host=True, with_cluster_track=False) for _ in range(NS)]
        for i in range(2):
            trk.track_timeframe_host_begin(*h_in, i % NS)
            trk.track_timeframe_host_end(h_csr[i % NS], i % NS)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for i in range(args.steps):
            trk.track_timeframe_host_begin(*h_in, i % NS)
            if i >= NS - 1:
                j = i - (NS - 1)
                trk.track_timeframe_host_end(h_csr[j % NS], j % NS)
        for j in range(max(0, args.steps - (NS - 1)), args.steps):
            trk.track_timeframe_host_end(h_csr[j % NS], j % NS)
        torch.cuda.synchronize(dev)
        ms_csr = (time.perf_counter() - t0) * 1e3 / args.steps
        d2h_csr = h_csr[0].bytes_out()
        del h_csr
        # the same, one frame at a time (no overlap), for reference
        trk.track_timeframe_host(*h_in, h_out[0])
        t0 = time.perf_counter()
        trk.track_timeframe_host(*h_in, h_out[0])
        ms_serial = (time.perf_counter() - t0) * 1e3
        e2e = {"ms": ms_e2e / args.steps, "ms_unpipelined": ms_serial, "ms_csr": ms_csr, "d2h_csr": d2h_csr,
               "h2d": int(sum(t.numel() * t.element_size() for t in h_in)), "d2h": h_out[0].bytes_out()}

    # ---- max over ranks
    ms_total, ms_e2e_max, n_total = aggregate_over_ranks(ms_total, e2e["ms"] if e2e else 0.0, tf.n, world, dev)
    if e2e:
        e2e["ms"] = ms_e2e_max
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms_total / args.steps
    value = n_total / (ms_step * 1e-3)
    peak, peak_src = hbm_peak()
    bytes_ = algorithmic_bytes(k)
    names = ["S1", "S2", "S3", "S4", "S5"]
    dom = int(np.argmax(stage))
    dom_kernel = {"S1": "S1 (sort+bin, 4 launches)", "S2": "k_neighbours", "S3": "S3 (cleaner, 6 launches)",
                  "S4": "k_tracklets", "S5": "S5 (selector, 16 launches)"}[names[dom]]
    achieved = bytes_[names[dom]] / (stage[dom] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom_kernel, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic(dom_kernel) if tf.name == "cfg5" else None, "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_[names[dom]],
                "kernel_ms": float(stage[dom]),
                # BASELINE.json asks for the HBM fraction, hence bound = "hbm"; what the kernel is really limited by:
                "counters": ncu_counters(dom_kernel) if tf.name == "cfg5" else None,
                "whole_path": {"algorithmic_bytes": bytes_["total"], "achieved": bytes_["total"] / (ms_step * 1e-3) / 1e9,
                               "frac_of_measured": bytes_["total"] / (ms_step * 1e-3) / 1e9 / peak,
                               "frac_of_8TBs": bytes_["total"] / (ms_step * 1e-3) / 1e9 / 8000.0,
                               "bins_per_cluster": k["n_bins"] / max(1, k["n_clusters"]),
                               "frac_of_measured_with_survey_S2_formula": bytes_["total_survey_S2"] / (ms_step * 1e-3) / 1e9 / peak,
                               "frac_of_measured_at_1p1_bins_per_cluster": bytes_["total_at_1p1_bins_per_cluster"] / (ms_step * 1e-3) / 1e9 / peak},
                "stage_ms": {n: float(v) for n, v in zip(names, stage)},
                "stage_bytes": {n: int(bytes_[n]) for n in names}}

    cpu = None if args.no_cpu_baseline else cpu_baseline(tf, P)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "ms_per_step_median": float(np.median(per_step)), "ms_per_step_best": float(per_step.min()),
        "repeats": int(per_step.size), "ms_per_step_cuda_graph": graph_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": tf.name, "n_clusters_per_gpu": tf.n, "n_clusters_total": n_total,
                   "parallelism": "replicas (one time frame per GPU, no collective)" if world > 1 else "single GPU",
                   "l2": "inputs larger than L2" if tf.n * 10 > 126e6 else "inputs fit L2 (small config)",
                   "cell_cm": [float(P["cell_y"]), float(P["cell_z"])], "generate_s": round(t_gen, 1),
                   "workspace_GB": round(trk.workspace_bytes / 1e9, 2)},
        "counters": {kk: int(v) for kk, v in k.items()},
        "parity_before_timing": parity,
        "optional_calls": opt,      # separate calls, not in the step; timed on the looper twin of the frame
        "roofline": roofline,
        "cpu_baseline": cpu,
        "gpu_launches": trk.launches_per_call() * args.steps,
        "clocks": clocks,
    }
    if e2e:
        line["e2e"] = {"value": n_total / (e2e["ms"] * 1e-3), "unit": UNIT, "ms_per_step": e2e["ms"],
                       "api": "tpc_track_timeframe_host_begin/_end (three staging slots)",
                       "ms_per_step_one_frame_at_a_time": e2e["ms_unpipelined"],
                       "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                       "without_cluster_track": {"what": "same pipeline, cluster_track = NULL (not downloaded; the CSR carries the assignment)",
                                                 "ms_per_step": e2e["ms_csr"], "value": tf.n * world / (e2e["ms_csr"] * 1e-3) if world == 1 else None,
                                                 "d2h_bytes_per_step": e2e["d2h_csr"]}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
