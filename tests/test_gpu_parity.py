"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): integer stages S1-S3 bit-exact on every input;
cluster-to-track assignment bit-exact on noise-free inputs; track parameters within 1e-4 relative,
covariance within 1e-3 relative; >= 99.5 % of oracle tracks matched (>= 90 % shared clusters) on noisy
inputs.  Because both sides follow the operation order of DESIGN.md section 3 without FMA contraction the
CUDA path is in fact expected to be bit-identical everywhere, and the tests report when it is.
"""
import numpy as np
import pytest
import torch

from tests.parity_util import compare_integer_stages, compare_tracklets, compare_tracks, run_gpu, run_oracle
from tpc_synth import default_params, generate_config

pytestmark = pytest.mark.gpu

PAR_TOL = 1e-4
COV_TOL = 1e-3


def _full_parity(tf, exact_assignment):
    P, trk, out = run_gpu(tf)
    o = run_oracle(tf, P)
    k = trk.counters()
    assert k["status"] == 0, k
    bad = compare_integer_stages(trk, o)
    assert not bad, bad
    t = compare_tracklets(trk, o)
    assert t["n_seeds"][0] == t["n_seeds"][1]
    assert t["par_rel"] <= PAR_TOL and t["cov_rel"] <= COV_TOL, t
    res = compare_tracks(out.numpy(), o, tf.n)
    assert res["matched_frac"] >= 0.995, res
    if exact_assignment:
        assert t["hit_mismatch_seeds"] == 0, t
        assert res["cluster_track_equal"] and res["csr_equal"], res
        g = out.numpy()
        for nm in ("sector", "first_row", "last_row", "n_clusters", "ndf"):
            assert np.array_equal(g[nm], o.get("trk_" + nm)), nm
        assert np.max(np.abs(g["par"] - o.get("trk_par").reshape(-1, 5)) /
                      np.maximum(np.abs(o.get("trk_par").reshape(-1, 5)), [1, 1, .1, .1, .1])) <= PAR_TOL
        assert np.array_equal(g["x_ref"], o.get("trk_x_ref").astype(np.float32))
        assert np.array_equal(g["z_ref"], o.get("trk_z_ref").astype(np.float32))
        assert np.array_equal(g["z_beam"], o.get("trk_z_beam").astype(np.float32))     # DESIGN.md 3.6, bit-exact
    # counters agree with the oracle's own sizes
    assert k["n_seeds"] == o.get("seed_head").shape[0]
    assert k["n_tracklets"] == int(o.get("t_kept").sum())
    assert k["n_tracks"] == o.get("trk_seed").shape[0]
    assert k["kf_steps"] == int(o.get("t_kf_steps")[0])
    return t, res


def test_cfg1_noise_free_bit_exact(cfg1_clean):
    t, res = _full_parity(cfg1_clean, exact_assignment=True)
    assert res["n_tracks"][0] > 30


def test_cfg1_smeared(cfg1):
    _full_parity(cfg1, exact_assignment=False)


def test_mini_event_all_sectors(mini_event):
    t, res = _full_parity(mini_event, exact_assignment=False)
    print(t, res)


def test_mini_timeframe_pileup(mini_tf):
    t, res = _full_parity(mini_tf, exact_assignment=False)
    print(t, res)


def test_native_time_input_bit_exact(mini_tf):
    """the z array holds native cluster times; S1 converts while it reads.  Every
    stage, the refit and z_beam bit-exact against the oracle on the same times; the sorted z the tracker works on is
    within the fp32 rounding of the time of the frame's own pseudo-z."""
    from tpc_synth import to_native_time
    tft, tp = to_native_time(mini_tf)
    P = default_params(mini_tf); P.update(tp)
    _, trk, out = run_gpu(tft, params=P)
    o = run_oracle(tft, P)
    assert trk.counters()["status"] == 0
    assert not compare_integer_stages(trk, o)
    t = compare_tracklets(trk, o)
    assert t["hit_mismatch_seeds"] == 0 and t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
    res = compare_tracks(out.numpy(), o, tft.n)
    assert res["cluster_track_equal"] and res["csr_equal"] and res["n_tracks"][0] > 1000, res
    g = out.numpy()
    assert np.array_equal(g["z_beam"], o.get("trk_z_beam").astype(np.float32))
    assert np.array_equal(g["z_ref"], o.get("trk_z_ref").astype(np.float32))
    z_in = np.empty(tft.n, np.float32); z_in[trk.stage_view("perm")] = trk.stage_view("yz").reshape(-1, 2)[:, 1]
    assert np.abs(z_in.astype(np.float64) - mini_tf.z).max() < 1e-3
    # the host path converts the same way
    _, trk_h, out_h = run_gpu(tft, params=P, host=True)
    assert np.array_equal(out_h.numpy()["cluster_track"], g["cluster_track"])


def test_native_time_input_rejects_bad_parameters_and_flags_overflowing_times(cfg1):
    import paper_2009_07515_b200 as tpc
    from tpc_synth import to_native_time
    tft, tp = to_native_time(cfg1)
    for bad in (dict(cm_per_time_unit=np.float32(0.0)), dict(cm_per_time_unit=np.float32(np.inf)),
                dict(drift_length=np.float32(np.nan))):
        P = default_params(cfg1); P.update(tp); P.update(bad)
        with pytest.raises((RuntimeError, ValueError)):
            tpc.Tracker(P, 1024, 1024, 64, 64, 1024)
    # a time so large that the z grid would need more rows than an int32 holds (or whose pseudo-z is not finite): a status
    # bit, nothing written out of bounds
    P = default_params(cfg1); P.update(tp)
    t = tft.z.copy(); t[17] = np.float32(3e38)
    import copy
    tfb = copy.copy(tft); tfb.z = t
    _, trk, out = run_gpu(tfb, params=P, caps=dict(max_bins=1 << 22), guard_bytes=1 << 20)
    assert out.numpy()["status"] & 3 and out.numpy()["n_tracks"] == 0 and trk.guards_intact()


def test_residual_codes_bit_exact_and_bad_steps_rejected(mini_tf, mini_event):
    """the optional 16-bit residual codes of tpc_tracker_refit equal the oracle's
    code for code at two resolutions (0.1 mm: the working point; 1 um: most codes saturate), the float residuals beside
    them are unchanged, entries of clusters that did not enter the fit are 0; half-given or non-positive arguments are
    INVALID_ARG."""
    for tf, steps in ((mini_tf, (0.01, 0.02)), (mini_event, (1e-4, 1e-4)), (mini_tf, (0.25, 7.0))):
        P, trk, out = run_gpu(tf)
        T = out.numpy()["n_tracks"]
        o = run_oracle(tf, P, last_stage=6).quantise_residuals(*steps)
        fit = trk.refit(T, tracks=out, steps=steps)
        assert fit["qres_y"].dtype == np.int16 and fit["qres_y"].size == o.get("fit_qres_y").size > 10_000
        assert np.array_equal(fit["qres_y"].astype(np.int32), o.get("fit_qres_y"))
        assert np.array_equal(fit["qres_z"].astype(np.int32), o.get("fit_qres_z"))
        assert np.array_equal(fit["res_y"], o.get("fit_res_y").astype(np.float32))
        assert np.array_equal(fit["par"], o.get("fit_par").astype(np.float32).reshape(-1, 5))
    assert (np.abs(fit["qres_y"]) <= 1).mean() > 0.99             # 2.5 mm steps: almost everything rounds to 0 or +-1
    buf = trk.new_fit(steps=(0.01, 0.01))
    for bad in (dict(res_step_y=0.0), dict(res_step_z=-1.0), dict(res_step_y=float("inf")), dict(res_step_z=float("nan")),
                dict(qres_z=None)):
        b = dict(buf); b.update(bad)
        if b.get("qres_z", 0) is None:
            del b["qres_z"]
        with pytest.raises(RuntimeError, match="invalid argument"):
            trk.refit_into(b, out=out)
    b = {k: v for k, v in buf.items() if k not in ("res_y", "res_z")}   # codes without the residuals
    with pytest.raises(RuntimeError, match="invalid argument"):
        trk.refit_into(b)
    trk.refit_into(buf, out=out)
    torch.cuda.synchronize()


def test_native_pad_and_time_input_bit_exact(mini_tf):
    """the y array holds native pad coordinates; S1 converts while it reads.  Every
    stage, the refit and the keep flags bit-exact against the oracle on the same pads - alone, and together with the native
    time (the detector's (pad, row, time) input); the sorted y the tracker works on is the frame's own y within the fp32
    rounding of the pad coordinate."""
    from tpc_synth import to_native_pad, to_native_time
    tfp, pp = to_native_pad(mini_tf)
    tfpt, tp = to_native_time(tfp)
    for frame, extra in ((tfp, pp), (tfpt, {**pp, **tp})):
        P = default_params(mini_tf); P.update(extra)
        _, trk, out = run_gpu(frame, params=P)
        o = run_oracle(frame, P, last_stage=6)
        assert trk.counters()["status"] == 0
        assert not compare_integer_stages(trk, o)
        t = compare_tracklets(trk, o)
        assert t["hit_mismatch_seeds"] == 0 and t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
        res = compare_tracks(out.numpy(), o, frame.n)
        assert res["cluster_track_equal"] and res["csr_equal"] and res["n_tracks"][0] > 1000, res
        g = out.numpy()
        fit = trk.refit(g["n_tracks"], tracks=out)
        assert np.array_equal(fit["par"], o.get("fit_par").astype(np.float32).reshape(-1, 5))
        assert np.array_equal(fit["res_y"], o.get("fit_res_y").astype(np.float32))
        keep = trk.protect(out, 1.0, 1.0)
        torch.cuda.synchronize()
        assert np.array_equal(keep.cpu().numpy()[: frame.n].astype(np.int32), o.protect(1.0, 1.0))
        y_in = np.empty(frame.n, np.float32); y_in[trk.stage_view("perm")] = trk.stage_view("yz").reshape(-1, 2)[:, 0]
        assert np.abs(y_in.astype(np.float64) - mini_tf.y).max() < 2e-5
    # the host path converts the same way
    _, trk_h, out_h = run_gpu(frame, params=P, host=True)
    assert np.array_equal(out_h.numpy()["cluster_track"], g["cluster_track"])


def test_native_pad_input_rejects_bad_tables_and_flags_non_finite_pads(cfg1):
    import copy
    import paper_2009_07515_b200 as tpc
    from tpc_synth import to_native_pad
    tfp, pp = to_native_pad(cfg1)
    R = cfg1.geometry.n_rows
    zero_pads = pp["n_pads"].copy(); zero_pads[7] = 0
    for bad in (dict(n_pads=zero_pads), dict(pad_pitch=np.where(np.arange(R) == 3, 0.0, pp["pad_pitch"]).astype(np.float32)),
                dict(pad_pitch=np.where(np.arange(R) == 3, np.inf, pp["pad_pitch"]).astype(np.float32)),
                dict(pad_pitch=np.where(np.arange(R) == 150, np.nan, pp["pad_pitch"]).astype(np.float32))):
        P = default_params(cfg1); P.update(pp); P.update(bad)
        with pytest.raises((RuntimeError, ValueError)):
            tpc.Tracker(P, 1024, 1024, 64, 64, 1024)
    P = default_params(cfg1); P.update(pp)
    for v in (np.inf, np.nan):
        tfb = copy.copy(tfp); tfb.y = tfp.y.copy(); tfb.y[11] = np.float32(v)
        _, trk, out = run_gpu(tfb, params=P, guard_bytes=1 << 20)
        assert out.numpy()["status"] & 1 and out.numpy()["n_tracks"] == 0 and trk.guards_intact()
    # a row id out of range with the pad flag on: rejected before the pad table is indexed
    tfb = copy.copy(tfp); tfb.row = tfp.row.copy(); tfb.row[5] = 200
    _, trk, out = run_gpu(tfb, params=P, guard_bytes=1 << 20)
    assert out.numpy()["status"] & 1 and trk.guards_intact()


def test_reports_bit_exactness(mini_event):
    """Not a requirement of north_star, but the design goal: identical op order => identical bits."""
    P, trk, out = run_gpu(mini_event)
    o = run_oracle(mini_event, P)
    t = compare_tracklets(trk, o)
    res = compare_tracks(out.numpy(), o, mini_event.n)
    assert t["hit_mismatch_seeds"] == 0 and t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
    assert res["cluster_track_equal"] and res["csr_equal"], res
    zb_g, zb_o = out.numpy()["z_beam"], o.get("trk_z_beam")
    assert zb_g.shape == zb_o.shape and np.array_equal(zb_g, zb_o.astype(np.float32))
    assert np.max(np.abs(zb_g - zb_o) / np.maximum(np.abs(zb_o), 1.0)) <= PAR_TOL   # the stated bar: 1e-4 relative


def test_host_path_equals_device_path(mini_event):
    P, trk_d, out_d = run_gpu(mini_event)
    _, trk_h, out_h = run_gpu(mini_event, host=True)
    a, b = out_d.numpy(), out_h.numpy()
    assert a["n_tracks"] == b["n_tracks"] and a["status"] == b["status"] == 0
    for k in a:
        if isinstance(a[k], np.ndarray):
            assert np.array_equal(a[k], b[k]), k


def test_host_paths_without_cluster_track(mini_event):
    """cluster_track = NULL on the host paths: nothing is copied there, everything else is unchanged."""
    tf = mini_event
    P, trk, out = run_gpu(tf, host=3)
    ref = out.numpy()
    ins = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (tf.sector, tf.row, tf.y, tf.z)]
    o2 = trk.new_tracks(tf.n, host=True, with_cluster_track=False)
    o2.cluster_track.fill_(-7)
    trk.track_timeframe_host(*ins, o2)
    a = o2.numpy()
    assert np.all(a["cluster_track"] == -7) and o2.bytes_out() == out.bytes_out() - 4 * tf.n
    for k in ref:
        if k != "cluster_track" and isinstance(ref[k], np.ndarray):
            assert np.array_equal(ref[k], a[k]), k
    o3 = trk.new_tracks(tf.n, host=True, with_cluster_track=False)
    o3.cluster_track.fill_(-7)
    trk.track_timeframe_host_begin(*ins, 1)
    trk.track_timeframe_host_end(o3, 1)
    b = o3.numpy()
    assert np.all(b["cluster_track"] == -7) and np.array_equal(b["trk_cl_idx"], ref["trk_cl_idx"]) and b["n_tracks"] == ref["n_tracks"]


def test_cuda_graph_path_gives_the_same_result_and_recaptures_on_new_arguments(mini_event, cfg1):
    """tpc_tracker_enable_graph: the cached graph replays while the arguments stay the same, is re-captured when they change
    (other buffers, other n), and every result equals the direct launches."""
    tf = mini_event
    P, trk, out = run_gpu(tf)
    ref = out.numpy()
    s = torch.cuda.Stream()
    trk.enable_graph(True)
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (tf.sector, tf.row, tf.y, tf.z)]
    o1 = trk.new_tracks(tf.n)
    with torch.cuda.stream(s):
        for _ in range(3):                                  # capture, then two replays
            trk.track_timeframe(*ins, o1, stream=s)
        s.synchronize()
    a = o1.numpy()
    for k in ref:
        if isinstance(ref[k], np.ndarray):
            assert np.array_equal(ref[k], a[k]), k
    # other input buffers with fewer clusters: re-capture
    keep = tf.sector < 9
    ins2 = [torch.from_numpy(np.ascontiguousarray(x[keep])).cuda() for x in (tf.sector, tf.row, tf.y, tf.z)]
    o2 = trk.new_tracks(int(keep.sum()))
    with torch.cuda.stream(s):
        trk.track_timeframe(*ins2, o2, stream=s); trk.track_timeframe(*ins2, o2, stream=s)
        s.synchronize()
    trk.enable_graph(False)
    o3 = trk.new_tracks(int(keep.sum()))
    trk.track_timeframe(*ins2, o3)
    torch.cuda.synchronize()
    b, c3 = o2.numpy(), o3.numpy()
    assert b["n_tracks"] == c3["n_tracks"] > 0 and np.array_equal(b["cluster_track"], c3["cluster_track"]) and np.array_equal(b["par"], c3["par"])
    # the stage views and the separate calls work after a replay as after a direct call
    trk.enable_graph(True)
    with torch.cuda.stream(s):
        trk.track_timeframe(*ins, o1, stream=s)
        s.synchronize()
    assert np.array_equal(trk.stage_view("perm"), run_oracle(tf, P, last_stage=1).get("perm"))


def test_graph_mode_inside_a_capture_of_the_callers_own(mini_event):
    """A framework that records its own CUDA graph around the tracker: with graph mode on, tpc_track_timeframe must not
    begin a second capture on that stream (it would fail and break the caller's) - its launches go into the caller's
    graph, and replaying that graph gives the result of the direct launches."""
    tf = mini_event
    P, trk, out = run_gpu(tf)
    ref = out.numpy()
    trk.enable_graph(True)
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (tf.sector, tf.row, tf.y, tf.z)]
    o1 = trk.new_tracks(tf.n)
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        trk.track_timeframe(*ins, o1, stream=torch.cuda.current_stream())
    o1.n_tracks.zero_()
    g.replay()
    torch.cuda.synchronize()
    a = o1.numpy()
    assert a["n_tracks"] == ref["n_tracks"] > 0
    for k in ref:
        if isinstance(ref[k], np.ndarray):
            assert np.array_equal(ref[k], a[k]), k
    # and the handle's own graph path still works afterwards on an ordinary stream
    with torch.cuda.stream(s):
        trk.track_timeframe(*ins, o1, stream=s); trk.track_timeframe(*ins, o1, stream=s)
        s.synchronize()
    assert np.array_equal(o1.numpy()["cluster_track"], ref["cluster_track"])


def test_repeatable_and_reusable(mini_event):
    """Two calls on one handle give identical results (ids come from scans, not from atomics)."""
    import paper_2009_07515_b200 as tpc
    tf = mini_event
    P, trk, out1 = run_gpu(tf)
    a = out1.numpy()
    ins = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (tf.sector, tf.row, tf.y, tf.z)]
    out2 = trk.new_tracks(tf.n)
    for _ in range(2):
        trk.track_timeframe(*ins, out2)
    torch.cuda.synchronize()
    b = out2.numpy()
    for k in a:
        if isinstance(a[k], np.ndarray):
            assert np.array_equal(a[k], b[k]), k


def test_edge_cases():
    import paper_2009_07515_b200 as tpc
    tf = generate_config("cfg1")
    P = default_params(tf)
    # empty input
    empty = generate_config("cfg1", n_tracks=0)
    assert empty.n == 0
    _, trk, out = run_gpu(empty, params=P, caps=dict(max_bins=1024))
    g = out.numpy()
    assert g["n_tracks"] == 0 and g["status"] == 0
    # ragged sizes around the vector width, single cluster, everything in one bin
    for n in (1, 2, 3, 5, 255, 257, 1023):
        sub = generate_config("cfg1")
        for f in ("sector", "row", "x", "y", "z", "track_id"):
            setattr(sub, f, getattr(sub, f)[:n].copy())
        Pn, trk, out = run_gpu(sub, params=P)
        o = run_oracle(sub, Pn)
        assert not compare_integer_stages(trk, o), n
        assert np.array_equal(out.numpy()["cluster_track"], o.get("cluster_track"))
    # duplicates: ties must keep input order (stable)
    dup = generate_config("cfg1")
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        a = getattr(dup, f)
        setattr(dup, f, np.concatenate([a, a]))
    Pd, trk, out = run_gpu(dup, params=P)
    o = run_oracle(dup, Pd)
    assert not compare_integer_stages(trk, o)
    assert np.array_equal(out.numpy()["cluster_track"], o.get("cluster_track"))
    # bad cluster -> status bit, no tracks
    bad = generate_config("cfg1")
    bad.row = bad.row.copy(); bad.row[7] = 200
    _, trk, out = run_gpu(bad, params=P)
    g = out.numpy()
    assert g["status"] & 1 and g["n_tracks"] == 0
    # capacity overflow is reported, never silent
    _, trk, out = run_gpu(tf, params=P, caps=dict(max_seeds=3))
    g = out.numpy()
    assert g["status"] & 4 and g["n_tracks"] == 0
    _, trk, out = run_gpu(tf, params=P, caps=dict(max_bins=100))
    assert out.numpy()["status"] & 2
    _, trk, out = run_gpu(tf, params=P, caps=dict(max_tracks=2))
    assert out.numpy()["status"] & 8


def test_full_size_whole_frame_every_array_exact():
    """cfg5 at full size, launched as bench.py launches it, compared with the oracle on ALL 36 sectors (DESIGN.md section
    5): sectors are independent (one z range per sector, section 3.1), so the oracle run on the clusters of one sector must
    reproduce the CUDA arrays restricted to it.  Every array is compared with np.array_equal - sorted order, grid
    (bin_start, bin_base, z range), raw and cleaned links, seeds, the tracklet tables (hits, rows, parameters,
    covariance, chi2), ownership, tracks (assignment, CSR, parameters, covariance, z_beam), the refit with its
    residuals, and the strategy-B keep flags.  No thresholds."""
    import time
    from tests.parity_util import check_sectors_parallel, collect_gpu_frame
    tf = generate_config("cfg5", device="cuda")
    P, trk, out = run_gpu(tf)
    k = trk.counters()
    assert k["status"] == 0 and k["n_clusters"] == tf.n > 50_000_000
    frame = collect_gpu_frame(tf, P, trk, out)
    del trk, out
    torch.cuda.empty_cache()
    t0 = time.perf_counter()
    bad, stats, procs = check_sectors_parallel(frame, range(P["n_sectors"]))
    dt = time.perf_counter() - t0
    assert sum(st["n"] for st in stats.values()) == tf.n
    assert sum(st["tracks"] for st in stats.values()) == k["n_tracks"] == frame["out"]["n_tracks"]
    assert sum(st["seeds"] for st in stats.values()) == k["n_seeds"]
    print(f"cfg5: {tf.n} clusters, {k['n_tracks']} tracks, 36 sectors checked by {procs} processes in {dt:.1f} s")
    assert not any(bad.values()), {s: b for s, b in bad.items() if b}


def test_wide_ownership_keys(mini_event):
    """S5 uses 32-bit ownership keys when every seed id fits 24 bits and 64-bit keys otherwise: a capacity above 2^24
    seeds forces the wide path (~12 GB of workspace), which must give the same tracks."""
    P, trk32, out32 = run_gpu(mini_event)
    _, trk64, out64 = run_gpu(mini_event, caps=dict(max_seeds=(1 << 24) + 1))
    a, b = out32.numpy(), out64.numpy()
    assert a["status"] == b["status"] == 0 and a["n_tracks"] == b["n_tracks"] > 0
    for k in a:
        if isinstance(a[k], np.ndarray):
            assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(trk32.stage_view("k_owned"), trk64.stage_view("k_owned")[: trk32.stage_view("k_owned").shape[0]])


@pytest.mark.parametrize("slots", [2, 3])
def test_pipelined_host_path(mini_event, mini_tf, slots):
    """tpc_track_timeframe_host_begin/_end with `slots` frames in flight gives, frame by frame, what the device path gives."""
    import paper_2009_07515_b200 as tpc
    frames = [mini_event, mini_tf, mini_event, mini_tf, mini_tf, mini_event, mini_event]
    P = default_params(mini_event)
    want = {}
    for tf in (mini_event, mini_tf):
        _, _, out = run_gpu(tf, params=P)
        want[id(tf)] = out.numpy()
    nmax = max(tf.n for tf in frames)
    c = tpc.suggest_capacities(nmax, P)
    nb = max(tpc.max_bins_bound(tf.sector, tf.z, P) for tf in frames)
    trk = tpc.Tracker(P, c["max_clusters"], nb, c["max_seeds"], c["max_tracks"], c["max_track_clusters"], host_io=slots)
    th = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
    pinned = {id(tf): [th(a) for a in (tf.sector, tf.row, tf.y, tf.z)] for tf in (mini_event, mini_tf)}
    outs = [trk.new_tracks(nmax, host=True) for _ in range(slots)]
    got = []

    def finish(i):
        trk.track_timeframe_host_end(outs[i % slots], i % slots)
        o = outs[i % slots]; o.n_in = frames[i].n
        got.append(o.numpy())

    for i in range(len(frames)):
        trk.track_timeframe_host_begin(*pinned[id(frames[i])], i % slots)
        if i >= slots - 1:
            finish(i - (slots - 1))
    for j in range(len(frames) - (slots - 1), len(frames)):
        finish(j)
    assert len(got) == len(frames)
    for tf, g in zip(frames, got):
        w = want[id(tf)]
        assert g["status"] == 0 and g["n_tracks"] == w["n_tracks"] > 0
        for k in w:
            if isinstance(w[k], np.ndarray):
                assert np.array_equal(g[k], w[k]), k
    # a slot used out of order, or one the tracker does not have, is refused
    with pytest.raises(RuntimeError):
        trk.track_timeframe_host_end(outs[0], 0)
    with pytest.raises(RuntimeError):
        trk.track_timeframe_host_begin(*pinned[id(mini_event)], slots)


def test_crowded_slab_falls_back_and_stays_exact():
    """5000 tracks (2 x 2250 per row) squeezed into +-5 cm of z of one sector, one bin row per (sector,row) bucket: the bucket's only z-slab
    holds more clusters than the shared-memory tables of the bin sort take (global-memory path), the link windows hold
    far more than kCap candidates (rectangle re-walk in S2), and bins hold many clusters (stable order by input index)."""
    tf = generate_config("cfg1", n_tracks=5000, seed=7)
    tf.z = (tf.z * np.float32(0.02)).astype(np.float32)
    P = default_params(tf, cell=4.0)
    P["cell_z"] = np.float32(16.0)
    Pg, trk, out = run_gpu(tf, params=P)
    o = run_oracle(tf, P)
    assert trk.counters()["status"] == 0
    assert int(np.diff(trk.stage_view("row_start")).max()) > 2048
    assert trk.counters()["s1_global_buckets"] > 0             # the fallback path really ran
    bad = compare_integer_stages(trk, o)
    assert not bad, bad
    t = compare_tracklets(trk, o)
    assert t["hit_mismatch_seeds"] == 0 and t["par_rel"] <= PAR_TOL and t["cov_rel"] <= COV_TOL, t
    res = compare_tracks(out.numpy(), o, tf.n)
    assert res["cluster_track_equal"] and res["csr_equal"], res


@pytest.mark.parametrize("which", ["cfg1", "mini_event", "mini_tf"])
def test_refit_parity(which, cfg1, mini_event, mini_tf):
    """tpc_tracker_refit against the oracle's refit: bit-exact, and within the stated bars."""
    tf = {"cfg1": cfg1, "mini_event": mini_event, "mini_tf": mini_tf}[which]
    P, trk, out = run_gpu(tf)
    o = run_oracle(tf, P, last_stage=6)
    g = out.numpy()
    T = g["n_tracks"]
    assert T == o.get("trk_seed").shape[0] > 0
    fit = trk.refit(T, tracks=out)
    assert np.array_equal(fit["n_fit"], o.get("fit_n")) and np.array_equal(fit["ndf"], o.get("fit_ndf"))
    # residuals to the extrapolated track, parallel to trk_cl_idx
    assert fit["res_y"].shape == g["trk_cl_idx"].shape
    assert np.array_equal(fit["res_y"], o.get("fit_res_y").astype(np.float32))
    assert np.array_equal(fit["res_z"], o.get("fit_res_z").astype(np.float32))
    ref = o.get("fit_par").reshape(-1, 5)
    assert np.max(np.abs(fit["par"] - ref) / np.maximum(np.abs(ref), [1, 1, .1, .1, .1])) <= PAR_TOL
    for nm, key in (("par", "fit_par"), ("cov", "fit_cov"), ("chi2", "fit_chi2"), ("x_ref", "fit_x_ref"), ("z_ref", "fit_z_ref")):
        want = o.get(key).astype(np.float32).reshape(fit[nm].shape)
        assert np.array_equal(fit[nm], want), nm
    # the refit leaves the tracks of the call untouched and can be repeated
    again = trk.refit(T)                                   # without residuals
    assert all(np.array_equal(fit[k], again[k]) for k in again)


def test_non_uniform_pad_row_pitch():
    """A 4-region pad-row pitch: up and down row distances differ at the region borders; every
    stage and the refit must still match the oracle bit for bit."""
    from tpc_synth import FOUR_REGION_PITCH, Geometry, generate
    from tpc_synth.generator import CONFIGS
    rec = dict(CONFIGS["cfg3"]); rec.update(n_collisions=2, seed=9)
    tf = generate(rec, geometry=Geometry(pitch_regions=FOUR_REGION_PITCH))
    t, res = _full_parity(tf, exact_assignment=True)
    assert t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
    P, trk, out = run_gpu(tf)
    o = run_oracle(tf, P, last_stage=6)
    fit = trk.refit(out.numpy()["n_tracks"])
    assert np.array_equal(fit["par"], o.get("fit_par").astype(np.float32).reshape(-1, 5))
    assert np.array_equal(fit["n_fit"], o.get("fit_n"))


@pytest.mark.parametrize("over", [
    dict(min_chain_len=2, max_gap=0, min_tracklet_hits=3, min_track_hits=2),
    dict(max_sinphi=np.float32(0.5), pick_chi2_cut=np.float32(4.0)),        # many propagation failures (phase A cut short)
    dict(min_chain_len=6, max_gap=8, link_T=np.float32(0.2), y_margin=np.float32(0.0)),
])
def test_other_cuts_and_rare_paths(over):
    """Different cuts push the rare branches: chains of two, no gap allowed, propagation failures inside phase A (the
    chain length is then counted past the failure), tight link cut.  Everything stays bit-exact."""
    tf = generate_config("cfg2", n_tracks=600, noise=0.2, seed=13)
    P = default_params(tf)
    P.update(over)
    Pg, trk, out = run_gpu(tf, params=P)
    o = run_oracle(tf, P, last_stage=6)
    assert trk.counters()["status"] == 0
    bad = compare_integer_stages(trk, o)
    assert not bad, bad
    t = compare_tracklets(trk, o)
    assert t["hit_mismatch_seeds"] == 0 and t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
    res = compare_tracks(out.numpy(), o, tf.n)
    assert res["cluster_track_equal"] and res["csr_equal"], res
    T = out.numpy()["n_tracks"]
    if T:
        fit = trk.refit(T)
        assert np.array_equal(fit["n_fit"], o.get("fit_n"))
        assert np.array_equal(fit["par"], o.get("fit_par").astype(np.float32).reshape(-1, 5))


@pytest.mark.parametrize("which,road", [("cfg1", (2.0, 2.0)), ("mini_event", (1.0, 3.0)), ("mini_tf", (0.5, 0.5)), ("mini_tf", (0.0, 0.0))])
def test_protect_parity(which, road, cfg1, mini_event, mini_tf):
    """tpc_tracker_protect (strategy B of PAPER.md:57-61) against the oracle: identical flags."""
    tf = {"cfg1": cfg1, "mini_event": mini_event, "mini_tf": mini_tf}[which]
    P, trk, out = run_gpu(tf)
    o = run_oracle(tf, P, last_stage=5)
    keep = trk.protect(out, *road)
    torch.cuda.synchronize()
    got = keep.cpu().numpy()[: tf.n].astype(np.int32)
    want = o.protect(*road)
    assert np.array_equal(got, want)
    assert np.all(got[out.numpy()["cluster_track"] >= 0] == 1)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4"])
def test_full_size_small_configs(name):
    """BASELINE.json configs[1..3] at their full sizes (0.8 M, 1.6 M, 3.0 M clusters): every stage, the refit and the
    protection flags bit-exact against the oracle."""
    tf = generate_config(name)
    t, res = _full_parity(tf, exact_assignment=True)
    assert t["par_bitexact"] and t["cov_bitexact"] and t["chi2_bitexact"], t
    P, trk, out = run_gpu(tf)
    o = run_oracle(tf, P, last_stage=6)
    T = out.numpy()["n_tracks"]
    fit = trk.refit(T, tracks=out)
    assert np.array_equal(fit["par"], o.get("fit_par").astype(np.float32).reshape(-1, 5))
    assert np.array_equal(fit["res_y"], o.get("fit_res_y").astype(np.float32))
    keep = trk.protect(out, 1.0, 1.0)
    torch.cuda.synchronize()
    assert np.array_equal(keep.cpu().numpy()[: tf.n].astype(np.int32), o.protect(1.0, 1.0))


@pytest.mark.parametrize("field,value,bit", [
    ("z", np.inf, 1), ("z", -np.inf, 1), ("z", np.nan, 1), ("y", np.inf, 1), ("y", np.nan, 1),
    ("z", 1e30, 2), ("z", -3e38, 2),
])
def test_non_finite_and_huge_coordinates_set_a_status_bit_and_write_nothing_out_of_bounds(field, value, bit, cfg1):
    """Precondition 'coordinates finite' (tpc_tracker.h): a NaN / Inf coordinate is a BAD_CLUSTER, a finite |z| so large
    that the z grid needs more rows than an int32 holds is a BINS_OVERFLOW - a status bit and zero tracks, never a wrapped
    bin count and writes outside the workspace (guard bytes on both sides of the arena stay intact).  The handle stays
    usable: the next, clean frame gives the clean result."""
    import copy
    tf = copy.copy(cfg1)
    P = default_params(cfg1)
    a = getattr(tf, field).copy(); a[1234] = value
    setattr(tf, field, a)
    caps = dict(max_bins=1 << 22)
    _, trk, out = run_gpu(tf, params=P, caps=caps, guard_bytes=1 << 20)
    g = out.numpy()
    assert g["status"] & bit and g["n_tracks"] == 0, g["status"]
    assert trk.guards_intact()
    ins = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (cfg1.sector, cfg1.row, cfg1.y, cfg1.z)]
    out2 = trk.new_tracks(cfg1.n)
    trk.track_timeframe(*ins, out2)
    torch.cuda.synchronize()
    o = run_oracle(cfg1, P, last_stage=5)
    assert out2.numpy()["status"] == 0 and np.array_equal(out2.numpy()["cluster_track"], o.get("cluster_track"))
    assert trk.guards_intact()
    from oracle import Oracle
    with pytest.raises(ValueError):                       # the oracle refuses the same inputs
        Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)


@pytest.mark.parametrize("S,R", [(46, 256), (47, 251), (255, 257 - 1), (36, 152)])
def test_many_sector_row_buckets_around_the_shared_histogram_limit(S, R):
    """S*R = 11776 is the last geometry whose (sector,row) histogram of k_zrange_count fits the 48 KB of shared memory a
    kernel gets without opting in; 11797 and 65280 take the global-atomics path.  Random clusters, S1-S3 bit-exact."""
    from tpc_synth import Geometry
    from tpc_synth.generator import TimeFrame
    g = Geometry(n_sectors=S, n_rows=R)
    rng = np.random.default_rng(S * 1000 + R)
    n = 40_000
    sector = rng.integers(0, S, n).astype(np.uint8); row = rng.integers(0, R, n).astype(np.uint8)
    ymax = g.row_x()[row] * g.tan_half_sector
    y = (rng.uniform(-1, 1, n) * ymax).astype(np.float32); z = rng.uniform(-250, 250, n).astype(np.float32)
    tf = TimeFrame(sector=sector, row=row, x=g.row_x().astype(np.float32)[row], y=y, z=z, track_id=np.full(n, -1, np.int32),
                   truth={}, geometry=g)
    P = default_params(tf, cell=8.0)
    Pg, trk, out = run_gpu(tf, params=P, guard_bytes=1 << 16)
    o = run_oracle(tf, P, last_stage=5)
    assert trk.counters()["status"] == 0
    bad = compare_integer_stages(trk, o)
    assert not bad, bad
    assert np.array_equal(out.numpy()["cluster_track"], o.get("cluster_track"))
    assert trk.guards_intact()
