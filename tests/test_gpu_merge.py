"""GPU parity of the track merger (tpc_tracker_merge) against the oracle: every intermediate array
(upward refit, best partners with their chi2, links) and every output (merged ids, CSR of segments, merged refit)
bit-exact, on a central event, a piled-up slice, the 4-region pitch, with other cuts, and at the full size of cfg2-cfg4."""
import numpy as np
import pytest
import torch

from tests.parity_util import run_gpu, run_oracle
from tpc_synth import default_params, generate_config

pytestmark = pytest.mark.gpu

CUTS = dict(max_rows=30, back_rows=1, edge=6.0, dz_win=50.0, chi2_cut=100.0, road_z0=2.0, road_z1=0.3)


def _merge_parity(tf, P=None, cuts=None, min_links=1):
    kw = dict(CUTS); kw.update(cuts or {})
    P, trk, out = run_gpu(tf, params=P)
    g = out.numpy()
    T = g["n_tracks"]
    m = trk.merge(T, kw)
    o = run_oracle(tf, P, last_stage=6).merge(**kw)
    links = _compare_merge(trk, m, o, T)
    assert links >= min_links, links
    return m, o, links


def _compare_merge(trk, m, o, T):
    """Every intermediate and output array of tpc_tracker_merge (`m` = Tracker.merge's host copies) against the oracle `o`
    after its merge(): asserts equality, returns the number of links."""
    f32 = np.float32
    mt = trk.caps[3]
    bad = []

    def eq(name, a, b):
        a = np.asarray(a); b = np.asarray(b)
        if a.shape != b.shape or not np.array_equal(a, b):
            bad.append(f"{name}: {a.shape} vs {b.shape}" if a.shape != b.shape else f"{name}: {int((a != b).sum())} of {a.size} differ")

    assert T == o.get("trk_seed").size
    # 3.9.1 upward refit
    eq("fit_row", trk.stage_view("fit_row"), o.get("fit_row"))
    eq("up_par", trk.stage_view("up_par").reshape(5, mt)[:, :T].T, o.get("up_par").astype(f32).reshape(-1, 5))
    eq("up_cov", trk.stage_view("up_cov").reshape(15, mt)[:, :T].T, o.get("up_cov").astype(f32).reshape(-1, 15))
    eq("up_x", trk.stage_view("up_x"), o.get("up_x_ref").astype(f32))
    eq("up_zref", trk.stage_view("up_zref"), o.get("up_z_ref").astype(f32))
    eq("up_row", trk.stage_view("up_row"), o.get("up_row"))
    eq("up_n", trk.stage_view("up_n"), o.get("up_n"))
    # 3.9.3 - 3.9.5 choice
    eq("best_b", trk.stage_view("mrg_best_b"), o.get("mrg_best_b"))
    eq("chi_b", trk.stage_view("mrg_chi_b"), o.get("mrg_chi2_b").astype(f32))
    key = trk.stage_view("mrg_best_a")
    eq("best_a", np.where(key == np.uint64(0xFFFFFFFFFFFFFFFF), -1, (key & np.uint64(0xFFFFFFFF)).astype(np.int64)), o.get("mrg_best_a"))
    for nm in ("next", "prev", "dir"):
        eq(nm, trk.stage_view("mrg_" + nm), o.get("mrg_" + nm))
    # 3.9.6 chains
    eq("n_merged", m["n_merged"], o.get("mrg_seg_start").size - 1)
    eq("merged_of_track", m["merged_of_track"], o.get("mrg_of_track"))
    eq("seg_start", m["seg_start"], o.get("mrg_seg_start"))
    eq("seg_idx", m["seg_idx"], o.get("mrg_seg_idx"))
    # 3.9.7 merged refit
    eq("par", m["par"], o.get("mrg_par").astype(f32).reshape(-1, 5))
    eq("cov", m["cov"], o.get("mrg_cov").astype(f32).reshape(-1, 15))
    for nm in ("x_ref", "z_ref", "chi2"):
        eq(nm, m[nm], o.get("mrg_" + nm).astype(f32))
    for nm in ("ndf", "n_fit", "sector", "n_clusters"):
        eq(nm, m[nm], o.get("mrg_" + nm))
    if bad:
        for nm in ("best_b", "best_a"):
            gk = trk.stage_view("mrg_" + nm)
            gk = np.where(gk == np.uint64(0xFFFFFFFFFFFFFFFF), -1, (gk & np.uint64(0xFFFFFFFF)).astype(np.int64)) if nm == "best_a" else gk
            w = np.nonzero(gk != o.get("mrg_" + nm))[0][:5]
            bad.append((nm, w.tolist(), gk[w].tolist(), o.get("mrg_" + nm)[w].tolist(), trk.stage_view("mrg_chi_b")[w].tolist(), o.get("mrg_chi2_b")[w].tolist()))
    assert not bad, bad
    return int((o.get("mrg_next") >= 0).sum())


def test_merge_central_event(mini_event):
    m, o, links = _merge_parity(mini_event, min_links=300)
    assert (o.get("mrg_dir") != 0).sum() > 300


def test_merge_piled_up_slice_and_repeat(mini_tf):
    m, o, links = _merge_parity(mini_tf, min_links=3000)
    # the call is repeatable on the same handle state (ids come from scans, choices from order-independent minima)
    P, trk, out = run_gpu(mini_tf)
    T = out.numpy()["n_tracks"]
    a = trk.merge(T); b = trk.merge(T)
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_merge_other_cuts_and_long_holes(mini_tf):
    """A wide row window and z window, a loose and a very tight chi2 cut, no neighbour search at all (edge = 0 keeps only
    ends outside the sector), rows removed from the frame so that same-sector links (dir = 0) occur."""
    import copy
    tf = copy.copy(mini_tf)
    keep = ~np.isin(tf.row, np.arange(70, 76))
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        setattr(tf, f, getattr(mini_tf, f)[keep].copy())
    m, o, links = _merge_parity(tf, cuts=dict(max_rows=40), min_links=3000)
    assert ((o.get("mrg_next") >= 0) & (o.get("mrg_dir") == 0)).sum() > 300
    _merge_parity(mini_tf, cuts=dict(max_rows=60, dz_win=120.0, chi2_cut=400.0, road_z0=1e9), min_links=3000)
    _merge_parity(mini_tf, cuts=dict(road_z0=0.05, road_z1=0.01), min_links=500)
    _merge_parity(mini_tf, cuts=dict(chi2_cut=2.0), min_links=100)
    _merge_parity(mini_tf, cuts=dict(edge=0.0, back_rows=0), min_links=0)


def test_merge_non_uniform_pitch():
    from tpc_synth import FOUR_REGION_PITCH, Geometry, generate
    from tpc_synth.generator import CONFIGS
    rec = dict(CONFIGS["cfg2"]); rec.update(n_tracks=600, seed=31)
    tf = generate(rec, geometry=Geometry(pitch_regions=FOUR_REGION_PITCH, x_last=85.0 + 0.75 * 62.5 + 1.0 * 34 + 1.2 * 30 + 1.5 * 25))
    _merge_parity(tf, min_links=200)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4"])
def test_merge_full_size_configs(name):
    tf = generate_config(name, device="cuda")
    m, o, links = _merge_parity(tf, min_links=5000)
    print(name, "tracks", o.get("trk_seed").size, "merged", m["n_merged"], "links", links)


def test_merge_at_time_frame_density():
    """Six whole sectors of the 50 kHz Pb-Pb time frame (cfg5: 11.4 ms of z, 5 % noise) as a frame of their own: three
    neighbours on the A side, three on the C side, ~15 M clusters."""
    from tpc_synth import select_sectors
    tf = generate_config("cfg5", device="cuda")
    sub, _ = select_sectors(tf, [0, 1, 2, 20, 21, 22])
    del tf
    P = default_params(sub)
    m, o, links = _merge_parity(sub, P=P, min_links=50000)
    print("tracks", o.get("trk_seed").size, "merged", m["n_merged"], "links", links)


def test_merge_at_the_density_and_z_span_of_the_time_frame_with_loopers():
    """The frame bench.py times the optional calls on: cfg5 (50 kHz Pb-Pb, 11.4 ms of z) WITH the returning legs of the
    loopers.  Twelve whole sectors - six neighbours around the 17|0 wrap on the A side and their mirror on the C side - as
    a frame of their own (~46 M clusters, 1.1 M tracks, the full +-28 500 cm of z): assignment, every intermediate of the
    merger and the merged refit against the oracle, np.array_equal.  apex / removable are not part of it: the oracle's apex
    step is an all-pairs scan by definition, quadratic in the merged tracks (two sectors of this frame took it 6.5 minutes
    on the B200 box - every array came out identical - and a two-sector cut holds almost no complete looper; DESIGN.md
    section 5)."""
    import time
    from tpc_synth import select_sectors
    tf = generate_config("cfg5", device="cuda", loopers=True)
    assert tf.n > 50_000_000 and int((tf.leg == 1).sum()) > 1_000_000
    P = default_params(tf)
    t0 = time.perf_counter()
    sub, _ = select_sectors(tf, [15, 16, 17, 0, 1, 2, 33, 34, 35, 18, 19, 20])
    assert float(sub.z.max()) - float(sub.z.min()) > 50_000
    _, trk, out = run_gpu(sub, params=P)
    g = out.numpy()
    T = g["n_tracks"]
    assert g["status"] == 0 and T > 200_000
    m = trk.merge(T, CUTS, fill=POISON)
    o = run_oracle(sub, P, last_stage=6)
    assert np.array_equal(g["cluster_track"], o.get("cluster_track"))
    links = _compare_merge(trk, m, o.merge(**CUTS), T)
    t1 = time.perf_counter()
    print(f"12 sectors of cfg5 + loopers: {sub.n} clusters, {T} tracks, {m['n_merged']} merged, {links} links ({t1 - t0:.0f} s)")
    assert links > 50_000


def test_merge_rejects_bad_arguments(cfg1):
    import ctypes as C
    import paper_2009_07515_b200 as tpc
    P, trk, out = run_gpu(cfg1)
    fit = trk.new_fit(); mg = trk.new_merged()
    trk.refit_into(fit)
    for bad in (dict(dz_win=0.0), dict(dz_win=float("inf")), dict(max_rows=-1), dict(chi2_cut=float("nan")), dict(edge=-1.0), dict(road_z0=-1.0)):
        with pytest.raises(RuntimeError):
            trk.merge_into(fit, mg, bad)
    trk.merge_into(fit, mg)
    torch.cuda.synchronize()
    assert int(mg["n_merged"].item()) >= 1


def test_buffers_smaller_than_the_frames_max_tracks_are_refused(cfg1):
    """refit / merge / apex / removable index their per-track buffers by track id up to n_tracks <= the max_tracks of the
    tpc_track_timeframe call: any buffer declared smaller than that is CAPACITY (-2) - no out-of-bounds access, no
    silently shortened result."""
    import ctypes as C
    import paper_2009_07515_b200 as tpc
    from paper_2009_07515_b200.binding import (_MERGED_FIELDS, tpc_apex_cuts_t, tpc_apex_t, tpc_fit_t, tpc_merge_cuts_t,
                                               tpc_merged_t, tpc_removal_cuts_t)
    P, trk, out = run_gpu(cfg1)
    lib, h, mt = trk.lib, trk._h, trk.caps[3]
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    fit = trk.new_fit(); mg = trk.new_merged(); ax = trk.new_apex()

    def fit_s(n):
        f = tpc_fit_t(); f.max_tracks = n
        for k in ("par", "cov", "x_ref", "z_ref", "chi2", "ndf", "n_fit"):
            setattr(f, k, fit[k].data_ptr())
        return f

    def mrg_s(n):
        m = tpc_merged_t(); m.max_tracks = n
        for k in _MERGED_FIELDS:
            setattr(m, k, mg[k].data_ptr())
        return m

    def apx_s(n):
        a = tpc_apex_t(); a.max_tracks = n
        a.apex_partner = ax["apex_partner"].data_ptr(); a.apex_leg = ax["apex_leg"].data_ptr()
        return a
    mc = tpc_merge_cuts_t(30, 1, 6.0, 50.0, 100.0, 2.0, 0.3)
    ac = tpc_apex_cuts_t(4, 0.6, 150.0, 0.1, 4.0, 0.1, 3.0)
    rc = tpc_removal_cuts_t(0.05, 0.85, 1.0, 1.0)
    cls = torch.zeros(cfg1.n, dtype=torch.uint8, device="cuda"); rem = torch.zeros_like(cls)
    small = mt - 1
    assert lib.tpc_tracker_refit(h, C.byref(fit_s(small)), st) == -2
    assert lib.tpc_tracker_refit(h, C.byref(fit_s(mt)), st) == 0
    assert lib.tpc_tracker_merge(h, C.byref(fit_s(small)), C.byref(mc), C.byref(mrg_s(mt)), st) == -2
    assert lib.tpc_tracker_merge(h, C.byref(fit_s(mt)), C.byref(mc), C.byref(mrg_s(small)), st) == -2
    assert lib.tpc_tracker_merge(h, C.byref(fit_s(mt)), C.byref(mc), C.byref(mrg_s(mt)), st) == 0
    assert lib.tpc_tracker_apex(h, C.byref(mrg_s(small)), C.byref(ac), C.byref(apx_s(mt)), st) == -2
    assert lib.tpc_tracker_apex(h, C.byref(mrg_s(mt)), C.byref(ac), C.byref(apx_s(small)), st) == -2
    assert lib.tpc_tracker_apex(h, C.byref(mrg_s(mt)), C.byref(ac), C.byref(apx_s(mt)), st) == 0
    ct = out.cluster_track.data_ptr()
    for f_n, m_n, a_n, want in ((small, mt, mt, -2), (mt, small, mt, -2), (mt, mt, small, -2), (mt, mt, mt + 1, -2), (mt, mt, mt, 0)):
        got = lib.tpc_tracker_removable(h, ct, C.byref(fit_s(f_n)), C.byref(mrg_s(m_n)), C.byref(apx_s(a_n)), C.byref(rc),
                                        cls.data_ptr(), rem.data_ptr(), st)
        assert got == want, (f_n, m_n, a_n, got)
    torch.cuda.synchronize()
    # a frame tracked with a smaller max_tracks lowers the bar accordingly
    out_small = tpc.Tracks(cfg1.n, 64, trk.caps[4], trk.device)
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (cfg1.sector, cfg1.row, cfg1.y, cfg1.z)]
    trk.track_timeframe(*ins, out_small)
    assert lib.tpc_tracker_refit(h, C.byref(fit_s(64)), st) == 0 and lib.tpc_tracker_refit(h, C.byref(fit_s(63)), st) == -2
    torch.cuda.synchronize()


def test_optional_calls_out_of_order_are_refused(cfg1):
    """refit -> merge -> apex -> removable read what their predecessors left in the workspace for the CURRENT frame: a call
    whose predecessor did not run after the last tpc_track_timeframe is INVALID_ARG, not a walk over stale counters."""
    import paper_2009_07515_b200 as tpc
    P = default_params(cfg1)
    c = tpc.suggest_capacities(cfg1.n, P)
    trk = tpc.Tracker(P, c["max_clusters"], tpc.max_bins_bound(cfg1.sector, cfg1.z, P), c["max_seeds"], c["max_tracks"], c["max_track_clusters"])
    fit = trk.new_fit(); mg = trk.new_merged(); ax = trk.new_apex()
    for call in (lambda: trk.refit_into(fit), lambda: trk.merge_into(fit, mg), lambda: trk.apex_into(mg, ax)):
        with pytest.raises(RuntimeError, match="invalid argument"):
            call()                                           # nothing tracked yet
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (cfg1.sector, cfg1.row, cfg1.y, cfg1.z)]
    out = trk.new_tracks(cfg1.n)
    trk.track_timeframe(*ins, out)
    with pytest.raises(RuntimeError, match="invalid argument"):
        trk.merge_into(fit, mg)                              # no refit of this frame
    trk.refit_into(fit)
    with pytest.raises(RuntimeError, match="invalid argument"):
        trk.apex_into(mg, ax)                                # no merge of this frame
    trk.merge_into(fit, mg); trk.apex_into(mg, ax)
    cls, rem = trk.removable(out)                            # refit + merge + apex + removable: fine
    trk.track_timeframe(*ins, out)                           # a new frame: everything above is stale
    with pytest.raises(RuntimeError, match="invalid argument"):
        trk.apex_into(mg, ax)
    with pytest.raises(RuntimeError, match="invalid argument"):
        trk.merge_into(fit, mg)
    trk.refit_into(fit); trk.merge_into(fit, mg); trk.apex_into(mg, ax)
    torch.cuda.synchronize()
    assert int(mg["n_merged"].item()) >= 1


# ------------------------------------------------------------------------------------------------ apex links (3.9.8)
APEX = dict(max_k=4, min_s=0.6, dz_win=150.0, tol_c=0.1, tol_z=4.0, tol_t=0.1, cut=3.0)


def _apex_parity(tf, cuts=None, min_pairs=1):
    kw = dict(APEX); kw.update(cuts or {})
    P, trk, out = run_gpu(tf)
    T = out.numpy()["n_tracks"]
    m = trk.merge(T, apex=kw)
    o = run_oracle(tf, P, last_stage=6).merge(**CUTS).apex(**kw)
    M = m["n_merged"]
    assert M == o.get("mrg_seg_start").size - 1 and np.array_equal(m["seg_idx"], o.get("mrg_seg_idx"))
    assert np.array_equal(trk.stage_view("apex_best")[:M], o.get("apx_best"))
    assert np.array_equal(trk.stage_view("apex_score")[:M], o.get("apx_score").astype(np.float32))
    assert np.array_equal(m["apex_partner"], o.get("apx_partner")) and np.array_equal(m["apex_leg"], o.get("apx_leg"))
    pairs = int((o.get("apx_partner") >= 0).sum()) // 2
    assert pairs >= min_pairs, pairs
    return m, o, pairs


def test_apex_links_bit_exact_on_looper_frames():
    tf = generate_config("cfg3", n_collisions=3, loopers=True)
    m, o, pairs = _apex_parity(tf, min_pairs=2000)
    # the pairs are what the generator says: the two legs of one truth track
    _apex_parity(generate_config("cfg2", n_tracks=1500, seed=8, loopers=True), min_pairs=500)
    _apex_parity(tf, cuts=dict(max_k=2, min_s=0.8, dz_win=40.0, tol_c=0.03, tol_z=1.0, tol_t=0.03, cut=1.0), min_pairs=20)
    _apex_parity(tf, cuts=dict(max_k=17, min_s=0.0, dz_win=400.0, tol_c=0.5, tol_z=20.0, tol_t=0.5, cut=10.0), min_pairs=2000)


def test_apex_links_without_loopers_and_bad_arguments(mini_event):
    m, o, pairs = _apex_parity(mini_event, min_pairs=0)
    P, trk, out = run_gpu(mini_event)
    fit = trk.new_fit(); mg = trk.new_merged(); ax = trk.new_apex()
    trk.refit_into(fit); trk.merge_into(fit, mg)
    for bad in (dict(dz_win=0.0), dict(tol_c=0.0), dict(tol_z=-1.0), dict(max_k=-1), dict(cut=float("nan"))):
        with pytest.raises(RuntimeError):
            trk.apex_into(mg, ax, bad)
    trk.apex_into(mg, ax)
    torch.cuda.synchronize()


def test_merge_and_apex_on_an_empty_frame_and_after_a_status_bit(cfg1):
    """No tracks: n_merged = 0 and nothing is written; a frame that ended with a status bit (capacity overflow) merges
    to nothing as well."""
    import copy
    import paper_2009_07515_b200 as tpc
    empty = copy.copy(cfg1)
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        setattr(empty, f, getattr(cfg1, f)[:0].copy())
    P = default_params(cfg1)
    trk = tpc.Tracker(P, 1024, 4096, 64, 64, 1024)
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (empty.sector, empty.row, empty.y, empty.z)]
    out = trk.new_tracks(0)
    trk.track_timeframe(*ins, out)
    m = trk.merge(0, apex=True)
    assert out.numpy()["n_tracks"] == 0 and m["n_merged"] == 0 and m["seg_start"].tolist() == [0] and m["apex_partner"].size == 0
    # seeds overflow -> status bit -> zero tracks -> zero merged tracks
    _, trk2, out2 = run_gpu(cfg1, caps=dict(max_seeds=4))
    assert out2.numpy()["status"] & 4 and out2.numpy()["n_tracks"] == 0
    m2 = trk2.merge(0, apex=True)
    assert m2["n_merged"] == 0


POISON = 0x7F7F7F7F
WILD = dict(max_rows=150, back_rows=150, edge=1000.0, dz_win=200.0, chi2_cut=1e30, road_z0=1e3, road_z1=1e3)


def test_link_cycles_get_minus_one_and_never_the_callers_garbage():
    """With cuts this loose (any row distance, any chi2) mutual links close into cycles: no chain head reaches those
    tracks, the oracle leaves them at -1 and so must the kernel, whatever the caller's buffer held;
    the hit removal then classifies them from their own segment (no index taken from a -1)."""
    tf = generate_config("cfg3", n_collisions=3, loopers=True)
    P, trk, out = run_gpu(tf)
    T = out.numpy()["n_tracks"]
    m = trk.merge(T, WILD, fill=POISON)
    o = run_oracle(tf, P, last_stage=6).merge(**WILD)
    want = o.get("mrg_of_track")
    assert int((want < 0).sum()) >= 50                     # the case is really there
    assert np.array_equal(m["merged_of_track"], want)
    assert m["n_merged"] == o.get("mrg_seg_start").size - 1
    assert np.array_equal(m["seg_start"], o.get("mrg_seg_start"))
    assert np.array_equal(m["seg_idx"][: int(m["seg_start"][-1])], o.get("mrg_seg_idx"))
    assert np.array_equal(m["par"], o.get("mrg_par").astype(np.float32).reshape(-1, 5))
    cuts = dict(min_pt=0.05, max_incl=0.85, road_y=1.0, road_z=1.0)
    cls, rem = trk.removable(out, cuts, merge_cuts=WILD, fill=POISON)
    oo = o.apex(**APEX).removable(**cuts)
    assert np.array_equal(cls.cpu().numpy().astype(np.int32), oo.get("rem_class"))
    assert np.array_equal(rem.cpu().numpy().astype(np.int32), oo.get("rem_remove"))


def test_merge_and_removal_after_a_status_bit_write_defined_values_into_poisoned_buffers(cfg1):
    """A frame aborted by a status bit has no tracks: the merger reports none and the hit removal marks every cluster as
    not attached and not removable, also when the caller's buffers were full of garbage."""
    _, trk, out = run_gpu(cfg1, caps=dict(max_seeds=4))
    assert out.numpy()["status"] & 4 and out.numpy()["n_tracks"] == 0
    m = trk.merge(0, apex=True, fill=POISON)
    assert m["n_merged"] == 0 and m["seg_start"].tolist() == [0]
    cls, rem = trk.removable(out, fill=POISON)
    assert int(cls.max().item()) == 0 and int(rem.max().item()) == 0


@pytest.mark.parametrize("S", [1, 2, 5])
def test_merge_in_odd_geometries(S, cfg1):
    """One sector (no neighbour), two sectors, an odd count: same results as the oracle, no neighbour arithmetic blows up."""
    import copy
    tf = copy.copy(cfg1)
    keep = (cfg1.sector == np.bincount(cfg1.sector).argmax()) & ~np.isin(cfg1.row, np.arange(60, 66))
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        setattr(tf, f, getattr(cfg1, f)[keep].copy())
    tf.sector = np.zeros_like(tf.sector)
    P = default_params(cfg1); P["n_sectors"] = S
    m, o, links = _merge_parity(tf, P=P, min_links=10)
    kw = dict(APEX)
    Pg, trk, out = run_gpu(tf, params=P)
    mm = trk.merge(out.numpy()["n_tracks"], apex=kw)
    oo = run_oracle(tf, P, last_stage=6).merge(**CUTS).apex(**kw)
    assert np.array_equal(mm["apex_partner"], oo.get("apx_partner"))


# ------------------------------------------------------------------------------------------------ strategy-A removal (3.8a)
@pytest.mark.parametrize("cuts", [dict(min_pt=0.05, max_incl=0.85, road_y=1.0, road_z=1.0),
                                  dict(min_pt=0.14, max_incl=0.6, road_y=3.0, road_z=0.5),
                                  dict(min_pt=0.0, max_incl=0.0, road_y=0.0, road_z=0.0)])
def test_strategy_a_removal_bit_exact(cuts):
    tf = generate_config("cfg3", n_collisions=3, loopers=True)
    P, trk, out = run_gpu(tf)
    cls, rem = trk.removable(out, cuts)
    o = run_oracle(tf, P, last_stage=6).merge(**CUTS).apex(**APEX).removable(**cuts)
    assert np.array_equal(cls.cpu().numpy().astype(np.int32), o.get("rem_class"))
    assert np.array_equal(rem.cpu().numpy().astype(np.int32), o.get("rem_remove"))
    assert (o.get("rem_class") == 2).sum() > 50000


def test_strategy_a_removal_rejects_bad_arguments_and_handles_empty_frames(cfg1):
    import paper_2009_07515_b200 as tpc
    P, trk, out = run_gpu(cfg1)
    for bad in (dict(min_pt=-1.0), dict(road_y=float("nan")), dict(max_incl=-0.1)):
        with pytest.raises(RuntimeError):
            trk.removable(out, bad)
    cls, rem = trk.removable(out)
    assert int(rem.sum().item()) == 0 and int((cls == 1).sum().item()) == int((out.cluster_track[: cfg1.n] >= 0).sum().item())
    trk2 = tpc.Tracker(default_params(cfg1), 1024, 4096, 64, 64, 1024)
    e = [torch.empty(0, dtype=dt, device="cuda") for dt in (torch.uint8, torch.uint8, torch.float32, torch.float32)]
    o2 = trk2.new_tracks(0)
    trk2.track_timeframe(*e, o2)
    cls, rem = trk2.removable(o2)
    assert cls.numel() == 0 and rem.numel() == 0
