"""Pins for the S4 phase logic of the oracle against generator truth (CPU only).

An isolated noise-free helix has exactly one right answer that does not depend on the oracle: every
cluster of the track belongs to it.  Removing rows from such a track exercises, one at a time,
  * phase B (upward extrapolation + pick-up across a hole the links cannot bridge),
  * the gap rule (a hole of max_gap rows is crossed, a hole of max_gap + 1 rows is not),
  * phase C (downward refit + pick-up below the seed head of clusters too few to seed a chain),
  * first_row / last_row / n_hits / ndf bookkeeping.
A wrong comparison in the gap counter, a phase that forgets to search, or a turn-round that restarts
from the wrong state fails one of these.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config, select_sectors


def _isolated_tracks(n_want=6, min_rows=90):
    """single noise-free helices whose clusters in their main sector form one contiguous row range"""
    out = []
    for seed in range(100, 160):
        tf = generate_config("cfg1", n_tracks=1, seed=seed, sigma=0.0)
        if tf.n == 0:
            continue
        s = np.bincount(tf.sector).argmax()
        sub, _ = select_sectors(tf, [s])
        rows = np.sort(sub.row.astype(int))
        if rows.size >= min_rows and np.array_equal(rows, np.arange(rows[0], rows[0] + rows.size)):
            out.append(sub)
        if len(out) == n_want:
            break
    assert len(out) == n_want
    return out


def _drop_rows(tf, rows_to_drop):
    keep = ~np.isin(tf.row.astype(int), list(rows_to_drop))
    idx = np.nonzero(keep)[0]
    sub, _ = select_sectors(tf, np.unique(tf.sector))
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        setattr(sub, f, getattr(tf, f)[idx].copy())
    return sub


def _run(tf, P):
    return Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32)


TRACKS = None


@pytest.fixture(scope="module")
def tracks():
    return _isolated_tracks()


@pytest.fixture(scope="module")
def params(tracks):
    return default_params(tracks[0], cell=4.0)


def test_intact_track_is_one_track_with_every_cluster(tracks, params):
    for tf in tracks:
        o = _run(tf, params)
        ct = o.get("cluster_track")
        assert o.get("trk_seed").size == 1 and np.all(ct == 0)
        r0, r1 = int(tf.row.min()), int(tf.row.max())
        assert o.get("trk_first_row")[0] == r0 and o.get("trk_last_row")[0] == r1
        assert o.get("trk_n_clusters")[0] == tf.n and o.get("trk_ndf")[0] == 2 * tf.n - 5
        assert o.get("trk_x_ref")[0] == np.float32(params["row_x"][r0])       # output state sits at the lowest hit row
        assert o.get("trk_chi2")[0] < 1e-2 * tf.n                             # noise-free: only fp32 rounding


@pytest.mark.parametrize("hole", [3, 4])
def test_phase_b_bridges_a_hole_of_up_to_max_gap_rows(tracks, params, hole):
    """links reach r+-2 at most, so a hole of >= 2 rows cuts the chain; phase B must pick the upper part up."""
    assert params["max_gap"] == 4
    for tf in tracks:
        r0 = int(tf.row.min())
        cut = r0 + 30
        sub = _drop_rows(tf, range(cut, cut + hole))
        o = _run(sub, params)
        assert np.all(o.get("link_up")[np.nonzero(o.get("s_row") == cut - 1)[0]] == -1)   # the chain really is cut
        ct = o.get("cluster_track")
        assert o.get("trk_seed").size == 1 and np.all(ct == 0), (hole, np.unique(ct))
        assert o.get("trk_n_clusters")[0] == sub.n
        assert o.get("trk_first_row")[0] == r0 and o.get("trk_last_row")[0] == int(tf.row.max())


def test_hole_of_max_gap_plus_one_rows_is_not_crossed(tracks, params):
    for tf in tracks:
        r0, r1 = int(tf.row.min()), int(tf.row.max())
        cut = r0 + 30
        hole = params["max_gap"] + 1
        sub = _drop_rows(tf, range(cut, cut + hole))
        o = _run(sub, params)
        ct = o.get("cluster_track")
        assert o.get("trk_seed").size == 2
        lower = sub.row.astype(int) < cut
        assert np.all(ct[lower] == 0) and np.all(ct[~lower] == 1)           # track ids in seed (= row) order
        assert list(o.get("trk_first_row")) == [r0, cut + hole] and list(o.get("trk_last_row")) == [cut - 1, r1]
        assert list(o.get("trk_n_clusters")) == [30, r1 - (cut + hole) + 1]


def test_phase_c_picks_up_below_the_seed_head(tracks, params):
    """three clusters below a 3-row hole cannot seed (min_chain_len = 4): only the downward pass can attach them"""
    assert params["min_chain_len"] == 4
    for tf in tracks:
        r0 = int(tf.row.min())
        sub = _drop_rows(tf, range(r0 + 3, r0 + 6))
        o = _run(sub, params)
        assert o.get("seed_head").size == 1
        head_row = int(o.get("s_row")[o.get("seed_head")[0]])
        assert head_row == r0 + 7            # row r0+6 has no downward candidate -> no link pair (section 3.2): phase C attaches it too
        ct = o.get("cluster_track")
        assert o.get("trk_seed").size == 1 and np.all(ct == 0)
        assert o.get("trk_first_row")[0] == r0 and o.get("trk_n_clusters")[0] == sub.n


def test_short_leftover_below_a_wide_hole_stays_unassigned(tracks, params):
    """3 clusters below a (max_gap+1)-row hole: unreachable for phase C and too few to seed -> no track, -1"""
    for tf in tracks:
        r0 = int(tf.row.min())
        hole = params["max_gap"] + 1
        sub = _drop_rows(tf, range(r0 + 3, r0 + 3 + hole))
        o = _run(sub, params)
        ct = o.get("cluster_track")
        low = sub.row.astype(int) < r0 + 3
        assert o.get("trk_seed").size == 1
        assert np.all(ct[low] == -1) and np.all(ct[~low] == 0)
        assert o.get("trk_first_row")[0] == r0 + 3 + hole


def test_tracklet_below_min_hits_is_dropped(tracks, params):
    tf = tracks[0]
    r0 = int(tf.row.min())
    n_keep = params["min_tracklet_hits"] - 1
    sub = _drop_rows(tf, range(r0 + n_keep, 256))
    o = _run(sub, params)
    assert o.get("seed_head").size == 1 and o.get("t_n_hits")[0] == n_keep and o.get("t_kept")[0] == 0
    assert o.get("trk_seed").size == 0 and np.all(o.get("cluster_track") == -1)
    sub = _drop_rows(tf, range(r0 + n_keep + 1, 256))
    o = _run(sub, params)
    assert o.get("trk_seed").size == 1 and np.all(o.get("cluster_track") == 0)
