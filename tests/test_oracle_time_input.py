"""Pins for the native time input of the oracle (clusters arrive in native pad,
row and TIME coordinates and cannot be converted ahead of time), CPU only.

* hand-written dyadic cases: every fp32 operation of `zc = drift_length - t * cm_per_time_unit` is exact on them, so the
  expected pseudo-z (with its A / C side sign) is typed into the test;
* the conversion is the ONLY thing the flag changes: the run on times equals the run on the pseudo-z obtained from the
  same times by numpy's separately rounded fp32 product and difference, array by array;
* round trip against the generator's own times (computed in double from the frame's pseudo-z): the tracker's z lands
  on the frame's z within the fp32 rounding of the time, on both sides of the TPC;
* vertex time: on the time path `-+ z_beam / v_drift` lands on the generated collision times.
"""
import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config, to_native_time


def _params(tf, **kw):
    P = default_params(tf)
    P.update(kw)
    return P


def test_hand_written_times_on_both_sides(cfg1):
    """L = 250 cm, 0.5 cm per time unit.  A side (sector 3): t = 0 -> +250, t = 100 -> +200, t = 500 -> +0, t = 601 ->
    -50.5 (a cluster read out after the full drift time of the frame start belongs to a later collision: negative pseudo-z).
    C side (sector 21): the same times with the opposite sign.  Kills: sign of the C side, A/C boundary at n_sectors / 2,
    `t * c - L` for `L - t * c`, a forgotten drift length, division for multiplication."""
    P = _params(cfg1, z_is_time=1, cm_per_time_unit=np.float32(0.5), drift_length=np.float32(250.0))
    t = np.array([0.0, 100.0, 500.0, 601.0], np.float32)
    want = np.array([250.0, 200.0, 0.0, -50.5], np.float32)
    for sector, sign in ((3, 1.0), (17, 1.0), (18, -1.0), (21, -1.0)):
        sec = np.full(4, sector, np.uint8)
        row = np.array([5, 5, 5, 5], np.uint8)
        y = np.array([-3.0, -1.0, 1.0, 3.0], np.float32)      # one bin each along y at most: order by z decides
        o = Oracle(P).run(sec, row, y, t, last_stage=1)
        zs = o.get("zs"); perm = o.get("perm")
        got = np.empty(4, np.float32); got[perm] = zs
        assert np.array_equal(got, (sign * want).astype(np.float32)), (sector, got)
        assert not np.signbit(got[2])                          # 0 - (+0) = +0: no negative zero enters the z range
        assert o.get("zmin")[sector] == got.min() and o.get("zmax")[sector] == got.max()


def test_flag_changes_nothing_but_the_conversion(mini_tf):
    tft, tp = to_native_time(mini_tf)
    P = _params(mini_tf, **tp)
    c, L = np.float32(tp["cm_per_time_unit"]), np.float32(tp["drift_length"])
    prod = (tft.z * c).astype(np.float32)                     # numpy rounds the product ...
    zc = (L - prod).astype(np.float32)                        # ... and the difference separately
    z = np.where(tft.sector < 18, zc, np.float32(0.0) - zc).astype(np.float32)
    a = Oracle(P).run(tft.sector, tft.row, tft.y, tft.z, last_stage=6)
    b = Oracle(_params(mini_tf)).run(tft.sector, tft.row, tft.y, z, last_stage=6)
    for nm in ("perm", "zs", "ys", "bin_start", "zmin", "zmax", "nz", "link_up", "link_dn", "seed_head", "t_hit", "t_par",
               "cluster_track", "trk_cl_idx", "trk_par", "trk_cov", "trk_z_ref", "trk_z_beam", "fit_par", "fit_res_z"):
        assert np.array_equal(a.get(nm), b.get(nm)), nm
    assert a.get("trk_seed").size > 100


def test_round_trip_against_the_generated_times():
    tf = generate_config("cfg5", n_collisions=4, seed=77)        # a slice of the 11.4 ms frame: |z'| up to 28 500 cm
    tft, tp = to_native_time(tf)
    assert tft.z.min() >= 0.0 and tft.z.max() > 50_000           # times count from the frame start, 57 000 units long
    o = Oracle(_params(tf, **tp)).run(tft.sector, tft.row, tft.y, tft.z, last_stage=1)
    z_in = np.empty(tf.n, np.float32); z_in[o.get("perm")] = o.get("zs")
    # the time is an fp32 of magnitude <= 2^16: half an ulp is 2^-8 time units = 0.002 cm; product and difference add
    # two more roundings of numbers below 2^15 cm
    err = np.abs(z_in.astype(np.float64) - tf.z.astype(np.float64))
    assert err.max() < 0.005, err.max()
    a_side = tf.sector < 18
    assert np.all(np.sign(z_in[a_side & (np.abs(tf.z) > 1)]) == np.sign(tf.z[a_side & (np.abs(tf.z) > 1)]))
    assert np.all(np.sign(z_in[~a_side & (np.abs(tf.z) > 1)]) == np.sign(tf.z[~a_side & (np.abs(tf.z) > 1)]))
    assert (z_in[~a_side] > 1).any() and (z_in[a_side] < -1).any()   # both signs occur on both sides (later collisions)


def test_vertex_time_from_the_time_path():
    tf = generate_config("cfg3", n_collisions=3, seed=21)
    tft, tp = to_native_time(tf)
    o = Oracle(_params(tf, **tp)).run(tft.sector, tft.row, tft.y, tft.z)
    ct = o.get("cluster_track"); zb = o.get("trk_z_beam"); sector = o.get("trk_sector")
    g = tf.geometry
    t_est, t_true = [], []
    for k in range(zb.size):
        ids = tf.track_id[ct == k]
        if ids.size < 40 or ids.min() < 0 or ids.min() != ids.max():
            continue
        tid = int(ids[0])
        t_est.append(-zb[k] / g.v_drift if sector[k] < g.n_azimuthal else zb[k] / g.v_drift)
        t_true.append(tf.truth["t_coll"][tid])
    t_est = np.array(t_est); t_true = np.array(t_true)
    assert t_est.size > 500
    dt = t_est - t_true                                        # off only by z_v / v_drift (sigma 2 us)
    assert abs(dt.mean()) < 0.3 and 1.2 < dt.std() < 3.0, (dt.mean(), dt.std())
    assert np.corrcoef(t_est, t_true)[0, 1] > 0.99
