"""Pins for the strategy-A hit removal of the oracle, CPU only.

* definition, brute force: the class of every cluster recomputed in numpy from the track-level results (apex label, merged
  q/pT, sin(phi) at both ends of the segment), the protection by GOOD tracks only as an all-pairs rectangle test per
  (sector, row) in numpy fp32, removable = class >= 2 and not protected;
* properties: nothing attached to a good track is ever removable; a huge road removes nothing that shares a row with a good
  track; a zero road removes exactly the clusters of classes >= 2;
* generator truth with returning branches: most clusters of returning legs go, almost none of the outgoing ones; with
  min_pt raised into the generated spectrum the low-momentum class follows the true pT.
"""
import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config

f32 = np.float32


def _run(tf, **cuts):
    P = default_params(tf)
    return Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=6).merge().apex().removable(**cuts)


def _brute(tf, o, min_pt, max_incl, road_y, road_z):
    ct = o.get("cluster_track"); nt = o.get("trk_seed").size
    mo = o.get("mrg_of_track"); leg = o.get("apx_leg")
    mq = o.get("mrg_par").reshape(-1, 5)[:, 4].astype(f32)
    s_in = np.abs(o.get("fit_par").reshape(-1, 5)[:, 2].astype(f32)); s_out = np.abs(o.get("up_par").reshape(-1, 5)[:, 2].astype(f32))
    cls_t = np.ones(nt, np.int32)
    for k in range(nt):
        m = mo[k]
        if m >= 0 and leg[m] == 1:
            cls_t[k] = 2
        elif m >= 0 and f32(np.abs(mq[m]) * f32(min_pt)) > f32(1):
            cls_t[k] = 3
        elif s_in[k] > f32(max_incl) and s_out[k] > f32(max_incl):
            cls_t[k] = 4
    cls = np.where(ct >= 0, cls_t[np.maximum(ct, 0)], 0)
    good = (ct >= 0) & (cls == 1)
    keep = np.zeros(tf.n, bool)
    key = tf.sector.astype(np.int64) * 256 + tf.row
    y, z = tf.y.astype(f32), tf.z.astype(f32)
    ry, rz = f32(road_y), f32(road_z)
    for k in np.unique(key[good]):
        idx = np.nonzero(key == k)[0]
        own = idx[good[idx]]
        inside = (y[idx][:, None] >= (y[own] - ry)[None, :]) & (y[idx][:, None] <= (y[own] + ry)[None, :]) & \
                 (z[idx][:, None] >= (z[own] - rz)[None, :]) & (z[idx][:, None] <= (z[own] + rz)[None, :])
        keep[idx[inside.any(axis=1)]] = True
    return cls, np.where(good, ct, -1), ((cls >= 2) & ~keep).astype(np.int32)


def test_classes_and_removal_equal_the_definition():
    tf = generate_config("cfg3", n_collisions=1, seed=9, loopers=True, noise=0.2)
    for cuts in (dict(min_pt=0.05, max_incl=0.85, road_y=1.0, road_z=1.0), dict(min_pt=0.14, max_incl=0.6, road_y=3.0, road_z=0.5)):
        o = _run(tf, **cuts)
        cls, good, rem = _brute(tf, o, **cuts)
        assert np.array_equal(o.get("rem_class"), cls) and np.array_equal(o.get("rem_good_track"), good)
        assert np.array_equal(o.get("rem_remove"), rem)
        assert set(np.unique(cls)) >= {0, 1, 2} and rem.sum() > 1000


def test_properties():
    tf = generate_config("cfg3", n_collisions=1, seed=9, loopers=True)
    o = _run(tf, road_y=0.0, road_z=0.0)
    cls = o.get("rem_class")
    assert np.array_equal(o.get("rem_remove"), (cls >= 2).astype(np.int32))       # zero road: exactly the classes >= 2
    r1 = _run(tf, road_y=1.0, road_z=1.0).get("rem_remove")
    r9 = _run(tf, road_y=1e6, road_z=1e6).get("rem_remove")
    assert np.all(r1 <= (cls >= 2)) and np.all(r9 <= r1) and r9.sum() < r1.sum()
    assert not np.any(r1[cls == 1]) and not np.any(r1[cls == 0])                   # good and unattached clusters are never removed
    # a huge road: nothing in a (sector, row) that holds a cluster of a good track goes
    key = tf.sector.astype(np.int64) * 256 + tf.row
    assert not np.any(r9[np.isin(key, np.unique(key[cls == 1]))])


def test_against_generator_truth():
    tf = generate_config("cfg3", n_collisions=2, loopers=True)
    o = _run(tf)
    cls, rem = o.get("rem_class"), o.get("rem_remove")
    ret = tf.leg == 1
    out = (tf.leg == 0) & (tf.track_id >= 0)
    assert (cls[ret] == 2).mean() > 0.65 and rem[ret].mean() > 0.65                # most of the returning legs go
    assert (cls[out] == 2).mean() < 0.005 and rem[out].mean() < 0.02               # almost none of the outgoing ones
    # low momentum: no generated track is below 50 MeV/c; with the cut raised to 150 MeV/c the class follows the true pT
    o.removable(min_pt=0.15)
    cls = o.get("rem_class")
    pt = np.abs(1.0 / tf.truth["q_over_pt"])[np.maximum(tf.track_id, 0)]
    att = out & (cls > 0) & (cls != 2)
    assert (cls[att & (pt < 0.14)] == 3).mean() > 0.98 and (cls[att & (pt > 0.17)] == 3).mean() < 0.01
