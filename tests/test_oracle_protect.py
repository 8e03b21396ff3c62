"""Pins for the oracle's cluster protection, "strategy B", CPU only.

* brute force: all pairs inside every (sector, row), same closed-rectangle predicate written in numpy fp32;
* properties: attached clusters are always kept, the kept set grows with the road, a zero road keeps exactly the attached
  clusters (and their exact duplicates);
* generator truth: the noise goes, the signal of the found tracks stays.
"""
import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config

f32 = np.float32


def _run(name, **over):
    tf = generate_config(name, **over)
    P = default_params(tf)
    return tf, P, Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)


def _brute(tf, o, road_y, road_z):
    ct = o.get("cluster_track")
    keep = (ct >= 0).astype(np.int32)
    key = tf.sector.astype(np.int64) * 256 + tf.row
    y, z = tf.y.astype(f32), tf.z.astype(f32)
    ry, rz = f32(road_y), f32(road_z)
    for k in np.unique(key):
        idx = np.nonzero(key == k)[0]
        own = idx[ct[idx] >= 0]
        if own.size == 0:
            continue
        ylo, yhi = (y[own] - ry)[None, :], (y[own] + ry)[None, :]          # fp32 bounds, closed rectangle (section 3.1)
        zlo, zhi = (z[own] - rz)[None, :], (z[own] + rz)[None, :]
        yi, zi = y[idx][:, None], z[idx][:, None]
        inside = (yi >= ylo) & (yi <= yhi) & (zi >= zlo) & (zi <= zhi)
        keep[idx[inside.any(axis=1)]] = 1
    return keep


def test_protection_equals_brute_force():
    for name, over, road in (("cfg2", dict(n_tracks=500, noise=0.3), (2.0, 3.0)), ("cfg3", dict(n_collisions=2), (0.7, 0.4)),
                             ("cfg1", {}, (5.0, 5.0))):
        tf, P, o = _run(name, **over)
        got = o.protect(*road)
        assert np.array_equal(got, _brute(tf, o, *road)), name
        assert 0 < got.sum()


def test_protection_properties():
    tf, P, o = _run("cfg3", n_collisions=2, noise=0.2)
    ct = o.get("cluster_track")
    k0 = o.protect(0.0, 0.0).copy()
    k1 = o.protect(1.0, 1.0).copy()
    k3 = o.protect(3.0, 3.0).copy()
    assert np.all(k1[ct >= 0] == 1) and np.all(k0[ct >= 0] == 1)
    assert np.all(k1 >= k0) and np.all(k3 >= k1) and k3.sum() > k1.sum() > k0.sum() - 1
    assert k0.sum() == (ct >= 0).sum()                      # nothing but the attached clusters (no exact duplicates here)
    sig = tf.track_id >= 0
    assert k1[~sig].mean() < 0.10                           # the noise goes ...
    seg = tf.track_id.astype(np.int64) * 64 + tf.sector      # a track inside one sector
    segs, cnt = np.unique(seg[(ct >= 0) & sig], return_counts=True)
    found = np.isin(seg, segs[cnt >= 20]) & sig
    assert found.sum() > 50000 and k1[found].mean() > 0.97  # ... the clusters of the found track segments stay
