"""Pins for the beam-line z estimate of the oracle, CPU only.

* closed form: for a circle through the origin the path length to (x, y) is R * theta with sin(theta/2) = d / (2R) -
  evaluated here with libm asin in double, which the oracle does not use;
* special cases: zero curvature (path = chord), a point on the beam line (z unchanged), charge symmetry;
* generator truth: primaries come from (0, 0, z_v) at time t_coll, so the estimate must land on the pseudo-z of their
  vertex, z_v -+ v_drift * t_coll (A / C side) - which is how continuous readout gets its vertex time.
"""
import math

import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config

KB = float(np.float32(-0.00299792458) * np.float32(0.5))


def _oracle():
    tf = generate_config("cfg1")
    return Oracle(default_params(tf))


def test_matches_closed_form_arc_length():
    o = _oracle()
    rng = np.random.default_rng(6)
    worst64 = worst32 = 0.0
    for _ in range(3000):
        R = rng.uniform(45.0, 5000.0)                       # pT 0.07 .. 7.5 GeV/c at 0.5 T
        theta = rng.uniform(0.01, 0.98 * math.pi)           # turning angle between the origin and the point
        sign = rng.choice([-1.0, 1.0])
        x = R * math.sin(theta)
        y = sign * R * (1.0 - math.cos(theta))
        q = sign * 1.0 / (abs(KB) * R)
        tanl, z = rng.uniform(-0.9, 0.9), rng.uniform(-250, 250)
        d = math.hypot(x, y)
        want = z - tanl * (2.0 * R * math.asin(min(1.0, d / (2.0 * R))))
        got64 = o.beam_z(x, y, z, tanl, q, precision=64)
        got32 = o.beam_z(x, y, z, tanl, q, precision=32)
        path = R * theta
        worst64 = max(worst64, abs(got64 - want) / path)
        worst32 = max(worst32, abs(got32 - want) / path)
    assert worst64 < 2e-6, worst64                          # truncation of the 5-term series at sin(theta/8) <= 0.38: 1.2e-6
    assert worst32 < 5e-6, worst32                          # a few fp32 roundings


def test_special_cases():
    o = _oracle()
    # no curvature: the path is the chord
    assert math.isclose(o.beam_z(120.0, -50.0, 10.0, 0.3, 0.0), 10.0 - 0.3 * 130.0, rel_tol=1e-12)
    # on the beam line nothing moves
    assert o.beam_z(0.0, 0.0, 42.0, 0.7, 3.0) == 42.0
    # the estimate does not depend on the sign of the charge or of y
    a = o.beam_z(150.0, 20.0, 5.0, 0.5, 2.0)
    assert a == o.beam_z(150.0, 20.0, 5.0, 0.5, -2.0) == o.beam_z(150.0, -20.0, 5.0, 0.5, 2.0)
    # a chord longer than the diameter is impossible for a primary: clamped to half a turn, finite
    R = 1.0 / (abs(KB) * 10.0)
    assert math.isclose(o.beam_z(3 * R, 0.0, 0.0, 1.0, 10.0), -(3 * R) * (math.pi / 2), rel_tol=1e-5)


def test_lands_on_the_vertex_pseudo_z_of_generated_primaries():
    tf = generate_config("cfg3", n_collisions=3, seed=21)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)
    ct = o.get("cluster_track")
    zb = o.get("trk_z_beam")
    sector = o.get("trk_sector")
    g = tf.geometry
    res, t_est, t_true = [], [], []
    for k in range(zb.size):
        ids = tf.track_id[ct == k]
        if ids.size < 40 or ids.min() < 0 or ids.min() != ids.max():
            continue                                        # long, pure tracks only
        tid = int(ids[0])
        a_side = sector[k] < g.n_azimuthal
        shift = -g.v_drift * tf.truth["t_coll"][tid] if a_side else g.v_drift * tf.truth["t_coll"][tid]
        res.append(zb[k] - (tf.truth["z_v"][tid] + shift))
        # vertex time under the paper's assumption (vertex at z = 0)
        t_est.append(-zb[k] / g.v_drift if a_side else zb[k] / g.v_drift)
        t_true.append(tf.truth["t_coll"][tid])
    res = np.array(res); t_est = np.array(t_est); t_true = np.array(t_true)
    assert res.size > 500
    assert abs(np.median(res)) < 0.05 and np.percentile(np.abs(res), 90) < 1.0, (np.median(res), np.percentile(np.abs(res), 90))
    # the time estimate is off only by z_v / v_drift (sigma 5 cm / 2.5 cm/us = 2 us)
    dt = t_est - t_true
    assert abs(dt.mean()) < 0.3 and 1.2 < dt.std() < 3.0, (dt.mean(), dt.std())
    assert np.corrcoef(t_est, t_true)[0, 1] > 0.99
