"""Pins for the native pad input of the oracle (clusters arrive in native PAD,
row and time coordinates and cannot be converted ahead of time), CPU only.

* hand-written dyadic cases: every fp32 operation of `y = (p - (n_pads_r - 1) / 2) * pitch_r` is exact on them, so the
  expected y is typed into the test (odd and even pad counts, two pitches, fractional centroids);
* the conversion is the ONLY thing the flag changes: the run on pad coordinates equals the run on the y obtained from the
  same pads by numpy's separately rounded fp32 difference and product, array by array, through every stage;
* round trip against the generator's own pad coordinates (computed in double from the frame's y): the tracker's y lands
  on the frame's y within the fp32 rounding of the pad coordinate, and the mirror symmetry of the pad plane holds
  (pad p and pad n_pads - 1 - p give y and -y);
* together with the time input (section 3.0a): a frame given in (pad, row, time) gives the tracks of the same frame in cm.
"""
import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config, to_native_pad, to_native_time


def _params(tf, **kw):
    P = default_params(tf)
    P.update(kw)
    return P


def _y_in_input_order(o, n):
    y = np.empty(n, np.float32)
    y[o.get("perm")] = o.get("ys")
    return y


def test_hand_written_pads(cfg1):
    """Row 5: 9 pads of 0.5 cm, centre pad = 4: p = 0 -> -2, 4 -> 0, 8 -> +2, 6.25 -> +1.125.  Row 70: 10 pads of 0.25 cm,
    the axis lies between pads 4 and 5: p = 4.5 -> 0, 0 -> -1.125, 9 -> +1.125, 5.5 -> +0.25.  Kills: n_pads / 2 for
    (n_pads - 1) / 2, a swapped sign, division by the pitch, the table of another row, the product before the difference."""
    R = cfg1.geometry.n_rows
    n_pads = np.full(R, 64, np.int32); pitch = np.full(R, 1.0, np.float32)
    n_pads[5], pitch[5] = 9, 0.5
    n_pads[70], pitch[70] = 10, 0.25
    P = _params(cfg1, y_is_pad=1, n_pads=n_pads, pad_pitch=pitch)
    row = np.array([5, 5, 5, 5, 70, 70, 70, 70], np.uint8)
    pad = np.array([0.0, 4.0, 8.0, 6.25, 4.5, 0.0, 9.0, 5.5], np.float32)
    want = np.array([-2.0, 0.0, 2.0, 1.125, 0.0, -1.125, 1.125, 0.25], np.float32)
    for sector in (0, 17, 18, 35):                               # the pad plane is the same on both sides
        sec = np.full(8, sector, np.uint8)
        z = np.linspace(10.0, 80.0, 8).astype(np.float32)
        o = Oracle(P).run(sec, row, pad, z, last_stage=1)
        assert np.array_equal(_y_in_input_order(o, 8), want), sector


def test_flag_changes_nothing_but_the_conversion(mini_tf):
    tfp, pp = to_native_pad(mini_tf)
    P = _params(mini_tf, **pp)
    centre = (np.float32(0.5) * (pp["n_pads"] - 1).astype(np.float32)).astype(np.float32)
    d = (tfp.y - centre[tfp.row]).astype(np.float32)            # numpy rounds the difference ...
    y = (d * pp["pad_pitch"][tfp.row]).astype(np.float32)       # ... and the product separately
    a = Oracle(P).run(tfp.sector, tfp.row, tfp.y, tfp.z, last_stage=6)
    b = Oracle(_params(mini_tf)).run(tfp.sector, tfp.row, y, tfp.z, last_stage=6)
    for nm in ("perm", "zs", "ys", "bin_start", "zmin", "zmax", "nz", "link_up", "link_dn", "seed_head", "t_hit", "t_par",
               "cluster_track", "trk_cl_idx", "trk_par", "trk_cov", "trk_z_ref", "trk_z_beam", "fit_par", "fit_res_y"):
        assert np.array_equal(a.get(nm), b.get(nm)), nm
    assert a.get("trk_seed").size > 100


def test_round_trip_and_mirror_symmetry(mini_event):
    tf = mini_event
    tfp, pp = to_native_pad(tf)
    # inside the pad plane of the row, up to the smearing of a cluster on the sector edge (0.1 cm sigma, pads >= 0.4 cm)
    assert tfp.y.min() >= -1.5 and np.all(tfp.y <= pp["n_pads"][tf.row] + 0.5)
    assert pp["n_pads"].min() >= 60 and pp["n_pads"].max() <= 160 and np.all(pp["n_pads"] % 2 == 0)
    P = _params(tf, **pp)
    o = Oracle(P).run(tfp.sector, tfp.row, tfp.y, tfp.z, last_stage=1)
    y_in = _y_in_input_order(o, tf.n)
    # a pad coordinate below 2^8 carries half an ulp of 2^-17 pads = 5e-6 cm; difference and product add two roundings of
    # numbers below 64 cm (half an ulp 2e-6 cm each)
    err = np.abs(y_in.astype(np.float64) - tf.y.astype(np.float64))
    assert err.max() < 2e-5, err.max()
    # mirror: p -> n_pads - 1 - p is exact in fp32 for these magnitudes only up to rounding of the input; use dyadic pads
    rows = np.arange(tf.geometry.n_rows).astype(np.uint8)
    p = np.full(rows.size, 7.25, np.float32)
    q = (pp["n_pads"][rows] - 1 - p.astype(np.float64)).astype(np.float32)
    sec = np.zeros(rows.size, np.uint8); z = np.full(rows.size, 5.0, np.float32)
    ya = _y_in_input_order(Oracle(P).run(sec, rows, p, z, last_stage=1), rows.size)
    yb = _y_in_input_order(Oracle(P).run(sec, rows, q, z, last_stage=1), rows.size)
    assert np.array_equal(ya, -yb) and np.all(ya < 0)


def test_pad_row_time_frame_gives_the_tracks_of_the_frame_in_cm(mini_tf):
    """(pad, row, time) in, as the detector delivers them: same track count and (up to the few clusters whose rounding
    moved them across a cut) same assignment as the frame in cm."""
    tfp, pp = to_native_pad(mini_tf)
    tft, tp = to_native_time(tfp)
    a = Oracle(_params(mini_tf, **pp, **tp)).run(tft.sector, tft.row, tft.y, tft.z)
    b = Oracle(_params(mini_tf)).run(mini_tf.sector, mini_tf.row, mini_tf.y, mini_tf.z)
    ca, cb = a.get("cluster_track"), b.get("cluster_track")
    assert abs(a.get("trk_seed").size - b.get("trk_seed").size) <= 3
    assert ((ca >= 0) == (cb >= 0)).mean() > 0.999
