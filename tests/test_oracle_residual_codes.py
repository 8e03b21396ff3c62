"""Pins for the residual encoding of the oracle ("tailored custom fixed or floating
point data formats using only exactly as many bits as needed", "Hits attached to tracks are stored as
residuals to the extrapolated track position, which have a smaller entropy than absolute hit positions"), CPU only.

* hand-written dyadic residuals: product and rounding are exact on them, so the expected codes - ties to even on both
  signs, no negative zero surprise, saturation at +-32767 - are typed into the test;
* the frame's codes equal numpy's separately rounded fp32 product followed by numpy's own round-half-even;
* decoding (code * step) reproduces every unsaturated residual within half a step;
* the purpose: at the same resolution the codes of the residuals carry several bits less entropy than the codes of the
  absolute positions, and they fit a byte almost always.
"""
import numpy as np

from oracle import Oracle
from tpc_synth import default_params, generate_config


def test_hand_written_codes():
    """step = 0.25 cm.  0.125 -> 0.5 -> 0 and 0.375 -> 1.5 -> 2 (ties to even), 0.625 -> 2.5 -> 2, 0.3 -> 1.2 -> 1, the
    mirror images, the range ends.  Kills: round half away from zero, truncation, floor, division by the step's
    reciprocal, saturation at 32768 or at the int16 minimum, a missing saturation."""
    res = np.array([0.0, 0.125, 0.375, 0.625, 0.3, -0.125, -0.375, -0.625, -0.3, 0.25, -0.25, 8191.75, 8191.875, 1e6,
                    -8191.75, -8191.875, -1e6, np.inf, -np.inf], np.float32)
    want = np.array([0, 0, 2, 2, 1, 0, -2, -2, -1, 1, -1, 32767, 32767, 32767, -32767, -32767, -32767, 32767, -32767], np.int32)
    assert np.array_equal(Oracle.quantise_values(res, 0.25), want)
    # another step: 1/64 cm; 3/128 -> 1.5 -> 2, 5/128 -> 2.5 -> 2, 1/128 -> 0.5 -> 0
    res = np.array([3 / 128, 5 / 128, 1 / 128, -3 / 128, 1.0], np.float32)
    assert np.array_equal(Oracle.quantise_values(res, 1 / 64), np.array([2, 2, 0, -2, 64], np.int32))


def test_frame_codes_equal_numpy_and_decode_within_half_a_step(mini_tf):
    tf = mini_tf
    P = default_params(tf)
    sy, sz = 0.01, 0.02
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6).quantise_residuals(sy, sz)
    for nm, step in (("y", sy), ("z", sz)):
        res = o.get("fit_res_" + nm).astype(np.float32)
        q = o.get("fit_qres_" + nm)
        assert q.shape == res.shape and q.size > 100_000
        inv = np.float32(1.0) / np.float32(step)
        v = (res * inv).astype(np.float32)                     # numpy rounds the product to fp32 ...
        want = np.clip(np.rint(v), -32767, 32767).astype(np.int32)   # ... and rounds half to even itself
        assert np.array_equal(q, want), nm
        ok = np.abs(q) < 32767
        assert ok.mean() > 0.999
        err = np.abs(q[ok].astype(np.float64) * step - res[ok].astype(np.float64))
        assert err.max() <= 0.5 * step * (1 + 1e-5), (nm, err.max())
        assert (np.abs(q) <= 127).mean() > 0.99                # at 0.1 / 0.2 mm almost every residual fits a byte


def test_codes_of_residuals_carry_less_entropy_than_codes_of_positions(mini_tf):
    tf = mini_tf
    P = default_params(tf)
    step = 0.01
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6).quantise_residuals(step, step)
    idx = o.get("trk_cl_idx")

    def bits(codes):
        _, cnt = np.unique(codes, return_counts=True)
        p = cnt / cnt.sum()
        return float(-(p * np.log2(p)).sum())
    by, bz = bits(o.get("fit_qres_y")), bits(o.get("fit_qres_z"))
    py = bits(Oracle.quantise_values(tf.y[idx], step))
    pz = bits(np.round(tf.z[idx].astype(np.float64) / step).astype(np.int64))   # z spans more than 16 bits of steps
    assert by < py - 5 and bz < pz - 5, (by, py, bz, pz)
    assert by < 7 and bz < 7                                    # ~6 bits per coordinate at 0.1 mm
