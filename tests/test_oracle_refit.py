"""Pins for the oracle's refit over owned clusters ("Track Fit"), CPU only.

* Bz = 0: the refit equals the closed-form weighted straight-line regression over exactly the clusters the track owns
  (numpy lstsq, evaluated at the lowest owned row), covariance = (A^T W A)^-1;
* noise-free helices: refitted q/pT within 1e-4 relative of generator truth (the bar BASELINE.json sets for the filter);
* smeared input: pulls of q/pT ~ N(0,1), chi2/ndf ~ 1 (ndf = 2 n_fit - 5);
* bookkeeping: every owned cluster is used, the state sits at the lowest owned row, z_ref is the top cluster's z.
"""
import math

import numpy as np

from oracle import Oracle
from tpc_synth import Geometry, default_params, generate, generate_config
from tpc_synth.generator import CONFIGS


def _truth_of_tracks(tf, o):
    ct = o.get("cluster_track")
    out = []
    for k in range(o.get("trk_seed").size):
        ids = tf.track_id[ct == k]
        v, c = np.unique(ids, return_counts=True)
        out.append((int(v[np.argmax(c)]), c.max() / ids.size, ids.size))
    return out


def test_refit_equals_weighted_line_fit_at_zero_field():
    rec = dict(CONFIGS["cfg1"]); rec.update(sigma=1e-3, n_tracks=30, seed=3)
    tf = generate(rec, geometry=Geometry(bz_tesla=0.0))
    P = default_params(tf)
    P["err_y2"] = np.float32(1e-6); P["err_z2"] = np.float32(1e-6)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=64, last_stage=6)
    nt = o.get("trk_seed").size
    assert nt >= 25
    st, pos = o.get("trk_cl_start"), o.get("trk_cl_pos")
    ys, zs, rows = o.get("ys").astype(np.float64), o.get("zs").astype(np.float64), o.get("s_row")
    rx = P["row_x"].astype(np.float64)
    par = o.get("fit_par").reshape(-1, 5); cov = o.get("fit_cov").reshape(-1, 15)
    checked = 0
    for k in range(nt):
        c = pos[st[k]:st[k + 1]]
        if c.size < 40:
            continue
        x, y, z = rx[rows[c]], ys[c], zs[c]
        assert o.get("fit_n")[k] == c.size
        A = np.stack([np.ones_like(x), x - x[0]], 1)             # evaluated at the lowest owned row
        coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        assert abs(par[k, 0] - coef[0]) < 2e-5
        tanphi = par[k, 2] / math.sqrt(1 - par[k, 2] ** 2)
        assert abs(tanphi - coef[1]) < 2e-6
        covyb = np.linalg.inv(A.T @ A) * 1e-6
        assert math.isclose(cov[k, 0], covyb[0, 0], rel_tol=5e-3)   # C_yy; the diffuse prior is negligible
        # z against the path length l = (x - x0) sqrt(1 + tan^2 phi)
        l = (x - x[0]) * math.sqrt(1 + coef[1] ** 2)
        Az = np.stack([np.ones_like(l), l], 1)
        cz, *_ = np.linalg.lstsq(Az, z - z[-1], rcond=None)         # z_ref = z of the top cluster
        assert abs(par[k, 1] - cz[0]) < 2e-5 and abs(par[k, 3] - cz[1]) < 2e-6
        assert o.get("fit_z_ref")[k] == z[-1] and o.get("fit_x_ref")[k] == rx[rows[c[0]]]
        checked += 1
    assert checked >= 15


def test_noise_free_refit_qpt_within_1e4_of_truth():
    tf = generate_config("cfg1", sigma=0.0)
    P = default_params(tf)
    for prec, tol in ((64, 2e-6), (32, 1e-4)):
        o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=prec, last_stage=6)
        par = o.get("fit_par").reshape(-1, 5)
        worst, n = 0.0, 0
        for k, (tid, purity, nc) in enumerate(_truth_of_tracks(tf, o)):
            assert purity == 1.0
            if nc < 70:
                continue
            q_true = tf.truth["q_over_pt"][tid]
            worst = max(worst, abs(par[k, 4] - q_true) / abs(q_true)); n += 1
            assert math.isclose(par[k, 3], tf.truth["tanl"][tid], rel_tol=10 * tol, abs_tol=10 * tol)
        assert n >= 25 and worst < tol, (prec, worst)


def test_refit_pulls_chi2_and_bookkeeping():
    tf = generate_config("cfg1", n_tracks=400, seed=11)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6)
    par = o.get("fit_par").reshape(-1, 5); cov = o.get("fit_cov").reshape(-1, 15)
    chi2, ndf, nfit = o.get("fit_chi2"), o.get("fit_ndf"), o.get("fit_n")
    assert np.array_equal(nfit, o.get("trk_n_clusters"))            # no propagation failure on this sample
    assert np.array_equal(ndf, 2 * nfit - 5) and np.all(chi2 >= 0)
    assert np.array_equal(o.get("fit_x_ref"), P["row_x"].astype(np.float64)[o.get("trk_first_row")])
    pulls, c2 = [], []
    for k, (tid, purity, nc) in enumerate(_truth_of_tracks(tf, o)):
        if purity < 1.0 or nc < 60:
            continue
        pulls.append((par[k, 4] - tf.truth["q_over_pt"][tid]) / math.sqrt(cov[k, 14]))
        c2.append(chi2[k] / ndf[k])
    pulls = np.array(pulls)
    assert pulls.size > 150
    assert abs(pulls.mean()) < 0.25 and 0.8 < pulls.std() < 1.25, (pulls.mean(), pulls.std())
    assert 0.85 < np.mean(c2) < 1.15, np.mean(c2)


def test_residuals_to_the_extrapolated_track():
    """"Hits attached to tracks are stored as residuals to the extrapolated track position, which have a
    smaller entropy than absolute hit positions."  The refit reports that residual (the innovation) per owned cluster."""
    # (i) noise-free: the model predicts the next cluster to a few 10 um (first steps: chord vs tangent direction)
    tf = generate_config("cfg1", sigma=0.0)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=64, last_stage=6)
    st = o.get("trk_cl_start"); ry, rz = o.get("fit_res_y"), o.get("fit_res_z")
    assert ry.shape == o.get("trk_cl_idx").shape
    for k in range(st.size - 1):
        if st[k + 1] - st[k] < 40:
            continue
        assert ry[st[k + 1] - 1] == 0.0 and rz[st[k + 1] - 1] == 0.0        # the top cluster seeds the fit
        assert np.abs(ry[st[k]:st[k + 1]]).max() < 1e-2 and np.abs(rz[st[k]:st[k + 1]]).max() < 1e-2
        assert np.abs(ry[st[k]:st[k + 1] - 10]).max() < 1e-4                  # once the curvature has settled
    # (ii) the loop recomposed in Python from the single-step entries (pinned above) gives the same residuals and state
    k = int(np.argmax(np.diff(st)))
    pos = o.get("trk_cl_pos")[st[k]:st[k + 1]]
    ys, zs, rows = o.get("ys").astype(np.float64), o.get("zs").astype(np.float64), o.get("s_row")
    rx = P["row_x"].astype(np.float64)
    top, nxt = pos[-1], pos[-2]
    dx, dy, dz = rx[rows[top]] - rx[rows[nxt]], ys[top] - ys[nxt], zs[top] - zs[nxt]
    dl = math.sqrt(dx * dx + dy * dy)
    par = np.array([ys[top], 0.0, dy / dl, dz / dl, o.get("trk_par").reshape(-1, 5)[k, 4]])
    cov = np.zeros(15)
    for i, v in zip((0, 2, 5, 9, 14), (P["err_y2"], P["err_z2"], P["init_c_ss"], P["init_c_tt"], P["init_c_qq"])):
        cov[i] = float(v)
    chi2, cur = 0.0, rows[top]
    for i in range(pos.size - 2, -1, -1):
        c = pos[i]
        ok, par, cov, _ = o.kf_propagate(par, cov, rx[cur], rx[rows[c]])
        assert ok
        assert ry[st[k] + i] == ys[c] - par[0] and rz[st[k] + i] == (zs[c] - zs[top]) - par[1]
        par, cov, chi2 = o.kf_update(par, cov, ys[c], zs[c] - zs[top], chi2)
        cur = rows[c]
    assert np.array_equal(par, o.get("fit_par").reshape(-1, 5)[k]) and chi2 == o.get("fit_chi2")[k]
    # (iii) smeared: residual ~ measurement error + prediction error, centred; far fewer bits than the positions
    tf = generate_config("cfg3", n_collisions=2)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=6)
    ry, rz, idx = o.get("fit_res_y"), o.get("fit_res_z"), o.get("trk_cl_idx")
    assert abs(ry.mean()) < 5e-3 and 0.10 < ry.std() < 0.17 and 0.10 < rz.std() < 0.17

    def bits(v, q=0.01):                                     # entropy of the values quantised to 0.1 mm
        _, cnt = np.unique(np.round(v / q).astype(np.int64), return_counts=True)
        p = cnt / cnt.sum()
        return float(-(p * np.log2(p)).sum())
    assert bits(ry) < bits(tf.y[idx]) - 5 and bits(rz) < bits(tf.z[idx]) - 5
