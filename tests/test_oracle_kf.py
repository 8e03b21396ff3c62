"""Pins for the oracle's Kalman-filter pieces and stages S4/S5 (CPU only).  DESIGN.md section 3.4-3.5.

* helix step vs the closed-form circle (asin form) and Jacobian vs central finite differences of that closed form;
* KF at Bz=0 vs the closed-form weighted straight-line regression;
* noise-free helices: fitted q/pT within 1e-4 relative of generator truth (BASELINE.json north_star);
* smeared input: pulls ~ N(0,1), chi2/ndf ~ 1;
* invariants (chi2 >= 0, C positive definite, <= 1 hit per row, gaps <= max_gap, every cluster in <= 1 track);
* S5 vs brute-force ownership.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config

KB = -0.00299792458


def _params(**over):
    tf = generate_config("cfg1")
    P = default_params(tf)
    P.update(over)
    return tf, P


def helix_closed_form(p, kb, dx):
    """Exact circle in xy, uniform Bz: sin(phi) linear in x; arc from the angle difference."""
    y, z, s, t, q = p
    c = kb * q
    s1 = s + c * dx
    phi0, phi1 = math.asin(s), math.asin(s1)
    if abs(c) > 1e-14:
        y1 = y + (math.cos(phi0) - math.cos(phi1)) / c
        arc = (phi1 - phi0) / c
    else:
        y1 = y + dx * math.tan(phi0)
        arc = dx / math.cos(phi0)
    return np.array([y1, z + t * arc, s1, t, q])


def _unpack15(c15):
    C = np.zeros((5, 5))
    m = 0
    for i in range(5):
        for j in range(i + 1):
            C[i, j] = C[j, i] = c15[m]
            m += 1
    return C


def _pack15(C):
    return np.array([C[i, j] for i in range(5) for j in range(i + 1)])


def test_helix_step_matches_closed_form_circle():
    _, P = _params()
    o = Oracle(P)
    kb = float(np.float32(KB) * np.float32(0.5))
    rng = np.random.default_rng(1)
    worst = 0.0
    for _ in range(2000):
        s = rng.uniform(-0.85, 0.85)
        q = rng.uniform(-10, 10)
        dx = rng.uniform(-4.5, 4.5)
        if abs(s + kb * q * dx) >= 0.9:
            continue
        p = np.array([rng.uniform(-30, 30), rng.uniform(-200, 200), s, rng.uniform(-0.9, 0.9), q])
        ok, p1, _, _ = o.kf_propagate(p, np.zeros(15), 100.0, 100.0 + dx, precision=64)
        assert ok
        want = helix_closed_form(p, kb, dx)
        worst = max(worst, np.max(np.abs(p1 - want) / np.maximum(1.0, np.abs(want))))
    assert worst < 1e-10, worst
    # fp32 instance: a few ulp of the coordinates
    p = np.array([10.0, 5.0, 0.3, 0.5, 1.5])
    ok, p1, _, _ = o.kf_propagate(p, np.zeros(15), 100.0, 101.06, precision=32)
    assert ok and np.allclose(p1, helix_closed_form(p, kb, float(np.float32(101.06) - np.float32(100.0))), rtol=2e-6, atol=2e-6)


def test_helix_step_fails_beyond_max_sinphi():
    _, P = _params()
    o = Oracle(P)
    ok, p1, _, _ = o.kf_propagate([0, 0, 0.94, 0, -10.0], np.zeros(15), 100.0, 104.0)   # s1 = 0.94 + 0.06 > 0.95
    assert not ok
    ok, _, _, _ = o.kf_propagate([0, 0, 0.96, 0, 0.0], np.zeros(15), 100.0, 101.0)
    assert not ok


def test_jacobian_matches_finite_differences_of_closed_form():
    _, P = _params()
    o = Oracle(P)
    kb = float(np.float32(KB) * np.float32(0.5))
    rng = np.random.default_rng(2)
    for _ in range(300):
        s = rng.uniform(-0.8, 0.8)
        q = rng.uniform(-8, 8)
        dx = rng.uniform(-4.5, 4.5)
        if abs(s + kb * q * dx) >= 0.85:
            continue
        p = np.array([rng.uniform(-3, 3), rng.uniform(-1, 1), s, rng.uniform(-0.9, 0.9), q])   # small y, z: FD round-off
        ok, _, _, J = o.kf_propagate(p, np.zeros(15), 100.0, 100.0 + dx)
        assert ok
        Jfd = np.zeros((5, 5))
        for j in range(5):
            h = 1e-6 * max(1.0, abs(p[j]))
            pp, pm = p.copy(), p.copy()
            pp[j] += h
            pm[j] -= h
            Jfd[:, j] = (helix_closed_form(pp, kb, dx) - helix_closed_form(pm, kb, dx)) / (2 * h)
        scale = np.maximum(np.abs(Jfd), 1e-6)
        rel = np.abs(J - Jfd) / scale
        # dz/dq is a Simpson quadrature: 0.5 % ; every other entry is exact
        mask = np.ones((5, 5), bool)
        mask[1, 4] = False
        assert np.all(np.abs(J - Jfd)[mask] <= 2e-6 * np.maximum(1.0, np.abs(Jfd))[mask]), (J, Jfd)
        assert abs(J[1, 4] - Jfd[1, 4]) <= 5e-3 * abs(Jfd[1, 4]) + 2e-9, (J[1, 4], Jfd[1, 4], rel[1, 4])


def test_covariance_transport_is_J_C_Jt():
    _, P = _params()
    o = Oracle(P)
    rng = np.random.default_rng(3)
    A = rng.normal(size=(5, 5))
    C = A @ A.T + np.eye(5)
    p = np.array([3.0, -7.0, 0.2, 0.4, 2.0])
    ok, _, c1, J = o.kf_propagate(p, _pack15(C), 120.0, 122.12)
    assert ok and np.allclose(_unpack15(c1), J @ C @ J.T, rtol=1e-12, atol=1e-12)


def test_update_is_textbook_kalman():
    _, P = _params()
    o = Oracle(P)
    rng = np.random.default_rng(4)
    A = rng.normal(size=(5, 5))
    C = A @ A.T + np.eye(5)
    p = np.array([3.0, -7.0, 0.2, 0.4, 2.0])
    m = np.array([3.4, -6.1])
    H = np.zeros((2, 5))
    H[0, 0] = H[1, 1] = 1
    V = np.diag([float(P["err_y2"]), float(P["err_z2"])])
    S = H @ C @ H.T + V
    K = C @ H.T @ np.linalg.inv(S)
    r = m - H @ p
    p1, c1, chi2 = o.kf_update(p, _pack15(C), m[0], m[1], chi2=1.5)
    assert np.allclose(p1, p + K @ r, rtol=1e-12)
    assert np.allclose(_unpack15(c1), C - K @ H @ C, rtol=1e-11, atol=1e-12)
    assert math.isclose(chi2, 1.5 + r @ np.linalg.inv(S) @ r, rel_tol=1e-12)


def test_kf_equals_weighted_line_fit_at_zero_field():
    """Bz = 0, Q = 0: the filter over a point list equals weighted straight-line regression in (x, y) and (l, z)
    (up to the weak prior on the slopes and EKF linearisation, both negligible at sigma = 1e-3 cm)."""
    _, P = _params(bz_tesla=np.float32(0.0), err_y2=np.float32(1e-6), err_z2=np.float32(1e-6))
    o = Oracle(P)
    rng = np.random.default_rng(5)
    x = P["row_x"].astype(np.float64)[10:90]
    for _ in range(20):
        a, b = rng.uniform(-10, 10), rng.uniform(-0.4, 0.4)          # y = a + b (x - x0)
        zt = rng.uniform(-0.9, 0.9)
        y = a + b * (x - x[0]) + rng.normal(0, 1e-3, x.size)
        l = (x - x[0]) * math.sqrt(1 + b * b)
        z = 17.0 + zt * l + rng.normal(0, 1e-3, x.size)
        ok, par, cov, chi2 = o.kf_fit(x, y, z, precision=64)
        assert ok
        # closed-form regression, evaluated at the last point
        A = np.stack([np.ones_like(x), x - x[-1]], 1)
        coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        covyb = np.linalg.inv(A.T @ A) * 1e-6
        assert abs(par[0] - coef[0]) < 2e-5
        tanphi = par[2] / math.sqrt(1 - par[2] ** 2)
        assert abs(tanphi - coef[1]) < 2e-6
        C = _unpack15(cov)
        assert math.isclose(C[0, 0], covyb[0, 0], rel_tol=2e-3)
        dsdb = (1 + coef[1] ** 2) ** -1.5                          # s = b / sqrt(1 + b^2)
        assert math.isclose(C[2, 2], covyb[1, 1] * dsdb ** 2, rel_tol=5e-3)
        Az = np.stack([np.ones_like(l), l - l[-1]], 1)
        cz, *_ = np.linalg.lstsq(Az, z - z[0], rcond=None)
        assert abs(par[1] - cz[0]) < 2e-5 and abs(par[3] - cz[1]) < 2e-6
        assert abs(par[4]) < 1e-12 or True                          # q is unobservable at Bz = 0
        assert chi2 >= 0 and 0.5 < chi2 / (2 * x.size - 4) < 1.6


def _match_tracks(tf, o):
    """for every reconstructed track: majority truth id and purity"""
    ct = o.get("cluster_track")
    nt = o.get("trk_seed").size
    out = []
    for k in range(nt):
        ids = tf.track_id[ct == k]
        v, c = np.unique(ids, return_counts=True)
        out.append((int(v[np.argmax(c)]), c.max() / ids.size, ids.size))
    return out


@pytest.mark.parametrize("prec,tol,min_nc", [(64, 2e-6, 70), (64, 1e-4, 30), (32, 1e-4, 30)])
def test_noise_free_helix_qpt_within_1e4_of_truth(prec, tol, min_nc):
    """north_star: "against the analytic helix for noise-free tracks (fitted q/pT within 1e-4 relative)".
    Short segments carry the bias of the N(0, init_c_qq) prior on q/pT (sigma_q^2 / init_c_qq relative) and the
    fp32 rounding of the input coordinates; with >= 70 rows the double instance is at the 1e-6 level."""
    tf = generate_config("cfg1", sigma=0.0)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=prec)
    par = o.get("trk_par").reshape(-1, 5)
    m = _match_tracks(tf, o)
    assert len(m) >= 40
    worst = 0.0
    for k, (tid, purity, nc) in enumerate(m):
        assert purity == 1.0
        if nc < min_nc:
            continue
        q_true = tf.truth["q_over_pt"][tid]
        worst = max(worst, abs(par[k, 4] - q_true) / abs(q_true))
        assert math.isclose(par[k, 3], tf.truth["tanl"][tid], rel_tol=10 * tol, abs_tol=10 * tol)
    assert worst < tol, worst


def test_pulls_and_chi2_on_smeared_input():
    tf = generate_config("cfg1", n_tracks=400, seed=11)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32)
    par = o.get("trk_par").reshape(-1, 5)
    cov = o.get("trk_cov").reshape(-1, 15)
    chi2, ndf = o.get("trk_chi2"), o.get("trk_ndf")
    pulls, c2 = [], []
    for k, (tid, purity, nc) in enumerate(_match_tracks(tf, o)):
        if purity < 1.0 or nc < 60:
            continue
        pulls.append((par[k, 4] - tf.truth["q_over_pt"][tid]) / math.sqrt(cov[k, 14]))
        c2.append(chi2[k] / ndf[k])
    pulls = np.array(pulls)
    assert pulls.size > 150
    assert abs(pulls.mean()) < 0.25 and 0.8 < pulls.std() < 1.25, (pulls.mean(), pulls.std())
    assert 0.85 < np.mean(c2) < 1.15, np.mean(c2)


@pytest.mark.parametrize("name,over", [("cfg1", {}), ("cfg2", dict(n_tracks=600)), ("cfg3", dict(n_collisions=2))])
def test_s4_s5_invariants_and_brute_force_ownership(name, over):
    tf = generate_config(name, **over)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)
    R = P["n_rows"]
    hit = o.get("t_hit").reshape(-1, R)
    K = hit.shape[0]
    s_row, s_sec = o.get("s_row"), o.get("s_sector")
    kept, nh = o.get("t_kept"), o.get("t_n_hits")
    first, last = o.get("t_first_row"), o.get("t_last_row")
    cov = o.get("t_cov").reshape(-1, 15)
    assert np.all(o.get("t_chi2") >= 0)
    for k in range(K):
        rows = np.nonzero(hit[k] >= 0)[0]
        assert np.array_equal(s_row[hit[k, rows]], rows)            # the hit of row r lies in row r
        assert np.all(s_sec[hit[k, rows]] == o.get("t_sector")[k])
        assert rows.size == nh[k] and rows[0] == first[k] and rows[-1] <= last[k]
        assert np.all(np.diff(rows) <= P["max_gap"] + 1)
        assert np.all(np.linalg.eigvalsh(_unpack15(cov[k])) > 0)
        assert kept[k] == (nh[k] >= P["min_tracklet_hits"])
    # brute-force ownership: enumerate, per cluster, every kept tracklet containing it
    tid_of = o.get("tracklet_of_seed")
    best = {}
    for k in np.nonzero(kept)[0]:
        key = (int(nh[k]), -int(tid_of[k]))
        for c in hit[k][hit[k] >= 0]:
            if c not in best or key > best[c][0]:
                best[int(c)] = (key, int(k))
    owned = np.zeros(K, np.int64)
    for c, (_, k) in best.items():
        owned[k] += 1
    assert np.array_equal(owned, o.get("k_owned"))
    survivors = [k for k in range(K) if kept[k] and owned[k] >= P["min_track_hits"]]
    assert np.array_equal(o.get("trk_seed"), survivors)
    ct = o.get("cluster_track")
    perm = o.get("perm")
    want = np.full(tf.n, -1, np.int32)
    rank = {k: i for i, k in enumerate(survivors)}
    for c, (_, k) in best.items():
        if k in rank:
            want[perm[c]] = rank[k]
    assert np.array_equal(ct, want)
    # CSR consistency; every cluster in at most one track
    st, idx = o.get("trk_cl_start"), o.get("trk_cl_idx")
    assert st[0] == 0 and st[-1] == idx.size and np.unique(idx).size == idx.size
    assert np.array_equal(np.diff(st), o.get("trk_n_clusters")) and np.all(np.diff(st) >= P["min_track_hits"])
    for i in range(len(survivors)):
        assert np.all(ct[idx[st[i]:st[i + 1]]] == i)


def test_end_to_end_truth_efficiency():
    """Guards against a vacuous oracle: tracks of a central-event-like sample are found and pure."""
    tf = generate_config("cfg2", n_tracks=1500)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)
    ct = o.get("cluster_track")
    sig = tf.track_id >= 0
    key = tf.track_id[sig].astype(np.int64) * 64 + tf.sector[sig]
    uniq, inv, cnt = np.unique(key, return_inverse=True, return_counts=True)
    big = np.nonzero(cnt >= 20)[0]
    cts = ct[sig]
    found = 0
    for g in big:
        seg = cts[inv == g]
        seg = seg[seg >= 0]
        if seg.size and np.bincount(seg).max() >= 0.5 * cnt[g]:
            found += 1
    assert found / big.size > 0.97, found / big.size
    fakes = 0
    for tid, purity, nc in _match_tracks(tf, o):
        fakes += purity < 0.7
    assert fakes <= 0.02 * o.get("trk_seed").size
    noise_assigned = (ct[~sig] >= 0).mean() if (~sig).any() else 0.0
    assert noise_assigned < 0.02
