"""Pins for the oracle's track merger ("Track Fit"), CPU only.

* the frame rotation (3.9.2): parameters against the rigid rotation written with libm, covariance against the Jacobian
  obtained by central finite differences of "turn the perturbed state, move it back onto the new plane";
* the upward refit (3.9.1): closed-form weighted line fit at Bz = 0 evaluated at the TOP row, q/pT within 1e-4 of truth;
* isolated noise-free helices have one right answer that does not depend on the oracle: a helix crossing a sector border
  is ONE track holding every cluster of both (or all three) segments - in both directions, on both sides, across the
  17 -> 0 wrap; the two tracks a hole of max_gap + 1 rows leaves are one track; a segment of another track is not taken,
  and of two possible continuations the right one is;
* candidate set, score and choice (3.9.3-3.9.5) against a brute force over ALL pairs of tracks recomposed in Python from
  the single-step entries; mutual links, chains and ids against their definition;
* a merged track of one segment is refitted exactly like the refit of section 3.7 (same operations, same bits); across a
  border the merged fit reaches q/pT within 1e-4 of truth and beats the segments;
* generator truth on a piled-up slice: purity and efficiency of the merging.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config, select_sectors

CUTS = dict(max_rows=30, back_rows=1, edge=6.0, dz_win=50.0, chi2_cut=100.0, road_z0=2.0, road_z1=0.3)
A20 = math.radians(20.0)


def _majority_truth(tf, o):
    ct = o.get("cluster_track")
    out = []
    for k in range(o.get("trk_seed").size):
        ids = tf.track_id[ct == k]
        v, c = np.unique(ids, return_counts=True)
        out.append((int(v[np.argmax(c)]), c.max() / ids.size))
    return out


# ------------------------------------------------------------------------------------------------ rotation
def _rigid(par, x, alpha):
    y, z, s, t, q = par
    return x * math.cos(alpha) + y * math.sin(alpha), [y * math.cos(alpha) - x * math.sin(alpha), z,
                                                       math.sin(math.asin(s) - alpha), t, q]


def test_rotation_is_rigid_and_its_jacobian_matches_finite_differences(cfg1):
    """Kills: alpha with the wrong sign in x' or y', cos for sin, a missing slide term (d y'/d y = 1), d z'/d y dropped,
    the curvature term of d s'/d y dropped, d s'/d s inverted."""
    o = Oracle(default_params(cfg1))
    rng = np.random.default_rng(9)
    n_ok = 0
    for _ in range(200):
        x = rng.uniform(85, 245); alpha = rng.choice([-A20, A20])
        par = np.array([rng.uniform(-30, 30), rng.uniform(-200, 200), rng.uniform(-0.8, 0.8), rng.uniform(-0.9, 0.9),
                        rng.uniform(-5, 5)])
        L = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 0.05])[:, None]
        Cm = L @ L.T + np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-5])
        cov15 = np.array([Cm[i, j] for i in range(5) for j in range(i + 1)])
        ok, p1, c1, x1 = o.kf_rotate(par, cov15, x, math.sin(alpha), math.cos(alpha))
        xr, pr = _rigid(par, x, alpha)
        if abs(pr[2]) >= 0.95:
            assert not ok
            continue
        assert ok and abs(x1 - xr) < 1e-11 and np.allclose(p1, pr, rtol=0, atol=1e-11)
        # Jacobian by central differences: perturb, turn rigidly, move back onto the plane x' = x1 with the (separately
        # pinned) helix step
        J = np.zeros((5, 5))
        for i, eps in enumerate([1e-4, 1e-4, 1e-6, 1e-6, 1e-5]):
            d = []
            for sg in (1, -1):
                pp = par.copy(); pp[i] += sg * eps
                xq, pq = _rigid(pp, x, alpha)
                okp, pq, _, _ = o.kf_propagate(pq, np.zeros(15), xq, x1)
                assert okp
                d.append(pq)
            J[:, i] = (d[0] - d[1]) / (2 * eps)
        want = J @ Cm @ J.T
        got = np.zeros((5, 5))
        for m, (i, j) in enumerate((i, j) for i in range(5) for j in range(i + 1)):
            got[i, j] = got[j, i] = c1[m]
        scale = np.sqrt(np.outer(np.diag(want), np.diag(want)))
        assert np.max(np.abs(got - want) / scale) < 2e-6, np.max(np.abs(got - want) / scale)
        n_ok += 1
    assert n_ok > 150
    # a state too steep for the new frame is refused and left untouched
    par = np.array([1.0, 2.0, -0.8, 0.1, 0.5])
    ok, p1, c1, _ = o.kf_rotate(par, np.arange(15.0), 100.0, math.sin(A20), math.cos(A20))
    assert not ok and np.array_equal(p1, par) and np.array_equal(c1, np.arange(15.0))


# ------------------------------------------------------------------------------------------------ isolated helices
def _single_tracks():
    """noise-free single helices from the nominal geometry, with their per-sector cluster counts"""
    out = []
    for seed in range(300, 700):
        tf = generate_config("cfg1", n_tracks=1, seed=seed, sigma=0.0, pt=("uniform", 0.15, 1.2))
        if tf.n < 60:
            continue
        cnt = np.bincount(tf.sector, minlength=36)
        out.append((tf, cnt))
    return out


SINGLES = None


@pytest.fixture(scope="module")
def singles():
    return _single_tracks()


def _run_merge(tf, P=None, prec=32, **cuts):
    P = P or default_params(tf, cell=4.0)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=prec, last_stage=6)
    kw = dict(CUTS); kw.update(cuts)
    return o.merge(**kw)


def test_helix_crossing_a_sector_border_is_one_track(singles):
    """Every cluster of both (all) segments ends up in ONE merged track.  Covers dir = +1 and -1, the A and the C side and
    the wrap between azimuthal sectors 0 and 17.  Kills: the neighbour taken on the wrong side, the rotation applied with
    the wrong sign (the chi2 explodes), A/C sides mixed in the neighbour index, a row window that excludes the same row."""
    seen = set(); n = 0
    for tf, cnt in singles:
        secs = np.nonzero(cnt >= 15)[0]
        if secs.size < 2 or cnt[secs].sum() < tf.n - 8:
            continue
        o = _run_merge(tf)
        nt = o.get("trk_seed").size
        if nt < 2:
            continue
        sec = o.get("trk_sector")
        if len(set(sec.tolist())) != nt:
            continue                                          # two segments in one sector: the hole test covers that
        ss, si = o.get("mrg_seg_start"), o.get("mrg_seg_idx")
        assert ss.size == 2 and ss[-1] == nt, (tf.name, sec, o.get("mrg_best_b"), o.get("mrg_chi2_b"))
        assert np.array_equal(np.sort(si), np.arange(nt)) and np.all(o.get("mrg_of_track") == 0)
        # inner to outer: rows (and radius) grow along the chain
        fr = o.get("trk_first_row")[si]
        assert np.all(np.diff(fr) >= -1)
        assert o.get("mrg_n_clusters")[0] == o.get("trk_n_clusters").sum() >= 0.85 * tf.n
        assert o.get("mrg_n_fit")[0] == o.get("mrg_n_clusters")[0]
        for a in si[:-1]:
            d = int(o.get("mrg_dir")[a]); b = int(o.get("mrg_next")[a])
            assert d in (-1, 1) and sec[b] // 18 == sec[a] // 18 and sec[b] % 18 == (sec[a] % 18 + d) % 18
            seen.add((d, int(sec[a]) // 18, (int(sec[a]) % 18, int(sec[b]) % 18) in ((17, 0), (0, 17))))
        n += 1
    assert n >= 25
    assert {(1, 0), (-1, 0), (1, 1), (-1, 1)} <= {(d, side) for d, side, _ in seen}   # both directions, both sides
    assert any(w for _, _, w in seen)                                                   # the 17 <-> 0 wrap


def _main_sector(tf, cnt, min_rows=110):
    s = int(cnt.argmax())
    sub, _ = select_sectors(tf, [s])
    rows = np.sort(sub.row.astype(int))
    ok = rows.size >= min_rows and np.array_equal(rows, np.arange(rows[0], rows[0] + rows.size))
    return sub if ok else None


def _subset(tf, keep):
    idx = np.nonzero(keep)[0]
    sub, _ = select_sectors(tf, np.unique(tf.sector))
    for f in ("sector", "row", "x", "y", "z", "track_id"):
        setattr(sub, f, getattr(tf, f)[idx].copy())
    return sub


def _long_ones(singles, n_want=5):
    out = []
    for tf, cnt in singles:
        sub = _main_sector(tf, cnt)
        if sub is not None:
            out.append(sub)
        if len(out) == n_want:
            break
    assert len(out) == n_want
    return out


def test_the_two_tracks_around_a_long_hole_become_one(singles):
    """tests/test_oracle_phases.py shows that a hole of max_gap + 1 rows is not crossed by the finder: two tracks.  The
    merger joins them (same sector, dir = 0), and the merged fit over all clusters reaches the truth."""
    for tf in _long_ones(singles):
        r0 = int(tf.row.min()) + 45
        P = default_params(tf, cell=4.0)
        holed = _subset(tf, ~np.isin(tf.row, np.arange(r0, r0 + P["max_gap"] + 1)))
        o = _run_merge(holed, P)
        assert o.get("trk_seed").size == 2
        assert np.array_equal(o.get("mrg_seg_start"), [0, 2]) and np.array_equal(o.get("mrg_seg_idx"), [0, 1])
        assert o.get("mrg_dir")[0] == 0 and o.get("mrg_next")[0] == 1 and o.get("mrg_prev")[1] == 0
        assert o.get("mrg_n_fit")[0] == holed.n
        q_true = tf.truth["q_over_pt"][0]
        assert abs(o.get("mrg_par")[4] - q_true) < 1e-4 * abs(q_true)
        assert o.get("mrg_x_ref")[0] == np.float32(P["row_x"][holed.row.min()])
        # too long a hole for the row window: left alone
        o2 = _run_merge(_subset(tf, ~np.isin(tf.row, np.arange(r0, r0 + 12))), P, max_rows=12)   # fit_row_B = r_A + 13
        assert o2.get("trk_seed").size == 2 and o2.get("mrg_seg_start").size == 3
        o3 = _run_merge(_subset(tf, ~np.isin(tf.row, np.arange(r0, r0 + 12))), P, max_rows=13)
        assert o3.get("mrg_seg_start").size == 2


def test_foreign_segments_are_not_taken_and_the_right_continuation_is_chosen(singles):
    """Lower part L of a helix, its own upper part U, and a copy U2 of the upper part shifted in z.
    * shift 5 cm: outside the chi2 cut - with U removed, L and U2 stay two tracks;
    * shift 0.25 cm: U2 is a candidate of L (chi2 below the cut) but U fits better: L - U merge, U2 stays alone;
    Kills: first candidate instead of best, best without the mutual test, z left out of the score."""
    for tf in _long_ones(singles, 3):
        r0 = int(tf.row.min()) + 50
        P = default_params(tf, cell=4.0)
        lower = tf.row < r0
        upper = tf.row >= r0 + 6

        def frame(shift, with_u):
            parts = [_subset(tf, lower)] + ([_subset(tf, upper)] if with_u else [])
            u2 = _subset(tf, upper); u2.z = (u2.z + np.float32(shift)).astype(np.float32)
            parts.append(u2)
            out = _subset(tf, np.zeros(tf.n, bool))
            for f in ("sector", "row", "x", "y", "z", "track_id"):
                setattr(out, f, np.concatenate([getattr(p, f) for p in parts]))
            return out
        o = _run_merge(frame(5.0, False), P)
        assert o.get("trk_seed").size == 2 and o.get("mrg_seg_start").size == 3 and np.all(o.get("mrg_next") < 0)
        tfc = frame(0.25, True)
        o = _run_merge(tfc, P)
        nt = o.get("trk_seed").size
        assert nt == 3
        zs_top = [o.get("zs")[o.get("trk_cl_pos")[o.get("trk_cl_start")[k + 1] - 1]] for k in range(nt)]
        first = o.get("trk_first_row")
        L = int(np.argmin(first))
        ups = [k for k in range(nt) if k != L]
        U = min(ups, key=lambda k: zs_top[k]) if tfc.z[upper.sum() + lower.sum():].mean() > tfc.z[lower.sum():lower.sum() + upper.sum()].mean() else max(ups, key=lambda k: zs_top[k])
        U2 = [k for k in ups if k != U][0]
        assert o.get("mrg_next")[L] == U and o.get("mrg_prev")[U] == L and o.get("mrg_prev")[U2] < 0
        assert o.get("mrg_best_a")[U2] == L                    # U2 did want L: only the mutual test keeps it out
        assert o.get("mrg_of_track")[L] == o.get("mrg_of_track")[U] != o.get("mrg_of_track")[U2]


def test_choice_is_the_best_not_the_first_and_links_are_mutual(singles):
    """(i) the foreign continuation comes FIRST in z order (shift -0.25 cm as well as +0.25): the best is still taken;
    (ii) two lower parts (L and a copy shifted by 0.25 cm) want the same upper part U: only the better one gets it, the
    other stays alone (without the mutual test U's back link is overwritten by the last taker);
    (iii) a continuation that starts on the very next row (a 1.5 cm kink the finder does not follow) is a candidate:
    the row window starts at r_A + 1.  Kills: first-candidate, no-mutual-test, row window off by one."""
    tf = _long_ones(singles, 1)[0]
    P = default_params(tf, cell=4.0)
    r0 = int(tf.row.min()) + 50
    lower, upper = tf.row < r0, tf.row >= r0 + 6

    def build(parts):
        out = _subset(tf, np.zeros(tf.n, bool))
        for f in ("sector", "row", "x", "y", "z", "track_id"):
            setattr(out, f, np.concatenate([getattr(p_, f) for p_ in parts]))
        return out

    def shifted(mask, dz):
        q = _subset(tf, mask); q.z = (q.z + np.float32(dz)).astype(np.float32)
        return q
    for dz in (0.25, -0.25):                                  # (i)
        o = _run_merge(build([_subset(tf, lower), _subset(tf, upper), shifted(upper, dz)]), P)
        assert o.get("trk_seed").size == 3
        first = o.get("trk_first_row"); L = int(np.argmin(first))
        ztop = lambda k: o.get("zs")[o.get("trk_cl_pos")[o.get("trk_cl_start")[k + 1] - 1]]   # noqa: E731
        zref = float(tf.z[np.argmax(tf.row)])
        U = min((k for k in range(3) if k != L), key=lambda k: abs(ztop(k) - zref))
        assert o.get("mrg_next")[L] == U, dz
    o = _run_merge(build([_subset(tf, lower), shifted(lower, 0.25), _subset(tf, upper)]), P)   # (ii)
    assert o.get("trk_seed").size == 3
    first = o.get("trk_first_row"); U = int(np.argmax(first))
    lows = [k for k in range(3) if k != U]
    assert all(o.get("mrg_best_b")[k] == U for k in lows)                      # both want U
    taker = int(o.get("mrg_best_a")[U])
    other = [k for k in lows if k != taker][0]
    assert o.get("mrg_chi2_b")[taker] < o.get("mrg_chi2_b")[other]
    assert o.get("mrg_next")[taker] == U and o.get("mrg_prev")[U] == taker and o.get("mrg_next")[other] < 0
    assert o.get("mrg_seg_start").size == 3 and o.get("mrg_of_track")[other] != o.get("mrg_of_track")[U]
    kink = build([_subset(tf, tf.row < r0), shifted(tf.row >= r0, 1.5)])        # (iii)
    o = _run_merge(kink, P, chi2_cut=1e6)
    assert o.get("trk_seed").size == 2
    lo, hi = int(np.argmin(o.get("trk_first_row"))), int(np.argmax(o.get("trk_first_row")))
    assert o.get("fit_row")[hi] == o.get("up_row")[lo] + 1 == r0 and o.get("mrg_next")[lo] == hi
    assert _run_merge(kink, P).get("mrg_next")[lo] < 0                         # at the default cut the kink is no continuation


# ------------------------------------------------------------------------------------------------ definitions
def _cov5(c15):
    C = np.zeros((5, 5))
    for m, (i, j) in enumerate((i, j) for i in range(5) for j in range(i + 1)):
        C[i, j] = C[j, i] = c15[m]
    return C


def test_candidates_score_choice_links_and_chains_against_brute_force(mini_tf):
    """All pairs of tracks, no z ordering, the score recomposed from the single-step entries (fp32)."""
    tf = generate_config("cfg2", n_tracks=500, seed=13)
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6).merge(**CUTS)
    nt = o.get("trk_seed").size
    f32 = np.float32
    sec = o.get("trk_sector"); fr = o.get("fit_row"); ur = o.get("up_row")
    fp = o.get("fit_par").reshape(-1, 5); fc = o.get("fit_cov").reshape(-1, 15); fx = o.get("fit_x_ref"); fz = o.get("fit_z_ref")
    up = o.get("up_par").reshape(-1, 5); uc = o.get("up_cov").reshape(-1, 15); ux = o.get("up_x_ref"); uz = o.get("up_z_ref")
    z_in = (fz.astype(f32) + fp[:, 1].astype(f32)).astype(f32)
    z_out = (uz.astype(f32) + up[:, 1].astype(f32)).astype(f32)
    ymax = (P["row_x"] * P["tan_half_sector"]).astype(f32)
    th = f32(P["tan_half_sector"]); den = f32(1) + th * th
    sin_a, cos_a = f32(f32(2) * th) / den, f32(f32(1) - th * th) / den
    assert abs(float(sin_a) - math.sin(A20)) < 1e-6 and abs(float(cos_a) - math.cos(A20)) < 1e-6
    best_b = np.full(nt, -1); best_a = np.full(nt, -1); chi_b = np.full(nt, np.inf); chi_a = np.full(nt, np.inf); dir_b = np.zeros(nt, int)
    n_pairs = 0
    takes_part = (o.get("up_n") >= 2) & (o.get("fit_n") >= 2)     # both refits got past their first cluster
    for a in range(nt):
        for b in range(nt):
            if a == b or sec[a] // 18 != sec[b] // 18 or not (takes_part[a] and takes_part[b]):
                continue
            if sec[a] == sec[b]:
                d = 0
                if not (ur[a] + 1 <= fr[b] <= ur[a] + CUTS["max_rows"]):
                    continue
            else:
                ya = f32(up[a, 0])
                if not (abs(ya) >= f32(ymax[ur[a]] - f32(CUTS["edge"]))):
                    continue
                d = 1 if ya >= 0 else -1
                if sec[b] % 18 != (sec[a] % 18 + d) % 18:
                    continue
                if not (ur[a] - CUTS["back_rows"] <= fr[b] <= ur[a] + CUTS["max_rows"]):
                    continue
            if not (f32(z_out[a] - f32(CUTS["dz_win"])) <= z_in[b] <= f32(z_out[a] + f32(CUTS["dz_win"]))):
                continue
            par, cov, x = up[a].copy(), uc[a].copy(), ux[a]
            if d:
                ok, par, cov, x = o.kf_rotate(par, cov, x, float(sin_a) * d, float(cos_a), precision=32)
                if not ok:
                    continue
            # the road: a straight continuation of the (turned) outer state
            with np.errstate(invalid="ignore"):
                zslope = f32(f32(par[3]) / np.sqrt(f32(f32(1) - f32(f32(par[2]) * f32(par[2])))))
            dxb = f32(f32(fx[b]) - f32(x))
            z_lin = f32(z_out[a] + f32(dxb * zslope))
            if not (abs(f32(z_in[b] - z_lin)) <= f32(f32(CUTS["road_z0"]) + f32(f32(CUTS["road_z1"]) * abs(dxb)))):
                continue
            ok, par, cov, _ = o.kf_propagate(par, cov, x, fx[b], precision=32)
            if not ok:
                continue
            n_pairs += 1
            dlt = [f32(fp[b, 0]) - f32(par[0]), z_in[b] - f32(f32(uz[a]) + f32(par[1])), f32(fp[b, 2]) - f32(par[2]),
                   f32(fp[b, 3]) - f32(par[3]), f32(fp[b, 4]) - f32(par[4])]
            Cd = np.diag(_cov5(cov)).astype(f32); Bd = np.diag(_cov5(fc[b])).astype(f32)
            chi = f32(0)
            for i in range(5):
                chi = f32(chi + f32(f32(dlt[i] * dlt[i]) / f32(Cd[i] + Bd[i])))
            if not chi <= f32(CUTS["chi2_cut"]):
                continue
            if chi < chi_b[a] or (chi == chi_b[a] and b < best_b[a]):
                chi_b[a], best_b[a], dir_b[a] = chi, b, d
            if chi < chi_a[b] or (chi == chi_a[b] and a < best_a[b]):
                chi_a[b], best_a[b] = chi, a
    assert n_pairs > 300 and (best_b >= 0).sum() > 250
    assert np.array_equal(best_b, o.get("mrg_best_b")) and np.array_equal(best_a, o.get("mrg_best_a"))
    got = o.get("mrg_chi2_b")
    assert np.array_equal(np.where(best_b >= 0, chi_b, -1.0).astype(np.float32), got.astype(np.float32))
    # links = mutual best; chains = heads in ascending id followed through `next`
    nxt = np.array([b if b >= 0 and best_a[b] == a else -1 for a, b in enumerate(best_b)])
    assert np.array_equal(nxt, o.get("mrg_next"))
    prv = np.full(nt, -1); prv[nxt[nxt >= 0]] = np.nonzero(nxt >= 0)[0]
    assert np.array_equal(prv, o.get("mrg_prev"))
    assert np.array_equal(np.where(nxt >= 0, dir_b, 0), o.get("mrg_dir"))
    seg, start = [], [0]
    for h in range(nt):
        if prv[h] >= 0:
            continue
        k = h
        while k >= 0:
            seg.append(k); k = nxt[k]
        start.append(len(seg))
    assert np.array_equal(seg, o.get("mrg_seg_idx")) and np.array_equal(start, o.get("mrg_seg_start"))
    mo = o.get("mrg_of_track")
    for m in range(len(start) - 1):
        assert np.all(mo[seg[start[m]:start[m + 1]]] == m)
    assert sorted(seg) == list(range(nt))                          # a partition of the tracks


# ------------------------------------------------------------------------------------------------ the fits
def test_upward_refit_equals_weighted_line_fit_at_zero_field_and_reaches_truth():
    from tpc_synth import Geometry, generate
    from tpc_synth.generator import CONFIGS
    rec = dict(CONFIGS["cfg1"]); rec.update(sigma=1e-3, n_tracks=30, seed=3)
    tf = generate(rec, geometry=Geometry(bz_tesla=0.0))
    P = default_params(tf)
    P["err_y2"] = np.float32(1e-6); P["err_z2"] = np.float32(1e-6)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=64, last_stage=6).merge(**CUTS)
    st, pos = o.get("trk_cl_start"), o.get("trk_cl_pos")
    ys, zs, rows = o.get("ys").astype(np.float64), o.get("zs").astype(np.float64), o.get("s_row")
    rx = P["row_x"].astype(np.float64)
    par = o.get("up_par").reshape(-1, 5); cov = o.get("up_cov").reshape(-1, 15)
    checked = 0
    for k in range(o.get("trk_seed").size):
        c = pos[st[k]:st[k + 1]]
        if c.size < 40:
            continue
        x, y, z = rx[rows[c]], ys[c], zs[c]
        assert o.get("up_n")[k] == c.size and o.get("up_row")[k] == rows[c[-1]] and o.get("up_x_ref")[k] == x[-1]
        A = np.stack([np.ones_like(x), x - x[-1]], 1)            # evaluated at the TOP owned row
        coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        assert abs(par[k, 0] - coef[0]) < 2e-5
        assert abs(par[k, 2] / math.sqrt(1 - par[k, 2] ** 2) - coef[1]) < 2e-6
        assert math.isclose(cov[k, 0], (np.linalg.inv(A.T @ A) * 1e-6)[0, 0], rel_tol=5e-3)
        l = (x - x[-1]) * math.sqrt(1 + coef[1] ** 2)
        cz, *_ = np.linalg.lstsq(np.stack([np.ones_like(l), l], 1), z - z[0], rcond=None)   # z_ref = z of the BOTTOM cluster
        assert abs(par[k, 1] - cz[0]) < 2e-5 and abs(par[k, 3] - cz[1]) < 2e-6
        assert o.get("up_z_ref")[k] == z[0]
        checked += 1
    assert checked >= 15
    # helices: q/pT at the outer end within 1e-4 (fp32) of truth
    tf = generate_config("cfg1", sigma=0.0)
    o = Oracle(default_params(tf)).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6).merge(**CUTS)
    up = o.get("up_par").reshape(-1, 5)
    n = 0
    for k, (tid, purity) in enumerate(_majority_truth(tf, o)):
        if o.get("trk_n_clusters")[k] < 70:
            continue
        assert purity == 1.0 and abs(up[k, 4] - tf.truth["q_over_pt"][tid]) < 1e-4 * abs(tf.truth["q_over_pt"][tid])
        n += 1
    assert n >= 25


def test_merged_fit_of_one_segment_is_the_refit_and_across_borders_it_reaches_truth(singles, mini_tf):
    o = _run_merge(mini_tf, default_params(mini_tf))
    ss, si = o.get("mrg_seg_start"), o.get("mrg_seg_idx")
    one = np.nonzero(np.diff(ss) == 1)[0]
    assert one.size > 300
    k = si[ss[one]]
    for nm in ("par", "cov", "chi2", "x_ref", "z_ref"):
        w = {"par": 5, "cov": 15}.get(nm, 1)
        assert np.array_equal(o.get("mrg_" + nm).reshape(-1, w)[one], o.get("fit_" + nm).reshape(-1, w)[k]), nm
    assert np.array_equal(o.get("mrg_n_fit")[one], o.get("fit_n")[k]) and np.array_equal(o.get("mrg_sector")[one], o.get("trk_sector")[k])
    # across borders, noise-free, double precision: the merged fit sees the whole lever arm
    n = 0
    for tf, cnt in singles:
        secs = np.nonzero(cnt >= 25)[0]
        if secs.size != 2 or cnt[secs].sum() < tf.n - 4:
            continue
        o = _run_merge(tf, prec=64)
        if o.get("trk_seed").size != 2 or o.get("mrg_seg_start").size != 2:
            continue
        q = tf.truth["q_over_pt"][0]
        em = abs(o.get("mrg_par")[4] - q) / abs(q)
        assert em < 1e-6, em                                  # double: the truncation of the arc series only
        assert o.get("mrg_sector")[0] == o.get("trk_sector")[o.get("mrg_seg_idx")[0]]
        assert abs(o.get("mrg_par")[3] - tf.truth["tanl"][0]) < 1e-4
        n += 1
        if n == 12:
            break
    assert n >= 8


def test_merging_against_generator_truth(mini_tf):
    """Piled-up slice with noise: merged tracks of several segments are pure, and most truth tracks found in several
    segments come out as one."""
    o = _run_merge(mini_tf, default_params(mini_tf))
    tr = _majority_truth(mini_tf, o)
    maj = np.array([t for t, _ in tr]); pur = np.array([p for _, p in tr])
    ss, si, mo = o.get("mrg_seg_start"), o.get("mrg_seg_idx"), o.get("mrg_of_track")
    multi = np.nonzero(np.diff(ss) > 1)[0]
    assert multi.size > 1000
    pure = sum(1 for m in multi if len(set(maj[si[ss[m]:ss[m + 1]]])) == 1)
    assert pure >= 0.998 * multi.size, (pure, multi.size)
    good = (maj >= 0) & (pur > 0.8)
    v, c = np.unique(maj[good], return_counts=True)
    split = v[c > 1]
    full = sum(1 for t in split if len(set(mo[good & (maj == t)])) == 1)
    assert split.size > 1000 and full >= 0.95 * split.size, (full, split.size)
    # the merged fit uses the whole lever arm: its q/pT is closer to the truth than the fit of the innermost segment alone
    mq = o.get("mrg_par").reshape(-1, 5)[:, 4]; fq = o.get("fit_par").reshape(-1, 5)[:, 4]
    em, es = [], []
    for m in multi:
        segs = si[ss[m]:ss[m + 1]]
        if len(set(maj[segs])) != 1 or maj[segs[0]] < 0 or o.get("mrg_n_fit")[m] != o.get("mrg_n_clusters")[m]:
            continue
        q = mini_tf.truth["q_over_pt"][maj[segs[0]]]
        em.append((mq[m] - q) / abs(q)); es.append((fq[segs[0]] - q) / abs(q))
    em, es = np.array(em), np.array(es)
    assert em.size > 1000 and np.median(np.abs(em)) < 0.7 * np.median(np.abs(es)), (np.median(np.abs(em)), np.median(np.abs(es)))


def test_odd_geometries_do_not_break_the_neighbour_arithmetic(singles):
    """One sector (no neighbour at all), two sectors (each side has a single sector: its neighbour is itself, skipped),
    an odd sector count: the merger and the apex search run and only join what lies in one sector."""
    tf = _long_ones(singles, 1)[0]
    r0 = int(tf.row.min()) + 45
    holed = _subset(tf, ~np.isin(tf.row, np.arange(r0, r0 + 5)))
    for S in (1, 2, 5):
        P = default_params(tf, cell=4.0); P["n_sectors"] = S
        holed.sector = np.zeros_like(holed.sector)
        o = Oracle(P).run(holed.sector, holed.row, holed.y, holed.z, last_stage=6).merge(**CUTS).apex()
        assert o.get("trk_seed").size == 2 and np.array_equal(o.get("mrg_seg_idx"), [0, 1]) and o.get("mrg_dir")[0] == 0, S
        assert np.all(o.get("apx_partner") < 0)
