"""Pins for looper following - the apex links of the oracle's merger ("secondary legs of
looping tracks", "the following of looping tracks") - and for the generator's returning branch, CPU only.

* generator: the returning clusters lie on the circle through the origin fixed by the truth parameters and have the z of
  the arc length from the vertex (global geometry with libm, no sector frames); the outgoing clusters do not change;
* an isolated noise-free looper has one right answer: its two legs are each other's apex partner and the returning one
  is labelled secondary - both charges (both curl directions), both sides, two and three sectors between the two ends;
* the score recomposed in Python in double with libm (asin for the arc, cos / sin of k sector angles for the frames),
  for every pair of a piled-up slice: same best partners, same scores; mutual links and labels against their definition;
* no links on frames without loopers; purity / efficiency / labels against generator truth.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config

KB = float(np.float32(-0.00299792458) * np.float32(0.5))
APEX = dict(max_k=4, min_s=0.6, dz_win=150.0, tol_c=0.1, tol_z=4.0, tol_t=0.1, cut=3.0)


def _run(tf, prec=32, P=None):
    P = P or default_params(tf)
    return Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=prec, last_stage=6).merge().apex(**APEX)


def test_generator_returning_branch_is_on_the_same_helix():
    a = generate_config("cfg2", n_tracks=300)
    b = generate_config("cfg2", n_tracks=300, loopers=True)
    out = (b.leg == 0) & (b.track_id >= 0)
    assert np.array_equal(a.y[a.track_id >= 0], b.y[out]) and np.array_equal(a.z[a.track_id >= 0], b.z[out])
    assert np.array_equal(a.sector[a.track_id >= 0], b.sector[out]) and (b.leg == 1).sum() > 0.2 * out.sum()
    c = generate_config("cfg1", n_tracks=40, seed=5, sigma=0.0, pt=("uniform", 0.1, 0.2), loopers=True)
    rx = c.geometry.row_x()
    n_ret = 0
    for t in range(40):
        m = c.track_id == t
        if not m.any():
            continue
        cv = KB * c.truth["q_over_pt"][t]; p0 = c.truth["phi0"][t]; R = 1.0 / abs(cv)
        Cx, Cy = -math.sin(p0) / cv, math.cos(p0) / cv                      # centre of the circle through the origin
        alpha = ((c.sector[m] % 18) + 0.5) * math.radians(20.0)
        xl, yl = rx[c.row[m]], c.y[m].astype(np.float64)
        X, Y = xl * np.cos(alpha) - yl * np.sin(alpha), xl * np.sin(alpha) + yl * np.cos(alpha)
        assert np.abs(np.hypot(X - Cx, Y - Cy) - R).max() < 1e-4
        turn = ((np.arctan2(Y - Cy, X - Cx) - math.atan2(-Cy, -Cx)) * np.sign(cv)) % (2 * math.pi)
        assert np.abs(c.z[m] - (c.truth["z_v"][t] + c.truth["tanl"][t] * turn * R)).max() < 1e-4
        # the returning branch is the later part of the turn, beyond the apex
        if (c.leg[m] == 1).any():
            assert turn[c.leg[m] == 1].min() > math.pi / 2 > 0 and turn[c.leg[m] == 0].max() < turn[c.leg[m] == 1].min()
            n_ret += 1
    assert n_ret >= 15


def _loopers(n_want=40):
    out = []
    for seed in range(1000, 1400):
        tf = generate_config("cfg1", n_tracks=1, seed=seed, sigma=0.0, pt=("uniform", 0.105, 0.175), loopers=True)
        if (tf.leg == 1).sum() >= 30 and (tf.leg == 0).sum() >= 30:
            out.append(tf)
        if len(out) == n_want:
            break
    return out


def test_isolated_looper_legs_find_each_other_and_are_labelled():
    """Kills: the curl direction taken the wrong way round (no candidate sector), the centre formula with the wrong sign of
    cos(phi)/c, frames turned the wrong way, the z advance with the wrong sign of tan(lambda), A / C sides swapped in the
    label."""
    seen = set(); n = 0
    for tf in _loopers():
        o = _run(tf, P=default_params(tf, cell=4.0))
        ss, si = o.get("mrg_seg_start"), o.get("mrg_seg_idx")
        if ss.size != 3:
            continue                                            # both legs found, each as one merged track
        p = o.get("apx_partner")
        assert np.array_equal(p, [1, 0]), (tf.name, p, o.get("apx_best"), o.get("apx_score"))
        ct = o.get("cluster_track"); mo = o.get("mrg_of_track")
        for m in (0, 1):
            legs = tf.leg[np.isin(ct, np.nonzero(mo == m)[0])]
            assert legs.min() == legs.max() == o.get("apx_leg")[m], (tf.name, m, np.bincount(legs), o.get("apx_leg"))
        tails = si[ss[1:] - 1]
        sec = o.get("trk_sector")[tails]
        k = min((sec[0] - sec[1]) % 18, (sec[1] - sec[0]) % 18)
        seen.add((int(np.sign(tf.truth["q_over_pt"][0])), int(sec[0]) // 18, int(k)))
        n += 1
    assert n >= 20
    assert {q for q, _, _ in seen} == {-1, 1} and {s for _, s, _ in seen} == {0, 1} and len({k for _, _, k in seen}) >= 2, seen


def test_score_and_choice_against_a_recomposition_with_libm():
    """Every pair of merged tracks of a piled-up slice, double precision: centres, the chord's arc with asin, frames with
    cos / sin of k sector angles - none of the oracle's series or recurrences."""
    tf = generate_config("cfg3", n_collisions=1, seed=41, loopers=True)
    o = _run(tf, prec=64)
    ss, si = o.get("mrg_seg_start"), o.get("mrg_seg_idx")
    nm = ss.size - 1
    tail = si[ss[1:] - 1]
    up = o.get("up_par").reshape(-1, 5)[tail]; ux = o.get("up_x_ref")[tail]; zo = o.get("up_z_ref")[tail] + up[:, 1]
    sec = o.get("trk_sector")[tail]; un = o.get("up_n")[tail]
    kbf = float(np.float32(KB))
    c = kbf * up[:, 4]
    steep = (un >= 2) & (np.abs(up[:, 2]) >= APEX["min_s"]) & (np.abs(up[:, 2]) < 1) & (c != 0)
    with np.errstate(divide="ignore", invalid="ignore"):
        xc = ux - up[:, 2] / c; yc = up[:, 0] + np.sqrt(1 - up[:, 2] ** 2) / c; R = 1 / np.abs(c)
    th = float(np.float32(np.float32(default_params(tf)["tan_half_sector"])))
    alpha = 2 * math.atan(th)
    best = np.full(nm, -1); score = np.full(nm, np.inf)
    for A in np.nonzero(steep)[0]:
        d = 1 if up[A, 2] >= 0 else -1
        for B in np.nonzero(steep)[0]:
            if A == B or sec[A] // 18 != sec[B] // 18 or c[A] * c[B] >= 0 or abs(zo[B] - zo[A]) > APEX["dz_win"]:
                continue
            k = ((sec[B] % 18) - (sec[A] % 18)) * d % 18
            if k > APEX["max_k"]:
                continue
            ang = d * k * alpha                                  # B's frame is A's frame turned by ang
            rot = lambda x, y: (x * math.cos(ang) - y * math.sin(ang), x * math.sin(ang) + y * math.cos(ang))  # noqa: E731
            xcb, ycb = rot(xc[B], yc[B]); xb, yb = rot(ux[B], up[B, 0])
            Rm = 0.5 * (R[A] + R[B])
            h = 0.5 * math.hypot(xb - ux[A], yb - up[A, 0]) / Rm
            if not h < 0.98:
                continue
            arc = 2 * Rm * math.asin(h)
            sc = ((xc[A] - xcb) ** 2 + (yc[A] - ycb) ** 2) / (APEX["tol_c"] * Rm) ** 2 \
                + ((zo[B] - (zo[A] + up[A, 3] * arc)) / APEX["tol_z"]) ** 2 + ((up[A, 3] + up[B, 3]) / APEX["tol_t"]) ** 2
            if sc <= APEX["cut"] and (sc < score[A] or (sc == score[A] and B < best[A])):
                score[A], best[A] = sc, B
    assert (best >= 0).sum() > 100
    assert np.array_equal(best, o.get("apx_best"))
    got = o.get("apx_score")
    # the arc: two half-angle steps + the 5-term series truncate at 63/2816 h1^10 <= 1.8e-4 of an arc <= 200 cm; with
    # |tan(lambda)| <= 0.9 and |dz| <= sqrt(3) tol_z inside the cut that is <= 0.016 in the score
    assert np.abs(got[best >= 0] - score[best >= 0]).max() < 0.016
    partner = np.array([b if b >= 0 and best[b] == a else -1 for a, b in enumerate(best)])
    assert np.array_equal(partner, o.get("apx_partner"))
    leg = np.zeros(nm, int)
    for a, b in enumerate(partner):
        if b >= 0:
            later = zo[a] > zo[b] if sec[a] < 18 else zo[a] < zo[b]
            leg[a] = int(later or (zo[a] == zo[b] and a > b))
    assert np.array_equal(leg, o.get("apx_leg"))
    assert np.all(leg[partner >= 0] + leg[partner[partner >= 0]] == 1)             # one primary, one secondary per pair


def test_no_links_without_loopers_and_truth_quality_with_them(cfg1):
    assert np.all(_run(cfg1).get("apx_partner") < 0)                                # pT >= 0.5 GeV/c: nothing curls up
    tf = generate_config("cfg3", n_collisions=2, loopers=True)
    o = _run(tf)
    ct = o.get("cluster_track"); nt = o.get("trk_seed").size
    order = np.argsort(ct, kind="stable"); lo = np.searchsorted(ct[order], np.arange(nt)); hi = np.searchsorted(ct[order], np.arange(nt), side="right")
    maj = np.full(nt, -1); mleg = np.full(nt, -1)
    for k in range(nt):
        ids = tf.track_id[order[lo[k]:hi[k]]]; lg = tf.leg[order[lo[k]:hi[k]]]
        if (ids >= 0).any():
            v, cnt = np.unique(ids[ids >= 0] * 2 + lg[ids >= 0], return_counts=True)
            maj[k], mleg[k] = v[cnt.argmax()] // 2, v[cnt.argmax()] % 2
    ss, si = o.get("mrg_seg_start"), o.get("mrg_seg_idx")
    head = si[ss[:-1]]
    T, L = maj[head], mleg[head]
    p, leg = o.get("apx_partner"), o.get("apx_leg")
    pairs = [(a, p[a]) for a in range(ss.size - 1) if p[a] > a]
    good = [(a, b) for a, b in pairs if T[a] == T[b] >= 0 and L[a] != L[b]]
    both = {}
    for m in range(ss.size - 1):
        if T[m] >= 0:
            both.setdefault(int(T[m]), set()).add(int(L[m]))
    possible = sum(1 for v in both.values() if v == {0, 1})
    assert len(pairs) > 1500 and len(good) >= 0.99 * len(pairs) and len(good) >= 0.85 * possible, (len(pairs), len(good), possible)
    right = sum(1 for a, b in good if leg[a] == L[a] and leg[b] == L[b])
    assert right >= 0.98 * len(good), (right, len(good))
