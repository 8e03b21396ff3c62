"""Pins for the two CHOICES the oracle makes among several candidates (CPU only):

  * S4 search (`Oracle::search`): the nearest gated cluster of a row -
    gate `d2 <= cut`, strict-minimum `d2`, ties -> lowest sorted position, window half-widths
    `sqrt(cut * (C + err))`, weights `1 / (C + err)`;
  * S2 link cut and pair choice: minimal `Dv` over all (up, down) pairs,
    ties -> smallest u then smallest d, accepted iff `Dv <= link_T * (dxu*dxd)^2`.

Every case is HAND-BUILT from dyadic numbers, so each fp32 operation of the reading is exact and the right
answer is known without running any code (it is written into the test as an input index).  On top of that the
search is compared with a numpy fp32 scan of the WHOLE ROW in position order (no grid, no bins), which pins the
bin cover and the visiting order.  Each docstring lists the plausible mistakes ("mutations") that its case kills.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import FOUR_REGION_PITCH, Geometry, default_params, generate_config
from tpc_synth.generator import TimeFrame

f32 = np.float32
SEC, ROW = 3, 40
ZMIN, ZMAX = 1000.0, 1100.0           # anchors (in row 0) fix the sector's z range: zmin = 1000 exactly


def _params(cell=2.0, cut=16.0, err=0.25, geometry=None):
    g = geometry or Geometry()
    tf = TimeFrame(sector=np.zeros(0, np.uint8), row=np.zeros(0, np.uint8), x=np.zeros(0, f32), y=np.zeros(0, f32),
                   z=np.zeros(0, f32), track_id=np.zeros(0, np.int32), truth={}, geometry=g)
    P = default_params(tf, cell=cell)
    P.update(pick_chi2_cut=f32(cut), err_y2=f32(err), err_z2=f32(err))
    return P


def _row_oracle(P, pts, row=ROW, sec=SEC, anchors=True):
    """S1 on hand-placed clusters of one (sector,row) (+ two anchors in row 0 that fix zmin/zmax).  Returns the
    oracle and `pos_of`, the sorted position of every input index."""
    pts = np.asarray(pts, dtype=np.float64).reshape(-1, 2)
    n = pts.shape[0]
    sector = np.full(n, sec, np.uint8); rows = np.full(n, row, np.uint8)
    y = pts[:, 0].astype(f32); z = pts[:, 1].astype(f32)
    assert np.array_equal(y.astype(np.float64), pts[:, 0]) and np.array_equal(z.astype(np.float64), pts[:, 1]), "not fp32-exact"
    if anchors:
        sector = np.concatenate([sector, [sec, sec]]).astype(np.uint8)
        rows = np.concatenate([rows, [0, 0]]).astype(np.uint8)
        y = np.concatenate([y, [0.0, 0.0]]).astype(f32); z = np.concatenate([z, [ZMIN, ZMAX]]).astype(f32)
    o = Oracle(P).run(sector, rows, y, z, last_stage=1)
    perm = o.get("perm")
    pos_of = np.empty_like(perm); pos_of[perm] = np.arange(perm.size)
    return o, pos_of, perm


def _cov(c00, c11):
    c = np.zeros(15); c[0] = c00; c[2] = c11; c[5] = c[9] = c[14] = 1.0
    return c


def _search(o, perm, y0, zref, zrel, c00, c11):
    """input index of the cluster the oracle's search returns (or -1)"""
    j = o.search([y0, zrel, 0.0, 0.0, 0.0], _cov(c00, c11), zref, SEC, ROW)
    return -1 if j < 0 else int(perm[j])


def _scan_whole_row(o, P, y0, zref, zrel, c00, c11, sec=SEC, row=ROW):
    """DESIGN.md 3.4.3 as a numpy fp32 scan over EVERY cluster of the row in ascending position - no grid."""
    rs = o.get("row_start"); R = P["n_rows"]
    j0, j1 = int(rs[sec * R + row]), int(rs[sec * R + row + 1])
    ys, zs = o.get("ys"), o.get("zs")
    cut = f32(P["pick_chi2_cut"])
    y0, zref, zrel = f32(y0), f32(zref), f32(zrel)
    sy2 = f32(f32(c00) + f32(P["err_y2"])); sz2 = f32(f32(c11) + f32(P["err_z2"]))
    hy = np.sqrt(f32(cut * sy2)); hz = np.sqrt(f32(cut * sz2))
    zabs = f32(zref + zrel)
    ylo, yhi, zlo, zhi = f32(y0 - hy), f32(y0 + hy), f32(zabs - hz), f32(zabs + hz)
    wy, wz = f32(f32(1) / sy2), f32(f32(1) / sz2)
    best, arg, n_gated = f32(np.inf), -1, 0
    for j in range(j0, j1):
        if not (ys[j] >= ylo and ys[j] <= yhi and zs[j] >= zlo and zs[j] <= zhi):
            continue
        dy = f32(ys[j] - y0); dz = f32(f32(zs[j] - zref) - zrel)
        d2 = f32(f32(f32(dy * dy) * wy) + f32(f32(dz * dz) * wz))
        if d2 <= cut:
            n_gated += 1
            if d2 < best:
                best, arg = d2, j
    return arg, n_gated


# state used by the hand cases: y = 1, z_ref = 1040, z_rel = 0.5 (absolute z 1040.5); C00 + err = 1 exactly
Y0, ZREF, ZREL = 1.0, 1040.0, 0.5
ZABS = ZREF + ZREL


def test_search_tie_inside_one_bin_goes_to_the_lower_input_index():
    """Two clusters at IDENTICAL coordinates (same bin, d2 = 0.5 each): stable S1 order puts the first input first, and
    the strict `d2 < best` keeps it.  Kills: `<=` (last minimum wins), ties -> highest position."""
    P = _params()
    o, pos_of, perm = _row_oracle(P, [(Y0 + 0.5, ZABS + 0.5), (Y0 + 0.5, ZABS + 0.5), (Y0 - 3.0, ZABS - 3.0)])
    assert pos_of[0] < pos_of[1]
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == 0


def test_search_tie_across_bin_rows_goes_to_the_lowest_position_not_the_first_input():
    """Equal d2 = 1 at z + 1 (input 0) and z - 1 (input 1); cell 2 cm puts them in different bin rows, the lower z first.
    Kills: ties -> lowest INPUT index, `<=`, z rows walked downward."""
    P = _params()
    o, pos_of, perm = _row_oracle(P, [(Y0, ZABS + 1.0), (Y0, ZABS - 1.0)])
    assert pos_of[1] < pos_of[0]
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == 1


def test_search_takes_the_minimum_not_the_first_or_the_largest():
    """In position order: d2 = 4 (z - 2), d2 = 1 (y + 1), d2 = 9 (z + 3), all inside the gate (cut 16).
    Kills: first gated candidate, max for min, last candidate."""
    P = _params()
    o, pos_of, perm = _row_oracle(P, [(Y0, ZABS - 2.0), (Y0 + 1.0, ZABS), (Y0, ZABS + 3.0)])
    assert pos_of[0] < pos_of[1] < pos_of[2]
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == 1


def test_search_weights_are_inverse_variances_each_on_its_own_axis():
    """sy2 = 1, sz2 = 4.  A = (dy 1.5, dz 0): d2 = 2.25;  B = (dy 0, dz 2): d2 = 1  ->  B.
    Kills: `* sy2` for `/ sy2` (A 2.25 vs B 16 -> A), sy2 <-> sz2 swapped (A 0.5625 vs B 4 -> A), unweighted Euclid
    distance (A 2.25 vs B 4 -> A)."""
    P = _params()
    o, pos_of, perm = _row_oracle(P, [(Y0 + 1.5, ZABS), (Y0, ZABS + 2.0)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 3.75) == 1


def test_search_gate_beats_euclidean_nearness():
    """cut = 4, sy2 = 1, sz2 = 4.  A = (dy 2.25, dz 0) is nearer in cm but d2 = 5.0625 > cut (and outside the window,
    hy = 2); B = (dy 0, dz 3) has d2 = 2.25.  -> B; A alone -> nothing.  Kills: no gate, gate on cm distance, window
    half-width without the cut or without the sqrt (hz = sqrt(4*4) = 4 must contain dz = 3; `cut*sz2` = 16 would too,
    `sz2` = 4 would, `sqrt(sz2)` = 2 would NOT)."""
    P = _params(cut=4.0)
    o, pos_of, perm = _row_oracle(P, [(Y0 + 2.25, ZABS), (Y0, ZABS + 3.0)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 3.75) == 1
    o, pos_of, perm = _row_oracle(P, [(Y0 + 2.25, ZABS)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 3.75) == -1


def test_search_gate_is_closed_and_a_rectangle_member_above_the_cut_is_refused():
    """cut = 25, sy2 = sz2 = 1, window +-5.  (dy 3, dz 4): d2 = 25 == cut exactly -> accepted.  dz one fp32 ulp of the
    absolute z larger (4 + 2^-13): d2 > 25 -> refused although it lies inside the window rectangle.  (dy 4.5, dz 4.5) is
    inside the rectangle with d2 = 40.5 -> refused.  Kills: `<` for `<=` in the gate, rectangle membership taken as the
    gate, gate applied to one axis only."""
    P = _params(cut=25.0)
    o, pos_of, perm = _row_oracle(P, [(Y0 + 3.0, ZABS + 4.0)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == 0
    z_up = float(np.nextafter(f32(ZABS + 4.0), f32(np.inf)))
    assert z_up - (ZABS + 4.0) == 2.0 ** -13
    o, pos_of, perm = _row_oracle(P, [(Y0 + 3.0, z_up)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == -1
    o, pos_of, perm = _row_oracle(P, [(Y0 + 4.5, ZABS + 4.5)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == -1
    # ... and the accepted one wins over a farther gated one whatever the order
    o, pos_of, perm = _row_oracle(P, [(Y0 - 4.0, ZABS - 3.0), (Y0 + 3.0, ZABS + 4.0), (Y0 + 1.0, ZABS + 4.0)])
    assert _search(o, perm, Y0, ZREF, ZREL, 0.75, 0.75) == 2         # d2 = 25, 25, 17


def test_search_z_is_taken_relative_to_z_ref():
    """The state carries z - z_ref: the same geometry shifted to another z_ref / z_rel split must give the
    same answer.  Kills: dz = zs - z_rel (z_ref dropped), window centred on z_rel."""
    P = _params()
    pts = [(Y0, ZABS - 2.0), (Y0 + 1.0, ZABS), (Y0, ZABS + 3.0)]
    o, pos_of, perm = _row_oracle(P, pts)
    for zref, zrel in ((ZREF, ZREL), (ZABS, 0.0), (ZMIN, ZABS - ZMIN), (ZABS + 8.0, -8.0)):
        assert _search(o, perm, Y0, zref, zrel, 0.75, 0.75) == 1


@pytest.mark.parametrize("edge", ["zmin", "zmax", "ymax", "ymin"])
def test_search_window_clamped_at_the_first_and_last_bins(edge):
    """The window reaches past the grid on one side: the bin cover is clamped, the members are still found - also a
    cluster that lies OUTSIDE the pad row in y (clamped into the edge bin by S1).  Checked against the hand answer and
    the whole-row scan.  Kills: unclamped bin indices, an off-by-one at the last bin (iy1 + 1), windows cut at the grid."""
    P = _params()
    ymax = float(f32(P["row_x"][ROW]) * f32(P["tan_half_sector"]))
    yedge = float(np.floor(ymax * 4) / 4)                              # dyadic, just inside the pad row
    if edge == "zmin":
        st = (Y0, ZMIN, 1.0)
        pts = [(Y0, ZMIN), (Y0 + 0.5, ZMIN + 0.25), (Y0, ZMIN + 4.5)]
        want = 1                                                      # d2 = 1, 0.8125, 12.25
    elif edge == "zmax":
        st = (Y0, ZMAX, -1.0)
        pts = [(Y0, ZMAX - 4.5), (Y0 + 0.5, ZMAX - 0.25), (Y0, ZMAX)]
        want = 1                                                      # d2 = 12.25, 0.8125, 1
    elif edge == "ymax":
        st = (yedge, ZREF, ZREL)
        pts = [(yedge - 3.0, ZABS), (yedge + 1.5, ZABS), (yedge + 0.5, ZABS + 1.0)]    # the 2nd and 3rd lie beyond ymax
        want = 2                                                      # d2 = 9, 2.25, 1.25
    else:
        st = (-yedge, ZREF, ZREL)
        pts = [(-yedge + 3.0, ZABS), (-yedge - 1.5, ZABS), (-yedge - 0.5, ZABS - 1.0)]
        want = 2
    o, pos_of, perm = _row_oracle(P, pts)
    got = _search(o, perm, st[0], st[1], st[2], 0.75, 0.75)
    assert got == want
    arg, n_gated = _scan_whole_row(o, P, st[0], st[1], st[2], 0.75, 0.75)
    assert n_gated == 3 and int(perm[arg]) == want


@pytest.mark.parametrize("cell", [2.0, 3.7, 16.0])
def test_search_equals_a_whole_row_scan_on_crowded_rows(cell):
    """600 clusters (with exact duplicates) in one row, 400 random states with windows covering one to many bin rows:
    the grid search must return what a scan of the whole row in position order returns.  Kills: a bin row skipped or
    visited twice, windows straddling bin rows handled wrongly, iy0/iy1 swapped, visiting order not ascending."""
    rng = np.random.default_rng(7)
    P = _params(cell=cell, cut=15.0, err=0.01)
    ymax = float(P["row_x"][ROW] * P["tan_half_sector"])
    y = rng.uniform(-ymax, ymax, 600).astype(f32); z = rng.uniform(ZMIN, ZMAX, 600).astype(f32)
    y[500:] = y[:100]; z[500:] = z[:100]                              # duplicates: equal d2, tie by position
    o, pos_of, perm = _row_oracle(P, np.stack([y, z], 1).astype(np.float64))
    found = multi = 0
    for _ in range(400):
        y0 = float(f32(rng.uniform(-ymax - 1, ymax + 1))); zabs = rng.uniform(ZMIN - 3, ZMAX + 3)
        zref = float(f32(zabs + rng.uniform(-20, 20))); zrel = float(f32(zabs - zref))
        c00, c11 = float(f32(rng.uniform(0, 2.0))), float(f32(rng.uniform(0, 6.0)))
        j = o.search([y0, zrel, 0.0, 0.0, 0.0], _cov(c00, c11), zref, SEC, ROW)
        arg, n_gated = _scan_whole_row(o, P, y0, zref, zrel, c00, c11)
        assert j == arg
        found += j >= 0; multi += n_gated >= 2
    assert found > 200 and multi > 100                                # not vacuous: most queries chose among several


# ------------------------------------------------------------------------------------------------ S2
# 4-region pad-row pitch: rows 61, 62, 63 sit at x = 130.75, 131.5, 132.375 (all fp32-exact), so for a cluster of row 62
# the distance up (0.875) differs from the distance down (0.75); row 64 is at 133.375.
G4 = Geometry(pitch_regions=FOUR_REGION_PITCH)
R_ME, S_ME = 62, 5
DXU, DXD, DXU2 = 0.875, 0.75, 1.875


def _links(pts_by_row, T=1.0, cell=0.25):
    """S2 on hand-placed clusters {row: [(y, z), ...]} of one sector; returns (input index of up link, of down link) of
    the FIRST cluster given for row 62, or (-1, -1)."""
    rx = G4.row_x()
    assert (rx[61], rx[62], rx[63], rx[64]) == (130.75, 131.5, 132.375, 133.375)
    P = _params(cell=cell, geometry=G4)
    P["link_T"] = f32(T)
    rows, y, z = [], [], []
    for r, pts in pts_by_row.items():
        for (yy, zz) in pts:
            rows.append(r); y.append(yy); z.append(zz)
    me = rows.index(R_ME)
    y = np.array(y, np.float64); z = np.array(z, np.float64)
    assert np.array_equal(y.astype(f32).astype(np.float64), y)
    o = Oracle(P).run(np.full(len(rows), S_ME, np.uint8), np.array(rows, np.uint8), y.astype(f32), z.astype(f32), last_stage=2)
    perm = o.get("perm"); pos_of = np.empty_like(perm); pos_of[perm] = np.arange(perm.size)
    lu, ld = int(o.get("link_up_raw")[pos_of[me]]), int(o.get("link_dn_raw")[pos_of[me]])
    return (-1 if lu < 0 else int(perm[lu])), (-1 if ld < 0 else int(perm[ld]))


def _up(v):
    return float(np.nextafter(f32(v), f32(np.inf)))


def _down(v):
    return float(np.nextafter(f32(v), f32(-np.inf)))


@pytest.mark.parametrize("T,yu", [(1.0, 0.875), (0.25, 0.4375)])
def test_link_cut_at_just_under_and_just_over(T, yu):
    """me = (0, 50) in row 62, d = (0, 50) in row 61, u = (yu, 50) in row 63:  Dy = dxd*yu, Dz = 0, Dv = (0.75*yu)^2 and
    the cut is T*(0.875*0.75)^2 - equal for yu = 0.875*sqrt(T), every operation exact.  At and one ulp below the cut the
    pair is accepted, one ulp above it is refused.  Kills: `<` for `<=`, the cut without the square (T*dxu*dxd = 0.656
    would accept), link_T left out or applied to the un-squared product, dxu*dxu or dxd*dxd for dxu*dxd."""
    z = 50.0
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(yu, z)]}, T=T) == (2, 1)
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(_down(yu), z)]}, T=T) == (2, 1)
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(_up(yu), z)]}, T=T) == (-1, -1)
    # the same along z (Dz carries the deviation, Dy = 0)
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(0.0, z + yu)]}, T=T) == (2, 1)
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(0.0, _up(z + yu))]}, T=T) == (-1, -1)


def test_link_cut_uses_the_row_distances_of_the_widened_step():
    """Row 63 empty -> the up link widens to row 64, dxu = 1.875: (0.75*yu)^2 <= (1.875*0.75)^2 iff yu <= 1.875.
    Kills: the k = 1 distance used for a k = 2 link (cut and score), widening that forgets the cut table."""
    z = 50.0
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 64: [(DXU2, z)]}) == (2, 1)
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 64: [(_up(DXU2), z)]}) == (-1, -1)
    # k = 1 has priority: with a row-63 candidate present (far off the line, refused) row 64 is not looked at
    assert _links({62: [(0.0, z)], 61: [(0.0, z)], 63: [(1.5, z)], 64: [(0.0, z)]}) == (-1, -1)


def test_link_score_is_zero_on_a_straight_line_through_unequal_row_distances():
    """d = (-0.75 k, .), me = (0, .), u = (+0.875 k, .) are collinear in (x, y) and (x, z) for any k: Dv = 0 exactly and
    the pair survives link_T = 1e-6.  Kills: dxu <-> dxd swapped in the score (Dy = 0.875^2 - 0.75^2 = 0.203), a sign
    error in either bracket."""
    for k in (1.0, -0.5):
        got = _links({62: [(0.0, 50.0)], 61: [(-DXD * k, 50.0 - 2 * DXD * k)], 63: [(DXU * k, 50.0 + 2 * DXU * k)]}, T=1e-6, cell=2.0)
        assert got == (2, 1)


def test_link_pair_choice_is_the_global_minimum_over_all_pairs():
    """u in {0.3, -0.6}, d in {-0.2, 0.5} (inputs 1, 2 and 3, 4):  Dy = 0.75 yu + 0.875 yd = 0.05, 0.6625, -0.625, -0.0125
    -> the pair (-0.6, 0.5) = inputs (2, 4).  Kills: nearest u and nearest d chosen separately (0.3 and -0.2), a sign
    error in (y - yd) (picks (0.3, 0.5)), first pair."""
    z = 50.0
    got = _links({62: [(0.0, z)], 63: [(0.3125, z), (-0.625, z)], 61: [(-0.1875, z), (0.5, z)]})
    # dyadic stand-ins: 0.75*0.3125 = 0.234375, 0.75*(-0.625) = -0.46875, 0.875*(-0.1875) = -0.1640625, 0.875*0.5 = 0.4375
    # sums: 0.0703125, 0.671875, -0.6328125, -0.03125 -> (-0.625, 0.5)
    assert got == (2, 4)


def test_link_ties_go_to_the_smallest_up_position_then_the_smallest_down_position():
    """u = +-0.5 (inputs 1, 2; the later input has the lower y, hence the lower bin and position), d = 0: equal Dv ->
    input 2.  Then d = +-0.5 with u = 0 -> the lower-y d.  Kills: `<=` (last pair), ties by input index."""
    z = 50.0
    assert _links({62: [(0.0, z)], 63: [(0.5, z), (-0.5, z)], 61: [(0.0, z)]}) == (2, 3)
    assert _links({62: [(0.0, z)], 63: [(0.0, z)], 61: [(0.5, z), (-0.5, z)]}) == (1, 3)
    # both at once: four pairs, Dy = +-0.375 +- 0.4375; |Dy| = 0.0625 for (u=+0.5, d=-0.5) and (u=-0.5, d=+0.5): the
    # smaller u position (y = -0.5, input 2) wins, with its partner d = +0.5 (input 3)
    assert _links({62: [(0.0, z)], 63: [(0.5, z), (-0.5, z)], 61: [(0.5, z), (-0.5, z)]}) == (2, 3)
