"""Pins for the oracle's integer stages S1-S3 (CPU only).

S1 is pinned to a library routine (numpy lexsort = stable sort) plus an independent per-cluster
recomputation of the bin id; S2's grid lookup to a brute-force all-pairs search over whole rows
(BASELINE.json north_star: "checked on tiny inputs against brute-force all-pairs neighbour search");
S3 to its invariants and a brute-force chain walk.  DESIGN.md section 3.1-3.3.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config

f32 = np.float32


def _run(tf, last_stage, **over):
    P = default_params(tf)
    P.update(over)
    return P, Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=last_stage)


def _bins_independent(tf, P):
    """bin id of every input cluster from the DESIGN.md 3.1 formulas, numpy fp32, no oracle code."""
    R = P["n_rows"]
    rx = P["row_x"].astype(f32)
    ymax = (rx * f32(P["tan_half_sector"])).astype(f32)
    inv_cy = f32(1.0) / f32(P["cell_y"])
    inv_cz = f32(1.0) / f32(P["cell_z"])
    ny = (np.floor((f32(2.0) * ymax) * inv_cy) + 1).astype(np.int64)
    zmin = np.full(P["n_sectors"], np.inf, f32)
    zmax = np.full(P["n_sectors"], -np.inf, f32)
    np.minimum.at(zmin, tf.sector, tf.z)
    np.maximum.at(zmax, tf.sector, tf.z)
    has = zmin <= zmax
    nz = np.where(has, np.floor(((zmax - zmin).astype(f32) * inv_cz).astype(f32)) + 1, 0).astype(np.int64)
    nbins_sr = (nz[:, None] * ny[None, :]).reshape(-1)
    base = np.concatenate([[0], np.cumsum(nbins_sr)])
    s = tf.sector.astype(np.int64)
    r = tf.row.astype(np.int64)
    iy = np.floor(((tf.y + ymax[r]).astype(f32) * inv_cy).astype(f32)).astype(np.int64)
    iz = np.floor(((tf.z - zmin[s]).astype(f32) * inv_cz).astype(f32)).astype(np.int64)
    iy = np.clip(iy, 0, ny[r] - 1)
    iz = np.clip(iz, 0, nz[s] - 1)
    return base[s * R + r] + iz * ny[r] + iy, base


@pytest.mark.parametrize("name,over", [("cfg1", {}), ("cfg2", dict(n_tracks=300)), ("cfg3", dict(n_collisions=2))])
def test_s1_matches_stable_sort_and_independent_bins(name, over):
    tf = generate_config(name, **over)
    P, o = _run(tf, 1)
    gbin, base = _bins_independent(tf, P)
    assert np.array_equal(o.get("gbin").astype(np.int64), gbin)
    assert np.array_equal(o.get("bin_base").astype(np.int64), base)
    perm = o.get("perm")
    # library routine: lexsort is a stable sort, last key is the primary
    want = np.lexsort((np.arange(tf.n), gbin))
    assert np.array_equal(perm, want)
    assert np.array_equal(np.sort(perm), np.arange(tf.n))           # a permutation
    assert np.array_equal(o.get("ys"), tf.y[perm]) and np.array_equal(o.get("zs"), tf.z[perm])
    bs = o.get("bin_start")
    assert bs[0] == 0 and bs[-1] == tf.n and np.all(np.diff(bs) >= 0)
    assert np.array_equal(np.diff(bs), np.bincount(gbin, minlength=bs.size - 1))
    rs = o.get("row_start")
    sr = tf.sector.astype(np.int64) * P["n_rows"] + tf.row
    assert np.array_equal(np.diff(rs), np.bincount(sr, minlength=P["n_sectors"] * P["n_rows"]))


def test_s1_ties_keep_input_order():
    tf = generate_config("cfg1")
    # duplicate every cluster: equal keys must stay in input order
    dup = lambda a: np.concatenate([a, a])  # noqa: E731
    P = default_params(tf)
    o = Oracle(P).run(dup(tf.sector), dup(tf.row), dup(tf.y), dup(tf.z), last_stage=1)
    perm = o.get("perm")
    pairs = perm.reshape(-1)  # equal clusters i and i+n fall in one bin; i must precede i+n
    pos = np.empty_like(pairs)
    pos[perm] = np.arange(perm.size)
    assert np.all(pos[: tf.n] < pos[tf.n:])


def test_s1_degenerate_inputs():
    tf = generate_config("cfg1")
    P = default_params(tf)
    e = np.empty(0)
    o = Oracle(P).run(e, e, e, e, last_stage=5)
    assert o.get("perm").size == 0 and o.get("trk_seed").size == 0
    # out-of-range y / a single cluster / identical z for a whole sector
    o = Oracle(P).run([3], [7], [1e6], [12.5], last_stage=5)
    assert o.get("perm").tolist() == [0] and o.get("nz")[3] == 1 and o.get("cluster_track").tolist() == [-1]
    with pytest.raises(ValueError):
        Oracle(P).run([36], [0], [0.0], [0.0])
    with pytest.raises(ValueError):
        Oracle(P).run([0], [152], [0.0], [0.0])


def _brute_links(o, P, idx):
    """All-pairs search over whole rows with the window predicate and score of DESIGN.md 3.2, numpy fp32."""
    ys, zs = o.get("ys"), o.get("zs")
    ss, rr = o.get("s_sector"), o.get("s_row")
    rs = o.get("row_start")
    R = P["n_rows"]
    rx = P["row_x"].astype(f32)
    ay, az, b, T = f32(P["link_ay"]), f32(P["link_az"]), f32(P["link_b"]), f32(P["link_T"])
    lu = np.full(ys.size, -1, np.int32)
    ld = np.full(ys.size, -1, np.int32)

    def cand(s, t, r, y, z):
        dx = f32(abs(f32(rx[t] - rx[r])))
        yc = f32(y * f32(rx[t] / rx[r]))
        wy = f32(f32(ay * dx) + b)
        wz = f32(f32(az * dx) + b)
        j0, j1 = rs[s * R + t], rs[s * R + t + 1]
        yy, zz = ys[j0:j1], zs[j0:j1]
        m = (yy >= f32(yc - wy)) & (yy <= f32(yc + wy)) & (zz >= f32(z - wz)) & (zz <= f32(z + wz))
        return j0 + np.nonzero(m)[0], dx

    for i in idx:
        s, r, y, z = int(ss[i]), int(rr[i]), ys[i], zs[i]
        U = D = np.empty(0, np.int64)
        for k in (1, 2):
            if r + k < R and U.size == 0:
                U, dxu = cand(s, r + k, r, y, z)
        for k in (1, 2):
            if r - k >= 0 and D.size == 0:
                D, dxd = cand(s, r - k, r, y, z)
        if U.size == 0 or D.size == 0:
            continue
        Dy = (dxd * (ys[U] - y).astype(f32)).astype(f32)[:, None] - (dxu * (y - ys[D]).astype(f32)).astype(f32)[None, :]
        Dz = (dxd * (zs[U] - z).astype(f32)).astype(f32)[:, None] - (dxu * (z - zs[D]).astype(f32)).astype(f32)[None, :]
        Dv = ((Dy * Dy).astype(f32) + (Dz * Dz).astype(f32)).astype(f32)
        a = int(np.argmin(Dv))                          # first minimum in (u asc, d asc) order
        dd = f32(dxu * dxd)
        if Dv.flat[a] <= f32(T * f32(dd * dd)):
            lu[i] = U[a // D.size]
            ld[i] = D[a % D.size]
    return lu, ld


@pytest.mark.parametrize("name,over,cell", [
    ("cfg1", {}, None), ("cfg1", {}, 7.3),
    ("cfg2", dict(n_tracks=400), None), ("cfg3", dict(n_collisions=2, noise=0.3), 3.1),
])
def test_s2_grid_search_equals_brute_force(name, over, cell):
    tf = generate_config(name, **over)
    P = default_params(tf, cell=cell)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=2)
    n = tf.n
    rng = np.random.default_rng(0)
    idx = np.arange(n) if n <= 7000 else np.sort(rng.choice(n, 6000, replace=False))
    lu, ld = _brute_links(o, P, idx)
    assert np.array_equal(o.get("link_up_raw")[idx], lu[idx])
    assert np.array_equal(o.get("link_dn_raw")[idx], ld[idx])
    assert (lu[idx] >= 0).mean() > 0.5                  # not vacuous


def test_s2_straight_tracks_have_zero_deviation():
    """Bz=0, sigma=0: the true (up, down) pair is collinear, so every interior cluster links to its own track."""
    tf = generate_config("cfg1", sigma=0.0, pt=("uniform", 1e6, 2e6))     # pT -> inf: straight lines
    P, o = _run(tf, 3)
    perm = o.get("perm")
    tid = tf.track_id[perm]
    lu, ld = o.get("link_up_raw"), o.get("link_dn_raw")
    has = lu >= 0
    assert has.mean() > 0.9
    assert np.all(tid[lu[has]] == tid[has]) and np.all(tid[ld[has]] == tid[has])


@pytest.mark.parametrize("name,over", [("cfg1", {}), ("cfg2", dict(n_tracks=500)), ("cfg3", dict(n_collisions=2))])
def test_s3_invariants_and_chain_walk(name, over):
    tf = generate_config(name, **over)
    P, o = _run(tf, 3)
    lur, ldr = o.get("link_up_raw"), o.get("link_dn_raw")
    lu, ld = o.get("link_up"), o.get("link_dn")
    n = tf.n
    i = np.arange(n)
    # definition, vectorised differently from the oracle loop
    want_lu = np.where((lur >= 0) & (ldr[np.maximum(lur, 0)] == i), lur, -1)
    want_ld = np.where((ldr >= 0) & (lur[np.maximum(ldr, 0)] == i), ldr, -1)
    assert np.array_equal(lu, want_lu) and np.array_equal(ld, want_ld)
    # mutual: lu[i]=j <=> ld[j]=i
    up = lu >= 0
    assert np.array_equal(ld[lu[up]], i[up])
    dn = ld >= 0
    assert np.array_equal(lu[ld[dn]], i[dn])
    # links go strictly upward in row, same sector
    rr, ss = o.get("s_row"), o.get("s_sector")
    assert np.all(rr[lu[up]] > rr[up]) and np.all(rr[lu[up]] - rr[up] <= 2) and np.all(ss[lu[up]] == ss[up])
    # chains are vertex-disjoint simple paths: brute-force walk from every head
    heads = np.nonzero((lu >= 0) & (ld < 0))[0]
    seen = np.zeros(n, bool)
    lens = []
    for h in heads:
        c, L = h, 0
        while c >= 0:
            assert not seen[c]
            seen[c] = True
            L += 1
            c = lu[c]
        lens.append(L)
    lens = np.array(lens)
    assert seen.sum() == ((lu >= 0) | (ld >= 0)).sum()
    keep = lens >= P["min_chain_len"]
    assert np.array_equal(o.get("seed_head"), heads[keep]) and np.array_equal(o.get("seed_len"), lens[keep])
    assert keep.sum() > 0


def test_s2_brute_force_and_straight_lines_on_non_uniform_pitch():
    """Pad rows with a 4-region pitch (0.75 / 1.0 / 1.2 / 1.5 cm): the distances to the row above and below differ at the
    region borders, so a swapped dx_up / dx_down table or window would show.  Brute force as above; and straight,
    noise-free tracks (Bz = 0) must still link every interior cluster to its own track with zero deviation."""
    from tpc_synth import FOUR_REGION_PITCH, Geometry, generate
    from tpc_synth.generator import CONFIGS
    g = Geometry(pitch_regions=FOUR_REGION_PITCH)
    rx = g.row_x()
    assert not np.allclose(np.diff(rx), np.diff(rx)[0])
    rec = dict(CONFIGS["cfg2"]); rec.update(n_tracks=300)
    tf = generate(rec, geometry=g)
    P = default_params(tf, cell=5.0)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=2)
    idx = np.arange(tf.n) if tf.n <= 7000 else np.sort(np.random.default_rng(1).choice(tf.n, 6000, replace=False))
    lu, ld = _brute_links(o, P, idx)
    assert np.array_equal(o.get("link_up_raw")[idx], lu[idx]) and np.array_equal(o.get("link_dn_raw")[idx], ld[idx])
    assert (lu[idx] >= 0).mean() > 0.5
    # straight lines through the region borders
    rec = dict(CONFIGS["cfg1"]); rec.update(sigma=0.0)
    tf = generate(rec, geometry=Geometry(pitch_regions=FOUR_REGION_PITCH, bz_tesla=0.0))
    P = default_params(tf)
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, last_stage=3)
    perm = o.get("perm"); up = o.get("link_up"); rows = o.get("s_row")
    tid = tf.track_id[perm]
    linked = up >= 0
    assert np.all(tid[up[linked]] == tid[linked])                     # links never leave the track
    border = np.isin(rows, [62, 63, 96, 97, 126, 127])
    assert linked[border].mean() > 0.9                                 # and the region borders are linked through
