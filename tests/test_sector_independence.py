"""Sectors are independent (DESIGN.md sections 3.1, 5): the oracle run on a whole frame equals, sector by sector, the oracle
run on the clusters of that sector alone.  This is the property the whole-frame GPU parity test rests on
(tests/test_gpu_parity.py::test_full_size_whole_frame_every_array_exact); here the per-sector checker of
tests/parity_util.py is exercised on CPU, with the whole-frame ORACLE standing where the CUDA arrays stand there, and
shown not to be vacuous (a single flipped element is reported)."""
import numpy as np

from tests.parity_util import check_sectors_parallel
from oracle import Oracle
from tpc_synth import default_params

f32 = np.float32


def _frame_from_oracle(tf, P, road=(1.0, 1.0)):
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z, precision=32, last_stage=6)
    T = o.get("trk_seed").shape[0]
    out = dict(n_tracks=T, status=0, sector=o.get("trk_sector"), cluster_track=o.get("cluster_track"),
               trk_cl_start=o.get("trk_cl_start"), trk_cl_idx=o.get("trk_cl_idx"),
               par=o.get("trk_par").astype(f32).reshape(-1, 5), cov=o.get("trk_cov").astype(f32).reshape(-1, 15))
    for nm in ("first_row", "last_row", "n_clusters", "ndf"):
        out[nm] = o.get("trk_" + nm)
    for nm in ("x_ref", "z_ref", "chi2", "z_beam"):
        out[nm] = o.get("trk_" + nm).astype(f32)
    fit = dict(par=o.get("fit_par").astype(f32).reshape(-1, 5), cov=o.get("fit_cov").astype(f32).reshape(-1, 15),
               n_fit=o.get("fit_n"), ndf=o.get("fit_ndf"), res_y=o.get("fit_res_y").astype(f32), res_z=o.get("fit_res_z").astype(f32))
    for nm in ("x_ref", "z_ref", "chi2"):
        fit[nm] = o.get("fit_" + nm).astype(f32)
    F = dict(tf=tf, P=P, out=out, fit=fit, keep=o.protect(*road), road=road,
             yz=np.stack([o.get("ys"), o.get("zs")], 1).reshape(-1),
             srow=(o.get("s_sector") * 256 + o.get("s_row")).astype(np.uint16),
             t_par=o.get("t_par").astype(f32), t_cov=o.get("t_cov").astype(f32), t_chi2=o.get("t_chi2").astype(f32),
             t_zref=o.get("t_z_ref").astype(f32))
    for nm in ("perm", "bin_start", "row_start", "bin_base", "zmin", "zmax", "nz", "link_up_raw", "link_dn_raw", "link_up",
               "link_dn", "seed_head", "seed_len", "t_hit", "t_first_row", "t_last_row", "t_n_hits", "tracklet_of_seed", "k_owned"):
        F[nm] = o.get(nm)
    return F


def test_whole_frame_oracle_equals_per_sector_oracle(mini_tf):
    P = default_params(mini_tf)
    F = _frame_from_oracle(mini_tf, P)
    bad, stats, procs = check_sectors_parallel(F, range(P["n_sectors"]), procs=4)
    assert not any(bad.values()), {s: b for s, b in bad.items() if b}
    assert sum(st["n"] for st in stats.values()) == mini_tf.n
    assert sum(st["tracks"] for st in stats.values()) == F["out"]["n_tracks"] > 100


def test_the_sector_checker_reports_a_single_flipped_element(mini_event):
    P = default_params(mini_event)
    F = _frame_from_oracle(mini_event, P)
    R = P["n_rows"]
    s = 7
    a = int(F["row_start"][s * R])
    for name, mutate in (
        ("link_up", lambda: F["link_up"].__setitem__(a + 5, F["link_up"][a + 5] + 1)),
        ("bin_start", lambda: F["bin_start"].__setitem__(int(F["bin_base"][s * R]) + 3, F["bin_start"][int(F["bin_base"][s * R]) + 3] + 1)),
        ("t_cov", lambda: F["t_cov"].__setitem__(15 * int(np.searchsorted(F["seed_head"], a)) + 4,
                                                 np.nextafter(F["t_cov"][15 * int(np.searchsorted(F["seed_head"], a)) + 4], f32(np.inf)))),
        ("keep", lambda: F["keep"].__setitem__(int(np.nonzero(mini_event.sector == s)[0][0]), 1 - F["keep"][int(np.nonzero(mini_event.sector == s)[0][0])])),
    ):
        mutate()
        bad, _, _ = check_sectors_parallel(F, [s, s + 1], procs=1)
        assert any(m.startswith(name) for m in bad[s]), (name, bad[s])
        assert not bad[s + 1]
        F = _frame_from_oracle(mini_event, P)
