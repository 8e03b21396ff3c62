"""Synthetic, seeded TPC time frames (stand-ins for the paper's simulated data).

The ALICE simulated time frames the paper measures on are
not available; BASELINE.json ``configs`` describes five synthetic workloads of
the same shape.  This module produces them:

* geometry: 36 sectors (18 azimuthal x 2 sides), 152 pad rows at
  x = 85 .. 245 cm (uniform pitch), Bz = 0.5 T, drift velocity 2.5 cm/us over
  250 cm (100 us drift window; BASELINE.json configs[2]; PAPER.md:29 says 90 us);
* primary helices from (0, 0, z_v): phi0 ~ U[0, 2pi), charge +-1, tan(lambda)
  ~ U[-0.9, 0.9], pT per config; first outgoing branch only - with the recipe key
  ``loopers=True`` also the RETURNING branch of tracks that curl up inside the TPC
  (second intersection of the circle with every pad-row line, truth-labelled in
  ``TimeFrame.leg``; "secondary legs of looping tracks");
* one cluster per crossed (sector, row): exact circle / row-line intersection
  in double precision in the sector-local frame, Gaussian smearing in y and z;
* continuous readout: the cluster z handed to the tracker is
  the *pseudo-z* computed with vertex time 0: A side z' = z - v_d t_coll,
  C side z' = z + v_d t_coll;
* uniform noise clusters; emission order (collision, track, row) then noise,
  i.e. NOT grouped by sector / row.

Random numbers come from numpy's counter-based Philox keyed by
(seed, stream), so the output does not depend on chunking or on the device the
double-precision geometry is evaluated on (``device='cuda'`` only speeds the
arithmetic up; all draws are made on the host).

Nothing here is part of the tracking method: no binning, no links, no fit.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

C_LIGHT_KB = -0.00299792458  # curvature [1/cm] = C_LIGHT_KB * Bz[T] * (q/pT [c/GeV])


@dataclass(frozen=True)
class Geometry:
    n_sectors: int = 36
    n_rows: int = 152
    x_first: float = 85.0
    x_last: float = 245.0
    half_sector_deg: float = 10.0
    bz_tesla: float = 0.5
    v_drift: float = 2.5          # cm / us
    drift_length: float = 250.0   # cm
    # optional non-uniform pad-row pitch: ((pitch_cm, n_rows), ...) regions from x_first outwards, n_rows summing to
    # n_rows (a second geometry that makes the up and down row distances differ)
    pitch_regions: tuple = ()

    def row_x(self) -> np.ndarray:
        if self.pitch_regions:
            steps = np.concatenate([np.full(int(n), float(p)) for p, n in self.pitch_regions])
            assert steps.shape[0] == self.n_rows
            return self.x_first + np.concatenate([[0.0], np.cumsum(steps[1:] * 0.5 + steps[:-1] * 0.5)])
        r = np.arange(self.n_rows, dtype=np.float64)
        return self.x_first + r * (self.x_last - self.x_first) / (self.n_rows - 1)

    @property
    def tan_half_sector(self) -> float:
        return math.tan(math.radians(self.half_sector_deg))

    @property
    def n_azimuthal(self) -> int:
        return self.n_sectors // 2


@dataclass
class TimeFrame:
    sector: np.ndarray      # uint8 [N]
    row: np.ndarray         # uint8 [N]
    x: np.ndarray           # float32 [N]  (= pad-row centre, row_x[row])
    y: np.ndarray           # float32 [N]
    z: np.ndarray           # float32 [N]  pseudo-z
    track_id: np.ndarray    # int32 [N], -1 for noise   (truth, never seen by a tracker)
    truth: dict             # per generated track: q_over_pt, tanl, phi0, z_v, t_coll (float64), collision
    geometry: Geometry = field(default_factory=Geometry)
    tf_length_us: float = 0.0
    sigma: float = 0.1
    name: str = ""
    leg: np.ndarray | None = None   # int8 [N]: 0 outgoing branch, 1 returning branch of a looper (recipe key `loopers`); truth

    @property
    def n(self) -> int:
        return int(self.sector.shape[0])


# --------------------------------------------------------------------------- RNG
def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed) & 0xFFFFFFFFFFFFFFFF, int(stream)]))


_STREAM_COLLISIONS = 0
_STREAM_NOISE = 1
_STREAM_TRACKS = 2
_STREAM_SMEAR0 = 1000
_STREAM_SMEAR_RET0 = 2_000_000   # smear normals of the returning branches (recipe key `loopers`)
_SMEAR_CHUNK = 8192  # tracks per smear stream; fixed, part of the recipe


# the 4-region pitch of SURVEY.md section 8c-2 (0.75 / 1.0 / 1.2 / 1.5 cm x 63 / 34 / 30 / 25 rows)
FOUR_REGION_PITCH = ((0.75, 63), (1.0, 34), (1.2, 30), (1.5, 25))


# ------------------------------------------------------------------- configs
# Recipes for BASELINE.json configs[0..4] (names cfg1..cfg5 follow SURVEY.md section 8d).
CONFIGS = {
    "cfg1": dict(kind="single_sector", n_tracks=40, pt=("uniform", 0.5, 5.0), zv_sigma=0.0,
                 sigma=0.1, noise=0.0, seed=0, tf_us=0.0),
    "cfg2": dict(kind="event", n_tracks=8000, pt=("power3", 0.1, 20.0), zv_sigma=5.0,
                 sigma=0.1, noise=0.02, seed=2, tf_us=0.0),
    "cfg3": dict(kind="timeframe", n_collisions=10, mult=("exp", 1600.0), pt=("power3", 0.1, 20.0),
                 zv_sigma=5.0, sigma=0.1, noise=0.05, seed=3, tf_us=100.0),
    "cfg4": dict(kind="timeframe", n_collisions=1000, mult=("poisson", 30.0), pt=("power3", 0.1, 20.0),
                 zv_sigma=5.0, sigma=0.1, noise=0.03, seed=4, tf_us=1000.0),
    "cfg5": dict(kind="timeframe", n_collisions=570, mult=("exp", 1600.0), pt=("power3", 0.1, 20.0),
                 zv_sigma=5.0, sigma=0.1, noise=0.05, seed=5, tf_us=11400.0),
}


def generate_config(name: str, device: str = "cpu", **override) -> TimeFrame:
    """Generate one of the BASELINE.json workloads.  ``override`` replaces recipe keys
    (e.g. ``n_collisions=20`` for a reduced cfg5, ``sigma=0.0`` for the noise-free twin)."""
    rec = dict(CONFIGS[name])
    rec.update(override)
    tf = generate(rec, device=device)
    tf.name = name if not override else name + "+" + ",".join(f"{k}={v}" for k, v in sorted(override.items()))
    return tf


# ------------------------------------------------------------------ generator
def _draw_pt(rng: np.random.Generator, spec, n: int) -> np.ndarray:
    kind = spec[0]
    if kind == "uniform":
        return rng.uniform(spec[1], spec[2], n)
    if kind == "power3":            # pdf ~ pT^-3 above pT_min  ->  pT = pT_min (1-u)^(-1/2), capped
        u = rng.random(n)
        return np.minimum(spec[1] * (1.0 - u) ** -0.5, spec[2])
    raise ValueError(kind)


def generate(rec: dict, geometry: Geometry | None = None, device: str = "cpu") -> TimeFrame:
    g = geometry or Geometry()
    seed = int(rec["seed"])
    n_az = g.n_azimuthal
    sect_w = 2.0 * math.pi / n_az

    # ---- collisions: multiplicity, time, vertex z
    rc = _rng(seed, _STREAM_COLLISIONS)
    if rec["kind"] in ("single_sector", "event"):
        n_trk = np.array([int(rec["n_tracks"])], dtype=np.int64)
        t_coll = np.zeros(1)
    else:
        nc = int(rec["n_collisions"])
        mk, mean = rec["mult"]
        if mk == "exp":
            n_trk = np.maximum(1, np.rint(rc.exponential(mean, nc))).astype(np.int64)
        elif mk == "poisson":
            n_trk = rc.poisson(mean, nc).astype(np.int64)
        else:
            raise ValueError(mk)
        t_coll = rc.uniform(0.0, float(rec["tf_us"]), nc)
    z_v = rc.normal(0.0, 1.0, n_trk.shape[0]) * float(rec["zv_sigma"])

    # ---- per-track parameters
    n_tot = int(n_trk.sum())
    rt = _rng(seed, _STREAM_TRACKS)
    coll_of = np.repeat(np.arange(n_trk.shape[0], dtype=np.int64), n_trk)
    if rec["kind"] == "single_sector":
        half = math.radians(g.half_sector_deg)
        phi0 = rt.uniform(0.0, 2.0 * half, n_tot)          # inside azimuthal sector 0
    else:
        phi0 = rt.uniform(0.0, 2.0 * math.pi, n_tot)
    charge = np.where(rt.random(n_tot) < 0.5, -1.0, 1.0)
    tanl = rt.uniform(-0.9, 0.9, n_tot)
    pt = _draw_pt(rt, rec["pt"], n_tot)
    qpt = charge / pt
    trk_zv = z_v[coll_of]
    trk_t = t_coll[coll_of]

    dev = torch.device(device)
    f64 = torch.float64
    row_x = torch.tensor(g.row_x(), dtype=f64, device=dev)                  # [R]
    ymax = row_x * g.tan_half_sector
    sigma = float(rec["sigma"])
    rho_probe = row_x * (0.5 * (1.0 + 1.0 / math.cos(math.radians(g.half_sector_deg))))
    cand_off = torch.tensor([-1, 0, 1], dtype=torch.int64, device=dev)      # sector candidates
    # big chunks on a GPU, cache-sized on the host; always a multiple of the smear-stream size
    chunk = _SMEAR_CHUNK * (16 if dev.type == "cuda" else 1)

    out_sector, out_row, out_y, out_z, out_tid, out_leg = [], [], [], [], [], []
    for c0 in range(0, n_tot, chunk):
        c1 = min(n_tot, c0 + chunk)
        m = c1 - c0
        # smear normals: one (y, z) pair per (track, row), drawn per fixed-size stream
        n1 = np.empty((m, g.n_rows)); n2 = np.empty((m, g.n_rows))
        for s0 in range(c0, c1, _SMEAR_CHUNK):
            s1 = min(c1, s0 + _SMEAR_CHUNK)
            rs = _rng(seed, _STREAM_SMEAR0 + s0 // _SMEAR_CHUNK)
            nn = rs.standard_normal((s1 - s0, g.n_rows, 2))
            n1[s0 - c0:s1 - c0] = nn[..., 0]
            n2[s0 - c0:s1 - c0] = nn[..., 1]
        T = lambda a: torch.as_tensor(a, dtype=f64).to(dev)  # noqa: E731
        p0 = T(phi0[c0:c1])[:, None, None]                 # [m,1,1]
        cv = (C_LIGHT_KB * g.bz_tesla) * T(qpt[c0:c1])[:, None, None]
        tl = T(tanl[c0:c1])[:, None, None]
        zv = T(trk_zv[c0:c1])[:, None, None]
        tc = T(trk_t[c0:c1])[:, None, None]
        X = row_x[None, :, None]                           # [1,R,1]
        # which azimuthal sector holds the helix point at radius ~x_r
        u_probe = 0.5 * cv * rho_probe[None, :, None]
        reach = u_probe.abs() < 1.0
        az = p0 + torch.asin(u_probe.clamp(-1.0, 1.0))
        a_guess = torch.floor(az / sect_w).to(torch.int64)
        a = torch.remainder(a_guess + cand_off[None, None, :], n_az)       # [m,R,3]
        alpha = (a.to(f64) + 0.5) * sect_w
        ploc = torch.remainder(p0 - alpha + math.pi, 2.0 * math.pi) - math.pi
        s_0 = torch.sin(ploc); c_0 = torch.cos(ploc)
        s_1 = s_0 + cv * X
        ok = reach & (c_0 > 0) & (s_1.abs() < 0.95)
        c_1 = torch.sqrt((1.0 - s_1 * s_1).clamp_min(0.0))
        y = X * (s_0 + s_1) / (c_0 + c_1)
        chord = torch.sqrt(X * X + y * y)
        u = 0.5 * cv * chord
        ser = torch.where(u.abs() > 1e-6, torch.asin(u.clamp(-1, 1)) / torch.where(u == 0, torch.ones_like(u), u),
                          1.0 + u * u / 6.0)
        z = zv + tl * (chord * ser)
        ok &= (y.abs() <= ymax[None, :, None]) & (z.abs() < g.drift_length)
        c_side = z < 0
        sec = a + c_side.to(torch.int64) * n_az
        ysm = y + sigma * T(n1)[:, :, None]
        zsm = z + sigma * T(n2)[:, :, None]
        zps = torch.where(c_side, zsm + g.v_drift * tc, zsm - g.v_drift * tc)
        rows = torch.arange(g.n_rows, device=dev)[None, :, None].expand_as(a)
        tids = (torch.arange(c0, c1, device=dev))[:, None, None].expand_as(a)
        out_sector.append(sec[ok].to(torch.uint8).cpu())
        out_row.append(rows[ok].to(torch.uint8).cpu())
        out_y.append(ysm[ok].to(torch.float32).cpu())
        out_z.append(zps[ok].to(torch.float32).cpu())
        out_tid.append(tids[ok].to(torch.int32).cpu())
        out_leg.append(torch.zeros(int(ok.sum()), dtype=torch.int8))
        if rec.get("loopers", False):
            # the returning branch: the circle through the origin meets the row line x = X of a sector frame a second
            # time, with cos(phi) < 0 (the particle comes back inwards), at y = (c_0 + c_1) / c, after the turning angle
            # 2 (pi - asin|u|) for the chord u = c chord / 2.  Its azimuth at radius rho is phi0 + sgn(c) pi - asin(u).
            sgn = torch.sign(cv)
            az_r = p0 + sgn * math.pi - torch.asin(u_probe.clamp(-1.0, 1.0))
            a_r = torch.remainder(torch.floor(az_r / sect_w).to(torch.int64) + cand_off[None, None, :], n_az)
            alpha_r = (a_r.to(f64) + 0.5) * sect_w
            ploc_r = torch.remainder(p0 - alpha_r + math.pi, 2.0 * math.pi) - math.pi
            s_0r = torch.sin(ploc_r); c_0r = torch.cos(ploc_r)
            s_1r = s_0r + cv * X
            ok_r = reach & (cv != 0) & (s_1r.abs() < 0.95)
            c_1r = torch.sqrt((1.0 - s_1r * s_1r).clamp_min(0.0))
            cvs = torch.where(cv == 0, torch.ones_like(cv), cv)
            y_r = (c_0r + c_1r) / cvs
            chord_r = torch.sqrt(X * X + y_r * y_r)
            u_r = (0.5 * cvs.abs() * chord_r).clamp(0.0, 1.0)
            arc_r = 2.0 * (math.pi - torch.asin(u_r)) / cvs.abs()
            z_r = zv + tl * arc_r
            ok_r &= (y_r.abs() <= ymax[None, :, None]) & (z_r.abs() < g.drift_length)
            c_side_r = z_r < 0
            sec_r = a_r + c_side_r.to(torch.int64) * n_az
            n1r = np.empty((m, g.n_rows)); n2r = np.empty((m, g.n_rows))
            for s0 in range(c0, c1, _SMEAR_CHUNK):
                s1 = min(c1, s0 + _SMEAR_CHUNK)
                nn = _rng(seed, _STREAM_SMEAR_RET0 + s0 // _SMEAR_CHUNK).standard_normal((s1 - s0, g.n_rows, 2))
                n1r[s0 - c0:s1 - c0] = nn[..., 0]
                n2r[s0 - c0:s1 - c0] = nn[..., 1]
            ysm_r = y_r + sigma * T(n1r)[:, :, None]
            zsm_r = z_r + sigma * T(n2r)[:, :, None]
            zps_r = torch.where(c_side_r, zsm_r + g.v_drift * tc, zsm_r - g.v_drift * tc)
            out_sector.append(sec_r[ok_r].to(torch.uint8).cpu())
            out_row.append(rows[ok_r].to(torch.uint8).cpu())
            out_y.append(ysm_r[ok_r].to(torch.float32).cpu())
            out_z.append(zps_r[ok_r].to(torch.float32).cpu())
            out_tid.append(tids[ok_r].to(torch.int32).cpu())
            out_leg.append(torch.ones(int(ok_r.sum()), dtype=torch.int8))

    cat = lambda lst, dt: (torch.cat(lst).numpy() if lst else np.empty(0, dt))  # noqa: E731
    sector = cat(out_sector, np.uint8); row = cat(out_row, np.uint8)
    yy = cat(out_y, np.float32); zz = cat(out_z, np.float32); tid = cat(out_tid, np.int32)
    leg = cat(out_leg, np.int8)

    # ---- noise clusters
    n_sig = sector.shape[0]
    n_noise = int(round(float(rec["noise"]) * n_sig))
    if n_noise > 0:
        rn = _rng(seed, _STREAM_NOISE)
        nsec = rn.integers(0, g.n_sectors, n_noise)
        nrow = rn.integers(0, g.n_rows, n_noise)
        ny = rn.uniform(-1.0, 1.0, n_noise) * (g.row_x()[nrow] * g.tan_half_sector)
        span = g.v_drift * float(rec["tf_us"])
        uz = rn.random(n_noise)
        a_side = nsec < n_az
        lo = np.where(a_side, -span, -g.drift_length)
        hi = np.where(a_side, g.drift_length, span)
        if span == 0.0:                                       # single event: physical half only
            lo = np.where(a_side, 0.0, -g.drift_length)
            hi = np.where(a_side, g.drift_length, 0.0)
        nz = lo + uz * (hi - lo)
        sector = np.concatenate([sector, nsec.astype(np.uint8)])
        row = np.concatenate([row, nrow.astype(np.uint8)])
        yy = np.concatenate([yy, ny.astype(np.float32)])
        zz = np.concatenate([zz, nz.astype(np.float32)])
        tid = np.concatenate([tid, np.full(n_noise, -1, np.int32)])
        leg = np.concatenate([leg, np.zeros(n_noise, np.int8)])

    x = g.row_x().astype(np.float32)[row]
    truth = dict(q_over_pt=qpt, tanl=tanl, phi0=phi0, z_v=trk_zv, t_coll=trk_t, collision=coll_of)
    return TimeFrame(sector=sector, row=row, x=x, y=yy, z=zz, track_id=tid, truth=truth, geometry=g,
                     tf_length_us=float(rec["tf_us"]), sigma=sigma, leg=leg)


# --------------------------------------------------------------- harness rules
def choose_cell(tf: TimeFrame, lo: float = 2.0, hi: float = 16.0, scale: float = 0.5) -> float:
    """Grid cell size handed to BOTH the oracle and the CUDA path (neither derives it):
    clamp(scale * sqrt(mean over non-empty (sector,row) of area / n_clusters), lo, hi), in double.
    The cell only changes how many clusters a window query has to look at, never which ones it accepts
    (DESIGN.md 3.1): scale = 0.5 (a quarter of a cluster per bin on average) was the fastest of a sweep on cfg5
    (profiles/r01b_summary.md)."""
    g = tf.geometry
    if tf.n == 0:
        return lo
    sr = tf.sector.astype(np.int64) * g.n_rows + tf.row
    cnt = np.bincount(sr, minlength=g.n_sectors * g.n_rows).astype(np.float64)
    zmin = np.full(g.n_sectors, np.inf); zmax = np.full(g.n_sectors, -np.inf)
    np.minimum.at(zmin, tf.sector, tf.z.astype(np.float64))
    np.maximum.at(zmax, tf.sector, tf.z.astype(np.float64))
    zspan = np.where(np.isfinite(zmin), zmax - zmin, 0.0)
    width = 2.0 * g.row_x() * g.tan_half_sector
    area = (zspan[:, None] * width[None, :]).reshape(-1)
    nz = cnt > 0
    per = area[nz] / cnt[nz]
    return float(min(hi, max(lo, scale * math.sqrt(float(per.mean())))))


def default_params(tf: TimeFrame, cell: float | None = None) -> dict:
    """Tracker parameters as a plain dict; both bindings marshal it."""
    g = tf.geometry
    c = choose_cell(tf) if cell is None else float(cell)
    return dict(
        n_sectors=g.n_sectors, n_rows=g.n_rows, row_x=g.row_x().astype(np.float32),
        tan_half_sector=np.float32(g.tan_half_sector), bz_tesla=np.float32(g.bz_tesla),
        err_y2=np.float32(0.01), err_z2=np.float32(0.01),
        cell_y=np.float32(c), cell_z=np.float32(c),
        link_ay=np.float32(1.2), link_az=np.float32(1.8), link_b=np.float32(0.6), link_T=np.float32(1.0),
        min_chain_len=4, max_gap=4, min_tracklet_hits=10, min_track_hits=10,
        pick_chi2_cut=np.float32(15.0), max_sinphi=np.float32(0.95), y_margin=np.float32(2.0),
        init_c_ss=np.float32(1.0), init_c_tt=np.float32(10.0), init_c_qq=np.float32(100.0),
    )


def to_native_time(tf: TimeFrame, time_unit_us: float = 0.2) -> tuple[TimeFrame, dict]:
    """The same time frame with the NATIVE time coordinate in place of the pseudo-z: a cluster is read
    out at t = t_coll + (L - |z_true|) / v_d after the start of the frame, i.e. t = (L -+ z') / v_d for the pseudo-z z'
    on the A / C side; here in units of `time_unit_us` (0.2 us = one TPC time bin), evaluated in double from the frame's
    own z', cast to fp32 last.  Returns (frame whose `z` holds t, the three tpc_params_t entries that describe it)."""
    g = tf.geometry
    side = np.where(tf.sector < g.n_azimuthal, 1.0, -1.0)
    t = (g.drift_length - side * tf.z.astype(np.float64)) / (g.v_drift * float(time_unit_us))
    out = TimeFrame(sector=tf.sector, row=tf.row, x=tf.x, y=tf.y, z=t.astype(np.float32), track_id=tf.track_id,
                    truth=tf.truth, geometry=g, tf_length_us=tf.tf_length_us, sigma=tf.sigma, name=tf.name + "+time", leg=tf.leg)
    return out, dict(z_is_time=1, cm_per_time_unit=np.float32(g.v_drift * float(time_unit_us)),
                     drift_length=np.float32(g.drift_length))


def to_native_pad(tf: TimeFrame, pitch_inner: float = 0.4375, pitch_outer: float = 0.625, n_inner: int = 63) -> tuple[TimeFrame, dict]:
    """The same time frame with the NATIVE pad coordinate in place of the sector-local y: row r has
    n_pads_r pads of width pitch_r (narrow pads on the first `n_inner` rows, wide ones outside - the ALICE read-out chambers
    have 4-6 mm pads), symmetric about the sector axis and enough of them to cover +-ymax_r; a cluster at y has the
    pad coordinate p = y / pitch_r + (n_pads_r - 1) / 2 (pad centres at the integers), evaluated in double from the
    frame's own y, cast to fp32 last.  Returns (frame whose `y` holds p, the three tpc_params_t entries that describe it)."""
    g = tf.geometry
    rx = g.row_x()
    pitch = np.where(np.arange(g.n_rows) < n_inner, float(pitch_inner), float(pitch_outer))
    n_pads = (2 * np.ceil(rx * g.tan_half_sector / pitch)).astype(np.int32)
    p = tf.y.astype(np.float64) / pitch[tf.row] + 0.5 * (n_pads[tf.row] - 1)
    out = TimeFrame(sector=tf.sector, row=tf.row, x=tf.x, y=p.astype(np.float32), z=tf.z, track_id=tf.track_id,
                    truth=tf.truth, geometry=g, tf_length_us=tf.tf_length_us, sigma=tf.sigma, name=tf.name + "+pad", leg=tf.leg)
    return out, dict(y_is_pad=1, n_pads=n_pads, pad_pitch=pitch.astype(np.float32))


def select_sectors(tf: TimeFrame, sectors) -> tuple[TimeFrame, np.ndarray]:
    """Sub-frame holding only the clusters of ``sectors`` (order kept) + their input indices."""
    keep = np.isin(tf.sector, np.asarray(list(sectors), dtype=np.uint8))
    idx = np.nonzero(keep)[0]
    sub = TimeFrame(sector=tf.sector[idx], row=tf.row[idx], x=tf.x[idx], y=tf.y[idx], z=tf.z[idx],
                    track_id=tf.track_id[idx], truth=tf.truth, geometry=tf.geometry,
                    tf_length_us=tf.tf_length_us, sigma=tf.sigma, name=tf.name + f"[sectors {list(sectors)}]",
                    leg=None if tf.leg is None else tf.leg[idx])
    return sub, idx
