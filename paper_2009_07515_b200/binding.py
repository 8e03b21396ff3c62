"""ctypes binding of libtpc_tracker.so - same names as include/tpc_tracker.h, argument marshalling only.

PyTorch supplies device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is NO CPU fallback: importing works without a GPU (so the ABI can be checked), but
creating a tracker needs a CUDA device and a missing library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

# ------------------------------------------------------------------ C structs (include/tpc_tracker.h)
c_f32p = C.POINTER(C.c_float)


class tpc_params_t(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.c_void_p),
        ("tan_half_sector", C.c_float), ("bz_tesla", C.c_float), ("err_y2", C.c_float), ("err_z2", C.c_float),
        ("cell_y", C.c_float), ("cell_z", C.c_float),
        ("link_ay", C.c_float), ("link_az", C.c_float), ("link_b", C.c_float), ("link_T", C.c_float),
        ("min_chain_len", C.c_int32), ("max_gap", C.c_int32), ("min_tracklet_hits", C.c_int32),
        ("min_track_hits", C.c_int32),
        ("pick_chi2_cut", C.c_float), ("max_sinphi", C.c_float), ("y_margin", C.c_float),
        ("init_c_ss", C.c_float), ("init_c_tt", C.c_float), ("init_c_qq", C.c_float),
        ("z_is_time", C.c_int32), ("cm_per_time_unit", C.c_float), ("drift_length", C.c_float),
        ("y_is_pad", C.c_int32), ("n_pads", C.c_void_p), ("pad_pitch", C.c_void_p),
    ]


# pseudo-z and y in cm unless asked otherwise
_PARAM_DEFAULTS = {"z_is_time": 0, "cm_per_time_unit": 0.0, "drift_length": 0.0, "y_is_pad": 0}


class tpc_clusters_t(C.Structure):
    _fields_ = [("n", C.c_int64), ("sector", C.c_void_p), ("row", C.c_void_p), ("x", C.c_void_p), ("y", C.c_void_p),
                ("z", C.c_void_p)]


_TRACK_FIELDS = ["n_tracks", "status", "sector", "first_row", "last_row", "n_clusters", "par", "cov", "x_ref", "z_ref",
                 "chi2", "ndf", "trk_cl_start", "trk_cl_idx", "cluster_track", "z_beam"]


class tpc_tracks_t(C.Structure):
    _fields_ = [("max_tracks", C.c_int64), ("max_track_clusters", C.c_int64)] + [(f, C.c_void_p) for f in _TRACK_FIELDS]


class tpc_fit_t(C.Structure):
    _fields_ = [("max_tracks", C.c_int64)] + [(f, C.c_void_p) for f in ("par", "cov", "x_ref", "z_ref", "chi2", "ndf", "n_fit",
                                                                       "trk_cl_start", "res_y", "res_z", "qres_y", "qres_z")] + \
               [("res_step_y", C.c_float), ("res_step_z", C.c_float)]


class tpc_merge_cuts_t(C.Structure):
    _fields_ = [("max_rows", C.c_int32), ("back_rows", C.c_int32), ("edge", C.c_float), ("dz_win", C.c_float),
                ("chi2_cut", C.c_float), ("road_z0", C.c_float), ("road_z1", C.c_float)]


_MERGED_FIELDS = ["n_merged", "merged_of_track", "seg_start", "seg_idx", "par", "cov", "x_ref", "z_ref", "chi2", "ndf", "n_fit",
                  "sector", "n_clusters"]


class tpc_merged_t(C.Structure):
    _fields_ = [("max_tracks", C.c_int64)] + [(f, C.c_void_p) for f in _MERGED_FIELDS]


class tpc_apex_cuts_t(C.Structure):
    _fields_ = [("max_k", C.c_int32), ("min_s", C.c_float), ("dz_win", C.c_float), ("tol_c", C.c_float), ("tol_z", C.c_float),
                ("tol_t", C.c_float), ("cut", C.c_float)]


class tpc_apex_t(C.Structure):
    _fields_ = [("max_tracks", C.c_int64), ("apex_partner", C.c_void_p), ("apex_leg", C.c_void_p)]


class tpc_removal_cuts_t(C.Structure):
    _fields_ = [("min_pt", C.c_float), ("max_incl", C.c_float), ("road_y", C.c_float), ("road_z", C.c_float)]


REMOVAL_CUTS = dict(min_pt=0.05, max_incl=0.85, road_y=1.0, road_z=1.0)
APEX_CUTS = dict(max_k=4, min_s=0.6, dz_win=150.0, tol_c=0.1, tol_z=4.0, tol_t=0.1, cut=3.0)
MERGE_CUTS = dict(max_rows=30, back_rows=1, edge=6.0, dz_win=50.0, chi2_cut=100.0, road_z0=2.0, road_z1=0.3)


class tpc_counters_t(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("n_bins", C.c_int64), ("n_seeds", C.c_int64), ("n_tracklets", C.c_int64),
                ("n_tracks", C.c_int64), ("n_track_clusters", C.c_int64), ("n_linked", C.c_int64),
                ("kf_steps", C.c_int64), ("n_hits", C.c_int64), ("status", C.c_int32), ("s1_global_buckets", C.c_int32)]


class tpc_stage_view_t(C.Structure):
    _fields_ = [("ptr", C.c_void_p), ("n", C.c_int64), ("elem_bytes", C.c_int32), ("is_float", C.c_int32)]


VIEWS = {name: i for i, name in enumerate([
    "perm", "yz", "srow", "bin_start", "row_start", "bin_base", "zmin", "zmax", "nz",
    "link_up_raw", "link_dn_raw", "link_up", "link_dn", "seed_head", "seed_len",
    "t_hit", "t_first_row", "t_last_row", "t_n_hits", "t_par", "t_cov", "t_chi2", "t_zref",
    "tracklet_of_seed", "k_owned",
    "fit_row", "up_par", "up_cov", "up_x", "up_zref", "up_row", "up_n",
    "mrg_best_b", "mrg_best_a", "mrg_chi_b", "mrg_next", "mrg_prev", "mrg_dir", "apex_best", "apex_score"])}

PROTECT_STATIC_MAX_CLUSTERS = 4194304   # TPC_PROTECT_STATIC_MAX_CLUSTERS of include/tpc_tracker.h

STATUS_BITS = {1: "BAD_CLUSTER", 2: "BINS_OVERFLOW", 4: "SEEDS_OVERFLOW", 8: "TRACKS_OVERFLOW", 16: "CHAIN_CYCLE"}

EXPORTS = [
    "tpc_tracker_workspace_bytes", "tpc_tracker_create", "tpc_track_timeframe", "tpc_track_timeframe_host",
    "tpc_track_timeframe_host_begin", "tpc_track_timeframe_host_end", "tpc_tracker_refit", "tpc_tracker_merge", "tpc_tracker_apex", "tpc_tracker_removable", "tpc_tracker_protect", "tpc_tracker_protect_static",
    "tpc_tracker_counters", "tpc_tracker_enable_graph", "tpc_tracker_enable_stage_timing", "tpc_tracker_stage_ms", "tpc_tracker_stage_view",
    "tpc_tracker_launches_per_call", "tpc_tracker_destroy", "tpc_error_string",
]

_lib = None


def library_path() -> str:
    return _build.LIB


def load_library(build: bool = True) -> C.CDLL:
    """Loads (building first if stale and nvcc is there) libtpc_tracker.so.  Raises if unavailable."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build:
        try:
            path = _build.build()
        except Exception as e:  # nvcc missing on the box: use the shipped .so if it is there
            if not os.path.exists(path):
                raise RuntimeError(f"libtpc_tracker.so is missing and could not be built: {e}") from e
    if not os.path.exists(path):
        raise RuntimeError("libtpc_tracker.so is missing: run `python -m paper_2009_07515_b200.build` (no CPU fallback)")
    lib = C.CDLL(path)
    P = C.POINTER
    lib.tpc_tracker_workspace_bytes.restype = C.c_size_t
    lib.tpc_tracker_workspace_bytes.argtypes = [P(tpc_params_t), C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.c_int32]
    lib.tpc_tracker_create.restype = C.c_int
    lib.tpc_tracker_create.argtypes = [P(tpc_params_t), C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.c_int32,
                                       C.c_void_p, C.c_size_t, P(C.c_void_p)]
    for name in ("tpc_track_timeframe", "tpc_track_timeframe_host"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, P(tpc_clusters_t), P(tpc_tracks_t), C.c_void_p]
    lib.tpc_track_timeframe_host_begin.restype = C.c_int
    lib.tpc_track_timeframe_host_begin.argtypes = [C.c_void_p, P(tpc_clusters_t), C.c_int32]
    lib.tpc_track_timeframe_host_end.restype = C.c_int
    lib.tpc_track_timeframe_host_end.argtypes = [C.c_void_p, P(tpc_tracks_t), C.c_int32]
    lib.tpc_tracker_refit.restype = C.c_int
    lib.tpc_tracker_refit.argtypes = [C.c_void_p, P(tpc_fit_t), C.c_void_p]
    lib.tpc_tracker_merge.restype = C.c_int
    lib.tpc_tracker_merge.argtypes = [C.c_void_p, P(tpc_fit_t), P(tpc_merge_cuts_t), P(tpc_merged_t), C.c_void_p]
    lib.tpc_tracker_apex.restype = C.c_int
    lib.tpc_tracker_apex.argtypes = [C.c_void_p, P(tpc_merged_t), P(tpc_apex_cuts_t), P(tpc_apex_t), C.c_void_p]
    lib.tpc_tracker_removable.restype = C.c_int
    lib.tpc_tracker_removable.argtypes = [C.c_void_p, C.c_void_p, P(tpc_fit_t), P(tpc_merged_t), P(tpc_apex_t), P(tpc_removal_cuts_t),
                                          C.c_void_p, C.c_void_p, C.c_void_p]
    lib.tpc_tracker_protect.restype = C.c_int
    lib.tpc_tracker_protect.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
    lib.tpc_tracker_protect_static.restype = C.c_int
    lib.tpc_tracker_protect_static.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
    lib.tpc_tracker_counters.restype = C.c_int
    lib.tpc_tracker_counters.argtypes = [C.c_void_p, P(tpc_counters_t)]
    lib.tpc_tracker_enable_graph.restype = C.c_int
    lib.tpc_tracker_enable_graph.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_tracker_enable_stage_timing.restype = C.c_int
    lib.tpc_tracker_enable_stage_timing.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_tracker_stage_ms.restype = C.c_int
    lib.tpc_tracker_stage_ms.argtypes = [C.c_void_p, P(C.c_float)]
    lib.tpc_tracker_stage_view.restype = C.c_int
    lib.tpc_tracker_stage_view.argtypes = [C.c_void_p, C.c_int32, P(tpc_stage_view_t)]
    lib.tpc_tracker_launches_per_call.restype = C.c_int
    lib.tpc_tracker_launches_per_call.argtypes = [C.c_void_p]
    lib.tpc_tracker_destroy.restype = C.c_int
    lib.tpc_tracker_destroy.argtypes = [C.c_void_p]
    lib.tpc_error_string.restype = C.c_char_p
    lib.tpc_error_string.argtypes = [C.c_int]
    _lib = lib
    return lib


def _check(lib, rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"{what}: {lib.tpc_error_string(rc).decode()} ({rc})")


def pack_params(params: dict):
    """dict (tpc_synth.default_params) -> (tpc_params_t, keep-alive host tables: row_x and, with y_is_pad, the pad plane)."""
    rx = np.ascontiguousarray(params["row_x"], dtype=np.float32)
    keep = [rx]
    p = tpc_params_t()
    for name, _ in tpc_params_t._fields_:
        if name == "row_x":
            p.row_x = rx.ctypes.data
        elif name in ("n_pads", "pad_pitch"):
            if params.get("y_is_pad", 0):
                tab = np.ascontiguousarray(params[name], dtype=np.int32 if name == "n_pads" else np.float32)
                assert tab.shape[0] == params["n_rows"]
                keep.append(tab)
                setattr(p, name, tab.ctypes.data)
        else:
            v = params[name] if name in params else _PARAM_DEFAULTS[name]
            setattr(p, name, v.item() if hasattr(v, "item") else v)
    return p, keep


class Tracks:
    """Output buffers (torch tensors on `device`, or pinned host tensors) laid out as tpc_tracks_t wants."""

    def __init__(self, n_clusters: int, max_tracks: int, max_track_clusters: int, device, with_cluster_track: bool = True):
        host = torch.device(device).type == "cpu"
        assert host or with_cluster_track, "the device path always writes cluster_track"
        self.with_cluster_track = bool(with_cluster_track)
        kw = dict(device=device, pin_memory=True) if host else dict(device=device)
        i32 = lambda *s: torch.empty(*s, dtype=torch.int32, **kw)   # noqa: E731
        f32 = lambda *s: torch.empty(*s, dtype=torch.float32, **kw)  # noqa: E731
        self.max_tracks, self.max_track_clusters = int(max_tracks), int(max_track_clusters)
        self.n_tracks = i32(1); self.status = i32(1)
        self.sector = i32(max_tracks); self.first_row = i32(max_tracks); self.last_row = i32(max_tracks)
        self.n_clusters = i32(max_tracks)
        self.par = f32(5, max_tracks); self.cov = f32(15, max_tracks)
        self.x_ref = f32(max_tracks); self.z_ref = f32(max_tracks); self.chi2 = f32(max_tracks); self.ndf = i32(max_tracks)
        self.z_beam = f32(max_tracks)
        self.trk_cl_start = i32(max_tracks + 1); self.trk_cl_idx = i32(max_track_clusters)
        self.cluster_track = i32(max(1, n_clusters))
        self.n_in = int(n_clusters)

    def struct(self) -> tpc_tracks_t:
        s = tpc_tracks_t()
        s.max_tracks = self.max_tracks; s.max_track_clusters = self.max_track_clusters
        for f in _TRACK_FIELDS:
            setattr(s, f, getattr(self, f).data_ptr())
        if not self.with_cluster_track:
            s.cluster_track = None              # host paths: do not copy the per-cluster assignment back
        return s

    def bytes_out(self) -> int:
        """Bytes a host run copies back for the tracks found (d2h_bytes_per_step)."""
        T = int(self.n_tracks.item())
        ntc = int(self.trk_cl_start[T].item()) if T else 0
        return 8 + T * 4 * (9 + 5 + 15) + (T + 1) * 4 + ntc * 4 + (self.n_in * 4 if self.with_cluster_track else 0)

    def numpy(self) -> dict:
        """Host copies trimmed to the tracks found."""
        T = int(self.n_tracks.item())
        g = lambda t: t.detach().cpu().numpy()  # noqa: E731
        st = g(self.trk_cl_start)[: T + 1].copy()
        if T == 0:
            st = np.zeros(1, np.int32)
        return dict(
            n_tracks=T, status=int(self.status.item()),
            sector=g(self.sector)[:T].copy(), first_row=g(self.first_row)[:T].copy(), last_row=g(self.last_row)[:T].copy(),
            n_clusters=g(self.n_clusters)[:T].copy(), par=g(self.par)[:, :T].T.copy(), cov=g(self.cov)[:, :T].T.copy(),
            x_ref=g(self.x_ref)[:T].copy(), z_ref=g(self.z_ref)[:T].copy(), chi2=g(self.chi2)[:T].copy(),
            z_beam=g(self.z_beam)[:T].copy(),
            ndf=g(self.ndf)[:T].copy(), trk_cl_start=st, trk_cl_idx=g(self.trk_cl_idx)[: int(st[-1])].copy(),
            cluster_track=g(self.cluster_track)[: self.n_in].copy())


class Tracker:
    """tpc_tracker_create / tpc_track_timeframe / tpc_tracker_destroy with torch-owned memory."""

    def __init__(self, params: dict, max_clusters: int, max_bins: int, max_seeds: int, max_tracks: int,
                 max_track_clusters: int, host_io: int = 0, device="cuda:0", guard_bytes: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("tpc tracker needs a CUDA device: there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        self._p, self._rx = pack_params(params)
        self.params = params
        caps = [int(max_clusters), int(max_bins), int(max_seeds), int(max_tracks), int(max_track_clusters)]
        self.caps = caps
        nbytes = self.lib.tpc_tracker_workspace_bytes(C.byref(self._p), *caps, int(host_io))
        if nbytes == 0:
            raise ValueError("tpc_tracker_workspace_bytes rejected the parameters / capacities")
        self.workspace_bytes = int(nbytes)
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): canary bytes on both sides of the arena, see guards_intact()
            g = (int(guard_bytes) + 255) // 256 * 256
            self._arena = torch.full((nbytes + 2 * g,), 0xA5, dtype=torch.uint8, device=self.device)
            self._guard = g
            self.workspace = self._arena[g: g + nbytes]
            h = C.c_void_p()
            _check(self.lib, self.lib.tpc_tracker_create(C.byref(self._p), *caps, int(host_io), self.workspace.data_ptr(),
                                                         nbytes, C.byref(h)), "tpc_tracker_create")
        self._h = h

    def guards_intact(self) -> bool:
        """True iff no kernel wrote outside the workspace arena (only meaningful with guard_bytes > 0)."""
        torch.cuda.synchronize(self.device)
        g = self._guard
        return bool((self._arena[:g] == 0xA5).all().item() and (self._arena[self._arena.numel() - g:] == 0xA5).all().item())

    # -- lifetime
    def destroy(self):
        if getattr(self, "_h", None):
            self.lib.tpc_tracker_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- calls
    @staticmethod
    def _clusters(sector, row, y, z) -> tpc_clusters_t:
        c = tpc_clusters_t()
        c.n = int(sector.shape[0])
        c.sector = sector.data_ptr(); c.row = row.data_ptr(); c.x = None; c.y = y.data_ptr(); c.z = z.data_ptr()
        return c

    def new_tracks(self, n_clusters: int, host: bool = False, with_cluster_track: bool = True) -> Tracks:
        return Tracks(n_clusters, self.caps[3], self.caps[4], "cpu" if host else self.device, with_cluster_track)

    def track_timeframe(self, sector, row, y, z, out: Tracks, stream=None):
        """Device tensors in, device tensors out; enqueues on `stream` (default: torch's current stream)."""
        for t in (sector, row, y, z):
            assert t.is_cuda and t.is_contiguous()
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        c = self._clusters(sector, row, y, z)
        s = out.struct()
        _check(self.lib, self.lib.tpc_track_timeframe(self._h, C.byref(c), C.byref(s), C.c_void_p(st.cuda_stream)),
               "tpc_track_timeframe")

    def track_timeframe_host(self, sector, row, y, z, out: Tracks, stream=None):
        """Pinned host tensors in/out; H2D, S1..S5 and D2H inside the call; synchronises."""
        for t in (sector, row, y, z):
            assert (not t.is_cuda) and t.is_contiguous()
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        c = self._clusters(sector, row, y, z)
        s = out.struct()
        _check(self.lib, self.lib.tpc_track_timeframe_host(self._h, C.byref(c), C.byref(s), C.c_void_p(st.cuda_stream)),
               "tpc_track_timeframe_host")

    def track_timeframe_host_begin(self, sector, row, y, z, slot: int):
        """Pipelined host path (host_io=2): enqueue H2D + S1..S5 of one frame, do not wait."""
        for t in (sector, row, y, z):
            assert (not t.is_cuda) and t.is_contiguous()
        c = self._clusters(sector, row, y, z)
        _check(self.lib, self.lib.tpc_track_timeframe_host_begin(self._h, C.byref(c), int(slot)), "tpc_track_timeframe_host_begin")

    def track_timeframe_host_end(self, out: Tracks, slot: int):
        """Wait for the frame begun on `slot` and copy its tracks into the (pinned host) buffers of `out`."""
        s = out.struct()
        _check(self.lib, self.lib.tpc_track_timeframe_host_end(self._h, C.byref(s), int(slot)), "tpc_track_timeframe_host_end")

    def new_fit(self, residuals: bool = False, steps: "tuple[float, float] | None" = None) -> dict:
        """Device buffers for tpc_tracker_refit (layouts as in tpc_fit_t); with `residuals` also res_y / res_z; with
        `steps` = (step_y, step_z) in cm also the 16-bit residual codes qres_y / qres_z (implies the residuals)."""
        mt, dev = self.caps[3], self.device
        f32 = lambda *s: torch.empty(*s, dtype=torch.float32, device=dev)   # noqa: E731
        i32 = lambda *s: torch.empty(*s, dtype=torch.int32, device=dev)     # noqa: E731
        d = dict(par=f32(5, mt), cov=f32(15, mt), x_ref=f32(mt), z_ref=f32(mt), chi2=f32(mt), ndf=i32(mt), n_fit=i32(mt))
        if residuals or steps is not None:
            d.update(res_y=f32(self.caps[4]), res_z=f32(self.caps[4]))
        if steps is not None:
            d.update(qres_y=torch.empty(self.caps[4], dtype=torch.int16, device=dev),
                     qres_z=torch.empty(self.caps[4], dtype=torch.int16, device=dev),
                     res_step_y=float(steps[0]), res_step_z=float(steps[1]))
        return d

    def refit_into(self, fit: dict, stream=None, out: "Tracks | None" = None):
        """Enqueues tpc_tracker_refit for the tracks of the last track_timeframe call (does not synchronise).  Residuals
        (fit has res_y / res_z) need that call's outputs `out` for the CSR offsets."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        f = tpc_fit_t()
        f.max_tracks = self.caps[3]
        for k, v in fit.items():
            setattr(f, k, v.data_ptr() if torch.is_tensor(v) else v)
        if "res_y" in fit:
            f.trk_cl_start = out.trk_cl_start.data_ptr()
        _check(self.lib, self.lib.tpc_tracker_refit(self._h, C.byref(f), C.c_void_p(st.cuda_stream)), "tpc_tracker_refit")

    def refit(self, n_tracks: int, stream=None, tracks: "Tracks | None" = None, steps=None) -> dict:
        """Convenience: refit + host copies trimmed to n_tracks (with `tracks`, the call's outputs, also the residuals;
        with `steps` = (step_y, step_z) also their 16-bit codes)."""
        buf = self.new_fit(residuals=tracks is not None, steps=steps if tracks is not None else None)
        self.refit_into(buf, stream, out=tracks)
        torch.cuda.synchronize(self.device)
        T = int(n_tracks)
        out = {k: v.cpu().numpy() for k, v in buf.items() if torch.is_tensor(v)}
        extra = {}
        if tracks is not None:
            ntc = int(tracks.trk_cl_start[T].item()) if T else 0
            extra = dict(res_y=out["res_y"][:ntc].copy(), res_z=out["res_z"][:ntc].copy())
            if steps is not None:
                extra.update(qres_y=out["qres_y"][:ntc].copy(), qres_z=out["qres_z"][:ntc].copy())
        return dict(**extra, par=out["par"][:, :T].T.copy(), cov=out["cov"][:, :T].T.copy(), x_ref=out["x_ref"][:T].copy(),
                    z_ref=out["z_ref"][:T].copy(), chi2=out["chi2"][:T].copy(), ndf=out["ndf"][:T].copy(),
                    n_fit=out["n_fit"][:T].copy())

    def new_merged(self, fill: int = 0) -> dict:
        """Device buffers for tpc_tracker_merge (layouts as in tpc_merged_t); the integer ones pre-filled with `fill`
        (tests pass a poison value to see that every entry the header promises is really written)."""
        mt, dev = self.caps[3], self.device
        f32 = lambda *s: torch.empty(*s, dtype=torch.float32, device=dev)   # noqa: E731
        i32 = lambda *s: torch.full(s, int(fill), dtype=torch.int32, device=dev)     # noqa: E731
        return dict(n_merged=i32(1), merged_of_track=i32(mt), seg_start=i32(mt + 1), seg_idx=i32(mt), par=f32(5, mt),
                    cov=f32(15, mt), x_ref=f32(mt), z_ref=f32(mt), chi2=f32(mt), ndf=i32(mt), n_fit=i32(mt), sector=i32(mt),
                    n_clusters=i32(mt))

    def merge_into(self, fit: dict, merged: dict, cuts: dict | None = None, stream=None):
        """Enqueues tpc_tracker_merge for the tracks of the last track_timeframe call, whose refit (refit_into) is `fit`
        (does not synchronise)."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        f = tpc_fit_t()
        f.max_tracks = self.caps[3]
        for k in ("par", "cov", "x_ref", "z_ref", "chi2", "ndf", "n_fit"):
            setattr(f, k, fit[k].data_ptr())
        kw = dict(MERGE_CUTS); kw.update(cuts or {})
        c = tpc_merge_cuts_t(int(kw["max_rows"]), int(kw["back_rows"]), float(kw["edge"]), float(kw["dz_win"]), float(kw["chi2_cut"]),
                             float(kw["road_z0"]), float(kw["road_z1"]))
        m = tpc_merged_t()
        m.max_tracks = self.caps[3]
        for k in _MERGED_FIELDS:
            setattr(m, k, merged[k].data_ptr())
        _check(self.lib, self.lib.tpc_tracker_merge(self._h, C.byref(f), C.byref(c), C.byref(m), C.c_void_p(st.cuda_stream)),
               "tpc_tracker_merge")

    def apex_into(self, merged: dict, out: dict, cuts: dict | None = None, stream=None):
        """Enqueues tpc_tracker_apex for the merged tracks of the last merge_into call (does not synchronise);
        `out` = dict(apex_partner=int32[max_tracks], apex_leg=int32[max_tracks]) on the device."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        m = tpc_merged_t()
        m.max_tracks = self.caps[3]
        for k in _MERGED_FIELDS:
            setattr(m, k, merged[k].data_ptr())
        kw = dict(APEX_CUTS); kw.update(cuts or {})
        c = tpc_apex_cuts_t(int(kw["max_k"]), float(kw["min_s"]), float(kw["dz_win"]), float(kw["tol_c"]), float(kw["tol_z"]),
                            float(kw["tol_t"]), float(kw["cut"]))
        o = tpc_apex_t()
        o.max_tracks = self.caps[3]
        o.apex_partner = out["apex_partner"].data_ptr(); o.apex_leg = out["apex_leg"].data_ptr()
        _check(self.lib, self.lib.tpc_tracker_apex(self._h, C.byref(m), C.byref(c), C.byref(o), C.c_void_p(st.cuda_stream)),
               "tpc_tracker_apex")

    def removable(self, out: "Tracks", cuts: dict | None = None, merge_cuts: dict | None = None, apex_cuts: dict | None = None,
                  fill: int = 0):
        """Convenience: refit + merge + apex + tpc_tracker_removable for the last track_timeframe call (outputs `out`);
        returns (cls, remove) as uint8 device tensors [n].  `fill`: see new_merged."""
        fit = self.new_fit(); mg = self.new_merged(fill); ax = self.new_apex()
        self.refit_into(fit); self.merge_into(fit, mg, merge_cuts); self.apex_into(mg, ax, apex_cuts)
        n = max(1, out.n_in)
        cls = torch.zeros(n, dtype=torch.uint8, device=self.device); rem = torch.zeros(n, dtype=torch.uint8, device=self.device)
        self.removable_into(out, fit, mg, ax, cls, rem, cuts)
        torch.cuda.synchronize(self.device)
        return cls[: out.n_in], rem[: out.n_in]

    def removable_into(self, out: "Tracks", fit: dict, mg: dict, ax: dict, cls, rem, cuts: dict | None = None, stream=None):
        """Enqueues tpc_tracker_removable alone (does not synchronise, allocates nothing): `fit`, `mg`, `ax` are the buffers
        the refit_into / merge_into / apex_into calls of this frame wrote; cls / rem uint8 device tensors [n]."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        f = tpc_fit_t(); f.max_tracks = self.caps[3]
        for k in ("par", "cov", "x_ref", "z_ref", "chi2", "ndf", "n_fit"):
            setattr(f, k, fit[k].data_ptr())
        m = tpc_merged_t(); m.max_tracks = self.caps[3]
        for k in _MERGED_FIELDS:
            setattr(m, k, mg[k].data_ptr())
        a = tpc_apex_t(); a.max_tracks = self.caps[3]
        a.apex_partner = ax["apex_partner"].data_ptr(); a.apex_leg = ax["apex_leg"].data_ptr()
        kw = dict(REMOVAL_CUTS); kw.update(cuts or {})
        c = tpc_removal_cuts_t(float(kw["min_pt"]), float(kw["max_incl"]), float(kw["road_y"]), float(kw["road_z"]))
        _check(self.lib, self.lib.tpc_tracker_removable(self._h, out.cluster_track.data_ptr(), C.byref(f), C.byref(m), C.byref(a),
                                                         C.byref(c), cls.data_ptr(), rem.data_ptr(), C.c_void_p(st.cuda_stream)),
               "tpc_tracker_removable")

    def new_apex(self) -> dict:
        mt, dev = self.caps[3], self.device
        return dict(apex_partner=torch.zeros(mt, dtype=torch.int32, device=dev), apex_leg=torch.zeros(mt, dtype=torch.int32, device=dev))

    def merge(self, n_tracks: int, cuts: dict | None = None, apex: dict | bool | None = None, fill: int = 0) -> dict:
        """Convenience: refit + merge (+ apex links when `apex` is True or a dict of cuts) + host copies trimmed to the
        tracks / merged tracks found.  `fill`: see new_merged."""
        fit = self.new_fit(); mg = self.new_merged(fill)
        self.refit_into(fit)
        self.merge_into(fit, mg, cuts)
        extra = {}
        if apex:
            ax = self.new_apex()
            self.apex_into(mg, ax, apex if isinstance(apex, dict) else None)
        torch.cuda.synchronize(self.device)
        T = int(n_tracks); M = int(mg["n_merged"].item())
        if apex:
            extra = dict(apex_partner=ax["apex_partner"].cpu().numpy()[:M].copy(), apex_leg=ax["apex_leg"].cpu().numpy()[:M].copy())
        h = {k: v.cpu().numpy() for k, v in mg.items()}
        return dict(**extra, n_merged=M, merged_of_track=h["merged_of_track"][:T].copy(), seg_start=h["seg_start"][:M + 1].copy(),
                    seg_idx=h["seg_idx"][:T].copy(), par=h["par"][:, :M].T.copy(), cov=h["cov"][:, :M].T.copy(),
                    **{k: h[k][:M].copy() for k in ("x_ref", "z_ref", "chi2", "ndf", "n_fit", "sector", "n_clusters")})

    def protect(self, out: Tracks, road_y: float, road_z: float, keep=None, stream=None):
        """tpc_tracker_protect for the last track_timeframe call (whose outputs are `out`); returns the uint8 device
        tensor keep[n] (enqueued, not synchronised)."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        if keep is None:
            keep = torch.empty(max(1, out.n_in), dtype=torch.uint8, device=self.device)
        _check(self.lib, self.lib.tpc_tracker_protect(self._h, out.cluster_track.data_ptr(), float(road_y), float(road_z),
                                                      keep.data_ptr(), C.c_void_p(st.cuda_stream)), "tpc_tracker_protect")
        return keep

    def protect_static(self, out: Tracks, road_y: float, road_z: float, keep, stream=None):
        """tpc_tracker_protect_static: the flags of `protect` for a frame of at most PROTECT_STATIC_MAX_CLUSTERS clusters,
        computed without any device allocation - the per-cluster scratch is an array inside the library, not workspace or
        cudaMalloc memory (for callers whose framework owns all GPU memory, or that may not stall the device with an
        allocation).  `keep` (uint8 device tensor [n]) must be passed in: this wrapper does not allocate either.  One
        array per device, shared by everybody: calls that could overlap on the GPU must be ordered by the caller.  The
        first call on a device looks the array up; make it before any stream capture.  Raises on larger frames."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        assert keep.is_cuda and keep.dtype == torch.uint8 and keep.numel() >= out.n_in
        _check(self.lib, self.lib.tpc_tracker_protect_static(self._h, out.cluster_track.data_ptr(), float(road_y), float(road_z),
                                                             keep.data_ptr(), C.c_void_p(st.cuda_stream)), "tpc_tracker_protect_static")
        return keep

    def counters(self) -> dict:
        k = tpc_counters_t()
        _check(self.lib, self.lib.tpc_tracker_counters(self._h, C.byref(k)), "tpc_tracker_counters")
        return {f: getattr(k, f) for f, _ in tpc_counters_t._fields_}

    def enable_stage_timing(self, on: bool = True):
        _check(self.lib, self.lib.tpc_tracker_enable_stage_timing(self._h, int(on)), "tpc_tracker_enable_stage_timing")

    def enable_graph(self, on: bool = True):
        """Replay a cached CUDA graph of S1..S5 while the arguments of track_timeframe stay the same (non-default stream)."""
        _check(self.lib, self.lib.tpc_tracker_enable_graph(self._h, int(on)), "tpc_tracker_enable_graph")

    def stage_ms(self) -> list[float]:
        ms = (C.c_float * 5)()
        _check(self.lib, self.lib.tpc_tracker_stage_ms(self._h, ms), "tpc_tracker_stage_ms")
        return [float(v) for v in ms]

    def launches_per_call(self) -> int:
        return int(self.lib.tpc_tracker_launches_per_call(self._h))

    def stage_view(self, name: str) -> np.ndarray:
        """Host copy of one workspace array (debug / parity tests)."""
        v = tpc_stage_view_t()
        _check(self.lib, self.lib.tpc_tracker_stage_view(self._h, VIEWS[name], C.byref(v)), "tpc_tracker_stage_view")
        dt = {(4, 0): np.int32, (4, 1): np.float32, (2, 0): np.uint16, (8, 0): np.uint64}[(v.elem_bytes, v.is_float)]
        out = np.empty(v.n, dtype=dt)
        if v.n:
            # plain byte copy device -> host of a workspace slice
            off = v.ptr - self.workspace.data_ptr()
            src = self.workspace[off: off + v.n * v.elem_bytes]
            out.view(np.uint8)[:] = src.cpu().numpy()
        return out


def max_bins_bound(sector, z, params: dict) -> int:
    """Upper bound of N_b for sizing the workspace (host-side helper, numpy float64, +2 rows of slack per
    sector; the tracker computes the exact grids itself on the device)."""
    sector = np.asarray(sector); z = np.asarray(z, dtype=np.float64)
    S = int(params["n_sectors"])
    if params.get("z_is_time", 0):              # native time input: the span of the pseudo-z the device will compute
        zc = float(params["drift_length"]) - z * float(params["cm_per_time_unit"])
        z = np.where(sector < S // 2, zc, -zc)
    if sector.size == 0:
        return 1
    ok = np.isfinite(z) & (sector < S)          # non-finite / out-of-range clusters are rejected on the device (status bit)
    sector, z = sector[ok], z[ok]
    zmin = np.full(S, np.inf); zmax = np.full(S, -np.inf)
    np.minimum.at(zmin, sector, z); np.maximum.at(zmax, sector, z)
    span = np.where(np.isfinite(zmin), zmax - zmin, 0.0)
    nz = np.where(np.isfinite(zmin), np.floor(span / float(params["cell_z"])) + 3, 0)
    rx = np.asarray(params["row_x"], dtype=np.float64)
    ny = np.floor(2.0 * rx * float(params["tan_half_sector"]) / float(params["cell_y"])) + 2
    return int(min(nz.sum() * ny.sum(), float(2**31 - 3))) + 1   # the device raises BINS_OVERFLOW beyond int32


def suggest_capacities(n_clusters: int, params: dict) -> dict:
    """Loose capacities for a workload of n clusters (host-side sizing helper, no tracker arithmetic):
    seeds <= n / min_chain_len, tracks <= n / min_track_hits, attached clusters <= n."""
    n = max(1, int(n_clusters))
    return dict(max_clusters=n, max_seeds=max(1024, n // max(2, int(params["min_chain_len"])) + 1),
                max_tracks=max(1024, n // max(1, int(params["min_track_hits"])) + 1), max_track_clusters=n)
