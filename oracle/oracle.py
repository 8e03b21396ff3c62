"""ctypes wrapper around oracle/liboracle.so (argument marshalling only).

TEST INFRASTRUCTURE: see the header of tpc_oracle.cpp for who may import this.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_MAX_ROWS = 256


class _Params(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32),
        ("row_x", C.c_float * _MAX_ROWS),
        ("tan_half_sector", C.c_float), ("bz_tesla", C.c_float), ("err_y2", C.c_float), ("err_z2", C.c_float),
        ("cell_y", C.c_float), ("cell_z", C.c_float),
        ("link_ay", C.c_float), ("link_az", C.c_float), ("link_b", C.c_float), ("link_T", C.c_float),
        ("min_chain_len", C.c_int32), ("max_gap", C.c_int32), ("min_tracklet_hits", C.c_int32),
        ("min_track_hits", C.c_int32),
        ("pick_chi2_cut", C.c_float), ("max_sinphi", C.c_float), ("y_margin", C.c_float),
        ("init_c_ss", C.c_float), ("init_c_tt", C.c_float), ("init_c_qq", C.c_float),
        ("z_is_time", C.c_int32), ("cm_per_time_unit", C.c_float), ("drift_length", C.c_float),
        ("y_is_pad", C.c_int32), ("n_pads", C.c_int32 * _MAX_ROWS), ("pad_pitch", C.c_float * _MAX_ROWS),
    ]


_DEFAULTS = {"z_is_time": 0, "cm_per_time_unit": 0.0, "drift_length": 0.0, "y_is_pad": 0}


_KINDS = {0: np.int32, 1: np.float32, 2: np.float64, 3: np.uint64, 4: np.int64}
_lib = None


def oracle_lib_path() -> str:
    return _build.LIB


def build_oracle(force: bool = False) -> str:
    return _build.build(force)


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.c_void_p]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_run.restype = C.c_int
        lib.orc_run.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        lib.orc_get.restype = C.c_int
        lib.orc_get.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_void_p), C.POINTER(C.c_int64), C.POINTER(C.c_int)]
        lib.orc_kf_propagate.restype = C.c_int
        lib.orc_kf_propagate.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        lib.orc_kf_update.restype = None
        lib.orc_kf_update.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        lib.orc_kf_fit.restype = C.c_int
        lib.orc_kf_fit.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_void_p]
        lib.orc_quantise_residuals.restype = None
        lib.orc_quantise_residuals.argtypes = [C.c_void_p, C.c_float, C.c_float]
        lib.orc_quantise_values.restype = None
        lib.orc_quantise_values.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.c_void_p]
        lib.orc_protect.restype = None
        lib.orc_protect.argtypes = [C.c_void_p, C.c_float, C.c_float]
        lib.orc_merge.restype = None
        lib.orc_merge.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float, C.c_float]
        lib.orc_apex.restype = None
        lib.orc_apex.argtypes = [C.c_void_p, C.c_int] + [C.c_float] * 6
        lib.orc_removable.restype = None
        lib.orc_removable.argtypes = [C.c_void_p] + [C.c_float] * 4
        lib.orc_kf_rotate.restype = C.c_double
        lib.orc_kf_rotate.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double]
        lib.orc_search.restype = C.c_int
        lib.orc_search.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.c_int]
        lib.orc_beam_z.restype = C.c_double
        lib.orc_beam_z.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double]
        assert lib.orc_params_size() == C.sizeof(_Params)
        _lib = lib
    return _lib


def _pack(params: dict) -> _Params:
    p = _Params()
    rx = np.asarray(params["row_x"], dtype=np.float32)
    assert rx.shape[0] == params["n_rows"] <= _MAX_ROWS
    for name, _ in _Params._fields_:
        if name == "row_x":
            for i, v in enumerate(rx):
                p.row_x[i] = float(v)
        elif name in ("n_pads", "pad_pitch"):              # per-row tables of the native pad input (only with y_is_pad)
            if params.get("y_is_pad", 0):
                tab = np.asarray(params[name])
                assert tab.shape[0] == params["n_rows"]
                for i, v in enumerate(tab):
                    getattr(p, name)[i] = v.item()
        else:
            v = params[name] if name in params else _DEFAULTS[name]
            setattr(p, name, v.item() if hasattr(v, "item") else v)
    return p


class Oracle:
    """One oracle instance = one parameter set.  ``run`` executes stages 1..last_stage."""

    def __init__(self, params: dict):
        self._lib = _load()
        self._p = _pack(params)
        self._h = self._lib.orc_create(C.byref(self._p))
        self._keep = None

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.orc_destroy(self._h)
            self._h = None

    def run(self, sector, row, y, z, precision: int = 32, last_stage: int = 5) -> "Oracle":
        sector = np.ascontiguousarray(sector, dtype=np.uint8)
        row = np.ascontiguousarray(row, dtype=np.uint8)
        y = np.ascontiguousarray(y, dtype=np.float32)
        z = np.ascontiguousarray(z, dtype=np.float32)
        self._keep = (sector, row, y, z)
        rc = self._lib.orc_run(self._h, sector.shape[0], sector.ctypes.data, row.ctypes.data, y.ctypes.data,
                               z.ctypes.data, precision, last_stage)
        if rc != 0:
            raise ValueError(f"oracle rejected the input (rc={rc})")
        return self

    def quantise_residuals(self, step_y: float, step_z: float) -> "Oracle":
        """DESIGN.md section 3.7a on the residuals of the last run (last_stage = 6): fit_qres_y / fit_qres_z."""
        self._lib.orc_quantise_residuals(self._h, float(step_y), float(step_z))
        return self

    @staticmethod
    def quantise_values(res, step: float) -> np.ndarray:
        """The scalar rule of section 3.7a applied to given residuals (test entry)."""
        res = np.ascontiguousarray(res, dtype=np.float32)
        out = np.empty(res.shape[0], np.int32)
        _load().orc_quantise_values(res.ctypes.data, res.shape[0], float(step), out.ctypes.data)
        return out

    def protect(self, road_y: float, road_z: float) -> np.ndarray:
        """DESIGN.md section 3.8 on the tracks of the last run: keep flag per INPUT cluster."""
        self._lib.orc_protect(self._h, float(road_y), float(road_z))
        return self.get("keep")

    def merge(self, max_rows: int = 30, back_rows: int = 1, edge: float = 6.0, dz_win: float = 50.0,
              chi2_cut: float = 100.0, road_z0: float = 2.0, road_z1: float = 0.3) -> "Oracle":
        """DESIGN.md section 3.9 on the tracks and the refit of the last run (last_stage = 6): results under mrg_*."""
        self._lib.orc_merge(self._h, int(max_rows), int(back_rows), float(edge), float(dz_win), float(chi2_cut),
                            float(road_z0), float(road_z1))
        return self

    def apex(self, max_k: int = 4, min_s: float = 0.6, dz_win: float = 150.0, tol_c: float = 0.1, tol_z: float = 4.0,
             tol_t: float = 0.1, cut: float = 3.0) -> "Oracle":
        """DESIGN.md section 3.9.8 on the merged tracks of the last merge(): results under apx_*."""
        self._lib.orc_apex(self._h, int(max_k), float(min_s), float(dz_win), float(tol_c), float(tol_z), float(tol_t), float(cut))
        return self

    def removable(self, min_pt: float = 0.05, max_incl: float = 0.85, road_y: float = 1.0, road_z: float = 1.0) -> "Oracle":
        """DESIGN.md section 3.8a (strategy A) on the results of the last merge() + apex(): rem_class, rem_good_track, rem_remove."""
        self._lib.orc_removable(self._h, float(min_pt), float(max_incl), float(road_y), float(road_z))
        return self

    def kf_rotate(self, par, cov15, x, sa, ca, precision=64):
        par = np.array(par, dtype=np.float64); cov = np.array(cov15, dtype=np.float64)
        xn = self._lib.orc_kf_rotate(C.byref(self._p), precision, par.ctypes.data, cov.ctypes.data, float(x), float(sa), float(ca))
        return (not np.isnan(xn)), par, cov, float(xn)

    def get(self, name: str) -> np.ndarray:
        ptr = C.c_void_p(); n = C.c_int64(); kind = C.c_int()
        if self._lib.orc_get(self._h, name.encode(), C.byref(ptr), C.byref(n), C.byref(kind)) != 0:
            raise KeyError(name)
        dt = np.dtype(_KINDS[kind.value])
        if n.value == 0:
            return np.empty(0, dt)
        buf = (C.c_char * (n.value * dt.itemsize)).from_address(ptr.value)
        return np.frombuffer(buf, dtype=dt).copy()

    # ---- single Kalman-filter steps, for the pins
    def kf_propagate(self, par, cov15, x0, x1, precision=64):
        par = np.array(par, dtype=np.float64); cov = np.array(cov15, dtype=np.float64); jac = np.zeros(25)
        ok = self._lib.orc_kf_propagate(C.byref(self._p), precision, par.ctypes.data, cov.ctypes.data, float(x0),
                                        float(x1), jac.ctypes.data)
        return bool(ok), par, cov, jac.reshape(5, 5)

    def kf_update(self, par, cov15, ym, zm_rel, chi2=0.0, precision=64):
        par = np.array(par, dtype=np.float64); cov = np.array(cov15, dtype=np.float64); c2 = np.array([chi2], dtype=np.float64)
        self._lib.orc_kf_update(C.byref(self._p), precision, par.ctypes.data, cov.ctypes.data, float(ym), float(zm_rel),
                                c2.ctypes.data)
        return par, cov, float(c2[0])

    def search(self, par, cov15, zref, sector, row, precision=32) -> int:
        """DESIGN.md section 3.4.3 on the grid of the last run: sorted position of the nearest gated cluster or -1."""
        par = np.array(par, dtype=np.float64); cov = np.array(cov15, dtype=np.float64)
        return int(self._lib.orc_search(self._h, precision, par.ctypes.data, cov.ctypes.data, float(zref), int(sector), int(row)))

    def beam_z(self, x, y, z, tanl, qpt, precision=64) -> float:
        """z of the track at the beam line, assuming a primary from the origin."""
        return float(self._lib.orc_beam_z(C.byref(self._p), precision, float(x), float(y), float(z), float(tanl), float(qpt)))

    def kf_fit(self, x, y, z, precision=64):
        x = np.ascontiguousarray(x, dtype=np.float64); y = np.ascontiguousarray(y, dtype=np.float64)
        z = np.ascontiguousarray(z, dtype=np.float64)
        par = np.zeros(5); cov = np.zeros(15); c2 = np.zeros(1)
        ok = self._lib.orc_kf_fit(C.byref(self._p), precision, x.shape[0], x.ctypes.data, y.ctypes.data, z.ctypes.data,
                                  par.ctypes.data, cov.ctypes.data, c2.ctypes.data)
        return bool(ok), par, cov, float(c2[0])
