"""CPU oracle of the TPC sector-tracker hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It shares nothing with ``paper_1712_09416_b200/csrc`` (the CUDA path) and never imports it.
See the header of ``tpc_oracle.cpp`` for what it computes, the readings it takes and how it is pinned.
"""
from __future__ import annotations

import ctypes as C
import subprocess
from dataclasses import dataclass
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
SRC = HERE / "tpc_oracle.cpp"
LIB = HERE / "libtpcoracle.so"
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> Path:
    """g++ -O2 -ffp-contract=off: strict IEEE evaluation, no fused multiply-add."""
    if force or not LIB.exists() or LIB.stat().st_mtime < SRC.stat().st_mtime:
        r = subprocess.run(["g++", *CXXFLAGS, "-o", str(LIB), str(SRC)], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed:\n" + r.stdout + r.stderr)
    return LIB


class Params(C.Structure):
    """Mirror of ``oracle_params`` (tpc_oracle.cpp)."""
    _fields_ = [
        ("link_step", C.c_int32),
        ("nf_slope_y", C.c_float), ("nf_slope_z", C.c_float), ("nf_w0", C.c_float), ("nf_dmax", C.c_float),
        ("sin_max", C.c_float),
        ("var_s", C.c_float), ("var_t", C.c_float), ("var_q", C.c_float),
        ("chi2_link", C.c_float), ("chi2_ext", C.c_float),
        ("win_nsigma", C.c_float), ("win_min", C.c_float), ("win_max", C.c_float),
        ("max_gap", C.c_int32), ("edge_margin", C.c_float),
        ("min_tracklet_hits", C.c_int32), ("min_track_hits", C.c_int32),
        ("refit", C.c_int32),
        ("merge", C.c_int32), ("merge_dy", C.c_float), ("merge_dz", C.c_float), ("merge_ds", C.c_float),
        ("merge_dt", C.c_float), ("merge_max_gap", C.c_int32),
        ("seed_dedup", C.c_int32), ("checked", C.c_int32),
    ]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class _Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("sigma_y", C.c_float), ("sigma_z", C.c_float), ("bz", C.c_float)]


_FIELDS = ["link_up", "link_dn", "clink_up", "clink_dn", "nf_margin", "seed_offset", "start_hit",
           "tl_first_row", "tl_last_row", "tl_n_hits", "tl_par", "tl_chi2", "tl_margin", "tl_table",
           "trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "trk_seed", "trk_first_row",
           "trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2", "trk_margin", "hit_idx", "tl_cov", "trk_row_out", "trk_out", "trk_next", "trk_prev", "trk_global", "trk_merge_margin",
           "trk_g", "trk_g_ndf", "trk_g_n_hits", "trk_g_sector"]
_F64 = {"nf_margin", "tl_par", "tl_cov", "tl_chi2", "tl_margin", "trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl",
        "trk_qpt", "trk_chi2", "trk_margin", "trk_out", "trk_merge_margin", "trk_g"}

_lib = None


def lib():
    global _lib
    if _lib is None:
        l = C.CDLL(str(build()))
        l.oracle_track_event.restype = C.c_void_p
        l.oracle_track_event.argtypes = [C.POINTER(_Geometry), C.POINTER(Params), C.c_int32, C.c_int32, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32]
        l.oracle_free.argtypes = [C.c_void_p]
        l.oracle_sizes.argtypes = [C.c_void_p, C.c_void_p]
        l.oracle_copy.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        l.oracle_copy.restype = C.c_int32
        l.oracle_default_params.argtypes = [C.POINTER(Params)]
        l.oracle_transport.argtypes = [C.POINTER(_Geometry), C.POINTER(Params), C.c_int32, C.c_double, C.c_double,
                                       C.c_void_p, C.c_void_p]
        l.oracle_transport.restype = C.c_int32
        l.oracle_update.argtypes = [C.POINTER(_Geometry), C.POINTER(Params), C.c_double, C.c_double, C.c_void_p,
                                    C.c_void_p, C.c_void_p]
        l.oracle_max_threads.restype = C.c_int32
        l.oracle_rotate.restype = C.c_int32
        l.oracle_rotate.argtypes = [C.POINTER(_Geometry), C.POINTER(Params), C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        l.oracle_merge_tracks.restype = C.c_int32
        l.oracle_merge_tracks.argtypes = [C.POINTER(_Geometry), C.POINTER(Params), C.c_int32, C.c_int32] + [C.c_void_p] * 9
        _lib = l
    return _lib


def default_params() -> Params:
    p = Params()
    lib().oracle_default_params(C.byref(p))
    return p


def max_threads() -> int:
    return int(lib().oracle_max_threads())


@dataclass
class Geometry:
    n_sectors: int
    row_x: np.ndarray          # float32 [n_rows]
    tan_half_angle: float
    sigma_y: float
    sigma_z: float
    bz: float

    def _c(self):
        rx = np.ascontiguousarray(self.row_x, dtype=np.float32)
        g = _Geometry(self.n_sectors, rx.shape[0], rx.ctypes.data_as(C.POINTER(C.c_float)), self.tan_half_angle,
                      self.sigma_y, self.sigma_z, self.bz)
        return g, rx


class Result(dict):
    """Field name -> numpy array (int32, or float64 for the names in _F64); plus sizes."""
    __getattr__ = dict.__getitem__


def track_event(geom: Geometry, sector_offset, y, z, row, params: Params | None = None, precision: str = "double",
                n_threads: int = 0, stop_after: int = 0) -> Result:
    """Run O1..O7 on one event.  ``precision``: "double" or "float" (strict float32).  All hit indices in the
    result are indices into the caller's arrays."""
    l = lib()
    p = params if params is not None else default_params()
    g, _keep = geom._c()
    so = np.ascontiguousarray(sector_offset, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    z = np.ascontiguousarray(z, dtype=np.float32)
    row = np.ascontiguousarray(row, dtype=np.int32)
    n = int(y.shape[0])
    assert so.shape[0] == geom.n_sectors + 1 and so[-1] == n
    h = l.oracle_track_event(C.byref(g), C.byref(p), 1 if precision == "float" else 0, n, so.ctypes.data,
                             y.ctypes.data, z.ctypes.data, row.ctypes.data, n_threads, stop_after)
    if not h:
        raise ValueError("oracle_track_event: bad arguments")
    try:
        sz = np.zeros(5, np.int64)
        l.oracle_sizes(h, sz.ctypes.data)
        N, S, T, H, NR = (int(v) for v in sz)
        shapes = {"link_up": (N,), "link_dn": (N,), "clink_up": (N,), "clink_dn": (N,), "nf_margin": (N,),
                  "seed_offset": (geom.n_sectors + 1,), "start_hit": (S,), "tl_first_row": (S,), "tl_last_row": (S,),
                  "tl_n_hits": (S,), "tl_par": (S, 5), "tl_cov": (S, 5), "tl_chi2": (S,), "tl_margin": (S,), "tl_table": (S, NR),
                  "hit_idx": (H,), "trk_out": (T, 6), "trk_g": (T, 7)}
        out = Result(n_clusters=N, n_seeds=S, n_tracks=T, n_track_hits=H)
        for i, name in enumerate(_FIELDS):
            shape = shapes.get(name, (T,))
            if stop_after and stop_after < 5 and name.startswith("tl_"):
                shape = (0,) + shape[1:]
            a = np.zeros(shape, np.float64 if name in _F64 else np.int32)
            if a.size:
                l.oracle_copy(h, i, a.ctypes.data)
            out[name] = a
    finally:
        l.oracle_free(h)
    return out


def transport(geom: Geometry, x: float, x1: float, state, cov, params: Params | None = None,
              precision: str = "double"):
    """One helix transport step of the fit (state [y,z,sin phi,tg lambda,q/pT], 5x5 covariance)."""
    p = params if params is not None else default_params()
    g, _keep = geom._c()
    st = np.array(state, np.float64).copy()
    cv = np.array(cov, np.float64).reshape(5, 5).copy()
    rc = lib().oracle_transport(C.byref(g), C.byref(p), 1 if precision == "float" else 0, x, x1, st.ctypes.data,
                                cv.ctypes.data)
    return rc == 0, st, cv


def update(geom: Geometry, my: float, mz: float, state, cov, chi2: float = 0.0, params: Params | None = None):
    """One Kalman measurement update (y then z) in double."""
    p = params if params is not None else default_params()
    g, _keep = geom._c()
    st = np.array(state, np.float64).copy()
    cv = np.array(cov, np.float64).reshape(5, 5).copy()
    c2 = np.array([chi2], np.float64)
    lib().oracle_update(C.byref(g), C.byref(p), my, mz, st.ctypes.data, cv.ctypes.data, c2.ctypes.data)
    return st, cv, float(c2[0])


def merge_tracks(geom: Geometry, sector, first_row, par, row_out, out, params: Params | None = None,
                 precision: str = "double"):
    """O9 on caller-given segments: ``par`` [T,6] = x, y, z, sin phi, tg lambda, q/pT at the first fitted row,
    ``out`` [T,6] the outer state at pad row ``row_out``.  Returns next, prev, global (int32 [T]) and margin."""
    p = params if params is not None else default_params()
    g, _keep = geom._c()
    sector = np.ascontiguousarray(sector, np.int32); first_row = np.ascontiguousarray(first_row, np.int32)
    row_out = np.ascontiguousarray(row_out, np.int32)
    par = np.ascontiguousarray(par, np.float64).reshape(-1, 6); out = np.ascontiguousarray(out, np.float64).reshape(-1, 6)
    T = int(sector.shape[0])
    nx = np.zeros(T, np.int32); pv = np.zeros(T, np.int32); gl = np.zeros(T, np.int32); mg = np.zeros(T, np.float64)
    rc = lib().oracle_merge_tracks(C.byref(g), C.byref(p), 1 if precision == "float" else 0, T, sector.ctypes.data,
                                   first_row.ctypes.data, par.ctypes.data, row_out.ctypes.data, out.ctypes.data,
                                   nx.ctypes.data, pv.ctypes.data, gl.ctypes.data, mg.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_merge_tracks: bad arguments")
    return nx, pv, gl, mg


def rotate(geom: Geometry, x: float, angle: float, state, cov, params: Params | None = None):
    """One O10 rotation step in double: the fit given at ``x`` in one sector frame, expressed in a frame whose axis is
    turned by ``angle`` (rad; negative = the next sector in azimuth).  Returns ok, x', state, cov."""
    p = params if params is not None else default_params()
    g, _keep = geom._c()
    st = np.array(state, np.float64).copy()
    cv = np.array(cov, np.float64).reshape(5, 5).copy()
    xx = np.array([x], np.float64)
    rc = lib().oracle_rotate(C.byref(g), C.byref(p), xx.ctypes.data, float(np.sin(angle)), float(np.cos(angle)),
                             st.ctypes.data, cv.ctypes.data)
    return rc == 0, float(xx[0]), st, cv
