"""Thin ctypes binding of ``csrc/libtpctrack.so`` (the C ABI of ``include/tpctrack.h``).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  The functions carry the
names of the C entry points.  There is no CPU fallback: importing this module fails loudly when the library is
missing, and ``tpc_tracker_create`` fails when no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

import os

LIB_PATH = Path(os.environ.get("TPCTRACK_LIB") or Path(__file__).resolve().parent / "csrc" / "libtpctrack.so")

TPC_OK, TPC_ERR_ARG, TPC_ERR_GEOMETRY, TPC_ERR_CAPACITY, TPC_ERR_CUDA = 0, -1, -2, -3, -4
N_STAGES = 6   # TPC_N_STAGES
STAGE = {"clean": 3, "seeds": 4, "construct": 5, "select": 6}   # TPC_STAGE_*
DBG = {"link_up": 0, "link_dn": 1, "clink_up": 2, "clink_dn": 3, "start_hit": 4, "tl_rows": 5, "tl_par": 6,
       "tl_table": 7, "sorted": 8}


class tpc_geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("z_abs_max", C.c_float), ("sigma_y", C.c_float),
                ("sigma_z", C.c_float), ("sector_alpha", C.POINTER(C.c_float))]


class tpc_params(C.Structure):
    _fields_ = [("link_step", C.c_int32), ("nf_slope_y", C.c_float), ("nf_slope_z", C.c_float), ("nf_w0", C.c_float),
                ("nf_dmax", C.c_float), ("sin_max", C.c_float), ("var_s", C.c_float), ("var_t", C.c_float),
                ("var_q", C.c_float), ("chi2_link", C.c_float), ("chi2_ext", C.c_float), ("win_nsigma", C.c_float),
                ("win_min", C.c_float), ("win_max", C.c_float), ("max_gap", C.c_int32), ("edge_margin", C.c_float),
                ("min_tracklet_hits", C.c_int32), ("min_track_hits", C.c_int32), ("refit", C.c_int32),
                ("merge", C.c_int32), ("merge_dy", C.c_float), ("merge_dz", C.c_float), ("merge_ds", C.c_float),
                ("merge_dt", C.c_float), ("merge_max_gap", C.c_int32), ("seed_dedup", C.c_int32), ("checked", C.c_int32)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class tpc_event_in(C.Structure):
    _fields_ = [("n_clusters", C.c_int32), ("sector_offset", C.c_void_p), ("x", C.c_void_p), ("y", C.c_void_p),
                ("z", C.c_void_p), ("row", C.c_void_p), ("mem_space", C.c_int32)]


_OUT_I = ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf")
_OUT_F = ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2")
_OUT_F2 = ("trk_out_x", "trk_out_y", "trk_out_z", "trk_out_sinphi", "trk_out_tgl", "trk_out_qpt")   # refit = 1
_OUT_I2 = ("trk_next", "trk_prev", "trk_global")                                                                   # merge = 1
_OUT_F3 = ("trk_g_x", "trk_g_y", "trk_g_z", "trk_g_sinphi", "trk_g_tgl", "trk_g_qpt", "trk_g_chi2")   # merge = 1 (O10)
_OUT_I3 = ("trk_g_ndf", "trk_g_n_hits", "trk_g_sector")


class tpc_event_out(C.Structure):
    _fields_ = ([("n_tracks", C.c_int32), ("n_track_hits", C.c_int32)] + [(n, C.c_void_p) for n in _OUT_I]
                + [(n, C.c_void_p) for n in _OUT_F] + [("hit_idx", C.c_void_p)]
                + [(n, C.c_void_p) for n in _OUT_F2] + [(n, C.c_void_p) for n in _OUT_I2]
                + [(n, C.c_void_p) for n in _OUT_F3] + [(n, C.c_void_p) for n in _OUT_I3])


class tpc_counters(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_events", "n_clusters", "n_links", "n_seeds", "n_row_visits",
                                         "n_tracklet_hits", "n_tracks", "n_track_hits", "n_kernel_launches",
                                         "n_retries", "n_updates", "n_refit_visits", "n_tracklets")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class TpcError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("tpctrack status %d (%s): %s" % (status, tpc_status_string(status), text))
        self.status = status


def _load():
    if not LIB_PATH.exists():
        raise ImportError("%s is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a).  There is no CPU fallback." % LIB_PATH)
    lib = C.CDLL(str(LIB_PATH))
    lib.tpc_default_params.argtypes = [C.POINTER(tpc_params)]
    lib.tpc_tracker_create.restype = C.c_void_p
    lib.tpc_tracker_create.argtypes = [C.POINTER(tpc_geometry), C.c_float]
    lib.tpc_tracker_create_ex.restype = C.c_void_p
    lib.tpc_tracker_create_ex.argtypes = [C.POINTER(tpc_geometry), C.c_float, C.POINTER(tpc_params), C.c_int32, C.c_int64]
    lib.tpc_tracker_set_stream.argtypes = [C.c_void_p, C.c_void_p]
    lib.tpc_tracker_set_group_events.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_track_event.argtypes = [C.c_void_p, C.POINTER(tpc_event_in), C.POINTER(tpc_event_out)]
    lib.tpc_track_events.argtypes = [C.c_void_p, C.c_int32, C.POINTER(tpc_event_in), C.POINTER(tpc_event_out)]
    lib.tpc_submit_events.argtypes = [C.c_void_p, C.c_int32, C.POINTER(tpc_event_in), C.POINTER(C.c_int32)]
    lib.tpc_wait_events.argtypes = [C.c_void_p, C.c_int32, C.POINTER(tpc_event_out)]
    lib.tpc_tracker_destroy.argtypes = [C.c_void_p]
    lib.tpc_tracker_destroy.restype = None
    lib.tpc_status_string.restype = C.c_char_p
    lib.tpc_status_string.argtypes = [C.c_int]
    lib.tpc_last_error.restype = C.c_char_p
    lib.tpc_get_counters.argtypes = [C.c_void_p, C.POINTER(tpc_counters)]
    lib.tpc_tracker_set_profiling.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_get_stage_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    lib.tpc_debug_size.restype = C.c_int64
    lib.tpc_debug_size.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
    lib.tpc_debug_get.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t]
    lib.tpc_debug_inject.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t]
    lib.tpc_debug_resume.argtypes = [C.c_void_p, C.c_int32, C.POINTER(tpc_event_out)]
    lib.tpc_measure_fp32_peak.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.tpc_scan_exclusive_static.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.tpc_debug_scan_exclusive.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
    return lib


lib = _load()

EXPORTS = ("tpc_default_params", "tpc_tracker_create", "tpc_tracker_create_ex", "tpc_tracker_set_stream",
           "tpc_tracker_set_group_events",
           "tpc_track_event", "tpc_track_events", "tpc_submit_events", "tpc_wait_events", "tpc_tracker_destroy", "tpc_status_string", "tpc_last_error",
           "tpc_get_counters", "tpc_tracker_set_profiling", "tpc_get_stage_ms", "tpc_debug_size", "tpc_debug_get",
           "tpc_debug_inject", "tpc_debug_resume", "tpc_measure_fp32_peak", "tpc_scan_exclusive_static",
           "tpc_debug_scan_exclusive")


def tpc_status_string(status: int) -> str:
    return lib.tpc_status_string(status).decode()


def tpc_last_error() -> str:
    return lib.tpc_last_error().decode()


def tpc_measure_fp32_peak() -> tuple:
    """(fused multiply-add, un-fused multiply + add) FP32 TFLOP/s measured on the current device."""
    a, b = C.c_float(0), C.c_float(0)
    _check(lib.tpc_measure_fp32_peak(C.byref(a), C.byref(b)))
    return float(a.value), float(b.value)


SCAN_STATIC_MAX_N = 1 << 24   # TPC_SCAN_STATIC_MAX_N


def tpc_scan_exclusive_static(in_dev, n: int, out_dev, cuda_stream=None) -> None:
    """Exclusive prefix sum of ``n`` int32 values for callers that may not allocate device memory (a framework owns
    all of it, or cudaMalloc's device-wide stall is not acceptable where they run): the kernel's scratch words live in
    an array inside the library, so only the caller's ``in_dev`` [n] and ``out_dev`` [n + 1] (device pointers, as
    integers) are touched.  Enqueued on ``cuda_stream`` (integer handle, None = default stream); not waited for.
    ``n`` beyond ``SCAN_STATIC_MAX_N`` raises TpcError (TPC_ERR_CAPACITY).  All calls share the one array: do not let
    two of them overlap on the GPU.  See include/tpctrack.h."""
    _check(lib.tpc_scan_exclusive_static(in_dev, n, out_dev, cuda_stream))


def tpc_debug_scan_exclusive(in_dev, n: int, out_dev) -> None:
    """The same prefix sum with cudaMalloc'ed scratch, as the tracker runs it (tests only; synchronous)."""
    _check(lib.tpc_debug_scan_exclusive(in_dev, n, out_dev))


def tpc_default_params() -> tpc_params:
    p = tpc_params()
    lib.tpc_default_params(C.byref(p))
    return p


def _check(status):
    if status != TPC_OK:
        raise TpcError(status, tpc_last_error())


class Tracker:
    """Owns one ``tpc_tracker*``.  ``row_x``: float32 pad-row radii (host)."""

    def __init__(self, n_sectors, row_x, tan_half_angle, sigma_y, sigma_z, bz, params: tpc_params | None = None,
                 z_abs_max=250.0, max_events=0, max_clusters=0):
        self._rx = np.ascontiguousarray(row_x, dtype=np.float32)
        g = tpc_geometry(n_sectors, self._rx.shape[0], self._rx.ctypes.data_as(C.POINTER(C.c_float)), tan_half_angle,
                         z_abs_max, sigma_y, sigma_z, None)
        self.n_sectors, self.n_rows = n_sectors, int(self._rx.shape[0])
        self._h = lib.tpc_tracker_create_ex(C.byref(g), bz, C.byref(params) if params is not None else None,
                                            max_events, max_clusters)
        if not self._h:
            raise TpcError(TPC_ERR_CUDA, tpc_last_error())
        self._keep = None

    def close(self):
        if getattr(self, "_h", None):
            lib.tpc_tracker_destroy(self._h)
            self._h = None

    __del__ = close

    def set_stream(self, cuda_stream_ptr: int | None):
        _check(lib.tpc_tracker_set_stream(self._h, C.c_void_p(cuda_stream_ptr or 0)))

    def tpc_tracker_set_group_events(self, n: int):
        _check(lib.tpc_tracker_set_group_events(self._h, int(n)))

    # ---- marshalling ----
    @staticmethod
    def _ptr(a):
        if a is None:
            return None, 0
        if isinstance(a, np.ndarray):
            return a.ctypes.data, 0
        return a.data_ptr(), 1        # torch tensor

    def _marshal(self, events):
        n = len(events)
        ins = (tpc_event_in * n)()
        keep = []
        for i, ev in enumerate(events):
            so = np.ascontiguousarray(ev["sector_offset"], dtype=np.int32)
            keep.append(so)
            spaces = set()
            ptrs = {"x": None}
            for k in ("x", "y", "z", "row"):
                if k == "x" and ev.get("x") is None:     # optional: only the checked mode reads it
                    continue
                a = ev[k]
                if isinstance(a, np.ndarray):
                    want = np.int32 if k == "row" else np.float32
                    if a.dtype != want or not a.flags.c_contiguous:
                        a = np.ascontiguousarray(a, dtype=want)
                    keep.append(a)
                else:
                    assert a.is_cuda and a.is_contiguous(), "device inputs must be contiguous CUDA tensors"
                    keep.append(a)
                p, sp = self._ptr(a)
                ptrs[k] = p
                spaces.add(sp)
            assert len(spaces) == 1, "y, z, row must live in one memory space"
            ncl = int(so[-1])
            ins[i] = tpc_event_in(ncl, so.ctypes.data, ptrs["x"], ptrs["y"], ptrs["z"], ptrs["row"], spaces.pop())
        return ins, keep

    def tpc_track_events(self, events):
        """events: list of dicts with sector_offset (host int32), y, z (float32), row (int32), optionally x: all
        numpy (host) or all torch CUDA tensors (device).  Returns a list of raw ``tpc_event_out`` structs (pointers are
        library-owned; host or device like the input) -- see ``to_numpy``."""
        n = len(events)
        ins, keep = self._marshal(events)
        outs = (tpc_event_out * n)()
        self._keep = keep
        _check(lib.tpc_track_events(self._h, n, ins, outs))
        self._mem_space = ins[0].mem_space if n else 0
        return list(outs)

    def tpc_track_event(self, event):
        return self.tpc_track_events([event])[0]

    def tpc_submit_events(self, events) -> int:
        """Enqueue a batch (copies in + all kernels) and return its ticket; at most three batches in flight.  The
        events' arrays must stay unchanged until ``tpc_wait_events(ticket)`` returns."""
        n = len(events)
        ins, keep = self._marshal(events)
        ticket = C.c_int32(-1)
        _check(lib.tpc_submit_events(self._h, n, ins, C.byref(ticket)))
        if not hasattr(self, "_tickets"):
            self._tickets = {}
        self._tickets[ticket.value] = (n, ins, keep)
        return ticket.value

    def tpc_wait_events(self, ticket: int):
        """Wait for the batch of ``ticket``; returns its list of ``tpc_event_out`` (valid until the second submit
        after this call)."""
        n, ins, keep = self._tickets.pop(ticket)
        outs = (tpc_event_out * n)()
        _check(lib.tpc_wait_events(self._h, ticket, outs))
        self._mem_space = ins[0].mem_space if n else 0
        self._keep = keep
        return list(outs)

    def tpc_get_counters(self) -> dict:
        c = tpc_counters()
        _check(lib.tpc_get_counters(self._h, C.byref(c)))
        return c.as_dict()

    def tpc_tracker_set_profiling(self, on: bool):
        _check(lib.tpc_tracker_set_profiling(self._h, int(on)))

    def tpc_get_stage_ms(self):
        ms = (C.c_float * N_STAGES)()
        _check(lib.tpc_get_stage_ms(self._h, ms))
        return [float(v) for v in ms]

    def tpc_debug_get(self, what: str, event: int = 0) -> np.ndarray:
        w = DBG[what]
        nbytes = lib.tpc_debug_size(self._h, w, event)
        if nbytes < 0:
            raise TpcError(int(nbytes), tpc_last_error())
        dt = np.float32 if what == "tl_par" else np.int32
        a = np.zeros(nbytes // 4, dt)
        _check(lib.tpc_debug_get(self._h, w, event, a.ctypes.data, a.nbytes))
        if what == "tl_rows":
            a = a.reshape(-1, 3)
        elif what == "tl_par":
            a = a.reshape(-1, 6)
        elif what == "tl_table":
            a = a.reshape(-1, self.n_rows)
        return a

    def tpc_debug_inject(self, what: str, a: np.ndarray, event: int = 0):
        """Overwrite an intermediate of the last call (layout of ``tpc_debug_get``)."""
        a = np.ascontiguousarray(a, dtype=np.float32 if what == "tl_par" else np.int32)
        _check(lib.tpc_debug_inject(self._h, DBG[what], event, a.ctypes.data, a.nbytes))

    def tpc_debug_resume(self, from_stage: str, n_events: int = 1):
        """Run the path again from ``from_stage`` ("clean", "seeds", "construct", "select") on the work space."""
        outs = (tpc_event_out * n_events)()
        _check(lib.tpc_debug_resume(self._h, STAGE[from_stage], outs))
        return list(outs)

    @staticmethod
    def as_tensor(ptr, n, dt):
        """Zero-copy torch view of a library-owned device array."""
        import torch

        class _Dev:
            pass
        d = _Dev()
        d.__cuda_array_interface__ = {"shape": (n,), "typestr": "<i4" if dt == np.int32 else "<f4",
                                      "data": (int(ptr), False), "version": 2}
        return torch.as_tensor(d, device="cuda")

    def to_numpy(self, out: tpc_event_out) -> dict:
        """Copy one event's outputs into numpy arrays."""
        T, H = out.n_tracks, out.n_track_hits
        res = {"n_tracks": T, "n_track_hits": H}

        def fetch(ptr, n, dt):
            if n == 0 or not ptr:
                return np.zeros(0, dt)
            if self._mem_space == 0:
                return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(C.c_int32 if dt == np.int32 else C.c_float)),
                                             shape=(n,)).copy()
            return self.as_tensor(ptr, n, dt).cpu().numpy()

        for k in _OUT_I:
            res[k] = fetch(getattr(out, k), T, np.int32)
        for k in _OUT_F:
            res[k] = fetch(getattr(out, k), T, np.float32)
        res["hit_idx"] = fetch(out.hit_idx, H, np.int32)
        for k in _OUT_F2:          # present with refit = 1
            if getattr(out, k):
                res[k] = fetch(getattr(out, k), T, np.float32)
        for k in _OUT_I2 + _OUT_I3:          # present with merge = 1
            if getattr(out, k):
                res[k] = fetch(getattr(out, k), T, np.int32)
        for k in _OUT_F3:
            if getattr(out, k):
                res[k] = fetch(getattr(out, k), T, np.float32)
        return res
