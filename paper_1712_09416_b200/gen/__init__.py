"""Seeded synthetic TPC events: the inputs of both the CPU oracle (tests) and the CUDA path.

Holds geometry tables and workload recipes only -- none of the tracker's arithmetic.
The events stand in for the ALICE Pb-Pb / p-Pb data the paper ran on, which is not available;
the five recipes are BASELINE.json ``configs`` (lines 7-11) as read in SURVEY.md 8(d).1.
"""
from __future__ import annotations

import ctypes as C
import math
from dataclasses import dataclass, field
from typing import List

import numpy as np

from .. import _build

N_ROWS = 159
TAN_HALF_ANGLE = math.tan(math.radians(10.0))
Z_MAX = 250.0
R_MAX = 247.0
BZ = 0.5


def row_x() -> np.ndarray:
    """Pad-row radii in cm (BASELINE.json:7: 63 rows at 0.75 cm pitch from 85.225, 64 at 1.0, 32 at 1.5;
    start radii of groups 2 and 3 are the reading S17 of SURVEY.md 8(c).4: 135.1 and 199.35 cm)."""
    a = 85.225 + 0.75 * np.arange(63)
    b = 135.1 + 1.0 * np.arange(64)
    c = 199.35 + 1.5 * np.arange(32)
    return np.concatenate([a, b, c]).astype(np.float64)


def sector_alpha(n_sectors: int = 36) -> np.ndarray:
    """Centre azimuth of each sector in rad: alpha_s = (20*(s mod 18)+10) deg; s>=18 is the C side (z<0)."""
    s = np.arange(n_sectors)
    return np.radians(20.0 * (s % 18) + 10.0)


class _Cfg(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_double)),
        ("tan_half_angle", C.c_double), ("z_max", C.c_double), ("r_max", C.c_double), ("bz", C.c_double),
        ("n_primaries", C.c_int32), ("frac_secondaries", C.c_double),
        ("pt_mode", C.c_int32), ("pt_a", C.c_double), ("pt_b", C.c_double), ("eta_max", C.c_double),
        ("sigma_y", C.c_double), ("sigma_z", C.c_double), ("inefficiency", C.c_double),
        ("noise_frac", C.c_double), ("loopers", C.c_int32), ("max_turns", C.c_int32), ("shuffle", C.c_int32),
    ]


@dataclass
class Recipe:
    """One workload recipe (a BASELINE.json config)."""
    name: str
    n_sectors: int = 36
    n_primaries: int = 60
    frac_secondaries: float = 0.0
    pt_mode: int = 1            # 0 uniform [pt_a, pt_b]; 1 pt_a + Exp(mean pt_b)
    pt_a: float = 0.1
    pt_b: float = 0.5
    eta_max: float = 0.9
    sigma: float = 0.06
    inefficiency: float = 0.02
    noise_frac: float = 0.05
    loopers: bool = False
    max_turns: int = 3
    shuffle: bool = True
    bz: float = BZ
    n_events: int = 1
    config_id: int = 0          # seeds: event e of config c uses 1000*c + e


# BASELINE.json:7-11
RECIPES = {
    "single_sector": Recipe("single_sector", n_sectors=1, n_primaries=50, pt_mode=0, pt_a=0.2, pt_b=5.0,
                            sigma=0.06, noise_frac=0.05, config_id=1),
    "pp": Recipe("pp", n_primaries=60, sigma=0.06, noise_frac=0.05, config_id=2),
    "semicentral": Recipe("semicentral", n_primaries=2000, frac_secondaries=0.15, sigma=0.06, noise_frac=0.10,
                          config_id=3),
    "central": Recipe("central", n_primaries=8000, frac_secondaries=0.20, sigma=0.08, noise_frac=0.10,
                      loopers=True, config_id=4),
    "central_batch16": Recipe("central_batch16", n_primaries=8000, frac_secondaries=0.20, sigma=0.08,
                              noise_frac=0.10, loopers=True, n_events=16, config_id=5),
    # not a BASELINE.json config: SURVEY.md 8(f).4 "higher-occupancy events (2-3x cluster density)": 2.5 x central
    "dense": Recipe("dense", n_primaries=20000, frac_secondaries=0.20, sigma=0.08, noise_frac=0.10, loopers=True,
                    config_id=6),
}

TRK_COLS = ("pt", "charge", "eta", "phi", "vx", "vy", "vz", "primary")


@dataclass
class Event:
    """float32 SoA clusters grouped by sector (+ truth the tracker never sees)."""
    n_sectors: int
    sector_offset: np.ndarray  # int32 [n_sectors+1]
    x: np.ndarray              # float32 [N]  (= row_x[row])
    y: np.ndarray              # float32 [N]  sector-local
    z: np.ndarray              # float32 [N]  signed
    row: np.ndarray            # int32 [N]
    label: np.ndarray          # int32 [N]   generator track id, -1 = noise
    tracks: np.ndarray         # float64 [n_tracks, 8]  columns TRK_COLS
    sigma: float = 0.06
    bz: float = BZ
    seed: int = 0
    recipe: str = ""

    @property
    def n_clusters(self) -> int:
        return int(self.x.shape[0])


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(str(_build.build_gen()))
        lib.tpcgen_generate.restype = C.c_void_p
        lib.tpcgen_generate.argtypes = [C.POINTER(_Cfg), C.c_uint64]
        lib.tpcgen_free.argtypes = [C.c_void_p]
        lib.tpcgen_n_clusters.argtypes = [C.c_void_p]
        lib.tpcgen_n_tracks.argtypes = [C.c_void_p]
        lib.tpcgen_n_clusters.restype = C.c_int32
        lib.tpcgen_n_tracks.restype = C.c_int32
        lib.tpcgen_copy.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        _lib = lib
    return _lib


def generate(recipe: Recipe | str, event: int = 0, seed: int | None = None) -> Event:
    """One event of ``recipe``; the seed defaults to 1000*config_id + event."""
    if isinstance(recipe, str):
        recipe = RECIPES[recipe]
    lib = _load()
    rx = np.ascontiguousarray(row_x())
    if seed is None:
        seed = 1000 * recipe.config_id + event
    cfg = _Cfg(recipe.n_sectors, N_ROWS, rx.ctypes.data_as(C.POINTER(C.c_double)), TAN_HALF_ANGLE, Z_MAX, R_MAX,
               recipe.bz, recipe.n_primaries, recipe.frac_secondaries, recipe.pt_mode, recipe.pt_a, recipe.pt_b,
               recipe.eta_max, recipe.sigma, recipe.sigma, recipe.inefficiency, recipe.noise_frac,
               int(recipe.loopers), recipe.max_turns, int(recipe.shuffle))
    h = lib.tpcgen_generate(C.byref(cfg), C.c_uint64(seed))
    if not h:
        raise RuntimeError("tpcgen_generate failed")
    try:
        n, nt = lib.tpcgen_n_clusters(h), lib.tpcgen_n_tracks(h)
        so = np.zeros(recipe.n_sectors + 1, np.int32)
        x = np.zeros(n, np.float32); y = np.zeros(n, np.float32); z = np.zeros(n, np.float32)
        row = np.zeros(n, np.int32); label = np.zeros(n, np.int32)
        trk = np.zeros((nt, len(TRK_COLS)), np.float64)
        lib.tpcgen_copy(h, *[a.ctypes.data for a in (so, x, y, z, row, label, trk)])
    finally:
        lib.tpcgen_free(h)
    return Event(recipe.n_sectors, so, x, y, z, row, label, trk, sigma=recipe.sigma, bz=recipe.bz, seed=seed,
                 recipe=recipe.name)


def generate_batch(recipe: Recipe | str) -> List[Event]:
    if isinstance(recipe, str):
        recipe = RECIPES[recipe]
    return [generate(recipe, e) for e in range(recipe.n_events)]


def tiny_sector(n_tracks: int = 6, seed: int = 7, noise_frac: float = 0.3, sigma: float = 0.06,
                n_sectors: int = 1) -> Event:
    """A small sector for brute-force pins (few tracks, heavy noise so that ambiguities occur)."""
    r = Recipe("tiny", n_sectors=n_sectors, n_primaries=n_tracks, pt_mode=0, pt_a=0.3, pt_b=3.0, sigma=sigma,
               noise_frac=noise_frac, config_id=0)
    return generate(r, seed=seed)
