"""Seeded synthetic TPC time frames (input generator only -- no tracking arithmetic).

Shapes follow BASELINE.json configs 1-5; recipe in DESIGN.md "Input recipe".  The heavy
lifting is `tpc_synth.c` (float64, counter-based RNG), compiled on first use with gcc.
Both the oracle tests and the CUDA path read the arrays this module returns.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_synth.c")
_SO = os.path.join(_HERE, "libtpc_synth.so")

N_ROWS = 152
X_FIRST, X_LAST = 85.0, 245.0
BZ_TESLA = 0.5
VDRIFT_CM_PER_US = 2.58
SIGMA_Y, SIGMA_Z = 0.1, 0.15
TAN_HALF_ANGLE = float(np.tan(np.deg2rad(10.0)))


def row_x() -> np.ndarray:
    """fp32 pad-row x positions, 85..245 cm linearly spaced (BASELINE.json config 1)."""
    r = np.arange(N_ROWS, dtype=np.float64)
    return (X_FIRST + (X_LAST - X_FIRST) / (N_ROWS - 1) * r).astype(np.float32)


class _Cfg(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32),
        ("x_first", C.c_double), ("x_last", C.c_double), ("bz_tesla", C.c_double),
        ("seed", C.c_uint64), ("n_collisions", C.c_int32),
        ("mult_lo", C.c_int32), ("mult_hi", C.c_int32), ("mult_log_uniform", C.c_int32),
        ("pt_law", C.c_int32), ("pt_lo", C.c_double), ("pt_hi", C.c_double), ("pt_mean", C.c_double),
        ("eta_max", C.c_double), ("vz_sigma", C.c_double), ("phi_in_sector", C.c_int32),
        ("n_loopers", C.c_int32), ("looper_pt_lo", C.c_double), ("looper_pt_hi", C.c_double),
        ("time_window_us", C.c_double), ("vdrift", C.c_double),
        ("sigma_y", C.c_double), ("sigma_z", C.c_double), ("noise_frac", C.c_double),
        ("z_max", C.c_double), ("max_turns", C.c_int32),
    ]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.synth_generate.restype = C.c_void_p
        lib.synth_generate.argtypes = [C.POINTER(_Cfg)]
        lib.synth_free.argtypes = [C.c_void_p]
        lib.synth_n.restype = C.c_int64
        lib.synth_n.argtypes = [C.c_void_p]
        lib.synth_n_tracks.restype = C.c_int32
        lib.synth_n_tracks.argtypes = [C.c_void_p]
        for name, t in (("synth_xyz", C.c_float), ("synth_row", C.c_int32), ("synth_truth", C.c_int32),
                        ("synth_sector_offsets", C.c_int32), ("synth_track_par", C.c_double)):
            fn = getattr(lib, name)
            fn.restype = C.POINTER(t)
            fn.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


@dataclass
class Frame:
    """One synthetic time frame.  `clusters` is the 16-byte record the C-ABI takes."""
    clusters: np.ndarray        # structured (x,y,z f32, row i32), n
    sector_offsets: np.ndarray  # int32, n_sectors+1 (CSR)
    truth: np.ndarray           # int32 n: generator track id, -1 = noise (harness only)
    track_par: np.ndarray       # float64 (n_tracks, 8): pt, phi0, eta, q, vz, t0_us, collision, n_clusters
    n_sectors: int
    name: str

    @property
    def n(self) -> int:
        return int(self.clusters.shape[0])


CLUSTER_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("row", "<i4")])


def _base(seed: int) -> dict:
    return dict(n_sectors=36, n_rows=N_ROWS, x_first=X_FIRST, x_last=X_LAST, bz_tesla=BZ_TESLA, seed=seed,
                n_collisions=1, mult_lo=4000, mult_hi=4000, mult_log_uniform=0,
                pt_law=1, pt_lo=0.1, pt_hi=20.0, pt_mean=0.5, eta_max=0.9, vz_sigma=5.0, phi_in_sector=0,
                n_loopers=0, looper_pt_lo=0.05, looper_pt_hi=0.15, time_window_us=0.0, vdrift=VDRIFT_CM_PER_US,
                sigma_y=SIGMA_Y, sigma_z=SIGMA_Z, noise_frac=0.10, z_max=250.0, max_turns=10)


def config(k: int, scale: float = 1.0, seed: int | None = None) -> dict:
    """BASELINE.json config k (1-5).  `scale` < 1 shrinks multiplicities for quick tests."""
    c = _base(k if seed is None else seed)
    if k == 1:
        c.update(n_sectors=1, mult_lo=int(200 * scale), mult_hi=int(200 * scale), pt_law=0, pt_lo=0.2, pt_hi=10.0,
                 vz_sigma=0.0, phi_in_sector=1, noise_frac=0.05)
    elif k == 2:
        c.update(mult_lo=int(4000 * scale), mult_hi=int(4000 * scale))
    elif k == 3:
        c.update(mult_lo=int(2000 * scale), mult_hi=int(2000 * scale), n_loopers=int(1000 * scale))
    elif k == 4:
        c.update(n_collisions=5, mult_lo=int(4000 * scale), mult_hi=int(4000 * scale), time_window_us=100.0)
    elif k == 5:
        c.update(n_collisions=max(1, int(round(50 * scale))), mult_lo=50, mult_hi=4000, mult_log_uniform=1,
                 time_window_us=1000.0 * min(1.0, scale))
    else:
        raise ValueError("config must be 1..5")
    return c


def generate(cfg: dict | int, name: str | None = None, **over) -> Frame:
    if isinstance(cfg, int):
        name = name or f"config{cfg}"
        cfg = config(cfg)
    cfg = dict(cfg, **over)
    lib = _load()
    cc = _Cfg(**cfg)
    h = lib.synth_generate(C.byref(cc))
    if not h:
        raise MemoryError("synth_generate failed")
    try:
        n = lib.synth_n(h)
        nt = lib.synth_n_tracks(h)
        ns = cfg["n_sectors"]
        xyz = np.ctypeslib.as_array(lib.synth_xyz(h), shape=(max(n, 1), 3))[:n]
        cl = np.empty(n, dtype=CLUSTER_DTYPE)
        cl["x"], cl["y"], cl["z"] = xyz[:, 0], xyz[:, 1], xyz[:, 2]
        cl["row"] = np.ctypeslib.as_array(lib.synth_row(h), shape=(max(n, 1),))[:n]
        truth = np.ctypeslib.as_array(lib.synth_truth(h), shape=(max(n, 1),))[:n].copy()
        so = np.ctypeslib.as_array(lib.synth_sector_offsets(h), shape=(ns + 1,)).copy()
        tp = np.ctypeslib.as_array(lib.synth_track_par(h), shape=(max(nt, 1), 8))[:nt].copy()
    finally:
        lib.synth_free(h)
    return Frame(cl, so, truth, tp, ns, name or "custom")


def permute_within_sectors(fr: Frame, seed: int) -> tuple[Frame, np.ndarray]:
    """Return a frame with clusters shuffled inside each sector and the permutation p
    (new[i] = old[p[i]]).  Drives the order-independence pin (P5)."""
    rng = np.random.default_rng(seed)
    p = np.arange(fr.n)
    for s in range(fr.n_sectors):
        b, e = int(fr.sector_offsets[s]), int(fr.sector_offsets[s + 1])
        p[b:e] = b + rng.permutation(e - b)
    return Frame(fr.clusters[p].copy(), fr.sector_offsets.copy(), fr.truth[p].copy(), fr.track_par, fr.n_sectors,
                 fr.name + "+perm"), p
