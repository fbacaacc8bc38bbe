"""ctypes wrapper of oracle/tpcca_oracle.cpp (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpcca_oracle.cpp")

# DESIGN.md Table A defaults (the oracle keeps its own copy; the product's live in binding.py)
DEFAULT_PARAMS = dict(
    sigma_y=0.1, sigma_z=0.15,
    nbr_dydx=1.5, nbr_dzdx=1.5, nbr_margin_y=0.5, nbr_margin_z=0.75, triplet_cut=18.0,
    cov0=(1.0, 1.0, 0.25, 1.0, 100.0),
    pick_cut=16.0, reject_cut=25.0, max_gap=5, edge_margin=3.0, max_sinphi=0.95,
    min_seed_hits=4, min_tracklet_hits=10, min_track_hits=10, qual_scale=1000.0,
    tan_half_angle=float(np.tan(np.deg2rad(10.0))),
)


# DESIGN.md section 12 Table B defaults of the merger (the product keeps its own copy in binding.py)
DEFAULT_MERGE_PARAMS = dict(merge_chi2_cut=50.0, merge_dz_max=30.0, merge_edge_dist=10.0, merge_row_back=2,
                            merge_row_fwd=8, fit_reject_cut=30.0, shared_err_scale=2.0, ring=18)


DEFAULT_TIME_PARAMS = dict(vdrift=2.58, z_max=250.0)  # cm/us, cm (BASELINE.json config 4; TPC half length)


# DESIGN.md section 14 Table D defaults of the looper-leg finder and the cluster tags (the product keeps its own copy)
DEFAULT_LEG_PARAMS = dict(leg_min_qpt=4.0, leg_min_sinphi=0.5, leg_inner_min_sinphi=0.2, leg_apex_margin=2.0, leg_max_sector_gap=5,
                          leg_inner_max_sector_gap=9, leg_max_turn=2.9, leg_inner_max_turn=5.0, leg_centre_frac=0.05, leg_centre_abs=1.5, leg_radius_frac=0.2,
                          leg_dz_max=4.0, leg_dzds_tol=0.1, tag_qpt_low=20.0, tag_qpt_leg=5.0, tag_sinphi=0.8, ring=18)
TAG_LOW_PT, TAG_EXTRA_LEG, TAG_HIGH_INCLINATION = 1, 2, 4
# DESIGN.md section 15 Table E defaults of the fit through both legs of a turn
DEFAULT_LEG_FIT_PARAMS = dict(fit_rot_sinphi=0.5, fit_step_sinphi=0.7, fit_min_d=0.3, fit_reject_cut=30.0, shared_err_scale=2.0, ring=18)


class _FitParams(C.Structure):
    _fields_ = [("fit_rot_sinphi", C.c_float), ("fit_step_sinphi", C.c_float), ("fit_min_d", C.c_float), ("fit_reject_cut", C.c_float),
                ("shared_err_scale", C.c_float), ("ring", C.c_int32)]


class _LegParams(C.Structure):
    _fields_ = [("leg_min_qpt", C.c_float), ("leg_min_sinphi", C.c_float), ("leg_inner_min_sinphi", C.c_float),
                ("leg_apex_margin", C.c_float),
                ("leg_max_sector_gap", C.c_int32), ("leg_inner_max_sector_gap", C.c_int32), ("leg_max_turn", C.c_float),
                ("leg_inner_max_turn", C.c_float), ("leg_centre_frac", C.c_float),
                ("leg_centre_abs", C.c_float), ("leg_radius_frac", C.c_float), ("leg_dz_max", C.c_float),
                ("leg_dzds_tol", C.c_float), ("tag_qpt_low", C.c_float), ("tag_qpt_leg", C.c_float),
                ("tag_sinphi", C.c_float), ("ring", C.c_int32)]


def _leg_params(legs) -> "_LegParams":
    d = dict(DEFAULT_LEG_PARAMS)
    if isinstance(legs, dict):
        d.update(legs)
    return _LegParams(**d)


class _MergeParams(C.Structure):
    _fields_ = [("merge_chi2_cut", C.c_float), ("merge_dz_max", C.c_float), ("merge_edge_dist", C.c_float),
                ("merge_row_back", C.c_int32), ("merge_row_fwd", C.c_int32),
                ("fit_reject_cut", C.c_float), ("shared_err_scale", C.c_float), ("ring", C.c_int32)]


class _Params(C.Structure):
    _fields_ = [
        ("sigma_y", C.c_float), ("sigma_z", C.c_float),
        ("nbr_dydx", C.c_float), ("nbr_dzdx", C.c_float), ("nbr_margin_y", C.c_float), ("nbr_margin_z", C.c_float),
        ("triplet_cut", C.c_float), ("cov0", C.c_float * 5),
        ("pick_cut", C.c_float), ("reject_cut", C.c_float), ("max_gap", C.c_int32),
        ("edge_margin", C.c_float), ("max_sinphi", C.c_float),
        ("min_seed_hits", C.c_int32), ("min_tracklet_hits", C.c_int32), ("min_track_hits", C.c_int32),
        ("qual_scale", C.c_float), ("tan_half_angle", C.c_float),
    ]


TRACK_DTYPE = np.dtype([
    ("sector", "<i4"), ("first_row", "<i4"), ("last_row", "<i4"), ("n_hits", "<i4"),
    ("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("sinphi", "<f4"), ("dzds", "<f4"), ("qpt", "<f4"),
    ("cov", "<f4", (15,)), ("chi2", "<f4"), ("ndf", "<i4"), ("pad", "<i4", (5,)),
])
assert TRACK_DTYPE.itemsize == 128


def _host_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


def build(opt: str = "-O2", force: bool = False) -> str:
    # TPCCA_ORACLE_CXXFLAGS: extra compiler flags for a checking build of the oracle (e.g. -fsanitize=address,undefined,
    # with libasan preloaded into python; profiles/r2_sanitizer.md has the command)
    extra = os.environ.get("TPCCA_ORACLE_CXXFLAGS", "").split()
    so = os.path.join(_HERE, f"libtpcca_oracle{opt.replace('-', '_')}{'_chk' if extra else ''}.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        # -mfma only makes std::fma a single instruction where the host has it (the result is the same correctly
        # rounded value either way); -ffp-contract=off: the compiler itself never fuses
        hw = ["-mfma"] if _host_has_fma() else []
        subprocess.check_call(["g++", opt, "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"] + hw
                              + extra + ["-o", so, _SRC])
    return so


_libs: dict = {}


def _load(opt: str = "-O2"):
    if opt not in _libs:
        lib = C.CDLL(build(opt))
        lib.orc_track.restype = C.c_void_p
        lib.orc_track.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_float, C.POINTER(_Params), C.c_void_p,
                                  C.c_int64, C.c_void_p, C.c_int32]
        lib.orc_free.argtypes = [C.c_void_p]
        for name in ("orc_n_start", "orc_n_tracks"):
            getattr(lib, name).restype = C.c_int64
            getattr(lib, name).argtypes = [C.c_void_p]
        for name in ("orc_link_up_raw", "orc_link_down_raw", "orc_link_up", "orc_link_down", "orc_start_hits",
                     "orc_row_hit", "orc_assignment", "orc_tracks", "orc_track_tracklet"):
            getattr(lib, name).restype = C.c_void_p
            getattr(lib, name).argtypes = [C.c_void_p]
        lib.orc_tracklets.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.orc_merge.restype = C.c_int64
        lib.orc_merge.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_float, C.POINTER(_Params), C.c_void_p,
                                  C.POINTER(_MergeParams)]
        for name in ("orc_merged", "orc_track_merged", "orc_link_next", "orc_shared"):
            getattr(lib, name).restype = C.c_void_p
            getattr(lib, name).argtypes = [C.c_void_p]
        lib.orc_outer.argtypes = [C.c_void_p, C.c_void_p]
        lib.orc_legs.restype = C.c_int64
        lib.orc_legs.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_float, C.POINTER(_Params), C.c_void_p,
                                 C.POINTER(_LegParams)]
        for name in ("orc_leg_partner", "orc_leg_partner_in", "orc_leg_first", "orc_cluster_tags"):
            getattr(lib, name).restype = C.c_void_p
            getattr(lib, name).argtypes = [C.c_void_p]
        lib.orc_fit_legs.restype = C.c_int64
        lib.orc_fit_legs.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_float, C.POINTER(_Params), C.c_void_p,
                                     C.POINTER(_FitParams)]
        lib.orc_leg_fits.restype = C.c_void_p
        lib.orc_leg_fits.argtypes = [C.c_void_p]
        lib.orc_angle_upper.restype = C.c_float
        lib.orc_angle_upper.argtypes = [C.c_float, C.c_float]
        lib.orc_leg_end.argtypes = [C.c_int32, C.c_void_p, C.c_float, C.c_float, C.POINTER(_LegParams), C.c_void_p]
        lib.orc_leg_pair.restype = C.c_float
        lib.orc_leg_pair.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.POINTER(_LegParams)]
        lib.orc_time_estimate.argtypes = [C.c_void_p, C.c_int32, C.c_float, C.c_void_p, C.c_float, C.c_float, C.c_void_p]
        lib.orc_time_estimate_state.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_int32, C.c_float,
                                                C.c_float, C.c_void_p]
        lib.orc_rotate.restype = C.c_int32
        lib.orc_rotate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_int32, C.c_float, C.c_float]
        lib.orc_kf_transport.restype = C.c_int32
        lib.orc_kf_transport.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float]
        lib.orc_kf_update.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_float]
        lib.orc_refit_hits.restype = C.c_int32
        lib.orc_refit_hits.argtypes = [C.c_int32, C.c_void_p, C.c_float, C.c_float, C.POINTER(_Params), C.c_void_p]
        _libs[opt] = lib
    return _libs[opt]


def _params(p: dict | None) -> _Params:
    d = dict(DEFAULT_PARAMS)
    if p:
        d.update(p)
    cp = _Params()
    for k, v in d.items():
        if k == "cov0":
            cp.cov0 = (C.c_float * 5)(*v)
        else:
            setattr(cp, k, v)
    return cp


@dataclass
class OracleResult:
    link_up_raw: np.ndarray
    link_down_raw: np.ndarray
    link_up: np.ndarray
    link_down: np.ndarray
    start_hits: np.ndarray
    row_hit: np.ndarray          # (n_tracklets, n_rows) input indices or -1
    tracklet_ints: np.ndarray    # (n_tracklets, 4): valid, first_row, last_row, n_hits
    tracklet_floats: np.ndarray  # (n_tracklets, 23): x, p5, C15, chi2, z_ref
    assignment: np.ndarray
    tracks: np.ndarray           # TRACK_DTYPE
    track_tracklet: np.ndarray
    shared: np.ndarray = None        # uint8 per cluster (O6 / B7)
    outer: np.ndarray = None         # (n_tracks, 21): outer end x, y, z, sinphi, dzds, qpt, cov15 (O8)
    merged: np.ndarray = None        # TRACK_DTYPE, merged tracks (O10); only with merge=...
    track_merged: np.ndarray = None  # sector track -> merged track
    link_next: np.ndarray = None     # sector track -> continuation or -1 (O9)
    leg_partner: np.ndarray = None   # merged track -> merged track joined at the outer turning point or -1 (O12); with legs=...
    leg_partner_in: np.ndarray = None  # merged track -> merged track joined through the inner region or -1
    leg_first: np.ndarray = None     # merged track: 1 first / only leg, 0 additional leg
    cluster_tags: np.ndarray = None  # uint8 per cluster: TAG_* bits (O13)
    leg_fits: np.ndarray = None      # TRACK_DTYPE, one fit per pair of legs joined at a turning point (O14); with leg_fit=...
    time_sector: np.ndarray = None   # (n_tracks, 4): z_dca, z_shift, t0_us, dca_xy (O11); only with time=...
    time_merged: np.ndarray = None   # (n_merged, 4)


def _arr(ptr, n, dtype):
    if n == 0 or not ptr:
        return np.zeros(0, dtype=dtype)
    buf = (C.c_char * (n * np.dtype(dtype).itemsize)).from_address(ptr)
    return np.frombuffer(buf, dtype=dtype).copy()


def track(clusters: np.ndarray, sector_offsets: np.ndarray, row_x: np.ndarray, bz: float = 0.5,
          params: dict | None = None, brute: bool = False, opt: str = "-O2", merge: dict | bool | None = None,
          time: dict | bool | None = None, legs: dict | bool | None = None, leg_fit: dict | bool | None = None) -> OracleResult:
    """Steps O1-O7 on one frame.  `clusters`: structured (x,y,z f32,row i32); returns input-index-space results.
    merge: True or a dict of DEFAULT_MERGE_PARAMS overrides -> also steps O8-O10 (sector-segment merger + final fit).
    legs: True or a dict of DEFAULT_LEG_PARAMS overrides -> also O12-O13 (looper legs, cluster tags); needs merge.
    time: True or dict(vdrift=..., z_max=...) -> also O11 (z / time estimate) for the sector and, with merge, merged tracks."""
    lib = _load(opt)
    cl = np.ascontiguousarray(clusters)
    assert cl.dtype.itemsize == 16
    so = np.ascontiguousarray(sector_offsets, dtype=np.int32)
    rx = np.ascontiguousarray(row_x, dtype=np.float32)
    n, ns, nr = cl.shape[0], so.shape[0] - 1, rx.shape[0]
    cp = _params(params)
    h = lib.orc_track(ns, nr, rx.ctypes.data, bz, C.byref(cp), cl.ctypes.data, n, so.ctypes.data, int(brute))
    try:
        nt, ntr = lib.orc_n_start(h), lib.orc_n_tracks(h)
        ti = np.zeros((nt, 4), np.int32)
        tf = np.zeros((nt, 23), np.float32)
        if nt:
            lib.orc_tracklets(h, ti.ctypes.data, tf.ctypes.data)
        res = OracleResult(
            _arr(lib.orc_link_up_raw(h), n, np.int32), _arr(lib.orc_link_down_raw(h), n, np.int32),
            _arr(lib.orc_link_up(h), n, np.int32), _arr(lib.orc_link_down(h), n, np.int32),
            _arr(lib.orc_start_hits(h), nt, np.int32),
            _arr(lib.orc_row_hit(h), nt * nr, np.int32).reshape(nt, nr),
            ti, tf,
            _arr(lib.orc_assignment(h), n, np.int32),
            _arr(lib.orc_tracks(h), ntr, TRACK_DTYPE), _arr(lib.orc_track_tracklet(h), ntr, np.int32))
        res.shared = _arr(lib.orc_shared(h), n, np.uint8)
        res.outer = np.zeros((ntr, 21), np.float32)
        if ntr:
            lib.orc_outer(h, res.outer.ctypes.data)
        if merge:
            md = dict(DEFAULT_MERGE_PARAMS)
            if isinstance(merge, dict):
                md.update(merge)
            mp = _MergeParams(**md)
            nm = lib.orc_merge(h, nr, rx.ctypes.data, bz, C.byref(cp), cl.ctypes.data, C.byref(mp))
            res.merged = _arr(lib.orc_merged(h), nm, TRACK_DTYPE)
            res.track_merged = _arr(lib.orc_track_merged(h), ntr, np.int32)
            res.link_next = _arr(lib.orc_link_next(h), ntr, np.int32)
        if legs:
            assert merge, "legs need the merged tracks"
            lp = _leg_params(legs)
            lib.orc_legs(h, nr, rx.ctypes.data, bz, C.byref(cp), cl.ctypes.data, C.byref(lp))
            res.leg_partner = _arr(lib.orc_leg_partner(h), len(res.merged), np.int32)
            res.leg_partner_in = _arr(lib.orc_leg_partner_in(h), len(res.merged), np.int32)
            res.leg_first = _arr(lib.orc_leg_first(h), len(res.merged), np.uint8)
            res.cluster_tags = _arr(lib.orc_cluster_tags(h), n, np.uint8)
        if leg_fit:
            assert legs, "the pair fit needs the leg links"
            fd = dict(DEFAULT_LEG_FIT_PARAMS)
            if isinstance(leg_fit, dict):
                fd.update(leg_fit)
            fp = _FitParams(**fd)
            nf = lib.orc_fit_legs(h, nr, rx.ctypes.data, bz, C.byref(cp), cl.ctypes.data, C.byref(fp))
            res.leg_fits = _arr(lib.orc_leg_fits(h), nf, TRACK_DTYPE)
        if time:
            td = dict(DEFAULT_TIME_PARAMS)
            if isinstance(time, dict):
                td.update(time)
            res.time_sector = np.zeros((ntr, 4), np.float32)
            if ntr:
                lib.orc_time_estimate(h, 0, bz, cl.ctypes.data, td["vdrift"], td["z_max"], res.time_sector.ctypes.data)
            if merge:
                res.time_merged = np.zeros((len(res.merged), 4), np.float32)
                if len(res.merged):
                    lib.orc_time_estimate(h, 1, bz, cl.ctypes.data, td["vdrift"], td["z_max"], res.time_merged.ctypes.data)
        return res
    finally:
        lib.orc_free(h)


def kf_transport(x, p5, cov15, xnew, bz=0.5, max_sinphi=0.95, opt="-O2"):
    lib = _load(opt)
    xx = np.array([x], np.float32)
    p = np.array(p5, np.float32)
    c = np.array(cov15, np.float32)
    ok = lib.orc_kf_transport(xx.ctypes.data, p.ctypes.data, c.ctypes.data, xnew, bz, max_sinphi)
    return bool(ok), float(xx[0]), p, c


def rotate_frame(x, p5, cov15, sgn, tan_half_angle=DEFAULT_PARAMS["tan_half_angle"], bz=0.5, max_sinphi=0.95, opt="-O2"):
    """Frame change into the next (sgn = +1) or previous (sgn = -1) sector (B3)."""
    lib = _load(opt)
    xx = np.array([x], np.float32)
    p = np.array(p5, np.float32)
    c = np.array(cov15, np.float32)
    ok = lib.orc_rotate(xx.ctypes.data, p.ctypes.data, c.ctypes.data, tan_half_angle, sgn, bz, max_sinphi)
    return bool(ok), float(xx[0]), p, c


def time_estimate_state(state6, zmin_hits, zmax_hits, side, bz=0.5, vdrift=2.58, z_max=250.0, opt="-O2"):
    """O11 on one state (x, y, z, sinphi, dzds, qpt): returns (z_dca, z_shift, t0_us, dca_xy)."""
    lib = _load(opt)
    st = np.array(state6, np.float32)
    out = np.zeros(4, np.float32)
    lib.orc_time_estimate_state(st.ctypes.data, bz, zmin_hits, zmax_hits, side, vdrift, z_max, out.ctypes.data)
    return out


def kf_update(p5, cov15, chi2, ym, zm, sy2, sz2, opt="-O2"):
    lib = _load(opt)
    p = np.array(p5, np.float32)
    c = np.array(cov15, np.float32)
    ch = np.array([chi2], np.float32)
    lib.orc_kf_update(p.ctypes.data, c.ctypes.data, ch.ctypes.data, ym, zm, sy2, sz2)
    return p, c, float(ch[0])


def refit_hits(x, y, z, q0=0.0, bz=0.5, params=None, opt="-O2"):
    """O7 three-pass refit of a free-standing hit list (increasing x).  Returns (ok, out22)."""
    lib = _load(opt)
    n = len(x)
    cl = np.zeros(n, dtype=[("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("row", "<i4")])
    cl["x"], cl["y"], cl["z"] = x, y, z
    out = np.zeros(22, np.float32)
    cp = _params(params)
    ok = lib.orc_refit_hits(n, cl.ctypes.data, q0, bz, C.byref(cp), out.ctypes.data)
    return bool(ok), out


def angle_upper(y, x, opt="-O2"):
    """O12: the angle of (x, y), y > 0, in (0, pi) by the fp32 polynomial of DESIGN.md section 14."""
    return float(_load(opt).orc_angle_upper(float(y), float(x)))


def leg_end(state7, bz=0.5, x_last=245.0, legs=None, opt="-O2", sig=1):
    """O12 on one end (sector, x, y, z, sinphi, dzds, qpt), sig = +1 outer / -1 inner: returns (candidate, R, xc, yc, cos phi)."""
    lib = _load(opt)
    st = np.array(state7, np.float32)
    out = np.zeros(5, np.float32)
    lp = _leg_params(legs)
    lib.orc_leg_end(sig, st.ctypes.data, bz, x_last, C.byref(lp), out.ctypes.data)
    return bool(out[0]), float(out[1]), float(out[2]), float(out[3]), float(out[4])


def leg_pair(a7, b7, bz=0.5, x_last=245.0, tan_half_angle=DEFAULT_PARAMS["tan_half_angle"], legs=None, opt="-O2", sig=1):
    """O12 pair score of two ends of one kind (sig = +1 outer, -1 inner; a7 plays the lower id), negative = no match."""
    lib = _load(opt)
    a, b = np.array(a7, np.float32), np.array(b7, np.float32)
    lp = _leg_params(legs)
    return float(lib.orc_leg_pair(sig, a.ctypes.data, b.ctypes.data, bz, x_last, tan_half_angle, C.byref(lp)))
