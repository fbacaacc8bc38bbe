"""Thin ctypes binding of include/tpcca.h (argument marshalling only).

PyTorch supplies device memory and streams; every step of the path runs in the CUDA kernels of
`csrc/`.  There is no fallback: a missing or unloadable libtpcca.so raises at import of `load()`.
Names follow the C-ABI: tpcca_init / tpcca_track / tpcca_track_host / tpcca_get_intermediate / tpcca_free.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpcca.so")

LINK_UP_RAW, LINK_DOWN_RAW, LINK_UP, LINK_DOWN, START_HITS, TRACKLET_ROW_HITS, TRACKLET_INTS, TRACKLET_FLOATS, \
    TRACK_TRACKLET, TRACK_OUTER, SHARED, MERGE_LINK_NEXT = range(12)
STAGES = ("grid", "neighbours", "clean_start", "tracklets", "select", "refit")
KERNELS = ("k_slice_scatter", "k_slice_sort", "k_neighbours", "k_clean", "k_tl_e1", "k_tl_e2", "k_tl_e3a", "k_tl_e3b",
           "k_tracklet_weights", "k_select_own", "k_assign", "k_refit")

CLUSTER_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("row", "<i4")])
TRACK_DTYPE = np.dtype([
    ("sector", "<i4"), ("first_row", "<i4"), ("last_row", "<i4"), ("n_hits", "<i4"),
    ("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("sinphi", "<f4"), ("dzds", "<f4"), ("qpt", "<f4"),
    ("cov", "<f4", (15,)), ("chi2", "<f4"), ("ndf", "<i4"), ("pad", "<i4", (5,)),
])
HEADER_DTYPE = np.dtype([("n_tracks", "<i4"), ("n_tracklets", "<i4"), ("n_start_hits", "<i4"), ("status", "<i4")])


class Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float)]


class Params(C.Structure):
    _fields_ = [
        ("sigma_y", C.c_float), ("sigma_z", C.c_float),
        ("nbr_dydx", C.c_float), ("nbr_dzdx", C.c_float), ("nbr_margin_y", C.c_float), ("nbr_margin_z", C.c_float),
        ("triplet_cut", C.c_float), ("cov0", C.c_float * 5),
        ("pick_cut", C.c_float), ("reject_cut", C.c_float), ("max_gap", C.c_int32),
        ("edge_margin", C.c_float), ("max_sinphi", C.c_float),
        ("min_seed_hits", C.c_int32), ("min_tracklet_hits", C.c_int32), ("min_track_hits", C.c_int32),
        ("qual_scale", C.c_float),
        ("grid_bin_y", C.c_float), ("grid_bin_z_min", C.c_float), ("grid_bins_per_cluster", C.c_float),
        ("max_clusters", C.c_int64), ("max_tracklets", C.c_int32), ("max_tracks", C.c_int32),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
    ]


class MergeParams(C.Structure):
    _fields_ = [("merge_chi2_cut", C.c_float), ("merge_dz_max", C.c_float), ("merge_edge_dist", C.c_float),
                ("merge_row_back", C.c_int32), ("merge_row_fwd", C.c_int32),
                ("fit_reject_cut", C.c_float), ("shared_err_scale", C.c_float), ("ring", C.c_int32)]


class LegParams(C.Structure):
    _fields_ = [("leg_min_qpt", C.c_float), ("leg_min_sinphi", C.c_float), ("leg_inner_min_sinphi", C.c_float),
                ("leg_apex_margin", C.c_float), ("leg_max_sector_gap", C.c_int32), ("leg_inner_max_sector_gap", C.c_int32),
                ("leg_max_turn", C.c_float), ("leg_inner_max_turn", C.c_float), ("leg_centre_frac", C.c_float),
                ("leg_centre_abs", C.c_float), ("leg_radius_frac", C.c_float), ("leg_dz_max", C.c_float),
                ("leg_dzds_tol", C.c_float), ("tag_qpt_low", C.c_float), ("tag_qpt_leg", C.c_float),
                ("tag_sinphi", C.c_float), ("ring", C.c_int32)]


TAG_LOW_PT, TAG_EXTRA_LEG, TAG_HIGH_INCLINATION = 1, 2, 4


class LegFitParams(C.Structure):
    _fields_ = [("fit_rot_sinphi", C.c_float), ("fit_step_sinphi", C.c_float), ("fit_min_d", C.c_float),
                ("fit_reject_cut", C.c_float), ("shared_err_scale", C.c_float), ("ring", C.c_int32)]

_lib = None


def load():
    """Load libtpcca.so (built in-tree by build.py).  Raises if it is missing: no CPU fallback exists."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} not built: run `python -m paper_1811_11481_b200.build` "
                               "(or __graft_entry__.build()); this package has no CPU fallback")
        lib = C.CDLL(_SO)
        lib.tpcca_default_params.argtypes = [C.POINTER(Params)]
        lib.tpcca_workspace_bytes.restype = C.c_size_t
        lib.tpcca_workspace_bytes.argtypes = [C.POINTER(Geometry), C.POINTER(Params)]
        lib.tpcca_init.restype = C.c_void_p
        lib.tpcca_init.argtypes = [C.POINTER(Geometry), C.c_float, C.POINTER(Params)]
        for name in ("tpcca_track", "tpcca_track_host", "tpcca_track_host_async"):
            fn = getattr(lib, name)
            fn.restype = C.c_int
            fn.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.tpcca_default_merge_params.argtypes = [C.POINTER(MergeParams)]
        lib.tpcca_merge.restype = C.c_int
        lib.tpcca_merge.argtypes = [C.c_void_p, C.POINTER(MergeParams), C.c_void_p, C.c_void_p, C.c_void_p]
        lib.tpcca_default_leg_params.argtypes = [C.POINTER(LegParams)]
        lib.tpcca_find_legs.restype = C.c_int
        lib.tpcca_find_legs.argtypes = [C.c_void_p, C.POINTER(LegParams), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_void_p]
        lib.tpcca_default_leg_fit_params.argtypes = [C.POINTER(LegFitParams)]
        lib.tpcca_fit_legs.restype = C.c_int
        lib.tpcca_fit_legs.argtypes = [C.c_void_p, C.POINTER(LegFitParams), C.c_void_p, C.c_void_p]
        lib.tpcca_estimate_time.restype = C.c_int
        lib.tpcca_estimate_time.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.tpcca_wait.restype = C.c_int
        lib.tpcca_wait.argtypes = [C.c_void_p]
        lib.tpcca_get_intermediate.restype = C.c_int
        lib.tpcca_get_intermediate.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
        lib.tpcca_debug_workspace_layout.restype = C.c_int
        lib.tpcca_debug_workspace_layout.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        lib.tpcca_set_profiling.argtypes = [C.c_void_p, C.c_int]
        lib.tpcca_set_debug.argtypes = [C.c_void_p, C.c_int]
        lib.tpcca_get_stage_ms.restype = C.c_int
        lib.tpcca_get_stage_ms.argtypes = [C.c_void_p, C.c_void_p]
        lib.tpcca_get_kernel_ms.restype = C.c_int
        lib.tpcca_get_kernel_ms.argtypes = [C.c_void_p, C.c_void_p]
        lib.tpcca_get_stats.restype = C.c_int
        lib.tpcca_get_stats.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.tpcca_last_launch_count.restype = C.c_int
        lib.tpcca_last_launch_count.argtypes = [C.c_void_p]
        lib.tpcca_clean_links_static.restype = C.c_int
        lib.tpcca_clean_links_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                                 C.c_void_p, C.c_void_p]
        lib.tpcca_last_error.restype = C.c_char_p
        lib.tpcca_free.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def default_leg_fit_params() -> LegFitParams:
    p = LegFitParams()
    load().tpcca_default_leg_fit_params(C.byref(p))
    return p


def default_leg_params() -> LegParams:
    p = LegParams()
    load().tpcca_default_leg_params(C.byref(p))
    return p


def default_merge_params() -> MergeParams:
    p = MergeParams()
    load().tpcca_default_merge_params(C.byref(p))
    return p


def default_params() -> Params:
    p = Params()
    load().tpcca_default_params(C.byref(p))
    return p


class TpccaError(RuntimeError):
    pass


STATIC_MAX_CLUSTERS = 1 << 25  # TPCCA_STATIC_MAX_CLUSTERS of include/tpcca.h


def clean_links_static(link_up_raw, link_down_raw, n: int, out_link_up, out_link_down, out_start_hits, out_n_start,
                       stream: int | None = None) -> None:
    """tpcca_clean_links_static: mutual links and chain starts from raw links, for callers that cannot allocate device
    memory (no workspace, no cudaMalloc inside: the scratch is a fixed array in the library, so n <= STATIC_MAX_CLUSTERS and
    calls that overlap on one GPU race -- see include/tpcca.h).  All arguments are CUDA int32 tensors the caller made
    (marshalling only); enqueued on `stream` (default: torch's current stream), returns without waiting."""
    import torch
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    ptr = lambda t: t.data_ptr() if t is not None and t.numel() else None
    rc = lib.tpcca_clean_links_static(ptr(link_up_raw), ptr(link_down_raw), int(n), stream, ptr(out_link_up),
                                      ptr(out_link_down), ptr(out_start_hits), ptr(out_n_start))
    if rc != 0:
        raise TpccaError(f"tpcca error {rc}: {lib.tpcca_last_error().decode()}")


class Tracker:
    """tpcca_init ... tpcca_free around one handle; owns the workspace tensor (caller-owned memory of the C-ABI)."""

    def __init__(self, row_x: np.ndarray, n_sectors: int = 36, bz: float = 0.5, max_clusters: int = 1 << 20,
                 max_tracklets: int | None = None, max_tracks: int | None = None,
                 tan_half_angle: float = float(np.tan(np.deg2rad(10.0))), device: str = "cuda:0",
                 poison: int | None = None, **params):
        import torch
        self.torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise TpccaError("no CUDA device: the tpcca path has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._rx = np.ascontiguousarray(row_x, dtype=np.float32)
        self.n_rows, self.n_sectors = int(self._rx.shape[0]), int(n_sectors)
        self.geo = Geometry(self.n_sectors, self.n_rows, self._rx.ctypes.data_as(C.POINTER(C.c_float)), tan_half_angle)
        p = default_params()
        for k, v in params.items():
            if k == "cov0":
                p.cov0 = (C.c_float * 5)(*v)
            elif hasattr(p, k):
                setattr(p, k, v)
            else:
                raise TypeError(f"unknown parameter {k}")
        p.max_clusters = int(max_clusters)
        p.max_tracklets = int(max_tracklets if max_tracklets is not None else max(1024, max_clusters // 8))
        p.max_tracks = int(max_tracks if max_tracks is not None else p.max_tracklets)
        nbytes = self.lib.tpcca_workspace_bytes(C.byref(self.geo), C.byref(p))
        if nbytes == 0:
            raise TpccaError(self.lib.tpcca_last_error().decode())
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        if poison is not None:  # tests: scratch must never be read before it is written
            self.workspace.fill_(int(poison))
        base = (self.workspace.data_ptr() + 255) & ~255
        p.workspace, p.workspace_bytes = base, nbytes
        self.params = p
        self.max_clusters, self.max_tracklets, self.max_tracks = p.max_clusters, p.max_tracklets, p.max_tracks
        self.h = self.lib.tpcca_init(C.byref(self.geo), float(bz), C.byref(p))
        if not self.h:
            raise TpccaError(self.lib.tpcca_last_error().decode())
        self.out_tracks = torch.empty(16 + 128 * self.max_tracks, dtype=torch.uint8, device=self.device)
        self.out_assign = torch.empty(max(1, self.max_clusters), dtype=torch.int32, device=self.device)
        self.n = 0

    def close(self):
        if getattr(self, "h", None):
            self.lib.tpcca_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise TpccaError(f"tpcca error {rc}: {self.lib.tpcca_last_error().decode()}")

    def _stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    # ---- device-resident call: clusters is a torch uint8/float32 CUDA tensor holding n 16-byte records
    def track(self, clusters_dev, n: int, sector_offsets: np.ndarray):
        so = np.ascontiguousarray(sector_offsets, dtype=np.int32)
        assert so.shape[0] == self.n_sectors + 1
        self._so = so
        self.n = int(n)
        self._check(self.lib.tpcca_track(self.h, clusters_dev.data_ptr() if n else None, n, so.ctypes.data,
                                         self._stream(), self.out_tracks.data_ptr(), self.out_assign.data_ptr()))

    def upload(self, clusters: np.ndarray):
        t = self.torch.from_numpy(np.ascontiguousarray(clusters).view(np.uint8).reshape(-1))
        return t.to(self.device)

    def header(self) -> dict:
        h = self.out_tracks[:16].cpu().numpy().view(HEADER_DTYPE)[0]
        return {k: int(h[k]) for k in HEADER_DTYPE.names}

    def tracks(self) -> np.ndarray:
        nt = self.header()["n_tracks"]
        return self.out_tracks[16:16 + 128 * nt].cpu().numpy().view(TRACK_DTYPE).copy()

    def assignment(self) -> np.ndarray:
        return self.out_assign[:self.n].cpu().numpy().copy()

    # ---- end to end from host buffers (pinned numpy-backed torch tensors recommended)
    def track_host(self, clusters_host, n: int, sector_offsets: np.ndarray, out_tracks_host, out_assign_host):
        so = np.ascontiguousarray(sector_offsets, dtype=np.int32)
        self._so = so
        self.n = int(n)
        self._check(self.lib.tpcca_track_host(self.h, clusters_host.data_ptr() if n else None, n, so.ctypes.data,
                                              self._stream(), out_tracks_host.data_ptr(), out_assign_host.data_ptr()))

    def track_host_async(self, clusters_host, n: int, sector_offsets: np.ndarray, out_tracks_host, out_assign_host):
        """tpcca_track_host_async: enqueue only; at most two frames in flight; pair every call with wait()."""
        so = np.ascontiguousarray(sector_offsets, dtype=np.int32)
        self._so = so
        self.n = int(n)
        self._check(self.lib.tpcca_track_host_async(self.h, clusters_host.data_ptr() if n else None, n, so.ctypes.data,
                                                    self._stream(), out_tracks_host.data_ptr(),
                                                    out_assign_host.data_ptr()))

    def wait(self):
        self._check(self.lib.tpcca_wait(self.h))

    def intermediate(self, what: int) -> np.ndarray:
        torch = self.torch
        hd = self.header()
        ns, nt = hd["n_start_hits"], hd["n_tracks"]
        if what <= LINK_DOWN or what == SHARED:
            shape, dt = (self.n,), torch.int32
        elif what == TRACK_OUTER:
            shape, dt = (nt, 24), torch.float32
        elif what == START_HITS:
            shape, dt = (ns,), torch.int32
        elif what == TRACKLET_ROW_HITS:
            shape, dt = (ns, self.n_rows), torch.int32
        elif what == TRACKLET_INTS:
            shape, dt = (ns, 4), torch.int32
        elif what == TRACKLET_FLOATS:
            shape, dt = (ns, 8), torch.float32
        else:
            shape, dt = (nt,), torch.int32
        numel = int(np.prod(shape))
        dst = torch.empty(max(4, numel), dtype=dt, device=self.device)
        self._check(self.lib.tpcca_get_intermediate(self.h, what, dst.data_ptr(), dst.numel() * 4, self._stream()))
        return dst[:numel].reshape(shape).cpu().numpy()

    # ---- sector-segment merger + final fit on the results of the last track() (tpcca_merge)
    def merge(self, **params):
        torch = self.torch
        mp = default_merge_params()
        for k, v in params.items():
            if not hasattr(mp, k):
                raise TypeError(f"unknown merge parameter {k}")
            setattr(mp, k, v)
        if getattr(self, "out_merged", None) is None:
            self.out_merged = torch.empty(16 + 128 * self.max_tracks, dtype=torch.uint8, device=self.device)
            self.out_track_merged = torch.empty(max(1, self.max_tracks), dtype=torch.int32, device=self.device)
        self._check(self.lib.tpcca_merge(self.h, C.byref(mp), self._stream(), self.out_merged.data_ptr(),
                                         self.out_track_merged.data_ptr()))

    def merged_header(self) -> dict:
        h = self.out_merged[:16].cpu().numpy().view(HEADER_DTYPE)[0]
        return dict(n_merged=int(h["n_tracks"]), n_links=int(h["n_tracklets"]), n_fit_failed=int(h["n_start_hits"]),
                    status=int(h["status"]))

    def merged(self) -> np.ndarray:
        nm = self.merged_header()["n_merged"]
        return self.out_merged[16:16 + 128 * nm].cpu().numpy().view(TRACK_DTYPE).copy()

    def track_merged(self) -> np.ndarray:
        return self.out_track_merged[:self.header()["n_tracks"]].cpu().numpy().copy()

    # ---- looper legs and cluster tags on the results of the last merge() (tpcca_find_legs)
    def find_legs_enqueue(self, **params):
        """tpcca_find_legs, enqueue only (results stay in out_leg_partner / out_leg_first / out_tags / out_leg_summary)."""
        torch = self.torch
        lp = default_leg_params()
        for k, v in params.items():
            if not hasattr(lp, k):
                raise TypeError(f"unknown leg parameter {k}")
            setattr(lp, k, v)
        n = max(1, int(self.n))
        if getattr(self, "out_leg_partner", None) is None:
            self.out_leg_partner = torch.empty(max(1, self.max_tracks), dtype=torch.int32, device=self.device)
            self.out_leg_partner_in = torch.empty(max(1, self.max_tracks), dtype=torch.int32, device=self.device)
            self.out_leg_first = torch.empty(max(1, self.max_tracks), dtype=torch.uint8, device=self.device)
            self.out_leg_summary = torch.empty(8, dtype=torch.int32, device=self.device)
        if getattr(self, "out_tags", None) is None or self.out_tags.numel() < n:
            self.out_tags = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._check(self.lib.tpcca_find_legs(self.h, C.byref(lp), self._stream(), self.out_leg_partner.data_ptr(),
                                             self.out_leg_partner_in.data_ptr(), self.out_leg_first.data_ptr(),
                                             self.out_tags.data_ptr(), self.out_leg_summary.data_ptr()))

    def find_legs(self, **params):
        """Returns (leg_partner[n_merged], leg_partner_inner[n_merged], leg_first[n_merged], cluster_tags[n], summary dict)."""
        self.find_legs_enqueue(**params)
        nm = self.merged_header()["n_merged"]
        sm = self.out_leg_summary.cpu().numpy()
        return (self.out_leg_partner[:nm].cpu().numpy().copy(), self.out_leg_partner_in[:nm].cpu().numpy().copy(),
                self.out_leg_first[:nm].cpu().numpy().copy(), self.out_tags[:int(self.n)].cpu().numpy().copy(),
                dict(n_links_outer=int(sm[0]), n_links_inner=int(sm[1]), n_tag_low_pt=int(sm[2]), n_tag_extra_leg=int(sm[3]),
                     n_tag_high_inclination=int(sm[4])))

    # ---- one fit through both legs of every pair joined at a turning point (tpcca_fit_legs), after find_legs()
    def fit_legs_enqueue(self, **params):
        torch = self.torch
        fp = default_leg_fit_params()
        for k, v in params.items():
            if not hasattr(fp, k):
                raise TypeError(f"unknown leg fit parameter {k}")
            setattr(fp, k, v)
        if getattr(self, "out_leg_fits", None) is None:
            self.out_leg_fits = torch.empty(16 + 128 * self.max_tracks, dtype=torch.uint8, device=self.device)
        self._check(self.lib.tpcca_fit_legs(self.h, C.byref(fp), self._stream(), self.out_leg_fits.data_ptr()))

    def fit_legs(self, **params) -> tuple:
        """Returns (records TRACK_DTYPE[n_pairs], n_failed)."""
        self.fit_legs_enqueue(**params)
        h = self.out_leg_fits[:16].cpu().numpy().view(HEADER_DTYPE)[0]
        n = int(h["n_tracks"])
        return self.out_leg_fits[16:16 + 128 * n].cpu().numpy().view(TRACK_DTYPE).copy(), int(h["n_tracklets"])

    def estimate_time(self, vdrift: float = 2.58, z_max: float = 250.0, merged: bool = True):
        """tpcca_estimate_time: (n_tracks, 4) and, after merge(), (n_merged, 4) arrays of z_dca, z_shift, t0_us, dca_xy."""
        torch = self.torch
        ts = torch.empty(4 * max(1, self.max_tracks), dtype=torch.float32, device=self.device)
        tm = torch.empty(4 * max(1, self.max_tracks), dtype=torch.float32, device=self.device) if merged else None
        self._check(self.lib.tpcca_estimate_time(self.h, vdrift, z_max, self._stream(), ts.data_ptr(),
                                                 tm.data_ptr() if merged else None))
        nt = self.header()["n_tracks"]
        out_s = ts[:4 * nt].reshape(nt, 4).cpu().numpy()
        if not merged:
            return out_s, None
        nm = self.merged_header()["n_merged"]
        return out_s, tm[:4 * nm].reshape(nm, 4).cpu().numpy()

    def workspace_layout(self) -> list:
        """[(offset, bytes)] of every array carved out of the workspace (tpcca_debug_workspace_layout)."""
        out, i = [], 0
        off, nb = C.c_size_t(), C.c_size_t()
        while self.lib.tpcca_debug_workspace_layout(self.h, i, C.byref(off), C.byref(nb)) == 0:
            out.append((int(off.value), int(nb.value)))
            i += 1
        return out

    def set_debug(self, on: bool):
        self.lib.tpcca_set_debug(self.h, int(on))

    def set_profiling(self, on):
        """0 / False off, 1 / True stage events, 2 stage + per-kernel events."""
        self.lib.tpcca_set_profiling(self.h, int(on))

    def kernel_ms(self) -> dict:
        ms = (C.c_float * len(KERNELS))()
        self._check(self.lib.tpcca_get_kernel_ms(self.h, ms))
        return dict(zip(KERNELS, [float(v) for v in ms]))

    def stage_ms(self) -> dict:
        ms = (C.c_float * len(STAGES))()
        self._check(self.lib.tpcca_get_stage_ms(self.h, ms))
        return dict(zip(STAGES, [float(v) for v in ms]))

    def stats(self) -> dict:
        st = (C.c_int64 * 9)()
        self._check(self.lib.tpcca_get_stats(self.h, st, self._stream()))
        return dict(n_bins=int(st[0]), row_steps=int(st[1]), searches=int(st[2]), track_hits=int(st[3]),
                    tracklet_hits=int(st[4]), steps_e1=int(st[5]), steps_e2=int(st[6]), steps_e3a=int(st[7]),
                    steps_e3b=int(st[8]))

    def launch_count(self) -> int:
        return int(self.lib.tpcca_last_launch_count(self.h))
