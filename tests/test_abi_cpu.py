"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/tpcca.h declares,
sizes workspaces, validates arguments and refuses to run without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1811_11481_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "tpcca.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(tpcca_[a-z_]+)\s*\(", hdr))
    assert {"tpcca_init", "tpcca_track", "tpcca_free", "tpcca_track_host", "tpcca_get_intermediate", "tpcca_merge",
            "tpcca_track_host_async", "tpcca_wait", "tpcca_default_merge_params", "tpcca_get_kernel_ms",
            "tpcca_estimate_time", "tpcca_find_legs", "tpcca_default_leg_params", "tpcca_debug_workspace_layout",
            "tpcca_fit_legs", "tpcca_default_leg_fit_params"} <= names
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts_match_header():
    assert C.sizeof(binding.Params) % 8 == 0
    assert binding.TRACK_DTYPE.itemsize == 128 and binding.HEADER_DTYPE.itemsize == 16
    assert binding.CLUSTER_DTYPE.itemsize == 16
    p = binding.default_params()
    assert abs(p.triplet_cut - 18.0) < 1e-6 and p.min_track_hits == 10 and abs(p.cov0[4] - 100.0) < 1e-6
    assert p.max_gap == 5 and abs(p.grid_bins_per_cluster - 2.0) < 1e-6 and abs(p.grid_bin_y - 6.0) < 1e-6


def test_defaults_equal_oracle_defaults():
    """The product and the oracle keep separate copies of DESIGN.md Table A; they must agree."""
    import oracle
    p = binding.default_params()
    for k, v in oracle.DEFAULT_PARAMS.items():
        if k == "tan_half_angle":
            continue
        got = list(p.cov0) if k == "cov0" else getattr(p, k)
        assert np.allclose(got, v, rtol=1e-7), k


def test_merge_defaults_equal_oracle_defaults(lib):
    import oracle
    mp = binding.default_merge_params()
    for k, v in oracle.DEFAULT_MERGE_PARAMS.items():
        assert np.isclose(getattr(mp, k), v), k
    assert {f[0] for f in binding.MergeParams._fields_} == set(oracle.DEFAULT_MERGE_PARAMS)


def test_workspace_bytes_and_argument_checks(lib, row_x):
    rx = np.ascontiguousarray(row_x)
    g = binding.Geometry(36, 152, rx.ctypes.data_as(C.POINTER(C.c_float)), synth.TAN_HALF_ANGLE)
    p = binding.default_params()
    p.max_clusters, p.max_tracklets, p.max_tracks = 1 << 20, 1 << 17, 1 << 17
    b1 = lib.tpcca_workspace_bytes(C.byref(g), C.byref(p))
    p.max_clusters = 1 << 21
    b2 = lib.tpcca_workspace_bytes(C.byref(g), C.byref(p))
    assert 0 < b1 < b2 < (1 << 32)
    g.n_sectors = 0
    assert lib.tpcca_workspace_bytes(C.byref(g), C.byref(p)) == 0
    assert b"n_sectors" in lib.tpcca_last_error()
    assert lib.tpcca_track(None, None, 0, None, None, None, None) == -2  # TPCCA_ERR_NOT_INIT


def test_init_fails_loudly_without_device(lib, row_x):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    rx = np.ascontiguousarray(row_x)
    g = binding.Geometry(36, 152, rx.ctypes.data_as(C.POINTER(C.c_float)), synth.TAN_HALF_ANGLE)
    p = binding.default_params()
    p.max_clusters, p.max_tracklets, p.max_tracks = 1024, 128, 128
    p.workspace, p.workspace_bytes = 256, 1 << 40
    assert not lib.tpcca_init(C.byref(g), 0.5, C.byref(p))
    assert b"no CPU fallback" in lib.tpcca_last_error()
    with pytest.raises(binding.TpccaError):
        binding.Tracker(row_x)
