"""GPU parity of tpcca_merge (sector-segment merger + final fit) against the oracle's O8-O10."""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import synth
from tests import scenarios
from tests.parity import PARAM_ATOL, PARAM_RTOL, run_gpu

pytestmark = pytest.mark.gpu


def compare_merge(fr, row_x, tracker=None, params=None, merge=None):
    """Outer ends, shared flags, links, merged ids bit-exact; merged records within the parameter tolerance (and, the
    operation sequence being identical, byte-identical: returned as `exact`)."""
    merge = merge or {}
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, params=params, merge=merge or True)
    t = run_gpu(fr, row_x, tracker, **(params or {}))
    assert t.header()["n_tracks"] == len(orc.tracks)
    assert np.array_equal(t.assignment(), orc.assignment)
    shared = t.intermediate(B.SHARED)
    assert np.array_equal(np.maximum(shared, 0), orc.shared.astype(np.int32))
    outer = t.intermediate(B.TRACK_OUTER)[:, :21]
    ok = orc.tracks["ndf"] >= 0
    np.testing.assert_allclose(outer[ok], orc.outer[ok], rtol=PARAM_RTOL, atol=PARAM_ATOL)
    t.merge(**merge)
    t.torch.cuda.synchronize()
    hd = t.merged_header()
    assert hd["n_merged"] == len(orc.merged), (hd, len(orc.merged))
    assert hd["n_links"] == int((orc.link_next >= 0).sum())
    assert hd["n_fit_failed"] == int((orc.merged["pad"][:, 2] < 0).sum())
    assert np.array_equal(t.intermediate(B.MERGE_LINK_NEXT), orc.link_next)
    assert np.array_equal(t.track_merged(), orc.track_merged)
    m = t.merged()
    for f in ("sector", "first_row", "last_row", "n_hits", "ndf", "pad"):
        assert np.array_equal(m[f], orc.merged[f]), f
    for f in ("x", "y", "z", "sinphi", "dzds", "qpt", "chi2"):
        np.testing.assert_allclose(m[f], orc.merged[f], rtol=PARAM_RTOL, atol=PARAM_ATOL, err_msg=f)
    np.testing.assert_allclose(m["cov"], orc.merged["cov"], rtol=1e-3, atol=1e-9)
    return t, orc, m.tobytes() == orc.merged.tobytes() and outer[ok].tobytes() == orc.outer[ok].tobytes()


@pytest.mark.parametrize("cfg,scale", [(2, 0.25), (2, 1.0), (3, 0.5), (4, 0.2), (5, 0.1), (1, 1.0)])
def test_merge_parity_configs(row_x, cfg, scale):
    fr = synth.generate(synth.config(cfg, scale=scale))
    t, orc, exact = compare_merge(fr, row_x)
    if cfg != 1:
        assert (orc.link_next >= 0).sum() > 100 and len(orc.merged) < len(orc.tracks)
    else:
        assert len(orc.merged) == len(orc.tracks)  # a standalone sector has no neighbours
    assert exact, "identical operation sequence: merged records should be bit-identical"


def test_merge_parity_full_frame(row_x):
    """Config 5 at full size (15.2 M clusters, 210 k sector tracks) in the capacities bench.py uses."""
    fr = synth.generate(synth.config(5, seed=5))
    t = B.Tracker(row_x, n_sectors=36, max_clusters=fr.n, max_tracklets=max(1 << 16, fr.n // 8),
                  max_tracks=max(1 << 16, fr.n // 24))
    t, orc, exact = compare_merge(fr, row_x, tracker=t)
    assert len(orc.merged) > 50000 and exact


def test_merge_parity_hand_built(row_x):
    """The scenarios of tests/test_merge_pins.py through the CUDA path: every ring position, each predicate of the match,
    competing partners, rejection, shared clusters."""
    cases = []
    for sector, side in ((3, +1), (3, -1), (17, +1), (18, -1), (35, +1), (0, -1)):
        cases.append((scenarios.helix_in_two_sectors(row_x, sector=sector, side=side)[0], None))
    early = dict(x0=85.0, y0=4.0, z0=25.0, sinphi0=0.2, tanl=0.5, qpt=-1.1, bz=0.5)
    two = lambda **kw: scenarios.helix_in_two_sectors(row_x, sector=7, side=+1, par=early, **kw)[0]  # noqa: E731
    cases += [(two(z_shift_b=3.0), None), (two(z_shift_b=0.03), None), (two(drop_rows_b=8), None), (two(drop_rows_b=7), None),
              (two(drop_rows_a_end=6), dict(merge_edge_dist=0.7)), (two(drop_rows_a_end=6), dict(merge_edge_dist=2.0)),
              (two(), dict(merge_dz_max=0.4)), (two(), dict(merge_dz_max=0.8)), (two(extend_a=3), None), (two(extend_a=4), None),
              (two(qpt_b=1.1), None), (two(qpt_b=-1.1), None), (two(copy_a_dz=-0.4), dict(merge_chi2_cut=1e6)),
              (two(), dict(ring=0)), (two(), dict(merge_chi2_cut=0.0)),
              (two(rng=np.random.default_rng(21)), None)]
    fr, _ = scenarios.helix_in_two_sectors(row_x, sector=9, side=-1)
    fr.clusters["y"][60] += 0.35
    cases += [(fr, None), (fr, dict(fit_reject_cut=6.0))]
    cl, _ = scenarios.crossing_helices(row_x)
    so = np.zeros(37, np.int32)
    so[1:] = len(cl)
    cross = synth.Frame(cl, so, np.full(len(cl), -1, np.int32), np.zeros((0, 8)), 36, "crossing")
    cases += [(cross, None), (cross, dict(shared_err_scale=1.0))]
    for fr, merge in cases:
        t, orc, exact = compare_merge(fr, row_x, merge=merge)
        assert exact


def test_merge_twice_and_after_each_frame(row_x):
    """tpcca_merge may be called again on the same frame (same result) and after the next frame on the same handle."""
    fr1 = synth.generate(synth.config(2, scale=0.2, seed=91))
    fr2 = synth.generate(synth.config(3, scale=0.2, seed=92))
    t = B.Tracker(row_x, max_clusters=max(fr1.n, fr2.n), max_tracklets=max(fr1.n, fr2.n) // 4)
    compare_merge(fr1, row_x, tracker=t)
    m1 = t.merged().tobytes()
    t.merge()
    t.torch.cuda.synchronize()
    assert t.merged().tobytes() == m1
    compare_merge(fr2, row_x, tracker=t)
    compare_merge(fr1, row_x, tracker=t)
    assert t.merged().tobytes() == m1


def test_merge_argument_checks(row_x):
    fr = synth.generate(synth.config(2, scale=0.05, seed=3))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    mp = B.default_merge_params()
    import ctypes as C
    import torch
    om = torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8, device="cuda")
    tm = torch.empty(t.max_tracks, dtype=torch.int32, device="cuda")
    assert t.lib.tpcca_merge(t.h, C.byref(mp), t._stream(), om.data_ptr(), tm.data_ptr()) == -1  # no frame yet
    run_gpu(fr, row_x, t)
    assert t.lib.tpcca_merge(t.h, None, t._stream(), om.data_ptr(), tm.data_ptr()) == -1
    assert t.lib.tpcca_merge(t.h, C.byref(mp), t._stream(), om.data_ptr() + 4, tm.data_ptr()) == -1
    assert t.lib.tpcca_merge(None, C.byref(mp), t._stream(), om.data_ptr(), tm.data_ptr()) == -2
    for bad_ring in (-1, 1, 65):  # ring 1: a sector would be its own neighbour (self links, chains without a head)
        mp.ring = bad_ring
        assert t.lib.tpcca_merge(t.h, C.byref(mp), t._stream(), om.data_ptr(), tm.data_ptr()) == -1, bad_ring
    assert b"ring" in t.lib.tpcca_last_error()
    # an empty frame merges to nothing
    empty = synth.Frame(np.zeros(0, synth.CLUSTER_DTYPE), np.zeros(37, np.int32), np.zeros(0, np.int32), np.zeros((0, 8)), 36, "e")
    run_gpu(empty, row_x, t)
    t.merge()
    t.torch.cuda.synchronize()
    assert t.merged_header() == dict(n_merged=0, n_links=0, n_fit_failed=0, status=0)
