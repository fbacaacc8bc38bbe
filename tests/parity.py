"""Shared helper of the GPU parity tests: run oracle and CUDA path on one frame and compare."""
import numpy as np

import oracle
from paper_1811_11481_b200 import binding as B

PARAM_RTOL, PARAM_ATOL = 1e-4, 1e-5  # north_star: relative 1e-4, or absolute 1e-5 in sinphi / tanlambda


def run_gpu(fr, row_x, tracker=None, **params):
    own = tracker is None
    if own:
        tracker = B.Tracker(row_x, n_sectors=fr.n_sectors, max_clusters=max(fr.n, 1024),
                            max_tracklets=max(1024, fr.n // 4), **params)
    dev = tracker.upload(fr.clusters) if fr.n else None
    tracker.track(dev, fr.n, fr.sector_offsets)
    tracker.torch.cuda.synchronize()
    return tracker


def compare(fr, row_x, tracker=None, params=None, check_intermediates=True):
    """Bit-exact: links, start hits, tracklet tables, assignment.  Parameters within tolerance."""
    params = params or {}
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, params=params)
    t = run_gpu(fr, row_x, tracker, **params)
    hd = t.header()
    assert hd["status"] == 0, hd
    assert hd["n_start_hits"] == len(orc.start_hits), (hd, len(orc.start_hits))
    assert hd["n_tracks"] == len(orc.tracks), (hd, len(orc.tracks))
    assert hd["n_tracklets"] == int(orc.tracklet_ints[:, 0].sum())
    if check_intermediates:
        for what, exp in ((B.LINK_UP_RAW, orc.link_up_raw), (B.LINK_DOWN_RAW, orc.link_down_raw),
                          (B.LINK_UP, orc.link_up), (B.LINK_DOWN, orc.link_down), (B.START_HITS, orc.start_hits),
                          (B.TRACKLET_INTS, None), (B.TRACKLET_ROW_HITS, orc.row_hit),
                          (B.TRACK_TRACKLET, orc.track_tracklet)):
            got = t.intermediate(what)
            if what == B.TRACKLET_INTS:
                exp = orc.tracklet_ints.copy()
                exp[exp[:, 0] == 0] = (0, -1, -1, 0)
            assert got.shape == exp.shape, (what, got.shape, exp.shape)
            bad = np.flatnonzero((got != exp).reshape(len(exp), -1).any(axis=1)) if len(exp) else []
            assert len(bad) == 0, (what, len(bad), bad[:5], got[bad[:3]], exp[bad[:3]])
        tf = t.intermediate(B.TRACKLET_FLOATS)
        valid = orc.tracklet_ints[:, 0] == 1
        exp = orc.tracklet_floats[:, [0, 1, 2, 3, 4, 5, 21, 22]]
        np.testing.assert_allclose(tf[valid], exp[valid], rtol=PARAM_RTOL, atol=PARAM_ATOL)
    assert np.array_equal(t.assignment(), orc.assignment)
    tr = t.tracks()
    for f in ("sector", "first_row", "last_row", "n_hits", "ndf"):
        assert np.array_equal(tr[f], orc.tracks[f]), f
    for f in ("x", "y", "z", "sinphi", "dzds", "qpt", "chi2"):
        np.testing.assert_allclose(tr[f], orc.tracks[f], rtol=PARAM_RTOL, atol=PARAM_ATOL, err_msg=f)
    np.testing.assert_allclose(tr["cov"], orc.tracks["cov"], rtol=1e-3, atol=1e-9)
    exact = tr.tobytes() == orc.tracks.tobytes()
    return t, orc, exact
