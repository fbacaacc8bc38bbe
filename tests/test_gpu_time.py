"""GPU parity of tpcca_estimate_time (O11) and the large-z single-precision case of PAPER.md:121."""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import synth
from tests.parity import run_gpu
from tests.test_gpu_merge import compare_merge

pytestmark = pytest.mark.gpu


def check_time(t, orc, zscale):
    ts, tm = t.estimate_time()
    # the oracle evaluates the definition in double precision from the same fp32 records; the kernel works in fp32:
    # a few ulp of z (z up to zscale) plus the fp32 turning angle over the curvature
    tol = 3e-3 + 1e-6 * zscale
    for got, exp in ((ts, orc.time_sector), (tm, orc.time_merged)):
        assert got.shape == exp.shape
        np.testing.assert_allclose(got[:, 0], exp[:, 0], rtol=0, atol=tol)
        np.testing.assert_allclose(got[:, 1], exp[:, 1], rtol=0, atol=tol)
        np.testing.assert_allclose(got[:, 2], exp[:, 2], rtol=0, atol=tol / 2.58)
        np.testing.assert_allclose(got[:, 3], exp[:, 3], rtol=2e-4, atol=2e-3)
        # the volume rule is a clamp: wherever the oracle clamps, the kernel clamps to the same bound
        cl = exp[:, 1] != exp[:, 0]
        assert np.array_equal(got[cl, 1], exp[cl, 1])


@pytest.mark.parametrize("cfg,scale", [(2, 0.3), (4, 0.2), (5, 0.1)])
def test_time_estimate_parity(row_x, cfg, scale):
    fr = synth.generate(synth.config(cfg, scale=scale))
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, time=True)
    t = run_gpu(fr, row_x)
    t.merge()
    check_time(t, orc, float(np.abs(fr.clusters["z"]).max()))
    assert (orc.time_merged[:, 1] != orc.time_merged[:, 0]).sum() > 10


def test_23ms_time_frame_single_precision_at_large_z(row_x):
    """PAPER.md:57 time frames of 10-23 ms, :121 "single precision floating point artifacts, which occur in the track fit at
    large z": 20 collisions spread over 23 ms put clusters at |z| up to 6e4 cm (one fp32 ulp = 4e-3 cm).  The path keeps z
    relative to a hit of the track, so links, assignment and the 128-byte records are still identical to the oracle, the
    merger too, and the time estimates agree to the ulp of z."""
    cfg = synth.config(5, scale=0.4, seed=23)
    cfg["time_window_us"] = 23000.0
    fr = synth.generate(cfg)
    zmax = float(np.abs(fr.clusters["z"]).max())
    assert zmax > 5.0e4 and fr.n > 1000000
    t, orc, exact = compare_merge(fr, row_x)
    assert exact and len(orc.merged) > 5000
    orc2 = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, time=True)
    check_time(t, orc2, zmax)
    # and the physics survives: efficiency as in a short frame
    from paper_1811_11481_b200 import score
    sc = score.score(orc.assignment, fr.truth, score.sector_of_cluster(fr.sector_offsets, fr.n), len(orc.tracks))
    assert sc["efficiency"] > 0.97 and sc["fake_rate"] < 0.01, sc


def test_time_estimate_argument_checks(row_x):
    import ctypes as C

    import torch
    fr = synth.generate(synth.config(2, scale=0.05, seed=3))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    out = torch.empty(4 * t.max_tracks, dtype=torch.float32, device="cuda")
    f = t.lib.tpcca_estimate_time
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr(), None) == -1      # no frame yet
    run_gpu(fr, row_x, t)
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr(), None) == 0
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr(), out.data_ptr()) == -1   # merged estimates need tpcca_merge
    assert f(t.h, 0.0, 250.0, t._stream(), out.data_ptr(), None) == -1
    assert f(t.h, 2.58, 250.0, t._stream(), None, None) == -1
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr() + 4, None) == -1
    t.merge()
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr(), out.data_ptr()) == 0
    run_gpu(fr, row_x, t)  # a new frame invalidates the merged tracks
    assert f(t.h, 2.58, 250.0, t._stream(), out.data_ptr(), out.data_ptr()) == -1
    torch.cuda.synchronize()


def test_merged_track_clamp_uses_every_segment(row_x):
    """tests/test_oracle_pins_r3.py::test_merged_track_is_shifted_inside_the_volume_by_all_its_clusters on the GPU: the largest
    z of a two-sector track lies in its outer segment and fixes the shift of the merged track."""
    from tests import scenarios
    par = dict(x0=85.0, y0=4.0, z0=175.0, sinphi0=0.12, tanl=1.1, qpt=-1.1, bz=0.5)
    with np.errstate(invalid="ignore"):
        fr, info = scenarios.helix_in_two_sectors(row_x, par=par)
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, time=True)
    t = run_gpu(fr, row_x)
    t.merge()
    check_time(t, orc, float(np.abs(fr.clusters["z"]).max()))
    ts, tm = t.estimate_time()
    assert len(tm) == 1 and tm[0, 1] == np.float32(fr.clusters["z"].max()) - np.float32(250.0) and tm[0, 1] > ts[0, 1]
