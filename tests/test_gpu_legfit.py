"""GPU parity of tpcca_fit_legs (one fit through both legs of a turn) against the oracle's O14: the
operation sequence is identical on both sides, so the 128-byte records are compared byte for byte."""
import ctypes as C

import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import synth
from tests import looper
from tests.parity import PARAM_ATOL, PARAM_RTOL, run_gpu

pytestmark = pytest.mark.gpu


def compare_fits(fr, row_x, tracker=None, fit=None):
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=True, leg_fit=fit or True)
    t = run_gpu(fr, row_x, tracker)
    t.merge()
    partner, *_ = t.find_legs()
    assert np.array_equal(partner, orc.leg_partner)
    got, n_failed = t.fit_legs(**(fit or {}))
    exp = orc.leg_fits
    assert len(got) == len(exp) and n_failed == int((exp["pad"][:, 2] == -1).sum())   # (ndf alone can be -1 with two hits used)
    for f in ("sector", "first_row", "last_row", "n_hits", "ndf", "pad"):
        assert np.array_equal(got[f], exp[f]), f
    for f in ("x", "y", "z", "sinphi", "dzds", "qpt", "chi2"):
        np.testing.assert_allclose(got[f], exp[f], rtol=PARAM_RTOL, atol=PARAM_ATOL, err_msg=f)
    assert got.tobytes() == exp.tobytes(), "identical operation sequence: the records should be bit-identical"
    return t, orc


@pytest.mark.parametrize("cfg,scale", [(3, 0.3), (3, 1.0), (2, 0.5), (4, 0.2), (5, 0.1), (1, 1.0)])
def test_leg_fit_parity_configs(row_x, cfg, scale):
    fr = synth.generate(synth.config(cfg, scale=scale))
    t, orc = compare_fits(fr, row_x)
    if cfg == 3:
        assert len(orc.leg_fits) >= 200 and (orc.leg_fits["ndf"] >= 0).mean() > 0.9


def test_leg_fit_parity_full_frame(row_x):
    fr = synth.generate(synth.config(5, seed=5))
    t = B.Tracker(row_x, n_sectors=36, max_clusters=fr.n, max_tracklets=max(1 << 16, fr.n // 8),
                  max_tracks=max(1 << 16, fr.n // 24))
    t, orc = compare_fits(fr, row_x, tracker=t)
    assert len(orc.leg_fits) > 10000


def test_leg_fit_parity_hand_built_and_parameters(row_x):
    parts = [looper.helix_clusters(row_x, 0.12, 0.7, 0.3, +1, z0=10.0, turns=2.0),
             looper.helix_clusters(row_x, 0.09, 2.9, -0.5, -1, z0=-10.0),
             looper.helix_clusters(row_x, 0.15, 5.0, 0.05, +1, z0=60.0)]
    fr, _ = looper.frame_from(parts)
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    for fit in (None, dict(fit_rot_sinphi=0.3, fit_step_sinphi=0.5), dict(fit_min_d=0.6), dict(fit_reject_cut=4.0),
                dict(ring=0), dict(shared_err_scale=3.0)):
        t2, orc = compare_fits(fr, row_x, tracker=t, fit=fit)
        assert len(orc.leg_fits) >= 3


def test_leg_fit_argument_checks(row_x):
    import torch
    fr = synth.generate(synth.config(3, scale=0.1, seed=4))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    fp = B.default_leg_fit_params()
    out = torch.empty(16 + 128 * t.max_tracks, dtype=torch.uint8, device="cuda")
    run_gpu(fr, row_x, t)
    t.merge()
    assert t.lib.tpcca_fit_legs(t.h, C.byref(fp), t._stream(), out.data_ptr()) == -1      # no tpcca_find_legs yet
    t.find_legs()
    assert t.lib.tpcca_fit_legs(t.h, None, t._stream(), out.data_ptr()) == -1
    assert t.lib.tpcca_fit_legs(t.h, C.byref(fp), t._stream(), None) == -1
    assert t.lib.tpcca_fit_legs(t.h, C.byref(fp), t._stream(), out.data_ptr() + 8) == -1
    assert t.lib.tpcca_fit_legs(None, C.byref(fp), t._stream(), out.data_ptr()) == -2
    for field, bad in (("fit_rot_sinphi", 0.95), ("fit_step_sinphi", 0.2), ("ring", -1), ("shared_err_scale", 0.0)):
        q = B.default_leg_fit_params()
        setattr(q, field, bad)
        assert t.lib.tpcca_fit_legs(t.h, C.byref(q), t._stream(), out.data_ptr()) == -1, field
    a, na = t.fit_legs()
    b, nb = t.fit_legs()
    assert a.tobytes() == b.tobytes() and na == nb and len(a) > 20
    t.merge()                                                                               # a new merge invalidates the links
    assert t.lib.tpcca_fit_legs(t.h, C.byref(fp), t._stream(), out.data_ptr()) == -1
