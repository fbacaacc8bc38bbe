"""GPU parity of tpcca_find_legs (looper legs + cluster tags) against the oracle's O12-O13:
leg partners, first-leg flags and cluster tags are integer results and must agree bit for bit."""
import ctypes as C

import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import binding as B
from paper_1811_11481_b200 import synth
from tests import looper
from tests.parity import run_gpu

pytestmark = pytest.mark.gpu


def compare_legs(fr, row_x, tracker=None, legs=None):
    orc = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=legs or True)
    t = run_gpu(fr, row_x, tracker)
    t.merge()
    partner, partner_in, first, tags, sm = t.find_legs(**(legs or {}))
    assert t.merged_header()["n_merged"] == len(orc.merged)
    assert np.array_equal(t.track_merged(), orc.track_merged)
    assert np.array_equal(partner, orc.leg_partner)
    assert np.array_equal(partner_in, orc.leg_partner_in)
    assert np.array_equal(first, orc.leg_first)
    assert np.array_equal(tags, orc.cluster_tags)
    assert sm["n_links_outer"] == int((orc.leg_partner >= 0).sum()) // 2
    assert sm["n_links_inner"] == int((orc.leg_partner_in >= 0).sum()) // 2
    assert sm["n_tag_low_pt"] == int(((orc.cluster_tags & 1) > 0).sum())
    assert sm["n_tag_extra_leg"] == int(((orc.cluster_tags & 2) > 0).sum())
    assert sm["n_tag_high_inclination"] == int(((orc.cluster_tags & 4) > 0).sum())
    return t, orc


@pytest.mark.parametrize("cfg,scale", [(3, 0.3), (3, 1.0), (2, 0.5), (4, 0.2), (5, 0.1), (1, 1.0)])
def test_legs_parity_configs(row_x, cfg, scale):
    fr = synth.generate(synth.config(cfg, scale=scale))
    t, orc = compare_legs(fr, row_x)
    if cfg == 3:
        assert (orc.leg_partner >= 0).sum() >= 400 and (orc.leg_partner_in >= 0).sum() >= 300


def test_legs_parity_full_frame(row_x):
    """Config 5 at full size in the capacities bench.py uses (107 k merged tracks)."""
    fr = synth.generate(synth.config(5, seed=5))
    t = B.Tracker(row_x, n_sectors=36, max_clusters=fr.n, max_tracklets=max(1 << 16, fr.n // 8),
                  max_tracks=max(1 << 16, fr.n // 24))
    t, orc = compare_legs(fr, row_x, tracker=t)
    assert (orc.leg_partner >= 0).sum() > 1000


def test_legs_parity_23ms_time_frame(row_x):
    """|z| up to 6e4 cm: z differences of nearby legs are still exact in fp32 (a few ulp of 4e-3 cm against
    a 4 cm window), and the z bins of the candidate buckets saturate (everything beyond 4096 cm falls into the last bin) --
    the links must not depend on that search structure."""
    cfg = synth.config(5, scale=0.4, seed=23)
    cfg["time_window_us"] = 23000.0
    fr = synth.generate(cfg)
    assert float(np.abs(fr.clusters["z"]).max()) > 5.0e4
    t, orc = compare_legs(fr, row_x)
    assert (orc.leg_partner >= 0).sum() > 200 and (orc.leg_partner_in >= 0).sum() > 200


def test_legs_parity_hand_built_loopers(row_x):
    """The float64 helices of the oracle pins: one looper of each charge, three turns at a 12 cm pitch, a 45 MeV/c secondary
    circling inside the TPC -- all in one frame."""
    parts = [looper.helix_clusters(row_x, 0.12, 0.7, 0.3, +1, z0=10.0, turns=2.0),
             looper.helix_clusters(row_x, 0.12, 2.9, -0.3, -1, z0=-10.0, turns=2.0),
             looper.helix_clusters(row_x, 0.13, -1.0, 0.022, +1, z0=60.0, turns=3.0),
             looper.helix_clusters(row_x, 0.045, 0.3, 0.25, +1, z0=120.0, origin=(150.0 * np.cos(4.0), 150.0 * np.sin(4.0)), turns=2.0)]
    fr, _ = looper.frame_from(parts)
    t, orc = compare_legs(fr, row_x)
    assert (orc.leg_partner >= 0).sum() >= 10 and (orc.leg_partner_in >= 0).sum() >= 6
    assert ((orc.cluster_tags & 1) > 0).sum() >= 40


def test_legs_parity_non_default_parameters(row_x):
    fr = synth.generate(synth.config(3, scale=0.3, seed=9))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    for legs in (dict(leg_dz_max=30.0, leg_centre_abs=6.0, leg_radius_frac=0.5), dict(ring=0), dict(leg_max_sector_gap=2),
                 dict(tag_sinphi=0.6, tag_qpt_leg=7.0, tag_qpt_low=6.0), dict(leg_max_turn=1.8, leg_min_sinphi=0.7),
                 dict(leg_inner_max_sector_gap=5, leg_inner_max_turn=3.5, leg_inner_min_sinphi=0.45)):
        compare_legs(fr, row_x, tracker=t, legs=legs)


def test_legs_twice_and_argument_checks(row_x):
    import torch
    fr = synth.generate(synth.config(3, scale=0.1, seed=4))
    t = B.Tracker(row_x, max_clusters=fr.n, max_tracklets=max(1024, fr.n // 4))
    lp = B.default_leg_params()
    pa = torch.empty(t.max_tracks, dtype=torch.int32, device="cuda")
    pin = torch.empty(t.max_tracks, dtype=torch.int32, device="cuda")
    fi = torch.empty(t.max_tracks, dtype=torch.uint8, device="cuda")
    tg = torch.empty(fr.n, dtype=torch.uint8, device="cuda")
    sm = torch.empty(8, dtype=torch.int32, device="cuda")
    args = (pa.data_ptr(), pin.data_ptr(), fi.data_ptr(), tg.data_ptr(), sm.data_ptr())
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), *args) == -1      # no frame yet
    run_gpu(fr, row_x, t)
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), *args) == -1      # no merge yet
    t.merge()
    assert t.lib.tpcca_find_legs(t.h, None, t._stream(), *args) == -1
    assert t.lib.tpcca_find_legs(None, C.byref(lp), t._stream(), *args) == -2
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), pa.data_ptr() + 2, *args[1:]) == -1
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), *args[:4], sm.data_ptr() + 4) == -1
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), args[0], None, *args[2:]) == -1
    for field, bad in (("leg_max_turn", 3.2), ("leg_inner_max_turn", 6.3), ("leg_min_sinphi", 0.0), ("leg_dz_max", 0.0), ("ring", -1), ("ring", 1), ("ring", 65)):
        q = B.default_leg_params()
        setattr(q, field, bad)
        assert t.lib.tpcca_find_legs(t.h, C.byref(q), t._stream(), *args) == -1, field
    a = t.find_legs()
    b = t.find_legs()
    assert all(np.array_equal(x, y) for x, y in zip(a[:4], b[:4])) and a[4] == b[4]
    # a new frame invalidates the merge; an empty frame has no legs and no tags
    empty = synth.Frame(np.zeros(0, synth.CLUSTER_DTYPE), np.zeros(37, np.int32), np.zeros(0, np.int32), np.zeros((0, 8)), 36, "e")
    run_gpu(empty, row_x, t)
    assert t.lib.tpcca_find_legs(t.h, C.byref(lp), t._stream(), *args) == -1
    t.merge()
    p, pi_, f, g, s = t.find_legs()
    assert len(p) == 0 and len(pi_) == 0 and len(g) == 0 and not any(s.values())


@pytest.mark.parametrize("seed", [1, 3])
def test_low_pt_tag_threshold_between_segment_and_merged_curvature(row_x, seed):
    """tests/test_oracle_pins_r3.py::test_low_pt_tag_follows_the_merged_tracks_curvature on the GPU."""
    from tests import scenarios
    par = dict(x0=85.0, y0=4.0, z0=25.0, sinphi0=0.12, tanl=0.5, qpt=-4.5, bz=0.5)
    with np.errstate(invalid="ignore"):
        fr, info = scenarios.helix_in_two_sectors(row_x, rng=np.random.default_rng(seed), par=par)
    base = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=True)
    thr = 0.5 * (abs(float(base.tracks["qpt"][0])) + abs(float(base.merged["qpt"][0])))
    t, orc = compare_legs(fr, row_x, legs=dict(tag_qpt_low=thr))
    assert ((orc.cluster_tags & 1) != 0).sum() in (0, int((orc.assignment >= 0).sum()))
