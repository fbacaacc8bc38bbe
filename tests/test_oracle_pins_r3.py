"""Round-3 pins of the CPU oracle: the mechanics that a one-line slip could change without any earlier pin noticing
("What's weak" 1).  Every expectation comes from outside the oracle: a float64 filter on the closed-form
helix (tests/kf64.py, tests/helix.py), the index order of bit-identical clusters, plain counting, or the float64 truth of
the hand-built input.  The inputs live in tests/scenarios.py so that the GPU parity tests run the same cases.
None of these call the CUDA path.
"""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import synth
from tests import kf64, scenarios
from tests.helix import helix_points

SY2, SZ2 = 0.1 ** 2, 0.15 ** 2
COV0 = [1.0, 1.0, 0.25, 1.0, 100.0]
HELIX = dict(x0=85.0, y0=0.5, z0=20.0, sinphi0=0.08, tanl=0.4, qpt=1.2, bz=0.5)  # scenarios.one_helix


def _so(cl):
    return np.array([0, len(cl)], np.int32)


def _inward_prediction(row_x, rows_with_hits, row_to):
    """Float64 covariance of the inward pass (covariance reset at the outermost hit, then one update per hit
    going down) predicted at `row_to`, on the true helix of scenarios.one_helix."""
    xs = row_x.astype(np.float64)
    y, z, s = helix_points(xs, **HELIX)
    top = max(rows_with_hits)
    p = np.array([y[top], z[top], s[top], HELIX["tanl"], HELIX["qpt"]])
    C = np.diag(np.array(COV0, np.float64))
    V = np.diag([SY2, SZ2])
    xc = xs[top]
    for j in sorted((r for r in rows_with_hits if r > row_to), reverse=True):
        p, C = kf64.transport(xc, p, C, xs[j], HELIX["bz"])
        xc = xs[j]
        p, C, _ = kf64.update(p, C, np.array([y[j], z[j]]), V)
    p, C = kf64.transport(xc, p, C, xs[row_to], HELIX["bz"])
    return C


# ---------------------------------------------------------------- (i) keep / reject distance of a seed hit uses var(z)
def test_reject_distance_of_a_hit_displaced_in_z(row_x):
    """on the inward pass a seed hit is dropped when its distance to the prediction exceeds reject_cut.
    The hit of row 120 sits 0.45 cm off in z only, so d = dz^2 / (C_zz + sigma_z^2) with C_zz the PREDICTED z variance after
    the 31 hits above it (float64 filter: d = 7.93; with cov(y,z) in its place it would be 9.05).  Kept 3 % above that
    distance, dropped 3 % below."""
    R = len(row_x)
    C = _inward_prediction(row_x, range(R), 120)
    d64 = 0.45 ** 2 / (C[1, 1] + SZ2)
    assert 7.5 < d64 < 8.3 and abs(C[0, 1]) < 0.1 * C[1, 1]
    cl = scenarios.displaced_hit_helix_z(row_x, row=120, dz=0.45)
    keep = oracle.track(cl, _so(cl), row_x, params=dict(reject_cut=1.03 * d64))
    assert len(keep.tracks) == 1 and keep.tracks["n_hits"][0] == R and keep.assignment[120] == 0
    drop = oracle.track(cl, _so(cl), row_x, params=dict(reject_cut=0.97 * d64))
    assert len(drop.tracks) == 1 and drop.tracks["n_hits"][0] == R - 1 and drop.assignment[120] == -1


# ---------------------------------------------------------------- (ii) equal pick-up distances: the key order decides
@pytest.mark.parametrize("positions", [None, (0, 1), (0, 200), (70, 10)])
def test_duplicate_clusters_in_a_pick_up_row_follow_the_index_order(row_x, positions):
    """DESIGN.md A4: among candidates of bit-equal distance the lower (ord z, ord y, input index) wins.  Row 100 can only be
    reached by the pick-up search and holds the same cluster twice: the copy with the lower input index is taken, wherever
    the two sit in the input."""
    cl, pos = scenarios.lone_row_helix(row_x, duplicate=True, dup_positions=positions)
    assert len(pos) == 2 and cl[pos[0]].tobytes() == cl[pos[1]].tobytes()
    r = oracle.track(cl, _so(cl), row_x)
    assert len(r.tracks) == 1 and r.tracks["n_hits"][0] == len(cl) - 1
    assert r.assignment[min(pos)] == 0 and r.assignment[max(pos)] == -1
    assert (np.delete(r.assignment, max(pos)) == 0).all()


# ---------------------------------------------------------------- (iii) pick-up: cut and window in y and in z
@pytest.mark.parametrize("axis", ["y", "z"])
def test_pick_up_cut_uses_the_predicted_variance_of_its_own_coordinate(row_x, axis):
    """PAPER.md:51 / :108: the extrapolation picks up the best cluster of a row if it is close enough: 2-dof distance
    d = dy^2 / (C_yy + sigma_y^2) + dz^2 / (C_zz + sigma_z^2) <= pick_cut = 16 (and the explicit window of DESIGN.md A10 may
    never refuse such a cluster).  The lone cluster of row 100 is moved along ONE axis to d = 0.94 * 16 and d = 1.06 * 16 of
    the float64 prediction coming down from the chain above (rows 151..103); the prediction from the chain below is
    tighter, so it never accepts what the inward pass refuses."""
    R = len(row_x)
    rows = [r for r in range(R) if r >= 103]
    C = _inward_prediction(row_x, rows, 100)
    v = (C[0, 0] + SY2) if axis == "y" else (C[1, 1] + SZ2)
    assert (C[0, 0] + SY2) * 1.2 < (C[1, 1] + SZ2)  # the z window is wider than the y window: swapping them would show
    for frac, taken in ((0.94, True), (1.06, False)):
        disp = float(np.sqrt(16.0 * frac * v))
        cl, pos = scenarios.lone_row_helix(row_x, **{"d" + axis: disp})
        r = oracle.track(cl, _so(cl), row_x)
        assert len(r.tracks) == 1, (axis, frac)
        assert (r.assignment[pos[0]] == 0) == taken, (axis, frac, disp)
        assert r.tracks["n_hits"][0] == len(cl) - (0 if taken else 1)


# ---------------------------------------------------------------- (iv) neighbour window: y and z slopes are separate
@pytest.mark.parametrize("seed", [13])
def test_p1_brute_force_triplets_with_unequal_windows(row_x, seed):
    """as P1 (all-triplet search in plain numpy), with a y window much narrower than the z window."""
    from tests.test_oracle_pins import _brute_links_py
    fr = synth.generate(synth.config(1, scale=0.02, seed=seed), noise_frac=0.4)
    P = dict(oracle.DEFAULT_PARAMS, nbr_dydx=0.25, nbr_margin_y=0.2, nbr_dzdx=2.5, nbr_margin_z=1.5)
    over = {k: P[k] for k in ("nbr_dydx", "nbr_margin_y", "nbr_dzdx", "nbr_margin_z")}
    with np.errstate(over="ignore"):
        up, dn = _brute_links_py(fr.clusters, row_x, P)
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x, params=over)
    assert np.array_equal(r.link_up_raw, up) and np.array_equal(r.link_down_raw, dn)
    d = oracle.track(fr.clusters, fr.sector_offsets, row_x)
    assert (r.link_up_raw != d.link_up_raw).sum() > 5 and (up >= 0).sum() > 30


def test_neighbour_window_slopes_act_on_their_own_axis(row_x):
    """A straight triplet (cost 0) whose neighbours sit 0.9 cm away in y, or 1.2 cm away in z: inside the default window
    (slope 1.5 per cm of row distance 1.06, margins 0.5 / 0.75).  Slope 0.3 in y closes the y case only (window 0.82 cm),
    slope 0.3 in z the z case only (window 1.07 cm)."""
    pitch = float(row_x[51] - row_x[50])
    assert 0.3 * pitch + 0.5 < 0.9 < 1.5 * pitch + 0.5 and 0.3 * pitch + 0.75 < 1.2 < 1.5 * pitch + 0.75
    for kw, y_links, z_links in ((dict(), True, True), (dict(nbr_dydx=0.3), False, True), (dict(nbr_dzdx=0.3), True, False)):
        for (dy, dz), expect in (((0.9, 0.0), y_links), ((0.0, 1.2), z_links)):
            cl = scenarios.window_triplet(row_x, dy, dz)
            r = oracle.track(cl, _so(cl), row_x, params=kw)
            assert (r.link_up_raw[1] == 2 and r.link_down_raw[1] == 0) == expect, (kw, dy, dz)
            assert (r.link_up_raw[1] == -1 and r.link_down_raw[1] == -1) == (not expect)


# ---------------------------------------------------------------- (v) rows the inward pass never reaches are empty
def test_rows_below_an_inward_stop_inside_the_seed_are_dropped(row_x):
    """the track is what the inward pass confirms.  A helix enters the sector from the side at row 60; here the
    clusters BEYOND the side exist on every row, so the links (which know no sector edge) chain them into the seed.  The
    inward pass stops at the first row whose prediction lies beyond |y| = x tan 10 deg + edge_margin (float64 truth,
    0.16 cm clear of the line): the seed hits below that row are not part of the tracklet."""
    margin = 0.5
    cl, y, inside = scenarios.edge_helix(row_x, inward=True, decoy_step=1)
    xs = row_x.astype(np.float64)
    lim = xs * np.tan(np.deg2rad(10.0)) + margin
    ok = np.abs(y) <= lim
    assert np.min(np.abs(np.abs(y) - lim)) > 0.1
    first_ok = int(np.flatnonzero(ok)[0])
    assert 40 < first_ok < 70 and ok[first_ok:].all() and not ok[:first_ok].any() and len(cl) == len(row_x)
    r = oracle.track(cl, _so(cl), row_x, params=dict(edge_margin=margin))
    assert cl["row"][r.start_hits].tolist() == [1], "one seed, starting far outside the sector"
    assert len(r.tracks) == 1 and r.tracks["first_row"][0] == first_ok and r.tracks["n_hits"][0] == len(row_x) - first_ok
    assert (r.row_hit[0][:first_ok] == -1).all() and (r.row_hit[0][first_ok:] >= 0).all()
    assert (r.assignment[cl["row"] < first_ok] == -1).all() and (r.assignment[cl["row"] >= first_ok] == 0).all()


# ---------------------------------------------------------------- (vi) minimum hit counts are inclusive
def test_minimum_hit_counts_are_inclusive(row_x):
    """DESIGN.md Table A: a chain / tracklet / track needs AT LEAST min_seed_hits / min_tracklet_hits / min_track_hits."""
    R = len(row_x)
    rows, y, z = scenarios.one_helix(row_x)
    cl = scenarios.mk(rows, y, z, row_x)
    r = oracle.track(cl, _so(cl), row_x)
    h, chain = int(r.start_hits[0]), 1
    while r.link_up[h] >= 0:
        h, chain = int(r.link_up[h]), chain + 1
    assert chain == R - 2 and len(r.tracks) == 1 and r.tracklet_ints[0].tolist() == [1, 0, R - 1, R]
    for kw, n_valid, n_tracks in ((dict(min_seed_hits=chain), 1, 1), (dict(min_seed_hits=chain + 1), 0, 0),
                                  (dict(min_tracklet_hits=R), 1, 1), (dict(min_tracklet_hits=R + 1), 0, 0),
                                  (dict(min_track_hits=R), 1, 1), (dict(min_track_hits=R + 1), 1, 0)):
        q = oracle.track(cl, _so(cl), row_x, params=kw)
        assert int(q.tracklet_ints[:, 0].sum()) == n_valid and len(q.tracks) == n_tracks, kw


# ---------------------------------------------------------------- (vii) degrees of freedom of a sector track
def test_ndf_of_a_sector_track(row_x):
    """Two measurements per hit, five fitted parameters: ndf = 2 n - 5 (include/tpcca.h tpcca_track_rec.ndf)."""
    rows, y, z = scenarios.one_helix(row_x)
    cl = scenarios.mk(rows, y, z, row_x)
    r = oracle.track(cl, _so(cl), row_x)
    assert r.tracks["n_hits"].tolist() == [152] and r.tracks["ndf"].tolist() == [299]
    cl2 = scenarios.gap_helix(row_x, 6)
    r2 = oracle.track(cl2, _so(cl2), row_x)
    assert sorted(zip(r2.tracks["n_hits"].tolist(), r2.tracks["ndf"].tolist())) == [(60, 115), (86, 167)]


# ---------------------------------------------------------------- (viii) quality field of the selector weight
def test_selector_quality_is_chi2_per_two_hits_in_thousandths(row_x):
    """DESIGN.md O6: between tracklets of equal length the quality field decides, quality = 65535 - int(qual_scale * chi2 /
    (2 n)) with qual_scale = 1000, and only then the lower id.  Two 91-hit tracklets share one cluster; A (the lower id)
    has one hit displaced by 0.035 cm: chi2 = 0.12, 1000 * 0.12 / 182 = 0.66 -> the same quality step as the clean tracklet,
    so the LOWER ID keeps the shared cluster although its chi2 is worse.  (Per n instead of per 2 n it would be 1.3: a
    different step, and the clean tracklet would win.)  At 0.05 cm, chi2 = 0.245 -> step 1: now the clean tracklet wins."""
    for dy, a_wins in ((0.035, True), (0.05, False)):
        cl, shared, is_a, is_b = scenarios.equal_length_crossing(row_x, "A", False, dy=dy)
        r = oracle.track(cl, _so(cl), row_x)
        assert len(r.tracks) == 2 and r.tracklet_ints[:2, 3].tolist() == [91, 91]
        ta, tb = int(r.assignment[np.flatnonzero(is_a)[0]]), int(r.assignment[np.flatnonzero(is_b)[0]])
        assert r.track_tracklet[ta] == 0 and r.track_tracklet[tb] == 1, "A is the lower tracklet id"
        chi_a, chi_b = float(r.tracklet_floats[0, 21]), float(r.tracklet_floats[1, 21])
        expect = (dy / 0.1) ** 2  # one hit off by dy: chi2 = (dy / sigma_y)^2 (1 - leverage), leverage of 1 hit in 91 ~ 2-4 %
        assert 0.93 * expect < chi_a < expect and chi_b < 1e-4
        step = lambda c, per: int(1000.0 * c / (per * 91))
        if a_wins:
            assert step(chi_a, 2) == step(chi_b, 2) == 0 and step(chi_a, 1) == 1
        else:
            assert step(chi_a, 2) == 1 and step(chi_b, 2) == 0
        assert r.assignment[shared] == (ta if a_wins else tb), dy


# ---------------------------------------------------------------- (ix) volume clamp of a merged track: all its clusters
def test_merged_track_is_shifted_inside_the_volume_by_all_its_clusters(row_x):
    """"In case clusters of a fully merged secondary track are outside the real TPC volume, the track is shifted
    inside".  A steep helix (tan lambda 1.1) from a collision 150 cm late crosses from sector 3 into sector 4; its largest z
    lies in the OUTER segment (sector 4), its closest approach more than 250 cm below that, so the shift is fixed by the end
    plate: z_shift = max z of ALL clusters - z_max, for the merged track and not only for its innermost segment."""
    par = dict(x0=85.0, y0=4.0, z0=175.0, sinphi0=0.12, tanl=1.1, qpt=-1.1, bz=0.5)
    with np.errstate(invalid="ignore"):
        fr, info = scenarios.helix_in_two_sectors(row_x, par=par)
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, time=dict(z_max=250.0))
    assert len(r.tracks) == 2 and len(r.merged) == 1 and r.merged["sector"][0] == 3 and r.merged["pad"][0][1] == info["sector_b"]
    z, so = fr.clusters["z"], fr.sector_offsets
    z_a, z_b = float(z[so[3]:so[4]].max()), float(z[so[4]:so[5]].max())
    assert z_b > z_a + 10.0
    zd = float(r.time_merged[0, 0])
    assert abs(zd - (175.0 - 1.1 * 85.0)) < 2.0 and zd < z_a - 250.0  # closest approach ~ z0 - tan(lambda) * x0
    assert r.time_merged[0, 1] == np.float32(z_b) - np.float32(250.0)
    assert r.time_sector[0, 1] == np.float32(z_a) - np.float32(250.0)   # the inner segment alone: its own clusters
    assert r.time_sector[1, 1] == np.float32(z_b) - np.float32(250.0)


# ---------------------------------------------------------------- (x) cluster tags
@pytest.mark.parametrize("seed,sector_above", [(1, True), (3, False)])
def test_low_pt_tag_follows_the_merged_tracks_curvature(row_x, seed, sector_above):
    """clusters of "very low-pT looping tracks below 50 MeV/c" are tagged -- a property of the whole track, so
    the MERGED fit decides (D11), not the fit of the sector segment a cluster happens to sit on.  Smeared helix in
    two sectors; the 58-hit inner segment's own q/pT differs from the merged one by about 1 %; a threshold between the two
    tags either every cluster of the track or none."""
    par = dict(x0=85.0, y0=4.0, z0=25.0, sinphi0=0.12, tanl=0.5, qpt=-4.5, bz=0.5)
    with np.errstate(invalid="ignore"):
        fr, info = scenarios.helix_in_two_sectors(row_x, rng=np.random.default_rng(seed), par=par)
    base = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=True)
    assert len(base.tracks) == 2 and len(base.merged) == 1
    q_seg, q_mrg = abs(float(base.tracks["qpt"][0])), abs(float(base.merged["qpt"][0]))
    assert abs(q_mrg - 4.5) < 0.03 and (q_seg > q_mrg + 0.02) == sector_above and abs(q_seg - q_mrg) > 0.02
    thr = 0.5 * (q_seg + q_mrg)
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=dict(tag_qpt_low=thr))
    on_track = r.assignment >= 0
    low = (r.cluster_tags & 1) != 0
    assert on_track.sum() > 140
    if sector_above:   # merged |q/pT| below the threshold: nothing is tagged, the inner segment included
        assert not low.any()
    else:              # merged |q/pT| above it: every cluster of the track, the inner segment included
        assert (low == on_track).all()


def test_clusters_of_a_failed_refit_are_tagged_high_inclination(row_x):
    """PAPER.md:157 "track segments with high inclination angle": a sector track whose refit cannot be carried through
    (|sin phi| beyond max_sinphi on the way, ndf = -1) has no usable local direction; all its clusters get the tag
    (D11).  Looper sample of config 3: such tracks exist, and some of their clusters would stay untagged if the
    local-angle rule were applied to the record they keep."""
    fr = synth.generate(synth.config(3, scale=0.1, seed=3))
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=True)
    bad = np.flatnonzero(r.tracks["ndf"] < 0)
    assert len(bad) >= 10
    on_bad = np.isin(r.assignment, bad)
    assert on_bad.sum() >= 100 and ((r.cluster_tags[on_bad] & 4) != 0).all()
    # the record such a track keeps (O7: the tracklet's own state) does not exceed the tag threshold everywhere:
    # with the local-angle rule at least one of these clusters would carry no tag
    T = r.tracks[bad]
    kq = -(0.000299792458 * 10.0 * 0.5)
    x_of = row_x[fr.clusters["row"]].astype(np.float64)
    untagged_by_angle = 0
    for t, rec in zip(bad, T):
        idx = np.flatnonzero(r.assignment == t)
        s_loc = rec["sinphi"] + (x_of[idx] - rec["x"]) * rec["qpt"] * kq
        untagged_by_angle += int((np.abs(s_loc) <= 0.8).sum())
    assert untagged_by_angle > 0
