"""Pins of the oracle's sector-segment merger and final fit (steps O8-O10) against what the paper and
the mathematics fix.  PAPER.md:51 "The second phase merges the track segments found in the individual sectors and performs
the final track fit with the full Kalman filter"; :69 outlier rejection by predicted chi2; :70 enlarged errors for clusters
shared between tracks; :71 three passes.  None of these call the CUDA path."""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import score, synth
from tests import kf64, scenarios
from tests.helix import helix_points

P = oracle.DEFAULT_PARAMS
M = oracle.DEFAULT_MERGE_PARAMS


def _track(fr, row_x, merge=True, **params):
    return oracle.track(fr.clusters, fr.sector_offsets, row_x, params=params or None, merge=merge)


def rot64(xc, p, C, sgn, bz=0.5):
    """Float64 frame change by sgn * 20 degrees, derived independently: rotate the point and the direction, then slide
    along the helix back onto the plane x' = const of the unperturbed point; Jacobian by central differences."""
    a = np.deg2rad(20.0) * sgn
    xref = xc * np.cos(a) + p[0] * np.sin(a)

    def f(q):
        xq = xc * np.cos(a) + q[0] * np.sin(a)
        st = np.array([-xc * np.sin(a) + q[0] * np.cos(a), q[1], np.sin(np.arcsin(q[2]) - a), q[3], q[4]])
        return kf64.fmap(st, xq, xref, bz) if xq != xref else st

    J = np.zeros((5, 5))
    for j in range(5):
        e = np.zeros(5)
        e[j] = 1e-6 if j != 4 else 1e-3
        J[:, j] = (f(p + e) - f(p - e)) / (2 * e[j])
    return xref, f(p), J @ C @ J.T


# ---------------------------------------------------------------- frame rotation (B3)
@pytest.mark.parametrize("sgn", [+1, -1])
@pytest.mark.parametrize("x,y,s", [(120.0, 18.0, 0.3), (200.0, -30.0, -0.45), (90.0, 2.0, 0.0)])
def test_rotation_is_the_plane_rotation_by_the_sector_angle(x, y, s, sgn):
    """The frame change is the rotation of point and direction by +-20 degrees; cos / sin 20 come from tan 10 by the
    double-angle formulas.  Against numpy float64 trigonometry; the sin(phi) row of C scales with d sin(phi') / d sin(phi)."""
    C = np.zeros(15, np.float32)
    C[[0, 2, 5, 9, 14]] = [0.01, 0.02, 1e-4, 1e-4, 0.01]
    C[3] = 2e-4   # cov(sinphi, y)
    C[8] = -3e-5  # cov(dzds, sinphi)
    ok, x1, p1, C1 = oracle.rotate_frame(x, [y, 7.0, s, 0.6, 1.3], C, sgn)
    a = np.deg2rad(20.0) * sgn
    assert ok
    assert abs(x1 - (x * np.cos(a) + y * np.sin(a))) < 2e-5 and abs(p1[0] - (-x * np.sin(a) + y * np.cos(a))) < 2e-5
    assert abs(p1[2] - np.sin(np.arcsin(s) - a)) < 2e-7
    assert p1[1] == 7.0 and abs(p1[3] - 0.6) < 1e-7 and abs(p1[4] - 1.3) < 1e-7
    # covariance: against the float64 finite-difference Jacobian of the frame change (a shifted point slides along the
    # track back onto the new plane: dy'/dy = cos(phi)/cos(phi'), dz'/dy = -t sin(a)/cos(phi'), ds'/ds = cos(phi')/cos(phi))
    Cm = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            Cm[i, j] = Cm[j, i] = C[k]
            k += 1
    _, _, Ce = rot64(x, np.array([y, 7.0, s, 0.6, 1.3]), Cm, sgn)
    got = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            got[i, j] = got[j, i] = C1[k]
            k += 1
    scale = np.sqrt(np.outer(np.diag(Ce), np.diag(Ce)))
    assert np.max(np.abs(got - Ce) / scale) < 1e-4, np.abs(got - Ce) / scale
    # there and back again
    ok, x2, p2, C2 = oracle.rotate_frame(x1, p1, C1, -sgn)
    assert ok and abs(x2 - x) < 3e-5 and abs(p2[0] - y) < 3e-5 and abs(p2[2] - s) < 3e-7 and np.allclose(C2, C, rtol=2e-6)


def test_rotation_fails_beyond_max_sinphi():
    ok, *_ = oracle.rotate_frame(100.0, [0, 0, 0.8, 0, 0], np.zeros(15), -1)  # phi 53 -> 73 degrees: sin 0.956
    assert not ok
    ok, *_ = oracle.rotate_frame(100.0, [0, 0, 0.8, 0, 0], np.zeros(15), +1)
    assert ok


# ---------------------------------------------------------------- two halves of one helix (O8-O10)
@pytest.mark.parametrize("sector,side", [(3, +1), (3, -1), (17, +1), (18, -1), (35, +1), (0, -1)])
def test_two_halves_of_one_helix_merge_to_one_track(row_x, sector, side):
    """A noiseless float64 helix that leaves a sector through its side: the two sector segments are linked, give ONE merged
    track holding every cluster, and the final fit recovers the helix (in the inner sector's frame, at the innermost hit)
    to float precision -- in every ring position, both z sides, both directions (ring closure 17 -> 0, 18 <- 35)."""
    fr, info = scenarios.helix_in_two_sectors(row_x, sector=sector, side=side)
    r = _track(fr, row_x)
    assert len(r.tracks) == 2 and len(r.merged) == 1
    ia = int(np.flatnonzero(r.tracks["sector"] == sector)[0])
    ib = 1 - ia
    assert r.tracks["sector"][ib] == info["sector_b"]
    assert r.link_next[ia] == ib and r.link_next[ib] == -1 and (r.track_merged == 0).all()
    m = r.merged[0]
    assert m["n_hits"] == fr.n == r.tracks["n_hits"].sum() and m["ndf"] == 2 * fr.n - 5
    assert m["sector"] == sector and m["first_row"] == info["rows_a"][0] and m["last_row"] == info["rows_b"][-1]
    assert list(m["pad"]) == [2, info["sector_b"], 0, 0, ia]
    r0 = info["rows_a"][0]
    assert m["x"] == row_x[r0]
    assert abs(m["y"] - info["y_a"][r0]) < 3e-5 and abs(m["z"] - info["z_a"][r0]) < 3e-5
    assert abs(m["sinphi"] - info["s_a"][r0]) < 2e-6 and abs(m["dzds"] - info["par"]["tanl"]) < 1e-6
    assert abs(m["qpt"] - info["par"]["qpt"]) < 1e-5 * abs(info["par"]["qpt"])
    assert m["chi2"] < 1e-4
    # the merged fit is better constrained than the inner segment's own fit (more hits, longer lever arm)
    assert m["cov"][14] < r.tracks["cov"][ia][14]


def test_merged_fit_equals_a_float64_filter_across_the_boundary(row_x):
    """Smeared version: the oracle's three-pass merged fit against a float64 extended Kalman filter written here that changes
    frame by an exact rotation (point and direction; C propagated with the finite-difference Jacobian of the frame
    change, rot64 above)."""
    rng = np.random.default_rng(21)
    fr, info = scenarios.helix_in_two_sectors(row_x, sector=5, side=+1, rng=rng)
    r = _track(fr, row_x)
    assert len(r.merged) == 1 and r.merged["pad"][0][0] == 2 and r.merged["n_hits"][0] == fr.n
    cl = fr.clusters
    na = len(info["rows_a"])
    sec = np.r_[np.zeros(na, int), np.ones(fr.n - na, int)]  # 0: inner sector frame, 1: rotated by +20 degrees
    x, y, z = cl["x"].astype(np.float64), cl["y"].astype(np.float64), cl["z"].astype(np.float64)

    n = fr.n
    ds = np.hypot(x[-1] - x[-2], y[-1] - y[-2])
    p = np.array([y[-1], z[-1], (y[-1] - y[-2]) / ds, (z[-1] - z[-2]) / ds, float(r.tracks["qpt"][1])])
    xc, cur = x[-1], 1
    V = np.diag([P["sigma_y"] ** 2, P["sigma_z"] ** 2])
    for order in (range(n - 1, -1, -1), range(n), range(n - 1, -1, -1)):
        C, chi2 = np.diag(np.asarray(P["cov0"], np.float64)), 0.0
        for j in order:
            if sec[j] != cur:
                xc, p, C = rot64(xc, p, C, +1 if sec[j] > cur else -1)
                cur = sec[j]
            p, C = kf64.transport(xc, p, C, x[j], 0.5)
            xc = x[j]
            p, C, c = kf64.update(p, C, np.array([y[j], z[j]]), V)
            chi2 += c
    m = r.merged[0]
    sig = np.sqrt(np.diag(C))
    got = np.array([m["y"], m["z"], m["sinphi"], m["dzds"], m["qpt"]], np.float64)
    assert np.all(np.abs(got - p) < 2e-3 * sig), ((got - p) / sig)
    assert np.all(np.abs(got - p) < 2e-5 * np.maximum(1.0, np.abs(p))), (got - p)
    assert abs(m["chi2"] - chi2) < 1e-4 * chi2 and m["ndf"] == 2 * n - 5


# ---------------------------------------------------------------- neighbours that do not match stay apart (O9)
def test_non_matching_neighbours_stay_apart(row_x):
    base, info = scenarios.helix_in_two_sectors(row_x, sector=7, side=+1)
    assert len(_track(base, row_x).merged) == 1
    # the continuation displaced by 3 cm in z (20 sigma): two tracks; by 0.3 mm: still one
    for dz, n_merged in ((3.0, 2), (0.03, 1)):
        fr, _ = scenarios.helix_in_two_sectors(row_x, sector=7, side=+1, z_shift_b=dz)
        r = _track(fr, row_x)
        assert len(r.tracks) == 2 and len(r.merged) == n_merged, dz
    # beyond the row window (merge_row_fwd = 8): first_row(B) - last_row(A) = 9 -> apart; 8 -> merged
    early = dict(info["par"], sinphi0=0.2)  # leaves the sector at row 90: a long continuation
    for drop, n_merged in ((8, 2), (7, 1)):
        fr, i2 = scenarios.helix_in_two_sectors(row_x, sector=7, side=+1, par=early, drop_rows_b=drop)
        r = _track(fr, row_x)
        assert len(r.tracks) == 2 and r.tracks["first_row"][1] - r.tracks["last_row"][0] == drop + 1
        assert len(r.merged) == n_merged, drop
    # a different particle in the neighbour sector (opposite curvature, other dip angle) is not a continuation
    other = dict(info["par"], qpt=-info["par"]["qpt"], tanl=-0.2)
    fo, _ = scenarios.helix_in_two_sectors(row_x, sector=7, side=+1, par=other)
    b_other = fo.clusters[fo.sector_offsets[8]:fo.sector_offsets[9]]
    a_base = base.clusters[base.sector_offsets[7]:base.sector_offsets[8]]
    so = np.zeros(37, np.int32)
    so[8:] = len(a_base)
    so[9:] += len(b_other)
    mix = synth.Frame(np.concatenate([a_base, b_other]), so, np.full(so[-1], -1, np.int32), np.zeros((0, 8)), 36, "mix")
    r = _track(mix, row_x)
    if len(r.tracks) == 2:
        assert len(r.merged) == 2 and (r.link_next == -1).all()
    # and with chi2 cut 0 nothing merges at all
    r = _track(base, row_x, merge=dict(merge_chi2_cut=0.0))
    assert len(r.merged) == 2


def test_one_partner_per_end(row_x):
    """DESIGN.md B4: links are mutual best matches.  Two continuations compete for one outer end -- the true one and a copy
    displaced by 0.4 cm in z; only the better one is linked, the other stays a track of its own."""
    fr, info = scenarios.helix_in_two_sectors(row_x, sector=7, side=+1)
    sb = info["sector_b"]
    b = fr.clusters[fr.sector_offsets[sb]:fr.sector_offsets[sb + 1]]
    b2 = b.copy()
    b2["z"] += 0.4
    cl = np.concatenate([fr.clusters[:fr.sector_offsets[sb + 1]], b2])
    so = fr.sector_offsets.copy()
    so[sb + 1:] += len(b2)
    f2 = synth.Frame(cl, so, np.full(len(cl), -1, np.int32), np.zeros((0, 8)), 36, "two_partners")
    r = _track(f2, row_x)
    assert len(r.tracks) == 3 and len(r.merged) == 2 and (r.link_next >= 0).sum() == 1
    a = int(np.flatnonzero(r.tracks["sector"] == 7)[0])
    nxt = r.link_next[a]
    # the linked partner is the undisplaced copy: its clusters are the first len(b) of sector sb
    owned = np.flatnonzero(r.assignment == nxt)
    assert (owned < fr.sector_offsets[sb] + len(b)).all()


# ---------------------------------------------------------------- final fit: rejection and shared-cluster inflation
def test_final_fit_rejects_outliers_by_predicted_chi2(row_x):
    """a hit displaced by 3.5 sigma survives the sector tracking (d ~ 12 < 16) and the default final cut (30),
    but is left out of the final fit at fit_reject_cut = 6: one rejected hit, ndf two lower, smaller chi2, assignment kept."""
    fr, info = scenarios.helix_in_two_sectors(row_x, sector=9, side=-1)
    fr.clusters["y"][60] += 0.35
    keep = _track(fr, row_x)
    drop = _track(fr, row_x, merge=dict(fit_reject_cut=6.0))
    for r in (keep, drop):
        assert len(r.merged) == 1 and r.merged["n_hits"][0] == fr.n and (r.assignment >= 0).all()
    assert keep.merged["pad"][0][2] == 0 and keep.merged["ndf"][0] == 2 * fr.n - 5
    assert drop.merged["pad"][0][2] == 1 and drop.merged["ndf"][0] == 2 * (fr.n - 1) - 5
    assert drop.merged["chi2"][0] < 0.1 and keep.merged["chi2"][0] > 8.0


def test_shared_clusters_get_enlarged_errors(row_x):
    """PAPER.md:70 "clusters shared between multiple tracks" get an enlarged error.  Two crossing helices: the crossing
    cluster is collected by both tracklets and owned by the longer track -> it is the one shared cluster; in the owner's
    final fit its sigma is doubled.  Checked against the float64 filter with per-hit errors."""
    cl, is_a = scenarios.crossing_helices(row_x)
    # smear so that the weight of one hit matters
    rng = np.random.default_rng(4)
    cl = cl.copy()
    cl["y"] += rng.normal(0, 0.03, len(cl)).astype(np.float32)
    cl["z"] += rng.normal(0, 0.05, len(cl)).astype(np.float32)
    so = np.zeros(37, np.int32)
    so[1:] = len(cl)
    fr = synth.Frame(cl, so, np.full(len(cl), -1, np.int32), np.zeros((0, 8)), 36, "crossing")
    r = _track(fr, row_x)
    assert len(r.tracks) == 2 and len(r.merged) == 2
    shared = np.flatnonzero(r.shared)
    assert len(shared) == 1 and cl["row"][shared[0]] == 90 and is_a[shared[0]]
    owner = r.assignment[shared[0]]
    assert r.merged["pad"][r.track_merged[owner]][3] == 1 and r.merged["pad"][r.track_merged[1 - owner]][3] == 0
    hits = np.flatnonzero(r.assignment == owner)
    hits = hits[np.argsort(cl["row"][hits])]
    x, y, z = (cl[f][hits].astype(np.float64) for f in ("x", "y", "z"))
    res = {}
    for scale in (1.0, 2.0):
        ds = np.hypot(x[-1] - x[-2], y[-1] - y[-2])
        p = np.array([y[-1], z[-1], (y[-1] - y[-2]) / ds, (z[-1] - z[-2]) / ds, float(r.tracks["qpt"][owner])])
        xc = x[-1]
        for order in (range(len(x) - 1, -1, -1), range(len(x)), range(len(x) - 1, -1, -1)):
            C = np.diag(np.asarray(P["cov0"], np.float64))
            for j in order:
                f = scale if hits[j] == shared[0] else 1.0
                p, C = kf64.transport(xc, p, C, x[j], 0.5)
                xc = x[j]
                p, C, _ = kf64.update(p, C, np.array([y[j], z[j]]), np.diag([(0.1 * f) ** 2, (0.15 * f) ** 2]))
        res[scale] = p
    m = r.merged[r.track_merged[owner]]
    got = np.array([m["y"], m["z"], m["sinphi"], m["dzds"], m["qpt"]], np.float64)
    tol = 2e-5 * np.maximum(1.0, np.abs(res[2.0]))
    assert np.all(np.abs(got - res[2.0]) < tol), (got - res[2.0])
    assert np.any(np.abs(res[1.0] - res[2.0]) > 5 * tol), "the inflation is visible at this tolerance"
    # without inflation (scale 1) the merged fit of an unmerged track is the sector refit again (it only starts from the
    # refitted q/pT instead of the tracklet's: a rounding-level difference)
    r1 = _track(fr, row_x, merge=dict(shared_err_scale=1.0))
    for f in ("y", "z", "sinphi", "dzds", "qpt", "chi2"):
        assert np.allclose(r1.merged[f], r1.tracks[f][r1.merged["pad"][:, 4]], rtol=2e-5, atol=1e-6), f


# ---------------------------------------------------------------- invariants on a full event
@pytest.fixture(scope="module")
def event(row_x):
    fr = synth.generate(synth.config(2, scale=0.1, seed=6))
    return fr, _track(fr, row_x)


def test_merge_invariants(event):
    fr, r = event
    nt, nm = len(r.tracks), len(r.merged)
    assert nm < nt and (r.link_next >= 0).sum() == nt - nm > 100
    # every sector track in exactly one merged track; merged ids follow the heads in id order
    assert r.track_merged.min() == 0 and r.track_merged.max() == nm - 1
    heads = r.merged["pad"][:, 4]
    assert (np.diff(heads) > 0).all() and np.array_equal(r.track_merged[heads], np.arange(nm))
    prev = np.full(nt, -1)
    for a in np.flatnonzero(r.link_next >= 0):
        b = r.link_next[a]
        assert prev[b] == -1, "one partner per inner end"
        prev[b] = a
        sa, sb = r.tracks["sector"][a], r.tracks["sector"][b]
        assert sa // 18 == sb // 18 and (sa - sb) % 18 in (1, 17), "adjacent sectors of one side"
        dr = r.tracks["first_row"][b] - r.tracks["last_row"][a]
        assert -M["merge_row_back"] <= dr <= M["merge_row_fwd"]
        assert r.track_merged[a] == r.track_merged[b]
    assert np.array_equal(np.flatnonzero(prev < 0), heads)
    nh = np.bincount(r.track_merged, weights=r.tracks["n_hits"], minlength=nm)
    assert np.array_equal(nh.astype(int), r.merged["n_hits"])
    assert np.array_equal(np.bincount(r.track_merged, minlength=nm), r.merged["pad"][:, 0])
    ok = r.merged["pad"][:, 2] >= 0
    assert ok.mean() > 0.85 and (r.merged["ndf"][~ok] == -1).all()
    assert np.array_equal(r.merged["ndf"][ok], 2 * (r.merged["n_hits"][ok] - r.merged["pad"][ok][:, 2]) - 5)


def test_merge_joins_the_same_particle_and_lowers_the_clone_rate(event):
    fr, r = event
    sec = score.sector_of_cluster(fr.sector_offsets, fr.n)
    lab = np.array([np.bincount(fr.truth[r.assignment == t] + 1).argmax() - 1 for t in range(len(r.tracks))])
    a = np.flatnonzero(r.link_next >= 0)
    assert (lab[a] == lab[r.link_next[a]]).mean() > 0.995
    am = np.where(r.assignment >= 0, r.track_merged[np.maximum(r.assignment, 0)], -1)
    one = np.zeros_like(sec)  # score per particle, not per (particle, sector)
    before = score.score(r.assignment, fr.truth, one, len(r.tracks))
    after = score.score(am, fr.truth, one, len(r.merged))
    assert after["efficiency"] >= before["efficiency"] and after["fake_rate"] <= before["fake_rate"] + 1e-3
    assert after["clone_rate"] < before["clone_rate"] - 0.15, (before, after)


def test_merge_permutation_invariance(event, row_x):
    fr, r = event
    fp, p = synth.permute_within_sectors(fr, seed=123)
    rp = _track(fp, row_x)
    assert rp.merged.tobytes() == r.merged.tobytes()
    assert np.array_equal(rp.track_merged, r.track_merged) and np.array_equal(rp.link_next, r.link_next)


def test_merge_optimisation_level_independent(row_x):
    fr = synth.generate(synth.config(2, scale=0.03, seed=16))
    a = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, opt="-O2")
    b = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, opt="-O0")
    assert a.merged.tobytes() == b.merged.tobytes() and np.array_equal(a.link_next, b.link_next)
    assert np.array_equal(a.shared, b.shared) and a.outer.tobytes() == b.outer.tobytes()


def test_no_ring_no_merging(row_x):
    """A single standalone sector (config 1) or ring = 0 has no neighbours: every sector track is its own merged track."""
    fr = synth.generate(synth.config(1, scale=0.2, seed=1))
    r = _track(fr, row_x)
    assert len(r.merged) == len(r.tracks) > 10 and (r.link_next == -1).all()
    fr2, _ = scenarios.helix_in_two_sectors(row_x, sector=3, side=+1)
    r2 = _track(fr2, row_x, merge=dict(ring=0))
    assert len(r2.merged) == 2


# ---------------------------------------------------------------- the predicates of O9, one at a time
EARLY = dict(x0=85.0, y0=4.0, z0=25.0, sinphi0=0.2, tanl=0.5, qpt=-1.1, bz=0.5)  # leaves the sector at row 90


def _n_merged(row_x, merge=True, **kw):
    fr, info = scenarios.helix_in_two_sectors(row_x, sector=7, side=kw.pop("side", +1), par=EARLY, **kw)
    r = _track(fr, row_x, merge=merge)
    return len(r.merged), r, fr, info


def test_only_ends_near_the_sector_side_are_merged(row_x):
    """B2: the outer end of A must lie within merge_edge_dist of the sector's side.  A's last 6 rows are removed, so it ends
    ~1.3 cm inside: merged at the default 10 cm and at 2 cm, apart at 0.7 cm (the rest of the match is untouched)."""
    n, r, fr, info = _n_merged(row_x, drop_rows_a_end=6)
    a = int(np.flatnonzero(r.tracks["sector"] == 7)[0])
    dist = r.outer[a][0] * scenarios.TAN10 - abs(r.outer[a][1])
    assert 1.0 < dist < 1.6 and n == 1
    assert _n_merged(row_x, merge=dict(merge_edge_dist=0.7), drop_rows_a_end=6)[0] == 2
    assert _n_merged(row_x, merge=dict(merge_edge_dist=2.0), drop_rows_a_end=6)[0] == 1


def test_z_window(row_x):
    """B2: |z_B - z_A| <= merge_dz_max between the two ends.  One row apart the ends differ by tan(lambda) * arc ~ 0.6 cm."""
    n, r, fr, info = _n_merged(row_x)
    a = int(np.flatnonzero(r.tracks["sector"] == 7)[0])
    dz = abs(r.tracks["z"][1 - a] - r.outer[a][2])
    assert n == 1 and 0.3 < dz < 0.9
    assert _n_merged(row_x, merge=dict(merge_dz_max=float(dz) * 0.9))[0] == 2
    assert _n_merged(row_x, merge=dict(merge_dz_max=float(dz) * 1.1))[0] == 1


def test_row_window_backwards(row_x):
    """B2: first_row(B) - last_row(A) >= -merge_row_back (= -2): the segments may overlap by rows near the boundary (the
    row planes of two sectors differ).  A keeps its clusters 3 / 4 rows beyond the side: overlap 2 merges, 3 does not."""
    for ext, n_merged in ((3, 1), (4, 2)):
        n, r, fr, info = _n_merged(row_x, extend_a=ext)
        a = int(np.flatnonzero(r.tracks["sector"] == 7)[0])
        assert r.tracks["first_row"][1 - a] - r.tracks["last_row"][a] == 1 - ext
        assert n == n_merged, ext


def test_curvature_is_part_of_the_match(row_x):
    """B3: chi2 runs over all five parameters.  The continuation starts at the same point with the same direction and dip
    but the opposite curvature: position, sin(phi) and dz/ds agree at the boundary, q/pT does not -> no merge."""
    n_same, *_ = _n_merged(row_x, qpt_b=EARLY["qpt"])
    n_flip, r, fr, info = _n_merged(row_x, qpt_b=-EARLY["qpt"])
    assert n_same == 1 and len(r.tracks) == 2 and n_flip == 2
    a = int(np.flatnonzero(r.tracks["sector"] == 7)[0])
    assert r.tracks["qpt"][a] * r.tracks["qpt"][1 - a] < 0


def test_links_are_mutual_not_greedy(row_x):
    """B4: two inner segments compete for one continuation -- the true one and a copy displaced by -0.4 cm in z, which has
    the LOWER track id (ids follow z).  The continuation's best partner is the true one; a greedy first-come link would
    give it to the copy."""
    n, r, fr, info = _n_merged(row_x, merge=dict(merge_chi2_cut=1e6), copy_a_dz=-0.4)  # both candidates pass the cut
    assert len(r.tracks) == 3 and n == 2
    ids_a = np.flatnonzero(r.tracks["sector"] == 7)
    b = int(np.flatnonzero(r.tracks["sector"] == info["sector_b"])[0])
    true_a = ids_a[np.argmax(r.tracks["z"][ids_a])]
    assert true_a == ids_a.max(), "the displaced copy comes first in id order"
    assert r.link_next[true_a] == b and r.link_next[ids_a.min()] == -1
