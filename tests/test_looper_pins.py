"""Pins of the oracle's looper-leg finder and cluster tags (steps O12-O13) against what the paper and
the mathematics fix.  PAPER.md:123 "additional legs of looping tracks do not point to the vertex ... special low-pT track
merging"; :157 clusters to remove: "very low-pT looping tracks below 50 MeV/c, additional legs of tracks below 200 MeV/c,
and track segments with high inclination angle".  Helices come from tests/looper.py (float64 closed form, written for the
tests), so which cluster lies on which leg is known by construction.  None of these call the CUDA path."""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import synth
from tests import looper

L = oracle.DEFAULT_LEG_PARAMS
KQ = -0.00299792458 * 0.5  # curvature per q/pT at Bz = 0.5 T (tests/helix.py convention)


def _run(fr, row_x, legs=True, **kw):
    return oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, legs=legs, **kw)


def _merged_of_cluster(res):
    a = res.assignment
    return np.where(a >= 0, res.track_merged[np.maximum(a, 0)], -1)


# ---------------------------------------------------------------- the angle polynomial
def test_angle_polynomial_is_arctan2_on_the_upper_half_plane():
    """O12 needs the turning angle without libm: octant reduction + Abramowitz-Stegun 4.4.49.  Against numpy float64."""
    worst = 0.0
    for a in np.r_[np.linspace(1e-3, np.pi - 1e-3, 721), [np.pi / 4, np.pi / 2, 3 * np.pi / 4]]:
        for r in (0.3, 1.0, 57.0):
            y, x = np.float32(r * np.sin(a)), np.float32(r * np.cos(a))
            worst = max(worst, abs(oracle.angle_upper(y, x) - np.arctan2(float(y), float(x))))
    assert worst < 6e-7, worst  # 2e-8 of the polynomial + fp32 rounding of an angle of order pi


# ---------------------------------------------------------------- one end: circle from the state
@pytest.mark.parametrize("q", [+1, -1])
@pytest.mark.parametrize("R,cx,cy,s", [(80.0, 70.0, 30.0, 0.9), (60.0, 100.0, -20.0, -0.7), (150.0, 60.0, 10.0, 0.6)])
def test_end_geometry_is_the_circle_through_the_state(R, cx, cy, s, q):
    """Radius 1/|k| and centre (x - s/k, y + c/k): a state ON a float64 circle must give back that circle."""
    w = -q  # Bz > 0: positive charge turns clockwise
    # point of the circle where the fit direction (cos phi > 0) has sin(phi) = s: tangent = w * (-sin a, cos a)
    c = np.sqrt(1 - s * s)
    a = np.arctan2(-w * c, w * s)  # solves w*(-sin a) = c ... direction (c, s)
    x, y = cx + R * np.cos(a), cy + R * np.sin(a)
    qpt = q / (R * abs(KQ))
    cand, Ro, xc, yc, co = oracle.leg_end([3, x, y, 12.0, s, 0.2, qpt], x_last=245.0)
    assert abs(Ro - R) < 1e-4 * R and abs(xc - cx) < 2e-4 * R and abs(yc - cy) < 2e-4 * R and abs(co - c) < 1e-6
    assert cand == (cx + R <= 247.0) or abs(cx + R - 247.0) < 1e-3


def test_candidate_cuts():
    """q = -7 at Bz = 0.5 T: k = +0.0105 / cm, R = 95.3 cm; with sin(phi) = +0.9 the centre lies at x - 0.9 R and the
    turning point at x + 0.1 R."""
    base = dict(x=160.0, y=5.0, z=0.0, s=0.9, t=0.1, q=-7.0)

    def cand(**kw):
        d = dict(base, **kw)
        return oracle.leg_end([0, d["x"], d["y"], d["z"], d["s"], d["t"], d["q"]], x_last=245.0)[0]

    assert cand() and cand(q=7.0, s=-0.9)                               # mirror image
    assert not cand(q=-3.9) and cand(q=-4.1) and cand(q=4.1, s=-0.9)    # leg_min_qpt = 4 (pT < 250 MeV/c)
    assert not cand(s=0.49) and cand(s=0.51)                            # leg_min_sinphi = 0.5
    assert not cand(q=7.0)              # sin(phi) moving AWAY from +-1 along the fit direction: the turning point is far outside
    assert cand(x=237.0) and not cand(x=238.0)                          # 237 + 9.53 <= 245 + 2 < 238 + 9.53


# ---------------------------------------------------------------- pairs: two ends of one float64 circle
def _two_ends(q, j, sec_a=3, R=90.0, tanl=0.35, sa=0.9, sb=0.92, za=40.0):
    """Outer end of the outgoing leg in sector sec_a (sin phi = +-sa towards the apex) and outer end of the returning leg
    j sectors further in the turning sense, on ONE float64 helix.  Returns (a7, b7, turn angle)."""
    w = -q
    k = w / R                      # d(phi)/ds, signed
    qpt = k / KQ
    # A: fit direction = physical direction, azimuth phi_a in A's frame, sin(phi_a) = w * sa (heading for the apex)
    phi_a = np.arcsin(w * sa)
    xa, ya = 150.0, 4.0
    cx, cy = xa - np.sin(phi_a) / k, ya + np.cos(phi_a) / k
    # B: physical azimuth in B's frame = pi - asin(w*sb) ... returning leg: its FIT direction has sin(phi) = -w*sb
    al = np.deg2rad(20.0 * j) * w  # B's frame axis relative to A's
    phi_b_fit = np.arcsin(-w * sb)          # in B's frame
    phi_b_phys = phi_b_fit + np.pi + al     # in A's frame
    turn = ((phi_b_phys - phi_a) * w) % (2 * np.pi)
    # point of the circle with physical azimuth phi_b_phys: centre + R * (sin, -cos) * w
    xb_a = cx + np.sin(phi_b_phys) / k
    yb_a = cy - np.cos(phi_b_phys) / k
    xb = xb_a * np.cos(al) + yb_a * np.sin(al)
    yb = -xb_a * np.sin(al) + yb_a * np.cos(al)
    zb = za + tanl * R * turn
    base = (sec_a // 18) * 18
    sec_b = base + (sec_a - base + w * j) % 18
    a7 = [sec_a, xa, ya, za, np.sin(phi_a), tanl, qpt]
    b7 = [sec_b, xb, yb, zb, -w * sb, -tanl, -qpt]
    return a7, b7, turn


@pytest.mark.parametrize("q", [+1, -1])
@pytest.mark.parametrize("j", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("sec_a", [3, 17, 18, 26])
def test_two_ends_of_one_helix_match_with_score_zero(q, j, sec_a):
    a7, b7, turn = _two_ends(q, j, sec_a)
    if turn > L["leg_max_turn"]:
        assert oracle.leg_pair(a7, b7) < 0
        return
    sc = oracle.leg_pair(a7, b7)
    assert 0 <= sc < 2e-4, (sc, turn)
    assert abs(oracle.leg_pair(b7, a7) - sc) < 2e-4  # either leg may carry the lower id


def test_each_term_of_the_score_is_what_table_d_says():
    a7, b7, turn = _two_ends(+1, 2)
    R = 90.0
    # z off by 2 cm: (2 / leg_dz_max)^2 -- this also pins arc = turn * R (a chord or a wrong angle would not give zero above)
    b = list(b7); b[3] += 2.0
    assert abs(oracle.leg_pair(a7, b) - 0.25) < 2e-3
    b = list(b7); b[3] += 4.1
    assert oracle.leg_pair(a7, b) < 0
    # dz/ds off by 0.05: the mean slope moves z by 0.025 * arc as well
    b = list(b7); b[5] += 0.05
    arc = turn * R
    want = (0.05 / 0.1) ** 2 + ((0.025 * arc) / 4.0) ** 2
    got = oracle.leg_pair(a7, b)
    assert (got < 0 and 0.025 * arc > 4.0) or abs(got - want) < 0.02 * want, (got, want)
    b = list(b7); b[5] += 0.11
    assert oracle.leg_pair(a7, b) < 0
    # centre off by 3 cm (shift B along its frame's y): tol = 0.05 R + 1.5 = 6 cm -> (3/6)^2
    b = list(b7); b[2] += 3.0
    assert abs(oracle.leg_pair(a7, b) - 0.25) < 5e-3
    b = list(b7); b[2] += 6.2
    assert oracle.leg_pair(a7, b) < 0
    b = list(b7); b[5] += 0.11; b[3] -= 0.055 * arc   # z made consistent with the new mean slope: only the slope sum is off
    assert oracle.leg_pair(a7, b) < 0
    b = list(b7); b[5] += 0.09; b[3] -= 0.045 * arc
    assert abs(oracle.leg_pair(a7, b) - 0.81) < 0.02
    # same sign of sin(phi) with opposite curvature: the ends lie half a turn apart, beyond leg_max_turn < pi
    b = list(b7); b[4] = -b[4]
    assert oracle.leg_pair(a7, b) < 0
    # the partner must lie AHEAD in the turning sense, at most leg_max_sector_gap sectors, on the same z side
    b = list(b7); b[0] = (a7[0] + 2) % 18      # q = +1 turns clockwise: sector 3 -> 1; sector 5 is behind
    assert oracle.leg_pair(a7, b) < 0
    b = list(b7); b[0] = b7[0] + 18
    assert oracle.leg_pair(a7, b) < 0
    a6, b6, t6 = _two_ends(+1, 6, sa=0.95, sb=0.95)  # 6 sectors ahead with a turn of 156 degrees: only the gap cut rejects it
    assert t6 < L["leg_max_turn"] and oracle.leg_pair(a6, b6) < 0 <= oracle.leg_pair(a6, b6, legs=dict(leg_max_sector_gap=6))
    assert oracle.leg_pair(a7, b7, legs=dict(leg_max_turn=float(turn) - 0.01)) < 0 <= oracle.leg_pair(a7, b7, legs=dict(leg_max_turn=float(turn) + 0.01))


def test_a_broken_flat_track_is_not_a_pair_of_legs():
    """Two outer ends on ONE circle traversed in the SAME sense (a flat track broken in two: B ends at sin(phi) = -0.9,
    A further along at +0.9, same z because dz/ds = 0): centre, radius, z and slope sum all agree, the turning angle from
    A to B reversed is 52 degrees -- only the curvature signs say that these are not the two legs of a turn."""
    R, q = 90.0, -1
    k = 1.0 / R
    qpt = k / KQ
    cx, cy = 100.0, 0.0
    pa, pb = np.arcsin(0.9), np.arcsin(-0.9)
    a7 = [4, cx + np.sin(pa) / k, cy - np.cos(pa) / k, 50.0, 0.9, 0.0, qpt]
    b7 = [4, cx + np.sin(pb) / k, cy - np.cos(pb) / k, 50.0, -0.9, 0.0, qpt]
    assert oracle.leg_end(a7)[0] and oracle.leg_end(b7)[0]
    assert oracle.leg_pair(a7, b7) < 0 and oracle.leg_pair(b7, a7) < 0


def test_radius_term():
    a7, b7, _ = _two_ends(-1, 1, R=90.0)
    # B's radius 4 % smaller with its centre kept in place: move the end point towards the centre accordingly
    w, R = 1, 90.0
    k_b = b7[6] * KQ
    cxb, cyb = b7[1] - b7[4] / k_b, b7[2] + np.sqrt(1 - b7[4] ** 2) / k_b
    f = 0.96
    b = list(b7)
    b[6] = b7[6] / f
    b[1] = cxb + (b7[1] - cxb) * f
    b[2] = cyb + (b7[2] - cyb) * f
    Rm = 0.5 * (R + f * R)
    want = ((R - f * R) / (0.2 * Rm)) ** 2
    got = oracle.leg_pair(a7, b)
    # the arc shortens with the mean radius: z term (tanl * turn * (R - Rm)) on top
    a7_, b7_, turn = _two_ends(-1, 1, R=90.0)
    want += ((0.35 * turn * (R - Rm)) / 4.0) ** 2
    assert abs(got - want) < 0.03 * want + 1e-3, (got, want)
    # a flat helix (no z term): radius 25 % smaller around the same centre -> only the radius cut (20 % of the mean) rejects
    a0, b0, _ = _two_ends(-1, 1, R=90.0, tanl=0.0)
    for f, ok in ((0.75, False), (0.85, True)):
        b = list(b0)
        b[6] = b0[6] / f
        b[1] = cxb + (b0[1] - cxb) * f
        b[2] = cyb + (b0[2] - cyb) * f
        sc = oracle.leg_pair(a0, b)
        assert (sc >= 0) == ok, (f, sc)
        if ok:
            assert abs(sc - ((1 - f) / (0.2 * 0.5 * (1 + f))) ** 2) < 0.01


# ---------------------------------------------------------------- inner ends: the passage below the first pad row
def _end_on_circle(cx, cy, R, w, a, z, tanl):
    """Fitted-state view (sector, x, y, z, sin phi, dz/ds, q/pT) of the point at angle `a` of a float64 circle (centre
    (cx, cy) in the global frame, sense of rotation w = +-1), side A: the fit runs with cos(phi) > 0 in the sector frame,
    so a particle flying inward is described against its flight (sin phi, dz/ds and q/pT change sign)."""
    gx, gy = cx + R * np.cos(a), cy + R * np.sin(a)
    sec = int(np.floor((np.degrees(np.arctan2(gy, gx)) % 360.0) / 20.0))
    al = np.deg2rad(20.0 * sec + 10.0)
    x = gx * np.cos(al) + gy * np.sin(al)
    y = -gx * np.sin(al) + gy * np.cos(al)
    ta = a + w * np.pi / 2 - al                      # direction of flight in the sector frame
    k = w / R
    qpt = k / KQ
    if np.cos(ta) > 0:
        return [sec, x, y, z, np.sin(ta), tanl, qpt]
    return [sec, x, y, z, -np.sin(ta), -tanl, -qpt]


def _inner_pair(R, w, tanl=0.3, d=0.0, phi=0.4, r_in=85.0, z1=50.0):
    """Two points at radius r_in of a circle that passes at distance d from the beam line: where the particle dives below
    the first pad row (end of a returning leg) and where it comes out again (start of the next outgoing leg).
    Returns (returning leg's inner end, outgoing leg's inner end, turning angle between them)."""
    rc = R + d                                      # distance of the centre from the beam line
    cx, cy = rc * np.cos(phi), rc * np.sin(phi)
    # points of the circle at distance r_in from the origin: angle g from the direction centre -> origin
    cosg = (R * R + rc * rc - r_in * r_in) / (2 * R * rc)
    g = np.arccos(cosg)
    a0 = phi + np.pi                                # point of the circle nearest to the beam line
    a_in, a_out = a0 - w * g, a0 + w * g            # flight order: a_in, nearest point, a_out
    turn = 2 * g
    e_in = _end_on_circle(cx, cy, R, w, a_in, z1, tanl)
    e_out = _end_on_circle(cx, cy, R, w, a_out, z1 + tanl * R * turn, tanl)
    return e_in, e_out, turn


@pytest.mark.parametrize("w", [+1, -1])
@pytest.mark.parametrize("R,d", [(95.0, 0.0), (80.0, 0.0), (55.0, 0.0), (47.0, 0.0), (70.0, 6.0), (120.0, -4.0)])
@pytest.mark.parametrize("phi", [0.4, 2.0, 5.9])
def test_two_inner_ends_of_one_helix_match_with_score_zero(R, d, w, phi):
    """Through the region below the first pad row the particle turns by 2*acos(...) -- more than half a turn for R < 60 cm
    -- and, passing close to the beam line, comes out up to nine sectors away on either side."""
    e_in, e_out, turn = _inner_pair(R, w, d=d, phi=phi)
    assert 1.2 < turn < 5.0
    for a7, b7 in ((e_in, e_out), (e_out, e_in)):   # either leg may carry the lower id
        sc = oracle.leg_pair(a7, b7, sig=-1)
        assert 0 <= sc < 5e-4, (sc, turn, e_in, e_out)
    assert oracle.leg_pair(e_in, e_out, sig=+1) < 0          # as OUTER ends these two do not continue into each other


def test_inner_pair_terms():
    e_in, e_out, turn = _inner_pair(80.0, +1, tanl=0.3)
    R = 80.0
    # z: along the continuation of an inner end the slope has the opposite sign of the fitted one
    b = list(e_out); b[3] += 2.0
    assert abs(oracle.leg_pair(e_in, b, sig=-1) - 0.25) < 3e-3
    b = list(e_out); b[3] -= 2 * 0.3 * R * turn      # the z a wrong slope sign would predict
    assert oracle.leg_pair(e_in, b, sig=-1) < 0
    # turn limit and sector limit of the inner kind are their own parameters
    assert oracle.leg_pair(e_in, e_out, sig=-1, legs=dict(leg_inner_max_turn=float(turn) - 0.01)) < 0
    assert oracle.leg_pair(e_in, e_out, sig=-1, legs=dict(leg_inner_max_turn=float(turn) + 0.01, leg_max_turn=0.1)) >= 0
    dsec = (e_out[0] - e_in[0]) % 18
    dsec = min(dsec, 18 - dsec)
    assert dsec >= 4
    assert oracle.leg_pair(e_in, e_out, sig=-1, legs=dict(leg_inner_max_sector_gap=dsec - 1)) < 0
    assert oracle.leg_pair(e_in, e_out, sig=-1, legs=dict(leg_inner_max_sector_gap=dsec, leg_max_sector_gap=0)) >= 0
    # candidates: the inner kind has its own sin(phi) threshold and no turning-point condition
    st = [3, 85.0, 2.0, 10.0, 0.3, 0.2, 7.0]
    assert oracle.leg_end(st, sig=-1)[0] and not oracle.leg_end(st, sig=+1)[0]
    st[4] = 0.15
    assert not oracle.leg_end(st, sig=-1)[0]
    big = [3, 85.0, 2.0, 10.0, 0.3, 0.2, 4.5]      # R = 148 cm: the helix leaves the TPC on its way out, but it came from below
    assert oracle.leg_end(big, sig=-1)[0] and not oracle.leg_end([3, 240.0, 2.0, 10.0, -0.9, 0.2, 4.5], sig=+1)[0]
    # more than half a turn: the angle comes from the lower half plane (R = 47 cm: 258 degrees)
    e_in, e_out, turn = _inner_pair(47.0, -1, tanl=0.2)
    assert turn > np.pi + 0.5
    b = list(e_out); b[3] += 1.0
    assert abs(oracle.leg_pair(e_in, b, sig=-1) - 1.0 / 16) < 2e-3   # pins arc = turn * R beyond pi


def test_two_turns_are_chained_through_the_inner_region(row_x):
    """Two full turns of a 120 MeV/c particle: outgoing 1 -(turning point)- returning 1 -(inner region)- outgoing 2
    -(turning point)- returning 2.  One chain, its first leg is outgoing 1, every other leg is tagged as additional."""
    for q in (+1, -1):
        p = looper.helix_clusters(row_x, 0.12, 0.7, 0.3, q, z0=10.0, turns=2.0, z_max=400.0)
        fr, info = looper.frame_from([p])
        res = _run(fr, row_x)
        am = _merged_of_cluster(res)
        nm = len(res.merged)
        assert nm == 4
        th = np.array([info["theta"][am == m].mean() for m in range(nm)])
        order = np.argsort(th)                      # flight order of the four legs
        o1, r1, o2, r2 = order
        assert res.leg_partner[o1] == r1 and res.leg_partner[o2] == r2
        assert res.leg_partner_in[r1] == o2 and res.leg_partner_in[o2] == r1
        assert res.leg_partner_in[o1] == -1 and res.leg_partner_in[r2] == -1
        assert list(res.leg_first[order]) == [1, 0, 0, 0]
        extra = (res.cluster_tags & oracle.TAG_EXTRA_LEG) > 0
        assert np.array_equal(extra, (am >= 0) & (am != o1))


# ---------------------------------------------------------------- whole path on hand-built loopers
def test_noiseless_looper_outgoing_and_returning_leg_are_linked(row_x):
    """One 120 MeV/c particle from the origin: the chain of sector segments up to the turning point and the chain coming
    back are two merged tracks (the merger cannot pass |sin phi| = 0.95); O12 links exactly these two; the first leg is the
    outgoing one; O13 tags every cluster of the returning leg and nothing else as additional leg."""
    for q in (+1, -1):
        p = looper.helix_clusters(row_x, 0.12, 0.7, 0.3 * q, q, z0=10.0 * q)
        fr, info = looper.frame_from([p])
        res = _run(fr, row_x)
        assert len(res.merged) == 2
        assert list(res.leg_partner) == [1, 0] and sorted(res.leg_first) == [0, 1]
        am = _merged_of_cluster(res)
        first = int(np.argmax(res.leg_first))
        assert info["outgoing"][am == first].all() and not info["outgoing"][am == 1 - first].any()
        extra = (res.cluster_tags & oracle.TAG_EXTRA_LEG) > 0
        assert np.array_equal(extra, am == 1 - first)
        assert not (res.cluster_tags & oracle.TAG_LOW_PT).any()


def test_high_inclination_tag_is_the_local_sinphi(row_x):
    """sin(phi) is linear in x along a helix, so the tag of every tracked cluster can be checked against the float64 truth;
    clusters within 0.01 of the threshold may go either way (the fit is not the truth)."""
    p = looper.helix_clusters(row_x, 0.10, 2.1, -0.4, -1, z0=-30.0)
    fr, info = looper.frame_from([p])
    res = _run(fr, row_x)
    on = res.assignment >= 0
    tag = (res.cluster_tags & oracle.TAG_HIGH_INCLINATION) > 0
    s = np.abs(info["sinphi"])
    clear = on & (np.abs(s - L["tag_sinphi"]) > 0.01)
    assert clear.sum() > 60 and np.array_equal(tag[clear], (s > L["tag_sinphi"])[clear])
    assert not tag[~on].any() and (res.cluster_tags[~on] == 0).all()
    res2 = _run(fr, row_x, legs=dict(tag_sinphi=0.6))
    tag2 = (res2.cluster_tags & oracle.TAG_HIGH_INCLINATION) > 0
    clear2 = on & (np.abs(s - 0.6) > 0.01)
    assert np.array_equal(tag2[clear2], (s > 0.6)[clear2]) and tag2.sum() > tag.sum()


def test_turns_of_a_flat_looper_pair_up_turn_by_turn(row_x):
    """Three turns with a pitch of 12 cm in z: six legs on one circle in xy.  The z term must pair the legs of the SAME
    turn (mutual best, not first come): partner's mean turn angle differs by less than one turn."""
    p = looper.helix_clusters(row_x, 0.13, -1.0, 0.022, +1, z0=5.0, turns=3.0)
    fr, info = looper.frame_from([p])
    res = _run(fr, row_x)
    am = _merged_of_cluster(res)
    nm = len(res.merged)
    assert nm == 6 and (res.leg_partner >= 0).all()
    turn_of = [int(np.floor(info["theta"][am == m].mean() / (2 * np.pi))) for m in range(nm)]
    for m in range(nm):
        assert res.leg_partner[res.leg_partner[m]] == m
        assert turn_of[m] == turn_of[res.leg_partner[m]], (m, turn_of)
    assert sorted(turn_of) == [0, 0, 1, 1, 2, 2]
    # with a z window wider than the pitch the pairing is still right: the score decides, not the first candidate in range
    res = _run(fr, row_x, legs=dict(leg_dz_max=30.0))
    assert all(turn_of[m] == turn_of[res.leg_partner[m]] for m in range(nm))


def test_very_low_pt_track_inside_the_tpc_is_tagged(row_x):
    """A 45 MeV/c secondary (R = 30 cm) born at r = 150 cm circles inside the TPC: every tracked cluster carries the
    low-pT tag (|q/pT| > 20); a 120 MeV/c particle carries none."""
    lo = looper.helix_clusters(row_x, 0.045, 0.3, 0.25, +1, z0=20.0, origin=(150.0 * np.cos(0.45), 150.0 * np.sin(0.45)), turns=2.0)
    hi = looper.helix_clusters(row_x, 0.12, 3.0, 0.3, -1, z0=10.0)
    fr, info = looper.frame_from([lo, hi])
    res = _run(fr, row_x)
    on = res.assignment >= 0
    low = (res.cluster_tags & oracle.TAG_LOW_PT) > 0
    assert (on & (fr.truth == 0)).sum() >= 40
    assert low[on & (fr.truth == 0)].all() and not low[fr.truth == 1].any()


def test_additional_leg_tag_has_its_own_momentum_threshold(row_x):
    """PAPER.md:157 removes "additional legs of tracks below 200 MeV/c": legs are linked up to 250 MeV/c (leg_min_qpt = 4)
    but tagged only above tag_qpt_leg = 5 (1/GeV).  A 150 MeV/c looper (|q/pT| = 6.7): tagged with the default threshold,
    linked but untagged once the threshold is 7."""
    p = looper.helix_clusters(row_x, 0.15, 1.3, 0.2, -1, z0=15.0)
    fr, info = looper.frame_from([p])
    for thr, tagged in ((5.0, True), (7.0, False)):
        res = _run(fr, row_x, legs=dict(tag_qpt_leg=thr))
        assert (res.leg_partner >= 0).sum() == 2, res.leg_partner
        n = int(((res.cluster_tags & oracle.TAG_EXTRA_LEG) > 0).sum())
        assert (n >= 20) if tagged else (n == 0), (thr, n)


def test_stiff_tracks_have_no_legs_and_no_tags(row_x):
    fr = synth.generate(synth.config(1, scale=0.3))
    res = _run(fr, row_x, legs=dict(ring=0))
    pt_ok = np.abs(res.merged["qpt"]) < 4.0
    assert (res.leg_partner[pt_ok] < 0).all() and (res.leg_first == 1)[pt_ok].all()
    assert not (res.cluster_tags & (oracle.TAG_LOW_PT | oracle.TAG_EXTRA_LEG)).any()


# ---------------------------------------------------------------- event level
@pytest.fixture(scope="module")
def event(row_x):
    fr = synth.generate(synth.config(3, scale=0.3, seed=3))
    return fr, _run(fr, row_x)


def _chains(res):
    """Union of both kinds of links: chain label of every merged track."""
    nm = len(res.merged)
    parent = np.arange(nm)

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x

    for lp in (res.leg_partner, res.leg_partner_in):
        for m in np.where(lp >= 0)[0]:
            parent[find(m)] = find(lp[m])
    return np.array([find(m) for m in range(nm)])


def test_leg_invariants(event):
    fr, res = event
    lf = res.leg_first
    nm = len(res.merged)
    q = res.merged["qpt"]
    for lp, n_min in ((res.leg_partner, 400), (res.leg_partner_in, 300)):
        linked = np.where(lp >= 0)[0]
        assert len(linked) >= n_min and len(linked) % 2 == 0
        assert np.array_equal(lp[lp[linked]], linked) and (lp[linked] != linked).all()   # an involution without fixed points
        assert (q[linked] * q[lp[linked]] < 0).all()                                     # neighbouring legs are fitted in opposite senses
    # exactly one first leg per chain, and it is the leg whose inner end lies at the smallest |z|
    root = _chains(res)
    z = np.abs(res.merged["z"])
    for r in np.unique(root):
        members = np.where(root == r)[0]
        firsts = members[lf[members] == 1]
        assert len(firsts) == 1
        assert z[firsts[0]] == z[members].min()
    tags = res.cluster_tags
    assert (tags[res.assignment < 0] == 0).all() and (tags < 8).all()
    am = _merged_of_cluster(res)
    extra = (tags & oracle.TAG_EXTRA_LEG) > 0
    want = (am >= 0) & (lf[np.maximum(am, 0)] == 0) & (np.abs(q[np.maximum(am, 0)]) > L["tag_qpt_leg"])
    assert np.array_equal(extra, want)


def test_legs_join_the_same_particle(event):
    """Against the generator's truth: both legs of every link carry the same particle label, and that particle is a looper
    (pT < 250 MeV/c).  PAPER.md:129 style labels: majority truth id of a track's clusters."""
    fr, res = event
    am = _merged_of_cluster(res)
    nm = len(res.merged)
    lab = np.full(nm, -1)
    order = np.argsort(am, kind="stable")
    a = am[order]
    for m in range(nm):
        s, e = np.searchsorted(a, m), np.searchsorted(a, m, side="right")
        l = fr.truth[order[s:e]]
        l = l[l >= 0]
        if len(l):
            lab[m] = np.bincount(l).argmax()
    for lp in (res.leg_partner, res.leg_partner_in):
        linked = np.where(lp > np.arange(nm))[0]
        same = lab[linked] == lab[lp[linked]]
        assert same.mean() >= 0.99, same.mean()
        assert (fr.track_par[lab[linked], 0] < 0.25).all()
    linked = np.where(res.leg_partner > np.arange(nm))[0]
    # a sizeable share of the loopers that reach the TPC have their first turn linked
    loopers = np.where((fr.track_par[:, 0] < 0.15) & (fr.track_par[:, 0] > 0.07))[0]
    found = np.isin(loopers, lab[linked]).mean()
    assert found > 0.6, found


def test_legs_permutation_invariance(event, row_x):
    fr, res = event
    fr2, p = synth.permute_within_sectors(fr, 11)
    res2 = _run(fr2, row_x)
    assert np.array_equal(res2.leg_partner, res.leg_partner) and np.array_equal(res2.leg_first, res.leg_first)
    assert np.array_equal(res2.leg_partner_in, res.leg_partner_in)
    assert np.array_equal(res2.cluster_tags, res.cluster_tags[p])


def test_legs_optimisation_level_independent(row_x):
    fr = synth.generate(synth.config(3, scale=0.1, seed=5))
    a = _run(fr, row_x)
    b = _run(fr, row_x, opt="-O0")
    assert np.array_equal(a.leg_partner, b.leg_partner) and np.array_equal(a.cluster_tags, b.cluster_tags)
    assert np.array_equal(a.leg_partner_in, b.leg_partner_in) and np.array_equal(a.leg_first, b.leg_first)
