"""Pins of the oracle's z / time estimate (step O11)."""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import synth
from tests.helix import KAPPA_PER_T, helix_points

V = oracle.DEFAULT_TIME_PARAMS["vdrift"]


def _brute_dca(state, bz=0.5):
    """Closest approach of the helix to the beam line by brute force: walk the circle in small steps of the turning angle
    (float64), take the point nearest to the origin, refine by a parabola."""
    x, y, z, s, t, q = [float(v) for v in state]
    k = -KAPPA_PER_T * bz * q
    phi = np.arcsin(s)
    if abs(k) < 1e-15:
        lam = np.linspace(-400, 100, 2000001)
        px, py = x + lam * np.cos(phi), y + lam * np.sin(phi)
        ds = lam
    else:
        dphi = np.linspace(-np.pi, np.pi, 4000001)
        px = x + (np.sin(phi + dphi) - np.sin(phi)) / k
        py = y - (np.cos(phi + dphi) - np.cos(phi)) / k
        ds = dphi / k
    r2 = px * px + py * py
    i = int(np.argmin(r2))
    a, b, c = r2[i - 1], r2[i], r2[i + 1]
    off = 0.5 * (a - c) / (a - 2 * b + c)
    return z + t * (ds[i] + off * (ds[1] - ds[0])), np.sqrt(max(b, 0.0))


@pytest.mark.parametrize("state", [(85.0, 20.3, 46.7, 0.168, 0.5, 1.0), (120.0, -30.0, -200.0, -0.4, -0.9, -3.0),
                                   (85.0, 5.0, 10.0, 0.05, 0.2, 0.0), (200.0, 10.0, 1500.0, 0.3, 0.7, 0.05),
                                   (100.0, 12.0, 60000.0, -0.2, 0.4, 6.0), (90.0, -14.0, -3.0, 0.6, -1.1, -8.0)])
def test_dca_is_the_closest_approach(state):
    """O11: z at the point of the helix nearest to the beam line, against brute force on the float64 circle; covers both
    signs of the curvature, the straight line, a stiff track, a 23 ms frame (z = 6e4 cm) and a looper-like radius."""
    zb, rb = _brute_dca(state)
    out = oracle.time_estimate_state(state, state[2], state[2], +1, z_max=1e9)
    assert abs(out[0] - zb) < 2e-4 * max(1.0, abs(zb) * 1e-2), (out, zb)
    assert abs(abs(out[3]) - rb) < 1e-3 * max(1.0, rb), (out, rb)


def test_straight_line_limit_is_continuous():
    a = oracle.time_estimate_state((85.0, 5.0, 10.0, 0.05, 0.2, 0.0), 10, 10, 1, z_max=1e9)
    b = oracle.time_estimate_state((85.0, 5.0, 10.0, 0.05, 0.2, 1e-6), 10, 10, 1, z_max=1e9)
    assert np.allclose(a, b, atol=1e-4)


@pytest.mark.parametrize("side", [+1, -1])
@pytest.mark.parametrize("pt,q,phi0,eta,zv,t0", [(0.3, 1, 0.1, 0.5, 3.0, 40.0), (1.5, -1, -0.05, 0.8, -4.0, 600.0),
                                                 (0.15, -1, -0.5, 0.3, 1.0, 5.0), (5.0, 1, 0.02, 0.6, 0.0, 22000.0)])
def test_primary_from_the_beam_line_gives_its_collision_time(row_x, pt, q, phi0, eta, zv, t0, side):
    """a primary helix from (0, 0, z_v) of a collision at time t0 (clusters shifted by side * v * t0,
    PAPER.md:93): the tracked, refitted track's z at closest approach is z_v + side * v * t0 and the time estimate is t0
    up to z_v / v -- for 5 us to 22 ms (z up to 5.7e4 cm: PAPER.md:121 single precision at large z), both drift sides."""
    tl = np.sinh(eta) * side
    xs = row_x.astype(np.float64)
    y, z, s = helix_points(xs, 0.0, 0.0, zv, np.sin(phi0), tl, q / pt, 0.5)
    ok = np.isfinite(y) & (np.abs(y) <= xs * np.tan(np.deg2rad(10))) & (np.abs(z) <= 250) & (z * side > 0)
    rows = np.flatnonzero(ok)
    assert len(rows) > 15
    cl = np.zeros(len(rows), synth.CLUSTER_DTYPE)
    cl["row"], cl["x"], cl["y"], cl["z"] = rows, row_x[rows], y[rows], z[rows] + side * V * t0
    so = np.zeros(37, np.int32)
    so[(4 if side > 0 else 22) + 1:] = len(cl)
    r = oracle.track(cl, so, row_x, merge=True, time=True)
    assert len(r.tracks) == 1 and len(r.merged) == 1
    zd, sh, t_est, dca = r.time_merged[0]
    zexp = zv + side * V * t0
    assert abs(zd - zexp) < 2e-3 + 4e-7 * abs(zexp), (zd, zexp)   # fp32: a few ulp of z
    assert abs(dca) < 2e-3
    assert abs(t_est - t0 - side * zv / V) < 1e-3 + 1e-6 * t0 or sh != zd
    assert np.allclose(r.time_sector[0], r.time_merged[0], rtol=1e-5, atol=2e-3)


def test_clusters_are_shifted_inside_the_drift_volume():
    """a secondary's closest approach says nothing about its vertex; if the shift would put clusters outside
    the physical drift volume [0, z_max] of their side, the shift is moved to the nearest value that keeps them inside."""
    st = (85.0, 5.0, 1000.0, 0.05, 2.0, 1.0)  # steep track: z at closest approach ~ 1000 - 2 * 85
    zd = oracle.time_estimate_state(st, 1000.0, 1000.0, +1, z_max=1e9)[0]
    assert 820 < zd < 840
    # clusters span [1000, 1200]: shift must be >= 1200 - 250 = 950 (else the last cluster sits beyond the end plate)
    out = oracle.time_estimate_state(st, 1000.0, 1200.0, +1)
    assert out[0] == zd and out[1] == 950.0 and abs(out[2] - 950.0 / V) < 1e-3
    # clusters span [700, 900] with z_dca = 830: a cluster would get z - shift < 0 -> shift <= 700
    out = oracle.time_estimate_state(st, 700.0, 900.0, +1)
    assert out[1] == 700.0
    # inside the allowed interval nothing moves
    out = oracle.time_estimate_state(st, 900.0, 1000.0, +1)
    assert out[1] == out[0] == zd
    # side C is the mirror image: -z_max <= z - shift <= 0
    stc = (85.0, 5.0, -1000.0, 0.05, -2.0, 1.0)
    out = oracle.time_estimate_state(stc, -1200.0, -1000.0, -1)
    assert abs(out[0] + zd) < 1e-3 and out[1] == -950.0 and abs(out[2] - 950.0 / V) < 1e-3


def test_time_estimates_on_a_time_frame(row_x):
    """Config 4 (5 collisions in 100 us): for particles that cross the TPC once, z at closest approach equals
    z_v + side * v * t0 to 1 mm (68 %), so the time estimate is t0 + side * z_v / v: t0 up to the vertex spread
    (sigma 5 cm / v = 1.9 us), which is what the paper's "assumed as z-position ... of the primary vertex" accepts."""
    fr = synth.generate(synth.config(4, scale=0.05, seed=4))
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x, merge=True, time=True)
    am = np.where(r.assignment >= 0, r.track_merged[np.maximum(r.assignment, 0)], -1)
    tp = fr.track_par
    ez, et = [], []
    for m in range(len(r.merged)):
        idx = np.flatnonzero(am == m)
        lab = np.bincount(fr.truth[idx] + 1).argmax() - 1
        if lab < 0:
            continue
        pitch = 2 * np.pi * tp[lab, 0] / (KAPPA_PER_T * 0.5) * abs(np.sinh(tp[lab, 2]))
        if pitch < 500:  # the generator lets helices go round again; later turns have another z at closest approach
            continue
        side = 1 if r.merged["sector"][m] < 18 else -1
        ez.append(r.time_merged[m, 0] - (tp[lab, 4] + side * V * tp[lab, 5]))
        if r.time_merged[m, 1] == r.time_merged[m, 0]:  # not clamped by the volume rule
            et.append(r.time_merged[m, 2] - (tp[lab, 5] + side * tp[lab, 4] / V))
    ez, et = np.abs(ez), np.abs(et)
    assert len(ez) > 300
    assert np.percentile(ez, 68) < 0.1 and np.percentile(ez, 95) < 0.3, np.percentile(ez, [68, 95])
    # the time estimate is t0 + side * z_v / v (the vertex is assumed at z = 0): exact up to the z_dca error
    assert len(et) > 0.9 * len(ez) and np.percentile(et, 68) < 0.1 / V, np.percentile(et, 68)
