"""Pins of the CPU oracle against what the paper and the mathematics fix (P1-P11).

None of these call the CUDA path.  Each pin is chosen so that a plausible mistake in the oracle
(dropped Jacobian term, wrong curvature sign, transposed covariance index, non-mutual link,
grid search missing a candidate) fails it.
"""
import numpy as np
import pytest

import oracle
from paper_1811_11481_b200 import score, synth
from tests.helix import KAPPA_PER_T, helix_points

CL = synth.CLUSTER_DTYPE


def _mk(rows, y, z, rx):
    cl = np.zeros(len(rows), CL)
    cl["row"] = rows
    cl["x"] = rx[rows]
    cl["y"] = y
    cl["z"] = z
    return cl


def _same(a, b):
    for f in ("link_up_raw", "link_down_raw", "link_up", "link_down", "start_hits", "row_hit", "assignment",
              "tracklet_ints", "track_tracklet"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert a.tracks.tobytes() == b.tracks.tobytes()
    assert a.tracklet_floats.tobytes() == b.tracklet_floats.tobytes()


# ---------------------------------------------------------------- P1
def _brute_links_py(cl, rx, P):
    """All-triplet search, no acceleration structure, numpy float32 scalars (O2)."""
    f = np.float32
    n = len(cl)
    up, dn = np.full(n, -1, np.int32), np.full(n, -1, np.int32)
    rows = cl["row"]
    R = len(rx)
    occupied = [np.flatnonzero(rows == r) for r in range(R)]
    inv_sy2 = f(1) / (f(P["sigma_y"]) * f(P["sigma_y"]))
    inv_sz2 = f(1) / (f(P["sigma_z"]) * f(P["sigma_z"]))

    def key(i):
        return (float(cl["z"][i]), float(cl["y"][i]), int(i))

    def fma(a, b, c):  # the fused multiply-add of DESIGN.md section 3: float32 x float32 is exact in float64
        return f(np.float64(a) * np.float64(b) + np.float64(c))

    for r in range(R):
        ru = r + 1 if r + 1 < R and len(occupied[r + 1]) else (r + 2 if r + 2 < R and len(occupied[r + 2]) else -1)
        rd = r - 1 if r - 1 >= 0 and len(occupied[r - 1]) else (r - 2 if r - 2 >= 0 and len(occupied[r - 2]) else -1)
        if ru < 0 or rd < 0:
            continue
        dxu, dxd = f(rx[ru]) - f(rx[r]), f(rx[r]) - f(rx[rd])
        t = dxd / (dxu + dxd)
        wyu, wzu = fma(dxu, f(P["nbr_dydx"]), f(P["nbr_margin_y"])), fma(dxu, f(P["nbr_dzdx"]), f(P["nbr_margin_z"]))
        wyd, wzd = fma(dxd, f(P["nbr_dydx"]), f(P["nbr_margin_y"])), fma(dxd, f(P["nbr_dzdx"]), f(P["nbr_margin_z"]))
        for h in occupied[r]:
            y0, z0 = cl["y"][h], cl["z"][h]
            best = None
            for u in occupied[ru]:
                yu, zu = cl["y"][u], cl["z"][u]
                if not (abs(yu - y0) <= wyu and abs(zu - z0) <= wzu):
                    continue
                for d in occupied[rd]:
                    yd, zd = cl["y"][d], cl["z"][d]
                    if not (abs(yd - y0) <= wyd and abs(zd - z0) <= wzd):
                        continue
                    ey = y0 - fma(t, yu - yd, yd)
                    ez = z0 - fma(t, zu - zd, zd)
                    cost = fma(ez * ez, inv_sz2, (ey * ey) * inv_sy2)
                    if not cost <= f(P["triplet_cut"]):
                        continue
                    cand = (float(cost), key(u), key(d), u, d)
                    if best is None or cand[:3] < best[:3]:
                        best = cand
            if best is not None:
                up[h], dn[h] = best[3], best[4]
    return up, dn


@pytest.mark.parametrize("seed", [11, 12])
def test_p1_brute_force_triplets_tiny(row_x, seed):
    fr = synth.generate(synth.config(1, scale=0.02, seed=seed), noise_frac=0.4)  # 4 tracks + heavy noise
    assert 100 < fr.n <= 700
    with np.errstate(over="ignore"):
        up, dn = _brute_links_py(fr.clusters, row_x, oracle.DEFAULT_PARAMS)
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x)
    assert np.array_equal(r.link_up_raw, up)
    assert np.array_equal(r.link_down_raw, dn)
    assert (up >= 0).sum() > 50


@pytest.mark.parametrize("cfg,scale", [(1, 0.05), (2, 0.01), (3, 0.01)])
def test_p1_structure_free_mode_equals_sorted_mode(row_x, cfg, scale):
    """The oracle's z-sorted search and its no-structure mode (every cluster of the row is a candidate)
    give identical results for every step (links, tracklets, assignment, tracks)."""
    fr = synth.generate(synth.config(cfg, scale=scale, seed=5))
    a = oracle.track(fr.clusters, fr.sector_offsets, row_x, brute=False)
    b = oracle.track(fr.clusters, fr.sector_offsets, row_x, brute=True)
    _same(a, b)
    assert len(a.tracks) > 0


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("pt,q,tanl,sinphi0", [(0.35, -1, 0.5, -0.33), (0.4, 1, 0.6, 0.3), (0.5, -1, -0.8, -0.1), (1.0, 1, 0.3, 0.12),
                                                (2.0, -1, 1.0, 0.0), (8.0, 1, -0.2, 0.02)])
def test_p2_noiseless_helix(row_x, pt, q, tanl, sinphi0):
    """A noiseless helix: links follow the true hits, one chain rows 1..R-2, one start hit, one track with all
    hits, and q/pT and tan(lambda) recovered (curvature sign DESIGN.md A15)."""
    R = len(row_x)
    qpt = q / pt
    y, z, s = helix_points(row_x.astype(np.float64), 85.0, 1.0, 30.0, sinphi0, tanl, qpt, 0.5)
    ok = np.abs(y) < row_x * np.tan(np.deg2rad(10))
    assert ok.all()
    cl = _mk(np.arange(R), y, z, row_x)
    r = oracle.track(cl, np.array([0, R], np.int32), row_x)
    idx = np.arange(R)
    exp_up = np.where((idx >= 1) & (idx <= R - 2), idx + 1, -1)
    exp_dn = np.where((idx >= 1) & (idx <= R - 2), idx - 1, -1)
    assert np.array_equal(r.link_up_raw, exp_up) and np.array_equal(r.link_down_raw, exp_dn)
    # cleaning cuts the links of the two end triplet centres whose partner is an end hit (A6)
    assert np.array_equal(r.link_up, np.where((idx >= 1) & (idx <= R - 3), idx + 1, -1))
    assert np.array_equal(r.link_down, np.where((idx >= 2) & (idx <= R - 2), idx - 1, -1))
    assert list(r.start_hits) == [1]
    assert len(r.tracks) == 1 and r.tracks["n_hits"][0] == R and (r.assignment == 0).all()
    t = r.tracks[0]
    assert t["x"] == row_x[0]
    # "to float precision" (north_star): achieved on these six helices 1.3e-6 relative in q/pT, 6e-8 in tan(lambda),
    # 3.3e-7 in sin(phi), 5 um in y, 70 um in z (z = 30..200 cm: 3 ulp); the bounds below are 3-8x those figures
    assert abs(t["qpt"] - qpt) <= 1e-5 * abs(qpt), (t["qpt"], qpt)
    assert abs(t["dzds"] - tanl) <= 1e-6 * max(1, abs(tanl)), (t["dzds"], tanl)
    assert abs(t["sinphi"] - sinphi0) <= 2e-6
    assert abs(t["y"] - 1.0) < 2e-5 and abs(t["z"] - 30.0) < 2e-4
    assert t["chi2"] < 1e-4  # noiseless: residuals are fp32 rounding only


def test_p2_curvature_sign(row_x):
    """Positive charge in +z field bends towards -y for a track along +x (d sinphi/dx = -0.003*B*q/pT < 0)."""
    R = len(row_x)
    y, z, s = helix_points(row_x.astype(np.float64), 85.0, 0.0, 0.0, 0.0, 0.1, +1.0 / 0.5, 0.5)
    assert y[-1] < -1.0
    cl = _mk(np.arange(R), y, z, row_x)
    r = oracle.track(cl, np.array([0, R], np.int32), row_x)
    assert len(r.tracks) == 1 and r.tracks["qpt"][0] > 1.9


# ---------------------------------------------------------------- P3-P5
@pytest.fixture(scope="module")
def cfg2_small(row_x):
    fr = synth.generate(synth.config(2, scale=0.05, seed=2))
    return fr, oracle.track(fr.clusters, fr.sector_offsets, row_x)


def test_p3_links_mutual_after_cleaning(cfg2_small):
    fr, r = cfg2_small
    h = np.flatnonzero(r.link_up >= 0)
    assert len(h) > 1000
    assert np.array_equal(r.link_down[r.link_up[h]], h)
    h = np.flatnonzero(r.link_down >= 0)
    assert np.array_equal(r.link_up[r.link_down[h]], h)
    # cleaning only removes
    assert ((r.link_up == r.link_up_raw) | (r.link_up == -1)).all()
    # start hits are exactly the chain heads
    sh = np.flatnonzero((r.link_down < 0) & (r.link_up >= 0))
    assert np.array_equal(np.sort(r.start_hits), sh)


def test_p4_exclusive_assignment(cfg2_small):
    fr, r = cfg2_small
    nt = len(r.tracks)
    assert nt > 100
    cnt = np.bincount(r.assignment[r.assignment >= 0], minlength=nt)
    assert np.array_equal(cnt, r.tracks["n_hits"])
    assert cnt.min() >= oracle.DEFAULT_PARAMS["min_track_hits"]
    sec = score.sector_of_cluster(fr.sector_offsets, fr.n)
    for t in range(0, nt, 7):
        h = np.flatnonzero(r.assignment == t)
        assert len(np.unique(fr.clusters["row"][h])) == len(h)  # one hit per row
        assert (sec[h] == r.tracks["sector"][t]).all()
        assert fr.clusters["row"][h].min() == r.tracks["first_row"][t]
        assert fr.clusters["row"][h].max() == r.tracks["last_row"][t]
    # every hit of a track comes from its tracklet's row table
    for t in range(0, nt, 11):
        rh = r.row_hit[r.track_tracklet[t]]
        assert set(np.flatnonzero(r.assignment == t)) <= set(rh[rh >= 0])


def test_p5_permutation_invariance(cfg2_small, row_x):
    fr, r = cfg2_small
    fp, p = synth.permute_within_sectors(fr, seed=99)
    rp = oracle.track(fp.clusters, fp.sector_offsets, row_x)
    assert len(rp.tracks) == len(r.tracks)
    # new[i] = old[p[i]]: assignment equal up to the permutation, track ids included (canonical order)
    assert np.array_equal(rp.assignment, r.assignment[p])
    inv = np.empty_like(p)
    inv[p] = np.arange(len(p))
    lu = np.where(r.link_up >= 0, inv[np.maximum(r.link_up, 0)], -1)
    assert np.array_equal(rp.link_up, lu[p])
    assert np.array_equal(rp.start_hits, inv[r.start_hits])
    assert np.array_equal(rp.tracks["n_hits"], r.tracks["n_hits"])
    assert rp.tracks.tobytes() == r.tracks.tobytes()


# ---------------------------------------------------------------- P6
@pytest.mark.parametrize("qpt,s0,tanl", [(2.0, 0.1, 0.7), (-4.0, -0.3, -1.2), (0.1, 0.6, 0.2), (0.0, 0.2, 0.5)])
def test_p6_transport_closed_form(qpt, s0, tanl):
    """sin(phi) linear in x, y on the circle, z = tan(lambda) * arc: one 100 cm step, 100 one-cm steps and the
    float64 helix agree."""
    x0, y0 = 90.0, 3.0
    p = [y0, 0.0, s0, tanl, qpt]
    C0 = np.zeros(15, np.float32)
    ok, x1, p1, _ = oracle.kf_transport(x0, p, C0, x0 + 40.0)
    assert ok
    y, z, s = helix_points([x0 + 40.0], x0, y0, 0.0, s0, tanl, qpt, 0.5)
    assert abs(p1[2] - s[0]) < 2e-6
    assert abs(p1[0] - y[0]) < 2e-5 * max(1, abs(y[0]))
    # the arc series is truncated after u^4: a single long step is slightly short at high curvature
    assert abs(p1[1] - z[0]) < 2e-3 * max(1, abs(z[0]))
    x, pp, C = x0, np.array(p, np.float32), C0
    for i in range(40):
        ok, x, pp, C = oracle.kf_transport(x, pp, C, x0 + (i + 1))
        assert ok
    assert abs(pp[2] - s[0]) < 5e-6
    assert abs(pp[0] - y[0]) < 1e-4
    assert abs(pp[1] - z[0]) < 1e-4 * max(1, abs(z[0]))
    # and back again: transport is reversible
    for i in range(40):
        ok, x, pp, C = oracle.kf_transport(x, pp, C, x0 + 39 - i)
    assert abs(pp[0] - y0) < 2e-4 and abs(pp[1]) < 2e-4 and abs(pp[2] - s0) < 1e-5


def test_p6_transport_fails_beyond_max_sinphi():
    ok, *_ = oracle.kf_transport(100.0, [0, 0, 0.9, 0, -10.0], np.zeros(15, np.float32), 110.0)
    assert not ok  # 0.9 + 10*0.015 > 0.95
    ok, *_ = oracle.kf_transport(100.0, [0, 0, 0.99, 0, 0.0], np.zeros(15, np.float32), 101.0)
    assert not ok
    # A11: the limit holds at BOTH ends of a step -- a state already beyond it may not be transported back inside
    ok, *_ = oracle.kf_transport(100.0, [0, 0, 0.96, 0, +4.0], np.zeros(15, np.float32), 110.0)  # s1 = 0.96 - 0.06
    assert not ok
    ok, x1, p1, _ = oracle.kf_transport(100.0, [0, 0, 0.94, 0, +4.0], np.zeros(15, np.float32), 110.0)
    assert ok and abs(p1[2] - 0.88004) < 1e-4
    # dx = 0 is the identity (first step of E3 and of every refit pass), whatever the state
    C = np.arange(15, dtype=np.float32)
    ok, x1, p1, C1 = oracle.kf_transport(100.0, [1, 2, 0.5, 0.3, 2.0], C, 100.0)
    assert ok and x1 == 100.0 and list(p1) == [1, 2, 0.5, 0.3, 2.0] and np.array_equal(C1, C)


@pytest.mark.parametrize("qpt,s0,tanl,dx", [(2.6, -0.2, 0.9, 100.0), (-2.6, 0.2, -0.7, 100.0), (2.6, 0.2, 0.9, -100.0)])
def test_p6_long_step_needs_both_series_terms(qpt, s0, tanl, dx):
    """One 100 cm step at |u| = |k L / 2| ~ 0.2: asin(u)/u - 1 = u^2/6 (7e-3) + 3u^4/40 (1.2e-4) + 15u^6/336 (3e-6).
    z against the float64 helix at 1e-5 relative needs both coefficients of the series of DESIGN.md section 3
    (dropping u^4 costs 1.2e-4, a wrong 1/6 much more); y and sin(phi) have no series and hold to fp32 rounding."""
    x0 = 100.0 if dx > 0 else 200.0
    ok, x1, p1, _ = oracle.kf_transport(x0, [3.0, 0.0, s0, tanl, qpt], np.zeros(15, np.float32), x0 + dx)
    assert ok
    y, z, s = helix_points([x0 + dx], x0, 3.0, 0.0, s0, tanl, qpt, 0.5)
    u = 0.5 * (-KAPPA_PER_T * 0.5 * qpt) * np.hypot(dx, y[0] - 3.0)
    assert 0.18 < abs(u) < 0.25
    assert abs(p1[2] - s[0]) < 1e-6
    assert abs(p1[0] - y[0]) < 1e-5 * abs(y[0] - 3.0) + 2e-6
    assert abs(p1[1] - z[0]) < 1e-5 * abs(z[0]), (p1[1], z[0])


def test_p6_jacobian_matches_finite_differences():
    """C <- F C F^T with F from the transport: compare the propagated covariance with a float64
    finite-difference Jacobian of the closed-form helix map (catches a dropped or transposed term)."""
    x0, dx, bz = 100.0, 12.0, 0.5
    p0 = np.array([2.0, 5.0, 0.25, 0.8, 1.5])

    def fmap(p):
        y, z, s = helix_points([x0 + dx], x0, p[0], p[1], p[2], p[3], p[4], bz)
        return np.array([y[0], z[0], s[0], p[3], p[4]])

    F = np.zeros((5, 5))
    for j in range(5):
        e = np.zeros(5)
        e[j] = 1e-6 * max(1.0, abs(p0[j]))
        F[:, j] = (fmap(p0 + e) - fmap(p0 - e)) / (2 * e[j])
    rng = np.random.default_rng(0)
    A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 0.1])[:, None]
    Cm = A @ A.T
    tri = [Cm[i, j] for i in range(5) for j in range(i + 1)]
    ok, x1, p1, C1 = oracle.kf_transport(x0, p0, tri, x0 + dx)
    exp = F @ Cm @ F.T
    got = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            got[i, j] = got[j, i] = C1[k]
            k += 1
    scale = np.sqrt(np.outer(np.diag(exp), np.diag(exp)))
    assert np.max(np.abs(got - exp) / scale) < 2e-3  # the neglected d(g) term is O(u^2) ~ 1e-5 here


# ---------------------------------------------------------------- P7
def test_p7_zero_field_is_linear_least_squares():
    """Bz = 0: the three-pass filter equals the weighted straight-line least-squares fit of y(x) and z(x) with the
    diagonal prior cov0 (textbook normal equations in float64).  sin(phi)=0 track so the model is exactly linear
    in (y, sinphi) to first order; compare value and covariance."""
    rng = np.random.default_rng(3)
    x = np.linspace(85, 245, 60)
    sy, sz = 0.1, 0.15
    ytrue = 1.0 + 0.02 * (x - 85)
    ztrue = -4.0 + 0.5 * (x - 85)
    y = ytrue + rng.normal(0, sy, x.size)
    z = ztrue + rng.normal(0, sz, x.size)
    ok, out = oracle.refit_hits(x, y, z, q0=0.0, bz=0.0)
    assert ok
    # float64 weighted LSQ on y = a + b (x - x0): params at x0 = innermost hit
    A = np.stack([np.ones_like(x), x - x[0]], 1)

    def lsq(v, sig, prior_var):
        N = A.T @ A / sig**2 + np.diag(1.0 / np.asarray(prior_var))
        return np.linalg.solve(N, A.T @ v / sig**2), np.linalg.inv(N)

    (a, b), covy = lsq(y, sy, [1e12, 1e12])
    (az, bz_), covz = lsq(z, sz, [1e12, 1e12])
    sinphi = b / np.sqrt(1 + b * b)
    dzds = bz_ / np.sqrt(1 + b * b)
    assert abs(out[1] - a) < 3e-3          # y at x0
    assert abs(out[3] - sinphi) < 1e-4     # sin(phi)
    assert abs(out[2] - az) < 5e-3         # z at x0
    assert abs(out[4] - dzds) < 2e-4       # dz/ds
    # covariance of y: (A^T W A)^-1 up to the prior (cov0 = 1 cm^2 vs 1e-4 information per hit: < 1 %)
    assert abs(out[6] - covy[0, 0]) / covy[0, 0] < 0.03
    assert abs(out[6 + 2] - covz[0, 0]) / covz[0, 0] < 0.03
    # q/pT unobservable at B = 0: stays at its start value, variance stays at the prior
    assert out[5] == 0.0 and abs(out[6 + 14] - 100.0) < 1e-3


def test_p7_single_update_is_textbook_gain():
    """One scalar update equals K = C H^T (H C H^T + v)^-1 in float64 for a full random covariance."""
    rng = np.random.default_rng(1)
    A = rng.normal(size=(5, 5))
    Cm = A @ A.T
    p = rng.normal(size=5)
    tri = [Cm[i, j] for i in range(5) for j in range(i + 1)]
    ym, zm, vy, vz = 0.3, -0.2, 0.01, 0.0225
    p1, C1, chi2 = oracle.kf_update(p, tri, 0.0, ym, zm, vy, vz)
    H = np.zeros((2, 5))
    H[0, 0] = H[1, 1] = 1
    V = np.diag([vy, vz])
    S = H @ Cm @ H.T + V
    K = Cm @ H.T @ np.linalg.inv(S)
    r = np.array([ym, zm]) - H @ p
    pe = p + K @ r
    Ce = (np.eye(5) - K @ H) @ Cm
    assert np.allclose(p1, pe, rtol=2e-4, atol=2e-5)
    got = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            got[i, j] = got[j, i] = C1[k]
            k += 1
    assert np.allclose(got, Ce, rtol=2e-3, atol=2e-4)
    assert abs(chi2 - r @ np.linalg.inv(S) @ r) < 1e-3 * max(1, chi2)


# ---------------------------------------------------------------- P8
def test_p8_pulls_and_chi2(row_x):
    """Smeared single helices: pulls of (y, z, sinphi, dzds, qpt) ~ N(0,1) and <chi2/ndf> ~ 1."""
    rng = np.random.default_rng(8)
    pulls, red = [], []
    xs = row_x.astype(np.float64)
    for i in range(400):
        pt = np.exp(rng.uniform(np.log(0.4), np.log(5)))
        q = rng.choice([-1.0, 1.0])
        s0, tl, y0, z0 = rng.uniform(-0.1, 0.1), rng.uniform(-1, 1), rng.uniform(-5, 5), rng.uniform(-100, 100)
        y, z, s = helix_points(xs, 85.0, y0, z0, s0, tl, q / pt, 0.5)
        ok, out = oracle.refit_hits(xs, y + rng.normal(0, 0.1, xs.size), z + rng.normal(0, 0.15, xs.size), 0.0, 0.5)
        assert ok
        true = np.array([y0, z0, s0, tl, q / pt])
        var = np.array([out[6 + k] for k in (0, 2, 5, 9, 14)])
        pulls.append((out[1:6] - true) / np.sqrt(var))
        red.append(out[21] / (2 * xs.size - 5))
    pulls = np.array(pulls)
    assert np.all(np.abs(pulls.mean(0)) < 0.2), pulls.mean(0)
    assert np.all(np.abs(pulls.std(0) - 1) < 0.15), pulls.std(0)
    assert abs(np.mean(red) - 1) < 0.05


# ---------------------------------------------------------------- P10 / P11
def test_p10_optimisation_level_independent(row_x):
    fr = synth.generate(synth.config(2, scale=0.02, seed=10))
    a = oracle.track(fr.clusters, fr.sector_offsets, row_x, opt="-O2")
    b = oracle.track(fr.clusters, fr.sector_offsets, row_x, opt="-O0")
    _same(a, b)
    c = oracle.track(fr.clusters, fr.sector_offsets, row_x, opt="-O2")
    _same(a, c)


def test_p11_config1_efficiency(row_x):
    fr = synth.generate(1)
    r = oracle.track(fr.clusters, fr.sector_offsets, row_x)
    sc = score.score(r.assignment, fr.truth, score.sector_of_cluster(fr.sector_offsets, fr.n), len(r.tracks))
    assert sc["efficiency"] > 0.98 and sc["fake_rate"] < 0.01, sc


def test_edge_cases(row_x):
    e = oracle.track(np.zeros(0, CL), np.zeros(37, np.int32), row_x)
    assert len(e.tracks) == 0 and len(e.start_hits) == 0
    # a sector with rows r and r+2 only (row skipping, A5): chain through every second row still links
    rows = np.arange(0, 152, 2)
    y, z, s = helix_points(row_x[rows].astype(np.float64), 85.0, 0.0, 10.0, 0.05, 0.4, 1.0, 0.5)
    cl = _mk(rows, y, z, row_x)
    r = oracle.track(cl, np.array([0, len(rows)], np.int32), row_x)
    assert (r.link_up_raw[1:-1] == np.arange(2, len(rows))).all()
    assert len(r.tracks) == 1 and r.tracks["n_hits"][0] == len(rows)
    # unequal row distances (rows 0,1,3,4,6,7,...): a straight inclined line still has zero triplet cost, because the
    # chord is evaluated at t = dxd / (dxu + dxd) (O2) -- with t = 1/2 or t swapped the middle hit would be
    # 0.5 cm off the chord (cost 28 > 18) and nothing would link
    rows = np.array([r_ for r_ in range(152) if r_ % 3 != 2])
    xs = row_x[rows].astype(np.float64)
    cl = _mk(rows, 0.5 * (xs - 85.0) - 20.0, 10.0 + 0.8 * (xs - 85.0), row_x)
    r = oracle.track(cl, np.array([0, len(rows)], np.int32), row_x, bz=0.0, params=dict(triplet_cut=0.01))
    assert (r.link_up_raw[1:-1] == np.arange(2, len(rows))).all() and (r.link_down_raw[1:-1] == np.arange(0, len(rows) - 2)).all()
    # every third row only: no links at all (one skip at most)
    rows = np.arange(0, 152, 3)
    y, z, s = helix_points(row_x[rows].astype(np.float64), 85.0, 0.0, 10.0, 0.05, 0.4, 1.0, 0.5)
    r = oracle.track(_mk(rows, y, z, row_x), np.array([0, len(rows)], np.int32), row_x)
    assert (r.link_up_raw == -1).all() and len(r.tracks) == 0


def test_golden_oracle_regression():
    """The oracle still reproduces tests/golden/oracle_regression.json (written by make_golden.py from the
    oracle alone): guards the oracle's arithmetic against unintended change."""
    import importlib.util
    import json
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = json.load(open(os.path.join(here, "oracle_regression.json")))
    assert len(stored) == len(mg.CASES)
    for exp in stored:
        got = mg.digest(exp["case"])
        assert got == exp, (got, exp)


# ---------------------------------------------------------------- mechanics of following, rejection and selection
from tests import scenarios  # noqa: E402


@pytest.mark.parametrize("missing,expect_tracks", [(5, 1), (6, 2)])
def test_gap_rule(row_x, missing, expect_tracks):
    """PAPER.md:51 "extrapolated through the TPC volume": `max_gap` = 5 consecutive rows without a cluster are
    bridged (both seeds then collect the same hits and the selector keeps one track); 6 are not (two tracks)."""
    R = len(row_x)
    cl = scenarios.gap_helix(row_x, missing)
    r = oracle.track(cl, np.array([0, len(cl)], np.int32), row_x)
    assert len(r.tracks) == expect_tracks
    if expect_tracks == 1:
        assert r.tracks["n_hits"][0] == R - missing and (r.assignment == 0).all()
    else:
        assert sorted(r.tracks["n_hits"]) == sorted([60, R - 60 - missing])
        assert (r.assignment[:60] == r.assignment[0]).all() and (r.assignment[60:] == r.assignment[-1]).all()
        assert r.assignment[0] != r.assignment[-1]


def test_outlier_rejection_on_the_inward_pass(row_x):
    """on the inward pass a hit of the seed that does not fit is rejected.  One hit displaced by 0.3 cm
    keeps its links (triplet cost 9 <= 18) and survives reject_cut = 25 (d ~ 9), but is dropped at reject_cut = 4."""
    R = len(row_x)
    cl = scenarios.displaced_hit_helix(row_x)
    so = np.array([0, R], np.int32)
    keep = oracle.track(cl, so, row_x)
    assert len(keep.tracks) == 1 and keep.tracks["n_hits"][0] == R and keep.assignment[80] == 0
    drop = oracle.track(cl, so, row_x, params=dict(reject_cut=4.0))
    assert len(drop.tracks) == 1 and drop.tracks["n_hits"][0] == R - 1
    assert drop.assignment[80] == -1 and (np.delete(drop.assignment, 80) == 0).all()
    assert drop.tracks["chi2"][0] < keep.tracks["chi2"][0]


def test_shared_cluster_goes_to_the_longer_track(row_x):
    """north_star (f) / PAPER.md:70: a cluster claimed by two tracklets goes to the one with more hits.  Two helices
    cross at row 90 and share that one cluster; the short one (rows 40-130) loses it."""
    R = len(row_x)
    cl, is_a = scenarios.crossing_helices(row_x)
    r = oracle.track(cl, np.array([0, len(cl)], np.int32), row_x)
    assert len(r.tracks) == 2
    ta = r.assignment[is_a]
    tb = r.assignment[~is_a]
    assert (ta == ta[0]).all() and ta[0] >= 0, "the long track keeps every cluster, the shared one included"
    assert (tb[tb >= 0] == tb[tb >= 0][0]).all() and tb[tb >= 0][0] != ta[0]
    assert R in r.tracks["n_hits"] and min(r.tracks["n_hits"]) <= 90


def test_canonical_orders(cfg2_small, row_x):
    """DESIGN.md A4 / O4 / O6: tracklet ids follow (sector, row, ord z, ord y, input index) of the start hit, track ids
    follow tracklet ids; both are what makes the output independent of the input order."""
    fr, r = cfg2_small
    sh = r.start_hits
    sec = score.sector_of_cluster(fr.sector_offsets, fr.n)[sh]
    c = fr.clusters[sh]

    def ordf(f):
        b = f.astype(np.float32).view(np.uint32).astype(np.uint64)
        return np.where(b & 0x80000000, (~b) & 0xFFFFFFFF, b | 0x80000000)

    keys = list(zip(sec.tolist(), c["row"].tolist(), ordf(c["z"]).tolist(), ordf(c["y"]).tolist(), sh.tolist()))
    assert keys == sorted(keys) and len(set(keys)) == len(keys)
    assert (np.diff(r.track_tracklet) > 0).all()
    # a start hit has an up-link and no down-link; every such cluster is a start hit
    is_start = (r.link_down < 0) & (r.link_up >= 0)
    assert np.array_equal(np.sort(sh), np.flatnonzero(is_start))


# ---------------------------------------------------------------- round 2: pins of the mechanics a one-line slip would break
from tests import kf64  # noqa: E402


def _run1(cl, row_x, **params):
    return oracle.track(cl, np.array([0, len(cl)], np.int32), row_x, params=params or None)


def test_refit_starts_from_the_tracklets_curvature(row_x):
    """DESIGN.md O7: the refit starts at the outermost hit with the two-hit chord and q/pT taken from the tracklet.  On a
    minimum-length (10 hits), strongly curved (pT = 0.1) track three passes have not yet forgotten the start value: the
    oracle must follow the float64 filter started with the SAME q0 (achieved 5e-6 relative), while the results for
    q0 = 0 and q0 = true differ by 1 % in q/pT.  (From 24 hits on the start value is immaterial: < 1e-7.)"""
    rng = np.random.default_rng(9)
    rows = np.arange(40, 50)
    xs = row_x[rows].astype(np.float64)
    qpt = 1 / 0.1
    y, z, s = helix_points(xs, xs[0], 1.0, 30.0, 0.1, 0.6, qpt, 0.5)
    ys = (y + rng.normal(0, 0.1, len(xs))).astype(np.float32).astype(np.float64)
    zs = (z + rng.normal(0, 0.15, len(xs))).astype(np.float32).astype(np.float64)
    P = oracle.DEFAULT_PARAMS
    res = {}
    for q0 in (0.0, qpt):
        ok, out = oracle.refit_hits(xs, ys, zs, q0=q0, bz=0.5)
        x3, p3, C3, chi3 = kf64.refit(xs, ys, zs, q0, 0.5, P["cov0"], P["sigma_y"], P["sigma_z"])
        assert ok and np.all(np.abs(out[1:6] - p3) <= 5e-5 * np.maximum(1.0, np.abs(p3))), (q0, out[1:6], p3)
        res[q0] = p3
    assert abs(res[0.0][4] - res[qpt][4]) > 5e-3 * qpt


@pytest.mark.parametrize("pt,q,s0,tl", [(0.3, 1, 0.3, 0.6), (0.25, -1, -0.35, -0.9)])
def test_refit_is_three_passes_inward_outward_inward(row_x, pt, q, s0, tl):
    """PAPER.md:71 "The final Kalman refit is iterated three times: inward, outward, and inward".  A curved, smeared
    helix, started from the two-hit chord with q/pT = 0: the oracle's refit must equal a float64 extended Kalman
    filter (tests/kf64.py: exact helix map, finite-difference Jacobian, joint 2-D update) run inward, outward, inward
    with the covariance reset per pass -- and NOT the same filter run once, which ends measurably elsewhere because the
    first pass linearises about the poor chord start (q/pT = 0).  Output at the innermost hit."""
    rng = np.random.default_rng(5)
    rows = np.arange(20, 130)
    xs = row_x[rows].astype(np.float64)
    y, z, s = helix_points(xs, xs[0], 1.0, 30.0, s0, tl, q / pt, 0.5)
    ys = (y + rng.normal(0, 0.1, len(xs))).astype(np.float32).astype(np.float64)
    zs = (z + rng.normal(0, 0.15, len(xs))).astype(np.float32).astype(np.float64)
    P = oracle.DEFAULT_PARAMS
    ok, out = oracle.refit_hits(xs, ys, zs, q0=0.0, bz=0.5)
    assert ok and out[0] == row_x[rows[0]]
    x3, p3, C3, chi3 = kf64.refit(xs, ys, zs, 0.0, 0.5, P["cov0"], P["sigma_y"], P["sigma_z"])
    x1, p1, C1, chi1 = kf64.refit(xs, ys, zs, 0.0, 0.5, P["cov0"], P["sigma_y"], P["sigma_z"], passes=("in",))
    sig = np.sqrt(np.diag(C3))
    got = out[1:6].astype(np.float64)
    # achieved: 2.2e-6 relative / 6e-4 sigma in the state, 1.3e-5 in the variances, 5e-6 in chi2
    assert np.all(np.abs(got - p3) <= 5e-6 * np.maximum(1.0, np.abs(p3))), (got, p3)
    assert np.all(np.abs(got - p3) <= 5e-3 * sig)
    var = np.array([out[6 + k] for k in (0, 2, 5, 9, 14)])
    assert np.allclose(var, np.diag(C3), rtol=1e-4)
    assert abs(out[21] - chi3) < 1e-4 * chi3
    # ... and ONE pass of the same float64 filter is measurably somewhere else: 2e-4 .. 7e-4 cm in y, 6e-5 .. 2e-4
    # relative in q/pT, 2e-4 .. 3e-3 in chi2, i.e. 40-300 x the bounds above
    assert abs(p1[0] - p3[0]) > 1e-4 and abs(p1[4] - p3[4]) > 5e-5 * abs(p3[4]) and abs(chi1 - chi3) > 1e-4 * chi3
    assert abs(got[0] - p1[0]) > 1e-4 and abs(got[4] - p1[4]) > 5e-5 * abs(p3[4])


def test_tracklet_covariance_is_one_inward_pass(row_x):
    """PAPER.md:66-68 / DESIGN.md A18: at the turn-round after the outward pass the covariance and chi2 are reset, so the
    tracklet's covariance is that of ONE pass over its hits.  Zero field, straight smeared track: var(y) and var(z~) at the
    innermost hit equal the float64 least-squares (A^T W A)^-1 -- information counted once, not twice -- and chi2 equals the
    least-squares residual sum (+ the z offset fixed by z_ref).  q/pT is unobservable at B = 0 and keeps the prior."""
    rng = np.random.default_rng(17)
    R = len(row_x)
    xs = row_x.astype(np.float64)
    y = 2.0 + 0.05 * (xs - xs[0]) + rng.normal(0, 0.1, R)
    z = 10.0 + 0.4 * (xs - xs[0]) + rng.normal(0, 0.15, R)
    cl = _mk(np.arange(R), y, z, row_x)
    r = oracle.track(cl, np.array([0, R], np.int32), row_x, bz=0.0)
    assert len(r.tracks) >= 1
    k = int(np.argmax(r.tracklet_ints[:, 3]))
    ti, tf = r.tracklet_ints[k], r.tracklet_floats[k]
    assert ti[0] == 1 and ti[3] >= 140
    hits = r.row_hit[k][r.row_hit[k] >= 0]
    xh = cl["x"][hits].astype(np.float64)
    A = np.stack([np.ones_like(xh), xh - xh[0]], 1)

    def lsq(v, sig):
        N = A.T @ A / sig**2
        sol = np.linalg.solve(N, A.T @ v / sig**2)
        return sol, np.linalg.inv(N), float(((v - A @ sol) ** 2).sum() / sig**2)

    (a, b), covy, chiy = lsq(cl["y"][hits].astype(np.float64), 0.1)
    (az, bz_), covz, chiz = lsq(cl["z"][hits].astype(np.float64), 0.15)
    C = tf[6:21]
    assert abs(C[0] - covy[0, 0]) < 0.02 * covy[0, 0], (C[0], covy[0, 0])   # prior 1 cm^2 vs 4e-4: 0.04 %
    assert abs(C[2] - covz[0, 0]) < 0.02 * covz[0, 0], (C[2], covz[0, 0])
    assert abs(C[14] - 100.0) < 1e-2
    assert abs(tf[21] - (chiy + chiz)) < 0.02 * (chiy + chiz), (tf[21], chiy + chiz)
    assert abs(tf[1] - a) < 2e-3 and abs((tf[2] + tf[22]) - az) < 2e-3


@pytest.mark.parametrize("mirror_z", [False, True])
def test_selector_equal_length_lower_id_wins(row_x, mirror_z):
    """DESIGN.md A4/A13: equal hit count and equal quality bucket (noiseless: chi2 ~ 0) -> the lower tracklet id owns the
    shared cluster.  Tracklet ids follow the start hits' (row, ord z, ...) order, both helices start on row 31, so the
    helix with the lower z there must own it; mirroring z swaps the owner."""
    cl, sh, is_a, is_b = scenarios.equal_length_crossing(row_x, None, mirror_z)
    r = _run1(cl, row_x)
    assert len(r.tracks) == 2
    ta, tb = np.unique(r.assignment[is_a]), np.unique(r.assignment[is_b])
    assert len(ta) == 1 and len(tb) == 1 and ta[0] >= 0 and tb[0] >= 0 and ta[0] != tb[0]
    za = cl["z"][is_a & (cl["row"] == 31)][0]
    zb = cl["z"][is_b & (cl["row"] == 31)][0]
    lower = ta[0] if za < zb else tb[0]
    assert lower == 0, "track ids follow tracklet ids"
    assert r.assignment[sh] == lower
    assert sorted(r.tracks["n_hits"]) == [90, 91]


@pytest.mark.parametrize("mirror_z", [False, True])
@pytest.mark.parametrize("displaced", ["A", "B"])
def test_selector_equal_length_better_chi2_wins(row_x, displaced, mirror_z):
    """north_star (f) "by track length and quality" / DESIGN.md A13: at equal hit count the tracklet with the lower
    chi2/ndf owns a shared cluster, whatever the ids.  One helix carries a hit displaced by 2.5 sigma (chi2 + 6, i.e.
    1000 * 6 / 182 = 33 quality buckets); the clean one must own the crossing cluster in all four id / role combinations."""
    cl, sh, is_a, is_b = scenarios.equal_length_crossing(row_x, displaced, mirror_z)
    r = _run1(cl, row_x)
    assert len(r.tracks) == 2
    ta, tb = np.unique(r.assignment[is_a]), np.unique(r.assignment[is_b])
    assert len(ta) == 1 and len(tb) == 1 and ta[0] >= 0 and tb[0] >= 0 and ta[0] != tb[0]
    clean = tb[0] if displaced == "A" else ta[0]
    assert r.assignment[sh] == clean
    assert r.tracks["n_hits"][clean] == 91 and r.tracks["n_hits"][1 - clean] == 90


@pytest.mark.parametrize("inward", [False, True])
def test_sector_edge_stop(row_x, inward):
    """PAPER.md:49 (tracking is sector-local) / DESIGN.md A11: following stops where the predicted |y| exceeds
    x tan(10 deg) + edge_margin.  On-helix decoy clusters beyond the sector's side (every third row, so the gap rule
    never fires and no links form) are collected while inside the 3 cm margin and never beyond it -- on the outward
    extrapolation E2 (helix leaving upwards) and on the inward pass E3 (helix entering from the side)."""
    cl, y, inside = scenarios.edge_helix(row_x, inward)
    lim = row_x.astype(np.float64) * np.tan(np.deg2rad(10.0)) + oracle.DEFAULT_PARAMS["edge_margin"]
    slack = np.abs(y) - lim
    assert np.abs(slack[~inside]).min() > 0.1  # no row sits on the line
    r = _run1(cl, row_x)
    assert len(r.tracks) == 1
    rows = cl["row"]
    dec = ~inside[rows]
    in_margin = slack[rows] < 0
    assert (dec & in_margin).sum() >= 3 and (dec & ~in_margin).sum() >= 10
    assert (r.assignment[in_margin] == 0).all(), "inside the margin every cluster is collected"
    assert (r.assignment[~in_margin] == -1).all(), "beyond x tan + margin nothing is collected"
    # without the margin the decoys are all dropped; with a huge one the helix is followed to the last decoy
    r0 = _run1(cl, row_x, edge_margin=0.0)
    assert (r0.assignment[dec] == -1).all() and (r0.assignment[~dec] == 0).all()
    r9 = _run1(cl, row_x, edge_margin=60.0)
    assert (r9.assignment == 0).all()


def test_e3_gap_rule_is_armed_only_below_the_start_row(row_x):
    """DESIGN.md section 2 (E3 gap rule): on the inward pass the stop after max_gap misses is armed only below the
    start hit's row.  Rows 99..103 are missing (E2 bridges 5 rows) and the last chain hit, row 98, is displaced by
    3 sigma: at reject_cut = 4 the inward pass rejects it, which makes six consecutive misses ABOVE the start row (1) --
    the pass must go on and keep rows 0..97.  The upper seed (start row 105) picks the displaced hit up (pick_cut = 16)."""
    cl = scenarios.e3_gap_above_start(row_x)
    r = _run1(cl, row_x, reject_cut=4.0)
    assert list(cl["row"][r.start_hits]) == [1, 105]
    assert r.tracklet_ints[0].tolist() == [1, 0, 151, 146]
    assert r.row_hit[0][98] == -1 and (r.row_hit[0][:98] == np.arange(98)).all()
    assert r.tracklet_ints[1].tolist() == [1, 0, 151, 147] and r.row_hit[1][98] == 98
    assert len(r.tracks) == 1 and r.tracks["n_hits"][0] == 147 and (r.assignment == 0).all()


def test_exact_ties_follow_the_key_order(row_x):
    """DESIGN.md A4: candidates of exactly equal cost are ordered by (ord z, ord y, input index) of the up cluster, then
    of the down cluster.  Mirror-image candidates give bit-equal costs (the error terms differ in sign only)."""
    f = np.float32
    x = row_x

    def links(up_pts, dn_pts, order):
        # centre cluster on row 50 at (0, 0); candidates on rows 51 / 49; `order` permutes the input positions
        pts = [(50, 0.0, 0.0)] + [(51, yy, zz) for yy, zz in up_pts] + [(49, yy, zz) for yy, zz in dn_pts]
        pts = [pts[i] for i in order]
        cl = _mk(np.array([p[0] for p in pts]), np.array([p[1] for p in pts], f), np.array([p[2] for p in pts], f), x)
        r = oracle.track(cl, np.array([0, len(cl)], np.int32), x)
        c = order.index(0)
        return pts[r.link_up_raw[c]], pts[r.link_down_raw[c]]

    for order in ([0, 1, 2, 3], [3, 2, 1, 0], [2, 0, 3, 1]):
        # two up candidates mirrored in z (same y): the lower z wins whatever the input order
        u, d = links([(0.05, +0.25), (0.05, -0.25)], [(0.0, 0.0)], order)
        assert u == (51, 0.05, -0.25) and d == (49, 0.0, 0.0)
        # mirrored in y at equal z: the lower y wins
        u, d = links([(+0.125, 0.1), (-0.125, 0.1)], [(0.0, 0.0)], order)
        assert u == (51, -0.125, 0.1)
        # the same up cluster with two mirrored down candidates: the down key decides
        u, d = links([(0.0, 0.0)], [(0.05, +0.25), (0.05, -0.25)], order)
        assert d == (49, 0.05, -0.25)
    # bit-identical duplicates: the lower input index wins
    for order in ([0, 1, 2, 3], [0, 2, 1, 3]):
        pts_up = [(0.05, 0.25), (0.05, 0.25)]
        pts = [(50, 0.0, 0.0)] + [(51, *p) for p in pts_up] + [(49, 0.0, 0.0)]
        pts = [pts[i] for i in order]
        cl = _mk(np.array([p[0] for p in pts]), np.array([p[1] for p in pts], f), np.array([p[2] for p in pts], f), x)
        r = oracle.track(cl, np.array([0, len(cl)], np.int32), x)
        dup = [i for i, p in enumerate(pts) if p[0] == 51]
        assert r.link_up_raw[0] == min(dup)
