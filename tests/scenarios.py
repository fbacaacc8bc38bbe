"""Small hand-built single-sector inputs (float64 closed-form helices, tests only) used by the oracle pins and by the
GPU parity tests: a helix with rows removed, a helix with one displaced hit, two crossing helices sharing a cluster."""
import numpy as np

from paper_1811_11481_b200 import synth
from tests.helix import helix_points

CL = synth.CLUSTER_DTYPE


def mk(rows, y, z, rx):
    cl = np.zeros(len(rows), CL)
    cl["row"] = rows
    cl["x"] = rx[rows]
    cl["y"] = y
    cl["z"] = z
    return cl


def one_helix(row_x, rows=None, **kw):
    rows = np.arange(len(row_x)) if rows is None else np.asarray(rows)
    par = dict(x0=85.0, y0=0.5, z0=20.0, sinphi0=0.08, tanl=0.4, qpt=1.2, bz=0.5)
    par.update(kw)
    y, z, _ = helix_points(row_x[rows].astype(np.float64), par["x0"], par["y0"], par["z0"], par["sinphi0"],
                           par["tanl"], par["qpt"], par["bz"])
    return rows, y, z


def gap_helix(row_x, missing):
    R = len(row_x)
    rows, y, z = one_helix(row_x, np.r_[np.arange(0, 60), np.arange(60 + missing, R)])
    return mk(rows, y, z, row_x)


def displaced_hit_helix(row_x, row=80, dy=0.3):
    rows, y, z = one_helix(row_x)
    y = y.copy()
    y[row] += dy
    return mk(rows, y, z, row_x)


def crossing_helices(row_x):
    """Returns (clusters sorted by row, mask of the long track's clusters)."""
    R = len(row_x)
    rows_a, ya, za = one_helix(row_x)
    rows_b = np.arange(40, 131)
    yb, zb, _ = helix_points(row_x[rows_b].astype(np.float64), float(row_x[90]), ya[90], za[90], -0.25, -0.6, -0.8, 0.5)
    keep = rows_b != 90  # the crossing cluster exists once
    rows = np.r_[rows_a, rows_b[keep]]
    cl = mk(rows, np.r_[ya, yb[keep]], np.r_[za, zb[keep]], row_x)
    order = np.argsort(rows, kind="stable")
    return cl[order], np.r_[np.ones(R, bool), np.zeros(int(keep.sum()), bool)][order]


def frame(cl):
    return synth.Frame(cl, np.array([0, len(cl)], np.int32), np.full(len(cl), -1, np.int32), np.zeros((0, 8)), 1, "scenario")


# ---------------------------------------------------------------- round-2 scenarios (selector weight, sector edge, E3)
def equal_length_crossing(row_x, displaced=None, mirror_z=False, dy=0.25):
    """Two helices over the SAME rows 30..120 that cross at row 75 and share that one cluster (it exists once).
    A: the gentle one; B: the steep one.  `displaced` = "A" / "B" moves one hit of that helix (row 50) by `dy` in y, which
    raises its chi2 and nothing else.  `mirror_z` flips the sign of every z (swaps which helix has the lower z at the
    first rows, i.e. the lower tracklet id).  Returns (clusters, index of the shared cluster, mask of A's own clusters,
    mask of B's own clusters); the shared cluster is in neither mask."""
    rows = np.arange(30, 121)
    ya, za, _ = helix_points(row_x[rows].astype(np.float64), float(row_x[75]), 2.0, 40.0, 0.05, 0.3, 0.9, 0.5)
    yb, zb, _ = helix_points(row_x[rows].astype(np.float64), float(row_x[75]), 2.0, 40.0, -0.22, -0.5, -0.7, 0.5)
    ya, yb = ya.copy(), yb.copy()
    if displaced == "A":
        ya[50 - 30] += dy
    elif displaced == "B":
        yb[50 - 30] += dy
    keep = rows != 75
    r = np.r_[rows, rows[keep]]
    y = np.r_[ya, yb[keep]]
    z = np.r_[za, zb[keep]]
    if mirror_z:
        z = -z
    is_a = np.r_[rows != 75, np.zeros(int(keep.sum()), bool)]
    is_b = np.r_[np.zeros(len(rows), bool), np.ones(int(keep.sum()), bool)]
    shared = np.r_[rows == 75, np.zeros(int(keep.sum()), bool)]
    order = np.argsort(r, kind="stable")
    cl = mk(r[order], y[order], z[order], row_x)
    return cl, int(np.flatnonzero(shared[order])[0]), is_a[order], is_b[order]


EDGE_OUT = dict(x0=85.0, y0=0.0, z0=15.0, sinphi0=0.26, tanl=0.35, qpt=-1.6, bz=0.5)    # leaves the sector upwards
EDGE_IN = dict(x0=245.0, y0=0.0, z0=15.0, sinphi0=-0.38, tanl=0.35, qpt=1.7, bz=0.5)    # enters it from the side


def edge_helix(row_x, inward=False, decoy_step=3):
    """A helix that crosses the sector's side (|y| = x tan 10 deg) at mid radius.  Real clusters exist on every row where
    the helix is inside the sector; beyond the side, on-helix "decoy" clusters sit on every `decoy_step`-th row only
    (too sparse to form links -- one row skip at most, A5 -- and dense enough that the gap rule never fires).
    outward (default): inside at the low rows, leaves upwards (pins the E2 stop).  inward: inside at the high rows, the
    decoys are below (pins the E3 stop).  The parameters keep every row beyond the side at least 0.14 cm away from the
    line |y| = x tan 10 deg + 3 cm.  Returns (clusters, float64 y of the helix on every row, in-sector mask per row)."""
    R = len(row_x)
    xs = row_x.astype(np.float64)
    par = EDGE_IN if inward else EDGE_OUT
    y, z, _ = helix_points(xs, par["x0"], par["y0"], par["z0"], par["sinphi0"], par["tanl"], par["qpt"], par["bz"])
    inside = np.abs(y) <= xs * np.tan(np.deg2rad(10.0))
    rows = np.arange(R)
    if inward:
        first_in = int(np.flatnonzero(inside)[0])
        decoy = (~inside) & ((first_in - rows) % decoy_step == 0) & (rows < first_in)
    else:
        last_in = int(np.flatnonzero(inside)[-1])
        decoy = (~inside) & ((rows - last_in) % decoy_step == 0) & (rows > last_in)
    use = inside | decoy
    return mk(rows[use], y[use], z[use], row_x), y, inside


def e3_gap_above_start(row_x):
    """Rows 99..103 removed (5 rows: E2 bridges them) and the last chain hit, row 98, displaced by 0.3 cm: on the inward
    pass with reject_cut = pick_cut = 6 that hit is rejected, which makes SIX consecutive misses above the start row."""
    R = len(row_x)
    rows, y, z = one_helix(row_x, np.r_[np.arange(0, 99), np.arange(104, R)])
    y = y.copy()
    y[98] += 0.3
    return mk(rows, y, z, row_x)


# ---------------------------------------------------------------- sector-boundary scenarios (merger)
TAN10 = float(np.tan(np.deg2rad(10.0)))


def helix_in_two_sectors(row_x, sector=3, side=+1, par=None, z_shift_b=0.0, drop_rows_b=0, rng=None, n_sectors=36,
                         drop_rows_a_end=0, extend_a=0, qpt_b=None, copy_a_dz=None):
    """One float64 helix that leaves `sector` through its +y (side = +1) or -y (side = -1) edge and continues in the
    neighbouring sector.  The helix is given in the frame of `sector` (A); its continuation is the SAME circle expressed in
    the neighbour's frame (B): reference point and direction rotated by side * 20 degrees.  Clusters exist on every row
    where the helix is inside the respective sector (|y| <= x tan 10 deg).  Variations: z_shift_b displaces B's clusters
    in z; drop_rows_b removes B's first rows; drop_rows_a_end removes A's last rows; extend_a keeps A's clusters on that
    many rows beyond its edge (the two segments then overlap in rows); qpt_b continues in B with another curvature from
    the point and direction the helix has on A's last in-sector row; copy_a_dz adds a second copy of A's clusters
    displaced by that much in z; rng smears (0.1 cm, 0.15 cm).
    Returns (frame, info) with info = dict(rows_a, rows_b, y_a, z_a, s_a: float64 truth on A's rows, sector_b)."""
    par = dict(x0=85.0, y0=4.0, z0=25.0, sinphi0=0.12, tanl=0.5, qpt=-1.1, bz=0.5) if par is None else dict(par)
    if side < 0:
        par.update(y0=-par["y0"], sinphi0=-par["sinphi0"], qpt=-par["qpt"])
        qpt_b = None if qpt_b is None else -qpt_b
    xs = row_x.astype(np.float64)
    ya, za, sa = helix_points(xs, par["x0"], par["y0"], par["z0"], par["sinphi0"], par["tanl"], par["qpt"], par["bz"])
    in_a = np.abs(ya) <= xs * TAN10
    last_in = int(np.flatnonzero(in_a)[-1])
    a = np.deg2rad(20.0) * side
    if qpt_b is None:
        xr, yr, zr, sr, qb = par["x0"], par["y0"], par["z0"], par["sinphi0"], par["qpt"]
    else:  # same point and direction on A's last in-sector row, other curvature beyond it
        xr, yr, zr, sr, qb = xs[last_in], ya[last_in], za[last_in], sa[last_in], qpt_b
    x0b = xr * np.cos(a) + yr * np.sin(a)
    y0b = -xr * np.sin(a) + yr * np.cos(a)
    s0b = np.sin(np.arcsin(sr) - a)
    with np.errstate(invalid="ignore"):
        yb, zb, sb = helix_points(xs, x0b, y0b, zr, s0b, par["tanl"], qb, par["bz"])
    in_b = np.isfinite(yb) & (np.abs(sb) < 0.98) & (np.abs(yb) <= xs * TAN10)
    rows_a = np.flatnonzero(in_a)
    if extend_a:
        rows_a = np.arange(rows_a[0], min(len(xs), last_in + 1 + extend_a))
    if drop_rows_a_end:
        rows_a = rows_a[:-drop_rows_a_end]
    rows_b = np.flatnonzero(in_b)[drop_rows_b:]
    ring = n_sectors // 2
    base = (sector // ring) * ring
    sector_b = base + (sector - base + side) % ring
    ca = mk(rows_a, ya[rows_a], za[rows_a], row_x)
    cb = mk(rows_b, yb[rows_b], zb[rows_b] + z_shift_b, row_x)
    if copy_a_dz is not None:
        c2 = ca.copy()
        c2["z"] += np.float32(copy_a_dz)
        ca = np.concatenate([ca, c2])
    if rng is not None:
        for c in (ca, cb):
            c["y"] += rng.normal(0, 0.1, len(c)).astype(np.float32)
            c["z"] += rng.normal(0, 0.15, len(c)).astype(np.float32)
    parts = {sector: ca, sector_b: cb}
    so = np.zeros(n_sectors + 1, np.int32)
    for s in range(n_sectors):
        so[s + 1] = so[s] + (len(parts[s]) if s in parts else 0)
    cl = np.concatenate([parts[s] for s in sorted(parts)])
    fr = synth.Frame(cl, so, np.full(len(cl), -1, np.int32), np.zeros((0, 8)), n_sectors, "two_sector_helix")
    return fr, dict(rows_a=rows_a, rows_b=rows_b, y_a=ya, z_a=za, s_a=sa, sector_b=sector_b, par=par)


# ---------------------------------------------------------------- round-3 scenarios (pins of tests/test_oracle_pins_r3.py)
def displaced_hit_helix_z(row_x, row=120, dz=0.45):
    """As displaced_hit_helix, but the hit is moved along z: its keep / reject distance on the inward pass is
    dz^2 / (var(z~) predicted + sigma_z^2) -- the z variance of the filter, not a y term."""
    rows, y, z = one_helix(row_x)
    z = z.copy()
    z[row] += dz
    return mk(rows, y, z, row_x)


def lone_row_helix(row_x, row=100, dy=0.0, dz=0.0, duplicate=False, dup_positions=None):
    """A helix whose row `row` cannot be linked (two rows removed on either side of it: DESIGN.md A5 allows one skipped row)
    and is therefore reached by the pick-up search only, from the chain below (E2) and again from the chain above (E3).
    The cluster of that row is moved by (dy, dz); with `duplicate` it exists twice, bit for bit, at the array positions
    `dup_positions` (default: appended).  Returns (clusters, positions of the lone row's cluster(s))."""
    R = len(row_x)
    rows = np.r_[np.arange(0, row - 2), [row], np.arange(row + 3, R)]
    rows, y, z = one_helix(row_x, rows)
    y, z = y.copy(), z.copy()
    i = int(np.flatnonzero(rows == row)[0])
    y[i] += dy
    z[i] += dz
    cl = mk(rows, y, z, row_x)
    if not duplicate:
        return cl, [i]
    lone = cl[i:i + 1]
    rest = np.delete(cl, i)
    p, q = dup_positions if dup_positions is not None else (len(rest), len(rest) + 1)
    out = np.insert(rest, min(p, len(rest)), lone)
    out = np.insert(out, min(q, len(out)), lone)
    pos = [int(k) for k in np.flatnonzero(out["row"] == row)]
    return out, pos


def window_triplet(row_x, dy=0.0, dz=0.0, row=50):
    """Three clusters on a straight line through rows row-1, row, row+1 (cost 0), the outer two displaced by -/+ (dy, dz)."""
    f = np.float32
    return mk(np.array([row - 1, row, row + 1]), np.array([-dy, 0.0, dy], f), np.array([10.0 - dz, 10.0, 10.0 + dz], f), row_x)
