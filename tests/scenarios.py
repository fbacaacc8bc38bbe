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
