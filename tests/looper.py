"""Full helices over all 36 sectors in float64, written for the tests only (independent of synth/ and oracle/).

A charged particle in a uniform field along z moves on a circle in the transverse plane; every pad row of every sector
is a chord x_local = x_row of that plane, so both crossings of a row (the outgoing and the returning leg) have a closed
form.  Used by the looper-leg pins: which clusters belong to which leg is known by construction.
"""
import numpy as np

from paper_1811_11481_b200 import synth

KAPPA_PER_T = 0.00299792458  # 1/cm per (T * c/GeV)
TAN10 = np.tan(np.deg2rad(10.0))


def helix_clusters(row_x, pt, phi0, tanl, q, z0=0.0, origin=(0.0, 0.0), bz=0.5, turns=1.0, z_max=250.0):
    """Clusters of one particle starting at `origin` (global x, y) and z0 with direction phi0 (global azimuth).

    Returns a list of dicts: sector (0..35, by the sign of z), row, x, y, z (sector-local), turn angle `theta` (>= 0, radians
    from the start), local sin(phi) of the PHYSICAL direction, `outgoing` (radius growing).  Side A (z >= 0) = sectors 0-17.
    """
    row_x = np.asarray(row_x, np.float64)
    R = pt / (KAPPA_PER_T * bz)
    # curvature of the azimuth along the path: d(phi)/ds = -kappa * Bz * q / pT  (tests/helix.py convention)
    w = -np.sign(q) if bz > 0 else np.sign(q)  # sense of rotation: +1 counter-clockwise
    cx = origin[0] - w * R * np.sin(phi0)
    cy = origin[1] + w * R * np.cos(phi0)
    a0 = np.arctan2(origin[1] - cy, origin[0] - cx)  # angle of the start point seen from the centre
    out = []
    for k in range(18):
        al = np.deg2rad(20.0 * k + 10.0)
        lcx = cx * np.cos(al) + cy * np.sin(al)
        lcy = -cx * np.sin(al) + cy * np.cos(al)
        for r, xr in enumerate(row_x):
            d = xr - lcx
            if abs(d) >= R:
                continue
            h = np.sqrt(R * R - d * d)
            for yl in (lcy + h, lcy - h):
                if abs(yl) > xr * TAN10:
                    continue
                # angle of the point seen from the centre, in the global frame
                gx = xr * np.cos(al) - yl * np.sin(al)
                gy = xr * np.sin(al) + yl * np.cos(al)
                a = np.arctan2(gy - cy, gx - cx)
                th = ((a - a0) * w) % (2 * np.pi)
                n = 0
                while th + 2 * np.pi * n <= turns * 2 * np.pi + 1e-12:
                    t = th + 2 * np.pi * n
                    n += 1
                    z = z0 + tanl * R * t
                    if abs(z) > z_max or (z >= 0) != (z0 >= 0 if z0 != 0 else tanl >= 0):
                        continue
                    # physical direction: tangent in the sense of rotation, in the local frame
                    ta = a + w * np.pi / 2 - al
                    out.append(dict(sector=k + (0 if z >= 0 else 18), row=r, x=xr, y=yl, z=z, theta=t,
                                    sinphi=np.sin(ta), outgoing=np.cos(ta) > 0))
    return out


def frame_from(particles, n_sectors=36):
    """Assemble a synth.Frame from lists of cluster dicts (one list per particle); truth = particle index.
    Returns (frame, per-cluster info arrays dict)."""
    rows = []
    for pid, cls in enumerate(particles):
        for c in cls:
            rows.append((c["sector"], c["row"], c["x"], c["y"], c["z"], pid, c["theta"], c["sinphi"], c["outgoing"]))
    rows.sort(key=lambda t: (t[0], t[1], t[4], t[3]))
    n = len(rows)
    cl = np.zeros(n, synth.CLUSTER_DTYPE)
    truth = np.zeros(n, np.int32)
    theta, sinphi, outgoing = np.zeros(n), np.zeros(n), np.zeros(n, bool)
    so = np.zeros(n_sectors + 1, np.int32)
    for i, t in enumerate(rows):
        cl[i] = (t[2], t[3], t[4], t[1])
        truth[i] = t[5]
        theta[i], sinphi[i], outgoing[i] = t[6], t[7], t[8]
        so[t[0] + 1] += 1
    so = np.cumsum(so).astype(np.int32)
    fr = synth.Frame(cl, so, truth, np.zeros((len(particles), 8)), n_sectors, "loopers")
    return fr, dict(theta=theta, sinphi=sinphi, outgoing=outgoing)
