"""Closed-form helix in float64, written for the tests only (independent of synth/ and oracle/).

Sector-local frame, uniform Bz along +z.  Lorentz force: d(phi)/ds = -0.3 * B[T] * (q/pT) / 100 per cm
(textbook: R[m] = pT[GeV/c] / (0.3 B[T])), so sin(phi) is linear in x.
"""
import numpy as np

KAPPA_PER_T = 0.00299792458  # 1/cm per (T * c/GeV)


def helix_points(xs, x0, y0, z0, sinphi0, tanl, qpt, bz):
    """Points of the helix through (x0,y0,z0) with direction sin(phi0) at the given x planes (outgoing branch)."""
    xs = np.asarray(xs, np.float64)
    k = -KAPPA_PER_T * bz * qpt
    s = sinphi0 + k * (xs - x0)
    c0, c = np.sqrt(1 - sinphi0**2), np.sqrt(1 - s**2)
    if abs(k) < 1e-14:
        y = y0 + (xs - x0) * sinphi0 / c0
        arc = (xs - x0) / c0
    else:
        y = y0 - (c - c0) / k
        arc = (np.arcsin(s) - np.arcsin(sinphi0)) / k
    z = z0 + tanl * arc
    return y, z, s
