"""Float64 extended Kalman filter on the closed-form helix, written for the tests only (independent of oracle/ and csrc/).

Transport = the exact helix map of tests/helix.py; its Jacobian is taken by central differences of that map (no formula
shared with the implementations); the measurement update is the textbook joint 2-D update K = C H^T (H C H^T + V)^-1.
PAPER.md:71: "The final Kalman refit is iterated three times: inward, outward, and inward".
"""
import numpy as np

from tests.helix import helix_points

H = np.zeros((2, 5))
H[0, 0] = H[1, 1] = 1.0


def fmap(p, x0, x1, bz):
    y, z, s = helix_points([x1], x0, p[0], p[1], p[2], p[3], p[4], bz)
    return np.array([y[0], z[0], s[0], p[3], p[4]])


def transport(x0, p, C, x1, bz):
    if x1 == x0:
        return p.copy(), C.copy()
    F = np.zeros((5, 5))
    for j in range(5):
        e = np.zeros(5)
        # q/pT gets a larger step: the closed form (c - c0) / k cancels badly for k ~ 1e-9 (error ~ 1e-7 / k)
        e[j] = (1e-3 if j == 4 else 1e-6) * max(1.0, abs(p[j]))
        F[:, j] = (fmap(p + e, x0, x1, bz) - fmap(p - e, x0, x1, bz)) / (2 * e[j])
    return fmap(p, x0, x1, bz), F @ C @ F.T


def update(p, C, m, V):
    S = H @ C @ H.T + V
    K = C @ H.T @ np.linalg.inv(S)
    r = m - H @ p
    return p + K @ r, (np.eye(5) - K @ H) @ C, float(r @ np.linalg.inv(S) @ r)


def refit(x, y, z, q0, bz, cov0, sy, sz, passes=("in", "out", "in")):
    """Start at the outermost hit with the chord from the second-outermost one and q/pT = q0 (O7); every pass
    resets C to diag(cov0) and chi2 to 0.  Returns (x, state, covariance, chi2 of the last pass)."""
    x, y, z = (np.asarray(a, np.float64) for a in (x, y, z))
    n = len(x)
    dx, dy, dz = x[-1] - x[-2], y[-1] - y[-2], z[-1] - z[-2]
    ds = np.hypot(dx, dy)
    p = np.array([y[-1], z[-1], dy / ds, dz / ds, q0])
    xc = x[-1]
    V = np.diag([sy * sy, sz * sz])
    C, chi2 = None, 0.0
    for d in passes:
        C, chi2 = np.diag(np.asarray(cov0, np.float64)), 0.0
        order = range(n - 1, -1, -1) if d == "in" else range(n)
        for j in order:
            p, C = transport(xc, p, C, x[j], bz)
            xc = x[j]
            p, C, c = update(p, C, np.array([y[j], z[j]]), V)
            chi2 += c
    return xc, p, C, chi2
