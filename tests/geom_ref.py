"""Independent numpy definitions used ONLY to pin the oracle (never by the product).

They restate the DEFINITION of signed distance, eqs.(5a-c), by routes that
share nothing with the paper's algorithm (§IV) that the oracle follows:
  * Minkowski difference: sd(P0,P) = signed distance of the origin to co{a - w};
  * brute force: dense boundary sampling (separated), dense direction sweep (overlap).
"""
import math

import numpy as np


def posed(fp, pose):
    x, y, th = pose
    c, s = math.cos(th), math.sin(th)
    return np.asarray(fp, float) @ np.array([[c, -s], [s, c]]).T + np.array([x, y])


def hull_ccw(pts):
    pts = np.unique(np.asarray(pts, float), axis=0)
    p = pts[np.lexsort((pts[:, 1], pts[:, 0]))]

    def half(seq):
        out = []
        for q in seq:
            while len(out) >= 2 and ((out[-1][0] - out[-2][0]) * (q[1] - out[-2][1])
                                     - (out[-1][1] - out[-2][1]) * (q[0] - out[-2][0])) <= 0:
                out.pop()
            out.append(q)
        return out
    lo, up = half(p), half(p[::-1])
    return np.array(lo[:-1] + up[:-1])


def sd_minkowski(robot_w, obst):
    """Signed distance of the origin to the Minkowski difference polygon co{a - w}."""
    D = hull_ccw((obst[:, None, :] - robot_w[None, :, :]).reshape(-1, 2))
    a, b = D, np.roll(D, -1, axis=0)
    e = b - a
    ln = np.hypot(e[:, 0], e[:, 1])
    # signed distance of origin to each supporting line, outward normal (CCW: right of travel)
    nout = np.stack([e[:, 1], -e[:, 0]], axis=1) / ln[:, None]
    sline = -(a * nout).sum(axis=1)                 # >0: origin outside that face
    if (sline <= 0).all():
        return float(sline.max())                   # inside: -(min distance to a face line)
    t = np.clip(-(a * e).sum(axis=1) / ln ** 2, 0.0, 1.0)
    q = a + t[:, None] * e
    return float(np.hypot(q[:, 0], q[:, 1]).min())


def boundary_samples(poly, k):
    a, b = poly, np.roll(poly, -1, axis=0)
    t = np.linspace(0.0, 1.0, k, endpoint=False)
    return (a[:, None, :] + t[None, :, None] * (b - a)[:, None, :]).reshape(-1, 2)


def dist_bruteforce(robot_w, obst, k=500):
    """Upper bound converging to dist from above: min over dense boundary samples."""
    p, q = boundary_samples(robot_w, k), boundary_samples(obst, k)
    best = np.inf
    for c in np.array_split(p, 16):
        d = np.hypot(c[:, None, 0] - q[None, :, 0], c[:, None, 1] - q[None, :, 1])
        best = min(best, float(d.min()))
    return best


def pen_bruteforce(robot_w, obst, k=200000):
    """min over k unit directions u of the overlap h_R(u) + h_O(-u): the translation
    along -u that just separates.  Converges to pen from above."""
    ang = np.linspace(0.0, 2.0 * math.pi, k, endpoint=False)
    u = np.stack([np.cos(ang), np.sin(ang)], axis=1)
    hr = (u @ robot_w.T).max(axis=1)
    ho = (-(u @ obst.T)).max(axis=1)
    return float((hr + ho).min())


def valid_polys(A, S):
    return [np.asarray(A[i][np.asarray(S[i]).astype(bool)], float) for i in range(len(A))]
