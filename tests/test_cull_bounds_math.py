"""The two lower bounds behind exact culling (psdf_cull_kernels.cuh), checked
as mathematics against the oracle on CPU: for every (pose, obstacle)

    sd^i >= |c_R - c_i| - R_i - r_R                       (bounding circles)
    sd^i >= max over the four box axes of the projection gap    (oriented bounding boxes)

with the boxes built by the packer's rule (footprint: robot-frame bounding box; obstacle:
smallest-area box aligned with one of its own edges).  Restated here in numpy, sharing no
code with the CUDA path; a bound that ever exceeded the oracle's signed distance would make
the culled kernel drop a relevant obstacle."""
import numpy as np

from oracle import psdf_oracle as O
from paper_2607_04310_b200 import workloads as W


def _obstacle_box(poly):
    """(centre, unit axis u, half extents (hx, hy), circle radius about the centre)."""
    best = None
    for k in range(len(poly)):
        t = poly[(k + 1) % len(poly)] - poly[k]
        t = t / np.linalg.norm(t)
        n = np.array([-t[1], t[0]])
        pt, pn = poly @ t, poly @ n
        area = (pt.max() - pt.min()) * (pn.max() - pn.min())
        if best is None or area < best[0]:
            best = (area, t, n, 0.5 * (pt.max() + pt.min()), 0.5 * (pn.max() + pn.min()))
    _, t, n, mt, mn = best
    c = mt * t + mn * n
    d = poly - c
    return c, t, np.array([np.abs(d @ t).max(), np.abs(d @ n).max()]), np.linalg.norm(d, axis=1).max()


def _bounds(footprint, pose, poly):
    lo, hi = footprint.min(0), footprint.max(0)
    c0, h0 = 0.5 * (lo + hi), 0.5 * (hi - lo)
    r0 = np.linalg.norm(footprint - c0, axis=1).max()
    cs, sn = np.cos(pose[2]), np.sin(pose[2])
    U, N = np.array([cs, sn]), np.array([-sn, cs])
    cR = pose[:2] + c0[0] * U + c0[1] * N
    c, u, h, R = _obstacle_box(poly)
    n = np.array([-u[1], u[0]])
    dd = c - cR
    circle = np.linalg.norm(dd) - R - r0

    def gap(axis):
        ext_o = h[0] * abs(u @ axis) + h[1] * abs(n @ axis)
        ext_r = h0[0] * abs(U @ axis) + h0[1] * abs(N @ axis)
        return abs(dd @ axis) - ext_o - ext_r

    return circle, max(gap(u), gap(n), gap(U), gap(N))


def test_lower_bounds_never_exceed_the_signed_distance():
    rng = np.random.default_rng(4310)
    footprints = [W.rectangle(0.6, 0.4), W.chamfered_rectangle(4.5, 1.8, 0.3), W.hex_robot(rng),
                  W.rectangle(4.5, 1.8) + np.array([1.35, 0.0])]        # last: reference point off-centre
    worst_c, worst_b, tight = -np.inf, -np.inf, 0
    n_cases = 0
    for fp in footprints:
        scale = float(np.abs(fp).max())
        polys = []
        for _ in range(60):
            if rng.random() < 0.5:
                poly = W.rectangle(float(rng.uniform(2, 5)), float(rng.uniform(1.5, 2.2)))
            else:
                poly = W.convex_kgon(rng, int(rng.integers(3, 13)), float(rng.uniform(0.2, 2.0)))
            polys.append(W.place(poly, rng.uniform(-6, 6, 2), float(rng.uniform(-np.pi, np.pi))))
        A, B, S = W.pad_scene(rng, polys, 12)
        poses = np.column_stack([rng.uniform(-8 - scale, 8 + scale, (40, 2)), rng.uniform(-np.pi, np.pi, 40)])
        ref = O.evaluate(fp.astype(np.float32), A, B, S, poses.astype(np.float32), per_obstacle=True)
        fp32 = fp.astype(np.float32).astype(np.float64)
        for n, pose in enumerate(poses.astype(np.float32).astype(np.float64)):
            for i in range(len(polys)):
                poly = A[i][S[i] == 1].astype(np.float64)
                circle, box = _bounds(fp32, pose, poly)
                sd = ref.per_obstacle[n, i]
                worst_c = max(worst_c, circle - sd)
                worst_b = max(worst_b, box - sd)
                tight += box > circle
                n_cases += 1
    assert worst_c <= 1e-9 and worst_b <= 1e-9, (worst_c, worst_b)
    assert tight > 0.5 * n_cases                      # the box bound is the tighter one most of the time
    # both signs were exercised
    assert (ref.per_obstacle < 0).any() and (ref.per_obstacle > 0).any()
