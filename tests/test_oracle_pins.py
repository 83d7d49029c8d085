"""Pins the oracle to things other than itself (③): hand-worked closed forms of the
definition (5a-c), the Minkowski-difference definition, dense brute force, finite
differences.  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import psdf_oracle as O
from paper_2607_04310_b200 import workloads as W
from tests import geom_ref as G

GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")
ENV = {"sqrt": math.sqrt, "cos": math.cos, "sin": math.sin, "pi": math.pi, "__builtins__": {}}
FP = {"rect": W.rectangle(0.6, 0.4), "sq": W.rectangle(1.0, 1.0)}


def _num(tok):
    return float(eval(tok, ENV))


def _poly(spec):
    t = spec.split()
    if t[0] == "box":
        x0, x1, y0, y1 = map(_num, t[1:])
        return np.array([[x0, y0], [x1, y0], [x1, y1], [x0, y1]])
    v = np.array(list(map(_num, t[1:]))).reshape(-1, 2)
    return v


def _scene(polys, E=None, M_extra=0):
    E = E or max(len(p) for p in polys)
    M = len(polys) + M_extra
    A = np.full((M, E, 2), 7.5)
    B = np.full((M, E, 2), -3.25)
    S = np.zeros((M, E), np.uint8)
    for i, p in enumerate(polys):
        k = len(p)
        A[i, :k], B[i, :k], S[i, :k] = p, np.roll(p, -1, axis=0), 1
    return A, B, S


def _cases(path=GOLD):
    out = []
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        f = [x.strip() for x in line.split("|")]
        out.append(f)
    return out


@pytest.mark.parametrize("case", _cases(), ids=lambda c: c[0])
def test_closed_forms(case):
    cid, fpn, pose, obst, val, grad, per, _ = case
    pose = [_num(t) for t in pose.split()]
    polys = [_poly(s) for s in obst.split(";")]
    A, B, S = _scene(polys)
    r = O.evaluate(FP[fpn], A, B, S, [pose], per_obstacle=True, window=-1.0)
    assert abs(r.value[0] - _num(val)) < 1e-12, cid
    if grad != "-":
        g = [_num(t) for t in grad.split()]
        assert np.allclose(r.grad[0], g, atol=1e-12), cid
        assert r.margin[0] > 1e-4
    else:
        assert r.margin[0] <= 1e-12          # listed "value only" because of a tie
    if per != "-":
        for k, tok in enumerate(per.split(None, 1)):
            if tok.strip() != "-":
                assert abs(r.per_obstacle[0, k] - _num(tok)) < 1e-12
    # the winner row and its branch (eq.(23): separated <=> value > 0; contact counts as not separated)
    assert r.branch[0] == (1 if _num(val) > 0 else 0), cid
    assert r.winner[0] == int(np.argmin(r.per_obstacle[0])), cid
    if cid == "P8":
        assert r.winner[0] == 1


MARGINS = os.path.join(os.path.dirname(__file__), "golden", "margins.txt")
_K = 0.3 * math.cos(0.3) + 0.2 * math.sin(0.3)
_YW = 0.2 * math.cos(0.3) - 0.3 * math.sin(0.3)


@pytest.mark.parametrize("case", _cases(MARGINS), ids=lambda c: c[0])
def test_margin_rule_exact(case):
    """Rule O7 / reading G9 pinned to hand-worked values: the gap of a loser with a different
    gradient, a same-gradient loser passing its own margin on (shifted by the gap), structural
    ties that share a witness, and a competitor inside one obstacle.  Replacing `gap + c[k].m`
    in the oracle's reduce() by INF fails M2, by `gap` fails M2, M3, M4 (and P2)."""
    cid, fpn, pose, obst, winner, margin, _ = case
    ENV.update(k=_K, yw=_YW)
    pose = [_num(t) for t in pose.split()]
    A, B, S = _scene([_poly(s) for s in obst.split(";")])
    for window in (-1.0, 0.2):                              # all duals, and the windowed mode bench/tests use
        r = O.evaluate(FP[fpn], A, B, S, [pose], per_obstacle=True, window=window)
        assert abs(r.margin[0] - _num(margin)) < 1e-12, (cid, window, r.margin[0], _num(margin))
        assert r.winner[0] == int(winner) and r.branch[0] == 1


def test_mpc_coeffs_hand_worked():
    """eqs.(26)-(28), on P8 (phi = 0.9-k = 0.554295012, grad (1, 0, -yw) with
    yw = 0.10241124): r_max = sqrt(0.3^2+0.2^2) = sqrt(0.13) = 0.360555128, rho_p = rho_theta = 0.1:
    gamma = 0.5*(0.360555128+0.554295012)*0.01 + 0.01 = 0.014574251,
    h - gamma = 0.554295012 - 0.01 - 0.014574251 = 0.529720761,  J_g = (-1, 0, +0.10241124)."""
    A, B, S = _scene([_poly("box 1 2 1 2"), _poly("box -2 -0.9 -0.3 0.4")])
    r = O.evaluate(FP["rect"], A, B, S, [(0.0, 0.0, 0.3)], window=-1.0)
    c = O.mpc_coeffs(r.value, r.grad, FP["rect"], 0.01, 0.1, 0.1)
    assert c.shape == (1, 4)
    assert np.abs(c[0] - np.array([0.529720761, -1.0, 0.0, 0.10241124])).max() < 5e-9
    # independent numbers: gamma of a literal phi, two stages, different radii
    c2 = O.mpc_coeffs([1.0, 2.0], [[0.6, 0.8, 0.1], [0.0, -1.0, -0.2]], [[3, 4], [-3, 4], [-3, -4], [3, -4]], 0.25, 0.2, 0.5)
    # r_max = 5: gamma = 0.5*(5+1)*0.25 + 0.1 = 0.85 ; 0.5*(5+2)*0.25 + 0.1 = 0.975
    assert np.allclose(c2, [[1.0 - 0.25 - 0.85, -0.6, -0.8, -0.1], [2.0 - 0.25 - 0.975, 0.0, 1.0, 0.2]], rtol=0, atol=1e-15)
    # no obstacle in view (reading G17): inactive constraint row
    c3 = O.mpc_coeffs([np.inf], [[0.0, 0.0, 0.0]], FP["rect"], 0.01, 0.1, 0.1)
    assert np.isposinf(c3[0, 0]) and (c3[0, 1:] == 0).all()


def test_axis_aligned_box_box_formula():
    """General closed form: gap sqrt(gx^2+gy^2) / overlap -min(ox,oy) for axis-aligned boxes."""
    rng = np.random.default_rng(7)
    for _ in range(300):
        w, h = rng.uniform(0.2, 2, 2)
        fp = W.rectangle(w, h)
        px, py = rng.uniform(-3, 3, 2)
        x0, y0 = rng.uniform(-3, 3, 2)
        x1, y1 = x0 + rng.uniform(0.2, 2), y0 + rng.uniform(0.2, 2)
        A, B, S = _scene([_poly(f"box {x0} {x1} {y0} {y1}")])
        th = rng.choice([0.0, math.pi])                     # half-turn keeps it axis-aligned
        got = O.evaluate(fp, A, B, S, [(px, py, th)]).value[0]
        gx = max(x0 - (px + w / 2), (px - w / 2) - x1)
        gy = max(y0 - (py + h / 2), (py - h / 2) - y1)
        if gx > 0 or gy > 0:
            want = math.hypot(max(gx, 0), max(gy, 0))
        else:
            want = -min(-gx, -gy)
        assert abs(got - want) < 1e-12


def _random_case(rng, penetrate=None):
    V = int(rng.integers(3, 9))
    fp = W.convex_kgon(rng, V, rng.uniform(0.3, 1.0))
    k = int(rng.integers(3, 9))
    ob = W.place(W.convex_kgon(rng, k, rng.uniform(0.3, 1.5)), rng.uniform(-2.5, 2.5, 2), 0.0)
    pose = np.array([rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-math.pi, math.pi)])
    return fp, ob, pose


def test_minkowski_definition_random():
    """sd of eqs.(5a-c) == signed distance of the origin to the Minkowski difference.
    Pins pools (14)-(16), SAT (17)-(22) and the selection (23) jointly, both signs."""
    rng = np.random.default_rng(11)
    npos = nneg = 0
    for _ in range(1500):
        fp, ob, pose = _random_case(rng)
        A, B, S = _scene([ob], E=10)
        got = O.evaluate(fp, A, B, S, [pose]).value[0]
        want = G.sd_minkowski(G.posed(fp, pose), ob)
        assert abs(got - want) < 1e-11, (got, want)
        npos += got > 0
        nneg += got < 0
    assert npos > 200 and nneg > 200


def test_bruteforce_tiny():
    rng = np.random.default_rng(13)
    seen = {True: 0, False: 0}
    for _ in range(40):
        fp, ob, pose = _random_case(rng)
        A, B, S = _scene([ob], E=10)
        got = O.evaluate(fp, A, B, S, [pose]).value[0]
        rw = G.posed(fp, pose)
        if got > 0:
            ub = G.dist_bruteforce(rw, ob)                  # from above, error <= ~perimeter/k
            assert got - 1e-12 <= ub <= got + 5e-3
        else:
            ub = G.pen_bruteforce(rw, ob)                   # from above, error O(angle step)
            assert -got - 1e-12 <= ub <= -got + 1e-3
        seen[got > 0] += 1
    assert seen[True] >= 5 and seen[False] >= 5


def test_finite_difference_gradient():
    """Central differences (h=1e-6, double) where the margin allows (reading G9)."""
    w = W.make_config(2)
    r = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    rng = np.random.default_rng(17)
    extra = np.stack([rng.uniform(0, 20, 400), rng.uniform(0, 20, 400),
                      rng.uniform(-math.pi, math.pi, 400)], axis=1)
    poses = np.concatenate([w.poses.astype(np.float64), extra])
    r = O.evaluate(w.footprint, w.A, w.B, w.S, poses)
    h = 1e-6
    ok = (r.margin > 1e-4) & (np.abs(r.value) > 1e-3)
    assert ok.mean() > 0.8
    fd = np.empty((len(poses), 3))
    for k in range(3):
        d = np.zeros(3)
        d[k] = h
        fd[:, k] = (O.evaluate_value_only(w.footprint, w.A, w.B, w.S, poses + d)
                    - O.evaluate_value_only(w.footprint, w.A, w.B, w.S, poses - d)) / (2 * h)
    err = np.abs(fd - r.grad)[ok]
    assert err.max() < 2e-5, err.max()
    # both branches were exercised
    assert (r.value[ok] < 0).sum() > 20 and (r.value[ok] > 0).sum() > 20


def test_gradient_closed_form_witness():
    """|grad_p phi| = 1 on both branches away from ties (unit gradient)."""
    w = W.make_config(3, n_traj=64)
    r = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    ok = (r.margin > 1e-4) & (np.abs(r.value) > 1e-3)
    gn = np.hypot(r.grad[ok, 0], r.grad[ok, 1])
    assert np.abs(gn - 1.0).max() < 1e-9
    rmax = np.hypot(w.footprint[:, 0], w.footprint[:, 1]).max()
    sep = ok & (r.value > 0)
    assert np.abs(r.grad[sep, 2]).max() <= rmax + 1e-9      # witness lies on the robot


def test_window_mode_equals_full_duals():
    w = W.make_config(2)
    a = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses, window=-1.0)
    b = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses, window=0.01)
    assert np.array_equal(a.value, b.value) and np.array_equal(a.grad, b.grad)
    assert np.array_equal(np.minimum(a.margin, 0.01), b.margin)


def test_component_min_and_trajectory_reduce_definitions():
    """NEXT-4 reductions: hand-worked values (the oracle's definitions against arithmetic done
    by hand), and the union property phi(E1 u E2) = min(phi(E1), phi(E2)) on an L-shaped
    obstacle given as two convex boxes."""
    from oracle import psdf_oracle as O
    pc = np.array([[3.0, -1.0, 2.0, 0.5], [0.25, 4.0, -2.0, np.inf]])
    out = O.component_min(pc, [1, 0, 1, 5], 3)                    # id 5 ignored, obstacle 2 has no component
    assert np.array_equal(out, np.array([[-1.0, 2.0, np.inf], [4.0, -2.0, np.inf]]))
    v = np.array([1.0, 0.2, 0.2, 3.0, -0.5, 0.6, 0.7, 0.1])
    mn, am, pen = O.trajectory_reduce(v, 2, 4, 0.5)
    assert np.array_equal(mn, [0.2, -0.5]) and np.array_equal(am, [1, 0])
    assert np.allclose(pen, [0.09 + 0.09, 1.0 + 0.16], rtol=0, atol=1e-15)
    # L-shape = box[0,2]x[0,1] u box[0,1]x[1,2]; rect robot (0.6x0.4) at (2,2,0) spans
    # [1.7,2.3]x[1.8,2.2]: it overlaps the first box in x (gap 0.8 in y) and the second in y
    # (gap 0.7 in x), so the components give (0.8, 0.7) and the obstacle 0.7
    rect = np.array([[-0.3, -0.2], [0.3, -0.2], [0.3, 0.2], [-0.3, 0.2]])
    def box(x0, x1, y0, y1):
        P = np.array([[x0, y0], [x1, y0], [x1, y1], [x0, y1]], np.float64)
        return P, np.roll(P, -1, axis=0)
    A1, B1 = box(0, 2, 0, 1); A2, B2 = box(0, 1, 1, 2)
    A = np.stack([A1, A2]); B = np.stack([B1, B2]); S = np.ones((2, 4), np.uint8)
    r = O.evaluate(rect, A, B, S, np.array([[2.0, 2.0, 0.0], [0.5, 0.5, 0.0]]), per_obstacle=True)
    d = O.component_min(r.per_obstacle, [0, 0], 1)[:, 0]
    assert np.allclose(r.per_obstacle[0], [0.8, 0.7], rtol=0, atol=1e-12)
    assert abs(d[0] - 0.7) < 1e-12 and np.array_equal(d, r.value)
    assert d[1] < 0                                                # inside the first component
