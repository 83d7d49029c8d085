"""Invariants that the mathematics fixes (SURVEY.md §8(c) 'Invariants'), checked on the
oracle.  A dropped term, wrong sign, transposed rotation or mask leak breaks one."""
import math

import numpy as np

from oracle import psdf_oracle as O
from paper_2607_04310_b200 import workloads as W


def _ev(w, poses=None, **kw):
    return O.evaluate(w.footprint, w.A, w.B, w.S, w.poses if poses is None else poses, **kw)


def test_rigid_motion_invariance():
    w = W.make_config(2)
    r0 = _ev(w)
    a, t = 0.7321, np.array([3.5, -11.25])
    c, s = math.cos(a), math.sin(a)
    R = np.array([[c, -s], [s, c]])
    A = w.A.astype(np.float64) @ R.T + t
    B = w.B.astype(np.float64) @ R.T + t
    poses = w.poses.astype(np.float64).copy()
    poses[:, :2] = poses[:, :2] @ R.T + t
    poses[:, 2] += a
    r1 = O.evaluate(w.footprint, A, B, w.S, poses)
    assert np.abs(r1.value - r0.value).max() < 1e-11
    ok = (r0.margin > 1e-4) & (np.abs(r0.value) > 1e-3)
    assert np.abs(r1.grad[ok, :2] - r0.grad[ok, :2] @ R.T).max() < 1e-9
    assert np.abs(r1.grad[ok, 2] - r0.grad[ok, 2]).max() < 1e-9


def test_uniform_scaling():
    w = W.make_config(1)
    lam = 3.25
    r0 = _ev(w)
    poses = w.poses.astype(np.float64).copy()
    poses[:, :2] *= lam
    r1 = O.evaluate(w.footprint.astype(np.float64) * lam, w.A.astype(np.float64) * lam,
                    w.B.astype(np.float64) * lam, w.S, poses)
    assert np.abs(r1.value - lam * r0.value).max() < 1e-11


def test_role_swap():
    """sd(P0(x), P) with the obstacle as footprint at identity and the posed robot as the
    obstacle is the same number (the definition is symmetric)."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        fp = W.convex_kgon(rng, int(rng.integers(3, 8)), 0.8)
        ob = W.place(W.convex_kgon(rng, int(rng.integers(3, 8)), 1.0), rng.uniform(-2, 2, 2), 0.0)
        pose = np.array([rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-3, 3)])
        E = 8

        def sc(p):
            A = np.zeros((1, E, 2)); B = np.zeros((1, E, 2)); S = np.zeros((1, E), np.uint8)
            A[0, :len(p)], B[0, :len(p)], S[0, :len(p)] = p, np.roll(p, -1, 0), 1
            return A, B, S
        v1 = O.evaluate(fp, *sc(ob), [pose]).value[0]
        c, s = math.cos(pose[2]), math.sin(pose[2])
        rw = fp @ np.array([[c, -s], [s, c]]).T + pose[:2]
        v2 = O.evaluate(ob, *sc(rw), [(0.0, 0.0, 0.0)]).value[0]
        assert abs(v1 - v2) < 1e-11


def test_masking_padding_permutation():
    w = W.make_config(2)
    r0 = _ev(w, per_obstacle=True)
    assert np.array_equal(r0.value, r0.per_obstacle.min(axis=1))          # eq.(6)
    rng = np.random.default_rng(3)
    # garbage in padded slots is inert
    A, B = w.A.copy(), w.B.copy()
    pad = w.S == 0
    A[pad] = rng.uniform(-1e3, 1e3, size=(pad.sum(), 2)).astype(np.float32)
    B[pad] = rng.uniform(-1e3, 1e3, size=(pad.sum(), 2)).astype(np.float32)
    r1 = O.evaluate(w.footprint, A, B, w.S, w.poses)
    assert np.array_equal(r1.value, r0.value) and np.array_equal(r1.grad, r0.grad)
    # obstacle permutation, duplicates, fully-masked extra rows, wider E
    perm = rng.permutation(w.M)
    r2 = O.evaluate(w.footprint, w.A[perm], w.B[perm], w.S[perm], w.poses, per_obstacle=True)
    assert np.array_equal(r2.value, r0.value)
    assert np.array_equal(r2.per_obstacle, r0.per_obstacle[:, perm])
    A3 = np.concatenate([w.A, w.A[:5], rng.uniform(0, 20, (4, w.E, 2)).astype(np.float32)])
    B3 = np.concatenate([w.B, w.B[:5], rng.uniform(0, 20, (4, w.E, 2)).astype(np.float32)])
    S3 = np.concatenate([w.S, w.S[:5], np.zeros((4, w.E), np.uint8)])
    r3 = O.evaluate(w.footprint, A3, B3, S3, w.poses, per_obstacle=True)
    assert np.array_equal(r3.value, r0.value)
    assert np.isinf(r3.per_obstacle[:, -4:]).all()
    A4 = np.concatenate([w.A, rng.uniform(0, 20, (w.M, 3, 2)).astype(np.float32)], axis=1)
    B4 = np.concatenate([w.B, rng.uniform(0, 20, (w.M, 3, 2)).astype(np.float32)], axis=1)
    S4 = np.concatenate([w.S, np.zeros((w.M, 3), np.uint8)], axis=1)
    r4 = O.evaluate(w.footprint, A4, B4, S4, w.poses)
    assert np.array_equal(r4.value, r0.value) and np.array_equal(r4.grad, r0.grad)
    # cyclic relabelling of an obstacle's edges changes nothing
    A5, B5, S5 = w.A.copy(), w.B.copy(), w.S.copy()
    for i in range(w.M):
        k = int(rng.integers(w.E))
        A5[i], B5[i], S5[i] = np.roll(A5[i], k, 0), np.roll(B5[i], k, 0), np.roll(S5[i], k, 0)
    r5 = O.evaluate(w.footprint, A5, B5, S5, w.poses)
    assert np.abs(r5.value - r0.value).max() < 1e-12


def test_union_is_min_and_empty_scene():
    w = W.make_config(2)
    h = w.M // 2
    ra = O.evaluate(w.footprint, w.A[:h], w.B[:h], w.S[:h], w.poses)
    rb = O.evaluate(w.footprint, w.A[h:], w.B[h:], w.S[h:], w.poses)
    r = _ev(w)
    assert np.array_equal(r.value, np.minimum(ra.value, rb.value))
    re = O.evaluate(w.footprint, w.A, w.B, np.zeros_like(w.S), w.poses)
    assert np.isinf(re.value).all() and (re.value > 0).all()
    assert (re.grad == 0).all() and (re.winner == -1).all()


def test_lipschitz_and_continuity_through_contact():
    """1-Lipschitz in p; continuous across phi=0."""
    w = W.make_config(1)
    k = int(w.meta["near_idx"][0])
    p0 = w.poses[k].astype(np.float64)
    r = O.evaluate(w.footprint, w.A, w.B, w.S, [p0])
    g = r.grad[0, :2] / max(np.hypot(*r.grad[0, :2]), 1e-12)
    ts = np.linspace(-0.6, 0.6, 4001)
    poses = np.stack([p0[0] + ts * g[0], p0[1] + ts * g[1], np.full_like(ts, p0[2])], axis=1)
    v = O.evaluate_value_only(w.footprint, w.A, w.B, w.S, poses)
    step = ts[1] - ts[0]
    assert np.abs(np.diff(v)).max() <= step * (1 + 1e-9)
    assert v.min() < 0 < v.max()
