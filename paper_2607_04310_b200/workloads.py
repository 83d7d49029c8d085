"""Seeded synthetic workloads for the PSDF hot path (BASELINE.json configs 1-5).

This module serves BOTH the oracle tests and the CUDA path (tests, bench.py).
It holds only input recipes: random polygons, random poses, padding.  None of
the method's arithmetic (eqs.(11)-(23)) lives here, and it imports
neither the oracle nor the CUDA binding.  The recipe is stated in DESIGN.md §4
and follows SURVEY.md §8(d); the paper's own workloads are "randomly generated
obstacle sets and query poses" and simulator scenes that are not
available, so these inputs stand in for them.

Everything is generated in float64 with numpy's PCG64 (`default_rng(seed)`),
rounded ONCE to float32, and those float32 arrays are the ground truth that
both the oracle and the GPU path receive.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEEDS = {1: 43101, 2: 43102, 3: 43103, 4: 43104, 5: 43105}

MIN_EDGE = 0.02                      # m; Assumption 1 with margin
MAX_ANGLE = math.radians(179.0)      # interior angle bound, same purpose


@dataclass
class Workload:
    name: str
    footprint: np.ndarray            # [V,2] f32, CCW, robot-local
    poses: np.ndarray                # [N,3] f32 (x, y, theta)
    A: np.ndarray                    # [M,E,2] f32 edge starts  (eq.10)
    B: np.ndarray                    # [M,E,2] f32 edge ends
    S: np.ndarray                    # [M,E] u8 validity mask
    want_per_obstacle: bool = False
    meta: dict = field(default_factory=dict)

    @property
    def N(self):
        return int(self.poses.shape[0])

    @property
    def M(self):
        return int(self.A.shape[0])

    @property
    def E(self):
        return int(self.A.shape[1])

    @property
    def V(self):
        return int(self.footprint.shape[0])

    def valid_edges(self) -> np.ndarray:
        return self.S.astype(np.int64).sum(axis=1)

    def n_pairs(self) -> int:
        """A pair = (pose, obstacle row with >=1 valid edge) — SURVEY.md §8(d)."""
        return self.N * int((self.valid_edges() > 0).sum())

    def subsample(self, n: int) -> "Workload":
        """First-n-by-stride subset of the poses (same scene) for CPU-sized parity."""
        if n >= self.N:
            return self
        idx = np.linspace(0, self.N - 1, n).astype(np.int64)
        return Workload(self.name + f"[sub{n}]", self.footprint, self.poses[idx].copy(),
                        self.A, self.B, self.S, self.want_per_obstacle, dict(self.meta))


# --------------------------------------------------------------------------- polygons
def _hull_ccw(pts: np.ndarray) -> np.ndarray:
    """Andrew monotone chain; returns hull vertices CCW, no repeated first point."""
    p = pts[np.lexsort((pts[:, 1], pts[:, 0]))]

    def half(seq):
        out = []
        for q in seq:
            while len(out) >= 2:
                a, b = out[-2], out[-1]
                if (b[0] - a[0]) * (q[1] - a[1]) - (b[1] - a[1]) * (q[0] - a[0]) <= 0.0:
                    out.pop()
                else:
                    break
            out.append(q)
        return out

    lo = half(p)
    up = half(p[::-1])
    return np.array(lo[:-1] + up[:-1], dtype=np.float64)


def _well_formed(poly: np.ndarray) -> bool:
    """Checks on the float32-rounded polygon: strictly convex CCW, edges >= MIN_EDGE,
    interior angles <= 179 deg."""
    q = poly.astype(np.float32).astype(np.float64)
    k = len(q)
    if k < 3:
        return False
    e = np.roll(q, -1, axis=0) - q
    ln = np.hypot(e[:, 0], e[:, 1])
    if (ln < MIN_EDGE).any():
        return False
    en = np.roll(e, -1, axis=0)
    cr = e[:, 0] * en[:, 1] - e[:, 1] * en[:, 0]
    dt = e[:, 0] * en[:, 0] + e[:, 1] * en[:, 1]
    turn = np.arctan2(cr, dt)                      # exterior angle at vertex j+1
    if (turn <= math.pi - MAX_ANGLE).any():        # interior = pi - turn
        return False
    return True


def disc_points(rng, n, radius):
    r = radius * np.sqrt(rng.random(n))
    a = 2.0 * math.pi * rng.random(n)
    return np.stack([r * np.cos(a), r * np.sin(a)], axis=1)


def hull_of_disc_points(rng, npts: int, radius: float) -> np.ndarray:
    """Config 1 literal: convex hull of `npts` uniform disc points (edge count falls
    where it falls)."""
    while True:
        h = _hull_ccw(disc_points(rng, npts, radius))
        if _well_formed(h):
            return h


def convex_kgon(rng, k: int, radius: float) -> np.ndarray:
    """Convex polygon with exactly k vertices: hull of 8k (k<=8) or 16k disc points,
    random k-subset of the hull vertices in cyclic order."""
    npts = 8 * k if k <= 8 else 16 * k
    while True:
        h = _hull_ccw(disc_points(rng, npts, radius))
        if len(h) < k:
            continue
        keep = np.sort(rng.choice(len(h), size=k, replace=False))
        poly = h[keep]
        if _well_formed(poly):
            return poly


def rectangle(L: float, W: float) -> np.ndarray:
    return np.array([[L / 2, -W / 2], [L / 2, W / 2], [-L / 2, W / 2], [-L / 2, -W / 2]],
                    dtype=np.float64)


def chamfered_rectangle(L: float, W: float, c: float) -> np.ndarray:
    x, y = L / 2, W / 2
    return np.array([[x, -y + c], [x, y - c], [x - c, y], [-x + c, y],
                     [-x, y - c], [-x, -y + c], [-x + c, -y], [x - c, -y]], dtype=np.float64)


def place(poly: np.ndarray, centre, yaw: float) -> np.ndarray:
    c, s = math.cos(yaw), math.sin(yaw)
    R = np.array([[c, -s], [s, c]])
    return poly @ R.T + np.asarray(centre)[None, :]


def pad_scene(rng, polys, E: int, extra_rows: int = 0):
    """Polygons (list of [k,2] CCW, world frame) -> padded A,B,S of eq.(10).
    Valid edges get S=1 at a RANDOM subset of the E slots (kept in cyclic order; the
    mask is not assumed to be a prefix); padded slots hold finite
    non-zero garbage.  `extra_rows` fully-masked rows are appended (M-bar >= M)."""
    M = len(polys) + extra_rows
    A = rng.uniform(-50.0, 150.0, size=(M, E, 2))
    B = rng.uniform(-50.0, 150.0, size=(M, E, 2))
    S = np.zeros((M, E), dtype=np.uint8)
    for i, poly in enumerate(polys):
        k = len(poly)
        assert 3 <= k <= E
        slots = np.sort(rng.choice(E, size=k, replace=False))
        A[i, slots] = poly
        B[i, slots] = np.roll(poly, -1, axis=0)
        S[i, slots] = 1
    A32 = A.astype(np.float32)
    B32 = B.astype(np.float32)
    # closed polygons must stay closed after rounding: B_j is bit-identical to A_next
    for i, poly in enumerate(polys):
        slots = np.nonzero(S[i])[0]
        B32[i, slots] = np.roll(A32[i, slots], -1, axis=0)
    return A32, B32, S


# --------------------------------------------------------------------------- poses
def near_contact_pose(rng, footprint, polys, s: float):
    """Pose whose footprint support vertex (in direction -n_out of a random obstacle
    face) sits at signed offset `s` from that face, over a random boundary point q:
    p = q + s*n_out - R(theta) v*.  s<0 penetrates.  Pure placement geometry
    (SURVEY.md §8(d) 'near-contact construction (no oracle needed)')."""
    i = int(rng.integers(len(polys)))
    poly = polys[i]
    j = int(rng.integers(len(poly)))
    a, b = poly[j], poly[(j + 1) % len(poly)]
    q = a + rng.uniform(0.15, 0.85) * (b - a)
    t = (b - a) / np.hypot(*(b - a))
    n_out = np.array([t[1], -t[0]])                 # CCW polygon: outward = right of travel
    th = rng.uniform(-math.pi, math.pi)
    c, sn = math.cos(th), math.sin(th)
    rv = footprint @ np.array([[c, -sn], [sn, c]]).T
    star = rv[np.argmax(rv @ (-n_out))]
    p = q + s * n_out - star
    return np.array([p[0], p[1], th])


def unicycle_rollouts(rng, n_traj, n_stage, lo, hi, vmax=1.5, wmax=1.0, dt=0.1):
    x = rng.uniform(lo, hi, n_traj)
    y = rng.uniform(lo, hi, n_traj)
    th = rng.uniform(-math.pi, math.pi, n_traj)
    out = np.empty((n_traj, n_stage, 3))
    for s in range(n_stage):
        out[:, s, 0], out[:, s, 1], out[:, s, 2] = x, y, th
        v = rng.uniform(0.0, vmax, n_traj)
        w = rng.uniform(-wmax, wmax, n_traj)
        x = x + dt * v * np.cos(th)
        y = y + dt * v * np.sin(th)
        th = th + dt * w
    return out.reshape(-1, 3)                        # pose index = traj*n_stage + stage


def bicycle_rollouts(rng, starts, n_stage, wheelbase=2.7, dt=0.1):
    n = len(starts)
    x, y, th = starts[:, 0].copy(), starts[:, 1].copy(), starts[:, 2].copy()
    out = np.empty((n, n_stage, 3))
    for s in range(n_stage):
        out[:, s, 0], out[:, s, 1], out[:, s, 2] = x, y, th
        v = rng.uniform(-1.0, 2.0, n)
        d = rng.uniform(-0.5, 0.5, n)
        x = x + dt * v * np.cos(th)
        y = y + dt * v * np.sin(th)
        th = th + dt * v / wheelbase * np.tan(d)
    return out.reshape(-1, 3)


def _replace(rng, poses, frac_idx, maker):
    idx = rng.choice(len(poses), size=frac_idx, replace=False)
    for k in idx:
        poses[k] = maker()
    return np.sort(idx)


# --------------------------------------------------------------------------- configs
RECT_ROBOT = rectangle(0.6, 0.4)


def config1() -> Workload:
    """MPC-sized: H=20, M=8 hulls of 8 disc points, E=8 (BASELINE.json configs[0])."""
    rng = np.random.default_rng(SEEDS[1])
    polys = [place(hull_of_disc_points(rng, 8, rng.uniform(0.2, 1.5)),
                   rng.uniform(0, 20, 2), 0.0) for _ in range(8)]
    A, B, S = pad_scene(rng, polys, 8)
    poses = np.stack([rng.uniform(0, 20, 20), rng.uniform(0, 20, 20),
                      rng.uniform(-math.pi, math.pi, 20)], axis=1)
    near = _replace(rng, poses, 4,
                    lambda: near_contact_pose(rng, RECT_ROBOT, polys, rng.uniform(-0.3, 0.3)))
    return Workload("cfg1_mpc", RECT_ROBOT.astype(np.float32), poses.astype(np.float32),
                    A, B, S, False, {"near_idx": near})


def _kgon_scene(rng, M, kmin, kmax, rmin, rmax, arena, E, extra_rows=0):
    polys = []
    for _ in range(M):
        k = int(rng.integers(kmin, kmax + 1))
        polys.append(place(convex_kgon(rng, k, rng.uniform(rmin, rmax)),
                           rng.uniform(0, arena, 2), 0.0))
    A, B, S = pad_scene(rng, polys, E, extra_rows)
    return polys, A, B, S


def config2() -> Workload:
    """Dense scene: N=50 one trajectory, M=64 k-gons k in 3..8, E=8, per-obstacle out."""
    rng = np.random.default_rng(SEEDS[2])
    polys, A, B, S = _kgon_scene(rng, 64, 3, 8, 0.2, 1.5, 20.0, 8)
    poses = unicycle_rollouts(rng, 1, 50, 6.0, 14.0)
    cent = np.array([p.mean(axis=0) for p in polys])

    def special():
        if rng.random() < 0.5:                     # narrow gap: midpoint of two nearest obstacles
            i = int(rng.integers(len(polys)))
            d = np.hypot(*(cent - cent[i]).T)
            d[i] = np.inf
            k = int(np.argmin(d))
            m = 0.5 * (cent[i] + cent[k])
            return np.array([m[0], m[1], rng.uniform(-math.pi, math.pi)])
        return near_contact_pose(rng, RECT_ROBOT, polys, rng.uniform(-0.3, 0.1))

    near = _replace(rng, poses, 15, special)
    return Workload("cfg2_dense", RECT_ROBOT.astype(np.float32), poses.astype(np.float32),
                    A, B, S, True, {"near_idx": near})


def config3(n_traj: int = 4096) -> Workload:
    """Sampled-trajectory batch: n_traj x 50 unicycle random walks, M=256, E=8."""
    rng = np.random.default_rng(SEEDS[3])
    polys, A, B, S = _kgon_scene(rng, 256, 3, 8, 0.2, 1.5, 40.0, 8)
    poses = unicycle_rollouts(rng, n_traj, 50, 0.0, 40.0)
    return Workload("cfg3_sampled", RECT_ROBOT.astype(np.float32), poses.astype(np.float32),
                    A, B, S, False, {"n_traj": n_traj, "n_stage": 50})


CAR = chamfered_rectangle(4.5, 1.8, 0.3)


def config4(n_traj: int = 1024) -> Workload:
    """Parking: 8-vertex car, n_traj x 100 bicycle rollouts, M=1024 (half parked-car
    rectangles, half k-gons k in 3..16), E=16, 60x60 m lot.  Obstacles sit in row
    bands (parking rows) separated by aisles; rollouts start in the aisles."""
    rng = np.random.default_rng(SEEDS[4])
    band_y = np.arange(4.0, 60.0, 12.0)             # 5 parking bands, 5.5 m deep
    aisle_y = band_y + 6.0                          # aisle centre lines between them
    polys = []
    for i in range(1024):
        yb = band_y[int(rng.integers(len(band_y)))] + rng.uniform(-2.2, 2.2)
        xb = rng.uniform(0, 60)
        if i % 2 == 0:
            poly = rectangle(rng.uniform(2.0, 5.0), rng.uniform(1.5, 2.2))
        else:
            poly = convex_kgon(rng, int(rng.integers(3, 17)), rng.uniform(0.2, 1.5))
        polys.append(place(poly, (xb, yb), rng.uniform(-math.pi, math.pi)))
    A, B, S = pad_scene(rng, polys, 16)
    starts = np.stack([rng.uniform(5, 55, n_traj),
                       aisle_y[rng.integers(len(aisle_y) - 1, size=n_traj)] + rng.uniform(-0.8, 0.8, n_traj),
                       rng.choice([0.0, math.pi], n_traj) + rng.uniform(-0.15, 0.15, n_traj)], axis=1)
    poses = bicycle_rollouts(rng, starts, 100)
    near = _replace(rng, poses, len(poses) // 4,
                    lambda: near_contact_pose(rng, CAR, polys, rng.uniform(-0.4, 0.2)))
    return Workload("cfg4_parking", CAR.astype(np.float32), poses.astype(np.float32),
                    A, B, S, False, {"near_idx": near, "n_traj": n_traj, "n_stage": 100})


def hex_robot(rng) -> np.ndarray:
    """6 points at radius 0.5 with jittered angles: exactly 6 hull vertices, CCW."""
    ang = (np.arange(6) + rng.uniform(-0.3, 0.3, 6)) * (math.pi / 3.0)
    return 0.5 * np.stack([np.cos(ang), np.sin(ang)], axis=1)


def config5(n_poses: int = 65536) -> Workload:
    """Throughput stress: 6-vertex robot, n_poses uniform poses, M=4096 k-gons k in
    3..12, R~U[0.2,2], E=12, 100x100 m.  ~10 % of the poses penetrate (near-contact
    construction with s<0); the other ~90 % are drawn uniformly and kept only when the
    robot's bounding circle clears every obstacle's generating disc (a conservative
    placement test on the generator's own discs, not a PSDF evaluation)."""
    from scipy.spatial import cKDTree
    rng = np.random.default_rng(SEEDS[5])
    robot = hex_robot(rng)
    M = 4096
    polys, cen, rad = [], np.empty((M, 2)), np.empty(M)
    for i in range(M):
        k = int(rng.integers(3, 13))
        rad[i] = rng.uniform(0.2, 2.0)
        cen[i] = rng.uniform(0, 100, 2)
        polys.append(place(convex_kgon(rng, k, rad[i]), cen[i], 0.0))
    A, B, S = pad_scene(rng, polys, 12)
    tree = cKDTree(cen)
    n_pen = n_poses // 10
    n_clear = n_poses - n_pen
    clear = np.empty((0, 2))
    while len(clear) < n_clear:
        cand = rng.uniform(0, 100, size=(4 * n_poses, 2))
        d, nb = tree.query(cand, k=32, distance_upper_bound=2.0 + 0.5 + 1e-3)
        hit = np.isfinite(d)                        # missing neighbours come back inf
        r_nb = np.where(hit, rad[np.minimum(nb, M - 1)], 0.0)
        ok = ~((hit & (d <= r_nb + 0.5 + 1e-3)).any(axis=1) | hit[:, -1])
        clear = np.concatenate([clear, cand[ok]])
    poses = np.empty((n_poses, 3))
    poses[:n_clear, :2] = clear[:n_clear]
    poses[:n_clear, 2] = rng.uniform(-math.pi, math.pi, n_clear)
    for k in range(n_clear, n_poses):
        poses[k] = near_contact_pose(rng, robot, polys, rng.uniform(-0.3, -0.005))
    poses = poses[rng.permutation(n_poses)]
    return Workload("cfg5_stress", robot.astype(np.float32), poses.astype(np.float32),
                    A, B, S, False, {})


def make_config(idx: int, **kw) -> Workload:
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[idx](**kw)


def table1_case(M: int, Bsz: int, seed: int = 43110) -> Workload:
    """Paper Table I shape: M random obstacles, B query
    poses; footprint / edges per obstacle are not stated in the paper:
    rectangle robot, k-gons k in 3..8, E=8, 20x20 m arena."""
    rng = np.random.default_rng(seed + 1000 * M + Bsz)
    polys, A, B, S = _kgon_scene(rng, M, 3, 8, 0.2, 1.5, 20.0, 8)
    poses = np.stack([rng.uniform(0, 20, Bsz), rng.uniform(0, 20, Bsz),
                      rng.uniform(-math.pi, math.pi, Bsz)], axis=1)
    return Workload(f"table1_M{M}_B{Bsz}", RECT_ROBOT.astype(np.float32),
                    poses.astype(np.float32), A, B, S, False, {})
