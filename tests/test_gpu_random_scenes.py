"""Randomised differential tests (a bounded slice of the long runs described in DESIGN.md §5.6,
§6.7): random footprints (V 3..16, off-centre reference point), random obstacle sets (rectangles
and k-gons, random mask positions, clockwise rows, fully masked rows), poses scattered over and
next to the obstacles, at offsets from the origin.  Every public path is checked against the
oracle or against another path that must agree bit for bit.  Need a B200: `pytest -m gpu`."""
import os

import numpy as np
import pytest

from tests.parity import compare

# Knobs for the long runs (defaults = the bounded slice the suite runs):
#   PSDF_RANDOM_SEED_BASE  first scene seed of test_random_scenes_every_path (default 510000)
#   PSDF_RANDOM_SCENES     scenes per block, four blocks (default 25)
#   PSDF_RANDOM_CULLED     number of culled-vs-dense scenes (default 12)
_SEED_BASE = int(os.environ.get("PSDF_RANDOM_SEED_BASE", "510000"))
_PER_BLOCK = int(os.environ.get("PSDF_RANDOM_SCENES", "25"))
_N_CULLED = int(os.environ.get("PSDF_RANDOM_CULLED", "12"))

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf, workloads as W
    assert torch.cuda.is_available()
    return torch, O, psdf, W


class _Ref:
    def __init__(self, ref, sl, per_obstacle=False, sign=1.0):
        self.value, self.grad, self.margin = ref.value[sl], sign * ref.grad[sl], ref.margin[sl]
        self.per_obstacle = ref.per_obstacle[sl] if per_obstacle else None


def _scene(W, seed):
    rng = np.random.default_rng(seed)
    V = int(rng.integers(3, 17))
    M = int(rng.choice([1, 2, 5, 20, 64, 130, 400]))
    arena = float(rng.choice([3.0, 10.0, 30.0]))
    off = float(rng.choice([0.0, 20.0, -60.0]))
    E = int(rng.choice([3, 4, 6, 8, 12]))
    rmax = float(rng.choice([0.3, 1.5, 4.0]))
    polys = []
    for _ in range(M):
        if E >= 4 and rng.random() < 0.4:
            poly = W.rectangle(float(rng.uniform(0.3, 3) * rmax), float(rng.uniform(0.1, 1) * rmax))
        else:
            rad = float(rng.uniform(0.5, 1.0) * rmax)
            poly = W.convex_kgon(rng, int(rng.integers(3, min(E, 3 + int(rad * 8)) + 1)), rad)
        polys.append(W.place(poly, rng.uniform(0, arena, 2) + off, float(rng.uniform(-np.pi, np.pi))))
    A, B, S = W.pad_scene(rng, polys, E, extra_rows=int(rng.integers(0, 4)))
    for i in range(0, M, 3):                                   # clockwise rows (reading G8)
        sl = np.nonzero(S[i])[0]
        A[i, sl], B[i, sl] = B[i, sl][::-1].copy(), A[i, sl][::-1].copy()
    ang = np.linspace(0, 2 * np.pi, V, endpoint=False) + rng.uniform(0, 1)
    fr = float(rng.choice([0.2, 1.0, 3.0]))
    footprint = (np.stack([fr * np.cos(ang), rng.uniform(0.3, 1.0) * fr * np.sin(ang)], 1)
                 + rng.uniform(-0.5, 0.5, 2) * fr).astype(np.float32)
    N = int(rng.choice([1, 7, 60, 600, 3000]))
    poses = np.empty((N, 3), np.float32)
    poses[:, :2] = rng.uniform(-0.2 * arena, 1.2 * arena, (N, 2)) + off
    nn = N // 3                                                # a third next to obstacle vertices
    if nn:
        k, kk = rng.integers(0, M, nn), rng.integers(0, E, nn)
        poses[:nn, :2] = np.array([polys[a][b % len(polys[a])] for a, b in zip(k, kk)]) + rng.normal(0, 0.3 * fr, (nn, 2))
    poses[:, 2] = rng.uniform(-7, 7, N)
    return rng, footprint, A, B, S, poses, f"seed {seed} V={V} M={M} E={E} arena={arena} off={off} N={N}"


@pytest.mark.parametrize("block", range(4))
def test_random_scenes_every_path(env, block):
    torch, O, psdf, W = env
    for seed in range(_SEED_BASE + _PER_BLOCK * block, _SEED_BASE + _PER_BLOCK * (block + 1)):
        rng, footprint, A, B, S, poses, tag = _scene(W, seed)
        N, Mrows = len(poses), A.shape[0]
        scene = psdf.Scene(footprint, A, B, S, max_poses=max(N, 8))
        idx = np.sort(rng.choice(N, min(N, 100), replace=False))
        ref = O.evaluate(footprint, A, B, S, poses[idx], per_obstacle=True)
        p = torch.from_numpy(poses).cuda()
        v, g, po = scene.eval(p, grad=True, per_obstacle=True)
        compare(ref, v.cpu().numpy()[idx], g.cpu().numpy()[idx], po.cpu().numpy()[idx], what=tag + " eval")
        # host path (single zero-copy launch or graph), all outputs
        vh, gh, poh = scene.eval_host(poses[idx], grad=True, per_obstacle=True)
        compare(ref, vh, gh, poh, what=tag + " eval_host")
        # serving mode (persistent kernel + mailbox): rows bit-equal to the host path, twice, then coefficients
        if len(idx) <= 512:
            try:
                scene.serve_begin(len(idx), idle_timeout_ms=200)
                for _ in range(2):
                    rows = scene.serve_step(poses[idx])
                    assert np.array_equal(rows[:, 0], vh) and np.array_equal(rows[:, 1:], gh), tag + " serve"
                scene.serve_begin(len(idx), coeffs=(0.3, 0.05, 0.02), idle_timeout_ms=200)
                rows = scene.serve_step(poses[idx])
                assert np.array_equal(rows, scene.mpc_coeffs_host(poses[idx], 0.3, 0.05, 0.02)), tag + " serve coeffs"
            finally:
                scene.serve_end()
        # MPC coefficients, eqs.(26)-(28)
        d_min, rho_p, rho_t = 0.3, 0.05, 0.02
        c = scene.mpc_coeffs_host(poses[idx], d_min, rho_p, rho_t)
        want = O.mpc_coeffs(ref.value, ref.grad, footprint, d_min, rho_p, rho_t)
        fin = np.isfinite(ref.value)
        # 1e-5 m + 4 ulp_fp32: these scenes reach |h - gamma| of tens of metres (reading G16)
        assert (np.abs(c[fin, 0] - want[fin, 0]) <= 1e-5 + 4 * np.abs(want[fin, 0]) * 2.0 ** -23).all(), tag
        assert np.isposinf(c[~fin, 0]).all() and (c[~fin, 1:] == 0).all(), tag
        compare(_Ref(ref, slice(None), sign=-1.0), vh, c[:, 1:], what=tag + " J_g")
        # time-varying row windows: pose n sees rows [w0, w1)
        w0 = rng.integers(0, Mrows, N)
        w1 = np.minimum(w0 + rng.integers(0, Mrows + 1, N), Mrows)
        win = np.stack([w0, w1], 1).astype(np.int32)
        vw, gw = scene.eval_windows(p, torch.from_numpy(win).cuda(), grad=True)
        vwh, gwh = scene.eval_windows_host(poses, win, grad=True)
        assert np.array_equal(vw.cpu().numpy(), vwh) and np.array_equal(gw.cpu().numpy(), gwh), tag
        for q, n in enumerate(idx[:30]):
            seg = ref.per_obstacle[q, w0[n]:w1[n]]
            want = seg.min() if seg.size and np.isfinite(seg).any() else np.inf
            got = float(vw[n])
            assert (np.isinf(want) and np.isinf(got)) or abs(got - want) <= 1e-5 + 4 * abs(want) * 2.0 ** -23, (tag, n)
        # NEXT-4 fused: random non-decreasing component map (rows in groups of 1..4), trajectories of a
        # random length that divides N
        sizes = []
        while sum(sizes) < Mrows:
            sizes.append(int(rng.integers(1, 5)))
        ids = np.repeat(np.arange(len(sizes)), sizes)[:Mrows].astype(np.int32)
        n_obs = min(int(ids.max()) + 1 + int(rng.integers(0, 2)), Mrows)      # (n_obstacles <= M)
        scene.set_components(ids, n_obs)
        vf_, gf_, pof = scene.eval(p, grad=True, per_obstacle=True)
        assert torch.equal(vf_, v) and torch.equal(gf_, g), tag + " components: value/grad"
        assert torch.equal(pof, psdf.psdf_component_min(po, torch.from_numpy(ids).cuda(), n_obs)), tag + " components: fused == stand-alone"
        want = O.component_min(ref.per_obstacle, ids, n_obs)
        got = pof.cpu().numpy().astype(np.float64)[idx]
        assert np.array_equal(np.isposinf(got), np.isposinf(want)), tag
        fin2 = np.isfinite(want)
        assert (np.abs(got[fin2] - want[fin2]) <= 1e-5 + 4 * np.abs(want[fin2]) * 2.0 ** -23).all(), tag + " components vs oracle"
        _, _, pofh = scene.eval_host(poses[idx], grad=True, per_obstacle=True)
        assert np.array_equal(pofh, pof.cpu().numpy()[idx]), tag + " components: host path"
        scene.set_components(None, 0)
        divs = [h for h in (1, 2, 3, 5, 7, 10, 30, 60, 100, 600) if N % h == 0]
        H = int(rng.choice(divs))
        vt, gt, mn, am, pen = scene.eval_trajectories(p, N // H, H, 0.4, grad=True)
        mn0, am0, pen0 = psdf.psdf_trajectory_reduce(v, N // H, H, 0.4)
        assert torch.equal(vt, v) and torch.equal(gt, g), tag + " trajectories: value/grad"
        assert torch.equal(mn, mn0) and torch.equal(am, am0) and torch.equal(pen, pen0), tag + f" trajectories H={H}"
        # update to shifted obstacles == fresh scene; device-resident update back == original
        sh = np.array([0.5, -0.25], np.float32)
        fresh = psdf.Scene(footprint, A + sh, B + sh, S, max_poses=max(N, 8))
        vf, gf, _ = fresh.eval(p, grad=True)
        scene.update(A + sh, B + sh, S)
        vu, gu, _ = scene.eval(p, grad=True)
        assert torch.equal(vu, vf) and torch.equal(gu, gf), tag + " host update"
        scene.update(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), torch.from_numpy(S).cuda())
        vu, gu, _ = scene.eval(p, grad=True)
        assert torch.equal(vu, v) and torch.equal(gu, g), tag + " device update"
        fresh.close()
        scene.close()


@pytest.mark.parametrize("seed", [902050 + 7 * k for k in range(_N_CULLED)])
def test_random_scenes_culled_equals_dense(env, seed):
    torch, O, psdf, W = env
    from tests.test_gpu_parity import _random_scene
    footprint, A, B, S, poses, info = _random_scene(seed)
    poses[11 % len(poses), 0] = np.nan
    try:
        scene = psdf.Scene(footprint, A, B, S, max_poses=len(poses))
    except psdf.PsdfError:
        pytest.skip("fp32 rounding at this offset made an obstacle degenerate")
    p = torch.from_numpy(poses).cuda()
    v, g, _ = scene.eval(p, grad=True)
    scene.set_culling(True)
    v1, g1, _ = scene.eval(p, grad=True)
    v2, _, _ = scene.eval(p, grad=False)
    torch.cuda.synchronize()
    same = lambda a, b: bool(((a == b) | (torch.isnan(a) & torch.isnan(b))).all())
    assert same(v1, v) and same(g1, g) and same(v2, v), info
    scene.close()
