"""Parity tests proper: CUDA path (through the C ABI) vs the oracle, element by element,
on the five BASELINE configs.  Need a B200: `pytest -m gpu`."""
import numpy as np
import pytest

from tests.parity import compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf
    assert torch.cuda.is_available()
    return torch, O, psdf


def _gpu_eval(torch, psdf, w, grad=True, per_obstacle=False, poses=None):
    poses = w.poses if poses is None else poses
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=max(len(poses), 1))
    p = torch.from_numpy(np.ascontiguousarray(poses)).cuda()
    v, g, po = scene.eval(p, grad=grad, per_obstacle=per_obstacle)
    torch.cuda.synchronize()
    out = (v.cpu().numpy(), None if g is None else g.cpu().numpy(), None if po is None else po.cpu().numpy())
    return scene, out


def _oracle(O, w, poses=None, per_obstacle=False):
    return O.evaluate(w.footprint, w.A, w.B, w.S, w.poses if poses is None else poses,
                      per_obstacle=per_obstacle)


@pytest.mark.parametrize("cfg", [1, 2])
def test_small_configs_device_and_host_paths(env, workloads_cache, cfg):
    torch, O, psdf = env
    w = workloads_cache(cfg)
    ref = _oracle(O, w, per_obstacle=True)
    scene, (v, g, po) = _gpu_eval(torch, psdf, w, grad=True, per_obstacle=True)
    st = compare(ref, v, g, po, what=w.name, per_obstacle_plain_tol=True)     # plain 1e-5 m per obstacle
    print(w.name, st)
    assert st["grad_compared"] > 0.5
    # host (CUDA graph) path, twice (capture, then replay), all output combinations
    for _ in range(2):
        v2, g2, po2 = scene.eval_host(w.poses, grad=True, per_obstacle=True)
        assert np.array_equal(v2, v) and np.array_equal(g2, g) and np.array_equal(po2, po)
    # pre-marshalled calls: same results, buffers rewritten in place
    vb, gb = np.zeros(w.N, np.float32), np.zeros((w.N, 3), np.float32)
    pb = w.poses.copy()
    call = scene.bind_eval_host(pb, vb, gb)
    call()
    assert np.array_equal(vb, v) and np.array_equal(gb, g)
    pb[:] = w.poses[::-1]
    call()
    assert np.array_equal(vb, v[::-1]) and np.array_equal(gb, g[::-1])
    cb = np.zeros((w.N, 4), np.float32)
    scene.bind_mpc_coeffs_host(pb, cb, 0.3, 0.05, 0.05)()
    assert np.array_equal(cb, scene.mpc_coeffs_host(pb, 0.3, 0.05, 0.05))
    v3, g3, po3 = scene.eval_host(w.poses, grad=False)
    assert g3 is None and po3 is None
    compare(ref, v3, what=w.name + " value-only host")
    # value-only device path gives the same value
    v4, _, _ = scene.eval(torch.from_numpy(w.poses).cuda(), grad=False)
    compare(ref, v4.cpu().numpy(), what=w.name + " value-only")
    scene.close()


@pytest.mark.parametrize("cfg,n", [(3, 5003), (4, 3001), (5, 2501)])
def test_scan_kernel_subsampled(env, workloads_cache, cfg, n):
    """Sizes the oracle finishes in seconds, several pose tiles, ragged tail, chunked
    obstacle ranges with the cross-chunk arg-min."""
    torch, O, psdf = env
    w = workloads_cache(cfg).subsample(n)
    ref = _oracle(O, w)
    scene, (v, g, _) = _gpu_eval(torch, psdf, w, grad=True)
    st = compare(ref, v, g, what=w.name)
    print(w.name, st, "penetrating frac", float((ref.value < 0).mean()))
    assert st["grad_compared"] > 0.5
    p = torch.from_numpy(w.poses).cuda()
    v0, _, _ = scene.eval(p, grad=False)                 # value-only variant
    compare(ref, v0.cpu().numpy(), what=w.name + " value-only")
    v1, g1, _ = scene.eval(p, grad=True)                 # workspace left clean: same answer again
    assert np.array_equal(v1.cpu().numpy(), v) and np.array_equal(g1.cpu().numpy(), g)
    scene.close()


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_sampled(env, workloads_cache, cfg):
    """BASELINE full sizes in the launch configuration bench.py times; the oracle checks
    a random sample of the outputs one by one."""
    torch, O, psdf = env
    w = workloads_cache(cfg)
    scene, (v, g, _) = _gpu_eval(torch, psdf, w, grad=True)
    rng = np.random.default_rng(99 + cfg)
    idx = np.sort(rng.choice(w.N, size={3: 4000, 4: 1500, 5: 1200}[cfg], replace=False))
    ref = _oracle(O, w, poses=w.poses[idx])
    st = compare(ref, v[idx], g[idx], what=w.name + " full")
    print(w.name, "full", st)
    # property that holds at any size: |grad_p| = 1 wherever finite and away from contact
    gn = np.hypot(g[:, 0], g[:, 1])
    far = np.abs(v) > 1e-3
    assert np.abs(gn[far] - 1.0).max() < 1e-4
    v0, _, _ = scene.eval(torch.from_numpy(w.poses).cuda(), grad=False)
    assert np.array_equal(v0.cpu().numpy(), v)
    scene.close()


def test_per_obstacle_large_batch(env, workloads_cache):
    torch, O, psdf = env
    w = workloads_cache(3).subsample(3000)
    ref = _oracle(O, w, per_obstacle=True)
    scene, (v, g, po) = _gpu_eval(torch, psdf, w, grad=True, per_obstacle=True)
    print(compare(ref, v, g, po, what="per-obstacle scan path"))
    assert np.array_equal(po.min(axis=1), v)
    scene.close()


@pytest.mark.parametrize("cfg,n", [(3, None), (4, None), (5, None), (5, 4099), (2, None)])
def test_culled_path_bit_identical_to_dense(env, workloads_cache, cfg, n):
    """psdf_set_culling (exact broad-phase culling, NEXT-3): same value and gradient bits as
    the dense path at BASELINE full sizes and on a ragged size; unique results, so compared
    exactly.  cfg 2 is below the culled path's size threshold: the switch must be inert."""
    torch, O, psdf = env
    w = workloads_cache(cfg)
    if n is not None:
        w = w.subsample(n)
    scene, (v, g, _) = _gpu_eval(torch, psdf, w, grad=True)
    p = torch.from_numpy(w.poses).cuda()
    scene.set_culling(True)
    for with_grad in (True, False):
        v1, g1, _ = scene.eval(p, grad=with_grad)
        torch.cuda.synchronize()
        assert np.array_equal(v1.cpu().numpy(), v)
        if with_grad:
            assert np.array_equal(g1.cpu().numpy(), g)
    # non-finite poses and a second call (workspace left clean)
    q = w.poses.copy()
    q[7, 0] = np.nan
    q[w.N // 2, 2] = np.inf
    v2, g2, _ = scene.eval(torch.from_numpy(q).cuda(), grad=True)
    v2, g2 = v2.cpu().numpy(), g2.cpu().numpy()
    bad = np.zeros(w.N, bool)
    bad[[7, w.N // 2]] = True
    assert np.isnan(v2[bad]).all() and np.array_equal(v2[~bad], v[~bad]) and np.array_equal(g2[~bad], g[~bad])
    if cfg == 5 and n is not None:
        # per-stage coefficients through the host path with culling on
        c = scene.mpc_coeffs_host(w.poses, 0.01, 0.1, 0.1)
        assert np.array_equal(c[:, 1:], -g)
    scene.set_culling(False)
    v3, _, _ = scene.eval(p, grad=False)
    assert np.array_equal(v3.cpu().numpy(), v)
    scene.close()


@pytest.mark.parametrize("cfg,n", [(5, 1), (5, 7), (4, 33), (5, 100), (3, 3)])
def test_few_poses_many_obstacles(env, workloads_cache, cfg, n):
    """Lane-split kernel with more than one warp (K > 32) and more than one CTA (C > 1) per
    pose: a handful of poses against up to 4096 obstacles, all outputs, twice (the cross-CTA
    workspace must be left clean), device and host paths."""
    torch, O, psdf = env
    w = workloads_cache(cfg)
    rng = np.random.default_rng(1000 * cfg + n)
    poses = w.poses[np.sort(rng.choice(w.N, n, replace=False))]
    ref = _oracle(O, w, poses=poses, per_obstacle=True)
    scene, (v, g, po) = _gpu_eval(torch, psdf, w, grad=True, per_obstacle=True, poses=poses)
    print(w.name, n, compare(ref, v, g, po, what=f"{w.name} n={n}"))
    p = torch.from_numpy(poses).cuda()
    v1, g1, _ = scene.eval(p, grad=True)
    assert np.array_equal(v1.cpu().numpy(), v) and np.array_equal(g1.cpu().numpy(), g)
    v2, _, _ = scene.eval(p, grad=False)
    assert np.array_equal(v2.cpu().numpy(), v)
    vh, gh, poh = scene.eval_host(poses, grad=True, per_obstacle=True)
    assert np.array_equal(vh, v) and np.array_equal(gh, g) and np.array_equal(poh, po)
    scene.close()


@pytest.mark.parametrize("n_poses,V", [(4500, 4), (40000, 6), (6000, 16)])
def test_culled_path_stress_cases(env, n_poses, V):
    """Culled path where its machinery is stressed: 600 near-duplicates of four overlapping
    obstacles (no bound can separate them: hundreds of candidate pairs per pose, so the
    shared-memory pair queue overflows and the walk resumes), poses far outside the obstacle grid, both CTA shapes (N below / above 32768), the
    smaller queue of 16-vertex footprints, a device-encoded scene, and a scene update (grid
    rebuilt).  Unique results: bit-identical to the dense path."""
    torch, O, psdf = env
    from paper_2607_04310_b200 import workloads as W
    rng = np.random.default_rng(4310 + n_poses)
    polys = []
    base = [(W.convex_kgon(rng, int(rng.integers(3, 9)), float(rng.uniform(0.6, 1.2))), rng.uniform(-1.0, 1.0, 2),
             float(rng.uniform(-np.pi, np.pi))) for _ in range(4)]
    for i in range(700):
        if i < 600:
            poly, centre, yaw = base[i % 4]
            polys.append(W.place(poly, centre + rng.uniform(-1e-3, 1e-3, 2), yaw))
        else:
            polys.append(W.place(W.convex_kgon(rng, int(rng.integers(3, 9)), float(rng.uniform(0.3, 1.2))),
                                 rng.uniform(-60, 60, 2), float(rng.uniform(-np.pi, np.pi))))
    A, B, S = W.pad_scene(rng, polys, 8, extra_rows=3)
    ang = np.linspace(0, 2 * np.pi, V, endpoint=False) + 0.1
    footprint = np.stack([0.7 * np.cos(ang), 0.35 * np.sin(ang)], 1).astype(np.float32)
    poses = np.empty((n_poses, 3), np.float32)
    poses[:, :2] = rng.uniform(-14, 14, (n_poses, 2))          # ring around the cluster: ub ~ distance to it
    poses[::7, :2] = rng.uniform(-2.5, 2.5, (len(poses[::7]), 2))   # inside the cluster (penetrating)
    poses[::31, :2] = rng.uniform(-80, 80, (len(poses[::31]), 2))
    poses[5, :2] = (1.0e4, -3.0e4)                              # far outside the obstacle grid
    poses[:, 2] = rng.uniform(-np.pi, np.pi, n_poses)
    p = torch.from_numpy(poses).cuda()

    def both(scene):
        scene.set_culling(False)
        v, g, _ = scene.eval(p, grad=True)
        scene.set_culling(True)
        scene.cull_stats()
        v1, g1, _ = scene.eval(p, grad=True)
        v2, _, _ = scene.eval(p, grad=False)
        torch.cuda.synchronize()
        pairs, edge_steps = scene.cull_stats()
        assert torch.equal(v1, v) and torch.equal(g1, g) and torch.equal(v2, v)
        return v.cpu().numpy(), pairs / 2.0 / n_poses

    scene = psdf.Scene(footprint, A, B, S, max_poses=n_poses)
    v, per_pose = both(scene)
    print(f"N={n_poses} V={V}: evaluated pairs per pose {per_pose:.1f}, penetrating {float((v < 0).mean()):.2f}")
    assert per_pose > 16.0                                      # the queue (16 or 8 entries per pose) did overflow
    # a sample against the oracle
    idx = np.sort(rng.choice(n_poses, 300, replace=False))
    idx = idx[idx != 5]                                         # fp32 cannot hold 1e-5 m at 3e4 m from the origin
    ref = O.evaluate(footprint, A, B, S, poses[idx])
    compare(ref, v[idx], what="culled stress")
    # scene update (values only): obstacles shifted, grid rebuilt
    shift = np.array([3.0, -2.0], np.float32)
    scene.update(A + shift, B + shift, S)
    both(scene)
    scene.close()
    # device-encoded scene
    s2 = psdf.Scene(footprint, torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), torch.from_numpy(S).cuda(),
                    max_poses=n_poses)
    v_dev, _ = both(s2)
    assert np.array_equal(v_dev, v)
    s2.close()


def test_culled_path_degenerate_grid(env):
    """All obstacle centres coincide (nested polygons): the obstacle grid has zero extent, every
    obstacle lands in one cell and the seed rectangle has to double ~30 times.  Still exact."""
    torch, O, psdf = env
    from paper_2607_04310_b200 import workloads as W
    rng = np.random.default_rng(77)
    base = W.rectangle(1.0, 1.0)
    polys = [W.place(base * (0.2 + 0.02 * i), (5.0, -3.0), 0.0) for i in range(80)]
    A, B, S = W.pad_scene(rng, polys, 6)
    footprint = W.rectangle(0.6, 0.4).astype(np.float32)
    n = 3000
    poses = np.column_stack([rng.uniform(-10, 20, n), rng.uniform(-18, 12, n), rng.uniform(-np.pi, np.pi, n)]).astype(np.float32)
    p = torch.from_numpy(poses).cuda()
    scene = psdf.Scene(footprint, A, B, S, max_poses=n)
    v, g, _ = scene.eval(p, grad=True)
    scene.set_culling(True)
    v1, g1, _ = scene.eval(p, grad=True)
    torch.cuda.synchronize()
    assert torch.equal(v1, v) and torch.equal(g1, g)
    ref = O.evaluate(footprint, A, B, S, poses[:400])
    compare(ref, v.cpu().numpy()[:400], what="nested obstacles")
    scene.close()


def _random_scene(seed):
    """One case of the randomised culled-vs-dense differential run (same draw order)."""
    from paper_2607_04310_b200 import workloads as W
    rng = np.random.default_rng(seed)
    V = int(rng.integers(3, 17))
    M = int(rng.choice([64, 70, 200, 700, 2500]))
    arena = float(rng.choice([3.0, 30.0, 300.0, 3000.0]))
    off = float(rng.choice([0.0, 0.0, 1000.0, -20000.0]))
    E = int(rng.choice([6, 8, 12, 16]))
    rmax = float(rng.choice([0.3, 1.5, 6.0]))
    polys = []
    for _ in range(M):
        if rng.random() < 0.4:
            poly = W.rectangle(float(rng.uniform(0.3, 3) * rmax), float(rng.uniform(0.1, 1) * rmax))
        else:
            rad = float(rng.uniform(0.5, 1.0) * rmax)
            poly = W.convex_kgon(rng, int(rng.integers(3, min(E, 3 + int(rad * 8)) + 1)), rad)
        polys.append(W.place(poly, rng.uniform(0, arena, 2) + off, float(rng.uniform(-np.pi, np.pi))))
    A, B, S = W.pad_scene(rng, polys, E, extra_rows=int(rng.integers(0, 3)))
    ang = np.sort(rng.uniform(0, 2 * np.pi, V))
    ang += np.linspace(0, 1e-3, V)
    gaps = np.diff(np.concatenate([ang, [ang[0] + 2 * np.pi]]))
    if gaps.min() < 0.15 or gaps.max() > 3.0:
        ang = np.linspace(0, 2 * np.pi, V, endpoint=False) + 0.05
    fr = float(rng.choice([0.2, 1.0, 4.0]))
    footprint = (np.stack([fr * np.cos(ang), 0.5 * fr * np.sin(ang)], 1) + rng.uniform(-0.5, 0.5, 2) * fr).astype(np.float32)
    N = int(rng.choice([2049, 5000, 33000, 70000]))
    poses = np.empty((N, 3), np.float32)
    poses[:, :2] = rng.uniform(-0.3 * arena, 1.3 * arena, (N, 2)) + off
    poses[:, 2] = rng.uniform(-7, 7, N)
    return footprint, A, B, S, poses, dict(V=V, M=M, arena=arena, off=off, N=N)


@pytest.mark.parametrize("seed", [902050, 900010, 900002])
def test_culled_path_far_from_the_origin(env, seed):
    """Scenes 2e4 m from the origin, where one fp32 ulp of a coordinate is 2 mm: the culling
    bounds must carry a safety term that grows with the coordinates.  A randomised differential
    run (2839 scenes) found 5, all at this offset, where a fixed 1e-4 m pad dropped the winner;
    seed 902050 is one of them (2500 obstacles crowded into 3 x 3 m, 70 000 poses)."""
    torch, O, psdf = env
    footprint, A, B, S, poses, info = _random_scene(seed)
    assert info["off"] == -20000.0
    scene = psdf.Scene(footprint, A, B, S, max_poses=len(poses))
    p = torch.from_numpy(poses).cuda()
    v, g, _ = scene.eval(p, grad=True)
    scene.set_culling(True)
    v1, g1, _ = scene.eval(p, grad=True)
    torch.cuda.synchronize()
    assert torch.equal(v1, v) and torch.equal(g1, g), info
    scene.close()
