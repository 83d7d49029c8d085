"""NEXT-4 reductions fused into the evaluation launch:
psdf_set_components folds convex components into per-obstacle values inside the kernels (no [N,M]
array), psdf_eval_trajectories reduces every trajectory in the launch that evaluates it.  Checked
against the oracle's plain definitions and bit for bit against the stand-alone kernels.
Need a B200: `pytest -m gpu`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf, workloads as W
    assert torch.cuda.is_available()
    return torch, O, psdf, W


def _check_components(torch, O, psdf, scene, w, S, ids, n_obs, poses, tag):
    """fused [N,n_obs] == stand-alone fold of the unfused [N,M] (bits) == oracle definition (1e-5 + 4 ulp)."""
    p = torch.from_numpy(poses).cuda()
    scene.set_components(None, 0)
    v0, g0, pc = scene.eval(p, grad=True, per_obstacle=True)
    assert pc.shape == (len(poses), w.M)
    want_bits = psdf.psdf_component_min(pc, torch.from_numpy(ids).cuda(), n_obs)
    scene.set_components(ids, n_obs)
    v1, g1, po = scene.eval(p, grad=True, per_obstacle=True)
    torch.cuda.synchronize()
    assert po.shape == (len(poses), n_obs), tag
    assert torch.equal(po, want_bits), tag
    assert torch.equal(v1, v0) and torch.equal(g1, g0), tag            # eq.(6): phi is the min over all components anyway
    assert torch.equal(po.min(dim=1).values, v1), tag
    ref = O.evaluate(w.footprint, w.A, w.B, S, poses[:300], per_obstacle=True)
    want = O.component_min(ref.per_obstacle, ids, n_obs)
    got = po.cpu().numpy().astype(np.float64)[:300]
    assert np.array_equal(np.isposinf(got), np.isposinf(want)), tag
    fin = np.isfinite(want)
    assert (np.abs(got[fin] - want[fin]) <= 1e-5 + 4 * np.abs(want[fin]) * 2.0 ** -23).all(), tag
    # host path, same bits (zero-copy launch for small batches, branched graph for large ones)
    vh, gh, poh = scene.eval_host(poses, grad=True, per_obstacle=True)
    assert np.array_equal(poh, po.cpu().numpy()) and np.array_equal(vh, v1.cpu().numpy()), tag
    return po


def test_components_fused_into_the_evaluation(env):
    torch, O, psdf, W = env
    # (1) MPC-sized: config 2, rows grouped three at a time; a group with no valid row, a trailing
    #     obstacle without components, single empty rows inside groups      -> lane-split kernel
    w = W.make_config(2)
    S = w.S.copy()
    S[6:9] = 0                                   # obstacle 2 has no valid component
    S[13] = 0
    S[w.M - 1] = 0
    ids = (np.arange(w.M) // 3).astype(np.int32)
    n_obs = int(ids.max()) + 2
    scene = psdf.Scene(w.footprint, w.A, w.B, S, max_poses=4096)
    po = _check_components(torch, O, psdf, scene, w, S, ids, n_obs, w.poses, "cfg2 lanes")
    assert torch.isposinf(po[:, 2]).all() and torch.isposinf(po[:, -1]).all()
    # more poses on the same scene: still the lane-split kernel, several poses per CTA
    rng = np.random.default_rng(5)
    many = np.column_stack([rng.uniform(0, 20, 1500), rng.uniform(0, 20, 1500), rng.uniform(-3, 3, 1500)]).astype(np.float32)
    _check_components(torch, O, psdf, scene, w, S, ids, n_obs, many, "cfg2 lanes, 1500 poses")
    # perception update (device tensors) with other rows emptied: tables follow
    S2 = w.S.copy()
    S2[0:3] = 0
    S2[20] = 0
    scene.update(torch.from_numpy(w.A).cuda(), torch.from_numpy(w.B).cuda(), torch.from_numpy(S2).cuda())
    po2 = _check_components(torch, O, psdf, scene, w, S2, ids, n_obs, w.poses, "cfg2 after device update")
    assert torch.isposinf(po2[:, 0]).all() and not torch.isposinf(po2[:, 2]).any()
    # invalid maps
    for bad in (ids[::-1].copy(), np.where(ids == 3, n_obs, ids).astype(np.int32), -np.ones(w.M, np.int32)):
        with pytest.raises(psdf.PsdfError) as e:
            scene.set_components(bad, n_obs)
        assert e.value.status == psdf.PSDF_ERR_INVALID_ARG
    scene.close()
    # (2) large batch: config 3 (256 rows in groups of 1..7), tile-scan kernel with chunked obstacle
    #     ranges (chunks must end between obstacles) and the branched host graph
    w = W.make_config(3).subsample(9000)
    rng = np.random.default_rng(6)
    sizes = []
    while sum(sizes) < w.M:
        sizes.append(int(rng.integers(1, 8)))
    ids = np.repeat(np.arange(len(sizes)), sizes)[:w.M].astype(np.int32)
    n_obs = int(ids.max()) + 1
    S = w.S.copy()
    S[ids == 5] = 0
    S[ids == n_obs - 1] = 0
    for host_scene in (True, False):
        if host_scene:
            scene = psdf.Scene(w.footprint, w.A, w.B, S, max_poses=w.N)
        else:
            scene = psdf.Scene(w.footprint, torch.from_numpy(w.A).cuda(), torch.from_numpy(w.B).cuda(),
                               torch.from_numpy(S).cuda(), max_poses=w.N)
        po = _check_components(torch, O, psdf, scene, w, S, ids, n_obs, w.poses, f"cfg3 scan host_scene={host_scene}")
        assert torch.isposinf(po[:, 5]).all() and torch.isposinf(po[:, n_obs - 1]).all()
        scene.close()
    # (3) one obstacle made of every row, and every row its own obstacle
    w = W.make_config(2)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    _check_components(torch, O, psdf, scene, w, w.S, np.zeros(w.M, np.int32), 1, w.poses, "one obstacle")
    _check_components(torch, O, psdf, scene, w, w.S, np.arange(w.M, dtype=np.int32), w.M, w.poses, "identity map")
    scene.close()


@pytest.mark.parametrize("case", ["scan", "scan_value_only", "lanes", "culled", "ragged"])
def test_trajectory_reductions_fused_into_the_evaluation(env, case):
    torch, O, psdf, W = env
    if case in ("scan", "scan_value_only", "culled"):
        w = W.make_config(3, n_traj=300)                    # 15 000 poses, H = 50: tiles of 64 poses straddle trajectories
        T, H = 300, 50
    elif case == "lanes":
        w = W.make_config(2)                                # 50 poses = 5 trajectories of 10 stages, lane-split kernel
        T, H = 5, 10
    else:
        w = W.make_config(3, n_traj=300).subsample(7 * 333) # H = 333 > tile, odd sizes
        T, H = 7, 333
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    scene.set_culling(case == "culled")
    p = torch.from_numpy(w.poses).cuda()
    d_safe = 0.5
    grad = case != "scan_value_only"
    for rep in range(3):                                    # the arrival counters are left clean
        v, g, mn, am, pen = scene.eval_trajectories(p, T, H, d_safe, grad=grad)
        v0, g0, _ = scene.eval(p, grad=grad)
        mn0, am0, pen0 = psdf.psdf_trajectory_reduce(v0, T, H, d_safe)
        torch.cuda.synchronize()
        assert torch.equal(v, v0) and (not grad or torch.equal(g, g0)), (case, rep)
        assert torch.equal(mn, mn0) and torch.equal(am, am0) and torch.equal(pen, pen0), (case, rep)
    # against the oracle's plain definitions, end to end
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    omn, oam, open_ = O.trajectory_reduce(ref.value, T, H, d_safe)
    assert np.abs(mn.cpu().numpy() - omn).max() <= 1e-5
    assert np.abs(pen.cpu().numpy() - open_).max() <= 1e-4 * max(1.0, open_.max())
    rmn, ram, _ = O.trajectory_reduce(v.cpu().numpy(), T, H, d_safe)      # definitions on the GPU's own fp32 values
    assert np.array_equal(mn.cpu().numpy().astype(np.float64), rmn) and np.array_equal(am.cpu().numpy(), ram)
    assert (open_ > 0).any()
    scene.close()
