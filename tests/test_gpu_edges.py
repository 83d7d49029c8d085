"""Edge cases of the C ABI on the GPU: empty / ragged inputs, masks, footprint sizes,
orientation, updates, capacity, NaN poses, MPC coefficients."""
import math

import numpy as np
import pytest

from tests.parity import compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf, workloads as W
    assert torch.cuda.is_available()
    return torch, O, psdf, W


def _run(torch, scene, poses, **kw):
    v, g, po = scene.eval(torch.from_numpy(np.ascontiguousarray(poses, np.float32)).cuda(), **kw)
    torch.cuda.synchronize()
    return v.cpu().numpy(), None if g is None else g.cpu().numpy(), None if po is None else po.cpu().numpy()


@pytest.mark.parametrize("V", [3, 5, 6, 7, 8, 9, 11, 13, 16])
def test_footprint_vertex_counts(env, V):
    """Rectangle, triangle, pentagon ... by changing only V0; V without a
    compiled instance is padded with collinear midpoints."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(100 + V)
    fp = W.convex_kgon(rng, V, 0.6).astype(np.float32)
    w = W.make_config(2)
    poses = np.stack([rng.uniform(0, 20, 600), rng.uniform(0, 20, 600), rng.uniform(-7, 7, 600)], 1).astype(np.float32)
    ref = O.evaluate(fp, w.A, w.B, w.S, poses, per_obstacle=True)
    scene = psdf.Scene(fp, w.A, w.B, w.S, max_poses=600)
    v, g, po = _run(torch, scene, poses, grad=True, per_obstacle=True)
    print(V, compare(ref, v, g, po, what=f"V={V}"))
    scene.close()


@pytest.mark.parametrize("V", [4, 8, 12, 16])
def test_symmetric_footprints_take_the_mirrored_edge_step(env, V):
    """Footprints that are centrally symmetric about the reference point (v_{l+V/2} == -v_l bitwise) are
    evaluated by edge_step2_sym (half of the dot products derived from the other half); the same outline
    with the reference point moved is not.  Both against the oracle, through the lane-split, the
    tile-scan (chunked) and the culled kernel, which must agree bit for bit with each other."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(300 + V)
    ang = np.sort(rng.uniform(0.05, np.pi - 0.05, V // 2))            # half of a convex outline, then its mirror image
    half = np.stack([0.8 * np.cos(ang), 0.45 * np.sin(ang)], 1).astype(np.float32)
    fp_sym = np.concatenate([half, -half]).astype(np.float32)
    fp_off = (fp_sym + np.float32(0.0625)).astype(np.float32)          # same outline, reference point moved
    w = W.make_config(3).subsample(6000)
    for fp, want_sym in ((fp_sym, True), (fp_off, False)):
        scene = psdf.Scene(fp, w.A, w.B, w.S, max_poses=w.N)
        assert scene.footprint_symmetric == want_sym
        ref = O.evaluate(fp, w.A, w.B, w.S, w.poses[:1500], per_obstacle=False)
        v, g, _ = _run(torch, scene, w.poses, grad=True)                # tile-scan kernel, chunked
        print(V, want_sym, compare(ref, v[:1500], g[:1500], what=f"V={V} sym={want_sym} scan"))
        vl, gl, pol = _run(torch, scene, w.poses[:100], grad=True, per_obstacle=True)   # lane-split kernel
        assert np.array_equal(vl, v[:100]) and np.array_equal(gl, g[:100])
        refp = O.evaluate(fp, w.A, w.B, w.S, w.poses[:100], per_obstacle=True)
        compare(refp, vl, gl, pol, what=f"V={V} sym={want_sym} lanes")
        scene.set_culling(True)
        vc, gc, _ = _run(torch, scene, w.poses, grad=True)              # culled kernel
        assert np.array_equal(vc, v) and np.array_equal(gc, g)
        vh, gh, _ = scene.eval_host(w.poses[:40], grad=True)            # MPC host path
        assert np.array_equal(vh, v[:40]) and np.array_equal(gh, g[:40])
        scene.close()


def test_empty_and_degenerate_inputs(env):
    torch, O, psdf, W = env
    w = W.make_config(2)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=64)
    # N = 0 is a no-op
    v, g, _ = scene.eval(torch.empty((0, 3), dtype=torch.float32, device="cuda"))
    assert v.numel() == 0 and g.numel() == 0
    # N = 1
    v, g, po = _run(torch, scene, w.poses[:1], grad=True, per_obstacle=True)
    compare(O.evaluate(w.footprint, w.A, w.B, w.S, w.poses[:1], per_obstacle=True), v, g, po)
    # capacity
    with pytest.raises(psdf.PsdfError) as e:
        scene.eval(torch.zeros((65, 3), dtype=torch.float32, device="cuda"))
    assert e.value.status == psdf.PSDF_ERR_CAPACITY
    # non-finite pose: NaN outputs, neighbours unaffected
    poses = w.poses[:8].copy()
    poses[3, 0] = np.nan
    poses[5, 2] = np.inf
    v, g, _ = _run(torch, scene, poses, grad=True)
    assert np.isnan(v[[3, 5]]).all() and np.isnan(g[[3, 5]]).all()
    keep = [0, 1, 2, 4, 6, 7]
    compare(O.evaluate(w.footprint, w.A, w.B, w.S, poses[keep]), v[keep], g[keep])
    # no valid obstacle at all: +inf, zero gradient, +inf per obstacle
    scene.update(w.A, w.B, np.zeros_like(w.S))
    v, g, po = _run(torch, scene, w.poses[:10], grad=True, per_obstacle=True)
    assert np.isposinf(v).all() and (g == 0).all() and np.isposinf(po).all()
    assert scene.num_obstacles == 0 and scene.num_edges == 0
    # degenerate update is rejected and leaves the scene in force
    S_bad = w.S.copy()
    S_bad[0, np.nonzero(S_bad[0])[0][0]] = 0
    with pytest.raises(psdf.PsdfError) as e:
        scene.update(w.A, w.B, S_bad)
    assert e.value.status == psdf.PSDF_ERR_DEGENERATE
    v, _, _ = _run(torch, scene, w.poses[:10], grad=False)
    assert np.isposinf(v).all()
    scene.close()


def test_masks_padding_orientation_update(env):
    torch, O, psdf, W = env
    w = W.make_config(2)
    rng = np.random.default_rng(8)
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses, per_obstacle=True)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    base = _run(torch, scene, w.poses, grad=True, per_obstacle=True)
    # garbage in padded slots, extra masked rows and wider E are inert (bit-identical)
    A, B = w.A.copy(), w.B.copy()
    pad = w.S == 0
    A[pad] = rng.uniform(-1e3, 1e3, (pad.sum(), 2)).astype(np.float32)
    B[pad] = rng.uniform(-1e3, 1e3, (pad.sum(), 2)).astype(np.float32)
    scene.update(A, B, w.S)
    again = _run(torch, scene, w.poses, grad=True, per_obstacle=True)
    for a, b in zip(base, again):
        assert np.array_equal(a, b)
    A2 = np.concatenate([np.concatenate([w.A, rng.uniform(0, 20, (w.M, 3, 2)).astype(np.float32)], 1),
                         rng.uniform(0, 20, (5, w.E + 3, 2)).astype(np.float32)])
    B2 = np.concatenate([np.concatenate([w.B, rng.uniform(0, 20, (w.M, 3, 2)).astype(np.float32)], 1),
                         rng.uniform(0, 20, (5, w.E + 3, 2)).astype(np.float32)])
    S2 = np.concatenate([np.concatenate([w.S, np.zeros((w.M, 3), np.uint8)], 1),
                         np.zeros((5, w.E + 3), np.uint8)])
    s2 = psdf.Scene(w.footprint, A2, B2, S2, max_poses=w.N)
    v, g, po = _run(torch, s2, w.poses, grad=True, per_obstacle=True)
    assert np.array_equal(v, base[0]) and np.array_equal(g, base[1])
    assert np.array_equal(po[:, :w.M], base[2]) and np.isposinf(po[:, w.M:]).all()
    s2.close()
    # clockwise obstacle rows give the same values (reading G8)
    A3, B3 = w.A.copy(), w.B.copy()
    for i in range(0, w.M, 2):
        sl = np.nonzero(w.S[i])[0]
        A3[i, sl], B3[i, sl] = w.B[i, sl][::-1].copy(), w.A[i, sl][::-1].copy()
    s3 = psdf.Scene(w.footprint, A3, B3, w.S, max_poses=w.N)
    v, g, po = _run(torch, s3, w.poses, grad=True, per_obstacle=True)
    compare(ref, v, g, po, what="clockwise rows")
    s3.close()
    # device-resident scene tensors
    s4 = psdf.Scene(w.footprint, torch.from_numpy(w.A).cuda(), torch.from_numpy(w.B).cuda(),
                    torch.from_numpy(w.S).cuda(), max_poses=w.N)
    v, g, po = _run(torch, s4, w.poses, grad=True, per_obstacle=True)
    for a, b in zip(base, (v, g, po)):
        assert np.array_equal(a, b)
    s4.close()
    scene.close()


def test_mpc_coefficients(env):
    """[h_s - gamma_s ; J_g,s] of eqs.(26)-(28), N=15 stages, d_min=0.01
    (PAPER.md:301), against oracle.mpc_coeffs (eq.(27) literally, hand-pinned in
    tests/test_oracle_pins.py) at the stated 1e-5 m."""
    torch, O, psdf, W = env
    from tests.parity import grad_mask
    w = W.table1_case(100, 15)
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=64)
    d_min, v_max, w_max, dt = 0.01, 1.0, 1.0, 0.1
    rho_p, rho_t = v_max * dt, w_max * dt
    c = scene.mpc_coeffs_host(w.poses, d_min, rho_p, rho_t)
    want = O.mpc_coeffs(ref.value, ref.grad, w.footprint, d_min, rho_p, rho_t)
    assert np.abs(c[:, 0] - want[:, 0]).max() <= 1e-5
    ok = grad_mask(ref)
    rel = np.linalg.norm(c[ok, 1:] - want[ok, 1:], axis=1) / np.linalg.norm(want[ok, 1:], axis=1)
    assert rel.max() <= 1e-3 and ok.mean() > 0.5
    v, g, _ = scene.eval_host(w.poses)
    assert np.array_equal(c[:, 1:], -g)
    # a stage that sees no obstacle (an obstacle-free perception frame, or an empty row window) is an
    # inactive constraint row (+inf, 0, 0, 0), never NaN (reading G17), also with rho_theta = 0
    scene.update(w.A, w.B, np.zeros_like(w.S))
    for rt in (rho_t, 0.0):
        c0 = scene.mpc_coeffs_host(w.poses, d_min, rho_p, rt)
        assert np.isposinf(c0[:, 0]).all() and (c0[:, 1:] == 0).all()
        assert np.array_equal(c0, O.mpc_coeffs(np.full(w.N, np.inf), np.zeros((w.N, 3)), w.footprint, d_min, rho_p, rt).astype(np.float32))
    scene.close()
    big = W.make_config(3, n_traj=60)                      # graph path (N > 512) on an empty scene
    s2 = psdf.Scene(big.footprint, big.A, big.B, np.zeros_like(big.S), max_poses=big.N)
    c1 = s2.mpc_coeffs_host(big.poses, d_min, rho_p, rho_t)
    assert np.isposinf(c1[:, 0]).all() and (c1[:, 1:] == 0).all()
    s2.close()


def test_table1_shapes(env):
    """Paper Table I grid M in {1,10,100} x B in {1,15,100}."""
    torch, O, psdf, W = env
    for M in (1, 10, 100):
        for Bsz in (1, 15, 100):
            w = W.table1_case(M, Bsz)
            ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
            scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=Bsz)
            v, g, _ = scene.eval_host(w.poses)
            compare(ref, v, g, what=w.name)
            scene.close()


def test_device_encode_edges(env):
    """On-device EncodeEdges (Alg.1 l.1-4): device-resident (A,B,S) are
    packed by the pack kernels; results must be bit-identical to the host packer, and a
    rejected device update must leave the old scene in force."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(77)
    for cfg, n in ((4, 700), (5, 600)):
        w = W.make_config(cfg).subsample(n)
        A, B, S = w.A.copy(), w.B.copy(), w.S.copy()
        for i in range(0, w.M, 3):                      # every third row clockwise
            sl = np.nonzero(S[i])[0]
            A[i, sl], B[i, sl] = w.B[i, sl][::-1].copy(), w.A[i, sl][::-1].copy()
        S[5::17] = 0                                    # some absent obstacles
        host = psdf.Scene(w.footprint, A, B, S, max_poses=n)
        dev = psdf.Scene(w.footprint, torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(),
                         torch.from_numpy(S).cuda(), max_poses=n)
        assert (dev.num_obstacles, dev.num_edges) == (host.num_obstacles, host.num_edges)
        a = _run(torch, host, w.poses, grad=True, per_obstacle=True)
        b = _run(torch, dev, w.poses, grad=True, per_obstacle=True)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        compare(O.evaluate(w.footprint, A, B, S, w.poses[:200], per_obstacle=True), b[0][:200], b[1][:200], b[2][:200])
        # device update with new values (perception update) == fresh host scene
        shift = rng.uniform(-0.5, 0.5, (w.M, 1, 2)).astype(np.float32)
        A2 = (A + shift).astype(np.float32)
        B2 = A2.copy()
        for i in range(w.M):                            # re-close the rows after the shift
            sl = np.nonzero(S[i])[0]
            if sl.size:
                B2[i, sl] = A2[i, np.roll(sl, -1)]         # B_j == A_next for either orientation
        try:
            host2 = psdf.Scene(w.footprint, A2, B2, S, max_poses=n)
        except psdf.PsdfError:
            host2 = None                                # fp32 rounding of the shift made an edge degenerate
        if host2 is not None:
            dev.update(torch.from_numpy(A2).cuda(), torch.from_numpy(B2).cuda(), torch.from_numpy(S).cuda())
            for x, y in zip(_run(torch, host2, w.poses, grad=True), _run(torch, dev, w.poses, grad=True)):
                assert x is None or np.array_equal(x, y)
            host2.close()
            dev.update(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), torch.from_numpy(S).cuda())
        # degenerate device updates are rejected, old scene stays
        bad = []
        S1 = S.copy(); r = int(np.nonzero(S.sum(1) > 3)[0][0]); S1[r, np.nonzero(S1[r])[0][1]] = 0
        bad.append((A, B, S1))                          # open row
        S2 = S.copy(); r2 = int(np.nonzero(S.sum(1) >= 3)[0][1]); S2[r2] = 0; S2[r2, :2] = 1
        bad.append((A, B, S2))                          # fewer than 3 edges
        A3, B3 = A.copy(), B.copy(); sl = np.nonzero(S[r])[0]
        A3[r, sl[1]] = B3[r, sl[0]] = A[r, sl[0]]
        bad.append((A3, B3, S))                         # zero-length edge
        A4, B4 = A.copy(), B.copy()
        c = A[r, sl].mean(0)
        A4[r, sl[1]] = B4[r, sl[0]] = (c - 0.3 * (A[r, sl[1]] - c)).astype(np.float32)   # past the diagonal
        bad.append((A4, B4, S))                         # dented (non-convex) polygon
        for Ab, Bb, Sb in bad:
            with pytest.raises(psdf.PsdfError) as e:
                dev.update(torch.from_numpy(Ab).cuda(), torch.from_numpy(Bb).cuda(), torch.from_numpy(Sb).cuda())
            assert e.value.status == psdf.PSDF_ERR_DEGENERATE
            with pytest.raises(psdf.PsdfError):
                host.update(Ab, Bb, Sb)                 # the host packer agrees
            for x, y in zip(a, _run(torch, dev, w.poses, grad=True, per_obstacle=True)):
                assert np.array_equal(x, y)
        host.close()
        dev.close()


def test_time_varying_row_windows(env):
    """Per-stage edge sets E_{k+s}: the scene holds H stage-wise obstacle sets,
    pose s is evaluated against its own stage's rows only; oracle = one evaluation per stage."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(321)
    base = W.table1_case(12, 1, seed=777)
    H, Ms, E = 15, base.M, base.E
    vel = rng.uniform(-1.0, 1.0, (Ms, 1, 2)).astype(np.float32)
    A = np.concatenate([(base.A + vel * np.float32(0.1 * s)).astype(np.float32) for s in range(H)])
    B = A.copy()
    S = np.concatenate([base.S] * H)
    for i in range(H * Ms):
        sl = np.nonzero(S[i])[0]
        B[i, sl] = A[i, np.roll(sl, -1)]
    n_per = 9
    poses = np.stack([rng.uniform(0, 20, H * n_per), rng.uniform(0, 20, H * n_per),
                      rng.uniform(-3.2, 3.2, H * n_per)], 1).astype(np.float32)
    stage = np.repeat(np.arange(H), n_per)
    win = np.stack([stage * Ms, (stage + 1) * Ms], 1).astype(np.int32)
    for device_scene in (False, True):
        if device_scene:
            scene = psdf.Scene(base.footprint, torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(),
                               torch.from_numpy(S).cuda(), max_poses=len(poses))
        else:
            scene = psdf.Scene(base.footprint, A, B, S, max_poses=len(poses))
        v, g = scene.eval_windows(torch.from_numpy(poses).cuda(), torch.from_numpy(win).cuda())
        torch.cuda.synchronize()
        v, g = v.cpu().numpy(), g.cpu().numpy()
        vh, gh = scene.eval_windows_host(poses, win)
        assert np.array_equal(v, vh) and np.array_equal(g, gh)
        for s in range(H):
            rows = slice(s * Ms, (s + 1) * Ms)
            ref = O.evaluate(base.footprint, A[rows], B[rows], S[rows], poses[stage == s])
            compare(ref, v[stage == s], g[stage == s], what=f"stage {s}")
        # full window == plain evaluation; clamped and empty windows
        full = np.tile(np.array([[-5, 10 ** 6]], np.int32), (len(poses), 1))
        vf, gf = scene.eval_windows_host(poses, full)
        v0, g0, _ = scene.eval_host(poses)
        assert np.array_equal(vf, v0) and np.array_equal(gf, g0)
        empty = np.tile(np.array([[7, 7]], np.int32), (len(poses), 1))
        ve, ge = scene.eval_windows_host(poses, empty)
        assert np.isposinf(ve).all() and (ge == 0).all()
        vv, gn = scene.eval_windows_host(poses, win, grad=False)
        assert gn is None and np.array_equal(vv, v)
        scene.close()


def test_component_min_and_trajectory_reduce(env):
    """NEXT-4 reductions through the C ABI vs the oracle's plain definitions."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(55)
    # non-convex obstacles: config-2 rows grouped 3 at a time into 22 obstacles (last group smaller)
    w = W.make_config(2)
    ids = (np.arange(w.M) // 3).astype(np.int32)
    ids[5] = 99                                                    # an id outside the range is ignored
    n_obs = int(np.ceil(w.M / 3)) + 1                              # plus one obstacle without components
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v, g, po = scene.eval(torch.from_numpy(w.poses).cuda(), grad=True, per_obstacle=True)
    out = psdf.psdf_component_min(po, torch.from_numpy(ids).cuda(), n_obs)
    torch.cuda.synchronize()
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses, per_obstacle=True)
    want = O.component_min(ref.per_obstacle, ids, n_obs)
    got = out.cpu().numpy().astype(np.float64)
    assert np.array_equal(np.isposinf(got), np.isposinf(want)) and np.isposinf(got[:, -1]).all()
    fin = np.isfinite(want)
    assert np.abs(got[fin] - want[fin]).max() <= 1e-5
    assert np.array_equal(got, O.component_min(po.cpu().numpy(), ids, n_obs))   # exact fold of the GPU's own values
    scene.close()
    # sampled trajectories: config-3-like batch, T x H with H not a multiple of 32
    w = W.make_config(3, n_traj=300)
    T, H = 300, w.N // 300
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v, _, _ = scene.eval(torch.from_numpy(w.poses).cuda(), grad=False)
    d_safe = 0.5
    mn, am, pen = psdf.psdf_trajectory_reduce(v, T, H, d_safe)
    torch.cuda.synchronize()
    vh = v.cpu().numpy()
    rmn, ram, rpen = O.trajectory_reduce(vh, T, H, d_safe)         # definitions on the same fp32 values
    assert np.array_equal(mn.cpu().numpy().astype(np.float64), rmn)
    assert np.array_equal(am.cpu().numpy(), ram)
    assert np.abs(pen.cpu().numpy() - rpen).max() <= 1e-5 * max(1.0, rpen.max())
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    omn, _, open_ = O.trajectory_reduce(ref.value, T, H, d_safe)   # and against the oracle end to end
    assert np.abs(mn.cpu().numpy() - omn).max() <= 1e-5
    assert np.abs(pen.cpu().numpy() - open_).max() <= 1e-4 * max(1.0, open_.max())
    assert (rpen > 0).any()
    scene.close()


def test_eval_is_cuda_graph_capturable(env):
    """psdf_eval only enqueues (no allocation, no synchronisation): it can be captured into a
    CUDA graph on the caller's stream and replayed on new pose contents; dense (chunked
    tile-scan), lane-split and culled paths."""
    torch, O, psdf, W = env
    for cfg, n, cull in ((3, 6000, False), (3, 6000, True), (2, 50, False)):
        w = W.make_config(cfg) if cfg == 2 else W.make_config(cfg, n_traj=n // 50)
        scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
        scene.set_culling(cull)
        poses = torch.from_numpy(w.poses).cuda()
        value = torch.empty(w.N, dtype=torch.float32, device="cuda")
        grad = torch.empty((w.N, 3), dtype=torch.float32, device="cuda")
        scene.eval(poses, value=value, grad=grad)                   # warm-up outside capture
        torch.cuda.synchronize()
        want_v, want_g = value.clone(), grad.clone()
        static = poses.clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            scene.eval(static, value=value, grad=grad)
        value.zero_(); grad.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(value, want_v) and torch.equal(grad, want_g)
        # new contents through the same graph
        shifted = w.poses.copy()
        shifted[:, 2] += np.float32(0.5)
        static.copy_(torch.from_numpy(shifted).cuda())
        g.replay()
        torch.cuda.synchronize()
        v2, g2, _ = scene.eval(torch.from_numpy(shifted).cuda(), grad=True)
        assert torch.equal(value, v2) and torch.equal(grad, g2)
        del g
        scene.close()


def test_autograd_module(env):
    """PSDF nn.Module: forward = value, backward = stored witness gradient times the upstream
    gradient; checked against the oracle's dual-number gradient through a scalar loss."""
    torch, O, psdf, W = env
    from paper_2607_04310_b200.autograd import PSDF
    w = W.make_config(2)
    mod = PSDF(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    poses = torch.from_numpy(w.poses).cuda().requires_grad_(True)
    phi = mod(poses)
    weights = torch.linspace(0.5, 2.0, w.N, device="cuda")
    (weights * phi).sum().backward()
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    assert np.abs(phi.detach().cpu().numpy() - ref.value).max() <= 1e-5
    from tests.parity import grad_mask
    ok = grad_mask(ref)
    want = weights.cpu().numpy()[:, None] * ref.grad
    got = poses.grad.cpu().numpy()
    rel = np.linalg.norm(got[ok] - want[ok], axis=1) / np.linalg.norm(want[ok], axis=1)
    assert rel.max() <= 1e-3 and ok.mean() > 0.5
    mod.scene.close()


def test_odd_footprint_padding_adds_no_witness_boundary(env):
    """A 15-vertex footprint is padded to 16 for the kernels.  Padding by splitting an edge at
    its midpoint put an artificial vertex-region boundary on that edge: at 18 m range fp32
    cannot separate the two collinear halves (d^2 differs by one ulp) and the witness snapped to
    the artificial vertex (gradient off by 6e-3; found by a randomised run against the oracle,
    this is that case).  Padding with copies of a vertex adds no boundary."""
    torch, O, psdf, W = env
    footprint = np.array([[1.1168420314788818, -0.327312171459198], [1.010167121887207, -0.12635846436023712],
                          [0.7492443323135376, 0.035527586936950684], [0.37918949127197266, 0.13035441935062408],
                          [-0.03601149469614029, 0.14172562956809998], [-0.4245666563510895, 0.06767500191926956],
                          [-0.7192912697792053, -0.07899341732263565], [-0.8692247271537781, -0.27291932702064514],
                          [-0.8484421968460083, -0.4805711805820465], [-0.6605371832847595, -0.6660441160202026],
                          [-0.33800017833709717, -0.7972680926322937], [0.06339926272630692, -0.8515533804893494],
                          [0.4742555320262909, -0.8195134997367859], [0.8235278129577637, -0.7066885232925415],
                          [1.0508238077163696, -0.5325868129730225]], np.float32)
    poly = np.array([[-92.06255340576172, -74.37434387207031], [-92.02520751953125, -74.52521514892578],
                     [-91.90606689453125, -74.4957275390625], [-91.94340515136719, -74.34485626220703]], np.float32)
    A = poly[None].copy()
    B = np.roll(poly, -1, axis=0)[None].copy()
    S = np.ones((1, 4), np.uint8)
    poses = np.array([[-77.1455078125, -85.82178497314453, 0.9523851275444031]], np.float32)
    ref = O.evaluate(footprint, A, B, S, poses)
    assert ref.margin[0] > 1e-3                          # a well-separated winner: the comparison is meaningful
    scene = psdf.Scene(footprint, A, B, S, max_poses=4)
    v, g, _ = _run(torch, scene, poses, grad=True)
    compare(ref, v, g, what="15-gon at 18 m")
    vh, gh, _ = scene.eval_host(poses, grad=True)
    compare(ref, vh, gh, what="15-gon at 18 m, host path")
    scene.close()
