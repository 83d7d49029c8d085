"""Serving mode (psdf_serve_begin / psdf_serve_step / psdf_serve_end, include/psdf.h): a persistent kernel
with a mailbox in mapped memory for one fixed MPC batch shape (Alg.1 l.5-11).  Rows must
be bit-identical to psdf_eval_host / psdf_mpc_coeffs_host and match the oracle; the kernel must survive its
idle time-out (restart), perception updates (restart on the new scene) and other calls made next to it.
Every wait is bounded (idle time-outs of <= 300 ms).  Need a B200: `pytest -m gpu`."""
import time

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


class _Ref:
    def __init__(self, ref, sign=1.0):
        self.value, self.grad, self.margin, self.per_obstacle = ref.value, sign * ref.grad, ref.margin, None


@pytest.mark.parametrize("case", ["cfg1", "cfg2", "table1_M100_B15", "M1000_B3", "V6_B33"])
def test_serve_rows_equal_host_path_and_oracle(env, case):
    torch, O, psdf, W = env
    if case == "cfg1":
        w = W.make_config(1)
    elif case == "cfg2":
        w = W.make_config(2)
    elif case == "table1_M100_B15":
        w = W.table1_case(100, 15)
    elif case == "M1000_B3":
        w = W.table1_case(1000, 3)                      # K = 256 lanes per pose, one CTA per pose
    else:
        w = W.make_config(5).subsample(33)              # asymmetric 6-gon, 4096 obstacles
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v, g, _ = scene.eval_host(w.poses, grad=True)
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses)
    try:
        scene.serve_begin(w.N, idle_timeout_ms=300)
        for rep in range(50):
            rows = scene.serve_step(w.poses)
            assert np.array_equal(rows[:, 0], v) and np.array_equal(rows[:, 1:], g), (case, rep)
        compare(ref, rows[:, 0], rows[:, 1:], what=case + " serve")
        # new poses every step (an MPC loop): reversed order, shifted headings
        for rep in range(10):
            q = w.poses[::-1].copy()
            q[:, 2] += np.float32(0.01 * rep)
            rows = scene.serve_step(q)
            vq, gq, _ = scene.eval_host(q, grad=True)   # the ordinary host path may be used next to the server
            assert np.array_equal(rows[:, 0], vq) and np.array_equal(rows[:, 1:], gq), (case, rep)
        # soak: rows are accepted by watching them arrive (no acknowledgement word): thousands of steps with
        # alternating pose sets, every row of every step checked
        qa, qb = w.poses.copy(), w.poses[::-1].copy()
        va, ga, _ = scene.eval_host(qa, grad=True)
        vb, gb, _ = scene.eval_host(qb, grad=True)
        buf = np.empty((w.N, 4), np.float32)
        for rep in range(2000):
            scene.serve_step(qa, out=buf)
            assert np.array_equal(buf[:, 0], va) and np.array_equal(buf[:, 1:], ga), (case, rep)
            scene.serve_step(qb, out=buf)
            assert np.array_equal(buf[:, 0], vb) and np.array_equal(buf[:, 1:], gb), (case, rep)
        # coefficient rows, eqs.(26)-(28)
        scene.serve_begin(w.N, coeffs=(0.01, 0.1, 0.1), idle_timeout_ms=300)
        c = scene.serve_step(w.poses)
        assert np.array_equal(c, scene.mpc_coeffs_host(w.poses, 0.01, 0.1, 0.1))
        want = O.mpc_coeffs(ref.value, ref.grad, w.footprint, 0.01, 0.1, 0.1)
        fin = np.isfinite(want[:, 0])
        assert (np.abs(c[fin, 0] - want[fin, 0]) <= 1e-5 + 4 * np.abs(want[fin, 0]) * 2.0 ** -23).all()
        compare(_Ref(ref, -1.0), rows[:, 0] * 0 + ref.value.astype(np.float32), c[:, 1:], what=case + " J_g")
    finally:
        scene.serve_end()
    torch.cuda.synchronize()                            # returns at once: the kernel is gone
    scene.close()


def test_serve_with_row_windows(env):
    """Per-stage edge sets E_{k+s} under the server: the scene holds H stage-wise obstacle sets,
    stage s sees its own rows; the window table is fixed at psdf_serve_begin, a perception update brings new
    values for all stages.  Rows equal psdf_eval_windows_host bit for bit and the oracle per stage."""
    torch, O, psdf, W = env
    rng = np.random.default_rng(99)
    base = W.table1_case(12, 1, seed=778)
    H, Ms = 15, base.M
    vel = rng.uniform(-1.0, 1.0, (Ms, 1, 2)).astype(np.float32)

    def stacked(t0):
        A = np.concatenate([(base.A + vel * np.float32(0.1 * (s + t0))).astype(np.float32) for s in range(H)])
        B = A.copy()
        S = np.concatenate([base.S] * H)
        for i in range(H * Ms):
            sl = np.nonzero(S[i])[0]
            B[i, sl] = A[i, np.roll(sl, -1)]
        return A, B, S

    A, B, S = stacked(0)
    poses = np.stack([rng.uniform(0, 20, H), rng.uniform(0, 20, H), rng.uniform(-3.2, 3.2, H)], 1).astype(np.float32)
    win = np.stack([np.arange(H) * Ms, (np.arange(H) + 1) * Ms], 1).astype(np.int32)
    scene = psdf.Scene(base.footprint, A, B, S, max_poses=H)
    try:
        scene.serve_begin(H, row_window=win, idle_timeout_ms=300)
        for t0 in (0, 1, 2):                                   # control cycles: obstacles move, all stages updated
            if t0:
                A, B, S = stacked(t0)
                scene.update(A, B, S)
            vw, gw = scene.eval_windows_host(poses, win)
            rows = scene.serve_step(poses)
            assert np.array_equal(rows[:, 0], vw) and np.array_equal(rows[:, 1:], gw), t0
            for s_ in range(H):
                r = slice(s_ * Ms, (s_ + 1) * Ms)
                ref = O.evaluate(base.footprint, A[r], B[r], S[r], poses[s_:s_ + 1])
                compare(ref, rows[s_:s_ + 1, 0], rows[s_:s_ + 1, 1:], what=f"cycle {t0} stage {s_}")
        # coefficient rows under windows; a stage whose window is empty is an inactive row (reading G17)
        win2 = win.copy()
        win2[4] = (7, 7)
        scene.serve_begin(H, coeffs=(0.01, 0.1, 0.1), row_window=win2, idle_timeout_ms=300)
        c = scene.serve_step(poses)
        vw, gw = scene.eval_windows_host(poses, win2)
        keep = np.arange(H) != 4
        want = O.mpc_coeffs(vw.astype(np.float64), gw.astype(np.float64), base.footprint, 0.01, 0.1, 0.1)
        assert np.isposinf(c[4, 0]) and (c[4, 1:] == 0).all() and np.isposinf(vw[4])
        assert np.array_equal(c[keep, 1:], -gw[keep]) and np.abs(c[keep, 0] - want[keep, 0]).max() <= 1e-5
        scene.serve_begin(H, idle_timeout_ms=300)              # and back to all rows
        v, g, _ = scene.eval_host(poses)
        rows = scene.serve_step(poses)
        assert np.array_equal(rows[:, 0], v) and np.array_equal(rows[:, 1:], g)
    finally:
        scene.serve_end()
    scene.close()


def test_serve_survives_timeout_update_and_errors(env):
    torch, O, psdf, W = env
    w = W.make_config(1)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=64)
    v, g, _ = scene.eval_host(w.poses, grad=True)
    with pytest.raises(psdf.PsdfError):                 # step before begin
        scene._serve_N = w.N
        scene.serve_step(w.poses)
    for bad_n in (0, 513):
        with pytest.raises(psdf.PsdfError) as e:
            scene.serve_begin(bad_n)
        assert e.value.status == psdf.PSDF_ERR_INVALID_ARG
    with pytest.raises(psdf.PsdfError) as e:
        scene.serve_begin(65)                           # beyond the scene's max_poses
    assert e.value.status == psdf.PSDF_ERR_CAPACITY
    try:
        scene.serve_begin(w.N, idle_timeout_ms=30)
        rows = scene.serve_step(w.poses)
        assert np.array_equal(rows[:, 0], v)
        # idle time-out: the kernel exits by itself, the next step starts it again
        time.sleep(0.12)
        t0 = time.perf_counter()
        torch.cuda.synchronize()                        # nothing left to wait for
        assert time.perf_counter() - t0 < 0.02
        for _ in range(3):
            rows = scene.serve_step(w.poses)
            assert np.array_equal(rows[:, 0], v) and np.array_equal(rows[:, 1:], g)
        # perception update while serving: the server restarts on the new scene
        sh = np.array([0.5, -0.25], np.float32)
        scene.update(w.A + sh, w.B + sh, w.S)
        v2, g2, _ = scene.eval_host(w.poses, grad=True)
        rows = scene.serve_step(w.poses)
        assert np.array_equal(rows[:, 0], v2) and np.array_equal(rows[:, 1:], g2) and not np.array_equal(v2, v)
        scene.update(torch.from_numpy(w.A).cuda(), torch.from_numpy(w.B).cuda(), torch.from_numpy(w.S).cuda())
        rows = scene.serve_step(w.poses)
        assert np.array_equal(rows[:, 0], v) and np.array_equal(rows[:, 1:], g)
        # an obstacle-free frame: +inf, zero gradient; a non-finite pose: NaN row, neighbours unaffected
        scene.update(w.A, w.B, np.zeros_like(w.S))
        rows = scene.serve_step(w.poses)
        assert np.isposinf(rows[:, 0]).all() and (rows[:, 1:] == 0).all()
        scene.update(w.A, w.B, w.S)
        q = w.poses.copy()
        q[3, 1] = np.nan
        rows = scene.serve_step(q)
        keep = np.arange(w.N) != 3
        assert np.isnan(rows[3]).all() and np.array_equal(rows[keep, 0], v[keep])
        # device path and culling switch next to the server
        vd, gd, _ = scene.eval(torch.from_numpy(w.poses).cuda(), grad=True)
        scene.set_culling(True)
        rows = scene.serve_step(w.poses)
        assert np.array_equal(rows[:, 0], v) and np.array_equal(vd.cpu().numpy(), v)
    finally:
        scene.serve_end()
    scene.close()
