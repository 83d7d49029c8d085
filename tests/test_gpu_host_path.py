"""The host entry points at full size (Alg.1 l.5-11: upload the states, evaluate,
bring the results back): psdf_eval_host / psdf_mpc_coeffs_host for N > 512 replay a captured graph
of {H2D, kernel, D2H} branches, the configuration bench.py's `e2e` figure is measured on.  Checked
bit for bit against psdf_eval and on a sample against the oracle, with ordinary and with pinned
caller buffers, dense and culled; plus the ordering rules of include/psdf.h (host calls next to an
asynchronous psdf_eval, updates across streams, one host thread per scene, allocation failures).
Need a B200: `pytest -m gpu`."""
import threading

import numpy as np
import pytest

from tests.parity import compare, grad_mask

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf, workloads as W
    assert torch.cuda.is_available()
    return torch, O, psdf, W


def _pinned(torch, shape, dtype=np.float32):
    t = torch.empty(shape, dtype=getattr(torch, np.dtype(dtype).name), pin_memory=True)
    return t.numpy()


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_eval_host_full_size(env, workloads_cache, cfg):
    torch, O, psdf, W = env
    w = workloads_cache(cfg)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    p = torch.from_numpy(w.poses).cuda()
    v, g, _ = scene.eval(p, grad=True)
    torch.cuda.synchronize()
    v, g = v.cpu().numpy(), g.cpu().numpy()
    rng = np.random.default_rng(500 + cfg)
    idx = np.sort(rng.choice(w.N, size={3: 3000, 4: 1200, 5: 1000}[cfg], replace=False))
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses[idx])
    pin_p, pin_v, pin_g = _pinned(torch, (w.N, 3)), _pinned(torch, (w.N,)), _pinned(torch, (w.N, 3))
    pin_p[:] = w.poses
    for culling in (False, True):
        scene.set_culling(culling)
        for rep in range(2):                                   # capture, then replay
            vh, gh, _ = scene.eval_host(w.poses, grad=True)    # ordinary memory: staged
            assert np.array_equal(vh, v) and np.array_equal(gh, g), (cfg, culling, rep)
        st = compare(ref, vh[idx], gh[idx], what=f"{w.name} eval_host culling={culling}")
        pin_v[:] = 0; pin_g[:] = 0
        for rep in range(2):
            scene.eval_host_into(pin_p, pin_v, pin_g)          # pinned memory: copied in place
            assert np.array_equal(pin_v, v) and np.array_equal(pin_g, g), (cfg, culling, rep, "pinned")
        v0, g0, _ = scene.eval_host(w.poses, grad=False)       # value-only graph
        assert g0 is None and np.array_equal(v0, v)
        c = scene.mpc_coeffs_host(w.poses, 0.01, 0.1, 0.1)     # [h - gamma ; J_g], eqs.(26)-(28)
        assert np.array_equal(c[:, 1:], -g)
        want = O.mpc_coeffs(ref.value, ref.grad, w.footprint, 0.01, 0.1, 0.1)
        assert (np.abs(c[idx, 0] - want[:, 0]) <= 1e-5 + 4 * np.abs(want[:, 0]) * 2.0 ** -23).all()
        print(w.name, "culling", culling, st)
    # a ragged size that is not a multiple of any chunk or tile, mixed pinned / ordinary buffers
    n = w.N - 4099
    scene.set_culling(False)
    g_buf = np.empty((n, 3), np.float32) if cfg == 4 else pin_g[:n]
    pin_v[:] = 0
    scene.eval_host_into(pin_p[:n], pin_v[:n], g_buf)
    assert np.array_equal(pin_v[:n], v[:n]) and np.array_equal(g_buf, g[:n]) and (pin_v[n:] == 0).all()
    vr, gr, _ = scene.eval_host(w.poses[:n], grad=True)
    assert np.array_equal(vr, v[:n]) and np.array_equal(gr, g[:n])
    scene.close()


def test_per_obstacle_graph_path(env, workloads_cache):
    """[N,M] per-obstacle output through the branched graph (N > 512), ordinary and pinned."""
    torch, O, psdf, W = env
    w = workloads_cache(3).subsample(9000)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v, g, po = scene.eval(torch.from_numpy(w.poses).cuda(), grad=True, per_obstacle=True)
    torch.cuda.synchronize()
    vh, gh, poh = scene.eval_host(w.poses, grad=True, per_obstacle=True)
    assert np.array_equal(vh, v.cpu().numpy()) and np.array_equal(gh, g.cpu().numpy()) and np.array_equal(poh, po.cpu().numpy())
    pp = _pinned(torch, (w.N, w.M))
    vv = np.empty(w.N, np.float32)
    scene.eval_host_into(w.poses, vv, None, pp)
    assert np.array_equal(pp, poh) and np.array_equal(vv, vh)
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses[:1500], per_obstacle=True)
    compare(ref, vh[:1500], gh[:1500], poh[:1500], what="per-obstacle graph path")
    scene.close()


def test_host_calls_next_to_async_eval(env, workloads_cache):
    """include/psdf.h ordering rule: the host entry points own a stream and a workspace, so they may
    run while an asynchronous psdf_eval of the same scene is in flight on the caller's stream.  Both
    use chunked kernels (cross-chunk keys and arrival counters in the workspace)."""
    torch, O, psdf, W = env
    w = workloads_cache(4)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    p = torch.from_numpy(w.poses).cuda()
    v_ref, g_ref, _ = scene.eval(p, grad=True)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    small = w.poses[:6000]
    win = np.tile(np.array([[0, w.M]], np.int32), (300, 1))
    overlapped = 0
    for it in range(6):
        v = torch.zeros(w.N, dtype=torch.float32, device="cuda")
        g = torch.zeros((w.N, 3), dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        scene.eval(p, value=v, grad=g, stream=side)             # ~3 ms in flight on `side`
        vh, gh, _ = scene.eval_host(small, grad=True)           # meanwhile, on the scene's stream
        c = scene.mpc_coeffs_host(small, 0.01, 0.1, 0.1)
        vw, gw = scene.eval_windows_host(w.poses[:300], win)
        overlapped += int(not side.query())                     # the device call was still running
        side.synchronize()
        assert torch.equal(v, v_ref) and torch.equal(g, g_ref), it
        assert np.array_equal(vh, v_ref[:6000].cpu().numpy()) and np.array_equal(gh, g_ref[:6000].cpu().numpy()), it
        assert np.array_equal(c[:, 1:], -gh)
        assert np.array_equal(vw, vh[:300]) and np.array_equal(gw, gh[:300])
    print("host calls returned while the device call was still in flight:", overlapped, "of 6")
    scene.close()


def test_update_after_eval_on_another_stream(env, workloads_cache):
    """Two updates in a row rewrite the buffer set an evaluation enqueued earlier on ANOTHER stream
    may still be reading: the update orders itself after it (include/psdf.h)."""
    torch, O, psdf, W = env
    w = workloads_cache(4)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    p = torch.from_numpy(w.poses).cuda()
    v_ref, g_ref, _ = scene.eval(p, grad=True)
    torch.cuda.synchronize()
    sh = np.array([0.25, -0.5], np.float32)
    A2, B2 = (w.A + sh).astype(np.float32), (w.B + sh).astype(np.float32)
    dA, dB, dS = torch.from_numpy(A2).cuda(), torch.from_numpy(B2).cuda(), torch.from_numpy(w.S).cuda()
    side = torch.cuda.Stream()
    for it in range(3):
        v = torch.zeros(w.N, dtype=torch.float32, device="cuda")
        g = torch.zeros((w.N, 3), dtype=torch.float32, device="cuda")
        scene.eval(p, value=v, grad=g, stream=side)
        scene.update(dA, dB, dS)                                 # on torch's current stream, not `side`
        scene.update(w.A, w.B, w.S)                              # rewrites the set the evaluation reads
        side.synchronize()
        assert torch.equal(v, v_ref) and torch.equal(g, g_ref), it
    scene.close()


def test_one_host_thread_per_scene(env, workloads_cache):
    """Concurrent use of one scene from two host threads is an error (PSDF_ERR_BUSY), not a race:
    every call either succeeds with the right result or reports BUSY and leaves its outputs alone."""
    torch, O, psdf, W = env
    w = workloads_cache(3)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v_ref, g_ref, _ = scene.eval_host(w.poses, grad=True)
    small = w.poses[:40].copy()
    stop = threading.Event()
    stats = {"ok": 0, "busy": 0, "bad": 0}

    def hammer():
        torch.cuda.set_device(0)
        while not stop.is_set():
            v = np.full(40, -7.0, np.float32)
            g = np.full((40, 3), -7.0, np.float32)
            try:
                scene.eval_host_into(small, v, g)
                good = np.array_equal(v, v_ref[:40]) and np.array_equal(g, g_ref[:40])
                stats["ok" if good else "bad"] += 1
            except psdf.PsdfError as e:
                untouched = (v == -7.0).all() and (g == -7.0).all()
                stats["busy" if (e.status == psdf.PSDF_ERR_BUSY and untouched) else "bad"] += 1

    t = threading.Thread(target=hammer)
    t.start()
    big_ok = big_busy = 0
    for _ in range(60):                                          # ~1 ms each: plenty of overlap
        try:
            v, g, _ = scene.eval_host(w.poses, grad=True)
            assert np.array_equal(v, v_ref) and np.array_equal(g, g_ref)
            big_ok += 1
        except psdf.PsdfError as e:
            assert e.status == psdf.PSDF_ERR_BUSY
            big_busy += 1
    stop.set()
    t.join()
    print("small calls", stats, "big calls ok/busy", big_ok, big_busy)
    assert stats["bad"] == 0 and stats["busy"] + big_busy > 0 and stats["ok"] > 0 and big_ok > 0
    scene.close()


def test_allocation_failure_is_reported_as_alloc(env):
    """cudaErrorMemoryAllocation maps to PSDF_ERR_ALLOC (not PSDF_ERR_CUDA) and the partly built scene
    is released: a 2.5e8-row scene wants ~300 GB of packed buffers.  The dummy device arrays are never
    read (allocation fails first); the library works normally afterwards."""
    torch, O, psdf, W = env
    import ctypes
    w = W.make_config(1)
    fp = np.ascontiguousarray(w.footprint, np.float32)
    dummy = torch.zeros(1024, dtype=torch.float32, device="cuda")
    free0 = torch.cuda.mem_get_info()[0]
    h = ctypes.c_void_p()
    rc = psdf.lib().psdf_create_scene(fp.ctypes.data, 4, dummy.data_ptr(), dummy.data_ptr(), dummy.data_ptr(),
                                      250_000_000, 8, psdf.PSDF_MEM_DEVICE, 16, None, ctypes.byref(h))
    assert rc == psdf.PSDF_ERR_ALLOC and not h.value
    assert torch.cuda.mem_get_info()[0] >= free0 - (64 << 20)    # nothing leaked
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    v, g, _ = scene.eval_host(w.poses)
    compare(O.evaluate(w.footprint, w.A, w.B, w.S, w.poses), v, g)
    scene.close()
