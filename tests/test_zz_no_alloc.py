"""psdf_eval_static_scratch: the evaluation entry point that allocates nothing (scratch in a file-scope
static device array of the library; include/psdf.h).  Its outputs against the existing path's
(psdf_eval), bit for bit as the other path-against-path tests do, on calls in a row that share the
array: a large batch, then a smaller ragged one (stale keys of the first call must not leak into it),
then the large one again; plus a sample against the oracle and the size limit.  Collected last on
purpose (the suite runs with pytest -x).  Need a B200: `pytest -m gpu`."""
import numpy as np
import pytest

from tests.parity import compare

pytestmark = pytest.mark.gpu


def test_static_scratch_entry_point_matches_psdf_eval():
    import torch
    from oracle import psdf_oracle as O
    from paper_2607_04310_b200 import psdf, workloads as W
    assert torch.cuda.is_available()
    w = W.make_config(3, n_traj=120)                     # 6000 poses x 256 obstacles: 94 pose tiles x 16 obstacle chunks
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=psdf.STATIC_SCRATCH_MAX_POSES + 64)
    p_big = torch.from_numpy(w.poses).cuda()
    p_small = torch.from_numpy(w.poses[1000:1000 + 2501].copy()).cuda()
    want = {}
    for name, p in (("big", p_big), ("small", p_small)):
        v, g, _ = scene.eval(p, grad=True)               # the existing path
        torch.cuda.synchronize()
        want[name] = (v.clone(), g.clone())
    # the entry point's code (everything behind its marker in psdf_api.cu) holds no allocating call
    import os, re
    src = open(os.path.join(os.path.dirname(psdf.LIB_PATH), "csrc", "psdf_api.cu")).read()
    tail = src[src.index("no-allocation entry point"):src.index("== serving mode")]
    tail = re.sub(r"//[^\n]*", "", tail)
    assert "psdf_eval_static_scratch" in tail and "cudaGetSymbolAddress" in tail
    assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaMallocHost|\bnew\b|malloc\(|std::vector", tail)
    value = torch.empty(w.N, dtype=torch.float32, device="cuda")
    grad = torch.empty((w.N, 3), dtype=torch.float32, device="cuda")
    for name, p in (("big", p_big), ("small", p_small), ("big", p_big), ("small", p_small)):   # calls in a row
        n = p.shape[0]
        value.fill_(-7.0); grad.fill_(-7.0)
        v, g = scene.eval_static_scratch(p, value=value[:n], grad=grad[:n])
        torch.cuda.synchronize()
        assert torch.equal(v, want[name][0]) and torch.equal(g, want[name][1]), name
        assert (value[n:] == -7.0).all()                 # nothing written past N
    v0, g0 = scene.eval_static_scratch(p_small, grad=False)    # value-only variant, then the existing path again
    assert g0 is None and torch.equal(v0, want["small"][0])
    v1, g1, _ = scene.eval(p_big, grad=True)
    assert torch.equal(v1, want["big"][0]) and torch.equal(g1, want["big"][1])
    # against the oracle, the tolerance of the parity tests
    idx = np.arange(0, w.N, 7)
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses[idx])
    v, g = scene.eval_static_scratch(p_big)
    compare(ref, v.cpu().numpy()[idx], g.cpu().numpy()[idx], what="static scratch vs oracle")
    # the size limit: rejected with a clear error, outputs untouched
    n_over = psdf.STATIC_SCRATCH_MAX_POSES + 1
    many = torch.zeros((n_over, 3), dtype=torch.float32, device="cuda")
    out = torch.full((n_over,), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(psdf.PsdfError) as e:
        scene.eval_static_scratch(many, value=out, grad=False)
    assert e.value.status == psdf.PSDF_ERR_CAPACITY and (out == -7.0).all()
    # at the limit it runs (scene of 256 obstacles, 65 536 poses), same bits as the existing path
    rng = np.random.default_rng(3)
    full = np.column_stack([rng.uniform(0, 40, n_over - 1), rng.uniform(0, 40, n_over - 1),
                            rng.uniform(-3.2, 3.2, n_over - 1)]).astype(np.float32)
    pf = torch.from_numpy(full).cuda()
    va, ga = scene.eval_static_scratch(pf)
    vb, gb, _ = scene.eval(pf, grad=True)
    assert torch.equal(va, vb) and torch.equal(ga, gb)
    scene.close()
