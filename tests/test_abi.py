"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol that
include/psdf.h declares, and its host logic (validation, error codes) behaves.  No compute."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def psdf():
    from paper_2607_04310_b200 import build
    build.build()
    from paper_2607_04310_b200 import psdf as m
    return m


def _declared(header):
    hdr = open(os.path.join(ROOT, "include", header)).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return set(re.findall(r"\b(psdf_[a-z0-9_]+)\s*\(", hdr))


def test_exports_match_header(psdf):
    """Every symbol include/psdf.h (product ABI) and include/psdf_bench.h (instrumentation) declare
    is exported, and the binding's lists are exactly the headers'."""
    declared = _declared("psdf.h")
    assert declared == set(psdf.EXPORTS), declared ^ set(psdf.EXPORTS)
    bench = _declared("psdf_bench.h")
    assert bench == set(psdf.BENCH_EXPORTS), bench ^ set(psdf.BENCH_EXPORTS)
    assert not (declared & bench)
    L = psdf.lib()
    for name in declared | bench:
        assert getattr(L, name) is not None
    assert "sm_100a" in psdf.psdf_version()
    assert psdf.lib().psdf_status_string(-2).decode().startswith("degenerate")
    assert psdf.lib().psdf_status_string(psdf.PSDF_ERR_ALLOC).decode() == "allocation failed"
    assert "another host thread" in psdf.lib().psdf_status_string(psdf.PSDF_ERR_BUSY).decode()
    # the status codes of the header and of the binding agree
    hdr = open(os.path.join(ROOT, "include", "psdf.h")).read()
    for name, val in re.findall(r"(PSDF_(?:OK|ERR_[A-Z_]+))\s*=\s*(-?\d+)", hdr):
        assert getattr(psdf, name) == int(val), name


def test_product_build_has_no_tuning_knobs(psdf):
    """The sweep knobs (PSDF_BD, PSDF_CHUNKS, PSDF_BRANCHES, PSDF_NO_ZERO_COPY) exist only in
    -DPSDF_TUNING measurement builds: the product library holds neither their names nor a getenv."""
    blob = open(psdf.LIB_PATH, "rb").read()
    for knob in (b"PSDF_BD", b"PSDF_CHUNKS", b"PSDF_BRANCHES", b"PSDF_NO_ZERO_COPY", b"PSDF_CULL_NP", b"PSDF_GRID_PER_CELL"):
        assert knob not in blob, knob
    src = open(os.path.join(ROOT, "paper_2607_04310_b200", "csrc", "psdf_api.cu")).read()
    outside = re.sub(r"#ifdef PSDF_TUNING.*?#endif", "", src, flags=re.S)
    assert "getenv" not in outside


def test_host_validation_without_gpu(psdf):
    from paper_2607_04310_b200 import workloads as W
    w = W.make_config(1)

    def status(fp, A, B, S, max_poses=8):
        try:
            s = psdf.Scene(fp, A, B, S, max_poses)
        except psdf.PsdfError as e:
            return e.status
        s.close()
        return 0

    assert status(w.footprint[::-1].copy(), w.A, w.B, w.S) == psdf.PSDF_ERR_DEGENERATE   # CW footprint
    assert status(w.footprint[:2], w.A, w.B, w.S) == psdf.PSDF_ERR_INVALID_ARG           # V < 3
    assert status(np.zeros((17, 2), np.float32), w.A, w.B, w.S) == psdf.PSDF_ERR_INVALID_ARG
    bow = np.array([[0, 0], [1, 1], [1, 0], [0, 1]], np.float32)
    assert status(bow, w.A, w.B, w.S) == psdf.PSDF_ERR_DEGENERATE                        # not convex
    S = w.S.copy()
    S[0, np.nonzero(S[0])[0][0]] = 0
    assert status(w.footprint, w.A, w.B, S) == psdf.PSDF_ERR_DEGENERATE                  # open row
    A = w.A.copy()
    j = np.nonzero(w.S[1])[0]
    A[1, j[1]] = A[1, j[0]]
    assert status(w.footprint, A, w.B, w.S) == psdf.PSDF_ERR_DEGENERATE
    assert status(w.footprint, w.A[:, :2], w.B[:, :2], w.S[:, :2]) == psdf.PSDF_ERR_INVALID_ARG  # E < 3
    assert status(w.footprint, w.A, w.B, w.S, max_poses=0) == psdf.PSDF_ERR_INVALID_ARG
    import torch
    if not torch.cuda.is_available():      # valid input but no device: a loud CUDA error, no fallback
        assert status(w.footprint, w.A, w.B, w.S) == psdf.PSDF_ERR_CUDA


def test_no_oracle_on_product_path():
    """The product never imports the oracle; the oracle never imports the product."""
    pkg = os.path.join(ROOT, "paper_2607_04310_b200")
    bad = re.compile(r"^\s*(import|from)\s+oracle|#include.*oracle|psdf_oracle", re.M)
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not bad.search(open(os.path.join(dp, f)).read()), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2607_04310_b200 import" not in txt and "import paper_2607" not in txt
            assert "csrc/" not in txt.replace("(paper_2607_04310_b200/csrc)", "")
