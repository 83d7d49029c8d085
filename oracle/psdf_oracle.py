"""ctypes wrapper over the double-precision CPU oracle (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs import this.  It never imports the CUDA binding.  Inputs of any float dtype are
widened to float64 exactly; see psdf_oracle.cpp for what is computed and the citations.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        _lib.psdf_oracle_eval.restype = ctypes.c_int
        _lib.psdf_oracle_eval.argtypes = [dp, ctypes.c_int, dp, dp, ctypes.POINTER(ctypes.c_uint8),
                                          ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, dp, dp, dp,
                                          dp, ip, ip, ctypes.c_double, ctypes.c_int]
        _lib.psdf_oracle_max_threads.restype = ctypes.c_int
    return _lib


def max_threads() -> int:
    return int(lib().psdf_oracle_max_threads())


@dataclass
class OracleResult:
    value: np.ndarray          # [N] f64   phi (eq.6)
    grad: np.ndarray           # [N,3] f64 d phi / d(x,y,theta)
    per_obstacle: np.ndarray   # [N,M] f64 sd^i (eq.23), +inf for empty rows (or None)
    margin: np.ndarray         # [N] f64   reading G9
    winner: np.ndarray         # [N] i32   argmin obstacle row (-1: none)
    branch: np.ndarray         # [N] i32   1 separated / 0 not separated, of the winner


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def evaluate(footprint, A, B, S, poses, per_obstacle=False, window=0.01, nthreads=0) -> OracleResult:
    fp = np.ascontiguousarray(footprint, dtype=np.float64)
    A = np.ascontiguousarray(A, dtype=np.float64)
    B = np.ascontiguousarray(B, dtype=np.float64)
    S = np.ascontiguousarray(S, dtype=np.uint8)
    poses = np.ascontiguousarray(poses, dtype=np.float64).reshape(-1, 3)
    V, (M, E), N = fp.shape[0], S.shape, poses.shape[0]
    assert fp.shape == (V, 2) and A.shape == (M, E, 2) and B.shape == (M, E, 2)
    value = np.empty(N)
    grad = np.empty((N, 3))
    per = np.empty((N, M)) if per_obstacle else None
    margin = np.empty(N)
    winner = np.empty(N, dtype=np.int32)
    branch = np.empty(N, dtype=np.int32)
    rc = lib().psdf_oracle_eval(_p(fp, ctypes.c_double), V, _p(A, ctypes.c_double),
                                _p(B, ctypes.c_double), _p(S, ctypes.c_uint8), M, E,
                                _p(poses, ctypes.c_double), N, _p(value, ctypes.c_double),
                                _p(grad, ctypes.c_double), _p(per, ctypes.c_double),
                                _p(margin, ctypes.c_double), _p(winner, ctypes.c_int),
                                _p(branch, ctypes.c_int), float(window), int(nthreads))
    if rc != 0:
        raise ValueError("psdf_oracle_eval: bad arguments")
    return OracleResult(value, grad, per, margin, winner, branch)


def evaluate_value_only(footprint, A, B, S, poses, nthreads=0) -> np.ndarray:
    """Plain-double pass only (no duals): what bench.py times as the CPU baseline."""
    fp = np.ascontiguousarray(footprint, dtype=np.float64)
    A = np.ascontiguousarray(A, dtype=np.float64)
    B = np.ascontiguousarray(B, dtype=np.float64)
    S = np.ascontiguousarray(S, dtype=np.uint8)
    poses = np.ascontiguousarray(poses, dtype=np.float64).reshape(-1, 3)
    V, (M, E), N = fp.shape[0], S.shape, poses.shape[0]
    value = np.empty(N)
    rc = lib().psdf_oracle_eval(_p(fp, ctypes.c_double), V, _p(A, ctypes.c_double),
                                _p(B, ctypes.c_double), _p(S, ctypes.c_uint8), M, E,
                                _p(poses, ctypes.c_double), N, _p(value, ctypes.c_double),
                                None, None, None, None, None, 0.01, int(nthreads))
    if rc != 0:
        raise ValueError("psdf_oracle_eval: bad arguments")
    return value


def component_min(per_component: np.ndarray, comp_to_obstacle, n_obstacles: int) -> np.ndarray:
    """Non-convex obstacles as unions of convex components (Assumption 1): the
    signed distance to obstacle o is the minimum over its components (eq.(6), PAPER.md:93-97,
    restricted to the components of o).  Plain definition, float64; +inf where o has none."""
    pc = np.asarray(per_component, np.float64)
    ids = np.asarray(comp_to_obstacle)
    out = np.full((pc.shape[0], int(n_obstacles)), np.inf)
    for o in range(int(n_obstacles)):
        cols = np.nonzero(ids == o)[0]
        if cols.size:
            out[:, o] = pc[:, cols].min(axis=1)
    return out


def trajectory_reduce(value: np.ndarray, T: int, H: int, d_safe: float):
    """Sampled-trajectory reductions (pose index = trajectory * H + stage): clearance
    min_s phi_s, its first arg-min stage, soft penalty sum_s max(0, d_safe - phi_s)^2.
    Plain definitions in float64."""
    v = np.asarray(value, np.float64).reshape(int(T), int(H))
    return v.min(axis=1), v.argmin(axis=1), (np.maximum(float(d_safe) - v, 0.0) ** 2).sum(axis=1)


def mpc_coeffs(value, grad, footprint, d_min: float, rho_p: float, rho_theta: float) -> np.ndarray:
    """Stage-wise QP parameter vectors [h_s - gamma_s ; J_g,s] of eqs.(26)-(28), PAPER.md:247-289,
    literally, in float64, from the PSDF values phi_s [N] and state gradients [N,3]:
        h_s     = phi_s - d_min
        J_g,s   = -grad_x phi_s
        r_max   = max_{v in V0} |v|_2                                       Prop.1
        gamma_s = 1/2 (r_max + phi_s) rho_theta^2 + rho_p rho_theta         eq.(27)
    Returns [N,4].  The paper is silent on a stage that sees no obstacle (phi_s = +inf, where
    eq.(27) reads inf - inf): the row is (+inf, 0, 0, 0), an inactive constraint (DESIGN.md
    reading G17)."""
    phi = np.asarray(value, np.float64).reshape(-1)
    g = np.asarray(grad, np.float64).reshape(-1, 3)
    fp = np.asarray(footprint, np.float64)
    r_max = max(float(np.hypot(v[0], v[1])) for v in fp)
    out = np.empty((phi.shape[0], 4))
    for s in range(phi.shape[0]):
        if np.isposinf(phi[s]):
            out[s] = (np.inf, 0.0, 0.0, 0.0)
            continue
        h_s = phi[s] - float(d_min)
        gamma_s = 0.5 * (r_max + phi[s]) * float(rho_theta) ** 2 + float(rho_p) * float(rho_theta)
        out[s, 0] = h_s - gamma_s
        out[s, 1:] = -g[s]
    return out
