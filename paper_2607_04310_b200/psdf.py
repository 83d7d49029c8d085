"""Thin ctypes binding over libpsdf.so (include/psdf.h), same names as the C ABI.

Argument marshalling only: every step of the hot path runs in the CUDA kernels.
PyTorch is used for device memory and streams.  There is NO CPU fallback: if the
library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpsdf.so")

PSDF_OK = 0
PSDF_ERR_INVALID_ARG = -1
PSDF_ERR_DEGENERATE = -2
PSDF_ERR_CAPACITY = -3
PSDF_ERR_CUDA = -4
PSDF_ERR_ALLOC = -5
PSDF_ERR_BUSY = -6
STATIC_SCRATCH_MAX_POSES = 65536      # PSDF_STATIC_SCRATCH_MAX_POSES of include/psdf.h
PSDF_MEM_HOST = 0
PSDF_MEM_DEVICE = 1

# include/psdf.h: the product ABI
EXPORTS = ["psdf_create_scene", "psdf_update_scene", "psdf_eval", "psdf_eval_static_scratch", "psdf_eval_host",
           "psdf_eval_windows", "psdf_eval_windows_host", "psdf_mpc_coeffs_host", "psdf_serve_begin", "psdf_serve_step",
           "psdf_serve_end", "psdf_component_min",
           "psdf_trajectory_reduce", "psdf_set_components", "psdf_eval_trajectories", "psdf_set_culling", "psdf_destroy_scene", "psdf_scene_num_obstacles",
           "psdf_scene_num_edges", "psdf_last_cuda_error", "psdf_status_string", "psdf_version"]
# include/psdf_bench.h: measurement instrumentation (bench.py, tests)
BENCH_EXPORTS = ["psdf_kernel_launches", "psdf_cull_stats", "psdf_measure_fp32_peak", "psdf_bench_host_latency",
                 "psdf_scene_footprint_symmetric", "psdf_bench_serve_latency"]

_lib = None


class PsdfError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        msg = lib().psdf_status_string(int(status)).decode()
        extra = f" (cudaError {lib().psdf_last_cuda_error()})" if status == PSDF_ERR_CUDA else ""
        super().__init__(f"{where}: {msg}{extra}")


def lib():
    """Loads libpsdf.so (built in-tree by paper_2607_04310_b200/build.py); fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_04310_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, fp_, u8p = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
    i = ctypes.c_int
    L.psdf_create_scene.restype = i
    L.psdf_create_scene.argtypes = [fp_, i, fp_, fp_, u8p, i, i, i, i, vp, ctypes.POINTER(vp)]
    L.psdf_update_scene.restype = i
    L.psdf_update_scene.argtypes = [vp, fp_, fp_, u8p, i, vp]
    L.psdf_eval.restype = i
    L.psdf_eval.argtypes = [vp, fp_, i, fp_, fp_, fp_, vp]
    L.psdf_eval_static_scratch.restype = i
    L.psdf_eval_static_scratch.argtypes = [vp, fp_, i, fp_, fp_, vp]
    L.psdf_eval_host.restype = i
    L.psdf_eval_host.argtypes = [vp, fp_, i, fp_, fp_, fp_]
    L.psdf_eval_windows.restype = i
    L.psdf_eval_windows.argtypes = [vp, fp_, i, vp, fp_, fp_, vp]
    L.psdf_eval_windows_host.restype = i
    L.psdf_eval_windows_host.argtypes = [vp, fp_, i, vp, fp_, fp_]
    L.psdf_mpc_coeffs_host.restype = i
    L.psdf_mpc_coeffs_host.argtypes = [vp, fp_, i, ctypes.c_float, ctypes.c_float, ctypes.c_float, fp_]
    L.psdf_serve_begin.restype = i
    L.psdf_serve_begin.argtypes = [vp, i, vp, i, ctypes.c_float, ctypes.c_float, ctypes.c_float, i]
    L.psdf_serve_step.restype = i
    L.psdf_serve_step.argtypes = [vp, fp_, fp_]
    L.psdf_serve_end.restype = i
    L.psdf_serve_end.argtypes = [vp]
    L.psdf_bench_serve_latency.restype = i
    L.psdf_bench_serve_latency.argtypes = [vp, fp_, fp_, i, ctypes.POINTER(ctypes.c_double)]
    L.psdf_set_components.restype = i
    L.psdf_set_components.argtypes = [vp, vp, i]
    L.psdf_eval_trajectories.restype = i
    L.psdf_eval_trajectories.argtypes = [vp, fp_, i, i, ctypes.c_float, fp_, fp_, fp_, vp, fp_, vp]
    L.psdf_set_culling.restype = i
    L.psdf_set_culling.argtypes = [vp, i]
    L.psdf_component_min.restype = i
    L.psdf_component_min.argtypes = [fp_, i, i, vp, i, fp_, vp]
    L.psdf_trajectory_reduce.restype = i
    L.psdf_trajectory_reduce.argtypes = [fp_, i, i, ctypes.c_float, fp_, vp, fp_, vp]
    L.psdf_cull_stats.restype = i
    L.psdf_cull_stats.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_ulonglong)]
    L.psdf_destroy_scene.restype = None
    L.psdf_destroy_scene.argtypes = [vp]
    L.psdf_scene_num_obstacles.restype = i
    L.psdf_scene_num_obstacles.argtypes = [vp]
    L.psdf_scene_num_edges.restype = i
    L.psdf_scene_num_edges.argtypes = [vp]
    L.psdf_scene_footprint_symmetric.restype = i
    L.psdf_scene_footprint_symmetric.argtypes = [vp]
    L.psdf_last_cuda_error.restype = i
    L.psdf_kernel_launches.restype = ctypes.c_longlong
    L.psdf_status_string.restype = ctypes.c_char_p
    L.psdf_status_string.argtypes = [i]
    L.psdf_version.restype = ctypes.c_char_p
    L.psdf_bench_host_latency.restype = i
    L.psdf_bench_host_latency.argtypes = [vp, fp_, i, fp_, fp_, fp_, fp_, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                          i, ctypes.POINTER(ctypes.c_double)]
    L.psdf_measure_fp32_peak.restype = i
    L.psdf_measure_fp32_peak.argtypes = [i, vp, ctypes.POINTER(ctypes.c_double)]
    _lib = L
    return L


def _check(status, where):
    if status != PSDF_OK:
        raise PsdfError(status, where)


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _dev_ptr(t, dtype_name, shape_last=None):
    import torch
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    assert t.dtype == getattr(torch, dtype_name), f"expected {dtype_name}, got {t.dtype}"
    return t.data_ptr()


def _stream_ptr(stream=None):
    """cudaStream_t of `stream` (a torch.cuda.Stream), else torch's current stream; the
    legacy default stream (NULL) when torch has no CUDA device to ask."""
    if stream is not None:
        return ctypes.c_void_p(stream.cuda_stream)
    try:
        import torch
        if torch.cuda.is_available():
            return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    except ImportError:
        pass
    return ctypes.c_void_p(0)


def psdf_kernel_launches() -> int:
    return int(lib().psdf_kernel_launches())


def psdf_version() -> str:
    return lib().psdf_version().decode()


def psdf_measure_fp32_peak(iters: int = 4096, stream=None) -> float:
    out = ctypes.c_double(0.0)
    _check(lib().psdf_measure_fp32_peak(int(iters), _stream_ptr(stream), ctypes.byref(out)),
           "psdf_measure_fp32_peak")
    return out.value


class Scene:
    """Owns a psdf_scene*.  Methods mirror the C entry points."""

    def __init__(self, footprint, A, B, S, max_poses, stream=None):
        fp, fp_ptr = _host(footprint, np.float32)
        self.V = int(fp.shape[0])
        if _is_torch(A):
            M, E = int(S.shape[0]), int(S.shape[1])
            pa, pb = _dev_ptr(A, "float32"), _dev_ptr(B, "float32")
            ps = _dev_ptr(S, "uint8")
            where = PSDF_MEM_DEVICE
            keep = (A, B, S)
        else:
            A_, pa = _host(A, np.float32)
            B_, pb = _host(B, np.float32)
            S_, ps = _host(S, np.uint8)
            M, E = int(S_.shape[0]), int(S_.shape[1])
            assert A_.shape == (M, E, 2) and B_.shape == (M, E, 2)
            where = PSDF_MEM_HOST
            keep = (A_, B_, S_)
        self.M, self.E, self.max_poses = M, E, int(max_poses)
        self.n_out = M                      # row length of the per-obstacle output (set_components changes it)
        h = ctypes.c_void_p()
        _check(lib().psdf_create_scene(fp_ptr, self.V, pa, pb, ps, M, E, where, int(max_poses),
                                       _stream_ptr(stream), ctypes.byref(h)), "psdf_create_scene")
        del keep
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            lib().psdf_destroy_scene(self._h)
            self._h = None

    def __del__(self):
        # at interpreter shutdown the module globals may already be gone: the process is about
        # to release the device anyway
        try:
            self.close()
        except Exception:
            pass

    @property
    def num_obstacles(self):
        return int(lib().psdf_scene_num_obstacles(self._h))

    @property
    def footprint_symmetric(self):
        """psdf_scene_footprint_symmetric (include/psdf_bench.h)."""
        return bool(lib().psdf_scene_footprint_symmetric(self._h))

    @property
    def num_edges(self):
        return int(lib().psdf_scene_num_edges(self._h))

    def set_culling(self, enable: bool):
        """psdf_set_culling: exact broad-phase culling for large batches (default off)."""
        _check(lib().psdf_set_culling(self._h, int(bool(enable))), "psdf_set_culling")

    def set_components(self, comp_to_obstacle, n_obstacles: int):
        """psdf_set_components: rows are convex components of n_obstacles obstacles (ids non-decreasing);
        per_obstacle outputs become [N, n_obstacles].  n_obstacles = 0 switches back."""
        if n_obstacles:
            comp, pc = _host(comp_to_obstacle, np.int32)
            assert comp.shape == (self.M,)
        else:
            pc = None
        _check(lib().psdf_set_components(self._h, pc, int(n_obstacles)), "psdf_set_components")
        self.n_out = int(n_obstacles) if n_obstacles else self.M

    def eval_trajectories(self, poses, T, H, d_safe, grad=True, stream=None):
        """psdf_eval_trajectories: device poses [T*H,3] -> (value, grad, min_value[T], argmin_stage[T], penalty[T])."""
        import torch
        N = int(T) * int(H)
        assert int(poses.shape[0]) == N
        dev = poses.device
        value = torch.empty(N, dtype=torch.float32, device=dev)
        g = torch.empty((N, 3), dtype=torch.float32, device=dev) if grad else None
        mn = torch.empty(int(T), dtype=torch.float32, device=dev)
        am = torch.empty(int(T), dtype=torch.int32, device=dev)
        pen = torch.empty(int(T), dtype=torch.float32, device=dev)
        _check(lib().psdf_eval_trajectories(self._h, _dev_ptr(poses, "float32"), int(T), int(H), float(d_safe),
                                            _dev_ptr(value, "float32"), _dev_ptr(g, "float32") if grad else None,
                                            _dev_ptr(mn, "float32"), _dev_ptr(am, "int32"), _dev_ptr(pen, "float32"),
                                            _stream_ptr(stream)), "psdf_eval_trajectories")
        return value, g, mn, am, pen

    def cull_stats(self, stream=None):
        """psdf_cull_stats: (evaluated (pose, obstacle) pairs, (pose, edge) steps) since the last call."""
        out = (ctypes.c_ulonglong * 2)()
        _check(lib().psdf_cull_stats(self._h, _stream_ptr(stream), out), "psdf_cull_stats")
        return int(out[0]), int(out[1])

    def update(self, A, B, S, stream=None):
        """psdf_update_scene: same (M,E), values only."""
        if _is_torch(A):
            args = (_dev_ptr(A, "float32"), _dev_ptr(B, "float32"), _dev_ptr(S, "uint8"), PSDF_MEM_DEVICE)
        else:
            A_, pa = _host(A, np.float32)
            B_, pb = _host(B, np.float32)
            S_, ps = _host(S, np.uint8)
            assert S_.shape == (self.M, self.E)
            args = (pa, pb, ps, PSDF_MEM_HOST)
        _check(lib().psdf_update_scene(self._h, *args, _stream_ptr(stream)), "psdf_update_scene")

    def eval(self, poses, value=None, grad=True, per_obstacle=False, stream=None):
        """psdf_eval on device tensors (async on the stream).  `grad` / `per_obstacle` may
        be False (not wanted), True (allocate) or a preallocated tensor."""
        import torch
        N = int(poses.shape[0])
        pp = _dev_ptr(poses, "float32")
        if value is None:
            value = torch.empty(N, dtype=torch.float32, device=poses.device)
        if grad is True:
            grad = torch.empty((N, 3), dtype=torch.float32, device=poses.device)
        if per_obstacle is True:
            per_obstacle = torch.empty((N, self.n_out), dtype=torch.float32, device=poses.device)
        want_g = grad is not False and grad is not None
        want_po = per_obstacle is not False and per_obstacle is not None
        pg = _dev_ptr(grad, "float32") if want_g else None
        po = _dev_ptr(per_obstacle, "float32") if want_po else None
        _check(lib().psdf_eval(self._h, pp, N, _dev_ptr(value, "float32"), pg, po, _stream_ptr(stream)),
               "psdf_eval")
        return value, (grad if want_g else None), (per_obstacle if want_po else None)

    def eval_static_scratch(self, poses, value=None, grad=True, stream=None):
        """psdf_eval_static_scratch: psdf_eval without any allocation inside the library (scratch in a
        static device array; N <= STATIC_SCRATCH_MAX_POSES).  Preallocated `value` / `grad` tensors may be
        passed so that the binding allocates nothing either."""
        import torch
        N = int(poses.shape[0])
        if value is None:
            value = torch.empty(N, dtype=torch.float32, device=poses.device)
        if grad is True:
            grad = torch.empty((N, 3), dtype=torch.float32, device=poses.device)
        want_g = grad is not False and grad is not None
        _check(lib().psdf_eval_static_scratch(self._h, _dev_ptr(poses, "float32"), N, _dev_ptr(value, "float32"),
                                              _dev_ptr(grad, "float32") if want_g else None, _stream_ptr(stream)),
               "psdf_eval_static_scratch")
        return value, (grad if want_g else None)

    def eval_host(self, poses, grad=True, per_obstacle=False):
        """psdf_eval_host on numpy arrays (CUDA-graph replay, returns after sync)."""
        poses, pp = _host(poses, np.float32)
        N = int(poses.shape[0])
        value = np.empty(N, np.float32)
        g = np.empty((N, 3), np.float32) if grad else None
        po = np.empty((N, self.n_out), np.float32) if per_obstacle else None
        _check(lib().psdf_eval_host(self._h, pp, N, value.ctypes.data,
                                    g.ctypes.data if g is not None else None,
                                    po.ctypes.data if po is not None else None), "psdf_eval_host")
        return value, g, po

    def eval_windows(self, poses, row_window, grad=True, stream=None):
        """psdf_eval_windows: device poses [N,3] float32 and row windows [N,2] int32."""
        import torch
        N = int(poses.shape[0])
        value = torch.empty(N, dtype=torch.float32, device=poses.device)
        g = torch.empty((N, 3), dtype=torch.float32, device=poses.device) if grad else None
        _check(lib().psdf_eval_windows(self._h, _dev_ptr(poses, "float32"), N, _dev_ptr(row_window, "int32"),
                                       _dev_ptr(value, "float32"), _dev_ptr(g, "float32") if grad else None,
                                       _stream_ptr(stream)), "psdf_eval_windows")
        return value, g

    def eval_windows_host(self, poses, row_window, grad=True):
        """psdf_eval_windows_host on numpy arrays."""
        poses, pp = _host(poses, np.float32)
        win, pw = _host(row_window, np.int32)
        N = int(poses.shape[0])
        assert win.shape == (N, 2)
        value = np.empty(N, np.float32)
        g = np.empty((N, 3), np.float32) if grad else None
        _check(lib().psdf_eval_windows_host(self._h, pp, N, pw, value.ctypes.data,
                                            g.ctypes.data if grad else None), "psdf_eval_windows_host")
        return value, g

    def eval_host_into(self, poses, value, grad=None, per_obstacle=None):
        """psdf_eval_host into caller-owned contiguous float32 numpy arrays (no allocation in
        the binding: the call an MPC loop makes every control cycle)."""
        N = int(poses.shape[0])
        for a in (poses, value, grad, per_obstacle):
            assert a is None or (a.dtype == np.float32 and a.flags.c_contiguous)
        _check(lib().psdf_eval_host(self._h, poses.ctypes.data, N, value.ctypes.data,
                                    grad.ctypes.data if grad is not None else None,
                                    per_obstacle.ctypes.data if per_obstacle is not None else None),
               "psdf_eval_host")

    def bind_eval_host(self, poses, value, grad=None, per_obstacle=None):
        """psdf_eval_host with the argument marshalling done ONCE: returns a zero-argument
        callable over caller-owned contiguous float32 numpy arrays (an MPC loop rewrites
        `poses` in place every control cycle and calls it; numpy's pointer extraction alone
        costs ~2 us per array per call).  The arrays are kept alive by the callable."""
        N = int(poses.shape[0])
        for a in (poses, value, grad, per_obstacle):
            assert a is None or (a.dtype == np.float32 and a.flags.c_contiguous)
        assert value.shape[0] == N and (grad is None or grad.shape == (N, 3))
        assert per_obstacle is None or per_obstacle.shape == (N, self.n_out)
        fn, h = lib().psdf_eval_host, self._h
        args = (h, poses.ctypes.data, N, value.ctypes.data, grad.ctypes.data if grad is not None else None,
                per_obstacle.ctypes.data if per_obstacle is not None else None)
        keep = (poses, value, grad, per_obstacle)

        def call(_keep=keep):
            status = fn(*args)
            if status != PSDF_OK:
                raise PsdfError(status, "psdf_eval_host")
        return call

    def bind_mpc_coeffs_host(self, poses, coeff, d_min, rho_p, rho_theta):
        """psdf_mpc_coeffs_host, pre-marshalled like bind_eval_host; coeff is [N,4] float32."""
        N = int(poses.shape[0])
        for a in (poses, coeff):
            assert a.dtype == np.float32 and a.flags.c_contiguous
        assert coeff.shape == (N, 4)
        fn = lib().psdf_mpc_coeffs_host
        args = (self._h, poses.ctypes.data, N, float(d_min), float(rho_p), float(rho_theta), coeff.ctypes.data)
        keep = (poses, coeff)

        def call(_keep=keep):
            status = fn(*args)
            if status != PSDF_OK:
                raise PsdfError(status, "psdf_mpc_coeffs_host")
        return call

    def bench_host_latency(self, poses, reps, grad=True, per_obstacle=False, coeffs=None):
        """psdf_bench_host_latency (include/psdf_bench.h): per-call microseconds of psdf_eval_host, or of
        psdf_mpc_coeffs_host when coeffs = (d_min, rho_p, rho_theta), timed inside the library."""
        poses, pp = _host(poses, np.float32)
        N = int(poses.shape[0])
        value = np.empty(N, np.float32)
        g = np.empty((N, 3), np.float32) if grad else None
        po = np.empty((N, self.n_out), np.float32) if per_obstacle else None
        c = np.empty((N, 4), np.float32) if coeffs else None
        d_min, rho_p, rho_theta = coeffs if coeffs else (0.0, 0.0, 0.0)
        out = (ctypes.c_double * int(reps))()
        _check(lib().psdf_bench_host_latency(self._h, pp, N, value.ctypes.data, g.ctypes.data if g is not None else None,
                                             po.ctypes.data if po is not None else None,
                                             c.ctypes.data if c is not None else None, float(d_min), float(rho_p),
                                             float(rho_theta), int(reps), out), "psdf_bench_host_latency")
        return np.frombuffer(out, dtype=np.float64).copy()

    def serve_begin(self, N, coeffs=None, idle_timeout_ms=200, row_window=None):
        """psdf_serve_begin: persistent-kernel serving of batches of exactly N poses; coeffs = (d_min, rho_p,
        rho_theta) for MPC coefficient rows, None for (value, grad) rows; row_window: optional [N,2] int32
        per-pose obstacle row windows, fixed for the session."""
        d_min, rho_p, rho_theta = coeffs if coeffs else (0.0, 0.0, 0.0)
        pw = None
        if row_window is not None:
            win, pw = _host(row_window, np.int32)
            assert win.shape == (int(N), 2)
        _check(lib().psdf_serve_begin(self._h, int(N), pw, 1 if coeffs else 0, float(d_min), float(rho_p),
                                      float(rho_theta), int(idle_timeout_ms)), "psdf_serve_begin")
        self._serve_N = int(N)

    def serve_step(self, poses, out=None):
        """psdf_serve_step: host poses [N,3] -> host rows [N,4]."""
        poses, pp = _host(poses, np.float32)
        assert poses.shape == (self._serve_N, 3)
        if out is None:
            out = np.empty((self._serve_N, 4), np.float32)
        _check(lib().psdf_serve_step(self._h, pp, out.ctypes.data), "psdf_serve_step")
        return out

    def bind_serve_step(self, poses, out):
        """psdf_serve_step pre-marshalled (as bind_eval_host): zero-argument callable over fixed float32 arrays."""
        assert poses.dtype == np.float32 and poses.flags.c_contiguous and poses.shape == (self._serve_N, 3)
        assert out.dtype == np.float32 and out.flags.c_contiguous and out.shape == (self._serve_N, 4)
        fn, args, keep = lib().psdf_serve_step, (self._h, poses.ctypes.data, out.ctypes.data), (poses, out)

        def call(_keep=keep):
            status = fn(*args)
            if status != PSDF_OK:
                raise PsdfError(status, "psdf_serve_step")
        return call

    def serve_end(self):
        _check(lib().psdf_serve_end(self._h), "psdf_serve_end")

    def bench_serve_latency(self, poses, reps):
        """psdf_bench_serve_latency (include/psdf_bench.h): per-step microseconds, timed inside the library."""
        poses, pp = _host(poses, np.float32)
        out4 = np.empty((self._serve_N, 4), np.float32)
        out = (ctypes.c_double * int(reps))()
        _check(lib().psdf_bench_serve_latency(self._h, pp, out4.ctypes.data, int(reps), out), "psdf_bench_serve_latency")
        return np.frombuffer(out, dtype=np.float64).copy()

    def mpc_coeffs_host(self, poses, d_min, rho_p, rho_theta):
        poses, pp = _host(poses, np.float32)
        N = int(poses.shape[0])
        coeff = np.empty((N, 4), np.float32)
        _check(lib().psdf_mpc_coeffs_host(self._h, pp, N, float(d_min), float(rho_p), float(rho_theta),
                                          coeff.ctypes.data), "psdf_mpc_coeffs_host")
        return coeff


def psdf_create_scene(footprint, A, B, S, max_poses, stream=None) -> Scene:
    return Scene(footprint, A, B, S, max_poses, stream)


def psdf_eval(scene: Scene, poses, **kw):
    return scene.eval(poses, **kw)


def psdf_eval_host(scene: Scene, poses, **kw):
    return scene.eval_host(poses, **kw)


def psdf_eval_windows(scene: Scene, poses, row_window, **kw):
    return scene.eval_windows(poses, row_window, **kw)


def psdf_eval_windows_host(scene: Scene, poses, row_window, **kw):
    return scene.eval_windows_host(poses, row_window, **kw)


def psdf_update_scene(scene: Scene, A, B, S, stream=None):
    return scene.update(A, B, S, stream)


def psdf_mpc_coeffs_host(scene: Scene, poses, d_min, rho_p, rho_theta):
    return scene.mpc_coeffs_host(poses, d_min, rho_p, rho_theta)


def psdf_component_min(per_component, comp_to_obstacle, n_obstacles, stream=None):
    """per_component: CUDA float32 [N,M]; comp_to_obstacle: CUDA int32 [M] -> float32 [N,n_obstacles]."""
    import torch
    N, M = int(per_component.shape[0]), int(per_component.shape[1])
    out = torch.empty((N, int(n_obstacles)), dtype=torch.float32, device=per_component.device)
    _check(lib().psdf_component_min(_dev_ptr(per_component, "float32"), N, M, _dev_ptr(comp_to_obstacle, "int32"),
                                    int(n_obstacles), _dev_ptr(out, "float32"), _stream_ptr(stream)),
           "psdf_component_min")
    return out


def psdf_trajectory_reduce(value, T, H, d_safe, stream=None):
    """value: CUDA float32 [T*H] -> (min_value[T], argmin_stage[T] int32, penalty[T])."""
    import torch
    assert value.numel() == int(T) * int(H)
    mn = torch.empty(int(T), dtype=torch.float32, device=value.device)
    am = torch.empty(int(T), dtype=torch.int32, device=value.device)
    pen = torch.empty(int(T), dtype=torch.float32, device=value.device)
    _check(lib().psdf_trajectory_reduce(_dev_ptr(value, "float32"), int(T), int(H), float(d_safe),
                                        _dev_ptr(mn, "float32"), _dev_ptr(am, "int32"), _dev_ptr(pen, "float32"),
                                        _stream_ptr(stream)), "psdf_trajectory_reduce")
    return mn, am, pen


def psdf_set_components(scene: Scene, comp_to_obstacle, n_obstacles: int):
    return scene.set_components(comp_to_obstacle, n_obstacles)


def psdf_eval_trajectories(scene: Scene, poses, T, H, d_safe, **kw):
    return scene.eval_trajectories(poses, T, H, d_safe, **kw)


def psdf_set_culling(scene: Scene, enable: bool):
    return scene.set_culling(enable)


def psdf_destroy_scene(scene: Scene):
    scene.close()
