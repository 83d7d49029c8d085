/* psdf_bench.h — measurement instrumentation of libpsdf.so, used by bench.py and the tests.
 * NOT part of the product ABI of include/psdf.h: nothing here computes
 * any part of the PSDF path.  Same library, same conventions (psdf_status, void* cuda_stream).
 */
#ifndef PSDF_BENCH_H_
#define PSDF_BENCH_H_

#include "psdf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Kernels launched by this library since it was loaded (a replayed CUDA graph counts its kernel
 * nodes): bench.py's `gpu_launches`. */
long long psdf_kernel_launches(void);

/* 1 if the scene's footprint was found centrally symmetric about its reference point at create
 * (v_{l+V/2} == -v_l bitwise, V a multiple of 4): the kernels then take the edge step that derives half of
 * the dot products from the other half.  Tests use it to know which variant ran. */
int psdf_scene_footprint_symmetric(const psdf_scene* scene);

/* Culled-path statistics (psdf_set_culling) accumulated since the last call (then reset):
 * out2[0] = number of evaluated (pose, obstacle) pairs, out2[1] = number of (pose, obstacle edge)
 * steps, over the stream-taking and the host entry points.  Synchronises `cuda_stream` and the
 * scene's own stream.  bench.py: evaluated-pair fraction and FLOPs of the culled path. */
psdf_status psdf_cull_stats(psdf_scene* scene, void* cuda_stream, unsigned long long* out2);

/* End-to-end latency of the host entry points measured INSIDE the library (steady_clock around the
 * C-ABI call, no interpreter in the timed region): `reps` calls of psdf_mpc_coeffs_host (coeff != NULL,
 * with d_min, rho_p, rho_theta) or of psdf_eval_host (value, grad, per_obstacle as there), one
 * duration in microseconds per call written to out_us[reps]. */
psdf_status psdf_bench_host_latency(psdf_scene* scene, const float* poses, int N, float* value, float* grad,
                                    float* per_obstacle, float* coeff, float d_min, float rho_p, float rho_theta,
                                    int reps, double* out_us);

/* The same for psdf_serve_step (serving mode begun by psdf_serve_begin): `reps` steps on the same poses,
 * one duration in microseconds per step. */
psdf_status psdf_bench_serve_latency(psdf_scene* scene, const float* poses, float* out, int reps, double* out_us);

/* FP32 FMA-only micro-kernel: achieved TFLOP/s on the current device (bench.py reports it beside
 * the nominal FP32 peak, MEASURED_PEAKS.json holding no FP32 figure). */
psdf_status psdf_measure_fp32_peak(int iters, void* cuda_stream, double* tflops_out);

#ifdef __cplusplus
}
#endif
#endif /* PSDF_BENCH_H_ */
