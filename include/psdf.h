/* psdf.h — C ABI of the B200-native PSDF hot path (arxiv/paper_2607_04310).
 *
 * What is computed (citations are PAPER.md line numbers, /root/reference/PAPER.md):
 *   the polygonal signed distance function
 *       phi(x, E) = min_i sd(P0(x), P^i)                               eq.(6)
 *   of a convex robot footprint posed at x = (p, theta),
 *       P0(x) = { R(theta) v + p | v in co(V0) }                       eq.(9)
 *   against the convex obstacle components encoded in the padded edge tensors
 *       A, B in R^{M x E x 2},  S in {0,1}^{M x E}                     eq.(10)
 *   where sd = dist - pen (eqs.(5a-c)) is evaluated exactly: point-to-
 *   segment minima over both vertex/edge pools when separated (eqs.(12)-(16),
 *   PAPER.md:153-177), SAT minimum overlap over both polygons' edge normals when not
 *   (eqs.(17)-(22)), selected by eq.(23); together
 *   with the state gradient d phi / d(x, y, theta), here the analytic
 *   gradient at the arg-min witness instead of an autodiff backward pass.
 *
 * Conventions.  Row-major, float32, metres / radians.  Every function returns a
 * psdf_status (0 ok, <0 error); nothing throws, aborts or prints.  On error the outputs
 * are untouched.  "device" pointers are CUDA device memory of the current device,
 * "host" pointers ordinary host memory.  `cuda_stream` is a cudaStream_t passed as
 * void* (NULL = legacy default stream).  The caller owns every I/O buffer and the stream;
 * the library copies the scene at create/update and owns that copy.
 *
 * Ordering and thread-safety (different scenes are always independent):
 *   - one host thread at a time per scene: a call that finds the scene inside another call of
 *     another thread returns PSDF_ERR_BUSY and does nothing;
 *   - the stream-taking evaluation calls (psdf_eval, psdf_eval_windows) share one small device
 *     workspace per scene: on one scene they must be ordered on ONE stream, or by the caller's own
 *     events; each only enqueues and returns;
 *   - the *_host calls run on the scene's own stream with a workspace of their own and return
 *     after synchronising it: they may be issued while an asynchronous psdf_eval of the same scene
 *     is still in flight on the caller's stream;
 *   - psdf_update_scene / psdf_set_culling wait for the scene's own stream; an update orders itself
 *     after earlier psdf_eval work by stream order when it is given the stream those calls used,
 *     and by a device-wide synchronisation when they used another one;
 *   - psdf_eval may be captured into a caller's CUDA graph (it only enqueues one kernel).  The
 *     captured node holds the scene's buffers and launch plan by value: such a graph must be
 *     captured again after psdf_update_scene or psdf_set_culling, and its replays ordered against
 *     updates by the caller.
 */
#ifndef PSDF_H_
#define PSDF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psdf_scene psdf_scene; /* opaque; owns packed device scene + workspace + graph */

typedef enum {
  PSDF_OK = 0,
  PSDF_ERR_INVALID_ARG = -1, /* null pointer, V outside [3,16], E<3, M<1, N<0 */
  PSDF_ERR_DEGENERATE = -2,  /* violates Assumption 1: edge shorter than 1e-6 m,
                                non-empty row with <3 valid edges, row that is not a closed
                                convex polygon, footprint not convex counter-clockwise */
  PSDF_ERR_CAPACITY = -3,    /* N > max_poses given at create */
  PSDF_ERR_CUDA = -4,        /* a CUDA call failed (psdf_last_cuda_error() has the code) */
  PSDF_ERR_ALLOC = -5,       /* host or device memory allocation failed */
  PSDF_ERR_BUSY = -6         /* the scene is inside another call of another host thread */
} psdf_status;

typedef enum { PSDF_MEM_HOST = 0, PSDF_MEM_DEVICE = 1 } psdf_mem;

/* EncodeEdges + upload (Alg.1 l.1-4; eq.(10)).
 *   footprint  host [V,2]   robot vertices in the robot-local frame, CCW
 *   A, B       [M,E,2]      edge start / end points, world frame; `where` says host or device
 *   S          [M,E] uint8  1 = valid edge, 0 = padded entry (any position, any garbage
 *                           in A/B there); a row with no valid entry is an absent obstacle
 *   max_poses  capacity for N in later psdf_eval / psdf_eval_host calls
 * Valid entries of a row, in slot order, must form one closed convex polygon
 * (B_j == A_next bitwise), either orientation.  Blocks until the upload has finished. */
psdf_status psdf_create_scene(const float* footprint, int V, const float* A, const float* B,
                              const uint8_t* S, int M, int E, psdf_mem where, int max_poses,
                              void* cuda_stream, psdf_scene** out);

/* Perception update: same (M,E), new values only.  On error the old scene
 * stays in force.  Blocks until the upload has finished. */
psdf_status psdf_update_scene(psdf_scene* scene, const float* A, const float* B, const uint8_t* S,
                              psdf_mem where, void* cuda_stream);

/* Batched evaluation (Alg.1 l.5-7), asynchronous on `cuda_stream`:
 * no host synchronisation, no allocation.
 *   poses         device [N,3]  (x, y, theta) per pose
 *   value         device [N]    phi                                    eq.(6)
 *   grad          device [N,3]  (d phi/dx, d phi/dy, d phi/dtheta), PLUS sign (the paper's
 *                               J_g = -grad);  NULL = value-only
 *   per_obstacle  device [N,M]  sd^i per obstacle row (eq.23), +INF for a row with no valid
 *                               edge ([N,n_obstacles] after psdf_set_components);  NULL = not wanted
 * No valid obstacle at all: value=+INF, grad=0.  Non-finite pose: NaN outputs.
 * At ties / kinks the gradient is that of one of the tied branches. */
psdf_status psdf_eval(const psdf_scene* scene, const float* poses, int N, float* value, float* grad,
                      float* per_obstacle, void* cuda_stream);

/* psdf_eval for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the chunked tile-scan evaluation with its scratch memory (cross-chunk
 * keys, arrival counters) in a file-scope static device array of the library, 1.03 MB, which every GPU
 * that loads the library holds until exit.  Same outputs as psdf_eval (value [N], grad [N,3] or NULL:
 * bit-identical), no per_obstacle output, no culling.  N > PSDF_STATIC_SCRATCH_MAX_POSES returns
 * PSDF_ERR_CAPACITY and does nothing.  The call itself enqueues three memsets of the scratch it will use
 * and one kernel on `cuda_stream`; it calls no cudaMalloc, cudaFree or allocating routine (the scene was
 * created beforehand; the first call on a device also looks the array's device address up, once).
 * ALL calls of the process on one GPU share the array, whatever scene they use: two such calls that overlap
 * on the GPU (different streams without an ordering between them) race and give wrong results; calls
 * ordered on one stream, or by events, are fine. */
#define PSDF_STATIC_SCRATCH_MAX_POSES 65536
psdf_status psdf_eval_static_scratch(const psdf_scene* scene, const float* poses, int N, float* value,
                                     float* grad, void* cuda_stream);

/* Same semantics with HOST buffers (Alg.1 l.5-11: upload the nominal states,
 * evaluate, bring the results back), on the scene's own stream; returns after synchronising it.
 * MPC-sized batches (N <= 512; with per_obstacle only up to 64 obstacles): ONE kernel launch; up
 * to 128 poses travel inside the launch, results are written to pinned, device-mapped staging, where
 * the host watches the rows arrive (no stream synchronise unless per_obstacle is wanted), and copied out.  Larger batches: replay of a captured CUDA graph of up to four branches
 * {H2D pose chunk, kernel, D2H result chunk} that overlap copies and kernels.  Buffers in pinned
 * (page-locked) host memory are read and written in place by the copy engines; ordinary memory
 * goes through the scene's pinned staging (one extra host copy each way); with culling on and pinned
 * buffers one kernel reads and writes them itself, without the copy engines.  Results are
 * bit-identical to psdf_eval on the same poses.  grad / per_obstacle may be NULL. */
psdf_status psdf_eval_host(psdf_scene* scene, const float* poses, int N, float* value, float* grad,
                           float* per_obstacle);

/* Serving mode for one fixed MPC batch shape (Alg.1 l.5-11: every control cycle uploads
 * the N nominal states and brings N coefficient rows back; N = 15 in the paper): a PERSISTENT
 * kernel and a mailbox in pinned, device-mapped memory, so that a cycle costs neither a kernel launch nor a
 * stream synchronisation.
 *   psdf_serve_begin   starts the kernel on a stream of its own for batches of exactly N poses
 *                      (N <= 512 and at most 128 pose groups, else PSDF_ERR_INVALID_ARG: use psdf_eval_host);
 *                      row_window: NULL, or host [N,2] int32 obstacle ROW windows as in psdf_eval_windows,
 *                      fixed for the session (time-varying environments: stage s sees the rows
 *                      of E_{k+s}; the mapping stays, psdf_update_scene brings the new values);
 *                      want_coeffs = 0: rows (phi, d phi/dx, d phi/dy, d phi/dtheta) as psdf_eval_host;
 *                      want_coeffs = 1: rows [h - gamma ; J_g] as psdf_mpc_coeffs_host with d_min, rho_p,
 *                      rho_theta.  idle_timeout_ms in [1, 10000]: a kernel that sees no request for that
 *                      long exits by itself (the next step starts it again, at the cost of one launch).
 *   psdf_serve_step    poses host [N,3] -> out host [N,4]; posts the poses, spins until every row has
 *                      arrived (the rows are blanked with a NaN pattern no result carries and watched
 *                      word by word: no fence, no acknowledgement), copies the rows out.  Results are bit-identical to psdf_eval_host /
 *                      psdf_mpc_coeffs_host.  Ordinary host memory is fine (N is small).
 *   psdf_serve_end     stops the kernel (psdf_destroy_scene does it too).
 * While the kernel runs it occupies a few CTAs and polls host memory over PCIe; a device-wide
 * synchronisation (cudaDeviceSynchronize, cudaFree) issued meanwhile waits until it exits, i.e. until
 * psdf_serve_end or the idle time-out.  psdf_update_scene, psdf_set_culling and psdf_set_components stop it
 * themselves and the next psdf_serve_step restarts it on the new scene; every other call of this header may
 * be used next to it.  Allocates (pinned memory, the window table) in psdf_serve_begin only. */
psdf_status psdf_serve_begin(psdf_scene* scene, int N, const int* row_window, int want_coeffs, float d_min,
                             float rho_p, float rho_theta, int idle_timeout_ms);
psdf_status psdf_serve_step(psdf_scene* scene, const float* poses, float* out);
psdf_status psdf_serve_end(psdf_scene* scene);

/* Time-varying environments ("batching {(x_{k+s}, E_{k+s})} instead"): the scene
 * holds the rows of all stage-wise edge sets one after another (e.g. M = H * M_stage rows) and
 * pose n is evaluated against the obstacle ROWS row_window[2n] <= i < row_window[2n+1] only
 * (clamped to [0, M]; an empty window gives value=+INF, grad=0).  Same outputs and conventions as
 * psdf_eval; row_window is a device [N,2] int32 array (host array for the _host variant, which
 * copies, evaluates on the scene's stream and synchronises).  Meant for MPC-sized batches: one
 * group of lanes per pose, any N <= max_poses. */
psdf_status psdf_eval_windows(const psdf_scene* scene, const float* poses, int N, const int* row_window,
                              float* value, float* grad, void* cuda_stream);
psdf_status psdf_eval_windows_host(psdf_scene* scene, const float* poses, int N, const int* row_window,
                                   float* value, float* grad);

/* MPC coefficient epilogue (Alg.1 l.7-11; eqs.(26)-(28)):
 * for each stage s writes coeff[s] = [ h_s - gamma_s ; J_g,s ] with h_s = phi_s - d_min,
 * J_g,s = -grad phi_s, gamma_s = 0.5 (r_max + phi_s) rho_theta^2 + rho_p rho_theta,
 * r_max = max_l |v_l|.  coeff: host [N,4].  A stage that sees no obstacle (phi = +INF, e.g. an
 * obstacle-free perception frame) gives the inactive row (+INF, 0, 0, 0), never NaN; a non-finite
 * pose gives NaN.  Same host path as psdf_eval_host. */
psdf_status psdf_mpc_coeffs_host(psdf_scene* scene, const float* poses, int N, float d_min,
                                 float rho_p, float rho_theta, float* coeff);

/* Exact broad-phase culling (beyond the paper; valid because phi is a minimum over obstacles,
 * eq.(6)).  When enabled, large batches (N > 2048, >= 64 obstacles) evaluated without
 * per_obstacle output go through one kernel that looks obstacles up in a uniform grid (rebuilt on
 * the device at every create/update) and skips every obstacle whose lower bound on sd^i (bounding
 * circles, then oriented bounding boxes of footprint and obstacle) exceeds an upper bound of phi
 * obtained from a nearby obstacle (the grid is built when culling is switched on and kept current by
 * every update from then on); surviving pairs use the same arithmetic and reductions as the
 * dense path, so value and grad are bit-identical to the dense result.  Default: disabled (dense,
 * branch-free evaluation). */
psdf_status psdf_set_culling(psdf_scene* scene, int enable);

/* Non-convex obstacles given as convex components (Assumption 1: "non-convex = union of
 * convex pieces"; eq.(6)), fused form: declares that the obstacle rows are components
 * of n_obstacles obstacles, comp_to_obstacle host [M] giving the obstacle id of every row,
 * non-decreasing and within [0, n_obstacles), n_obstacles <= M (the components of one obstacle are consecutive rows;
 * anything else is PSDF_ERR_INVALID_ARG).  From then on the `per_obstacle` output of psdf_eval and
 * psdf_eval_host is [N, n_obstacles] with per_obstacle[n,o] = min over the valid rows of obstacle o
 * (+INF if it has none), folded inside the evaluation kernels: no [N,M] array is formed.  value and
 * grad are unaffected (eq.(6) is a minimum over all components anyway).  n_obstacles = 0 switches
 * back to one value per row.  Synchronises the device. */
psdf_status psdf_set_components(psdf_scene* scene, const int* comp_to_obstacle, int n_obstacles);

/* Stand-alone form for any map: folds the per-component values of psdf_eval's `per_obstacle` output,
 * per_component device [N,M], into out device [N,n_obstacles] with
 * out[n,o] = min over rows i with comp_to_obstacle[i] == o (+INF if none); comp_to_obstacle is a
 * device [M] int32 array, ids outside [0,n_obstacles) are ignored.  Asynchronous on the stream. */
psdf_status psdf_component_min(const float* per_component, int N, int M, const int* comp_to_obstacle,
                               int n_obstacles, float* out, void* cuda_stream);

/* Sampled-trajectory batches, fused form: psdf_eval on the T*H poses (pose index = trajectory * H +
 * stage; value device [T*H], grad device [T*H,3] or NULL) with the per-trajectory reductions of
 * psdf_trajectory_reduce computed by the same launch (the CTA that completes a trajectory reduces it:
 * same routine, same bits as the stand-alone call).  Any of min_value / argmin_stage / penalty
 * (device [T]) may be NULL.  T*H <= max_poses.  Asynchronous on the stream. */
psdf_status psdf_eval_trajectories(const psdf_scene* scene, const float* poses, int T, int H, float d_safe,
                                   float* value, float* grad, float* min_value, int* argmin_stage,
                                   float* penalty, void* cuda_stream);

/* Stand-alone form (pose index = trajectory * H + stage): per trajectory the clearance
 * min_value[t] = min_s phi, its first arg-min stage, and the soft penalty
 * penalty[t] = sum_s max(0, d_safe - phi_s)^2 (fixed summation order: deterministic).  value is
 * psdf_eval's device [T*H] output; any of the three device outputs may be NULL. */
psdf_status psdf_trajectory_reduce(const float* value, int T, int H, float d_safe, float* min_value,
                                   int* argmin_stage, float* penalty, void* cuda_stream);

void psdf_destroy_scene(psdf_scene* scene);

/* Introspection (no CUDA work). */
int psdf_scene_num_obstacles(const psdf_scene* scene);   /* rows with >=1 valid edge */
int psdf_scene_num_edges(const psdf_scene* scene);       /* total valid edges */
int psdf_last_cuda_error(void);                          /* cudaError_t of the last failure */
const char* psdf_status_string(psdf_status status);
const char* psdf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSDF_H_ */
