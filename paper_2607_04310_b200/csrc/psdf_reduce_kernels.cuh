// Reductions on top of the PSDF outputs:
//   * component_min_kernel: non-convex obstacles are given as several convex components
//     (Assumption 1; eq.(6) PAPER.md:93-97 minimises over all components); this
//     folds per-component values sd^i [N,M] into per-obstacle values [N,n_obstacles] through a
//     component -> obstacle id map;
//   * trajectory_reduce_kernel: sampled-trajectory batches (N = T trajectories x H stages, pose
//     index = traj * H + stage): clearance min_s phi_s with its first arg-min stage and the soft
//     penalty sum_s max(0, d_safe - phi_s)^2, one warp per trajectory, fixed reduction order
//     (deterministic).
#pragma once
#include "psdf_device.cuh"

namespace psdf {

// one thread per (pose, obstacle): scans the components (M is small when per-obstacle output
// is wanted); id outside [0, n_obstacles) is ignored.
__global__ void component_min_kernel(const float* __restrict__ per_component, int N, int M,
                                     const int* __restrict__ comp_to_obstacle, int n_obstacles,
                                     float* __restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)N * n_obstacles) return;
  const int n = (int)(t / n_obstacles), o = (int)(t % n_obstacles);
  const float* row = per_component + (size_t)n * M;
  float m = kInf;
  for (int i = 0; i < M; ++i)
    if (__ldg(comp_to_obstacle + i) == o) m = fminf(m, __ldg(row + i));
  out[t] = m;
}

__global__ void trajectory_reduce_kernel(const float* __restrict__ value, int T, int H, float d_safe,
                                         float* __restrict__ min_value, int* __restrict__ argmin_stage,
                                         float* __restrict__ penalty) {
  const int lane = threadIdx.x & 31;
  const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (t >= T) return;
  const float* v = value + (size_t)t * H;
  unsigned long long best = ~0ull;          // (ordered key of phi) << 32 | stage: min = first arg-min
  float pen = 0.f;
  for (int s = lane; s < H; s += 32) {
    const float phi = __ldg(v + s);
    const unsigned long long key = ((unsigned long long)fkey(phi) << 32) | (unsigned)s;
    best = key < best ? key : best;
    const float d = fmaxf(d_safe - phi, 0.f);
    pen = fmaf(d, d, pen);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
    best = other < best ? other : best;
    pen += __shfl_xor_sync(0xffffffffu, pen, o);
  }
  if (lane == 0) {
    if (min_value) min_value[t] = H > 0 ? fkey_inv((uint32_t)(best >> 32)) : kInf;
    if (argmin_stage) argmin_stage[t] = H > 0 ? (int)(uint32_t)best : -1;
    if (penalty) penalty[t] = pen;
  }
}

}  // namespace psdf
